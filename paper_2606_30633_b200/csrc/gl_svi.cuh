// gl_svi.cuh -- SURVEY 8(f) NEXT-2: one SVI iteration around the hot path (Fig. 1).
//   draws z_i = mu + L xi_i (reparameterised; xi supplied by the caller)  ->  gl_logpost_grad on the draws (the hot path)
//   -> fixed-order reduction over the draws of g_i and g_i xi_i^T (this replaces the paper's cross-device pmean, Fig. 1
//   box 5: one GPU holds all n_VI draws)  ->  loss gradient w.r.t. (mu, packed lower-triangular L) and optimiser update.
// Readings: DESIGN.md section 12.  fp64 arithmetic on fp32 storage; no atomics (two-level fixed-order sums).
#pragma once
#include "gl_common.cuh"
#include "gl_particle.cuh"

namespace gl {

constexpr int SVI_NCHUNK = 32;          // first-level partial sums over the draws

// z[i][j] = mu[j] + sum_{k<=j} L[j][k] xi[i][k].  One thread per (draw, parameter).
__global__ void gl_svi_draw_kernel(int64_t n, int np, const float* __restrict__ mu, const float* __restrict__ Lp,
                                   const float* __restrict__ xi, float* __restrict__ z) {
    const int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= n * np) return;
    const int64_t i = e / np;
    const int j = (int)(e - i * np);
    const float* row = Lp + (size_t)j * (j + 1) / 2;
    const float* x = xi + i * np;
    double acc = (double)mu[j];
    for (int k = 0; k <= j; ++k) acc = fma((double)row[k], (double)x[k], acc);
    z[e] = (float)acc;
}

// Row of packed lower-triangle index t (t = j (j + 1) / 2 + k, k <= j).
__device__ __forceinline__ int tril_row(int t) {
    int j = 0;
    while ((j + 1) * (j + 2) / 2 <= t) ++j;
    return j;
}

// Slot q of the reduction: 0 = sum of logp over the finite draws, 1 = their count, 2 + j = sum_i g_ij,
// 2 + np + tril(j, k) = sum_i g_ij xi_ik.  grid = (ceil(nslot / 128), SVI_NCHUNK); part: [SVI_NCHUNK][nslot] doubles.
__global__ void gl_svi_reduce_kernel(int64_t n, int np, const float* __restrict__ logp, const float* __restrict__ grad,
                                     const float* __restrict__ xi, double* __restrict__ part) {
    const int ntril = np * (np + 1) / 2, nslot = 2 + np + ntril;
    const int q = blockIdx.x * blockDim.x + threadIdx.x;
    if (q >= nslot) return;
    const int64_t per = (n + SVI_NCHUNK - 1) / SVI_NCHUNK, i0 = blockIdx.y * per, i1 = (i0 + per < n) ? i0 + per : n;
    int j = 0, k = -1;
    if (q >= 2 + np) {                   // packed row-major lower triangle: t = j (j + 1) / 2 + k
        const int t = q - 2 - np;
        j = tril_row(t);
        k = t - j * (j + 1) / 2;
    } else if (q >= 2) j = q - 2;
    double s = 0.0;
    for (int64_t i = i0; i < i1; ++i) {
        const float lp = logp[i];
        if (!isfinite(lp)) continue;
        if (q == 0) s += (double)lp;
        else if (q == 1) s += 1.0;
        else if (k < 0) s += (double)grad[i * np + j];
        else s = fma((double)grad[i * np + j], (double)xi[i * np + k], s);
    }
    part[(size_t)blockIdx.y * nslot + q] = s;
}

__device__ __forceinline__ double svi_total(const double* __restrict__ part, int nslot, int q) {
    double s = 0.0;
    for (int c = 0; c < SVI_NCHUNK; ++c) s += part[(size_t)c * nslot + q];
    return s;
}

// Second-level sums, loss, loss gradient and optimiser update of theta = [mu; packed L].  ONE block of 256 threads.
// out_stats[0] = loss (Eq. 2 estimate), out_stats[1] = number of finite draws.
// dead: bit j set = dimension j is not part of the surrogate (a solved amplitude of backward modelling, whose log p~
// gradient is identically zero): its mu_j, every L entry of row or column j and their optimiser
// state are left untouched, and log L_jj / the (1/2) log 2 pi e of that dimension stay out of the loss.
__global__ void __launch_bounds__(256) gl_svi_update_kernel(const __grid_constant__ OptParams o, const __grid_constant__ DimMask dead, int np,
                                                            const double* __restrict__ part, float* __restrict__ mu,
                                                            float* __restrict__ Lp, float* __restrict__ m,
                                                            float* __restrict__ v, float* __restrict__ out_stats,
                                                            const double* __restrict__ diag_coef = nullptr) {
    // diag_coef: coefficient of the -1 / L_jj term of d loss / d L_jj: 1 for the pathwise estimator (NULL), (1/N) sum_i c_i for
    // the score-function estimator (gl_svi_score_* kernels below), read from device memory
    const int ntril = np * (np + 1) / 2, nslot = 2 + np + ntril;
    const double dcoef = diag_coef ? diag_coef[0] : 1.0;
    __shared__ double s_logdiag;
    const double N = svi_total(part, nslot, 1);                  // every thread: same fixed-order sum, same value
    if (threadIdx.x == 0) {                                      // sum_j log |L_jj| from the OLD L, fixed order
        double l = 0.0;
        for (int j = 0; j < np; ++j) if (!dead.test(j)) l += log(fabs((double)Lp[(size_t)j * (j + 1) / 2 + j]));
        s_logdiag = l;
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        const double loss = N > 0 ? -s_logdiag - 0.5 * (np - dead.count(np)) * 2.8378770664093453 - svi_total(part, nslot, 0) / N : INFINITY;
        out_stats[0] = (float)loss; out_stats[1] = (float)N;     // 2.8378... = 1 + ln 2 pi
    }
    if (!(N > 0)) return;
    for (int e = threadIdx.x; e < np + ntril; e += blockDim.x) {  // each thread owns its parameters
        double g = -svi_total(part, nslot, 2 + e) / N;            // d loss / d theta_e
        float* th = e < np ? mu + e : Lp + (e - np);
        if (e >= np) {
            const int t = e - np, j = tril_row(t), k = t - j * (j + 1) / 2;
            if (dead.test(j) || dead.test(k)) continue;
            if (k == j) g -= dcoef / (double)*th;
        } else if (dead.test(e)) continue;
        const double m1 = o.b1 * (double)m[e] + (1.0 - o.b1) * g;
        const double d = o.kind == 1 ? g - m1 : g;
        const double v1 = o.b2 * (double)v[e] + (1.0 - o.b2) * d * d + (o.kind == 1 ? o.eps_root : 0.0);
        const double t1 = (double)*th - o.lr * (m1 * o.c1) / (sqrt(v1 * o.c2) + o.eps);
        m[e] = (float)m1; v[e] = (float)v1; *th = (float)t1;
    }
}

// ----------------------------------------------------------------------------- score-function estimator (Eq. 3 as printed)
// grad_phi loss = (1/N) sum_i c_i grad_phi log q~(z_i), c_i = w_i - b_i, w_i = log q~(z_i) - log p~(z_i); needs log p~ only.
//   log q~(z_i) = -1/2 |xi_i|^2 - sum_j log L_jj - (n/2) log 2 pi;  d log q~/d mu_j = s_j,  d log q~/d L_jk = s_j xi_k - delta_jk / L_jj,
//   s = L^-T xi.  Readings: DESIGN.md section 12 (b_i = 0: as printed; leave-one-out mean: c_i = N/(N-1) (w_i - mean w)).
// The kernels below turn that into the quantities the pathwise path already reduces: a "pseudo-gradient" row
// G_i = -c_i s_i in place of grad log p~(z_i), so that gl_svi_reduce_kernel's sums of G_ij and G_ij xi_ik and
// gl_svi_update_kernel (with diag_coef = (1/N) sum_i c_i) produce exactly the score-function gradient.

// w_i for every draw (NaN marks a draw with a non-finite log p~).  One thread per draw.
__global__ void gl_svi_score_w_kernel(int64_t n, int np, const float* __restrict__ logp, const float* __restrict__ xi,
                                      const float* __restrict__ Lp, double* __restrict__ w) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const float lp = logp[i];
    if (!isfinite(lp)) { w[i] = nan(""); return; }
    double q = 0.0, ld = 0.0;
    for (int j = 0; j < np; ++j) {
        const double x = (double)xi[i * np + j];
        q = fma(x, x, q);
        ld += log(fabs((double)Lp[(size_t)j * (j + 1) / 2 + j]));
    }
    w[i] = -0.5 * q - ld - 0.5 * np * 1.8378770664093453 - (double)lp;         // ln 2 pi
}

// fixed-order sum over a strided subset per thread, then a fixed tree; ONE block of 256 threads
__device__ __forceinline__ double svi_block_sum(double v, double* sm) {
    sm[threadIdx.x] = v;
    __syncthreads();
    for (int o = 128; o > 0; o >>= 1) { if (threadIdx.x < o) sm[threadIdx.x] += sm[threadIdx.x + o]; __syncthreads(); }
    const double r = sm[0];
    __syncthreads();
    return r;
}
// w (in place) -> c;  scal[0] = (1/N) sum_i c_i (the diagonal coefficient), scal[1] = N, scal[2] = mean w
__global__ void __launch_bounds__(256) gl_svi_score_c_kernel(int64_t n, int baseline, double* __restrict__ w, double* __restrict__ scal) {
    __shared__ double sm[256];
    double sw = 0.0, cnt = 0.0;
    for (int64_t i = threadIdx.x; i < n; i += 256) { const double x = w[i]; if (x == x) { sw += x; cnt += 1.0; } }
    const double N = svi_block_sum(cnt, sm), W = svi_block_sum(sw, sm);
    const double wbar = N > 0 ? W / N : 0.0, f = (baseline && N > 1) ? N / (N - 1.0) : 1.0;
    double sc = 0.0;
    for (int64_t i = threadIdx.x; i < n; i += 256) {
        const double x = w[i];
        const double c = (x == x) ? (baseline ? f * (x - wbar) : x) : 0.0;
        w[i] = c; sc += c;
    }
    const double C = svi_block_sum(sc, sm);
    if (threadIdx.x == 0) { scal[0] = N > 0 ? C / N : 0.0; scal[1] = N; scal[2] = wbar; }
}

// G_i = -c_i L^-T xi_i (back-substitution, fp64), stored as the fp32 "gradient" rows the reduction reads.  One thread per draw.
__global__ void gl_svi_score_grad_kernel(int64_t n, int np, const float* __restrict__ Lp, const float* __restrict__ xi,
                                         const double* __restrict__ c, float* __restrict__ g) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    double s[128];
    const double ci = c[i];
    for (int j = np - 1; j >= 0; --j) {               // s_j = (xi_j - sum_{k > j} L_kj s_k) / L_jj
        double a = (double)xi[i * np + j];
        for (int k = j + 1; k < np; ++k) a = fma(-(double)Lp[(size_t)k * (k + 1) / 2 + j], s[k], a);
        s[j] = a / (double)Lp[(size_t)j * (j + 1) / 2 + j];
    }
    for (int j = 0; j < np; ++j) g[i * np + j] = (float)(-ci * s[j]);
}

}  // namespace gl
