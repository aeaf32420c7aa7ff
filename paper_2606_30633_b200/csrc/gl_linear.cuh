// gl_linear.cuh -- "backward" amplitude modelling (light intensities solved "by linear inversion";
// SURVEY 8(f) NEXT-4; reading S21 in DESIGN.md section 16).
//
// The model image is linear in the light amplitudes a_k (I of each Sersic block, the shapelet coefficients).  With
// amplitude_mode = 1 a call first renders the n_amp unit-amplitude component images A_k: ONE pass of steps B-C
// (gl_ray_comp_kernel: one deflection per ray, every component stored separately) and the step-D kernel once per
// component (obs = 0, w = 1: its g_pix output is -A_k), then one CTA per particle
// forms the normal equations  M_kl = sum A_k A_l / sigma^2,  b_k = sum A_k obs / sigma^2  in fp64, factors M = L L^T,
// writes a* = M^-1 b into PB and, step D being linear, g_pix and chi^2 at a* from the same component images; the
// transpose of step D and the ordinary adjoint then run at a*.  Since dL/da = 0 there, the gradient
// with respect to the other parameters is the ordinary adjoint's (envelope theorem); gl_finalize_kernel zeroes the
// amplitude entries.  Product path only; shares nothing with oracle/.
#pragma once
#include "gl_common.cuh"
#include "gl_conv.cuh"

namespace gl {

constexpr int AMP_MAX = 72;          // 2 + 66 + 3 = 71 amplitudes at most (two sources, n_max = 10, three lens Sersic blocks)

struct AmpMap {                      // component k -> its slot in PB
    int n;
    short off[AMP_MAX];              // PB offset of the amplitude
    unsigned char shp[AMP_MAX];      // 1: shapelet coefficient (PB holds a_k c_n1 c_n2 / beta_s: scale by PB[PB_SHP] = 1/beta_s and scl)
    float scl[AMP_MAX];              // c_n1 c_n2 of the scaled shapelet basis (gl_ray.cuh), 1 for the other amplitudes
};

// PB amplitudes := unit vector e_k (k < 0: every amplitude 1).  One thread per (particle, component).
template <class T>
__global__ void gl_amp_select_kernel(const __grid_constant__ AmpMap am, int k, int64_t Pc, T* __restrict__ pb) {
    const int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= Pc * am.n) return;
    const int64_t p = e / am.n; const int j = (int)(e - p * am.n);
    T* o = pb + p * PB_STRIDE;
    o[am.off[j]] = (j == k || k < 0) ? (am.shp[j] ? (T)((double)o[PB_SHP] * (double)am.scl[j]) : T(1)) : T(0);
}

// obs = 0 and w = 1 for the component passes: step E then leaves -A_k in its g_pix output.
template <class T>
__global__ void gl_amp_fill_kernel(size_t n, float* __restrict__ zero_obs, T* __restrict__ unit_w) {
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) { zero_obs[i] = 0.f; unit_w[i] = T(1); }
}

// system_id of the na * Pc virtual particles of the component passes (component-major).
__global__ void gl_amp_sid_kernel(const int32_t* __restrict__ sid, int64_t Pc, int na, int32_t* __restrict__ out) {
    const int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (e < Pc * na) out[e] = sid[e % Pc];
}

// Normal equations + Cholesky solve.  grid = Pc, 256 threads.
// comp: [n_amp][Pc][gpix_stride] = -A_k in the padded g_pix layout.  sys_w: 1/sigma^2.  out_amp may be NULL.
// A particle whose normal matrix is not positive definite (a component that leaves no light on the cutout) is
// marked invalid (PB_VALID = 0: logp = -INF, zero gradient).
// Pixels per shared-memory tile and its layout.  Few pairs (n_pair <= 128, the split mode below): as many pixels as fit
// the largest problem's footprint (multiple of 64, up to 1024), which amortises the two barriers per tile, row pitch
// TP + 1.  Many pairs (the tensor-core mode): 64 pixels, rows padded to a multiple of 8, row pitch TP + 4 (an FP64
// mma fragment load -- 8 rows x 4 consecutive pixels per half-warp pair -- is then bank-conflict free).
static inline bool amp_solve_mma(int n) { return (n + 1) * (n + 2) / 2 > 128; }
static inline int amp_solve_tp(int n) {
    if (amp_solve_mma(n)) return 64;
    int tp = (4608 / (n + 1) - 1) / 64 * 64;
    return tp < 64 ? 64 : (tp > 1024 ? 1024 : tp);
}
static inline size_t amp_solve_smem(int n) {
    const int np = n + 1, tp = amp_solve_tp(n);
    size_t ct = amp_solve_mma(n) ? (size_t)((np + 7) / 8 * 8) * (tp + 4) : (size_t)np * (tp + 1);
    if (ct < (size_t)n * n) ct = (size_t)n * n;
    if (ct < 256) ct = 256;
    const size_t npair = (size_t)np * (np + 1) / 2;
    return sizeof(double) * (ct + (npair > 256 ? npair : 256) + n);
}

// D(8x8) += A(8x4) B(4x8) in fp64 on the tensor cores.  Lane l holds a = A[l/4][l%4], b = B[l%4][l/4],
// (c0, c1) = C[l/4][2 (l%4) + {0, 1}].
__device__ __forceinline__ void dmma_m8n8k4(double& c0, double& c1, double a, double b) {
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                 : "+d"(c0), "+d"(c1) : "d"(a), "d"(b));
}
constexpr int AMP_TPW = 6;           // 8x8 output tiles per warp: 9 * 10 / 2 = 45 tiles at most over 8 warps

template <class T>
__global__ void __launch_bounds__(256) gl_amp_solve_kernel(const __grid_constant__ Geom G, const __grid_constant__ AmpMap am,
                                                           const T* __restrict__ comp, int64_t Pc,
                                                           const float* __restrict__ obs, const T* __restrict__ sys_w,
                                                           const int32_t* __restrict__ system_id, int64_t p_base,
                                                           T* __restrict__ pb, float* __restrict__ out_amp,
                                                           T* __restrict__ gpix, T* __restrict__ chi, int n_ctile, int TP) {
    extern __shared__ double amp_sm[];
    const int n = am.n, np = n + 1, NN = G.N * G.N, tid = threadIdx.x;
    const int64_t p = blockIdx.x;
    const int sys = system_id ? system_id[p_base + p] : 0;
    const int npair = np * (np + 1) / 2;
    const bool mma = npair > 128;                        // the normal matrix is a dense contraction over the pixels
    const int NR = mma ? (np + 7) / 8 * 8 : np, PT = mma ? TP + 4 : TP + 1;
    double* ct = amp_sm;                                 // [NR][PT] tile of A_k / sigma (row n: obs / sigma, then zero rows); later M [n][n]
    int ct_sz = NR * PT > n * n ? NR * PT : n * n;
    if (ct_sz < 256) ct_sz = 256;
    double* pr = amp_sm + ct_sz;                         // [npair] sums, pair (k, l), l <= k, at k(k+1)/2 + l
    double* rhs = pr + (npair > 256 ? npair : 256);     // [n]  (pr doubles as the 256-entry reduction buffer at the end)
    __shared__ int s_fail;
    if (tid == 0) s_fail = 0;
    // Split mode: S = 256 / npair threads share one pair, each taking every S-th pixel of a tile; their partial sums are
    // added in a fixed order at the end.  Tensor-core mode: M = A A^T in 8x8 tiles of the lower triangle, warp w owns
    // tiles w, w + 8, ...; one mma.m8n8k4 per tile and 4 pixels.
    const int S = mma ? 1 : 256 / npair;
    const int my = tid / S, g = tid - my * S;             // split mode: pair index, pixel lane
    const int lane = tid & 31, wrp = tid >> 5;
    auto tri = [](int i, int& k, int& l) {
        k = (int)((sqrt(8.0 * i + 1.0) - 1.0) * 0.5);
        while (k * (k + 1) / 2 > i) --k;
        while ((k + 1) * (k + 2) / 2 <= i) ++k;
        l = i - k * (k + 1) / 2;
    };
    int pk = 0, pl = 0;                                   // split mode: this thread's pair
    if (!mma && my < npair) tri(my, pk, pl);
    const int ntile = (NR >> 3) * ((NR >> 3) + 1) / 2;
    int ti[AMP_TPW], tj[AMP_TPW]; double c0[AMP_TPW], c1[AMP_TPW];
#pragma unroll
    for (int j = 0; j < AMP_TPW; ++j) {
        ti[j] = tj[j] = 0; c0[j] = c1[j] = 0;
        if (mma && wrp + 8 * j < ntile) tri(wrp + 8 * j, ti[j], tj[j]);
    }
    double acc = 0;
    const size_t gs = gpix_stride(G);
    for (int t0 = 0; t0 < NN; t0 += TP) {
        __syncthreads();
        for (int idx = tid; idx < NR * TP; idx += 256) {
            const int k = idx / TP, x = idx - k * TP, pix = t0 + x;
            double v = 0;
            if (pix < NN && k < np) {
                const int r = pix / G.N, q = pix - r * G.N;
                const double isg = sqrt((double)sys_w[(size_t)sys * NN + pix]);
                v = k < n ? -(double)comp[((size_t)k * Pc + p) * gs + (size_t)(r + G.PADg) * G.Wg + q + G.PADg]
                          : (double)obs[(size_t)sys * NN + pix];
                v *= isg;
            }
            ct[k * PT + x] = v;
        }
        __syncthreads();
        if (!mma) {
            if (my < npair) {
                const double* a = ct + pk * PT; const double* b = ct + pl * PT;
                for (int x = g; x < TP; x += S) acc = fma(a[x], b[x], acc);
            }
        } else {
#pragma unroll
            for (int j = 0; j < AMP_TPW; ++j) {
                if (wrp + 8 * j < ntile) {               // warp-uniform
                    const double* a = ct + (8 * ti[j] + (lane >> 2)) * PT + (lane & 3);
                    const double* b = ct + (8 * tj[j] + (lane >> 2)) * PT + (lane & 3);
#pragma unroll 4
                    for (int x0 = 0; x0 < TP; x0 += 4) dmma_m8n8k4(c0[j], c1[j], a[x0], b[x0]);
                }
            }
        }
    }
    __syncthreads();
    if (!mma) {
        ct[tid] = acc;                                    // [pair][S] partials (npair * S <= 256 <= ct_sz)
        __syncthreads();
        if (tid < npair) { double s = 0; for (int x = 0; x < S; ++x) s += ct[tid * S + x]; pr[tid] = s; }
    } else {
#pragma unroll
        for (int j = 0; j < AMP_TPW; ++j) {
            if (wrp + 8 * j < ntile) {
                const int row = 8 * ti[j] + (lane >> 2), col = 8 * tj[j] + 2 * (lane & 3);
                if (row < np && col <= row) pr[row * (row + 1) / 2 + col] = c0[j];
                if (row < np && col + 1 <= row) pr[row * (row + 1) / 2 + col + 1] = c1[j];
            }
        }
    }
    __syncthreads();
    // full symmetric M and rhs
    double* M = ct;
    for (int idx = tid; idx < n * n; idx += 256) {
        const int k = idx / n, l = idx - k * n; const int a = k > l ? k : l, b = k > l ? l : k;
        M[idx] = pr[a * (a + 1) / 2 + b];
    }
    for (int k = tid; k < n; k += 256) rhs[k] = pr[n * (n + 1) / 2 + k];
    __syncthreads();
    // Cholesky, column by column (lower triangle in place)
    for (int j = 0; j < n; ++j) {
        if (tid == 0) {
            const double d = M[j * n + j], d0 = pr[j * (j + 1) / 2 + j];
            if (!(d > 1e-13 * d0) || !isfinite(d)) { s_fail = 1; M[j * n + j] = 1.0; } else M[j * n + j] = sqrt(d);
        }
        __syncthreads();
        const double dj = M[j * n + j];
        for (int i = j + 1 + tid; i < n; i += 256) M[i * n + j] /= dj;
        __syncthreads();
        const int m = n - j - 1;                          // trailing update of the lower triangle
        for (int idx = tid; idx < m * m; idx += 256) {
            const int i = j + 1 + idx / m, k = j + 1 + idx % m;
            if (k <= i) M[i * n + k] -= M[i * n + j] * M[k * n + j];
        }
        __syncthreads();
    }
    if (tid == 0) {
        for (int i = 0; i < n; ++i) { double s = rhs[i]; for (int k = 0; k < i; ++k) s -= M[i * n + k] * rhs[k]; rhs[i] = s / M[i * n + i]; }
        for (int i = n - 1; i >= 0; --i) { double s = rhs[i]; for (int k = i + 1; k < n; ++k) s -= M[k * n + i] * rhs[k]; rhs[i] = s / M[i * n + i]; }
        for (int i = 0; i < n; ++i) if (!isfinite(rhs[i])) s_fail = 1;
    }
    __syncthreads();
    T* o = pb + p * PB_STRIDE;
    const bool fail = s_fail != 0;
    for (int k = tid; k < n; k += 256) {
        const double a = fail ? 0.0 : rhs[k];
        o[am.off[k]] = am.shp[k] ? (T)(a * (double)o[PB_SHP] * (double)am.scl[k]) : (T)a;
        if (out_amp) out_amp[(p_base + p) * n + k] = (float)a;
    }
    if (tid == 0 && fail) o[PB_VALID] = T(0);
    // Step E at a*: the model image is sum_k a*_k A_k (step D is linear), so g_pix and chi^2 follow from the component
    // images already in memory and the forward passes B-D need not run again.
    T* gp = gpix + (size_t)p * gs;
    zero_gpix_border(G, gp, tid, 256);
    double c2 = 0;
    for (int pix = tid; pix < NN; pix += 256) {
        const int r = pix / G.N, q = pix - r * G.N;
        const size_t at = (size_t)(r + G.PADg) * G.Wg + q + G.PADg;
        double m = 0;
        for (int k = 0; k < n; ++k) m = fma(-rhs[k], (double)comp[((size_t)k * Pc + p) * gs + at], m);
        const double w = (double)sys_w[(size_t)sys * NN + pix], res = m - (double)obs[(size_t)sys * NN + pix];
        gp[at] = fail ? T(0) : (T)(-res * w);
        c2 = fma(res * res, w, c2);
    }
    __syncthreads();                                      // pr is free again: block sum in fixed order
    pr[tid] = c2;
    __syncthreads();
    for (int o2 = 128; o2 > 0; o2 >>= 1) { if (tid < o2) pr[tid] += pr[tid + o2]; __syncthreads(); }
    for (int k = tid; k < n_ctile; k += 256) chi[(size_t)p * n_ctile + k] = k == 0 && !fail ? (T)pr[0] : T(0);
}


}  // namespace gl
