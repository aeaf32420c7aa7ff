// gl_conv.cuh -- step D (PSF convolution + binning), step E (chi-square) and the transpose of step D.
//
// Fused form (checked in tests/test_oracle_pins.py::test_conv_bin_vs_scipy_and_fused_keff_form):
//   model[p][q] = sum_{u,v < KE} kt[u][v] * I_ray[s p - c + u][s q - c + v],   KE = K + s - 1,
//   kt[u][v] = Delta^2/s^2 * k_eff[KE-1-u][KE-1-v],  k_eff = psf (*) ones(s,s)   (rays outside the cutout are 0)
// kt is stored PHASE-MAJOR: kt[a'][b'][u1][v1] with u = s*u1 + a', v = s*v1 + b', u1,v1 < U = ceil(KE/s) (zero padded).
//
// The ray image lives in HBM as s*s zero-bordered, shifted PHASE PLANES (gl_common.cuh): ray (s i1 + a, s j1 + b) is
// element [i1 + o_a][j1 + o_b] of plane (a, b), o_a = (a + c) div s.  With a' = (a + c) mod s the stride-s correlation
// becomes, per plane, a plain stride-1 "valid" correlation with U x U taps and no bounds checks:
//   model[p][q] = sum_{a,b} sum_{u1,v1 < U} kt[a'][b'][u1][v1] * plane_ab[p + u1][q + v1]                (step D)
//   gbar_ab[n + o_a][j'] = sum_{k,l < U} kt[a'][b'][U-1-k][U-1-l] * gp[n + o_a + k][j' + l]           (transpose)
// where gp is g_pix zero-padded by U-1 on every side and gbar is produced directly in the plane layout.
//
// Both directions run the same inner loop (gl_conv_*_sw): one thread owns 4 adjacent output columns of ONE plane and
// UR consecutive tap rows, keeps its UR x U taps and a UR-row sliding window of the input in registers, and sweeps
// down the image: per output row it loads one new input row segment (U+3 floats, 16-byte aligned) and issues
// 4*UR*U FMAs.  Step D then sums the s*s*ceil(U/UR) partial results per pixel through shared memory in a fixed
// order (deterministic), and applies step E in the same pass.
#pragma once
#include "gl_common.cuh"
#include "gl_math.cuh"

namespace gl {

// Per-system preparation, once per call.  grid = n_systems, block = 256.
//   sys_kt  [n_sys][s*s*U*U]   sys_w [n_sys][N*N] = 1/sigma^2   sys_sumlog [n_sys] = sum ln sigma
template <class T>
__global__ void gl_prep_kernel(const __grid_constant__ Geom G, const float* __restrict__ psf, const float* __restrict__ sigma,
                               T* __restrict__ sys_kt, T* __restrict__ sys_w, double* __restrict__ sys_sumlog,
                               double* __restrict__ math_tab_out) {
    const int sys = blockIdx.x;
    if (sys == 0 && math_tab_out != nullptr) fill_math_tab(math_tab_out);
    const int KE = G.K + G.s - 1, U = G.U, s = G.s;
    const float* ps = psf + (size_t)sys * G.K * G.K;
    T* kt = sys_kt + (size_t)sys * s * s * U * U;
    for (int t = threadIdx.x; t < s * s * U * U; t += blockDim.x) {
        int v1 = t % U, u1 = (t / U) % U, b = (t / (U * U)) % s, a = t / (U * U * s);
        int u = s * u1 + a, v = s * v1 + b;
        double acc = 0.0;
        if (u < KE && v < KE) {
            int m = KE - 1 - u, n = KE - 1 - v;           // k_eff[m][n] = sum_{di,dj<s} psf[m-di][n-dj]
            for (int di = 0; di < s; ++di) for (int dj = 0; dj < s; ++dj) {
                int r = m - di, cc = n - dj;
                if (r >= 0 && r < G.K && cc >= 0 && cc < G.K) acc += (double)ps[r * G.K + cc];
            }
        }
        kt[t] = (T)(acc * G.delta2 / (double)(s * s));
    }
    __shared__ double red[256];
    double sl = 0.0;
    const float* sg = sigma + (size_t)sys * G.N * G.N;
    T* w = sys_w + (size_t)sys * G.N * G.N;
    for (int t = threadIdx.x; sigma != nullptr && t < G.N * G.N; t += blockDim.x) {
        double sv = (double)sg[t];
        w[t] = (T)(1.0 / (sv * sv));
        sl += log(sv);
    }
    red[threadIdx.x] = sl; __syncthreads();
    for (int o = 128; o > 0; o >>= 1) { if (threadIdx.x < o) red[threadIdx.x] += red[threadIdx.x + o]; __syncthreads(); }
    if (threadIdx.x == 0) sys_sumlog[sys] = red[0];
}

// fixed-order block sum of one value per thread (blockDim.x a multiple of 32, <= 1024), result valid in thread 0
template <class T>
__device__ __forceinline__ T block_sum(T v, T* red /* 32 */) {
    v = warp_sum(v);
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = v;
    __syncthreads();
    T s = T(0);
    if (threadIdx.x == 0) {
        const int nw = blockDim.x >> 5;
        for (int w = 0; w < nw; ++w) s += red[w];
    }
    return s;
}

// Zero the border of this particle's padded g_pix image (the interior is written by the step-E epilogue).
template <class T>
__device__ __forceinline__ void zero_gpix_border(const Geom& G, T* __restrict__ gp, int first, int stride) {
    const int tot = G.Hg * G.Wg;
    for (int e = first; e < tot; e += stride) {
        const int r = e / G.Wg, cc = e - r * G.Wg;
        if (r < G.PADg || r >= G.PADg + G.N || cc < G.PADg || cc >= G.PADg + G.N) gp[e] = T(0);
    }
}

// Step E for one pixel: writes the model / g_pix and returns the chi^2 term.  obs is fp32 (C ABI), w = 1/sigma^2 in T.
template <class T>
__device__ __forceinline__ T pixel_epilogue(const Geom& G, T m, int pr, int pq, int sys, size_t p_out, int p,
                                            const float* __restrict__ obs, const T* __restrict__ sys_w,
                                            T* __restrict__ gpix, float* __restrict__ out_model) {
    const size_t NN = (size_t)G.N * G.N, pix = (size_t)pr * G.N + pq;
    if (out_model) out_model[p_out * NN + pix] = (float)m;
    if (!gpix) return T(0);
    const T r = m - (T)obs[(size_t)sys * NN + pix], w = sys_w[(size_t)sys * NN + pix];
    gpix[(size_t)p * gpix_stride(G) + (size_t)(pr + G.PADg) * G.Wg + pq + G.PADg] = -r * w;
    return r * r * w;
}

// ----------------------------------------------------------------------------- generic kernels (any s, K)
// One thread per detector pixel, taps and rays through L1/L2.  grid = (ceil(N*N/256), Pc).  chi: [Pc][gridDim.x].
template <class T>
__global__ void __launch_bounds__(256) gl_conv_fwd_generic(const __grid_constant__ Geom G, const T* __restrict__ ray,
                                                           const T* __restrict__ sys_kt, const T* __restrict__ sys_w,
                                                           const float* __restrict__ obs, const int32_t* __restrict__ system_id,
                                                           int64_t p_base, T* __restrict__ gpix, T* __restrict__ chi,
                                                           float* __restrict__ out_model) {
    __shared__ T red[32];
    const int p = blockIdx.y, NN = G.N * G.N, s = G.s, U = G.U;
    const int sys = system_id ? system_id[p_base + p] : 0;
    const T* kt = sys_kt + (size_t)sys * s * s * U * U;
    const T* I = ray + (size_t)p * ray_stride(G);
    if (gpix) zero_gpix_border(G, gpix + (size_t)p * gpix_stride(G), blockIdx.x * 256 + threadIdx.x, gridDim.x * 256);
    const int pix = blockIdx.x * 256 + threadIdx.x;
    T c2 = T(0);
    if (pix < NN) {
        const int pr = pix / G.N, pq = pix - pr * G.N;
        T acc = T(0);
        for (int a = 0; a < s; ++a) for (int b = 0; b < s; ++b) {
            const T* kr = kt + (size_t)(((a + G.c) % s) * s + (b + G.c) % s) * U * U;
            const T* pl = I + ((size_t)(a * s + b) * G.Hp + pr) * G.Wp + pq;
            for (int u1 = 0; u1 < U; ++u1)
                for (int v1 = 0; v1 < U; ++v1) acc = Real<T>::fma(kr[u1 * U + v1], pl[(size_t)u1 * G.Wp + v1], acc);
        }
        c2 = pixel_epilogue<T>(G, acc, pr, pq, sys, (size_t)(p_base + p), p, obs, sys_w, gpix, out_model);
    }
    if (chi) {
        T tot = block_sum(c2, red);
        if (threadIdx.x == 0) chi[(size_t)p * gridDim.x + blockIdx.x] = tot;
    }
}

// Generic transpose of step D: one thread per ray.  grid = (ceil(s*s*N*N/256), Pc).  gbar is written in plane layout.
template <class T>
__global__ void __launch_bounds__(256) gl_conv_bwd_generic(const __grid_constant__ Geom G, const T* __restrict__ gpix,
                                                           const T* __restrict__ sys_kt, const int32_t* __restrict__ system_id,
                                                           int64_t p_base, T* __restrict__ gbar) {
    const int p = blockIdx.y, s = G.s, U = G.U, N = G.N;
    const int idx = blockIdx.x * 256 + threadIdx.x;
    if (idx >= s * s * N * N) return;
    const int sys = system_id ? system_id[p_base + p] : 0;
    const int ph = idx / (N * N), rem = idx - ph * N * N, n = rem / N, j1 = rem - n * N;
    const int a = ph / s, b = ph - a * s, oa = phase_shift(G, a), ob = phase_shift(G, b);
    const T* kr = sys_kt + (size_t)sys * s * s * U * U + (size_t)(((a + G.c) % s) * s + (b + G.c) % s) * U * U;
    const T* g = gpix + (size_t)p * gpix_stride(G) + (size_t)(n + oa) * G.Wg + j1 + ob;
    T acc = T(0);
    for (int k = 0; k < U; ++k)
        for (int l = 0; l < U; ++l) acc = Real<T>::fma(kr[(U - 1 - k) * U + (U - 1 - l)], g[(size_t)k * G.Wg + l], acc);
    gbar[(size_t)p * ray_stride(G) + ((size_t)ph * G.Hp + n + oa) * G.Wp + j1 + ob] = acc;
}

// ----------------------------------------------------------------------------- sliding-window kernels
// 4 consecutive T, 4-element aligned: one 16-byte load for float, two for double.
__device__ __forceinline__ void load4(const float* __restrict__ p, float* w) {
    const float4 x = __ldg(reinterpret_cast<const float4*>(p));
    w[0] = x.x; w[1] = x.y; w[2] = x.z; w[3] = x.w;
}
__device__ __forceinline__ void load4(const double* __restrict__ p, double* w) {
    const double2 x = __ldg(reinterpret_cast<const double2*>(p)), y = __ldg(reinterpret_cast<const double2*>(p) + 1);
    w[0] = x.x; w[1] = x.y; w[2] = y.x; w[3] = y.y;
}
__device__ __forceinline__ void store4(float* p, const float* a) { *reinterpret_cast<float4*>(p) = make_float4(a[0], a[1], a[2], a[3]); }
__device__ __forceinline__ void store4(double* p, const double* a) {
    reinterpret_cast<double2*>(p)[0] = make_double2(a[0], a[1]); reinterpret_cast<double2*>(p)[1] = make_double2(a[2], a[3]);
}

template <class T, int U>
struct RowSeg {                                  // the U+3 input values that 4 adjacent outputs need from one row
    static constexpr int NEED = U + 3;
    static constexpr int NV4 = (NEED % 4 <= 1) ? NEED / 4 : (NEED + 3) / 4;
    static constexpr int NSC = (NEED % 4 <= 1) ? NEED % 4 : 0;
    static constexpr int NVAL = NV4 * 4 + NSC;
    static constexpr int WL = 4 * ((NEED + 3) / 4);                 // values a row segment may touch
    static __device__ __forceinline__ void load(T (&w)[NVAL], const T* __restrict__ p) {
#pragma unroll
        for (int v = 0; v < NV4; ++v) load4(p + 4 * v, &w[4 * v]);
#pragma unroll
        for (int i = 0; i < NSC; ++i) w[4 * NV4 + i] = __ldg(p + 4 * NV4 + i);
    }
};

template <class T, int U, int NVAL>
__device__ __forceinline__ void fma_row(T (&acc)[4], const T (&Tp)[U], const T (&w)[NVAL]) {
#pragma unroll
    for (int l = 0; l < U; ++l) {
#pragma unroll
        for (int q = 0; q < 4; ++q) acc[q] = Real<T>::fma(Tp[l], w[q + l], acc[q]);
    }
}

constexpr int CONV_R = 4;                        // output rows between two reductions

// Step D + E.  grid = (n_band, Pc); block = roundup32(ncgb * s*s * ceil(U/UR)); dynamic smem = conv_sw_smem(...).
// Thread t: column group g = t % ncgb (4 pixels), virtual phase vp = t / ncgb = (plane, tap-row group).
template <class T, int UR, int U, int NT_MAX>
__global__ void __launch_bounds__(NT_MAX) gl_conv_fwd_sw(const __grid_constant__ Geom G, int ncgb,
                                                         const T* __restrict__ ray, const T* __restrict__ sys_kt,
                                                         const T* __restrict__ sys_w, const float* __restrict__ obs,
                                                         const int32_t* __restrict__ system_id, int64_t p_base,
                                                         T* __restrict__ gpix, T* __restrict__ chi,
                                                         float* __restrict__ out_model) {
    constexpr int NRG = (U + UR - 1) / UR;
    constexpr int NVAL = RowSeg<T, U>::NVAL;
    extern __shared__ __align__(16) unsigned char conv_smem[];     // part [2][NVP][CONV_R][NQ]
    T* part = reinterpret_cast<T*>(conv_smem);
    __shared__ T red[32];
    const int s = G.s, N = G.N, NVP = s * s * NRG, NQ = 4 * ncgb;
    const int p = blockIdx.y, band = blockIdx.x, t = threadIdx.x;
    const bool active = t < ncgb * NVP;
    const int g = active ? t % ncgb : 0, vp = active ? t / ncgb : 0;
    const int rho = vp % NRG, ph = vp / NRG, a = ph / s, b = ph - a * s;
    const int sys = system_id ? system_id[p_base + p] : 0;
    if (gpix) zero_gpix_border(G, gpix + (size_t)p * gpix_stride(G), band * blockDim.x + t, gridDim.x * blockDim.x);
    T Tp[UR][U];
    {
        const T* kph = sys_kt + (size_t)sys * s * s * U * U + (size_t)(((a + G.c) % s) * s + (b + G.c) % s) * U * U;
#pragma unroll
        for (int k = 0; k < UR; ++k) {
            const int u1 = rho * UR + k;
#pragma unroll
            for (int l = 0; l < U; ++l) Tp[k][l] = (u1 < U) ? __ldg(kph + u1 * U + l) : T(0);
        }
    }
    const int gg = min(band * ncgb + g, (G.Wp - RowSeg<T, U>::WL) / 4);      // clamp keeps idle lanes in bounds
    const T* in = ray + (size_t)p * ray_stride(G) + ((size_t)ph * G.Hp + rho * UR) * G.Wp + 4 * gg;
    const size_t Wp = (size_t)G.Wp;
    T w[UR][NVAL];
#pragma unroll
    for (int k = 0; k < UR; ++k) RowSeg<T, U>::load(w[k], in + k * Wp);
    T c2 = T(0);
    int buf = 0;
    for (int pr0 = 0; pr0 < N; pr0 += UR) {
#pragma unroll
        for (int j = 0; j < UR; ++j) {
            const int pr = pr0 + j;
            if (pr < N) {
                T acc[4] = {T(0), T(0), T(0), T(0)};
                fma_row<T, U, NVAL>(acc, Tp[0], w[j % UR]);
                if (pr + 1 < N) RowSeg<T, U>::load(w[j % UR], in + (size_t)(pr + UR) * Wp);   // row for the next step
#pragma unroll
                for (int k = 1; k < UR; ++k) fma_row<T, U, NVAL>(acc, Tp[k], w[(j + k) % UR]);
                if (active) store4(&part[((size_t)(buf * NVP + vp) * CONV_R + (pr & (CONV_R - 1))) * NQ + 4 * g], acc);
                if ((pr & (CONV_R - 1)) == CONV_R - 1 || pr == N - 1) {
                    __syncthreads();
                    const int rows = (pr & (CONV_R - 1)) + 1, r0 = pr - rows + 1;
                    for (int o = t; o < rows * NQ; o += blockDim.x) {
                        const int r = o / NQ, q = o - r * NQ, pq = band * NQ + q;
                        T m = T(0);
                        for (int v = 0; v < NVP; ++v) m += part[((size_t)(buf * NVP + v) * CONV_R + r) * NQ + q];
                        if (pq < N) c2 += pixel_epilogue<T>(G, m, r0 + r, pq, sys, (size_t)(p_base + p), p, obs, sys_w, gpix, out_model);
                    }
                    buf ^= 1;
                }
            }
        }
    }
    if (chi) {
        const T tot = block_sum(c2, red);
        if (t == 0) chi[(size_t)p * gridDim.x + band] = tot;
    }
}

// Transpose of step D.  grid = (n_band, Pc); block = roundup32(ncgb * s*s * ceil(U/UR)).  gbar (plane layout)
// overwrites the ray buffer; only the N x N interior of each plane is meaningful afterwards.
template <class T, int UR, int U, int NT_MAX>
__global__ void __launch_bounds__(NT_MAX) gl_conv_bwd_sw(const __grid_constant__ Geom G, int ncgb,
                                                         const T* __restrict__ gpix, const T* __restrict__ sys_kt,
                                                         const int32_t* __restrict__ system_id, int64_t p_base,
                                                         T* __restrict__ gbar) {
    constexpr int NRG = (U + UR - 1) / UR;
    constexpr int NVAL = RowSeg<T, U>::NVAL;
    extern __shared__ __align__(16) unsigned char conv_smem[];     // part [2][NVP][CONV_R][NQ] (only if NRG > 1)
    T* part = reinterpret_cast<T*>(conv_smem);
    const int s = G.s, N = G.N, NPH = s * s, NVP = NPH * NRG, NQ = 4 * ncgb;
    const int p = blockIdx.y, band = blockIdx.x, t = threadIdx.x;
    const bool active = t < ncgb * NVP;
    const int g = active ? t % ncgb : 0, vp = active ? t / ncgb : 0;
    const int rho = vp % NRG, ph = vp / NRG, a = ph / s, b = ph - a * s, oa = phase_shift(G, a);
    const int sys = system_id ? system_id[p_base + p] : 0;
    T Tp[UR][U];
    {
        const T* kph = sys_kt + (size_t)sys * s * s * U * U + (size_t)(((a + G.c) % s) * s + (b + G.c) % s) * U * U;
#pragma unroll
        for (int k = 0; k < UR; ++k) {
            const int u1 = rho * UR + k;
#pragma unroll
            for (int l = 0; l < U; ++l) Tp[k][l] = (u1 < U) ? __ldg(kph + (U - 1 - u1) * U + (U - 1 - l)) : T(0);
        }
    }
    const int gcol = band * ncgb + g;
    const bool in_range = active && 4 * gcol + 3 < G.Wp && 4 * gcol + RowSeg<T, U>::WL <= G.Wg;
    const int gg = min(gcol, (G.Wg - RowSeg<T, U>::WL) / 4);
    const size_t Wg = (size_t)G.Wg, Wp = (size_t)G.Wp;
    const T* in = gpix + (size_t)p * gpix_stride(G) + (size_t)(oa + rho * UR) * Wg + 4 * gg;
    T* out = gbar + (size_t)p * ray_stride(G) + ((size_t)ph * G.Hp + oa) * Wp + 4 * gcol;
    T w[UR][NVAL];
#pragma unroll
    for (int k = 0; k < UR; ++k) RowSeg<T, U>::load(w[k], in + k * Wg);
    int buf = 0;
    for (int n0 = 0; n0 < N; n0 += UR) {
#pragma unroll
        for (int j = 0; j < UR; ++j) {
            const int n = n0 + j;
            if (n < N) {
                T acc[4] = {T(0), T(0), T(0), T(0)};
                fma_row<T, U, NVAL>(acc, Tp[0], w[j % UR]);
                if (n + 1 < N) RowSeg<T, U>::load(w[j % UR], in + (size_t)(n + UR) * Wg);
#pragma unroll
                for (int k = 1; k < UR; ++k) fma_row<T, U, NVAL>(acc, Tp[k], w[(j + k) % UR]);
                if constexpr (NRG == 1) {
                    if (in_range) store4(out + (size_t)n * Wp, acc);
                } else {
                    if (active) store4(&part[((size_t)(buf * NVP + vp) * CONV_R + (n & (CONV_R - 1))) * NQ + 4 * g], acc);
                    if ((n & (CONV_R - 1)) == CONV_R - 1 || n == N - 1) {
                        __syncthreads();
                        const int rows = (n & (CONV_R - 1)) + 1, r0 = n - rows + 1;
                        for (int o = t; o < rows * NPH * NQ; o += blockDim.x) {
                            const int q = o % NQ, r = (o / NQ) % rows, ph2 = o / (NQ * rows);
                            T m = T(0);
#pragma unroll
                            for (int v = 0; v < NRG; ++v) m += part[((size_t)(buf * NVP + ph2 * NRG + v) * CONV_R + r) * NQ + q];
                            const int col = band * NQ + q;
                            if (col < G.Wp)
                                gbar[(size_t)p * ray_stride(G) + ((size_t)ph2 * G.Hp + phase_shift(G, ph2 / s) + r0 + r) * Wp + col] = m;
                        }
                        buf ^= 1;
                    }
                }
            }
        }
    }
}

}  // namespace gl
