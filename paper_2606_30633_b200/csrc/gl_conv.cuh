// gl_conv.cuh -- step D (PSF convolution + binning), step E (chi-square) and the transpose of step D.
//
// Fused form (checked in tests/test_oracle_pins.py::test_conv_bin_vs_scipy_and_fused_keff_form):
//   model[p][q] = sum_{u,v < KE} kt[u][v] * I_ray[s p - c + u][s q - c + v],   KE = K + s - 1,
//   kt[u][v] = Delta^2/s^2 * k_eff[KE-1-u][KE-1-v],  k_eff = psf (*) ones(s,s)   (rays outside the cutout are 0)
// kt is stored PHASE-MAJOR: kt[a][b][u1][v1] with u = s*u1 + a, v = s*v1 + b, u1,v1 < U = ceil(KE/s) (zero padded),
// which turns the stride-s correlation into s^2 stride-1 correlations of the ray image's phase planes.
// The transpose is  gbar[i][j] = sum_{u1,v1} kt[a][b][u1][v1] * g[pp - u1][qq - v1],  pp = (i+c) div s, a = (i+c) mod s.
#pragma once
#include "gl_common.cuh"

namespace gl {

// Per-system preparation, once per call.  grid = n_systems, block = 256.
//   sys_kt  [n_sys][s*s*U*U]   sys_w [n_sys][N*N] = 1/sigma^2   sys_sumlog [n_sys] = sum ln sigma
__global__ void gl_prep_kernel(const __grid_constant__ Geom G, const float* __restrict__ psf, const float* __restrict__ sigma,
                               float* __restrict__ sys_kt, float* __restrict__ sys_w, float* __restrict__ sys_sumlog) {
    const int sys = blockIdx.x;
    const int KE = G.K + G.s - 1, U = G.U, s = G.s;
    const float* ps = psf + (size_t)sys * G.K * G.K;
    float* kt = sys_kt + (size_t)sys * s * s * U * U;
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
        kt[t] = (float)(acc * (double)G.delta2 / (double)(s * s));
    }
    __shared__ double red[256];
    double sl = 0.0;
    const float* sg = sigma + (size_t)sys * G.N * G.N;
    float* w = sys_w + (size_t)sys * G.N * G.N;
    for (int t = threadIdx.x; sigma != nullptr && t < G.N * G.N; t += blockDim.x) {
        double sv = (double)sg[t];
        w[t] = (float)(1.0 / (sv * sv));
        sl += log(sv);
    }
    red[threadIdx.x] = sl; __syncthreads();
    for (int o = 128; o > 0; o >>= 1) { if (threadIdx.x < o) red[threadIdx.x] += red[threadIdx.x + o]; __syncthreads(); }
    if (threadIdx.x == 0) sys_sumlog[sys] = (float)red[0];
}

// fixed-order block sum of one float per thread (NT threads), result valid in thread 0
template <int NT>
__device__ __forceinline__ float block_sum(float v, float* red /* NT/32 */) {
    v = warp_sum(v);
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = v;
    __syncthreads();
    float s = 0.f;
    if (threadIdx.x == 0) {
#pragma unroll
        for (int w = 0; w < NT / 32; ++w) s += red[w];
    }
    return s;
}

// Generic (any s, K) step D + E: one thread per detector pixel, taps and rays through L1/L2.  Used for shapes
// without a tiled specialisation.  grid = (ceil(N*N/256), Pc).  chi: [Pc][gridDim.x].
// out_model may be NULL; gpix may be NULL (gl_model_image).
__global__ void __launch_bounds__(256) gl_conv_fwd_generic(const __grid_constant__ Geom G, const float* __restrict__ ray,
                                                           const float* __restrict__ sys_kt, const float* __restrict__ sys_w,
                                                           const float* __restrict__ obs, const int32_t* __restrict__ system_id,
                                                           int64_t p_base, float* __restrict__ gpix, float* __restrict__ chi,
                                                           float* __restrict__ out_model) {
    __shared__ float red[8];
    const int p = blockIdx.y, NN = G.N * G.N, M = G.M, s = G.s, U = G.U;
    const int sys = system_id ? system_id[p_base + p] : 0;
    const float* kt = sys_kt + (size_t)sys * s * s * U * U;
    const float* I = ray + (size_t)p * M * M;
    const int pix = blockIdx.x * 256 + threadIdx.x;
    float c2 = 0.f;
    if (pix < NN) {
        const int pr = pix / G.N, pq = pix - pr * G.N;
        float acc = 0.f;
        for (int a = 0; a < s; ++a) for (int u1 = 0; u1 < U; ++u1) {
            const int i = s * pr - G.c + s * u1 + a;
            if (i < 0 || i >= M) continue;
            for (int b = 0; b < s; ++b) {
                const float* kr = kt + ((a * s + b) * U + u1) * U;
                for (int v1 = 0; v1 < U; ++v1) {
                    const int j = s * pq - G.c + s * v1 + b;
                    if (j >= 0 && j < M) acc = fmaf(kr[v1], I[i * M + j], acc);
                }
            }
        }
        if (out_model) out_model[(size_t)(p_base + p) * NN + pix] = acc;
        if (gpix) {
            const float r = acc - obs[(size_t)sys * NN + pix], w = sys_w[(size_t)sys * NN + pix];
            gpix[(size_t)p * NN + pix] = -r * w;
            c2 = r * r * w;
        }
    }
    if (chi) {
        float tot = block_sum<256>(c2, red);
        if (threadIdx.x == 0) chi[(size_t)p * gridDim.x + blockIdx.x] = tot;
    }
}

// Generic transpose of step D: one thread per ray.  grid = (ceil(M*M/256), Pc).  gbar overwrites the ray buffer.
__global__ void __launch_bounds__(256) gl_conv_bwd_generic(const __grid_constant__ Geom G, const float* __restrict__ gpix,
                                                           const float* __restrict__ sys_kt, const int32_t* __restrict__ system_id,
                                                           int64_t p_base, float* __restrict__ gbar) {
    const int p = blockIdx.y, M = G.M, s = G.s, U = G.U, N = G.N;
    const int idx = blockIdx.x * 256 + threadIdx.x;
    if (idx >= M * M) return;
    const int sys = system_id ? system_id[p_base + p] : 0;
    const float* kt = sys_kt + (size_t)sys * s * s * U * U;
    const float* g = gpix + (size_t)p * N * N;
    const int i = idx / M, j = idx - i * M;
    const int pp = (i + G.c) / s, a = (i + G.c) - pp * s, qq = (j + G.c) / s, b = (j + G.c) - qq * s;
    const float* kr = kt + (a * s + b) * U * U;
    float acc = 0.f;
    for (int u1 = 0; u1 < U; ++u1) {
        const int pr = pp - u1; if (pr < 0 || pr >= N) continue;
        for (int v1 = 0; v1 < U; ++v1) {
            const int pq = qq - v1;
            if (pq >= 0 && pq < N) acc = fmaf(kr[u1 * U + v1], g[pr * N + pq], acc);
        }
    }
    gbar[(size_t)p * M * M + idx] = acc;
}

}  // namespace gl
