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
// Both directions run the same inner loop (conv_slide): "input-stationary" sliding accumulators.  One thread owns CW
// adjacent output columns and a few phase planes; it walks down the input rows ONCE, and every input row segment
// (CW+U-1 values, loaded one step ahead) is scattered into the U output rows it contributes to, held as acc[U][CW]
// registers; the finished row leaves at the bottom and the accumulators shift by one.  Per step: U*U*CW FMAs on
// CW+U-1 loaded values, taps read from shared memory as 16-byte broadcasts.  Four adjacent lanes share a column
// group and split the s*s planes between them; step D sums their partial rows with two shuffles (fixed order) and
// applies step E in the same pass.  No tap or window registers -> ~100 registers in fp64, many resident warps.
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
    const int KE = G.KE, U = G.U, s = G.s;
    const float* ps = psf + (size_t)sys * G.K * G.K;
    T* kt = sys_kt + (size_t)sys * s * s * U * U;
    for (int t = threadIdx.x; t < s * s * U * U; t += blockDim.x) {
        int v1 = t % U, u1 = (t / U) % U, b = (t / (U * U)) % s, a = t / (U * U * s);
        int u = s * u1 + a, v = s * v1 + b;
        double acc = 0.0;
        if (u < KE && v < KE) {
            int m = KE - 1 - u, n = KE - 1 - v;           // psf_grid 0: k_eff[m][n] = sum_{di,dj<s} psf[m-di][n-dj]
            if (G.pgrid == 1) acc = (double)ps[(m / s) * G.K + n / s];     // psf_grid 1: box-expanded detector-grid taps
            else for (int di = 0; di < s; ++di) for (int dj = 0; dj < s; ++dj) {
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
        w[t] = G.noise_model == 1 ? (T)(sv * sv) : (T)(1.0 / (sv * sv));   // noise model 1: the background VARIANCE
        sl += G.noise_model == 1 ? 0.0 : log(sv);                        // (ln v is then part of the per-pixel term)
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
    T* gp = gpix + (size_t)p * gpix_stride(G) + (size_t)(pr + G.PADg) * G.Wg + pq + G.PADg;
    if (G.noise_model == 1) {                   // S12b: v = sigma^2 + max(m, 0) / t_exp; term = r^2 / v + ln v
        const bool pos = m > T(0);
        const double v = (double)w + (pos ? (double)m * G.inv_texp : 0.0), iv = 1.0 / v, vp = pos ? G.inv_texp : 0.0;
        const double rd = (double)r;
        *gp = (T)(-rd * iv + 0.5 * rd * rd * iv * iv * vp - 0.5 * vp * iv);
        return (T)(rd * rd * iv + log(v));
    }
    *gp = -r * w;
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

// ----------------------------------------------------------------------------- input-stationary sliding kernels
template <class T> struct Vec2;
template <> struct Vec2<float>  { using type = float2; };
template <> struct Vec2<double> { using type = double2; };

// Launch-invariant description of the sliding kernels (filled by conv_plan).
struct SlidePlan {
    int ncg;      // column groups per particle
    int tpp;      // threads per particle slot = ncg (one thread per column group, all phase planes)
    int ppc;      // particle slots per CTA
    int ps;       // tap stride between phases in shared memory (elements)
    int shared_taps;  // 1: one system -> one tap copy per CTA (uniform addresses); 0: one copy per slot
};

// acc[u][q] += sum_v tap[u][v] * seg[q + v] for one input row segment.  tap: shared memory, row pitch UP2 (even).
template <class T, int U, int CW, int SEG>
__device__ __forceinline__ void conv_slide(T (&acc)[U][CW], const T* __restrict__ tap, const T (&seg)[SEG]) {
    using V2 = typename Vec2<T>::type;
    constexpr int UP2 = (U + 1) & ~1;
#pragma unroll
    for (int u = 0; u < U; ++u) {
#pragma unroll
        for (int v = 0; v < UP2; v += 2) {
            const V2 k = *reinterpret_cast<const V2*>(tap + u * UP2 + v);
#pragma unroll
            for (int q = 0; q < CW; ++q) {
                acc[u][q] = Real<T>::fma(k.x, seg[q + v], acc[u][q]);
                if (v + 1 < U) acc[u][q] = Real<T>::fma(k.y, seg[q + v + 1], acc[u][q]);
            }
        }
    }
}

template <class T, int SEG>
__device__ __forceinline__ void load_seg(T (&seg)[SEG], const T* __restrict__ p) {
    using V2 = typename Vec2<T>::type;
#pragma unroll
    for (int v = 0; v < SEG; v += 2) {
        const V2 x = __ldg(reinterpret_cast<const V2*>(p + v));
        seg[v] = x.x; seg[v + 1] = x.y;
    }
}

// Step D + E.  grid = (ceil(Pc / ppc)); block = roundup32(ppc * tpp).  Dynamic smem: tap copies [n_copy][s*s][ps].
// Thread lt of a particle slot owns column group g = lt and walks through ALL s*s planes of every input row, so the
// tap address is uniform across a slot (a pure shared-memory broadcast: splitting the planes between lanes made the
// U = 16 kernels shared-memory bound) and an output row is complete inside one thread (no cross-lane reduction).
// PF: prefetch the next row segment into a second register buffer (off for U = 16 in fp64, where the registers buy more
// as a second resident CTA); MINB: minimum CTAs per SM handed to the register allocator.
#ifndef GL_CONV16_PF
#define GL_CONV16_PF 1
#endif
#ifndef GL_CONV16_MINB
#define GL_CONV16_MINB 1
#endif
template <class T, int U> __host__ __device__ constexpr bool conv_pf() { return !(U == 16 && sizeof(T) == 8) || GL_CONV16_PF; }
template <class T, int U> __host__ __device__ constexpr int conv_minb() { return (U == 16 && sizeof(T) == 8) ? GL_CONV16_MINB : 1; }

template <class T, int U, int CW, int LS, int NT_MAX>
__global__ void __launch_bounds__(NT_MAX, (conv_minb<T, U>())) gl_conv_fwd_is(const __grid_constant__ Geom G, const SlidePlan sp, int64_t Pc,
                                                         const T* __restrict__ ray, const T* __restrict__ sys_kt,
                                                         const T* __restrict__ sys_w, const float* __restrict__ obs,
                                                         const int32_t* __restrict__ system_id, int64_t p_base,
                                                         T* __restrict__ gpix, T* __restrict__ chi, float* __restrict__ out_model) {
    constexpr int SEG = (CW + U - 1 + 1) & ~1, UP2 = (U + 1) & ~1;
    extern __shared__ __align__(16) unsigned char conv_smem[];
    T* taps = reinterpret_cast<T*>(conv_smem);                   // [n_copy][s*s][ps]
    __shared__ T red[NT_MAX];
    const int s = G.s, N = G.N, NPH = s * s;
    const int slot = threadIdx.x / sp.tpp, lt = threadIdx.x - slot * sp.tpp;
    const int64_t p = (int64_t)blockIdx.x * sp.ppc + slot;
    const bool live = slot < sp.ppc && p < Pc;
    const int sys = (live && system_id) ? system_id[p_base + p] : 0;
    // stage the taps in PLANE order: plane (a,b) uses kt[(a+c)%s][(b+c)%s]
    const int copy = sp.shared_taps ? 0 : slot;
    {
        const int first = sp.shared_taps ? threadIdx.x : lt, stride = sp.shared_taps ? blockDim.x : sp.tpp;
        T* tp = taps + (size_t)copy * NPH * sp.ps;
        const T* kt = sys_kt + (size_t)sys * NPH * U * U;
        if (sp.shared_taps || slot < sp.ppc)
            for (int e = first; e < NPH * U * UP2; e += stride) {
                const int v = e % UP2, u = (e / UP2) % U, ph = e / (UP2 * U);
                const int a = ph / s, b = ph - a * s;
                tp[(size_t)ph * sp.ps + u * UP2 + v] = (v < U) ? kt[(size_t)(((a + G.c) % s) * s + (b + G.c) % s) * U * U + u * U + v] : T(0);
            }
    }
    if (live && gpix) zero_gpix_border(G, gpix + (size_t)p * gpix_stride(G), lt, sp.tpp);
    __syncthreads();
    // LS lanes share a column group and split the planes (LS = 4 where a particle has too few column groups to fill
    // the machine, with a shuffle reduction per output row; LS = 1: one thread walks all planes).
    const int g = lt / LS, pq = lt - g * LS;
    const bool active = live && g < sp.ncg;
    const unsigned amask = __ballot_sync(0xffffffffu, active);   // the LS lanes of a column group are active together
    T c2 = T(0);
    if (active) {
        const int nj = NPH / LS;                                 // planes per lane
        const size_t plane = (size_t)G.Hp * G.Wp;
        const T* in = ray + (size_t)p * ray_stride(G) + (size_t)CW * g;
        const T* tp = taps + (size_t)copy * NPH * sp.ps;
        T acc[U][CW];
#pragma unroll
        for (int u = 0; u < U; ++u)
#pragma unroll
            for (int q = 0; q < CW; ++q) acc[u][q] = T(0);
        constexpr bool PF = conv_pf<T, U>();
        T cur[SEG], nxt[PF ? SEG : 2];
        if constexpr (PF) load_seg<T, SEG>(nxt, in + (size_t)pq * plane);
        const int steps = G.Hp * nj;
        int i = 0, j = 0;
        for (int t = 0; t < steps; ++t) {
            int jn = j + 1, in_ = i;
            if (jn == nj) { jn = 0; in_ = i + 1; }
            if constexpr (PF) {
#pragma unroll
                for (int v = 0; v < SEG; ++v) cur[v] = nxt[v];
                if (t + 1 < steps) load_seg<T, SEG>(nxt, in + (size_t)(pq + LS * jn) * plane + (size_t)in_ * G.Wp);
            } else {
                load_seg<T, SEG>(cur, in + (size_t)(pq + LS * j) * plane + (size_t)i * G.Wp);
            }
            conv_slide<T, U, CW, SEG>(acc, tp + (size_t)(pq + LS * j) * sp.ps, cur);
            if (jn == 0) {                                       // input row i done: output row i - U + 1 is complete
                const int pr = i - (U - 1);
                if constexpr (LS == 1) {
                    if (pr >= 0) {
#pragma unroll
                        for (int q = 0; q < CW; ++q) {
                            const int pc = CW * g + q;
                            if (pc < N)
                                c2 += pixel_epilogue<T>(G, acc[U - 1][q], pr, pc, sys, (size_t)(p_base + p), (int)p, obs, sys_w, gpix, out_model);
                        }
                    }
                } else {
                    static_assert(LS == 1 || (LS == 4 && CW <= 4), "lane split: 4 lanes, at most 4 columns");
                    T m[CW];
#pragma unroll
                    for (int q = 0; q < CW; ++q) {
                        T v = acc[U - 1][q];
                        v += __shfl_xor_sync(amask, v, 1);
                        v += __shfl_xor_sync(amask, v, 2);
                        m[q] = v;
                    }
                    if (pr >= 0) {
                        T mine = m[0];
#pragma unroll
                        for (int q = 1; q < CW; ++q) mine = (pq == q) ? m[q] : mine;
                        const int pc = CW * g + pq;
                        if (pq < CW && pc < N)
                            c2 += pixel_epilogue<T>(G, mine, pr, pc, sys, (size_t)(p_base + p), (int)p, obs, sys_w, gpix, out_model);
                    }
                }
#pragma unroll
                for (int u = U - 1; u > 0; --u)
#pragma unroll
                    for (int q = 0; q < CW; ++q) acc[u][q] = acc[u - 1][q];
#pragma unroll
                for (int q = 0; q < CW; ++q) acc[0][q] = T(0);
            }
            i = in_; j = jn;
        }
    }
    if (chi) {                                                   // fixed-order sum over the slot's threads
        red[threadIdx.x] = c2;
        __syncthreads();
        if (lt == 0 && live) {
            T tot = T(0);
            for (int k = 0; k < sp.tpp; ++k) tot += red[slot * sp.tpp + k];
            chi[p] = tot;
        }
    }
}

// Transpose of step D.  Same mapping (sp is the BACKWARD SlidePlan: ncg covers the N + max plane shift output
// columns).  For plane (a,b), rows R in [oa, oa + N):
//   gbar_ab[R][j'] = sum_{k,l<U} F[k][l] gp[R + k][j' + l],  F[k][l] = kt[(a+c)%s][(b+c)%s][U-1-k][U-1-l]
// gbar (plane layout) overwrites the ray buffer; only the N x N interior of each plane is meaningful afterwards.
template <class T, int U, int CW, int LS, int NT_MAX>
__global__ void __launch_bounds__(NT_MAX, (conv_minb<T, U>())) gl_conv_bwd_is(const __grid_constant__ Geom G, const SlidePlan sp, int64_t Pc,
                                                         const T* __restrict__ gpix, const T* __restrict__ sys_kt,
                                                         const int32_t* __restrict__ system_id, int64_t p_base,
                                                         T* __restrict__ gbar) {
    using V2 = typename Vec2<T>::type;
    constexpr int SEG = (CW + U - 1 + 1) & ~1, UP2 = (U + 1) & ~1;
    extern __shared__ __align__(16) unsigned char conv_smem[];
    T* taps = reinterpret_cast<T*>(conv_smem);                   // [n_copy][s*s][ps], flipped
    const int s = G.s, N = G.N, NPH = s * s;
    const int slot = threadIdx.x / sp.tpp, lt = threadIdx.x - slot * sp.tpp;
    const int64_t p = (int64_t)blockIdx.x * sp.ppc + slot;
    const bool live = slot < sp.ppc && p < Pc;
    const int sys = (live && system_id) ? system_id[p_base + p] : 0;
    const int copy = sp.shared_taps ? 0 : slot;
    {
        const int first = sp.shared_taps ? threadIdx.x : lt, stride = sp.shared_taps ? blockDim.x : sp.tpp;
        T* tp = taps + (size_t)copy * NPH * sp.ps;
        const T* kt = sys_kt + (size_t)sys * NPH * U * U;
        if (sp.shared_taps || slot < sp.ppc)
            for (int e = first; e < NPH * U * UP2; e += stride) {
                const int v = e % UP2, u = (e / UP2) % U, ph = e / (UP2 * U);
                const int a = ph / s, b = ph - a * s;
                tp[(size_t)ph * sp.ps + u * UP2 + v] =
                    (v < U) ? kt[(size_t)(((a + G.c) % s) * s + (b + G.c) % s) * U * U + (U - 1 - u) * U + (U - 1 - v)] : T(0);
            }
    }
    __syncthreads();
    const int g = lt / LS, pq = lt - g * LS;
    if (!(live && g < sp.ncg)) return;
    const T* tp = taps + (size_t)copy * NPH * sp.ps;
    const T* gp = gpix + (size_t)p * gpix_stride(G) + (size_t)CW * g;
    const int rows = N + U - 1;
    for (int ph = pq; ph < NPH; ph += LS) {
        const int a = ph / s, oa = phase_shift(G, a);
        T* out = gbar + (size_t)p * ray_stride(G) + ((size_t)ph * G.Hp) * G.Wp + (size_t)CW * g;
        const T* in = gp + (size_t)oa * G.Wg;
        T acc[U][CW];
#pragma unroll
        for (int u = 0; u < U; ++u)
#pragma unroll
            for (int q = 0; q < CW; ++q) acc[u][q] = T(0);
        constexpr bool PF = conv_pf<T, U>();
        T cur[SEG], nxt[PF ? SEG : 2];
        if constexpr (PF) load_seg<T, SEG>(nxt, in);
        for (int r = 0; r < rows; ++r) {
            if constexpr (PF) {
#pragma unroll
                for (int v = 0; v < SEG; ++v) cur[v] = nxt[v];
                if (r + 1 < rows) load_seg<T, SEG>(nxt, in + (size_t)(r + 1) * G.Wg);
            } else {
                load_seg<T, SEG>(cur, in + (size_t)r * G.Wg);
            }
            conv_slide<T, U, CW, SEG>(acc, tp + (size_t)ph * sp.ps, cur);
            const int n = r - (U - 1);                           // finished output row (relative to oa)
            if (n >= 0) {
                T* o = out + (size_t)(oa + n) * G.Wp;
#pragma unroll
                for (int q = 0; q < CW; q += 2) { V2 v; v.x = acc[U - 1][q]; v.y = acc[U - 1][q + 1]; *reinterpret_cast<V2*>(o + q) = v; }
            }
#pragma unroll
            for (int u = U - 1; u > 0; --u)
#pragma unroll
                for (int q = 0; q < CW; ++q) acc[u][q] = acc[u - 1][q];
#pragma unroll
            for (int q = 0; q < CW; ++q) acc[0][q] = T(0);
        }
    }
}

// ----------------------------------------------------------------------------- two input rows per step (U = 11, 16)
// With many taps the 16-byte tap broadcasts saturate the shared-memory return path (512 B per warp per load, 128 B per
// clock per SM) before the FP64 pipe fills: measured 0.36-0.41 of the FP64 peak with one row per step.  Here every tap
// pair loaded feeds TWO input rows (rows i and i+1 of the same plane), i.e. 4*CW FMAs per load: A[s] is the accumulator
// of output row i + 1 - s, row i adds tap row u into A[u + 1], row i + 1 adds it into A[u]; after the pair, A[U] and
// A[U - 1] are complete and the accumulators shift by two.
template <class T, int U, int CW, int SEG>
__device__ __forceinline__ void conv_slide2(T (&A)[U + 1][CW], const T* __restrict__ tap, const T (&s0)[SEG], const T (&s1)[SEG]) {
    using V2 = typename Vec2<T>::type;
    constexpr int UP2 = (U + 1) & ~1;
#pragma unroll
    for (int u = 0; u < U; ++u) {
#pragma unroll
        for (int v = 0; v < UP2; v += 2) {
            const V2 k = *reinterpret_cast<const V2*>(tap + u * UP2 + v);
#pragma unroll
            for (int q = 0; q < CW; ++q) {
                A[u + 1][q] = Real<T>::fma(k.x, s0[q + v], A[u + 1][q]);
                A[u][q] = Real<T>::fma(k.x, s1[q + v], A[u][q]);
                if (v + 1 < U) {
                    A[u + 1][q] = Real<T>::fma(k.y, s0[q + v + 1], A[u + 1][q]);
                    A[u][q] = Real<T>::fma(k.y, s1[q + v + 1], A[u][q]);
                }
            }
        }
    }
}

template <class T, int U, int CW>
__device__ __forceinline__ void shift2(T (&A)[U + 1][CW]) {
#pragma unroll
    for (int u = U; u > 1; --u)
#pragma unroll
        for (int q = 0; q < CW; ++q) A[u][q] = A[u - 2][q];
#pragma unroll
    for (int q = 0; q < CW; ++q) { A[0][q] = T(0); A[1][q] = T(0); }
}

template <class T, int SEG>
__device__ __forceinline__ void load_seg_or_zero(T (&seg)[SEG], const T* __restrict__ p, bool ok) {
    if (ok) load_seg<T, SEG>(seg, p);
    else {
#pragma unroll
        for (int v = 0; v < SEG; ++v) seg[v] = T(0);
    }
}

// Step D + E, one thread per column group, all planes, two rows per step.  Launch geometry as gl_conv_fwd_is (LS = 1).
template <class T, int U, int CW, int NT_MAX>
__global__ void __launch_bounds__(NT_MAX) gl_conv_fwd_is2(const __grid_constant__ Geom G, const SlidePlan sp, int64_t Pc,
                                                          const T* __restrict__ ray, const T* __restrict__ sys_kt,
                                                          const T* __restrict__ sys_w, const float* __restrict__ obs,
                                                          const int32_t* __restrict__ system_id, int64_t p_base,
                                                          T* __restrict__ gpix, T* __restrict__ chi, float* __restrict__ out_model) {
    constexpr int SEG = (CW + U - 1 + 1) & ~1, UP2 = (U + 1) & ~1;
    extern __shared__ __align__(16) unsigned char conv_smem[];
    T* taps = reinterpret_cast<T*>(conv_smem);
    __shared__ T red[NT_MAX];
    const int s = G.s, N = G.N, NPH = s * s;
    const int slot = threadIdx.x / sp.tpp, lt = threadIdx.x - slot * sp.tpp;
    const int64_t p = (int64_t)blockIdx.x * sp.ppc + slot;
    const bool live = slot < sp.ppc && p < Pc;
    const int sys = (live && system_id) ? system_id[p_base + p] : 0;
    const int copy = sp.shared_taps ? 0 : slot;
    {
        const int first = sp.shared_taps ? threadIdx.x : lt, stride = sp.shared_taps ? blockDim.x : sp.tpp;
        T* tp = taps + (size_t)copy * NPH * sp.ps;
        const T* kt = sys_kt + (size_t)sys * NPH * U * U;
        if (sp.shared_taps || slot < sp.ppc)
            for (int e = first; e < NPH * U * UP2; e += stride) {
                const int v = e % UP2, u = (e / UP2) % U, ph = e / (UP2 * U);
                const int a = ph / s, b = ph - a * s;
                tp[(size_t)ph * sp.ps + u * UP2 + v] = (v < U) ? kt[(size_t)(((a + G.c) % s) * s + (b + G.c) % s) * U * U + u * U + v] : T(0);
            }
    }
    if (live && gpix) zero_gpix_border(G, gpix + (size_t)p * gpix_stride(G), lt, sp.tpp);
    __syncthreads();
    const int g = lt;
    T c2 = T(0);
    if (live && g < sp.ncg) {
        const size_t plane = (size_t)G.Hp * G.Wp;
        const T* in = ray + (size_t)p * ray_stride(G) + (size_t)CW * g;
        const T* tp = taps + (size_t)copy * NPH * sp.ps;
        T A[U + 1][CW];
#pragma unroll
        for (int u = 0; u <= U; ++u)
#pragma unroll
            for (int q = 0; q < CW; ++q) A[u][q] = T(0);
        for (int i = 0; i < G.Hp; i += 2) {
            const bool two = i + 1 < G.Hp;
            for (int j = 0; j < NPH; ++j) {
                T s0[SEG], s1[SEG];
                const T* row = in + (size_t)j * plane + (size_t)i * G.Wp;
                load_seg<T, SEG>(s0, row);
                load_seg_or_zero<T, SEG>(s1, row + G.Wp, two);
                conv_slide2<T, U, CW, SEG>(A, tp + (size_t)j * sp.ps, s0, s1);
            }
#pragma unroll
            for (int h = 0; h < 2; ++h) {                        // A[U] is output row i - U + 1, A[U - 1] is row i - U + 2
                const int pr = i - (U - 1) + h;
                if (pr >= 0 && pr < N) {
#pragma unroll
                    for (int q = 0; q < CW; ++q) {
                        const int pc = CW * g + q;
                        if (pc < N)
                            c2 += pixel_epilogue<T>(G, A[U - h][q], pr, pc, sys, (size_t)(p_base + p), (int)p, obs, sys_w, gpix, out_model);
                    }
                }
            }
            shift2<T, U, CW>(A);
        }
    }
    if (chi) {
        red[threadIdx.x] = c2;
        __syncthreads();
        if (lt == 0 && live) {
            T tot = T(0);
            for (int k = 0; k < sp.tpp; ++k) tot += red[slot * sp.tpp + k];
            chi[p] = tot;
        }
    }
}

// Transpose of step D, two rows per step.  Launch geometry as gl_conv_bwd_is (LS = 1).
template <class T, int U, int CW, int NT_MAX>
__global__ void __launch_bounds__(NT_MAX) gl_conv_bwd_is2(const __grid_constant__ Geom G, const SlidePlan sp, int64_t Pc,
                                                          const T* __restrict__ gpix, const T* __restrict__ sys_kt,
                                                          const int32_t* __restrict__ system_id, int64_t p_base,
                                                          T* __restrict__ gbar) {
    using V2 = typename Vec2<T>::type;
    constexpr int SEG = (CW + U - 1 + 1) & ~1, UP2 = (U + 1) & ~1;
    extern __shared__ __align__(16) unsigned char conv_smem[];
    T* taps = reinterpret_cast<T*>(conv_smem);
    const int s = G.s, N = G.N, NPH = s * s;
    const int slot = threadIdx.x / sp.tpp, lt = threadIdx.x - slot * sp.tpp;
    const int64_t p = (int64_t)blockIdx.x * sp.ppc + slot;
    const bool live = slot < sp.ppc && p < Pc;
    const int sys = (live && system_id) ? system_id[p_base + p] : 0;
    const int copy = sp.shared_taps ? 0 : slot;
    {
        const int first = sp.shared_taps ? threadIdx.x : lt, stride = sp.shared_taps ? blockDim.x : sp.tpp;
        T* tp = taps + (size_t)copy * NPH * sp.ps;
        const T* kt = sys_kt + (size_t)sys * NPH * U * U;
        if (sp.shared_taps || slot < sp.ppc)
            for (int e = first; e < NPH * U * UP2; e += stride) {
                const int v = e % UP2, u = (e / UP2) % U, ph = e / (UP2 * U);
                const int a = ph / s, b = ph - a * s;
                tp[(size_t)ph * sp.ps + u * UP2 + v] =
                    (v < U) ? kt[(size_t)(((a + G.c) % s) * s + (b + G.c) % s) * U * U + (U - 1 - u) * U + (U - 1 - v)] : T(0);
            }
    }
    __syncthreads();
    const int g = lt;
    if (!(live && g < sp.ncg)) return;
    const T* tp = taps + (size_t)copy * NPH * sp.ps;
    const T* gp = gpix + (size_t)p * gpix_stride(G) + (size_t)CW * g;
    const int rows = N + U - 1;
    for (int ph = 0; ph < NPH; ++ph) {
        const int a = ph / s, oa = phase_shift(G, a);
        T* out = gbar + (size_t)p * ray_stride(G) + ((size_t)ph * G.Hp) * G.Wp + (size_t)CW * g;
        const T* in = gp + (size_t)oa * G.Wg;
        T A[U + 1][CW];
#pragma unroll
        for (int u = 0; u <= U; ++u)
#pragma unroll
            for (int q = 0; q < CW; ++q) A[u][q] = T(0);
        for (int r = 0; r < rows; r += 2) {
            T s0[SEG], s1[SEG];
            load_seg<T, SEG>(s0, in + (size_t)r * G.Wg);
            load_seg_or_zero<T, SEG>(s1, in + (size_t)(r + 1) * G.Wg, r + 1 < rows);
            conv_slide2<T, U, CW, SEG>(A, tp + (size_t)ph * sp.ps, s0, s1);
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                const int n = r - (U - 1) + h;                   // finished output row (relative to oa)
                if (n >= 0 && n < N) {
                    T* o = out + (size_t)(oa + n) * G.Wp;
#pragma unroll
                    for (int q = 0; q < CW; q += 2) { V2 v; v.x = A[U - h][q]; v.y = A[U - h][q + 1]; *reinterpret_cast<V2*>(o + q) = v; }
                }
            }
            shift2<T, U, CW>(A);
        }
    }
}

}  // namespace gl
