// gl_conv_ct.cuh -- step D (+ E) and its transpose with the TAPS AS UNIFORM OPERANDS (single-system configurations).
//
// Why (gl_probe_pipe kinds 4 / 7 / 8, profiles/r2d): on B200 an FP64 FMA whose three operands are three different vector
// registers issues at 12.1 T lane-op/s, one with two vector registers and ONE UNIFORM operand (uniform register / constant
// bank) at the full 18.5 T: the limit is register-file reads per DFMA.  The tap-stationary kernels (gl_conv_ts.cuh) keep
// the taps in per-lane vector registers -- every DFMA reads tap, window and accumulator from the register file -- and top
// out at 0.47-0.65 of the peak.  Here all lanes of a warp work on the SAME phase plane and tap row at the same time (a lane
// = one column group of CW output columns), so the tap is warp-uniform: it sits in CONSTANT memory, reaches the FMA through
// a uniform register (SASS: LDCU + DFMA R, R, UR, R), costs no register-file read, no shared-memory traffic and no vector
// register.  The input-stationary sliding accumulators of gl_conv.cuh do the rest: a thread walks down the input rows once,
// every row segment (CW + U - 1 values, loaded one step ahead) is scattered into the U output rows it contributes to
// (acc[U][CW]), the finished row leaves at the bottom.  Tap rows whose output row lies outside the thread's row band are
// skipped (warp-uniform test), so the zero border rows of the padded planes cost nothing.
//
// The constant table is process-wide state: CT_NSLOT slots of CT_SLOT doubles; a single-system configuration takes a slot
// in gl_config_create and refills it from the caller's PSF on every call (cudaMemcpyToSymbolAsync, device to device, on the
// caller's stream).  Configurations without a slot, several systems (a particle's taps then depend on its system_id: not
// warp-uniform) and tap counts without an instance keep the tap-stationary kernels.
#pragma once
#include "gl_common.cuh"
#include "gl_conv.cuh"

namespace gl {

constexpr int CT_SLOT = 2112;          // doubles per slot: 16 planes x 11 x 12 (config 5); 4 x 16 x 16 and 16 x 6 x 6 fit too
constexpr int CT_NSLOT = 3;
__constant__ double c_ctap[CT_NSLOT][CT_SLOT];

template <class T>
__device__ __forceinline__ T ctap(int slot, int idx) {
    if constexpr (sizeof(T) == 8) return c_ctap[slot][idx];
    else return reinterpret_cast<const float*>(&c_ctap[slot][0])[idx];
}

// Tap table of ONE system in plane order, rows padded to UP2 = U rounded up to even: out[ph][u][UP2] with plane (a, b)
// using kt[(a + c) % s][(b + c) % s]; this is what the constant slot holds.
template <class T>
__global__ void gl_ctap_stage_kernel(const __grid_constant__ Geom G, int NPH, const T* __restrict__ sys_kt, T* __restrict__ out) {
    const int s = G.s, U = G.U, UP2 = (U + 1) & ~1;
    for (int e = blockIdx.x * blockDim.x + threadIdx.x; e < NPH * U * UP2; e += gridDim.x * blockDim.x) {
        const int v = e % UP2, u = (e / UP2) % U, ph = e / (UP2 * U);
        const int a = ph / s, b = ph - a * s;
        out[e] = (v < U) ? sys_kt[(size_t)(((a + G.c) % s) * s + (b + G.c) % s) * U * U + u * U + v] : T(0);
    }
}

struct CtPlan {
    int ncg;      // column groups per particle = threads per particle: thread t of the grid works on item t = (particle, column group)
    int n_bands;  // forward: row bands per particle (a function of the geometry only: the chi^2 partials depend on it)
    int rbh;      // forward: output rows per band
};
// CTAs are always CT_NT threads = 4 warps, one per scheduler: with 2, 3 or 5 warps per CTA the schedulers of an SM carry
// unequal shares of an FP64-bound kernel (measured on config 3: 5-warp CTAs 13.2 ms, 8-warp CTAs 8.4 ms for the same work).
constexpr int CT_NT = 128;      // no minimum-blocks bound: ptxas then settles at 168 registers (3 CTAs per SM) for the U = 11 transpose; (CT_NT, 1) took 182 and measured 30 % slower, (CT_NT, 3) spills at U = 16

// acc[u][q] += sum_v tap[u][v] seg[q + v] for the tap rows u in [ulo, uhi]; FLIP: the transpose's taps kt[U-1-u][U-1-v].
// Tap rows are taken in groups of GU = 4 with the tap column v as the OUTER loop inside a group, so that two FMAs into the same
// accumulator are GU * CW instructions apart (with u outermost they were CW apart: the kernel waited on the FP64 latency);
// a group runs if any of its rows is wanted -- the other rows of it then add into accumulators that are never emitted, which is
// the price of coarse groups at the edges of a row band (measured: at CW = 2 groups of 4 beat groups of 8, config 3 step D 7.17 ->
// 6.26 ms; at CW = 4 groups of 4 beat groups of 2 and 3).
template <class T, int U, int CW, int SEG, bool FLIP>
__device__ __forceinline__ void ct_slide(T (&acc)[U][CW], int slot, int tbase, const T (&seg)[SEG], int ulo, int uhi) {
    constexpr int UP2 = (U + 1) & ~1, GU = CW >= 4 ? ((16 / CW) < 1 ? 1 : 16 / CW) : 4;
#pragma unroll
    for (int u0 = 0; u0 < U; u0 += GU) {
        if (u0 + GU - 1 >= ulo && u0 <= uhi) {
#pragma unroll
            for (int v = 0; v < U; ++v) {
#pragma unroll
                for (int u = u0; u < (u0 + GU < U ? u0 + GU : U); ++u) {
                    const T k = ctap<T>(slot, tbase + (FLIP ? (U - 1 - u) * UP2 + (U - 1 - v) : u * UP2 + v));
#pragma unroll
                    for (int q = 0; q < CW; ++q) acc[u][q] = Real<T>::fma(k, seg[q + v], acc[u][q]);
                }
            }
        }
    }
}

template <class T, int U, int CW>
__device__ __forceinline__ void ct_shift(T (&acc)[U][CW]) {
#pragma unroll
    for (int u = U - 1; u > 0; --u)
#pragma unroll
        for (int q = 0; q < CW; ++q) acc[u][q] = acc[u - 1][q];
#pragma unroll
    for (int q = 0; q < CW; ++q) acc[0][q] = T(0);
}

// Step D + E.  grid = (ceil(Pc * ncg / CT_NT), n_bands).  chi: [Pc][n_bands * ncg], one partial per thread (summed in a
// fixed order by gl_finalize_kernel).
template <class T, int U, int CW>
__global__ void __launch_bounds__(CT_NT) gl_conv_fwd_ct(const __grid_constant__ Geom G, const CtPlan cp, int slot_c, int64_t Pc,
                                                        const T* __restrict__ ray, const T* __restrict__ sys_w,
                                                        const float* __restrict__ obs, int64_t p_base, T* __restrict__ gpix,
                                                        T* __restrict__ chi, float* __restrict__ out_model) {
    constexpr int SEG = (CW + U - 1 + 1) & ~1, UP2 = (U + 1) & ~1;
    const int N = G.N, NPH = G.binned ? 1 : G.s * G.s;         // binned (psf_grid 1, dedicated path): the image is plane 0
    const int64_t item = (int64_t)blockIdx.x * CT_NT + threadIdx.x;
    const int64_t p = item / cp.ncg;
    const int g = (int)(item - p * cp.ncg);
    const bool act = p < Pc;
    const int band = blockIdx.y, b0 = band * cp.rbh, b1 = min(N, b0 + cp.rbh);
    if (act && gpix && band == 0) zero_gpix_border(G, gpix + (size_t)p * gpix_stride(G), g, cp.ncg);
    // Every thread of the CTA runs the row walk -- the idle lanes of the last CTA on item 0, their results dropped -- so that
    // the loop is convergent code: inside a divergent branch ptxas cannot use the uniform datapath and the taps would come
    // through vector constant loads (LDC) into vector registers.
    const int64_t pa = act ? p : 0;
    const int ga = act ? g : 0;
    T c2 = T(0);
    {
        const size_t plane = (size_t)G.Hp * G.Wp;
        const T* in = ray + (size_t)pa * ray_stride(G) + (size_t)CW * ga;
        T acc[U][CW];
#pragma unroll
        for (int u = 0; u < U; ++u)
#pragma unroll
            for (int q = 0; q < CW; ++q) acc[u][q] = T(0);
        T cur[SEG], nxt[SEG];
        load_seg<T, SEG>(nxt, in + (size_t)b0 * G.Wp);
        const int i_end = b1 + U - 1;                                // input rows [b0, i_end)
        for (int i = b0; i < i_end; ++i) {
            for (int j = 0; j < NPH; ++j) {
#pragma unroll
                for (int v = 0; v < SEG; ++v) cur[v] = nxt[v];
                const int jn = j + 1 < NPH ? j + 1 : 0, in_ = j + 1 < NPH ? i : i + 1;
                if (in_ < i_end) load_seg<T, SEG>(nxt, in + (size_t)jn * plane + (size_t)in_ * G.Wp);
                // tap row u of input row i feeds output row i - u, wanted iff b0 <= i - u < b1
                ct_slide<T, U, CW, SEG, false>(acc, slot_c, j * (U * UP2), cur, i - b1 + 1, i - b0);
            }
            const int pr = i - (U - 1);                              // input row i done: output row i - U + 1 is complete
            if (pr >= b0 && act) {
#pragma unroll
                for (int q = 0; q < CW; ++q) {
                    const int pc = CW * g + q;
                    if (pc < N) c2 += pixel_epilogue<T>(G, acc[U - 1][q], pr, pc, 0, (size_t)(p_base + p), (int)p, obs, sys_w, gpix, out_model);
                }
            }
            ct_shift<T, U, CW>(acc);
        }
    }
    if (chi && act) chi[(p * cp.n_bands + band) * cp.ncg + g] = c2;
}

// Transpose of step D.  grid = (s*s, ceil(Pc * ncg / CT_NT)): one phase plane per CTA, every plane its own output; the plane is
// the FASTEST grid index, so the s*s CTAs that read the same g_pix rows run together and share them in L2 (with the plane as the
// slow index every plane re-read g_pix from DRAM: 4.0 GB per config-5 launch against 0.28 GB of g_pix).
//   gbar_ab[R][j'] = sum_{k,l<U} kt_ab[U-1-k][U-1-l] gp[R + k][j' + l],  R in [oa, oa + N)
template <class T, int U, int CW>
__global__ void __launch_bounds__(CT_NT) gl_conv_bwd_ct(const __grid_constant__ Geom G, const CtPlan cp, int slot_c, int64_t Pc,
                                                        const T* __restrict__ gpix, T* __restrict__ gbar) {
    using V2 = typename Vec2<T>::type;
    constexpr int SEG = (CW + U - 1 + 1) & ~1, UP2 = (U + 1) & ~1;
    const int N = G.N, s = G.s;
    const int64_t item = (int64_t)blockIdx.y * CT_NT + threadIdx.x;
    const int64_t p = item / cp.ncg;
    const int g = (int)(item - p * cp.ncg);
    const bool act = p < Pc;                                         // idle lanes walk item 0 (convergent loop, see the forward kernel)
    const int64_t pa = act ? p : 0;
    const int ga = act ? g : 0;
    const int ph = blockIdx.x, a = ph / s, oa = phase_shift(G, a);
    const T* in = gpix + (size_t)pa * gpix_stride(G) + (size_t)oa * G.Wg + (size_t)CW * ga;
    T* out = gbar + (size_t)pa * ray_stride(G) + ((size_t)ph * G.Hp + oa) * G.Wp + (size_t)CW * ga;
    T acc[U][CW];
#pragma unroll
    for (int u = 0; u < U; ++u)
#pragma unroll
        for (int q = 0; q < CW; ++q) acc[u][q] = T(0);
    T cur[SEG], nxt[SEG];
    load_seg<T, SEG>(nxt, in);
    const int rows = N + U - 1;
    for (int r = 0; r < rows; ++r) {
#pragma unroll
        for (int v = 0; v < SEG; ++v) cur[v] = nxt[v];
        if (r + 1 < rows) load_seg<T, SEG>(nxt, in + (size_t)(r + 1) * G.Wg);
        ct_slide<T, U, CW, SEG, true>(acc, slot_c, ph * (U * UP2), cur, r - N + 1, r);      // output row r - u in [0, N)
        const int n = r - (U - 1);
        if (n >= 0 && act) {
            T* o = out + (size_t)n * G.Wp;
#pragma unroll
            for (int q = 0; q < CW; q += 2) { V2 v; v.x = acc[U - 1][q]; v.y = acc[U - 1][q + 1]; *reinterpret_cast<V2*>(o + q) = v; }
        }
        ct_shift<T, U, CW>(acc);
    }
}

}  // namespace gl
