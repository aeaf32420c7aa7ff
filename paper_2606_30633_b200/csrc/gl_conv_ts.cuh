// gl_conv_ts.cuh -- step D (+ E) and its transpose, "tap-stationary" form fed by TMA (sm_100a).
//
// Why (profiles/r2a_cfg5_f64.md): the round-1 sliding kernels read every tap from shared memory once per FMA group; a
// 16-byte tap broadcast costs 4 shared-memory wavefronts = as many SM cycles as the 8 DFMAs it feeds, so shared-memory
// return bandwidth and FP64 issue were co-limiting at ~50 %, on 4-8 warps per SM whose input rows came through
// per-thread global loads (top stall long_scoreboard).  Here the roles are swapped:
//   * TAPS LIVE IN REGISTERS.  A lane owns ONE phase plane j and ONE group a of NU = ceil(U / G) tap rows (NU * U taps,
//     loaded once per CTA); LPG = NPH * G lanes cover all planes and tap rows of a column group of CW output columns.
//   * INPUT ROWS COME FROM SHARED MEMORY, filled by TMA: one cp.async.bulk.tensor box per input row (all NPH planes x the
//     CTA's column band + halo, zero-filled outside the tensor) into an S-stage ring guarded by full / empty mbarriers;
//     a lane reads only its CW + U - 1 window per row (16-byte loads; the row pitch is chosen = 16 mod 32 bytes so that the
//     planes of a quarter-warp hit distinct banks).  Per row step a lane does NU * U * CW FMAs on ~(CW + U - 1) loaded values.
//   * Sliding accumulators acc[NU][CW] as before (slot i = output row r - a NU - i), rotated at compile time instead of moved.
//     The finished slot of tap-row group a is handed to group a + 1 by ONE shuffle per value (a systolic chain: it is
//     exactly the initial value of the slot that group starts at the next row), the last group holds the plane's row.
//   * forward: every lane drops its plane's finished row into a small per-warp shared-memory buffer; once per fill the
//     warp sums the NPH planes of each output pixel in a fixed order and applies step E, one or two pixels per lane.
//     transpose: every plane is its own output, no reduction.
//   * persistent CTAs: a dedicated producer warp streams the rows of consecutive work items through the ring, so the
//     pipeline never drains between particles.
#pragma once
#include <cuda.h>
#include <type_traits>
#include "gl_common.cuh"
#include "gl_conv.cuh"

namespace gl {

// ----------------------------------------------------------------------------- PTX helpers (mbarrier, TMA)
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t* bar, int count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_fence_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
__device__ __forceinline__ void mbar_arrive(uint64_t* bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint64_t* bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ uint32_t mbar_try_wait(uint64_t* bar, uint32_t parity) {
    uint32_t ok;
    asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
                 : "=r"(ok) : "r"(smem_u32(bar)), "r"(parity) : "memory");
    return ok;
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
    while (!mbar_try_wait(bar, parity)) {}
}
__device__ __forceinline__ void tma_load_3d(void* dst, const CUtensorMap* tm, int c0, int c1, int c2, uint64_t* bar) {
    asm volatile("cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];"
                 ::"r"(smem_u32(dst)), "l"(tm), "r"(c0), "r"(c1), "r"(c2), "r"(smem_u32(bar)) : "memory");
}

// ----------------------------------------------------------------------------- plan
struct TsPlan {
    int wpc;          // warps per CTA
    int cg_per_cta;   // column groups per CTA (= wpc * CGW)
    int n_bands;      // CTAs per particle
    int ncg;          // column groups that carry output
    int boxw;         // columns of one TMA box (band + halo, padded for the bank-conflict-free pitch)
    int stages;       // ring depth
    int steps;        // input rows walked
    int row0;         // first input row (transpose: the smallest plane shift)
    int stage_elems;  // elements of one stage (multiple of 128 bytes)
    int pbuf_elems;   // forward: elements of one warp's partial-row buffer (0 for the transpose)
};

template <class T, int CW> struct SegVec {
    static constexpr int BYTES = ((CW * (int)sizeof(T)) % 16 == 0) ? 16 : 8;
    static constexpr int VE = BYTES / (int)sizeof(T);
};
template <class T, int U, int CW> __host__ __device__ constexpr int ts_segp() {
    return (CW + U - 1 + SegVec<T, CW>::VE - 1) / SegVec<T, CW>::VE * SegVec<T, CW>::VE;
}

template <class T, int CW, int SEGP>
__device__ __forceinline__ void ts_load_seg(T (&seg)[SEGP], const T* __restrict__ s) {
    constexpr int VE = SegVec<T, CW>::VE;
    if constexpr (SegVec<T, CW>::BYTES == 16) {
        using V = typename std::conditional<sizeof(T) == 8, double2, float4>::type;
#pragma unroll
        for (int v = 0; v < SEGP; v += VE) {
            const V x = *reinterpret_cast<const V*>(s + v);
            if constexpr (sizeof(T) == 8) { seg[v] = x.x; seg[v + 1] = x.y; }
            else { seg[v] = ((const T*)&x)[0]; seg[v + 1] = ((const T*)&x)[1]; seg[v + 2] = ((const T*)&x)[2]; seg[v + 3] = ((const T*)&x)[3]; }
        }
    } else {
        static_assert(sizeof(T) == 4, "8-byte windows: float only");
#pragma unroll
        for (int v = 0; v < SEGP; v += 2) {
            const float2 x = *reinterpret_cast<const float2*>(s + v);
            seg[v] = x.x; seg[v + 1] = x.y;
        }
    }
}

template <class T> __device__ __forceinline__ T shfl_up1(T v) { return __shfl_up_sync(0xffffffffu, v, 1); }

// compile-time loop: f(std::integral_constant<int, I>) for I = 0 .. N - 1
template <int I, int N, class F>
__device__ __forceinline__ void static_for(F&& f) {
    if constexpr (I < N) { f(std::integral_constant<int, I>{}); static_for<I + 1, N>(f); }
}

// One row step of the sliding accumulators, rotation ROT = (row index) mod NU known at compile time:
// logical slot i (output row r - a NU - i) lives in A[(i - ROT) mod NU].  Returns the finished row of this lane's group
// in out[] and re-arms that slot with the row handed over by the previous tap-row group (0 for the first group).
template <class T, int U, int G, int NU, int CW, int SEGP, int ROT>
__device__ __forceinline__ void ts_row_step(T (&A)[NU][CW], const T (&tap)[NU][U], const T (&seg)[SEGP], int a, T (&out)[CW]) {
#pragma unroll
    for (int i = 0; i < NU; ++i) {
        const int ph = (i - ROT + NU) % NU;
#pragma unroll
        for (int v = 0; v < U; ++v)
#pragma unroll
            for (int q = 0; q < CW; ++q) A[ph][q] = Real<T>::fma(tap[i][v], seg[q + v], A[ph][q]);
    }
    constexpr int fin = (NU - 1 - ROT + NU) % NU;
#pragma unroll
    for (int q = 0; q < CW; ++q) {
        out[q] = A[fin][q];
        if constexpr (G > 1) {
            const T rcv = shfl_up1(out[q]);
            A[fin][q] = a == 0 ? T(0) : rcv;
        } else A[fin][q] = T(0);
    }
}

// Launch bounds per tap count.  Registers are allocated per scheduler (16K each): 168 registers = 3 warps per
// scheduler, 128 = 4, above 168 only 2.  U = 6 (158-200 live registers) is capped at 168 by a 9-warp bound; U = 11
// (66 taps = 132 registers alone) keeps up to 255 registers at 2 warps per scheduler (the capped build spills and
// measured 40 % slower); U = 16 needs 128-156.
#ifndef GL_TS_MAXT6
#define GL_TS_MAXT6 288
#endif
#ifndef GL_TS_MAXT11
#define GL_TS_MAXT11 256
#endif
#ifndef GL_TS_MAXT16
#define GL_TS_MAXT16 256
#endif
#ifndef GL_TS_MINB16
#define GL_TS_MINB16 2
#endif
constexpr int GL_TS_MAXT = 288;       // largest block of any instance (plan check)
template <int U> __host__ __device__ constexpr int ts_maxt() { return U == 6 ? GL_TS_MAXT6 : (U == 11 ? GL_TS_MAXT11 : (U == 16 ? GL_TS_MAXT16 : 256)); }
template <int U> __host__ __device__ constexpr int ts_minb() { return U == 16 ? GL_TS_MINB16 : 1; }

// Shared-memory carve-up: ring [stages][stage_elems] T | full[stages], empty[stages] mbarriers
template <class T> __host__ __device__ inline size_t ts_smem_bytes(const TsPlan& pl) {
    return (size_t)pl.stages * pl.stage_elems * sizeof(T) + 2 * pl.stages * sizeof(uint64_t) + 128 +
           (size_t)pl.wpc * pl.pbuf_elems * sizeof(T);
}
// forward kernel: per-warp buffer of per-plane partial rows of one fill, [RPS][CGW * CW][NPH + 2] (plane index fastest;
// the + 2 makes the 16-byte reads of the plane sums and the 8-byte writes of the partials bank-conflict free)
__host__ __device__ constexpr int ts_pj(int NPH) { return NPH == 1 ? 1 : NPH + 2; }
__host__ __device__ constexpr int ts_pbuf_elems(int NPH, int G, int CW, int RPS) { return RPS * (32 / (NPH * G)) * CW * ts_pj(NPH); }

// Step E for one pixel from values already in registers (ob = obs, w = 1 / sigma^2, or sigma^2 with noise_model 1):
// returns the chi^2 term, g = d(-chi^2 / 2 [- ln v / 2]) / d model.  Same arithmetic as pixel_epilogue (gl_conv.cuh).
template <class T>
__device__ __forceinline__ T ts_pixel_terms(const Geom& G, T m, float ob, T w, T& g) {
    const T r = m - (T)ob;
    if (G.noise_model == 1) {
        const bool pos = m > T(0);
        const double v = (double)w + (pos ? (double)m * G.inv_texp : 0.0), iv = 1.0 / v, vp = pos ? G.inv_texp : 0.0;
        const double rd = (double)r;
        g = (T)(-rd * iv + 0.5 * rd * rd * iv * iv * vp - 0.5 * vp * iv);
        return (T)(rd * rd * iv + log(v));
    }
    g = -r * w;
    return r * r * w;
}

// psf_grid 1, dedicated path: the PSF acts at the pixel scale on the BINNED image, and with the
// half-width s (K - 1) / 2 every phase plane has the same shift, so binning is the element-wise sum of the s*s padded planes:
// plane 0 += planes 1 .. NPH - 1 (fixed order).  grid = (ceil(Hp Wp / 256), n_images), block = 256.
template <class T>
__global__ void __launch_bounds__(256) gl_bin_planes_kernel(const __grid_constant__ Geom Gm, T* __restrict__ ray) {
    const size_t plane = (size_t)Gm.Hp * Gm.Wp;
    const size_t e = (size_t)blockIdx.x * 256 + threadIdx.x;
    if (e >= plane) return;
    T* p0 = ray + (size_t)blockIdx.y * ray_stride(Gm) + e;
    T sum = p0[0];
    for (int ph = 1; ph < Gm.s * Gm.s; ++ph) sum += p0[(size_t)ph * plane];
    p0[0] = sum;
}

// ----------------------------------------------------------------------------- step D + E
// Persistent: grid = a few CTAs per SM, block = 32 * (wpc + 1): wpc consumer warps + ONE producer warp.  CTA b owns the
// work items (particle, column band) [b n / grid, (b + 1) n / grid), n = Pc * n_bands, and walks them as one stream of
// stage fills: a fill = RPS consecutive input rows (RPS a multiple of NU, so the accumulator rotation of row i of a fill
// is i mod NU at compile time) of all NPH planes; an item takes ceil(steps / RPS) fills, the rows past the tensor read as
// zeros.  The producer (lane 0 of the last warp) runs up to S fills ahead, across item boundaries, so the pipeline never
// drains between particles; consumers wait once per fill (full[st]) and release it once (empty[st]).
// tm: RAY as a 3-D tensor with the plane index in the MIDDLE, {Wp, NPH * Pc (stride Hp Wp), Hp (stride Wp)}, box
// {boxw, NPH, RPS} -> stage layout [RPS][NPH][boxw]: the planes of a row sit boxw apart (the conflict-free pitch).
// chi: [Pc][n_bands * wpc] per-warp partial sums (summed in a fixed order by gl_finalize_kernel).
template <class T, int U, int G, int NPH, int CW, int RPS>
__global__ void __launch_bounds__((ts_maxt<U>()), (ts_minb<U>())) gl_conv_fwd_ts(const __grid_constant__ CUtensorMap tm, const __grid_constant__ Geom Gm,
                                                             const TsPlan pl, int64_t Pc, const T* __restrict__ sys_kt,
                                                             const T* __restrict__ sys_w, const float* __restrict__ obs,
                                                             const int32_t* __restrict__ system_id, int64_t p_base,
                                                             T* __restrict__ gpix, T* __restrict__ chi, float* __restrict__ out_model) {
    constexpr int LPG = NPH * G, CGW = 32 / LPG, NU = (U + G - 1) / G, UPAD = NU * G, SEGP = ts_segp<T, U, CW>();
    static_assert(32 % LPG == 0 && CW % 2 == 0 && RPS % NU == 0, "lane layout");
    extern __shared__ __align__(128) unsigned char ts_smem[];
    T* ring = reinterpret_cast<T*>(ts_smem);
    uint64_t* full = reinterpret_cast<uint64_t*>(ring + (size_t)pl.stages * pl.stage_elems);
    uint64_t* empty = full + pl.stages;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int s = Gm.s, N = Gm.N, S = pl.stages, R = pl.steps, F = (R + RPS - 1) / RPS;
    const size_t NN = (size_t)N * N;
    const int64_t n_items = Pc * pl.n_bands;
    const int64_t i0 = (int64_t)blockIdx.x * n_items / gridDim.x, i1 = (int64_t)(blockIdx.x + 1) * n_items / gridDim.x;
    if (threadIdx.x == 0) {
        for (int k = 0; k < S; ++k) { mbar_init(full + k, 1); mbar_init(empty + k, pl.wpc); }
        mbar_fence_init();
    }
    __syncthreads();
    if (warp == pl.wpc) {                                           // ---- producer warp
        if (lane == 0) {
            const uint32_t tx = (uint32_t)(pl.boxw * RPS * NPH * sizeof(T));
            int st = 0, use = 0;
            for (int64_t it = i0; it < i1; ++it) {
                const int64_t pp = it / pl.n_bands;
                const int bb = (int)(it - pp * pl.n_bands);
                for (int f = 0; f < F; ++f) {
                    if (use > 0) mbar_wait(empty + st, (uint32_t)((use - 1) & 1));
                    mbar_arrive_expect_tx(full + st, tx);
                    tma_load_3d(ring + (size_t)st * pl.stage_elems, &tm, CW * bb * pl.cg_per_cta, (int)pp * NPH, f * RPS, full + st);
                    if (++st == S) { st = 0; ++use; }
                }
            }
        }
        return;
    }
    const int cgw = lane / LPG, j = (lane % LPG) / G, a = lane % G;
    const int cgl = warp * CGW + cgw;
    const int pa = j / s, pb = j - pa * s;
    const int ktplane = ((pa + Gm.c) % s) * s + (pb + Gm.c) % s;
    T tap[NU][U];
    int cur_sys = -1;
    const T* my = ring + (size_t)j * pl.boxw + CW * cgl;           // this lane's window: row 0 of stage 0
    constexpr int PJ = ts_pj(NPH);
    T* pbuf = reinterpret_cast<T*>(empty + pl.stages) + (size_t)warp * pl.pbuf_elems;     // this warp's partial-row buffer
    T* pb_w = pbuf + (size_t)cgw * CW * PJ + j;                                           // + (i CGW CW + q) PJ
    int st = 0; uint32_t ph = 0;
    for (int64_t it = i0; it < i1; ++it) {
        const int64_t p = it / pl.n_bands;
        const int band = (int)(it - p * pl.n_bands);
        const int sys = system_id ? system_id[p_base + p] : 0;
        if (sys != cur_sys) {                                       // uniform over the CTA
            const T* kt = sys_kt + ((size_t)sys * s * s + ktplane) * U * U;
#pragma unroll
            for (int i = 0; i < NU; ++i)
#pragma unroll
                for (int v = 0; v < U; ++v) tap[i][v] = (a * NU + i < U) ? kt[(a * NU + i) * U + v] : T(0);
            cur_sys = sys;
        }
        T* gp_img = gpix ? gpix + (size_t)p * gpix_stride(Gm) : nullptr;
        if (gp_img) zero_gpix_border(Gm, gp_img, band * (pl.wpc * 32) + threadIdx.x, pl.n_bands * (pl.wpc * 32));
        const int cg0 = band * pl.cg_per_cta + warp * CGW;         // first column group of this warp
        T A[NU][CW];
#pragma unroll
        for (int i = 0; i < NU; ++i)
#pragma unroll
            for (int q = 0; q < CW; ++q) A[i][q] = T(0);
        T c2 = T(0);
        constexpr int NOUT = (RPS * CGW * CW + 31) / 32;           // outputs of a fill per lane
        for (int f = 0; f < F; ++f) {
            // step-E operands of this lane's outputs of the fill: loaded now, used after the FMAs
            constexpr bool PFE = NOUT <= 4;                          // many outputs per lane (single-plane instances): load at use
            float ob_r[PFE ? NOUT : 1]; T w_r[PFE ? NOUT : 1];
#pragma unroll
            for (int k = 0; k < (PFE ? NOUT : 0); ++k) {
                const int o = lane + 32 * k, i = o / (CGW * CW), c = o - i * (CGW * CW);
                const int prow = f * RPS + i - (UPAD - 1), pc = CW * cg0 + c;
                const bool ok = o < RPS * CGW * CW && prow >= 0 && prow < N && pc < N && gp_img != nullptr;
                ob_r[k] = ok ? obs[(size_t)sys * NN + (size_t)prow * N + pc] : 0.f;
                w_r[k] = ok ? sys_w[(size_t)sys * NN + (size_t)prow * N + pc] : T(0);
            }
            mbar_wait(full + st, ph);
            const T* srow = my + (size_t)st * pl.stage_elems;
            static_for<0, RPS>([&](auto ic) {
                constexpr int i = decltype(ic)::value;
                T seg[SEGP];
                ts_load_seg<T, CW, SEGP>(seg, srow + i * (NPH * pl.boxw));
                T out[CW];
                ts_row_step<T, U, G, NU, CW, SEGP, (i % NU)>(A, tap, seg, a, out);
                if (a == G - 1) {                                   // this plane's row of the fill, plane index fastest
#pragma unroll
                    for (int q = 0; q < CW; ++q) pb_w[(i * CGW * CW + q) * PJ] = out[q];
                }
            });
            __syncwarp();
            if (lane == 0) mbar_arrive(empty + st);
            if (++st == S) { st = 0; ph ^= 1u; }
            // plane sums in a fixed order (j = 0 .. NPH - 1) and step E: lane l takes outputs l, l + 32, ... of the fill
#pragma unroll
            for (int k = 0; k < NOUT; ++k) {
                const int o = lane + 32 * k, i = o / (CGW * CW), c = o - i * (CGW * CW);
                const int prow = f * RPS + i - (UPAD - 1), pc = CW * cg0 + c;
                const bool ok = o < RPS * CGW * CW && prow >= 0 && prow < N && pc < N;
                float ob; T w;
                if constexpr (PFE) { ob = ob_r[k]; w = w_r[k]; }
                else {
                    const bool ld = ok && gp_img != nullptr;
                    ob = ld ? obs[(size_t)sys * NN + (size_t)prow * N + pc] : 0.f;
                    w = ld ? sys_w[(size_t)sys * NN + (size_t)prow * N + pc] : T(0);
                }
                const T* src = pbuf + (size_t)(o < RPS * CGW * CW ? o : 0) * PJ;
                T m = T(0);
                if constexpr (NPH == 1) m = src[0];
                else if constexpr (sizeof(T) == 8) {
#pragma unroll
                    for (int jj = 0; jj < NPH; jj += 2) { const double2 x = *reinterpret_cast<const double2*>(src + jj); m += x.x; m += x.y; }
                } else {
#pragma unroll
                    for (int jj = 0; jj < NPH; jj += 2) { const float2 x = *reinterpret_cast<const float2*>(src + jj); m += x.x; m += x.y; }
                }
                if (ok) {
                    if (out_model) out_model[(size_t)(p_base + p) * NN + (size_t)prow * N + pc] = (float)m;
                    if (gp_img) {
                        T g;
                        c2 += ts_pixel_terms<T>(Gm, m, ob, w, g);
                        gp_img[(size_t)(prow + Gm.PADg) * Gm.Wg + pc + Gm.PADg] = g;
                    }
                }
            }
            __syncwarp();
        }
        if (chi) {                                                  // fixed-order lane tree; one partial per warp
            const T tot = warp_sum(c2);
            if (lane == 0) chi[(size_t)p * (pl.n_bands * pl.wpc) + band * pl.wpc + warp] = tot;
        }
    }
}

// ----------------------------------------------------------------------------- transpose of step D
// gbar_j[Rr][c] = sum_{k,l<U} F_j[k][l] gp[Rr + k][c + l], F_j[k][l] = kt_j[U-1-k][U-1-l], rows Rr in [o_a(j), o_a(j) + N),
// written in the plane layout over the ray buffer.  All planes read the SAME padded g_pix rows (a pure shared-memory
// broadcast), so one row schedule from the smallest plane shift serves every plane; a lane stores only the rows of its
// own plane's interior.  Persistent, producer warp and fills as in the forward kernel.
// tm: GPIX as a 3-D tensor {Wg, Hg, Pc}, box {boxw, RPS, 1}.
template <class T, int U, int G, int NPH, int CW, int RPS>
__global__ void __launch_bounds__((ts_maxt<U>()), (ts_minb<U>())) gl_conv_bwd_ts(const __grid_constant__ CUtensorMap tm, const __grid_constant__ Geom Gm,
                                                             const TsPlan pl, int64_t Pc, const T* __restrict__ sys_kt,
                                                             const int32_t* __restrict__ system_id, int64_t p_base,
                                                             T* __restrict__ gbar) {
    constexpr int LPG = NPH * G, CGW = 32 / LPG, NU = (U + G - 1) / G, UPAD = NU * G, SEGP = ts_segp<T, U, CW>();
    static_assert(32 % LPG == 0 && RPS % NU == 0, "lane layout");
    extern __shared__ __align__(128) unsigned char ts_smem[];
    T* ring = reinterpret_cast<T*>(ts_smem);
    uint64_t* full = reinterpret_cast<uint64_t*>(ring + (size_t)pl.stages * pl.stage_elems);
    uint64_t* empty = full + pl.stages;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int s = Gm.s, N = Gm.N, S = pl.stages, R = pl.steps, F = (R + RPS - 1) / RPS;
    const int64_t n_items = Pc * pl.n_bands;
    const int64_t i0 = (int64_t)blockIdx.x * n_items / gridDim.x, i1 = (int64_t)(blockIdx.x + 1) * n_items / gridDim.x;
    if (threadIdx.x == 0) {
        for (int k = 0; k < S; ++k) { mbar_init(full + k, 1); mbar_init(empty + k, pl.wpc); }
        mbar_fence_init();
    }
    __syncthreads();
    if (warp == pl.wpc) {                                           // ---- producer warp
        if (lane == 0) {
            const uint32_t tx = (uint32_t)(pl.boxw * RPS * sizeof(T));
            int st = 0, use = 0;
            for (int64_t it = i0; it < i1; ++it) {
                const int64_t pp = it / pl.n_bands;
                const int bb = (int)(it - pp * pl.n_bands);
                for (int f = 0; f < F; ++f) {
                    if (use > 0) mbar_wait(empty + st, (uint32_t)((use - 1) & 1));
                    mbar_arrive_expect_tx(full + st, tx);
                    tma_load_3d(ring + (size_t)st * pl.stage_elems, &tm, CW * bb * pl.cg_per_cta, pl.row0 + f * RPS, (int)pp, full + st);
                    if (++st == S) { st = 0; ++use; }
                }
            }
        }
        return;
    }
    const int cgw = lane / LPG, j = (lane % LPG) / G, a = lane % G;
    const int cgl = warp * CGW + cgw;
    const int pa = j / s, pb = j - pa * s;
    const int ktplane = ((pa + Gm.c) % s) * s + (pb + Gm.c) % s;
    const int oa = phase_shift(Gm, pa);
    T tap[NU][U];
    int cur_sys = -1;
    const T* my = ring + CW * cgl;
    int st = 0; uint32_t ph = 0;
    for (int64_t it = i0; it < i1; ++it) {
        const int64_t p = it / pl.n_bands;
        const int band = (int)(it - p * pl.n_bands);
        const int sys = system_id ? system_id[p_base + p] : 0;
        if (sys != cur_sys) {
            const T* kt = sys_kt + ((size_t)sys * s * s + ktplane) * U * U;
#pragma unroll
            for (int i = 0; i < NU; ++i)
#pragma unroll
                for (int v = 0; v < U; ++v) tap[i][v] = (a * NU + i < U) ? kt[(U - 1 - (a * NU + i)) * U + (U - 1 - v)] : T(0);
            cur_sys = sys;
        }
        const int cg = band * pl.cg_per_cta + cgl;
        const bool writer = a == G - 1 && cg < pl.ncg;
        T* outp = gbar + (size_t)p * ray_stride(Gm) + (size_t)j * Gm.Hp * Gm.Wp + (size_t)CW * cg;
        T A[NU][CW];
#pragma unroll
        for (int i = 0; i < NU; ++i)
#pragma unroll
            for (int q = 0; q < CW; ++q) A[i][q] = T(0);
        for (int f = 0; f < F; ++f) {
            mbar_wait(full + st, ph);
            const T* srow = my + (size_t)st * pl.stage_elems;
            static_for<0, RPS>([&](auto ic) {
                constexpr int i = decltype(ic)::value;
                T seg[SEGP];
                ts_load_seg<T, CW, SEGP>(seg, srow + i * pl.boxw);
                T out[CW];
                ts_row_step<T, U, G, NU, CW, SEGP, (i % NU)>(A, tap, seg, a, out);
                const int Rr = pl.row0 + f * RPS + i - (UPAD - 1);  // finished output row of the last tap-row group
                if (writer && Rr >= oa && Rr < oa + N) {
                    T* o = outp + (size_t)Rr * Gm.Wp;
                    if constexpr (sizeof(T) == 8) {
#pragma unroll
                        for (int q = 0; q < CW; q += 2) { double2 v; v.x = out[q]; v.y = out[q + 1]; *reinterpret_cast<double2*>(o + q) = v; }
                    } else {
#pragma unroll
                        for (int q = 0; q < CW; q += 2) { float2 v; v.x = out[q]; v.y = out[q + 1]; *reinterpret_cast<float2*>(o + q) = v; }
                    }
                }
            });
            __syncwarp();
            if (lane == 0) mbar_arrive(empty + st);
            if (++st == S) { st = 0; ph ^= 1u; }
        }
    }
}

}  // namespace gl
