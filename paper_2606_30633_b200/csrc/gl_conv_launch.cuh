// gl_conv_launch.cuh -- geometry of the padded buffers and launch selection for step D / its transpose:
// input-stationary sliding kernels for the tap counts of the BASELINE.json configs (U = 6, 11, 16 with s*s a
// multiple of 4), generic kernels for every other shape.
#pragma once
#include "gl_common.cuh"
#include "gl_conv.cuh"

namespace gl {

#ifndef GL_CONV_CTA
#define GL_CONV_CTA 128
#endif

struct ConvPlan {
    int kind;                 // 0 generic, 1: U=6 CW=4, 2: U=11 CW=2, 3: U=16 CW=2
    int CW;                   // output columns per thread
    SlidePlan fwd, bwd;
    size_t fwd_smem, bwd_smem;
    int n_ctile;              // chi^2 partials per particle
};

static inline int round_up(int x, int m) { return (x + m - 1) / m * m; }

// Fill the layout fields of G (UP, Hp, Wp, Hg, Wg, PADg) and choose the kernels.  esize = sizeof(T).
static inline ConvPlan conv_plan(Geom& G, int esize, int n_systems) {
    ConvPlan pl{};
    const int U = G.U, N = G.N, NPH = G.s * G.s;
    pl.kind = 0;
    if ((NPH & 3) == 0) { if (U == 6) pl.kind = 1; else if (U == 11) pl.kind = 2; else if (U == 16) pl.kind = 3; }
    pl.CW = pl.kind == 1 ? 4 : 2;
    const int CW = pl.CW, SEG = (CW + U - 1 + 1) & ~1;
    const int ob_max = (G.s - 1 + G.c) / G.s;                    // largest plane shift
    const int ncg_f = (N + CW - 1) / CW, ncg_b = (N + ob_max + CW - 1) / CW;
    G.UP = U;
    G.Hp = N + U - 1;
    int wp = N + U - 1;
    if (wp < CW * (ncg_f - 1) + SEG) wp = CW * (ncg_f - 1) + SEG;
    if (wp < CW * ncg_b) wp = CW * ncg_b;
    G.Wp = round_up(wp, 4);
    G.PADg = U - 1;
    G.Hg = N + 2 * U;
    int wg = N + 2 * (U - 1);
    if (wg < CW * (ncg_b - 1) + SEG) wg = CW * (ncg_b - 1) + SEG;
    G.Wg = round_up(wg, 4);
    if (pl.kind == 0) {
        pl.n_ctile = (N * N + 255) / 256;
        return pl;
    }
    const int LS = pl.kind == 1 ? 4 : 1;                         // lanes per column group (conv_*_launch must agree)
    int ps = U * ((U + 1) & ~1);
    if (LS > 1) while ((2 * ps) % 32 != 8 && (2 * ps) % 32 != 24) ps += 2;   // 4 consecutive planes -> disjoint bank groups
    const int nt_max = 256;                 // launch bounds of the compiled specialisations
    auto mk = [&](int ncg, int cta_f64) {
        SlidePlan sp{};
        sp.ncg = ncg; sp.tpp = LS > 1 ? round_up(LS * ncg, 32) : ncg; sp.ps = ps; sp.shared_taps = n_systems == 1 ? 1 : 0;
        // particles per CTA: the count (<= 8) that wastes the fewest lanes of a CTA of at most GL_CONV_CTA threads
        sp.ppc = 1; double best = 0;
        for (int k = 1; k <= 8; ++k) {
            const int nt = round_up(k * sp.tpp, 32);
            if (nt > (LS > 1 ? GL_CONV_CTA : (esize == 8 ? cta_f64 : 256)) && k > 1) break;   // LS = 1: the fullest CTA the registers allow
            const double eff = (double)(k * LS * ncg) / nt;
            if (eff > best + 1e-9) { best = eff; sp.ppc = k; }
        }
        return sp;
    };
#ifndef GL_CONV_CTA_BWD64
#define GL_CONV_CTA_BWD64 160
#endif
    pl.fwd = mk(ncg_f, GL_CONV_CTA); pl.bwd = mk(ncg_b, GL_CONV_CTA_BWD64);   // fp64: 220 / 168 registers per thread at U = 16
    pl.fwd_smem = (size_t)esize * (pl.fwd.shared_taps ? 1 : pl.fwd.ppc) * NPH * ps;
    pl.bwd_smem = (size_t)esize * (pl.bwd.shared_taps ? 1 : pl.bwd.ppc) * NPH * ps;
    pl.n_ctile = 1;
    if (round_up(pl.fwd.tpp, 32) > nt_max || round_up(pl.bwd.tpp, 32) > nt_max || pl.fwd_smem > 200 * 1024 || pl.bwd_smem > 200 * 1024) {
        pl.kind = 0; pl.n_ctile = (N * N + 255) / 256;
    }
    return pl;
}

template <class T, int U, int CW, int LS, int NT_MAX>
static inline cudaError_t conv_fwd_is_launch(const ConvPlan& pl, const Geom& G, const T* ray, const T* sys_kt,
                                             const T* sys_w, const float* obs, const int32_t* system_id, int64_t p_base,
                                             int64_t Pc, T* gpix, T* chi, float* out_model, cudaStream_t st) {
    auto kern = gl_conv_fwd_is<T, U, CW, LS, NT_MAX>;
    if (pl.fwd_smem > 40 * 1024) {
        cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)pl.fwd_smem);
        if (e != cudaSuccess) return e;
    }
    const unsigned grid = (unsigned)((Pc + pl.fwd.ppc - 1) / pl.fwd.ppc);
    kern<<<grid, round_up(pl.fwd.ppc * pl.fwd.tpp, 32), pl.fwd_smem, st>>>(G, pl.fwd, Pc, ray, sys_kt, sys_w, obs, system_id, p_base, gpix,
                                                            chi, out_model);
    return cudaSuccess;
}

template <class T, int U, int CW, int LS, int NT_MAX>
static inline cudaError_t conv_bwd_is_launch(const ConvPlan& pl, const Geom& G, const T* gpix, const T* sys_kt,
                                             const int32_t* system_id, int64_t p_base, int64_t Pc, T* gbar, cudaStream_t st) {
    auto kern = gl_conv_bwd_is<T, U, CW, LS, NT_MAX>;
    if (pl.bwd_smem > 40 * 1024) {
        cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)pl.bwd_smem);
        if (e != cudaSuccess) return e;
    }
    const unsigned grid = (unsigned)((Pc + pl.bwd.ppc - 1) / pl.bwd.ppc);
    kern<<<grid, round_up(pl.bwd.ppc * pl.bwd.tpp, 32), pl.bwd_smem, st>>>(G, pl.bwd, Pc, gpix, sys_kt, system_id, p_base, gbar);
    return cudaSuccess;
}

template <class T, int U, int CW, int NT_MAX>
static inline cudaError_t conv_fwd_is2_launch(const ConvPlan& pl, const Geom& G, const T* ray, const T* sys_kt,
                                              const T* sys_w, const float* obs, const int32_t* system_id, int64_t p_base,
                                              int64_t Pc, T* gpix, T* chi, float* out_model, cudaStream_t st) {
    auto kern = gl_conv_fwd_is2<T, U, CW, NT_MAX>;
    if (pl.fwd_smem > 40 * 1024) {
        cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)pl.fwd_smem);
        if (e != cudaSuccess) return e;
    }
    const unsigned grid = (unsigned)((Pc + pl.fwd.ppc - 1) / pl.fwd.ppc);
    kern<<<grid, round_up(pl.fwd.ppc * pl.fwd.tpp, 32), pl.fwd_smem, st>>>(G, pl.fwd, Pc, ray, sys_kt, sys_w, obs, system_id, p_base,
                                                                          gpix, chi, out_model);
    return cudaSuccess;
}

template <class T, int U, int CW, int NT_MAX>
static inline cudaError_t conv_bwd_is2_launch(const ConvPlan& pl, const Geom& G, const T* gpix, const T* sys_kt,
                                              const int32_t* system_id, int64_t p_base, int64_t Pc, T* gbar, cudaStream_t st) {
    auto kern = gl_conv_bwd_is2<T, U, CW, NT_MAX>;
    if (pl.bwd_smem > 40 * 1024) {
        cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)pl.bwd_smem);
        if (e != cudaSuccess) return e;
    }
    const unsigned grid = (unsigned)((Pc + pl.bwd.ppc - 1) / pl.bwd.ppc);
    kern<<<grid, round_up(pl.bwd.ppc * pl.bwd.tpp, 32), pl.bwd_smem, st>>>(G, pl.bwd, Pc, gpix, sys_kt, system_id, p_base, gbar);
    return cudaSuccess;
}

// Step D + E.  Returns the number of kernels launched (negative on a CUDA error).
template <class T>
static inline int conv_fwd_launch(const ConvPlan& pl, const Geom& G, const T* ray, const T* sys_kt, const T* sys_w,
                                  const float* obs, const int32_t* system_id, int64_t p_base, int64_t Pc,
                                  T* gpix, T* chi, float* out_model, cudaStream_t st) {
    cudaError_t e = cudaSuccess;
    switch (pl.kind) {
        case 1: e = conv_fwd_is_launch<T, 6, 4, 4, 256>(pl, G, ray, sys_kt, sys_w, obs, system_id, p_base, Pc, gpix, chi, out_model, st); break;
        case 2: e = conv_fwd_is2_launch<T, 11, 2, 256>(pl, G, ray, sys_kt, sys_w, obs, system_id, p_base, Pc, gpix, chi, out_model, st); break;
        case 3: e = conv_fwd_is2_launch<T, 16, 2, 256>(pl, G, ray, sys_kt, sys_w, obs, system_id, p_base, Pc, gpix, chi, out_model, st); break;
        default: {
            dim3 grid((G.N * G.N + 255) / 256, (unsigned)Pc);
            gl_conv_fwd_generic<T><<<grid, 256, 0, st>>>(G, ray, sys_kt, sys_w, obs, system_id, p_base, gpix, chi, out_model);
        }
    }
    return e == cudaSuccess ? 1 : -1;
}

// Transpose of step D: gbar_ray overwrites the ray buffer.
template <class T>
static inline int conv_bwd_launch(const ConvPlan& pl, const Geom& G, const T* gpix, const T* sys_kt,
                                  const int32_t* system_id, int64_t p_base, int64_t Pc, T* gbar, cudaStream_t st) {
    cudaError_t e = cudaSuccess;
    switch (pl.kind) {
        case 1: e = conv_bwd_is_launch<T, 6, 4, 4, 256>(pl, G, gpix, sys_kt, system_id, p_base, Pc, gbar, st); break;
        case 2: e = conv_bwd_is2_launch<T, 11, 2, 256>(pl, G, gpix, sys_kt, system_id, p_base, Pc, gbar, st); break;
        case 3: e = conv_bwd_is2_launch<T, 16, 2, 256>(pl, G, gpix, sys_kt, system_id, p_base, Pc, gbar, st); break;
        default: {
            dim3 grid((G.s * G.s * G.N * G.N + 255) / 256, (unsigned)Pc);
            gl_conv_bwd_generic<T><<<grid, 256, 0, st>>>(G, gpix, sys_kt, system_id, p_base, gbar);
        }
    }
    return e == cudaSuccess ? 1 : -1;
}

}  // namespace gl
