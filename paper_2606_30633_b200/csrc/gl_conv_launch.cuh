// gl_conv_launch.cuh -- geometry of the padded buffers and launch selection for step D / its transpose:
// sliding-window specialisations for the tap counts of the BASELINE.json configs (U = 6, 11, 16), generic kernels
// for every other shape.  The tap rows per thread (UR) differ between the fp32 and the fp64 mode because a double
// takes two registers.
#pragma once
#include "gl_common.cuh"
#include "gl_conv.cuh"

namespace gl {

struct ConvPlan {
    int kind;                 // 0 generic, else index of the (UR, U) specialisation
    int UR;                   // tap rows per thread
    int nvp;                  // threads per column group: s*s*ceil(U/UR)
    int fwd_ncgb, fwd_nband, fwd_nt; size_t fwd_smem;
    int bwd_ncgb, bwd_nband, bwd_nt; size_t bwd_smem;
    int n_ctile;              // chi^2 partials per particle
};

// (UR, U, max threads per CTA) of the compiled specialisations: [0] fp32, [1] fp64
constexpr int CONV_SPEC[2][3][3] = {{{6, 6, 512}, {4, 11, 384}, {4, 16, 256}},
                                    {{3, 6, 512}, {2, 11, 384}, {2, 16, 256}}};

static inline int round_up(int x, int m) { return (x + m - 1) / m * m; }

// Fill the layout fields of G (UP, Hp, Wp, Hg, Wg, PADg) and choose the kernels.  esize = sizeof(T).
static inline ConvPlan conv_plan(Geom& G, int esize) {
    ConvPlan pl{};
    const int U = G.U, tsel = esize == 8 ? 1 : 0;
    int max_nt = 256;
    pl.kind = 0; pl.UR = U;
    for (int k = 0; k < 3; ++k)
        if (CONV_SPEC[tsel][k][1] == U) { pl.kind = k + 1; pl.UR = CONV_SPEC[tsel][k][0]; max_nt = CONV_SPEC[tsel][k][2]; }
    const int nrg = (U + pl.UR - 1) / pl.UR;
    const int WL = 4 * ((U + 3 + 3) / 4);
    const int NCG = (G.N + 3) / 4, NCGp = (G.N + U - 1 + 3) / 4;
    G.UP = nrg * pl.UR;
    G.Hp = G.N + G.UP - 1;
    G.Wp = 4 * (NCG - 1) + WL; if (G.Wp < 4 * NCGp) G.Wp = 4 * NCGp;
    G.PADg = U - 1;
    G.Hg = G.N + U + G.UP;
    G.Wg = 4 * (NCGp - 1) + WL;
    pl.nvp = G.s * G.s * nrg;
    if (pl.kind == 0) {
        pl.n_ctile = (G.N * G.N + 255) / 256;
        return pl;
    }
    auto split = [&](int ncg, int& ncgb, int& nband, int& nt) {
        int cap = max_nt / pl.nvp; if (cap < 1) cap = 1;
        nband = (ncg + cap - 1) / cap;
        ncgb = (ncg + nband - 1) / nband;
        nt = round_up(ncgb * pl.nvp, 32);
    };
    split(NCG, pl.fwd_ncgb, pl.fwd_nband, pl.fwd_nt);
    split(NCGp, pl.bwd_ncgb, pl.bwd_nband, pl.bwd_nt);
    pl.fwd_smem = (size_t)esize * 2 * (size_t)pl.nvp * CONV_R * 4 * pl.fwd_ncgb;
    pl.bwd_smem = nrg > 1 ? (size_t)esize * 2 * (size_t)pl.nvp * CONV_R * 4 * pl.bwd_ncgb : 0;
    pl.n_ctile = pl.fwd_nband;
    if (pl.fwd_nt > max_nt || pl.bwd_nt > max_nt || pl.fwd_smem > 200 * 1024 || pl.bwd_smem > 200 * 1024) {
        pl.kind = 0; pl.n_ctile = (G.N * G.N + 255) / 256;      // s*s*ceil(U/UR) threads do not fit one CTA: generic path
    }
    return pl;
}

template <class T, int UR, int U, int NT>
static inline cudaError_t conv_fwd_sw_launch(const ConvPlan& pl, const Geom& G, const T* ray, const T* sys_kt,
                                             const T* sys_w, const float* obs, const int32_t* system_id, int64_t p_base,
                                             int64_t Pc, T* gpix, T* chi, float* out_model, cudaStream_t st) {
    auto kern = gl_conv_fwd_sw<T, UR, U, NT>;
    if (pl.fwd_smem > 32 * 1024) {
        cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)pl.fwd_smem);
        if (e != cudaSuccess) return e;
    }
    kern<<<dim3(pl.fwd_nband, (unsigned)Pc), pl.fwd_nt, pl.fwd_smem, st>>>(G, pl.fwd_ncgb, ray, sys_kt, sys_w, obs, system_id,
                                                                          p_base, gpix, chi, out_model);
    return cudaSuccess;
}

template <class T, int UR, int U, int NT>
static inline cudaError_t conv_bwd_sw_launch(const ConvPlan& pl, const Geom& G, const T* gpix, const T* sys_kt,
                                             const int32_t* system_id, int64_t p_base, int64_t Pc, T* gbar, cudaStream_t st) {
    auto kern = gl_conv_bwd_sw<T, UR, U, NT>;
    if (pl.bwd_smem > 32 * 1024) {
        cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)pl.bwd_smem);
        if (e != cudaSuccess) return e;
    }
    kern<<<dim3(pl.bwd_nband, (unsigned)Pc), pl.bwd_nt, pl.bwd_smem, st>>>(G, pl.bwd_ncgb, gpix, sys_kt, system_id, p_base, gbar);
    return cudaSuccess;
}

template <class T> struct ConvSpec;
template <> struct ConvSpec<float>  { static constexpr int UR0 = 6, UR1 = 4, UR2 = 4; };
template <> struct ConvSpec<double> { static constexpr int UR0 = 3, UR1 = 2, UR2 = 2; };

// Step D + E.  Returns the number of kernels launched (negative on a CUDA error).
template <class T>
static inline int conv_fwd_launch(const ConvPlan& pl, const Geom& G, const T* ray, const T* sys_kt, const T* sys_w,
                                  const float* obs, const int32_t* system_id, int64_t p_base, int64_t Pc,
                                  T* gpix, T* chi, float* out_model, cudaStream_t st) {
    using S = ConvSpec<T>;
    cudaError_t e = cudaSuccess;
    switch (pl.kind) {
        case 1: e = conv_fwd_sw_launch<T, S::UR0, 6, 512>(pl, G, ray, sys_kt, sys_w, obs, system_id, p_base, Pc, gpix, chi, out_model, st); break;
        case 2: e = conv_fwd_sw_launch<T, S::UR1, 11, 384>(pl, G, ray, sys_kt, sys_w, obs, system_id, p_base, Pc, gpix, chi, out_model, st); break;
        case 3: e = conv_fwd_sw_launch<T, S::UR2, 16, 256>(pl, G, ray, sys_kt, sys_w, obs, system_id, p_base, Pc, gpix, chi, out_model, st); break;
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
    using S = ConvSpec<T>;
    cudaError_t e = cudaSuccess;
    switch (pl.kind) {
        case 1: e = conv_bwd_sw_launch<T, S::UR0, 6, 512>(pl, G, gpix, sys_kt, system_id, p_base, Pc, gbar, st); break;
        case 2: e = conv_bwd_sw_launch<T, S::UR1, 11, 384>(pl, G, gpix, sys_kt, system_id, p_base, Pc, gbar, st); break;
        case 3: e = conv_bwd_sw_launch<T, S::UR2, 16, 256>(pl, G, gpix, sys_kt, system_id, p_base, Pc, gbar, st); break;
        default: {
            dim3 grid((G.s * G.s * G.N * G.N + 255) / 256, (unsigned)Pc);
            gl_conv_bwd_generic<T><<<grid, 256, 0, st>>>(G, gpix, sys_kt, system_id, p_base, gbar);
        }
    }
    return e == cudaSuccess ? 1 : -1;
}

}  // namespace gl
