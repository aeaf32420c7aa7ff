// gl_conv_launch.cuh -- geometry of the padded buffers and launch selection for step D / its transpose:
// input-stationary sliding kernels for the tap counts of the BASELINE.json configs (U = 6, 11, 16 with s*s a
// multiple of 4), generic kernels for every other shape.
#pragma once
#include <algorithm>
#include <cmath>
#include <cstdlib>
#include "gl_common.cuh"
#include "gl_conv.cuh"
#include "gl_conv_ts.cuh"
#include "gl_conv_ct.cuh"

namespace gl {

#ifndef GL_CONV_CTA
#define GL_CONV_CTA 128
#endif

static inline int round_up(int x, int m) { return (x + m - 1) / m * m; }

struct ConvPlan {
    int kind;                 // 6: uniform taps (single system; gl_conv_ct.cuh); 7: the same on the binned plane of psf_grid 1; 0 generic, 1: U=6 CW=4, 2: U=11 CW=2, 3: U=16 CW=2 (round-1 sliding kernels), 4: tap-stationary + TMA,
                              // 5: psf_grid 1 dedicated: bin the planes, then tap-stationary on ONE plane with the K x K taps
    int CW;                   // output columns per thread
    SlidePlan fwd, bwd;
    size_t fwd_smem, bwd_smem;
    int n_ctile;              // chi^2 partials per particle
    int ts_id;                // kind 4: which (U, G, NPH, CW) instance (ts_variant)
    TsPlan tf, tb;            // kind 4: forward / transpose launch plans
    int ct_slot;              // kind 6 (uniform taps from constant memory, gl_conv_ct.cuh): slot of c_ctap
    CtPlan cf, cb;            // kind 6: forward / transpose launch plans
};

// Uniform-tap instances: output columns per thread for each compiled tap count
#ifndef GL_CT_CW6
#define GL_CT_CW6 4
#endif
#ifndef GL_CT_CW11
#define GL_CT_CW11 4
#endif
#ifndef GL_CT_CW16
#define GL_CT_CW16 2
#endif
#ifndef GL_CT_BAND_ROWS
#define GL_CT_BAND_ROWS 25
#endif
#ifndef GL_CT_TARGET_CTAS
#define GL_CT_TARGET_CTAS 1776.0      // 6 waves of 148 SMs x 2 resident CTAs
#endif
#ifndef GL_CT_CW16B
#define GL_CT_CW16B 4
#endif
// U = 6 (36 taps per plane) stays on the tap-stationary kernels: measured on config 2, 0.96 / 1.00 ms here against 0.95 / 0.71 ms
// there (too few FMAs per row step to amortise the row bookkeeping); GL_CT_U6=1 compiles the instance in for A/B runs.
#ifndef GL_CT_U6
#define GL_CT_U6 0
#endif
// U = 5, 7, 21 occur on the dedicated psf_grid = 1 path only (one binned plane, U = K taps per side)
static inline int ct_cw(int U) {                                                                                       // forward
    return (U == 6 && GL_CT_U6) ? GL_CT_CW6 : (U == 11 ? GL_CT_CW11 : (U == 16 ? GL_CT_CW16 : (U == 5 || U == 7 ? 4 : (U == 21 ? 2 : 0))));
}
static inline int ct_cwb(int U) { return U == 16 ? GL_CT_CW16B : ct_cw(U); }                                            // transpose
static inline bool ct_fits(int U, int NPH) { return ct_cw(U) > 0 && NPH * U * ((U + 1) & ~1) <= CT_SLOT; }

// The compiled tap-stationary instances: id -> (U, G, NPH, CW).  G tap-row groups x NPH planes = lanes per column group.
#ifndef GL_TS_CW11
#define GL_TS_CW11 4
#endif
#ifndef GL_TS_CW16
#define GL_TS_CW16 4
#endif
struct TsVariant { int U, G, NPH, CW, RPS, wmax_f, wmax_b, maxt; };   // wmax: consumer warps per CTA, forward / transpose
#ifndef GL_TS_RPS6
#define GL_TS_RPS6 6
#endif
#ifndef GL_TS_RPS11
#define GL_TS_RPS11 6
#endif
#ifndef GL_TS_RPS16
#define GL_TS_RPS16 8
#endif
#ifndef GL_TS_W6
#define GL_TS_W6 8, 8
#endif
#ifndef GL_TS_W11
#define GL_TS_W11 7, 4
#endif
#ifndef GL_TS_W16
#define GL_TS_W16 4, 4
#endif
#ifndef GL_TS_W1
#define GL_TS_W1 4, 4
#endif
// single-plane instances of the dedicated psf_grid = 1 path: (U = K, G, NPH = 1)
static constexpr TsVariant k_ts1_variants[] = {{5, 1, 1, 4, 5, GL_TS_W1, 256}, {7, 1, 1, 4, 7, GL_TS_W1, 256}, {11, 2, 1, 4, 6, GL_TS_W1, 256},
                                               {21, 8, 1, 4, 6, GL_TS_W1, 256}};     // K is odd; other K: box-expanded path
static inline int ts1_variant(int U) {
    for (int i = 0; i < (int)(sizeof(k_ts1_variants) / sizeof(k_ts1_variants[0])); ++i)
        if (k_ts1_variants[i].U == U) return i;
    return -1;
}
static constexpr TsVariant k_ts_variants[] = {{6, 1, 4, 4, GL_TS_RPS6, GL_TS_W6, GL_TS_MAXT6}, {6, 1, 16, 4, GL_TS_RPS6, GL_TS_W6, GL_TS_MAXT6},
                                              {11, 2, 4, GL_TS_CW11, GL_TS_RPS11, GL_TS_W11, GL_TS_MAXT11},
                                              {11, 2, 16, GL_TS_CW11, GL_TS_RPS11, GL_TS_W11, GL_TS_MAXT11},
                                              {16, 8, 4, GL_TS_CW16, GL_TS_RPS16, GL_TS_W16, GL_TS_MAXT16}};
static inline int ts_variant(int U, int NPH) {
    for (int i = 0; i < (int)(sizeof(k_ts_variants) / sizeof(k_ts_variants[0])); ++i)
        if (k_ts_variants[i].U == U && k_ts_variants[i].NPH == NPH) return i;
    return -1;
}
#ifndef GL_TS_STAGES
#define GL_TS_STAGES 3
#endif
// Launch plan of one direction.  ncols: output columns to cover; planes_in_box: NPH (forward) or 1 (transpose);
// pitch_rule: forward rows of different planes sit boxw apart -> boxw * esize = 16 (mod 32) keeps a quarter-warp's
// 16-byte loads on distinct banks.
static inline TsPlan ts_plan(const TsVariant& v, int wmax_default, int esize, int ncols, int planes_in_box, int steps, int row0, bool fwd) {
    TsPlan pl{};
    const int LPG = v.NPH * v.G, CGW = 32 / LPG, NU = (v.U + v.G - 1) / v.G;
    (void)NU;
    const int ve = ((v.CW * esize) % 16 == 0 ? 16 : 8) / esize;
    const int segp = (v.CW + v.U - 1 + ve - 1) / ve * ve;
    pl.ncg = (ncols + v.CW - 1) / v.CW;
    const int warps = (pl.ncg + CGW - 1) / CGW;
    int wmax = wmax_default, nst = GL_TS_STAGES;
    if (const char* e = std::getenv("GL_TS_WMAX")) { const int k = std::atoi(e); if (k >= 1) wmax = k; }   // tuning overrides
    if (const char* e = std::getenv("GL_TS_STAGES")) { const int k = std::atoi(e); if (k >= 2 && k <= 16) nst = k; }
    if (wmax > v.maxt / 32 - 1) wmax = v.maxt / 32 - 1;
    pl.n_bands = (warps + wmax - 1) / wmax;
    pl.wpc = (warps + pl.n_bands - 1) / pl.n_bands;
    // TMA: the first column of a band must sit on a 16-byte boundary
    while (pl.n_bands > 1 && (v.CW * pl.wpc * CGW * esize) % 16 != 0) ++pl.wpc;
    pl.n_bands = (warps + pl.wpc - 1) / pl.wpc;
    pl.cg_per_cta = pl.wpc * CGW;
    int bw = v.CW * (pl.cg_per_cta - 1) + segp;
    const int q = 16 / esize;                                   // TMA: box row a multiple of 16 bytes
    bw = round_up(bw, q);
    if (planes_in_box > 1) while ((bw * esize) % 32 != 16) bw += q;
    pl.boxw = bw;
    pl.stage_elems = round_up(bw * planes_in_box * v.RPS, 128 / esize);
    pl.stages = nst;
    pl.steps = steps; pl.row0 = row0;
    pl.pbuf_elems = fwd ? ts_pbuf_elems(v.NPH, v.G, v.CW, v.RPS) : 0;
    return pl;
}

// Fill the layout fields of G (UP, Hp, Wp, Hg, Wg, PADg) and choose the kernels.  esize = sizeof(T).
// What conv_plan may know about the batch: the workspace budget of a chunk and how many ray-image-sized buffers a particle
// keeps (1, or 3 with the (u, v) buffer); budget 0 = plenty of particles per launch (backward modelling: n_amp virtual particles each).
struct ConvChunkHint { size_t budget; int ray_bufs; };
static inline ConvPlan conv_plan(Geom& G, int esize, int n_systems, int ct_slot = -1, ConvChunkHint hint = ConvChunkHint{0, 1}) {
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
    G.binned = 0;
    pl.ct_slot = -1;
    // uniform taps (gl_conv_ct.cuh): one system, a free constant slot, a compiled tap count; GL_CONV_CT=0: off (A/B runs).
    // planes = s*s, or 1 on the dedicated psf_grid = 1 path (kind 7: the binned image in plane 0)
    auto try_ct = [&](int planes, int kind) -> bool {
        const char* e = std::getenv("GL_CONV_CT");
        if (ct_slot >= 0 && n_systems == 1 && ct_fits(U, planes) && !(e && e[0] == '0')) {
            const int cw = ct_cw(U), seg = (cw + U - 1 + 1) & ~1, cwb = ct_cwb(U), segb = (cwb + U - 1 + 1) & ~1;
            const int nf = (N + cw - 1) / cw, nb = (N + ob_max + cwb - 1) / cwb;
            int wp2 = G.Wp, wg2 = G.Wg;
            if (wp2 < cw * (nf - 1) + seg) wp2 = cw * (nf - 1) + seg;
            if (wp2 < cwb * nb) wp2 = cwb * nb;
            if (wg2 < cwb * (nb - 1) + segb) wg2 = cwb * (nb - 1) + segb;
            G.Wp = round_up(wp2, 4); G.Wg = round_up(wg2, 4);
            auto mkc = [&](int ncg) {
                CtPlan cp{};
                cp.ncg = ncg;
                // Row bands of the forward kernel: enough CTAs per launch to fill the machine several times over when a FULL chunk
                // is processed (config 5: 410-487 particles x 50 column groups = 190 CTAs per band against 296 resident: 1 band ran
                // 20.7 ms, 4 bands 14.2, 8 bands 13.6), but no thinner than GL_CT_BAND_ROWS rows (halo rows and partial tap groups
                // are redone per band).  A function of the configuration only: the chi^2 partials, hence the bit-identity of a
                // particle's result across batch sizes, depend on it.
                const size_t per_particle = (size_t)esize * ((size_t)hint.ray_bufs * G.s * G.s * G.Hp * G.Wp + (size_t)G.Hg * G.Wg);
                const double pc_full = hint.budget ? (double)hint.budget / (double)per_particle : 1e9;
                const double ctas_per_band = pc_full * ncg / CT_NT;
                int nb = (int)std::ceil(GL_CT_TARGET_CTAS / ctas_per_band);
                const int nb_max = N / GL_CT_BAND_ROWS < 1 ? 1 : N / GL_CT_BAND_ROWS;
                cp.n_bands = nb < 1 ? 1 : (nb > nb_max ? nb_max : nb);
                cp.rbh = (N + cp.n_bands - 1) / cp.n_bands;
                cp.n_bands = (N + cp.rbh - 1) / cp.rbh;
                return cp;
            };
            pl.cf = mkc(nf); pl.cb = mkc(nb);
            pl.kind = kind; pl.CW = cw; pl.ct_slot = ct_slot; pl.n_ctile = pl.cf.n_bands * pl.cf.ncg;
            return true;
        }
        return false;
    };
    {   // psf_grid 1: the dedicated bin-then-convolve path wherever a single-plane instance exists (GL_CONV_BIN=0: box-expanded)
        const char* e = std::getenv("GL_CONV_BIN");
        const int id = G.pgrid == 1 ? ts1_variant(U) : -1;
        if (id >= 0 && !(e && e[0] == '0')) {
            if (try_ct(1, 7)) { G.binned = 1; return pl; }      // uniform taps on the single binned plane
            const TsVariant& v = k_ts1_variants[id];
            const int NU = (v.U + v.G - 1) / v.G, UPAD = NU * v.G, o = G.c / G.s;     // every plane has the shift o = (K - 1) / 2
            TsPlan tf = ts_plan(v, v.wmax_f, esize, N, 1, N + UPAD - 1, 0, true);
            TsPlan tb = ts_plan(v, v.wmax_b, esize, N + o, 1, N + UPAD - 1, o, false);
            if (tf.boxw <= 256 && tb.boxw <= 256 && v.CW * tb.ncg <= G.Wp) {
                pl.kind = 5; pl.ts_id = id; pl.CW = v.CW; pl.tf = tf; pl.tb = tb; pl.n_ctile = tf.n_bands * tf.wpc;
                G.binned = 1;
                return pl;
            }
        }
    }
    if (pl.kind == 0) {
        pl.n_ctile = (N * N + 255) / 256;
        return pl;
    }
    if (try_ct(NPH, 6)) return pl;
    const int LS = pl.kind == 1 ? 4 : 1;                         // lanes per column group (conv_*_launch must agree)
    int ps = U * ((U + 1) & ~1);
    if (LS > 1) while ((2 * ps) % 32 != 8 && (2 * ps) % 32 != 24) ps += 2;   // 4 consecutive planes -> disjoint bank groups
    {   // tap-stationary kernels (gl_conv_ts.cuh) wherever an instance exists; GL_CONV_TS=0 keeps the round-1 kernels (A/B runs)
        const char* e = std::getenv("GL_CONV_TS");
        const int id = ts_variant(U, NPH);
        if (id >= 0 && !(e && e[0] == '0')) {
            const TsVariant& v = k_ts_variants[id];
            const int NU = (v.U + v.G - 1) / v.G, UPAD = NU * v.G;
            const int omin = G.c / G.s, omax = (G.s - 1 + G.c) / G.s;
            TsPlan tf = ts_plan(v, v.wmax_f, esize, N, NPH, N + UPAD - 1, 0, true);
            TsPlan tb = ts_plan(v, v.wmax_b, esize, N + ob_max, 1, N + (omax - omin) + UPAD - 1, omin, false);
            if (tf.boxw <= 256 && tb.boxw <= 256 && (tf.wpc + 1) * 32 <= v.maxt && (tb.wpc + 1) * 32 <= v.maxt &&
                v.CW * tb.ncg <= G.Wp) {
                pl.kind = 4; pl.ts_id = id; pl.CW = v.CW; pl.tf = tf; pl.tb = tb; pl.n_ctile = tf.n_bands * tf.wpc;
                return pl;
            }
        }
    }
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

// ----------------------------------------------------------------------------- tap-stationary launches (kind 4)
// cuTensorMapEncodeTiled through the runtime's driver entry point (no link-time dependency on libcuda).
typedef CUresult (*gl_encode_tiled_fn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                       const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                       CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
static inline gl_encode_tiled_fn gl_encode_tiled() {
    static gl_encode_tiled_fn fn = []() -> gl_encode_tiled_fn {
        void* f = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &f, cudaEnableDefault, &q) != cudaSuccess || q != cudaDriverEntryPointSuccess)
            return nullptr;
        return (gl_encode_tiled_fn)f;
    }();
    return fn;
}
// 3-D tensor {d0, d1, d2} of T at `base`, dim 0 contiguous, dims 1 and 2 with the given element strides; box {b0, b1, b2}; elements outside the tensor read as zero.
template <class T>
static inline bool ts_make_map(CUtensorMap* tm, const void* base, uint64_t d0, uint64_t d1, uint64_t d2, uint64_t stride1, uint64_t stride2,
                               uint32_t b0, uint32_t b1, uint32_t b2) {
    gl_encode_tiled_fn enc = gl_encode_tiled();
    if (!enc) return false;
    const cuuint64_t dims[3] = {d0, d1, d2};
    const cuuint64_t strides[2] = {stride1 * sizeof(T), stride2 * sizeof(T)};      // element strides of dims 1 and 2
    const cuuint32_t box[3] = {b0, b1, b2};
    const cuuint32_t es[3] = {1, 1, 1};
    return enc(tm, sizeof(T) == 8 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT64 : CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, const_cast<void*>(base), dims,
               strides, box, es, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
               CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

// Persistent grid: every SM gets as many CTAs as fit (shared-memory carve-out raised to the maximum, else the driver sizes
// it for ONE block), never more CTAs than work items.
template <class K>
static inline cudaError_t ts_grid(K kern, const TsPlan& pl, size_t smem, int64_t Pc, unsigned* grid) {
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(kern, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared);
    if (e != cudaSuccess) return e;
    int dev = 0, n_sm = 0, occ = 0;
    if ((e = cudaGetDevice(&dev)) != cudaSuccess) return e;
    if ((e = cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev)) != cudaSuccess) return e;
    if ((e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kern, (pl.wpc + 1) * 32, smem)) != cudaSuccess) return e;
    if (occ < 1) return cudaErrorLaunchOutOfResources;
    const int64_t items = Pc * pl.n_bands, cap = (int64_t)n_sm * occ;
    *grid = (unsigned)(items < cap ? items : cap);
    return cudaSuccess;
}

template <class T, int U, int G_, int NPH, int CW, int RPS>
static inline cudaError_t conv_fwd_ts_launch(const ConvPlan& pl, const Geom& G, const T* ray, const T* sys_kt, const T* sys_w,
                                             const float* obs, const int32_t* system_id, int64_t p_base, int64_t Pc, T* gpix,
                                             T* chi, float* out_model, cudaStream_t st, bool prebinned = false) {
    CUtensorMap tm;
    // plane index in the middle: {Wp, NPH * Pc (stride Hp Wp), Hp (stride Wp)} -> a box lands as [RPS][NPH][boxw];
    // binned path (NPH = 1): plane 0 of every particle, one ray_stride apart
    const uint64_t pstride = G.binned ? (uint64_t)ray_stride(G) : (uint64_t)G.Hp * G.Wp;
    if (!ts_make_map<T>(&tm, ray, (uint64_t)G.Wp, (uint64_t)NPH * (uint64_t)Pc, (uint64_t)G.Hp, pstride, (uint64_t)G.Wp,
                        (uint32_t)pl.tf.boxw, NPH, RPS))
        return cudaErrorInvalidValue;
    if (G.binned && !prebinned) gl_bin_planes_kernel<T><<<dim3((unsigned)(((size_t)G.Hp * G.Wp + 255) / 256), (unsigned)Pc), 256, 0, st>>>(G, const_cast<T*>(ray));
    auto kern = gl_conv_fwd_ts<T, U, G_, NPH, CW, RPS>;
    const size_t smem = ts_smem_bytes<T>(pl.tf);
    unsigned grid = 0;
    cudaError_t e = ts_grid(kern, pl.tf, smem, Pc, &grid);
    if (e != cudaSuccess) return e;
    kern<<<grid, (pl.tf.wpc + 1) * 32, smem, st>>>(tm, G, pl.tf, Pc, sys_kt, sys_w, obs, system_id, p_base, gpix, chi, out_model);
    return cudaSuccess;
}
template <class T, int U, int G_, int NPH, int CW, int RPS>
static inline cudaError_t conv_bwd_ts_launch(const ConvPlan& pl, const Geom& G, const T* gpix, const T* sys_kt,
                                             const int32_t* system_id, int64_t p_base, int64_t Pc, T* gbar, cudaStream_t st) {
    CUtensorMap tm;
    if (!ts_make_map<T>(&tm, gpix, (uint64_t)G.Wg, (uint64_t)G.Hg, (uint64_t)Pc, (uint64_t)G.Wg, (uint64_t)G.Hg * G.Wg, (uint32_t)pl.tb.boxw,
                        RPS, 1))
        return cudaErrorInvalidValue;
    auto kern = gl_conv_bwd_ts<T, U, G_, NPH, CW, RPS>;
    const size_t smem = ts_smem_bytes<T>(pl.tb);
    unsigned grid = 0;
    cudaError_t e = ts_grid(kern, pl.tb, smem, Pc, &grid);
    if (e != cudaSuccess) return e;
    kern<<<grid, (pl.tb.wpc + 1) * 32, smem, st>>>(tm, G, pl.tb, Pc, sys_kt, system_id, p_base, gbar);
    return cudaSuccess;
}
// ----------------------------------------------------------------------------- uniform-tap launches (kind 6)
template <class T, int U, int CW>
static inline cudaError_t conv_fwd_ct_launch(const ConvPlan& pl, const Geom& G, const T* ray, const T* sys_w, const float* obs,
                                             int64_t p_base, int64_t Pc, T* gpix, T* chi, float* out_model, cudaStream_t st) {
    const dim3 grid((unsigned)((Pc * pl.cf.ncg + CT_NT - 1) / CT_NT), (unsigned)pl.cf.n_bands);
    gl_conv_fwd_ct<T, U, CW><<<grid, CT_NT, 0, st>>>(G, pl.cf, pl.ct_slot, Pc, ray, sys_w, obs, p_base, gpix, chi, out_model);
    return cudaSuccess;
}
template <class T, int U, int CW>
static inline cudaError_t conv_bwd_ct_launch(const ConvPlan& pl, const Geom& G, const T* gpix, int64_t Pc, T* gbar, cudaStream_t st) {
    // grid.y carries the items (the plane is the fastest index, gl_conv_ct.cuh): at most 65535 CTAs per launch -> slices of particles
    const int64_t p_slice = std::max<int64_t>(1, (int64_t)65535 * CT_NT / pl.cb.ncg);
    for (int64_t p0 = 0; p0 < Pc; p0 += p_slice) {
        const int64_t n = std::min<int64_t>(p_slice, Pc - p0);
        const dim3 grid((unsigned)(G.binned ? 1 : G.s * G.s), (unsigned)((n * pl.cb.ncg + CT_NT - 1) / CT_NT));   // binned: plane 0 only
        gl_conv_bwd_ct<T, U, CW><<<grid, CT_NT, 0, st>>>(G, pl.cb, pl.ct_slot, n, gpix + (size_t)p0 * gpix_stride(G), gbar + (size_t)p0 * ray_stride(G));
    }
    return cudaSuccess;
}
// Refill the constant slot from the taps gl_prep_kernel wrote (system 0): plane-ordered table into `stage`, then a
// device-to-device copy into c_ctap on the same stream.  Returns the number of kernels launched, negative on error.
template <class T>
static inline int conv_ct_upload(const ConvPlan& pl, const Geom& G, const T* sys_kt, T* stage, cudaStream_t st) {
    const int nph = G.binned ? 1 : G.s * G.s;            // binned (psf_grid 1): every plane has the same taps, plane 0 is the image
    const int n = nph * G.U * ((G.U + 1) & ~1);
    gl_ctap_stage_kernel<T><<<(n + 255) / 256, 256, 0, st>>>(G, nph, sys_kt, stage);
    if (cudaMemcpyToSymbolAsync(c_ctap, stage, (size_t)n * sizeof(T), (size_t)pl.ct_slot * CT_SLOT * sizeof(double),
                                cudaMemcpyDeviceToDevice, st) != cudaSuccess)
        return -1;
    return 1;
}

#define GL_TS_DISPATCH(CALL)                                                                                       \
    switch (pl.ts_id) {                                                                                            \
        case 0: e = CALL(6, 1, 4, 4, GL_TS_RPS6); break;                                                           \
        case 1: e = CALL(6, 1, 16, 4, GL_TS_RPS6); break;                                                          \
        case 2: e = CALL(11, 2, 4, GL_TS_CW11, GL_TS_RPS11); break;                                                \
        case 3: e = CALL(11, 2, 16, GL_TS_CW11, GL_TS_RPS11); break;                                               \
        default: e = CALL(16, 8, 4, GL_TS_CW16, GL_TS_RPS16); break;                                               \
    }

#define GL_TS1_DISPATCH(CALL)                                                                                      \
    switch (pl.ts_id) {                                                                                            \
        case 0: e = CALL(5, 1, 1, 4, 5); break;                                                                    \
        case 1: e = CALL(7, 1, 1, 4, 7); break;                                                                    \
        case 2: e = CALL(11, 2, 1, 4, 6); break;                                                                   \
        default: e = CALL(21, 8, 1, 4, 6); break;                                                                  \
    }

// Step D + E.  Returns the number of kernels launched (negative on a CUDA error).
template <class T>
static inline int conv_fwd_launch(const ConvPlan& pl, const Geom& G, const T* ray, const T* sys_kt, const T* sys_w,
                                  const float* obs, const int32_t* system_id, int64_t p_base, int64_t Pc,
                                  T* gpix, T* chi, float* out_model, cudaStream_t st, bool prebinned = false) {
    // prebinned (psf_grid 1, dedicated path): plane 0 already holds the binned image (gl_ray_fwd_binned_kernel): no bin pass
    cudaError_t e = cudaSuccess;
    switch (pl.kind) {
        case 1: e = conv_fwd_is_launch<T, 6, 4, 4, 256>(pl, G, ray, sys_kt, sys_w, obs, system_id, p_base, Pc, gpix, chi, out_model, st); break;
        case 2: e = conv_fwd_is2_launch<T, 11, 2, 256>(pl, G, ray, sys_kt, sys_w, obs, system_id, p_base, Pc, gpix, chi, out_model, st); break;
        case 3: e = conv_fwd_is2_launch<T, 16, 2, 256>(pl, G, ray, sys_kt, sys_w, obs, system_id, p_base, Pc, gpix, chi, out_model, st); break;
        case 4: {
#define GL_TS_F(U_, G__, NPH_, CW_, RPS_) conv_fwd_ts_launch<T, U_, G__, NPH_, CW_, RPS_>(pl, G, ray, sys_kt, sys_w, obs, system_id, p_base, Pc, gpix, chi, out_model, st, prebinned)
            GL_TS_DISPATCH(GL_TS_F)
            break;
        }
        case 5: {
            GL_TS1_DISPATCH(GL_TS_F)
#undef GL_TS_F
            return e == cudaSuccess ? (prebinned ? 1 : 2) : -1;          // (bin +) step D
        }
        case 7:
            if (!prebinned) gl_bin_planes_kernel<T><<<dim3((unsigned)(((size_t)G.Hp * G.Wp + 255) / 256), (unsigned)Pc), 256, 0, st>>>(G, const_cast<T*>(ray));
            [[fallthrough]];
        case 6:
#define GL_CT_F(U_, CW_) conv_fwd_ct_launch<T, U_, CW_>(pl, G, ray, sys_w, obs, p_base, Pc, gpix, chi, out_model, st)
            switch (G.U) {
                case 5: e = GL_CT_F(5, 4); break;
                case 6: e = GL_CT_F(6, GL_CT_CW6); break;
                case 7: e = GL_CT_F(7, 4); break;
                case 11: e = GL_CT_F(11, GL_CT_CW11); break;
                case 16: e = GL_CT_F(16, GL_CT_CW16); break;
                default: e = GL_CT_F(21, 2); break;
            }
#undef GL_CT_F
            if (pl.kind == 7) return e == cudaSuccess ? (prebinned ? 1 : 2) : -1;   // (bin +) step D
            break;
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
        case 4: {
#define GL_TS_B(U_, G__, NPH_, CW_, RPS_) conv_bwd_ts_launch<T, U_, G__, NPH_, CW_, RPS_>(pl, G, gpix, sys_kt, system_id, p_base, Pc, gbar, st)
            GL_TS_DISPATCH(GL_TS_B)
            break;
        }
        case 5: {
            GL_TS1_DISPATCH(GL_TS_B)
#undef GL_TS_B
            break;
        }
        case 6:
        case 7:
#define GL_CT_B(U_, CW_) conv_bwd_ct_launch<T, U_, CW_>(pl, G, gpix, Pc, gbar, st)
            switch (G.U) {
                case 5: e = GL_CT_B(5, 4); break;
                case 6: e = GL_CT_B(6, GL_CT_CW6); break;
                case 7: e = GL_CT_B(7, 4); break;
                case 11: e = GL_CT_B(11, GL_CT_CW11); break;
                case 16: e = GL_CT_B(16, GL_CT_CW16B); break;
                default: e = GL_CT_B(21, 2); break;
            }
#undef GL_CT_B
            break;
        default: {
            dim3 grid((G.s * G.s * G.N * G.N + 255) / 256, (unsigned)Pc);
            gl_conv_bwd_generic<T><<<grid, 256, 0, st>>>(G, gpix, sys_kt, system_id, p_base, gbar);
        }
    }
    return e == cudaSuccess ? 1 : -1;
}

}  // namespace gl
