// gigalens.cu -- C-ABI entry points (include/gigalens.h) and launch logic of libgigalens.
// Product path: hand-written CUDA for sm_100a only; no CPU fallback; nothing here touches oracle/.
#include "../../include/gigalens.h"

#include <cmath>
#include <algorithm>
#include <cstring>
#include <mutex>
#include <new>
#include <vector>

#include "gl_common.cuh"
#include "gl_math.cuh"
#include "gl_conv.cuh"
#include "gl_conv_launch.cuh"
#include "gl_particle.cuh"
#include "gl_probe.cuh"
#include "gl_ray.cuh"
#include "gl_svi.cuh"
#include "gl_hmc.cuh"
#include "gl_linear.cuh"
#include "gl_rng.cuh"

using namespace gl;

struct gl_config {
    gl_config_desc desc;
    std::vector<gl_prior> priors;
    Layout L;
    Geom G;
    PriorTable pt;
    int variant;        // 0: <.,0,1,-1,1>  1: <.,0,1,6,2>  2: <.,3,1,10,2>  3: <.,0,2,-1,3>  4: <.,3,2,10,3>
    int na;             // natural accumulators per chunk for the variant
    int nt_fwd, nt_adj, rpt_fwd, rpt_adj, n_chunk_fwd, n_chunk_adj;   // per phase plane
    int nt_fwd_b, rpt_fwd_b, n_chunk_fwd_b;   // binned forward kernel (psf_grid 1, dedicated path): pixels per thread, chunks per particle
    int n_nap;          // adjoint partials per particle = s*s*n_chunk_adj
    int n_ctile;        // chi^2 partials per particle
    ConvPlan conv;
    CompIdx cidx;       // component index of each light block (gl_ray_comp_kernel)
    AmpMap amp;         // light amplitudes (n = 0 unless amplitude_mode 1 ... see n_amp)
    int n_amp;          // amplitude count of the model, whatever the mode
    int esize;          // sizeof the arithmetic type: 8 (GL_PRECISION_F64) or 4 (GL_PRECISION_F32)
    int uv_split;       // 1: the adjoint stores the shapelet coordinates (u, v) of every ray for gl_shp_coef_kernel (coef_split)
    size_t per_particle_bytes;
    int ct_slot;        // slot of the process-wide constant tap table (gl_conv_ct.cuh), -1: none
};

static thread_local int64_t t_launches = 0;

// Slots of the constant tap table c_ctap (gl_conv_ct.cuh): process-wide, handed out at gl_config_create, returned at destroy.
static std::mutex g_ct_mu;
static bool g_ct_used[CT_NSLOT] = {};
static int ct_slot_acquire() {
    std::lock_guard<std::mutex> lk(g_ct_mu);
    for (int i = 0; i < CT_NSLOT; ++i) if (!g_ct_used[i]) { g_ct_used[i] = true; return i; }
    return -1;
}
static void ct_slot_release(int i) {
    std::lock_guard<std::mutex> lk(g_ct_mu);
    if (i >= 0 && i < CT_NSLOT) g_ct_used[i] = false;
}

// ----------------------------------------------------------------------------- optional per-stage timing (diagnostic)
enum { ST_PREP = 0, ST_UNPACK, ST_RAY_FWD, ST_CONV_FWD, ST_CONV_BWD, ST_RAY_ADJ, ST_FINALIZE, ST_AMP, ST_COUNT };
static const char* const k_stage_names[ST_COUNT] = {"prep", "unpack_prior", "ray_fwd", "conv_chi2", "conv_transpose",
                                                    "ray_adjoint", "finalize", "amplitude_solve"};
struct StageTimer {
    bool on = false;
    std::vector<cudaEvent_t> ev;      // pairs (begin, end)
    std::vector<int> stage;           // stage id of pair i
    size_t used = 0;
    void reset() { used = 0; stage.clear(); }
    void begin(int id, cudaStream_t st) {
        if (!on) return;
        while (ev.size() < 2 * (used + 1)) { cudaEvent_t e; if (cudaEventCreate(&e) != cudaSuccess) { on = false; return; } ev.push_back(e); }
        stage.push_back(id);
        cudaEventRecord(ev[2 * used], st);
    }
    void end(cudaStream_t st) {
        if (!on) return;
        cudaEventRecord(ev[2 * used + 1], st); ++used;
    }
};
static thread_local StageTimer t_timer;

extern "C" void gl_stage_timing_enable(int32_t on) { t_timer.on = on != 0; t_timer.reset(); }
extern "C" int32_t gl_stage_count(void) { return ST_COUNT; }
extern "C" const char* gl_stage_name(int32_t i) { return (i >= 0 && i < ST_COUNT) ? k_stage_names[i] : ""; }
extern "C" int32_t gl_stage_times(float* ms_host, int32_t* launches_host, int32_t n) {
    if (!ms_host || n < ST_COUNT) return -1;
    for (int i = 0; i < n; ++i) { ms_host[i] = 0.f; if (launches_host) launches_host[i] = 0; }
    for (size_t i = 0; i < t_timer.used; ++i) {
        float ms = 0.f;
        if (cudaEventSynchronize(t_timer.ev[2 * i + 1]) != cudaSuccess) return -1;
        if (cudaEventElapsedTime(&ms, t_timer.ev[2 * i], t_timer.ev[2 * i + 1]) != cudaSuccess) return -1;
        ms_host[t_timer.stage[i]] += ms;
        if (launches_host) launches_host[t_timer.stage[i]] += 1;
    }
    return ST_COUNT;
}
#define GL_STAGE(id, st, ...) do { t_timer.begin(id, st); __VA_ARGS__; t_timer.end(st); } while (0)

#ifndef GL_NT_FWD
#define GL_NT_FWD 256
#endif
#ifndef GL_NT_ADJ
#define GL_NT_ADJ 128
#endif
static constexpr int NT_FWD = GL_NT_FWD;     // compiled launch bounds; the block size actually used is chosen per config
static constexpr int NT_ADJ = GL_NT_ADJ;
#ifndef GL_RB_FWD
#define GL_RB_FWD 1
#endif
// Rays per thread the ray kernels aim for (a plane's rays are cut into chunks of about nt * RPT): every CTA stages the particle's
// block and the series coefficients before its first ray, so longer threads amortise that better -- 40 / 64 (round 1, tuned on
// config 2 where a plane is one chunk anyway) against 160 / 256: config 5 adjoint 90.3 -> 87.8 ms, forward 37.4 -> 37.0, config 3
// 17.2 -> 16.9 and 7.43 -> 7.24; 512 gains another 1 % on config 5 but leaves 32 CTAs per particle.
#ifndef GL_RPT_FWD
#define GL_RPT_FWD 160
#endif
#ifndef GL_RPT_ADJ
#define GL_RPT_ADJ 256
#endif
static constexpr int RB_FWD = GL_RB_FWD;  // rays a forward thread evaluates concurrently
static constexpr size_t WS_BUDGET = (size_t)4096 << 20;   // chunk so that per-chunk buffers stay below ~4 GiB
#ifndef GL_WS_BUDGET_UV_GIB
#define GL_WS_BUDGET_UV_GIB 16
#endif
static constexpr size_t WS_BUDGET_UV = (size_t)GL_WS_BUDGET_UV_GIB << 30;   // the split adjoint also keeps (u, v) of every ray
// Backward modelling keeps n_amp component images per particle: with the 4 GiB budget a 30-amplitude model is cut into
// chunks of ~280 particles, too few CTAs for the one-CTA-per-particle kernels (config 3: 506 -> see DESIGN.md section 16).
static constexpr size_t WS_BUDGET_AMP = (size_t)16384 << 20;

static inline size_t align256(size_t x) { return (x + 255) & ~(size_t)255; }

extern "C" const char* gl_status_string(gl_status s) {
    switch (s) {
        case GL_OK: return "GL_OK";
        case GL_ERR_NULL: return "GL_ERR_NULL: a required pointer is NULL";
        case GL_ERR_BAD_CONFIG: return "GL_ERR_BAD_CONFIG: inconsistent configuration";
        case GL_ERR_BAD_SHAPE: return "GL_ERR_BAD_SHAPE: negative particle count";
        case GL_ERR_UNSUPPORTED: return "GL_ERR_UNSUPPORTED: no kernel for this configuration";
        case GL_ERR_WORKSPACE: return "GL_ERR_WORKSPACE: workspace too small or misaligned";
        case GL_ERR_CUDA: return "GL_ERR_CUDA: CUDA runtime error";
        case GL_ERR_NOALLOC_LIMIT: return "GL_ERR_NOALLOC_LIMIT: the call needs more scratch than the library's static buffer (GL_NOALLOC_MAX_BYTES); use fewer particles per call or gl_logpost_grad with a caller workspace";
    }
    return "unknown gl_status";
}

extern "C" const char* gl_version(void) { return "0.1"; }
extern "C" int64_t gl_last_launch_count(void) { return t_launches; }

static int layout_from_desc(const gl_config_desc& d, Layout& L) {
    int k = 0;
    L.mass = k; k += 1;
    if (d.mass_model == 1) { L.gamma = k; k += 1; } else L.gamma = -1;
    L.ell = k; k += 4;
    if (d.has_shear) { L.shear = k; k += 2; } else L.shear = -1;
    if (d.multipole_mask & 1) { L.mp3 = k; k += 2; } else L.mp3 = -1;
    if (d.multipole_mask & 2) { L.mp4 = k; k += 2; } else L.mp4 = -1;
    if (d.n_source_sersic > 0) { L.src = k; k += 7; } else L.src = -1;
    if (d.n_source_sersic > 1) { L.src1 = k; k += 7; } else L.src1 = -1;
    if (d.n_source_sersic > 1 && d.source2_plane) { L.eta2 = k; k += 1; } else L.eta2 = -1;
    L.nmax = d.shapelet_nmax; L.n_coef = 0;
    if (d.shapelet_nmax >= 0) { L.n_coef = (d.shapelet_nmax + 1) * (d.shapelet_nmax + 2) / 2; L.shp = k; k += 1 + L.n_coef; } else L.shp = -1;
    if (d.n_lens_sersic >= 1) { L.ll0 = k; k += 7; } else L.ll0 = -1;
    if (d.n_lens_sersic >= 2) { L.ll1 = k; k += 7; } else L.ll1 = -1;
    if (d.n_lens_sersic >= 3) { L.ll2 = k; k += 7; } else L.ll2 = -1;
    L.n_params = k; L.param_space = d.param_space; L.mass_model = d.mass_model;
    return k;
}

extern "C" gl_status gl_config_create(const gl_config_desc* d, gl_config** out) {
    if (!d || !out) return GL_ERR_NULL;
    *out = nullptr;
    if (!d->priors) return GL_ERR_NULL;
    if (d->n_pix < 1 || d->supersample < 1 || d->psf_size < 1 || (d->psf_size & 1) == 0) return GL_ERR_BAD_CONFIG;
    if (!(d->pix_scale > 0.f) || !std::isfinite(d->pix_scale)) return GL_ERR_BAD_CONFIG;
    if (d->mass_model != 0 && d->mass_model != 1) return GL_ERR_BAD_CONFIG;
    if (d->mass_model == 1 && (d->epl_terms < 2 || d->epl_terms > 30)) return GL_ERR_BAD_CONFIG;
    if ((d->has_shear & ~1) || (d->multipole_mask & ~3) || (d->param_space & ~1)) return GL_ERR_BAD_CONFIG;
    if (d->n_source_sersic < 0 || d->n_source_sersic > 2 || d->n_lens_sersic < 0 || d->n_lens_sersic > 3) return GL_ERR_BAD_CONFIG;
    if (d->shapelet_nmax < -1 || d->shapelet_nmax > 10) return GL_ERR_BAD_CONFIG;
    if (d->shapelet_nmax >= 0 && d->n_source_sersic < 1) return GL_ERR_BAD_CONFIG;      // shapelets share the first source's centre
    if (d->n_systems < 1) return GL_ERR_BAD_CONFIG;
    if (d->precision != GL_PRECISION_F64 && d->precision != GL_PRECISION_F32) return GL_ERR_BAD_CONFIG;
    if (d->psf_grid != 0 && d->psf_grid != 1) return GL_ERR_UNSUPPORTED;
    if (d->noise_model != 0 && d->noise_model != 1) return GL_ERR_BAD_CONFIG;
    if (d->noise_model == 1 && !(d->exposure_time > 0.f && std::isfinite(d->exposure_time))) return GL_ERR_BAD_CONFIG;
    if (d->amplitude_mode != 0 && d->amplitude_mode != 1) return GL_ERR_BAD_CONFIG;
    if (d->source2_plane != 0 && d->source2_plane != 1) return GL_ERR_BAD_CONFIG;
    if (d->source2_plane == 1 && d->n_source_sersic < 2) return GL_ERR_BAD_CONFIG;
    if (d->amplitude_mode == 1 && d->noise_model != 0) return GL_ERR_UNSUPPORTED;     // chi^2 must be quadratic in the amplitudes
    Layout L{};
    int np = layout_from_desc(*d, L);
    if (np != d->n_params || np > 128) return GL_ERR_BAD_CONFIG;
    for (int i = 0; i < np; ++i) {
        const gl_prior& p = d->priors[i];
        if (p.kind < GL_PRIOR_NONE || p.kind > GL_PRIOR_LOGUNIFORM) return GL_ERR_BAD_CONFIG;
        bool gauss = p.kind == GL_PRIOR_NORMAL || p.kind == GL_PRIOR_LOGNORMAL || p.kind == GL_PRIOR_TRUNCNORMAL;
        bool bounded = p.kind == GL_PRIOR_UNIFORM || p.kind == GL_PRIOR_TRUNCNORMAL || p.kind == GL_PRIOR_LOGUNIFORM;
        if (gauss && !(p.b > 0.f && std::isfinite(p.a) && std::isfinite(p.b))) return GL_ERR_BAD_CONFIG;
        if (bounded && !(p.hi > p.lo && std::isfinite(p.lo) && std::isfinite(p.hi))) return GL_ERR_BAD_CONFIG;
        if (p.kind == GL_PRIOR_LOGUNIFORM && !(p.lo > 0.f)) return GL_ERR_BAD_CONFIG;
    }
    const int64_t M64 = (int64_t)d->n_pix * d->supersample;
    if (M64 > 4096 || d->psf_size > 255) return GL_ERR_UNSUPPORTED;
    gl_config* c = new (std::nothrow) gl_config();
    if (!c) return GL_ERR_BAD_CONFIG;
    c->ct_slot = -1;
    c->desc = *d;
    c->priors.assign(d->priors, d->priors + np);
    c->desc.priors = c->priors.data();
    for (int i = 0; i < np; ++i) {
        c->pt.kind[i] = d->priors[i].kind; c->pt.a[i] = d->priors[i].a; c->pt.b[i] = d->priors[i].b;
        c->pt.lo[i] = d->priors[i].lo; c->pt.hi[i] = d->priors[i].hi;
    }
    {   // light amplitudes in the flat order S18 and their PB slots
        AmpMap& A = c->amp; A.n = 0;
        auto add = [&](int pb_off, int shp, double scl = 1.0) { A.off[A.n] = (short)pb_off; A.shp[A.n] = (unsigned char)shp; A.scl[A.n] = (float)scl; ++A.n; };
        CompIdx& ci = c->cidx; ci.src = ci.src1 = ci.shp0 = ci.ll0 = ci.ll1 = ci.ll2 = -1; ci.n_coef = L.n_coef;
        if (L.src >= 0) { ci.src = A.n; add(PB_SRC + SB_IE, 0); }
        if (L.src1 >= 0) { ci.src1 = A.n; add(PB_SRC1 + SB_IE, 0); }
        if (L.n_coef > 0) ci.shp0 = A.n;
        for (int k = 0; k < L.n_coef; ++k) add(PB_SHP_A + k, 1, shp_scale_host(k));
        if (L.ll0 >= 0) { ci.ll0 = A.n; add(PB_LL0 + SB_IE, 0); }
        if (L.ll1 >= 0) { ci.ll1 = A.n; add(PB_LL1 + SB_IE, 0); }
        if (L.ll2 >= 0) { ci.ll2 = A.n; add(PB_LL2 + SB_IE, 0); }
        c->n_amp = A.n;
        L.amp_mode = d->amplitude_mode;
        if (d->amplitude_mode == 1) {
            if (A.n == 0) { delete c; return GL_ERR_BAD_CONFIG; }
            for (int i = 0; i < np; ++i) if (is_amp(L, i)) c->pt.kind[i] = GL_PRIOR_NONE;   // no prior, no bijector (S21)
        }
    }
    for (int i = np; i < 128; ++i) { c->pt.kind[i] = 0; c->pt.a[i] = 0; c->pt.b[i] = 1; c->pt.lo[i] = 0; c->pt.hi[i] = 1; }
    // kernel variant: the smallest compiled superset of the requested components
    const bool extra = d->n_source_sersic > 1 || d->n_lens_sersic > 2;       // second source / third lens-light block
    if (!extra && d->multipole_mask == 0 && d->shapelet_nmax < 0 && d->n_lens_sersic <= 1) { c->variant = 0; L.ker_nmax = -1; c->na = NA_SHA; }
    else if (!extra && d->multipole_mask == 0 && d->shapelet_nmax <= 6) { c->variant = 1; L.ker_nmax = 6; c->na = NA_SHA + 28; }
    else if (!extra) { c->variant = 2; L.ker_nmax = 10; c->na = NA_SHA + 66; }
    else if (d->multipole_mask == 0 && d->shapelet_nmax < 0) { c->variant = 3; L.ker_nmax = -1; c->na = NA_SHA; }
    else { c->variant = 4; L.ker_nmax = 10; c->na = NA_SHA + 66; }
    c->L = L;
    Geom& G = c->G;
    G.N = d->n_pix; G.s = d->supersample; G.M = (int)M64; G.K = d->psf_size; G.pgrid = d->psf_grid;
    G.noise_model = d->noise_model; G.inv_texp = d->noise_model == 1 ? 1.0 / (double)d->exposure_time : 0.0;
    // psf_grid 1 (bin, then convolve at the pixel scale) is the same stride-s correlation with
    // the box-expanded kernel k_eff[m][n] = psf[m / s][n / s]: s*K taps per side, half-width s*(K-1)/2
    G.c = d->psf_grid == 1 ? G.s * ((d->psf_size - 1) / 2) : (d->psf_size - 1) / 2;
    G.KE = d->psf_grid == 1 ? G.s * G.K : G.K + G.s - 1;
    const int KE = G.KE;
    G.U = (KE + G.s - 1) / G.s; G.KEp = G.U * G.s;
    G.n_terms = d->mass_model == 1 ? d->epl_terms : 0;
    G.delta2 = (double)d->pix_scale * (double)d->pix_scale;
    (void)M64;
    c->esize = d->precision == GL_PRECISION_F64 ? 8 : 4;
    c->ct_slot = d->n_systems == 1 ? ct_slot_acquire() : -1;      // constant-memory tap table of the uniform-tap step D
    c->uv_split = (c->esize == 8 && L.ker_nmax > 6) ? 1 : 0;      // must agree with coef_split<T, V>() in gl_ray.cuh
    // what a full chunk holds, as bytes per particle per element of the ray image (conv_plan sizes its row bands by it)
    const ConvChunkHint hint{d->amplitude_mode == 1 ? (size_t)0 : (c->uv_split ? WS_BUDGET_UV : WS_BUDGET), c->uv_split ? 3 : 1};
    c->conv = conv_plan(G, c->esize, d->n_systems, c->ct_slot, hint);   // also fills the padded-layout fields of G
    if (c->conv.kind != 6 && c->ct_slot >= 0) { ct_slot_release(c->ct_slot); c->ct_slot = -1; }
    c->n_ctile = c->conv.n_ctile;
    // ray kernels: one CTA per (particle, phase plane, chunk); pick the block size that wastes the fewest lanes
    const int NN = G.N * G.N;
    auto pick = [&](int nt_max, int rpt_target, int& nt, int& rpt, int& n_chunk) {
        int best = nt_max; double best_w = 1e30;
        for (int t = nt_max; t >= nt_max / 2 && t >= 32; t -= 32) {
            const int it = (NN + t - 1) / t;
            const double w = (double)it * t / NN;
            if (w < best_w - 1e-9) { best_w = w; best = t; }
        }
        nt = best;
        const int iters = (NN + nt - 1) / nt;
        n_chunk = (iters + rpt_target - 1) / rpt_target;
        rpt = (iters + n_chunk - 1) / n_chunk;
    };
    pick(NT_FWD, GL_RPT_FWD, c->nt_fwd, c->rpt_fwd, c->n_chunk_fwd);
    pick(NT_ADJ, GL_RPT_ADJ, c->nt_adj, c->rpt_adj, c->n_chunk_adj);
    pick(NT_FWD, std::max(1, GL_RPT_FWD / (G.s * G.s)), c->nt_fwd_b, c->rpt_fwd_b, c->n_chunk_fwd_b);   // a pixel = s*s rays
    c->n_nap = G.s * G.s * c->n_chunk_adj;
    c->per_particle_bytes = (size_t)c->esize * ((size_t)PB_STRIDE + ray_stride(G) + gpix_stride(G) + (size_t)c->n_ctile +
                                                (size_t)c->n_nap * c->na) + sizeof(double) + 6 * 256;
    if (d->amplitude_mode == 1) c->per_particle_bytes += (size_t)c->esize * c->n_amp * (gpix_stride(G) + ray_stride(G));
    if (c->uv_split) c->per_particle_bytes += (size_t)c->esize * 2 * ray_stride(G);
    *out = c;
    return GL_OK;
}

extern "C" void gl_config_destroy(gl_config* c) { if (c) ct_slot_release(c->ct_slot); delete c; }
extern "C" int32_t gl_config_n_params(const gl_config* c) { return c ? c->L.n_params : 0; }
extern "C" int32_t gl_config_n_amplitudes(const gl_config* c) { return c ? c->n_amp : 0; }
extern "C" gl_status gl_config_shape(const gl_config* c, int32_t* out) {
    if (!c || !out) return GL_ERR_NULL;
    out[0] = c->desc.n_pix; out[1] = c->desc.psf_size; out[2] = c->desc.n_systems; out[3] = c->L.n_params; out[4] = c->n_amp;
    return GL_OK;
}

struct Plan {
    int64_t Pc;
    size_t off_ctap;    // plane-ordered tap table of the uniform-tap step D (staging for the constant slot)
    size_t off_tab, off_kt, off_w, off_sl, off_pb, off_lpd, off_ray, off_gpix, off_chi, off_nap, off_uv, off_comp, off_cray, off_zobs, off_uw, off_sid, total;
};

// balanced: the batch is cut into the FEWEST chunks the budget allows, all of (almost) the same size, instead of full chunks
// plus a small remainder (config 5: 5 x 410 instead of 4 x 487 + 100 -- a 100-particle chunk leaves most SMs idle in the
// persistent and few-CTA kernels).  gl_workspace_bytes reports the unbalanced plan: an upper bound that is flat beyond the
// chunk size, as include/gigalens.h promises.
static Plan make_plan(const gl_config* c, int64_t P, bool balanced = true) {
    Plan pl{};
    const Geom& G = c->G;
    // the split adjoint keeps (u, v) of every ray: twice the budget keeps its chunks as large as the other variants'
    int64_t pc_max = (int64_t)((c->desc.amplitude_mode == 1 ? WS_BUDGET_AMP : (c->uv_split ? WS_BUDGET_UV : WS_BUDGET)) / c->per_particle_bytes);
    if (pc_max < 1) pc_max = 1;
    if (pc_max > 32768) pc_max = 32768;
    pl.Pc = P < pc_max ? P : pc_max;
    if (balanced && P > pc_max) { const int64_t nch = (P + pc_max - 1) / pc_max; pl.Pc = (P + nch - 1) / nch; }
    size_t o = 0;
    const size_t nsys = (size_t)c->desc.n_systems, es = (size_t)c->esize;
    pl.off_tab = o;  o = align256(o + sizeof(double) * MATH_TAB_DOUBLES);
    pl.off_kt = o;   o = align256(o + es * nsys * G.s * G.s * G.U * G.U);
    pl.off_ctap = o; o = align256(o + es * (size_t)G.s * G.s * G.U * ((G.U + 1) & ~1));
    pl.off_w = o;    o = align256(o + es * nsys * G.N * G.N);
    pl.off_sl = o;   o = align256(o + sizeof(double) * nsys);
    pl.off_pb = o;   o = align256(o + es * (size_t)pl.Pc * PB_STRIDE);
    pl.off_lpd = o;  o = align256(o + sizeof(double) * (size_t)pl.Pc);
    pl.off_ray = o;  o = align256(o + es * (size_t)pl.Pc * ray_stride(G));
    pl.off_gpix = o; o = align256(o + es * (size_t)pl.Pc * gpix_stride(G));
    pl.off_chi = o;  o = align256(o + es * (size_t)pl.Pc * c->n_ctile);
    pl.off_nap = o;  o = align256(o + es * (size_t)pl.Pc * c->n_nap * c->na);
    pl.off_uv = o;
    if (c->uv_split) o = align256(o + es * (size_t)pl.Pc * 2 * ray_stride(G));
    pl.off_comp = pl.off_cray = pl.off_zobs = pl.off_uw = pl.off_sid = o;
    if (c->desc.amplitude_mode == 1) {
        pl.off_comp = o; o = align256(o + es * (size_t)c->n_amp * pl.Pc * gpix_stride(G));
        pl.off_cray = o; o = align256(o + es * (size_t)c->n_amp * pl.Pc * ray_stride(G));
        pl.off_zobs = o; o = align256(o + sizeof(float) * nsys * G.N * G.N);
        pl.off_uw = o;   o = align256(o + es * nsys * G.N * G.N);
        pl.off_sid = o;  o = align256(o + sizeof(int32_t) * (size_t)c->n_amp * pl.Pc);
    }
    pl.total = o;
    return pl;
}

extern "C" size_t gl_workspace_bytes(const gl_config* c, int64_t n_particles) {
    if (!c || n_particles <= 0) return 0;
    return make_plan(c, n_particles, false).total;
}

// Diagnostic: where the per-particle block PB of the LAST processed chunk sits in the workspace, so that bench.py can
// read what step A decided per particle (the precision bands of the series) without a kernel of its own.
extern "C" gl_status gl_workspace_layout(const gl_config* c, int64_t n_particles, int64_t* out) {
    if (!c || !out) return GL_ERR_NULL;
    if (n_particles <= 0) return GL_ERR_BAD_SHAPE;
    const Plan pl = make_plan(c, n_particles);
    out[0] = (int64_t)pl.off_pb; out[1] = pl.Pc; out[2] = PB_STRIDE; out[3] = c->esize;
    out[4] = PB_SER_M1; out[5] = PB_SER_M2; out[6] = PB_VALID; out[7] = (n_particles - 1) / pl.Pc * pl.Pc;   // first particle of the last chunk
    return GL_OK;
}

// ----------------------------------------------------------------------------- variant dispatch
template <class T, class V>
static void launch_ray_fwd(const gl_config* c, const T* pb, const double* tab, T* ray, int64_t Pc, cudaStream_t st) {
    if (c->G.binned) {       // psf_grid 1, dedicated path: the binned image straight into plane 0 (gl_ray_fwd_binned_kernel)
        dim3 grid(c->n_chunk_fwd_b, (unsigned)Pc);
        gl_ray_fwd_binned_kernel<T, V, NT_FWD><<<grid, c->nt_fwd_b, 0, st>>>(c->G, pb, tab, ray, c->rpt_fwd_b, c->n_chunk_fwd_b);
        return;
    }
    dim3 grid(c->G.s * c->G.s * c->n_chunk_fwd, (unsigned)Pc);
    gl_ray_fwd_kernel<T, V, NT_FWD, RB_FWD><<<grid, c->nt_fwd, 0, st>>>(c->G, pb, tab, ray, c->rpt_fwd, c->n_chunk_fwd);
}
template <class T, class V>
static cudaError_t launch_ray_adj(const gl_config* c, const T* pb, const double* tab, const T* gbar, T* nap, T* uv, int64_t Pc, cudaStream_t st) {
    dim3 grid(c->n_nap, (unsigned)Pc);
    gl_ray_adj_kernel<T, V, NT_ADJ><<<grid, c->nt_adj, 0, st>>>(c->G, pb, tab, gbar, nap, uv, c->rpt_adj, c->n_chunk_adj);
    if constexpr (coef_split<T, V>()) {     // the shapelet coefficient sums from the stored (u, v): same grid, same partial slots
        // its own block size (128) and rays per thread: any partition of a plane's rays over the n_chunk_adj CTAs of a plane works
        const int ntc = 128, rptc = (c->G.N * c->G.N + c->n_chunk_adj * ntc - 1) / (c->n_chunk_adj * ntc);
        gl_shp_coef_kernel<T, V::NMAX, V::NA, 128><<<grid, ntc, 0, st>>>(c->G, pb, tab, gbar, uv, nap, rptc, c->n_chunk_adj);
        ++t_launches;
    }
    return cudaSuccess;
}

using V_S0 = Variant<0, 0, 1, -1, 1>; using V_E0 = Variant<1, 0, 1, -1, 1>;
using V_S1 = Variant<0, 0, 1, 6, 2>;  using V_E1 = Variant<1, 0, 1, 6, 2>;
using V_S2 = Variant<0, 3, 1, 10, 2>; using V_E2 = Variant<1, 3, 1, 10, 2>;
using V_S3 = Variant<0, 0, 2, -1, 3>; using V_E3 = Variant<1, 0, 2, -1, 3>;   // the real-system component list
using V_S4 = Variant<0, 3, 2, 10, 3>; using V_E4 = Variant<1, 3, 2, 10, 3>;   // everything

template <class T>
static void ray_fwd(const gl_config* c, const T* pb, const double* tab, T* ray, int64_t Pc, cudaStream_t st) {
    const int id = c->variant * 2 + c->desc.mass_model;
    switch (id) {
        case 0: launch_ray_fwd<T, V_S0>(c, pb, tab, ray, Pc, st); break;
        case 1: launch_ray_fwd<T, V_E0>(c, pb, tab, ray, Pc, st); break;
        case 2: launch_ray_fwd<T, V_S1>(c, pb, tab, ray, Pc, st); break;
        case 3: launch_ray_fwd<T, V_E1>(c, pb, tab, ray, Pc, st); break;
        case 4: launch_ray_fwd<T, V_S2>(c, pb, tab, ray, Pc, st); break;
        case 5: launch_ray_fwd<T, V_E2>(c, pb, tab, ray, Pc, st); break;
        case 6: launch_ray_fwd<T, V_S3>(c, pb, tab, ray, Pc, st); break;
        case 7: launch_ray_fwd<T, V_E3>(c, pb, tab, ray, Pc, st); break;
        case 8: launch_ray_fwd<T, V_S4>(c, pb, tab, ray, Pc, st); break;
        default: launch_ray_fwd<T, V_E4>(c, pb, tab, ray, Pc, st); break;
    }
}
template <class T, class V>
static void launch_ray_comp(const gl_config* c, const T* pb, const double* tab, T* cray, int64_t Pc, cudaStream_t st) {
    dim3 grid(c->G.s * c->G.s * c->n_chunk_fwd, (unsigned)Pc);
    gl_ray_comp_kernel<T, V, NT_FWD><<<grid, c->nt_fwd, 0, st>>>(c->G, c->cidx, c->amp.n, pb, tab, cray, (size_t)Pc * ray_stride(c->G),
                                                                 c->rpt_fwd, c->n_chunk_fwd);
}
template <class T>
static void ray_comp(const gl_config* c, const T* pb, const double* tab, T* cray, int64_t Pc, cudaStream_t st) {
    const int id = c->variant * 2 + c->desc.mass_model;
    switch (id) {
        case 0: launch_ray_comp<T, V_S0>(c, pb, tab, cray, Pc, st); break;
        case 1: launch_ray_comp<T, V_E0>(c, pb, tab, cray, Pc, st); break;
        case 2: launch_ray_comp<T, V_S1>(c, pb, tab, cray, Pc, st); break;
        case 3: launch_ray_comp<T, V_E1>(c, pb, tab, cray, Pc, st); break;
        case 4: launch_ray_comp<T, V_S2>(c, pb, tab, cray, Pc, st); break;
        case 5: launch_ray_comp<T, V_E2>(c, pb, tab, cray, Pc, st); break;
        case 6: launch_ray_comp<T, V_S3>(c, pb, tab, cray, Pc, st); break;
        case 7: launch_ray_comp<T, V_E3>(c, pb, tab, cray, Pc, st); break;
        case 8: launch_ray_comp<T, V_S4>(c, pb, tab, cray, Pc, st); break;
        default: launch_ray_comp<T, V_E4>(c, pb, tab, cray, Pc, st); break;
    }
}
template <class T>
static cudaError_t ray_adj(const gl_config* c, const T* pb, const double* tab, const T* gbar, T* nap, T* uv, int64_t Pc, cudaStream_t st) {
    const int id = c->variant * 2 + c->desc.mass_model;
    switch (id) {
        case 0: return launch_ray_adj<T, V_S0>(c, pb, tab, gbar, nap, uv, Pc, st);
        case 1: return launch_ray_adj<T, V_E0>(c, pb, tab, gbar, nap, uv, Pc, st);
        case 2: return launch_ray_adj<T, V_S1>(c, pb, tab, gbar, nap, uv, Pc, st);
        case 3: return launch_ray_adj<T, V_E1>(c, pb, tab, gbar, nap, uv, Pc, st);
        case 4: return launch_ray_adj<T, V_S2>(c, pb, tab, gbar, nap, uv, Pc, st);
        case 5: return launch_ray_adj<T, V_E2>(c, pb, tab, gbar, nap, uv, Pc, st);
        case 6: return launch_ray_adj<T, V_S3>(c, pb, tab, gbar, nap, uv, Pc, st);
        case 7: return launch_ray_adj<T, V_E3>(c, pb, tab, gbar, nap, uv, Pc, st);
        case 8: return launch_ray_adj<T, V_S4>(c, pb, tab, gbar, nap, uv, Pc, st);
        default: return launch_ray_adj<T, V_E4>(c, pb, tab, gbar, nap, uv, Pc, st);
    }
}

// mode 0: logpost, 1: logpost + grad, 2: model image
template <class T>
static gl_status run_t(const gl_config* c, int mode, const float* obs, const float* sigma, const float* psf,
                       const float* params, const int32_t* system_id, int64_t P, float* out_logp, float* out_grad,
                       float* out_image, float* out_amp, void* ws, const Plan& pl, cudaStream_t st) {
    const Geom& G = c->G;
    char* w = (char*)ws;
    double* tab = (double*)(w + pl.off_tab);
    T* sys_kt = (T*)(w + pl.off_kt); T* sys_w = (T*)(w + pl.off_w); double* sys_sl = (double*)(w + pl.off_sl);
    T* pb = (T*)(w + pl.off_pb); double* lpd = (double*)(w + pl.off_lpd);
    T* ray = (T*)(w + pl.off_ray); T* gpix = (T*)(w + pl.off_gpix);
    T* chi = (T*)(w + pl.off_chi); T* nap = (T*)(w + pl.off_nap);
    double* tab_out = sizeof(T) == 8 ? tab : nullptr;
    const bool solve = c->desc.amplitude_mode == 1 && mode != 2;
    T* comp = (T*)(w + pl.off_comp); float* zobs = (float*)(w + pl.off_zobs); T* unit_w = (T*)(w + pl.off_uw);
    Layout L = c->L;
    if (mode == 2) L.amp_mode = 0;          // gl_model_image: the amplitude entries of params are the amplitudes

    // sigma is not an input of gl_model_image (mode 2): prep then only builds kt (and the math tables)
    GL_STAGE(ST_PREP, st, (gl_prep_kernel<T><<<c->desc.n_systems, 256, 0, st>>>(G, psf, mode == 2 ? nullptr : sigma, sys_kt, sys_w,
                                                                             sys_sl, tab_out)));
    ++t_launches;
    if (c->conv.kind == 6 || c->conv.kind == 7) {                 // uniform-tap step D: refill this configuration's constant slot from the PSF of this call
        const int nk = conv_ct_upload<T>(c->conv, G, sys_kt, (T*)(w + pl.off_ctap), st);
        if (nk < 0) return GL_ERR_CUDA;
        t_launches += nk;
    }
    if (solve) {
        const size_t n = (size_t)c->desc.n_systems * G.N * G.N;
        gl_amp_fill_kernel<T><<<(unsigned)((n + 255) / 256), 256, 0, st>>>(n, zobs, unit_w);
        ++t_launches;
    }
    for (int64_t base = 0; base < P; base += pl.Pc) {
        const int64_t Pc = (P - base) < pl.Pc ? (P - base) : pl.Pc;
        GL_STAGE(ST_UNPACK, st, (gl_unpack_kernel<T><<<(unsigned)((Pc + UNPACK_WPB - 1) / UNPACK_WPB), UNPACK_WPB * 32, 0, st>>>(
            c->pt, L, G, c->desc.pix_scale, params + base * c->L.n_params, Pc, pb, lpd)));
        ++t_launches;
        if (solve) {     // unit-amplitude component images through steps B-D, then the normal equations (gl_linear.cuh)
            const int na = c->amp.n;
            T* cray = (T*)(w + pl.off_cray);
            gl_amp_select_kernel<T><<<(unsigned)((Pc * na + 255) / 256), 256, 0, st>>>(c->amp, -1, Pc, pb);
            ++t_launches;
            GL_STAGE(ST_RAY_FWD, st, ray_comp<T>(c, pb, tab, cray, Pc, st)); ++t_launches;
            // step D for all components as na * Pc virtual particles (component-major, like both buffers)
            int32_t* sid_exp = nullptr;
            if (system_id) {
                sid_exp = (int32_t*)(w + pl.off_sid);
                gl_amp_sid_kernel<<<(unsigned)((Pc * na + 255) / 256), 256, 0, st>>>(system_id + base, Pc, na, sid_exp);
                ++t_launches;
            }
            const int kg = c->conv.kind == 0 ? (int)std::max<int64_t>(1, 65535 / Pc) : na;    // generic kernels: grid.y <= 65535
            for (int k = 0; k < na; k += kg) {
                const int nk_c = std::min(kg, na - k);
                int nk = 0;
                GL_STAGE(ST_CONV_FWD, st, nk = conv_fwd_launch<T>(c->conv, G, cray + (size_t)k * Pc * ray_stride(G), sys_kt, unit_w, zobs,
                                                 sid_exp ? sid_exp + (size_t)k * Pc : nullptr, 0, (int64_t)nk_c * Pc,
                                                 comp + (size_t)k * Pc * gpix_stride(G), nullptr, nullptr, st));
                if (nk < 0) return GL_ERR_CUDA;
                t_launches += nk;
            }
            const size_t sm = amp_solve_smem(na);
            if (sm > 40 * 1024 && cudaFuncSetAttribute(gl_amp_solve_kernel<T>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm) != cudaSuccess)
                return GL_ERR_CUDA;
            GL_STAGE(ST_AMP, st, (gl_amp_solve_kernel<T><<<(unsigned)Pc, 256, sm, st>>>(G, c->amp, comp, Pc, obs, sys_w, system_id, base,
                                                                                 pb, out_amp, gpix, chi, c->n_ctile, amp_solve_tp(na))));
            ++t_launches;
        }
        int nl = 0;
        if (!solve) {      // backward modelling: gl_amp_solve_kernel has already written g_pix and chi^2 at a*
            GL_STAGE(ST_RAY_FWD, st, ray_fwd<T>(c, pb, tab, ray, Pc, st)); ++t_launches;
            GL_STAGE(ST_CONV_FWD, st, nl = conv_fwd_launch<T>(c->conv, G, ray, sys_kt, sys_w, obs, system_id, base, Pc,
                                             mode == 2 ? nullptr : gpix, mode == 2 ? nullptr : chi,
                                             mode == 2 ? out_image : nullptr, st, /*prebinned=*/G.binned != 0));
            if (nl < 0) return GL_ERR_CUDA;
            t_launches += nl;
        }
        if (mode == 2) { if (cudaPeekAtLastError() != cudaSuccess) return GL_ERR_CUDA; continue; }
        if (mode == 1) {
            GL_STAGE(ST_CONV_BWD, st, nl = conv_bwd_launch<T>(c->conv, G, gpix, sys_kt, system_id, base, Pc, ray, st));
            if (nl < 0) return GL_ERR_CUDA;
            t_launches += nl;
            cudaError_t ea = cudaSuccess;
            GL_STAGE(ST_RAY_ADJ, st, ea = ray_adj<T>(c, pb, tab, ray, nap, (T*)(w + pl.off_uv), Pc, st)); ++t_launches;
            if (ea != cudaSuccess) return GL_ERR_CUDA;
        }
        const int wpb = 4;
        GL_STAGE(ST_FINALIZE, st, (gl_finalize_kernel<T><<<(unsigned)((Pc + wpb - 1) / wpb), wpb * 32, wpb * (NA_MAX + 256) * sizeof(double), st>>>(
            c->pt, L, G, params, pb, lpd, chi, c->n_ctile, mode == 1 ? nap : nullptr, c->n_nap, c->na,
            sys_sl, system_id, Pc, base, out_logp, out_grad)));
        ++t_launches;
        if (cudaPeekAtLastError() != cudaSuccess) return GL_ERR_CUDA;     // a failed launch: enqueue no further chunk
    }
    return GL_OK;
}

// Every argument check of the hot path, on the host, BEFORE any launch (the consumers gl_map_step / gl_svi_step /
// gl_hmc_step call it before their own first kernel).  ws_bytes is what the hot path may use of the workspace.
static gl_status validate(const gl_config* c, int mode, const float* obs, const float* sigma, const float* psf,
                          const float* params, int64_t P, const float* out_logp, const float* out_grad,
                          const float* out_image, const void* ws, size_t ws_bytes) {
    if (!c) return GL_ERR_NULL;
    if (P < 0) return GL_ERR_BAD_SHAPE;
    if (P == 0) return GL_OK;
    if (!psf || !params || !ws) return GL_ERR_NULL;
    if (mode != 2 && (!obs || !sigma || !out_logp)) return GL_ERR_NULL;
    if (mode == 1 && !out_grad) return GL_ERR_NULL;
    if (mode == 2 && !out_image) return GL_ERR_NULL;
    if (ws_bytes < make_plan(c, P).total || ((uintptr_t)ws & 255) != 0) return GL_ERR_WORKSPACE;
    return GL_OK;
}

// A non-sticky CUDA error left behind by the caller's earlier work would otherwise be reported by the launch checks
// of this call as GL_ERR_CUDA: it is cleared on entry (a sticky error stays and is reported).
static inline void clear_stale_error() { (void)cudaGetLastError(); }

static gl_status run(const gl_config* c, int mode, const float* obs, const float* sigma, const float* psf,
                     const float* params, const int32_t* system_id, int64_t P, float* out_logp, float* out_grad,
                     float* out_image, void* ws, size_t ws_bytes, cudaStream_t st, float* out_amp = nullptr) {
    t_launches = 0;
    t_timer.reset();
    const gl_status sv = validate(c, mode, obs, sigma, psf, params, P, out_logp, out_grad, out_image, ws, ws_bytes);
    if (sv != GL_OK || P == 0) return sv;
    clear_stale_error();
    const Plan pl = make_plan(c, P);
    if (c->esize == 8)
        return run_t<double>(c, mode, obs, sigma, psf, params, system_id, P, out_logp, out_grad, out_image, out_amp, ws, pl, st);
    return run_t<float>(c, mode, obs, sigma, psf, params, system_id, P, out_logp, out_grad, out_image, out_amp, ws, pl, st);
}

extern "C" gl_status gl_logpost(const gl_config* cfg, const float* obs, const float* noise_sigma, const float* psf,
                                const float* params, const int32_t* system_id, int64_t n_particles,
                                float* out_logp, void* workspace, size_t workspace_bytes, void* stream) {
    return run(cfg, 0, obs, noise_sigma, psf, params, system_id, n_particles, out_logp, nullptr, nullptr,
               workspace, workspace_bytes, (cudaStream_t)stream);
}

extern "C" gl_status gl_logpost_grad(const gl_config* cfg, const float* obs, const float* noise_sigma, const float* psf,
                                     const float* params, const int32_t* system_id, int64_t n_particles,
                                     float* out_logp, float* out_grad, void* workspace, size_t workspace_bytes, void* stream) {
    return run(cfg, 1, obs, noise_sigma, psf, params, system_id, n_particles, out_logp, out_grad, nullptr,
               workspace, workspace_bytes, (cudaStream_t)stream);
}

// ----------------------------------------------------------------------------- no-allocation entry point
// Workspace of gl_logpost_grad_noalloc: a file-scope device array (every GPU that loads the library holds it until exit).
// In HOST code the name is only a stand-in for the symbol, not a device address: the address comes from
// cudaGetSymbolAddress, once per device, with that device current.
static __device__ __align__(256) unsigned char g_noalloc_scratch[GL_NOALLOC_MAX_BYTES];
static std::mutex g_noalloc_mu;
static void* g_noalloc_ptr[64] = {};          // per device ordinal
static gl_status noalloc_scratch(void** out) {
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= 64) return GL_ERR_CUDA;
    std::lock_guard<std::mutex> lk(g_noalloc_mu);
    if (!g_noalloc_ptr[dev]) {
        void* p = nullptr;
        if (cudaGetSymbolAddress(&p, g_noalloc_scratch) != cudaSuccess || !p) return GL_ERR_CUDA;
        g_noalloc_ptr[dev] = p;
    }
    *out = g_noalloc_ptr[dev];
    return GL_OK;
}

extern "C" gl_status gl_logpost_grad_noalloc(const gl_config* cfg, const float* obs, const float* noise_sigma, const float* psf,
                                             const float* params, const int32_t* system_id, int64_t n_particles,
                                             float* out_logp, float* out_grad, void* stream) {
    t_launches = 0;
    if (!cfg) return GL_ERR_NULL;
    if (n_particles < 0) return GL_ERR_BAD_SHAPE;
    if (n_particles > 0 && make_plan(cfg, n_particles).total > GL_NOALLOC_MAX_BYTES) return GL_ERR_NOALLOC_LIMIT;
    void* ws = nullptr;
    if (n_particles > 0) {
        const gl_status s = noalloc_scratch(&ws);
        if (s != GL_OK) return s;
    }
    // Nothing to clear: the path rewrites every workspace element it reads (the caller-workspace form runs on
    // uninitialised memory too).  n_particles == 0 returns GL_OK inside run() before the workspace is looked at.
    return run(cfg, 1, obs, noise_sigma, psf, params, system_id, n_particles, out_logp, out_grad, nullptr,
               ws, GL_NOALLOC_MAX_BYTES, (cudaStream_t)stream);
}

extern "C" gl_status gl_draw_normal(uint64_t seed, uint64_t step, uint32_t stream_id, int64_t n_rows, int32_t n_cols,
                                    float* out, void* stream) {
    t_launches = 0;
    if (n_rows < 0 || n_cols < 0) return GL_ERR_BAD_SHAPE;
    if (stream_id > 255u || n_rows > 0xFFFFFFFFll || n_cols > (1 << 26)) return GL_ERR_BAD_CONFIG;
    if (n_rows == 0 || n_cols == 0) return GL_OK;
    if (!out) return GL_ERR_NULL;
    const int64_t n = n_rows * ((n_cols + 3) / 4);
    clear_stale_error();
    gl_draw_normal_kernel<<<(unsigned)((n + 255) / 256), 256, 0, (cudaStream_t)stream>>>(seed, step, stream_id, n_rows, n_cols, out);
    ++t_launches;
    return cudaPeekAtLastError() == cudaSuccess ? GL_OK : GL_ERR_CUDA;
}

extern "C" gl_status gl_draw_log_uniform(uint64_t seed, uint64_t step, uint32_t stream_id, int64_t n_rows, float* out, void* stream) {
    t_launches = 0;
    if (n_rows < 0) return GL_ERR_BAD_SHAPE;
    if (stream_id > 255u || n_rows > 0xFFFFFFFFll) return GL_ERR_BAD_CONFIG;
    if (n_rows == 0) return GL_OK;
    if (!out) return GL_ERR_NULL;
    clear_stale_error();
    gl_draw_log_uniform_kernel<<<(unsigned)((n_rows + 255) / 256), 256, 0, (cudaStream_t)stream>>>(seed, step, stream_id, n_rows, out);
    ++t_launches;
    return cudaPeekAtLastError() == cudaSuccess ? GL_OK : GL_ERR_CUDA;
}

extern "C" gl_status gl_linear_amplitudes(const gl_config* cfg, const float* obs, const float* noise_sigma, const float* psf,
                                          const float* params, const int32_t* system_id, int64_t n_particles,
                                          float* out_amp, float* out_logp, void* workspace, size_t workspace_bytes, void* stream) {
    if (!cfg) return GL_ERR_NULL;
    if (cfg->desc.amplitude_mode != 1) return GL_ERR_BAD_CONFIG;
    if (n_particles > 0 && !out_amp) return GL_ERR_NULL;
    return run(cfg, 0, obs, noise_sigma, psf, params, system_id, n_particles, out_logp, nullptr, nullptr,
               workspace, workspace_bytes, (cudaStream_t)stream, out_amp);
}

extern "C" gl_status gl_model_image(const gl_config* cfg, const float* psf, const float* params, const int32_t* system_id,
                                    int64_t n_particles, float* out_image, void* workspace, size_t workspace_bytes, void* stream) {
    return run(cfg, 2, nullptr, nullptr, psf, params, system_id, n_particles, nullptr, nullptr, out_image,
               workspace, workspace_bytes, (cudaStream_t)stream);
}

static gl_status check_opt(const gl_opt_desc* opt, int64_t step);
static OptParams opt_params(const gl_opt_desc* opt, int64_t step);
// parameters no optimiser may move: the solved amplitudes of backward modelling (amplitude_mode 1)
static DimMask dead_mask(const gl_config* c) {
    DimMask m{};
    if (c->desc.amplitude_mode == 1)
        for (int i = 0; i < c->L.n_params; ++i) if (is_amp(c->L, i)) m.w[i >> 5] |= 1u << (i & 31);
    return m;
}

extern "C" gl_status gl_map_step(const gl_config* cfg, const gl_opt_desc* opt, const float* obs, const float* noise_sigma,
                                 const float* psf, float* params, const int32_t* system_id, int64_t n_particles,
                                 float* opt_m, float* opt_v, int64_t step, float* out_logp, float* out_grad,
                                 void* workspace, size_t workspace_bytes, void* stream) {
    t_launches = 0;
    if (!cfg) return GL_ERR_NULL;
    { gl_status so = check_opt(opt, step); if (so != GL_OK) return so; }
    if (n_particles < 0) return GL_ERR_BAD_SHAPE;
    if (n_particles == 0) return GL_OK;
    if (!opt_m || !opt_v) return GL_ERR_NULL;
    cudaStream_t st = (cudaStream_t)stream;
    gl_status s = run(cfg, 1, obs, noise_sigma, psf, params, system_id, n_particles, out_logp, out_grad, nullptr,
                      workspace, workspace_bytes, st);
    if (s != GL_OK) return s;
    const OptParams o = opt_params(opt, step);
    const int64_t n_elem = n_particles * cfg->L.n_params;
    gl_opt_update_kernel<<<(unsigned)((n_elem + 255) / 256), 256, 0, st>>>(o, dead_mask(cfg), n_elem, cfg->L.n_params, out_logp, out_grad,
                                                                          params, opt_m, opt_v);
    ++t_launches;
    return cudaPeekAtLastError() == cudaSuccess ? GL_OK : GL_ERR_CUDA;
}

extern "C" gl_status gl_best_particle(const float* logp, int64_t n, int64_t* out_index, float* out_logp, void* stream) {
    t_launches = 0;
    if (n < 0) return GL_ERR_BAD_SHAPE;
    if (!out_index || !out_logp || (n > 0 && !logp)) return GL_ERR_NULL;
    clear_stale_error();
    gl_best_particle_kernel<<<1, 1024, 0, (cudaStream_t)stream>>>(logp, n, out_index, out_logp);
    t_launches = 1;
    return cudaPeekAtLastError() == cudaSuccess ? GL_OK : GL_ERR_CUDA;
}

struct SviPlan { size_t core, off_z, off_lp, off_g, off_part, total; };
static SviPlan svi_plan(const gl_config* c, int64_t n) {
    SviPlan p{};
    const size_t np = (size_t)c->L.n_params, nslot = 2 + np + np * (np + 1) / 2;
    p.core = make_plan(c, n).total;
    size_t o = p.core;
    p.off_z = o;    o = align256(o + sizeof(float) * (size_t)n * np);
    p.off_lp = o;   o = align256(o + sizeof(float) * (size_t)n);
    p.off_g = o;    o = align256(o + sizeof(float) * (size_t)n * np);
    p.off_part = o; o = align256(o + sizeof(double) * SVI_NCHUNK * nslot);
    p.total = o;
    return p;
}

extern "C" size_t gl_svi_workspace_bytes(const gl_config* c, int64_t n) {
    if (!c || n <= 0) return 0;
    return svi_plan(c, n).total;
}

static gl_status check_opt(const gl_opt_desc* opt, int64_t step) {
    if (!opt) return GL_ERR_NULL;
    if (opt->kind != GL_OPT_ADAM && opt->kind != GL_OPT_ADABELIEF) return GL_ERR_BAD_CONFIG;
    if (!(opt->lr > 0.f) || !(opt->b1 >= 0.f && opt->b1 < 1.f) || !(opt->b2 >= 0.f && opt->b2 < 1.f) || !(opt->eps >= 0.f) ||
        !(opt->eps_root >= 0.f) || step < 1)
        return GL_ERR_BAD_CONFIG;
    // an element whose gradient is exactly 0 from step 1 makes the update 0 / (sqrt(0) + eps): the denominator must not vanish
    if (opt->kind == GL_OPT_ADAM ? !(opt->eps > 0.f) : !(opt->eps > 0.f || opt->eps_root > 0.f)) return GL_ERR_BAD_CONFIG;
    return GL_OK;
}
static OptParams opt_params(const gl_opt_desc* opt, int64_t step) {
    OptParams o{};
    o.kind = opt->kind; o.lr = opt->lr; o.b1 = opt->b1; o.b2 = opt->b2; o.eps = opt->eps; o.eps_root = opt->eps_root;
    o.c1 = 1.0 / (1.0 - std::pow(o.b1, (double)step)); o.c2 = 1.0 / (1.0 - std::pow(o.b2, (double)step));
    return o;
}

extern "C" gl_status gl_svi_step(const gl_config* cfg, const gl_opt_desc* opt, const float* obs, const float* noise_sigma,
                                 const float* psf, float* mu, float* l_tril, const float* xi, const int32_t* system_id,
                                 int64_t n, float* opt_m, float* opt_v, int64_t step, float* out_stats,
                                 void* workspace, size_t workspace_bytes, void* stream) {
    t_launches = 0;
    if (!cfg) return GL_ERR_NULL;
    gl_status s = check_opt(opt, step);
    if (s != GL_OK) return s;
    if (n < 0) return GL_ERR_BAD_SHAPE;
    if (n == 0) return GL_OK;
    if (!mu || !l_tril || !xi || !opt_m || !opt_v || !out_stats || !workspace) return GL_ERR_NULL;
    const SviPlan pl = svi_plan(cfg, n);
    if (workspace_bytes < pl.total || ((uintptr_t)workspace & 255) != 0) return GL_ERR_WORKSPACE;
    cudaStream_t st = (cudaStream_t)stream;
    char* w = (char*)workspace;
    float* z = (float*)(w + pl.off_z); float* lp = (float*)(w + pl.off_lp); float* g = (float*)(w + pl.off_g);
    double* part = (double*)(w + pl.off_part);
    const int np = cfg->L.n_params, nslot = 2 + np + np * (np + 1) / 2;
    s = validate(cfg, 1, obs, noise_sigma, psf, z, n, lp, g, nullptr, workspace, pl.core);     // before the first launch
    if (s != GL_OK) return s;
    clear_stale_error();
    gl_svi_draw_kernel<<<(unsigned)((n * np + 255) / 256), 256, 0, st>>>(n, np, mu, l_tril, xi, z);
    s = run(cfg, 1, obs, noise_sigma, psf, z, system_id, n, lp, g, nullptr, workspace, pl.core, st);
    if (s != GL_OK) return s;
    const int64_t launches = t_launches + 1;
    gl_svi_reduce_kernel<<<dim3((nslot + 127) / 128, SVI_NCHUNK), 128, 0, st>>>(n, np, lp, g, xi, part);
    gl_svi_update_kernel<<<1, 256, 0, st>>>(opt_params(opt, step), dead_mask(cfg), np, part, mu, l_tril, opt_m, opt_v, out_stats);
    t_launches = launches + 2;
    return cudaPeekAtLastError() == cudaSuccess ? GL_OK : GL_ERR_CUDA;
}

// Score-function SVI iteration (Eq. 3 as printed): the hot path runs FORWARD ONLY (gl_logpost) on the draws; the gradient of the
// loss w.r.t. (mu, L) comes from log p~ and the surrogate's own score (gl_svi.cuh).  Same workspace as gl_svi_step: the draws'
// buffer holds c_i and three scalars once the hot path has consumed z, the gradient buffer holds the pseudo-gradient rows.
extern "C" gl_status gl_svi_step_score(const gl_config* cfg, const gl_opt_desc* opt, const float* obs, const float* noise_sigma,
                                       const float* psf, float* mu, float* l_tril, const float* xi, const int32_t* system_id,
                                       int64_t n, float* opt_m, float* opt_v, int64_t step, int32_t baseline, float* out_stats,
                                       void* workspace, size_t workspace_bytes, void* stream) {
    t_launches = 0;
    if (!cfg) return GL_ERR_NULL;
    gl_status s = check_opt(opt, step);
    if (s != GL_OK) return s;
    if (baseline != 0 && baseline != 1) return GL_ERR_BAD_CONFIG;
    if (cfg->desc.amplitude_mode == 1) return GL_ERR_UNSUPPORTED;          // surrogate on a subset of the dimensions: pathwise only
    if (n < 0) return GL_ERR_BAD_SHAPE;
    if (n == 0) return GL_OK;
    if (!mu || !l_tril || !xi || !opt_m || !opt_v || !out_stats || !workspace) return GL_ERR_NULL;
    const SviPlan pl = svi_plan(cfg, n);
    if (workspace_bytes < pl.total || ((uintptr_t)workspace & 255) != 0) return GL_ERR_WORKSPACE;
    const int np = cfg->L.n_params, nslot = 2 + np + np * (np + 1) / 2;
    if ((size_t)n * np * sizeof(float) < ((size_t)n + 4) * sizeof(double)) return GL_ERR_UNSUPPORTED;   // n_params < 3
    cudaStream_t st = (cudaStream_t)stream;
    char* w = (char*)workspace;
    float* z = (float*)(w + pl.off_z); float* lp = (float*)(w + pl.off_lp); float* g = (float*)(w + pl.off_g);
    double* part = (double*)(w + pl.off_part);
    s = validate(cfg, 0, obs, noise_sigma, psf, z, n, lp, nullptr, nullptr, workspace, pl.core);     // before the first launch
    if (s != GL_OK) return s;
    clear_stale_error();
    gl_svi_draw_kernel<<<(unsigned)((n * np + 255) / 256), 256, 0, st>>>(n, np, mu, l_tril, xi, z);
    s = run(cfg, 0, obs, noise_sigma, psf, z, system_id, n, lp, nullptr, nullptr, workspace, pl.core, st);
    if (s != GL_OK) return s;
    const int64_t launches = t_launches + 1;
    double* c = (double*)z;                       // z has been consumed: c_i [n], then scal[3]
    double* scal = c + n;
    gl_svi_score_w_kernel<<<(unsigned)((n + 127) / 128), 128, 0, st>>>(n, np, lp, xi, l_tril, c);
    gl_svi_score_c_kernel<<<1, 256, 0, st>>>(n, baseline, c, scal);
    gl_svi_score_grad_kernel<<<(unsigned)((n + 63) / 64), 64, 0, st>>>(n, np, l_tril, xi, c, g);
    gl_svi_reduce_kernel<<<dim3((nslot + 127) / 128, SVI_NCHUNK), 128, 0, st>>>(n, np, lp, g, xi, part);
    gl_svi_update_kernel<<<1, 256, 0, st>>>(opt_params(opt, step), dead_mask(cfg), np, part, mu, l_tril, opt_m, opt_v, out_stats, scal);
    t_launches = launches + 5;
    return cudaPeekAtLastError() == cudaSuccess ? GL_OK : GL_ERR_CUDA;
}

struct HmcPlan { size_t core, off_zd, off_xd, off_zf, off_g, off_lp, total; };
static HmcPlan hmc_plan(const gl_config* c, int64_t n) {
    HmcPlan p{};
    const size_t np = (size_t)c->L.n_params;
    p.core = make_plan(c, n).total;
    size_t o = p.core;
    p.off_zd = o; o = align256(o + sizeof(double) * (size_t)n * np);
    p.off_xd = o; o = align256(o + sizeof(double) * (size_t)n * np);
    p.off_zf = o; o = align256(o + sizeof(float) * (size_t)n * np);
    p.off_g = o;  o = align256(o + sizeof(float) * (size_t)n * np);
    p.off_lp = o; o = align256(o + sizeof(float) * (size_t)n);
    p.total = o;
    return p;
}

extern "C" size_t gl_hmc_workspace_bytes(const gl_config* c, int64_t n) {
    if (!c || n <= 0) return 0;
    return hmc_plan(c, n).total;
}

extern "C" gl_status gl_hmc_step(const gl_config* cfg, const float* obs, const float* noise_sigma, const float* psf,
                                 float* z, float* logp, float* grad, const float* l_tril, const float* xi, const float* log_u,
                                 const int32_t* system_id, int64_t n, float step_size, int32_t n_leapfrog,
                                 int32_t* out_accept, float* out_dh, void* workspace, size_t workspace_bytes, void* stream) {
    t_launches = 0;
    if (!cfg) return GL_ERR_NULL;
    if (!(step_size > 0.f) || !std::isfinite(step_size) || n_leapfrog < 1 || cfg->L.n_params > 128) return GL_ERR_BAD_CONFIG;
    if (n < 0) return GL_ERR_BAD_SHAPE;
    if (n == 0) return GL_OK;
    if (!z || !logp || !grad || !xi || !log_u || !out_accept || !out_dh || !workspace) return GL_ERR_NULL;
    const HmcPlan pl = hmc_plan(cfg, n);
    if (workspace_bytes < pl.total || ((uintptr_t)workspace & 255) != 0) return GL_ERR_WORKSPACE;
    cudaStream_t st = (cudaStream_t)stream;
    char* w = (char*)workspace;
    double* zd = (double*)(w + pl.off_zd); double* xd = (double*)(w + pl.off_xd);
    float* zf = (float*)(w + pl.off_zf); float* g1 = (float*)(w + pl.off_g); float* lp1 = (float*)(w + pl.off_lp);
    const int np = cfg->L.n_params;
    const double eps = (double)step_size;
    {   // before the first launch
        const gl_status sv = validate(cfg, 1, obs, noise_sigma, psf, zf, n, lp1, g1, nullptr, workspace, pl.core);
        if (sv != GL_OK) return sv;
        clear_stale_error();
    }
    int64_t launches = 0;
    for (int s = 0; s < n_leapfrog; ++s) {
        // half kick at the first step, the two half kicks of consecutive steps merged into one full kick afterwards
        gl_hmc_kick_drift_kernel<<<(unsigned)n, 128, 0, st>>>(np, l_tril, s == 0 ? grad : g1, s == 0 ? 0.5 * eps : eps, eps, 1,
                                                             s == 0, z, xi, zd, xd, zf);
        gl_status r = run(cfg, 1, obs, noise_sigma, psf, zf, system_id, n, lp1, g1, nullptr, workspace, pl.core, st);
        if (r != GL_OK) return r;
        launches += 1 + t_launches;
    }
    gl_hmc_kick_drift_kernel<<<(unsigned)n, 128, 0, st>>>(np, l_tril, g1, 0.5 * eps, eps, 0, 0, z, xi, zd, xd, zf);
    gl_hmc_accept_kernel<<<(unsigned)n, 128, 0, st>>>(np, xi, xd, zd, lp1, g1, log_u, z, logp, grad, out_accept, out_dh);
    t_launches = launches + 2;
    return cudaPeekAtLastError() == cudaSuccess ? GL_OK : GL_ERR_CUDA;
}

extern "C" size_t gl_workspace_bytes_host(const gl_config* c, int64_t n) {
    if (!c || n <= 0) return 0;
    const size_t np = (size_t)c->L.n_params;
    return make_plan(c, n).total + align256(sizeof(float) * (size_t)n * np) * 2 + align256(sizeof(float) * (size_t)n);
}

extern "C" gl_status gl_logpost_grad_host(const gl_config* c, const float* obs, const float* noise_sigma, const float* psf,
                                          const float* params_host, const int32_t* system_id, int64_t n,
                                          float* out_logp_host, float* out_grad_host, void* workspace, size_t workspace_bytes,
                                          void* stream) {
    t_launches = 0;
    if (!c) return GL_ERR_NULL;
    if (n < 0) return GL_ERR_BAD_SHAPE;
    if (n == 0) return GL_OK;
    if (!params_host || !out_logp_host || !workspace) return GL_ERR_NULL;
    if (workspace_bytes < gl_workspace_bytes_host(c, n) || ((uintptr_t)workspace & 255) != 0) return GL_ERR_WORKSPACE;
    cudaStream_t st = (cudaStream_t)stream;
    const size_t np = (size_t)c->L.n_params, core = make_plan(c, n).total;
    char* w = (char*)workspace;
    float* d_params = (float*)(w + core);
    float* d_grad = (float*)(w + core + align256(sizeof(float) * n * np));
    float* d_logp = (float*)(w + core + 2 * align256(sizeof(float) * n * np));
    if (cudaMemcpyAsync(d_params, params_host, sizeof(float) * n * np, cudaMemcpyHostToDevice, st) != cudaSuccess) return GL_ERR_CUDA;
    gl_status s = run(c, out_grad_host ? 1 : 0, obs, noise_sigma, psf, d_params, system_id, n, d_logp,
                      out_grad_host ? d_grad : nullptr, nullptr, workspace, core, st);
    if (s != GL_OK) return s;
    if (cudaMemcpyAsync(out_logp_host, d_logp, sizeof(float) * n, cudaMemcpyDeviceToHost, st) != cudaSuccess) return GL_ERR_CUDA;
    if (out_grad_host && cudaMemcpyAsync(out_grad_host, d_grad, sizeof(float) * n * np, cudaMemcpyDeviceToHost, st) != cudaSuccess)
        return GL_ERR_CUDA;
    return GL_OK;
}

// ----------------------------------------------------------------------------- pipe probe (measurement utility)
extern "C" gl_status gl_probe_pipe(int32_t kind, int32_t n_outer, void* workspace, size_t workspace_bytes, void* stream,
                                   double* tera_lane_ops_per_s_host, float* ms_host) {
    if (!workspace || !tera_lane_ops_per_s_host) return GL_ERR_NULL;
    if (kind < 0 || kind > 8 || n_outer < 1) return GL_ERR_BAD_SHAPE;
    if (workspace_bytes < 256) return GL_ERR_WORKSPACE;
    cudaStream_t st = (cudaStream_t)stream;
    int dev = 0, n_sm = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess)
        return GL_ERR_CUDA;
    const int ctas = n_sm * 8, nt = 256;
    cudaEvent_t e0, e1;
    if (cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess) return GL_ERR_CUDA;
    float* sink = (float*)workspace;
    auto launch = [&](int n) {
        switch (kind) {
            case 0: gl_probe_kernel<0><<<ctas, nt, 0, st>>>(n, 1.f, sink); break;
            case 1: gl_probe_kernel<1><<<ctas, nt, 0, st>>>(n, 1.f, sink); break;
            case 2: gl_probe_kernel<2><<<ctas, nt, 0, st>>>(n, 1.f, sink); break;
            case 3: gl_probe_kernel<3><<<ctas, nt, 0, st>>>(n, 1.f, sink); break;
            case 4: gl_probe_kernel<4><<<ctas, nt, 0, st>>>(n, 1.f, sink); break;
            case 5: gl_probe_kernel<5><<<ctas, nt, 0, st>>>(n, 1.f, sink); break;
            case 6: gl_probe_kernel<6><<<ctas, nt, 0, st>>>(n, 1.f, sink); break;
            case 7: gl_probe_kernel<7><<<ctas, nt, 0, st>>>(n, 1.f, sink); break;
            default: gl_probe_kernel<8><<<ctas, nt, 0, st>>>(n, 1.f, sink); break;
        }
    };
    launch(n_outer);                                   // warm-up
    cudaEventRecord(e0, st);
    launch(n_outer);
    cudaEventRecord(e1, st);
    float ms = 0.f;
    cudaError_t e = cudaEventSynchronize(e1);
    if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, e0, e1);
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    if (e != cudaSuccess || !(ms > 0.f)) return GL_ERR_CUDA;
    const double per = kind == 3 ? 2.0 : kind == 5 ? 8.0 : kind == 6 ? 9.0 : 1.0;    // lane-operations per chain step
    const double ops = (double)ctas * nt * (double)n_outer * PROBE_INNER * PROBE_CHAINS * per;
    *tera_lane_ops_per_s_host = ops / (ms * 1e-3) * 1e-12;
    if (ms_host) *ms_host = ms;
    return GL_OK;
}
