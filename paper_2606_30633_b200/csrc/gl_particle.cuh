// gl_particle.cuh -- step A (unpack + bijector + prior) and the per-particle tail of step F (chain rule),
// both in fp64: O(P * n_params) work, negligible next to the per-ray kernels.
#pragma once
#include "gl_common.cuh"

namespace gl {

struct PriorTable {                 // passed by value as a kernel parameter (<= 2.6 KB)
    int32_t kind[128];
    float a[128], b[128], lo[128], hi[128];
};

struct Layout {                     // offsets into the flat parameter vector (reading S18); -1 = absent
    int mass, gamma, ell, shear, mp3, mp4, src, src1, eta2, shp, ll0, ll1, ll2;   // eta2: deflection scale of the 2nd source's plane
    int n_params, n_coef, nmax, param_space, mass_model;
    int ker_nmax;                   // shapelet order the selected kernel variant is compiled for (>= nmax)
    int amp_mode;                   // 1: light amplitudes solved by linear inversion (gl_linear.cuh); their z entries are ignored
};
// Amplitude parameters in the flat order S18: I of each Sersic block, the shapelet coefficients.
__host__ __device__ inline bool is_amp(const Layout& L, int i) {
    return (L.src >= 0 && i == L.src + 6) || (L.src1 >= 0 && i == L.src1 + 6) || (L.ll0 >= 0 && i == L.ll0 + 6) ||
           (L.ll1 >= 0 && i == L.ll1 + 6) || (L.ll2 >= 0 && i == L.ll2 + 6) ||
           (L.shp >= 0 && i > L.shp && i <= L.shp + L.n_coef);
}
// z of parameter i as the kernels see it: a solved amplitude (amp_mode 1) reads as 1 whatever the caller stored
__device__ __forceinline__ double z_in(const Layout& L, const float* __restrict__ z, int i) {
    return (L.amp_mode == 1 && is_amp(L, i)) ? 1.0 : (double)z[i];
}

struct Xform { double theta, lp, logdet, dth_dz, dlp_dth, dlogdet_dz; bool ok; };

__device__ inline double d_softplus(double x) { return x > 0 ? x + log1p(exp(-x)) : log1p(exp(x)); }
__device__ inline double d_sigmoid(double x) { return x >= 0 ? 1.0 / (1.0 + exp(-x)) : exp(x) / (1.0 + exp(x)); }

// O1: theta = T(z), log prior density, log-determinant and their derivatives for one parameter.
__device__ inline Xform transform_one(const PriorTable& pt, int i, int param_space, double z) {
    const double HL2PI = 0.91893853320467274178;
    const int kind = pt.kind[i];
    const double a = pt.a[i], b = pt.b[i], lo = pt.lo[i], hi = pt.hi[i];
    Xform r; r.theta = z; r.logdet = 0; r.dth_dz = 1; r.dlogdet_dz = 0; r.lp = 0; r.dlp_dth = 0; r.ok = true;
    if (param_space == 0) {
        if (kind == 2) { r.theta = exp(z); r.logdet = z; r.dth_dz = r.theta; r.dlogdet_dz = 1; }
        else if (kind == 3 || kind == 4) {
            double s = d_sigmoid(z), w = hi - lo;
            r.theta = lo + w * s; r.logdet = log(w) - d_softplus(-z) - d_softplus(z);
            r.dth_dz = w * s * (1 - s); r.dlogdet_dz = 1 - 2 * s;
        } else if (kind == 5) {
            double s = d_sigmoid(z), w = log(hi) - log(lo), u = log(lo) + w * s;
            r.theta = exp(u); r.logdet = u + log(w) - d_softplus(-z) - d_softplus(z);
            r.dth_dz = r.theta * w * s * (1 - s); r.dlogdet_dz = w * s * (1 - s) + 1 - 2 * s;
        }
    }
    const double th = r.theta;
    if (kind == 1) { double e = (th - a) / b; r.lp = -0.5 * e * e - log(b) - HL2PI; r.dlp_dth = -e / b; }
    else if (kind == 2) {
        if (!(th > 0)) r.ok = false;
        else { double e = (log(th) - a) / b; r.lp = -0.5 * e * e - log(b) - HL2PI - log(th); r.dlp_dth = -e / (b * th) - 1 / th; }
    } else if (kind == 3) {
        if (th < lo || th > hi) r.ok = false; else r.lp = -log(hi - lo);
    } else if (kind == 4) {
        if (th < lo || th > hi) r.ok = false;
        else {
            double e = (th - a) / b;
            double Z = 0.5 * erfc(-((hi - a) / b) * 0.70710678118654752440) - 0.5 * erfc(-((lo - a) / b) * 0.70710678118654752440);
            r.lp = -0.5 * e * e - log(b) - HL2PI - log(Z); r.dlp_dth = -e / b;
        }
    } else if (kind == 5) {
        if (th < lo || th > hi) r.ok = false; else { r.lp = -log(th) - log(log(hi) - log(lo)); r.dlp_dth = -1 / th; }
    }
    if (!isfinite(z) || !isfinite(r.theta)) r.ok = false;
    return r;
}

struct Ell { double c, q, phi, cphi, sphi; };
__device__ inline Ell make_ell(double e1, double e2) {
    Ell E; E.c = sqrt(e1 * e1 + e2 * e2); E.phi = 0.5 * atan2(e2, e1); E.q = (1 - E.c) / (1 + E.c);
    sincos(E.phi, &E.sphi, &E.cphi); return E;
}
// (d/dq, d/dphi) -> (d/de1, d/de2); zero for c < 1e-10 (O9)
__device__ inline void ell_chain(double e1, double e2, const Ell& E, double dq, double dphi, double& de1, double& de2) {
    if (E.c < 1e-10) { de1 = 0; de2 = 0; return; }
    double dq_dc = -2.0 / ((1 + E.c) * (1 + E.c));
    de1 = dq * dq_dc * e1 / E.c + dphi * (-e2 / (2 * E.c * E.c));
    de2 = dq * dq_dc * e2 / E.c + dphi * (e1 / (2 * E.c * E.c));
}

// theta of parameter i from the warp's cache th[] (filled once per particle by the lanes in parallel: transform_one is
// a few hundred fp64 instructions, and the serial per-particle code below used to call it 2-3 times per parameter)
__device__ __forceinline__ double theta_at(const double* __restrict__ th, int i) { return th[i]; }

// Write one Sersic block [R, n, e1, e2, x0, y0, Ie] into PB; a negative `off` writes a neutral (Ie = 0) block.
template <class T>
__device__ inline void write_sersic(const double* __restrict__ th, int off, T* sb, double x_first, bool& ok) {
    double R = 1, n = 1, e1 = 0, e2 = 0, x0 = 0, y0 = 0, Ie = 0;
    if (off >= 0) {
        R = theta_at(th, off); n = theta_at(th, off + 1);
        e1 = theta_at(th, off + 2); e2 = theta_at(th, off + 3);
        x0 = theta_at(th, off + 4); y0 = theta_at(th, off + 5);
        Ie = theta_at(th, off + 6);
        if (!(R > 0) || !(n > 0) || !(e1 * e1 + e2 * e2 < 1.0)) { ok = false; R = 1; n = 1; e1 = e2 = 0; }
    }
    Ell E = make_ell(e1, e2);
    double bn = 1.9992 * n - 0.3271;
    sb[SB_XOFF] = (T)(x_first - x0); sb[SB_YOFF] = (T)(x_first - y0);
    const double sq = sqrt(E.q);
    sb[SB_C] = (T)E.cphi; sb[SB_S] = (T)E.sphi;
    sb[SB_A11] = (T)(sq * E.cphi); sb[SB_A12] = (T)(sq * E.sphi); sb[SB_A21] = (T)(-E.sphi / sq); sb[SB_A22] = (T)(E.cphi / sq);
    sb[SB_K1] = (T)(0.5 / n); sb[SB_K0] = (T)(-log2(R) / n);
    sb[SB_C1] = (T)(bn * 1.44269504088896340736); sb[SB_IE] = (T)Ie;
    sb[SB_KQ] = (T)(bn / n * sq); sb[SB_KQI] = (T)(bn / n / sq);
    sb[14] = sb[15] = T(0);
}

// Step A.  One WARP per particle (4 per CTA): the lanes transform the parameters in parallel into a shared-memory cache,
// lane 0 derives the per-particle scalars into a shared-memory PB row, all lanes copy the row out (coalesced).
// pb: [P][PB_STRIDE]; lpd: [P] = sum log prior + sum log-det (fp64, fixed-order lane tree).
// Terms of the EPL series below this size relative to the sum are dropped (fp64 mode).  The fp32 band of the series already
// contributes a rounding error of 1e-7 * 1e-4 = 1e-11 relative to the sum (knuth_banded in gl_ray.cuh); terms below 1e-12 are
// an order under that, so dropping them leaves the error budget of the series where it was (the parity margins of all
// configurations are unchanged to the printed digits) -- round 1 dropped only what is below the fp64 rounding, 3e-16, and paid one
// more group of four fp32 recurrence steps per polynomial for it (config 2: 12.34 -> 12.07 ms).
#ifndef GL_SERIES_DROP
#define GL_SERIES_DROP 1e-12
#endif
constexpr int UNPACK_WPB = 4;
template <class T>
__global__ void __launch_bounds__(UNPACK_WPB * 32) gl_unpack_kernel(const __grid_constant__ PriorTable pt, const __grid_constant__ Layout L,
                                 const __grid_constant__ Geom G, float pix_scale,
                                 const float* __restrict__ params, int64_t P, T* __restrict__ pb, double* __restrict__ lpd) {
    __shared__ double s_th[UNPACK_WPB][128];
    __shared__ __align__(16) T s_pb[UNPACK_WPB][PB_STRIDE];
    const int wib = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int64_t p = (int64_t)blockIdx.x * UNPACK_WPB + wib;
    if (p >= P) return;                                           // warp-uniform
    const float* z = params + p * L.n_params;
    double* th = s_th[wib];
    T* o = s_pb[wib];
    bool ok = true;
    double lp = 0;
    for (int i = lane; i < L.n_params; i += 32) {
        Xform x = transform_one(pt, i, L.param_space, z_in(L, z, i));
        ok = ok && x.ok; lp += x.lp + x.logdet; th[i] = x.theta;
    }
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) lp += __shfl_xor_sync(0xffffffffu, lp, d);
    ok = __all_sync(0xffffffffu, ok);
    for (int k = lane; k < PB_STRIDE; k += 32) o[k] = T(0);
    __syncwarp();
    // The derived scalars are independent per component: lanes 0-4 take one Sersic block each (absent blocks get the neutral
    // block), lane 5 the main deflector, shear, multipoles and grid, every lane a share of the shapelet coefficients and
    // ONE term of the series (ratios in parallel, running product / sum by a shuffle scan): a serial lane-0 version spent
    // ~35 us per call on dependent fp64 divisions and libdevice calls, most of the latency of a small batch.
    const double x_first = 0.0;   // ray coordinates are x_j = (j - (M-1)/2) * step about the grid centre: offsets are -x0
    {
        const int blk_off[5] = {L.src, L.ll0, L.ll1, L.src1, L.ll2};
        const int blk_pb[5] = {PB_SRC, PB_LL0, PB_LL1, PB_SRC1, PB_LL2};
        if (lane < 5) write_sersic<T>(th, blk_off[lane], o + blk_pb[lane], x_first, ok);
        if (lane == 3) o[PB_SRC1 + SB_ETA] = L.eta2 >= 0 ? (T)theta_at(th, L.eta2) : T(1);
    }
    double t = L.gamma >= 0 ? theta_at(th, L.gamma) - 1.0 : 1.0;
    double e1 = theta_at(th, L.ell), e2 = theta_at(th, L.ell + 1), thE = theta_at(th, L.mass);
    if (!(thE > 0) || !(t > 0 && t < 2) || !(e1 * e1 + e2 * e2 < 1.0)) { ok = false; thE = 1; t = 1; e1 = e2 = 0; }
    if (lane == 5) {
        const double step = (double)pix_scale / G.s;
        const double x0 = theta_at(th, L.ell + 2), y0 = theta_at(th, L.ell + 3);
        Ell E = make_ell(e1, e2);
        double b = thE * sqrt(E.q), f = (1 - E.q) / (1 + E.q);
        o[PB_M_XOFF] = (T)(x_first - x0); o[PB_M_YOFF] = (T)(x_first - y0);
        o[PB_M_C] = (T)E.cphi; o[PB_M_S] = (T)E.sphi; o[PB_M_Q] = (T)E.q; o[PB_M_B] = (T)b;
        o[PB_M_T] = (T)t; o[PB_M_F] = (T)f; o[PB_M_L2B] = (T)log2(b); o[PB_M_A] = (T)(2 * b / (1 + E.q));
        double qp = sqrt(fmax(1 - E.q * E.q, 0.0));
        o[PB_M_QP] = (T)qp; o[PB_M_BQP] = (T)(qp > 0 ? b / qp : 0.0);
        o[PB_M_F2] = (T)(f * f); o[PB_M_TM1] = (T)(t - 1);
        {   // kappa = KAPC * amp / R with amp = A (b/R)^(t-1) (the amplitude the ray kernels form in one exp2, PB_M_H1 / _H0)
            const double A = 2 * b / (1 + E.q);
            o[PB_M_KAPC] = (T)(0.5 * (2 - t) * b / A);
            o[PB_M_H1] = (T)(-0.5 * (t - 1)); o[PB_M_H0] = (T)((t - 1) * log2(b) + log2(A));
        }
        o[PB_G1] = L.shear >= 0 ? (T)theta_at(th, L.shear) : T(0);
        o[PB_G2] = L.shear >= 0 ? (T)theta_at(th, L.shear + 1) : T(0);
        o[PB_C3] = L.mp3 >= 0 ? (T)theta_at(th, L.mp3) : T(0);
        o[PB_S3] = L.mp3 >= 0 ? (T)theta_at(th, L.mp3 + 1) : T(0);
        o[PB_C4] = L.mp4 >= 0 ? (T)theta_at(th, L.mp4) : T(0);
        o[PB_S4] = L.mp4 >= 0 ? (T)theta_at(th, L.mp4 + 1) : T(0);
        o[PB_XFIRST] = (T)x_first; o[PB_STEP] = (T)step;
        if (L.mass_model == 1) {
            // precision bands of the series (knuth_banded in gl_ray.cuh): smallest k with 30 f^k below the threshold
            const double lf = f > 0 ? log(f) : -1e30;
            auto first_below = [&](double thr) { double k = ceil(log(thr / 30.0) / lf); return k < 1 ? 1 : (k > 64 ? 64 : (int)k); };
            const bool dbl = sizeof(T) == 8;
            const int k_top = first_below(dbl ? GL_SERIES_DROP : 3e-9) - 1;      // keep terms k <= kt, kt >= k_top
            const int k_dp = dbl ? first_below(1e-4) - 1 : k_top;       // fp32 steps only above 4 M1 >= k_dp (fp64 mode)
            int mt = (k_top - 1 + 3) / 4; if (mt < 1) mt = 1; if (mt > 7) mt = 7;
            int m1 = (k_dp + 3) / 4; if (m1 < 1) m1 = 1; if (m1 > mt) m1 = mt;
            o[PB_SER_M1] = (T)m1; o[PB_SER_M2] = (T)(mt - m1);
        }
    }
    // shapelets (coefficients pre-divided by beta_s and multiplied by the basis scale c_n1 c_n2 of gl_ray.cuh; orders above
    // the configured nmax are zero)
    if (L.ker_nmax >= 0) {
        double bs = 1.0;
        if (L.shp >= 0) { bs = theta_at(th, L.shp); if (!(bs > 0)) { ok = false; bs = 1; } }
        const double ibs = 1.0 / bs;
        if (lane == 6) { o[PB_SHP] = (T)ibs; o[PB_SHP + 1] = o[PB_SHP + 2] = o[PB_SHP + 3] = T(0); }
        const int nck = (L.ker_nmax + 1) * (L.ker_nmax + 2) / 2;
        for (int k = lane; k < nck; k += 32)
            o[PB_SHP_A + k] = (L.shp >= 0 && k < L.n_coef) ? (T)(theta_at(th, L.shp + 1 + k) * ibs * shp_scale(k)) : T(0);
    }
    // EPL series coefficients: a_n = prod_{k<=n} (2k-2+t)/(2k+2-t); d_m = (m+1) a_{m+1}; e_m = L_{m+1} a_{m+1}, with
    // L_n = sum_{k<=n} 4k/((2k+2-t)(2k-2+t)).  Lane n holds term n: inclusive scans over the lanes give a_n and L_n.
    if (L.mass_model == 1) {
        const double n = (double)lane;
        double an = lane == 0 ? 1.0 : (2.0 * n - 2.0 + t) / (2.0 * n + 2.0 - t);
        double Ln = lane == 0 ? 0.0 : 4.0 * n / ((2.0 * n + 2.0 - t) * (2.0 * n - 2.0 + t));
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            const double pa_ = __shfl_up_sync(0xffffffffu, an, d), pl_ = __shfl_up_sync(0xffffffffu, Ln, d);
            if (lane >= d) { an *= pa_; Ln += pl_; }
        }
        const bool keep = lane < G.n_terms;
        o[PB_SER_A + lane] = keep ? (T)an : T(0);
        if (lane >= 1) {
            o[PB_SER_D + lane - 1] = keep ? (T)(n * an) : T(0);
            o[PB_SER_E + lane - 1] = keep ? (T)(Ln * an) : T(0);
        } else { o[PB_SER_D + 31] = T(0); o[PB_SER_E + 31] = T(0); }
    }
    ok = __all_sync(0xffffffffu, ok);
    if (!isfinite(lp)) ok = false;
    if (lane == 0) { o[PB_VALID] = ok ? T(1) : T(0); lpd[p] = lp; }
    __syncwarp();
    T* dst = pb + p * PB_STRIDE;
    for (int k = lane; k < PB_STRIDE; k += 32) dst[k] = o[k];
}

// Chain rule for one Sersic block: natural sums T -> d logL / d[R, n, e1, e2, x0, y0, Ie], written to gth[off..off+6].
__device__ inline void sersic_chain(const double* __restrict__ th, int off, const double* T, double* gth) {
    double R = theta_at(th, off), n = theta_at(th, off + 1);
    double e1 = theta_at(th, off + 2), e2 = theta_at(th, off + 3), Ie = theta_at(th, off + 6);
    Ell E = make_ell(e1, e2);
    double bn = 1.9992 * n - 0.3271, k = bn / n;
    gth[off + 6] = T[SA_T0] / Ie;
    gth[off] = k * T[SA_T1] / R;
    gth[off + 1] = -1.9992 * (T[SA_T1] - T[SA_T0]) + bn * 0.69314718055994530942 * T[SA_T2] / n;
    // the sums were taken in the pre-scaled frame x' = sqrt(q) x_r, y' = y_r / sqrt(q) (gl_common.cuh): unscale here
    const double sq = sqrt(E.q);
    double gxr = -k * sq * T[SA_AX], gyr = -k * T[SA_AY] / sq;
    gth[off + 4] = -(E.cphi * gxr - E.sphi * gyr);
    gth[off + 5] = -(E.sphi * gxr + E.cphi * gyr);
    double dq = -k * 0.5 * (T[SA_BXX] - T[SA_BYY]) / E.q;
    double dphi = -k * (E.q - 1.0 / E.q) * T[SA_BXY];
    ell_chain(e1, e2, E, dq, dphi, gth[off + 2], gth[off + 3]);
}

// Tail of step E/F.  One WARP per particle.  Sums the per-tile chi^2 partials and the per-chunk natural
// accumulators in a fixed order (fp64), applies the chain rule natural -> theta -> z, adds prior and
// log-det terms, and writes out_logp / out_grad.  nap may be NULL (gl_logpost: no gradient).
template <class T>
__global__ void gl_finalize_kernel(const __grid_constant__ PriorTable pt, const __grid_constant__ Layout L,
                                   const __grid_constant__ Geom G,
                                   const float* __restrict__ params, const T* __restrict__ pb,
                                   const double* __restrict__ lpd, const T* __restrict__ chi, int n_ctile,
                                   const T* __restrict__ nap, int n_chunk, int na,
                                   const double* __restrict__ sys_sumlog, const int32_t* __restrict__ system_id,
                                   int64_t P, int64_t p_base, float* __restrict__ out_logp, float* __restrict__ out_grad) {
    extern __shared__ double fsm[];                     // per warp: nat[NA_MAX] + gth[128] + th[128]
    const int wib = threadIdx.x >> 5, lane = threadIdx.x & 31;
    int64_t p = (int64_t)blockIdx.x * (blockDim.x >> 5) + wib;
    if (p >= P) return;
    double* nat = fsm + (size_t)wib * (NA_MAX + 256);
    double* gth = nat + NA_MAX;
    double* th = gth + 128;                             // theta cache (see theta_at)
    const float* z = params + (p_base + p) * L.n_params;
    const bool valid = pb[p * PB_STRIDE + PB_VALID] != T(0);
    // chi^2: lanes stride over tiles, then a fixed xor-tree
    double c2 = 0;
    for (int k = lane; k < n_ctile; k += 32) c2 += (double)chi[p * n_ctile + k];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) c2 += __shfl_xor_sync(0xffffffffu, c2, o);
    const int sys = system_id ? system_id[p_base + p] : 0;
    double logp = -0.5 * c2 - sys_sumlog[sys] - 0.5 * G.N * G.N * 1.83787706640934548356 + lpd[p];
    bool good = valid && isfinite(logp);
    if (nap) {
        for (int k = lane; k < na; k += 32) {
            double s = 0;
            for (int ch = 0; ch < n_chunk; ++ch) s += (double)nap[((size_t)p * n_chunk + ch) * na + k];
            nat[k] = s;
        }
        for (int k = lane; k < L.n_params; k += 32) { gth[k] = 0; th[k] = transform_one(pt, k, L.param_space, z_in(L, z, k)).theta; }
        __syncwarp();
        // chain rule natural -> theta, one component per lane: lane 0 the mass block, shear and multipoles, lanes 1-5 one
        // Sersic block each; the shapelet terms that add to the first source's centre follow after a warp barrier
        if (lane == 0 && valid) {
            double thE = theta_at(th, L.mass);
            double t = L.gamma >= 0 ? theta_at(th, L.gamma) - 1.0 : 1.0;
            double e1 = theta_at(th, L.ell), e2 = theta_at(th, L.ell + 1);
            Ell E = make_ell(e1, e2);
            double q = E.q, b = thE * sqrt(q);
            double dL_db = -(t / b) * nat[NA_D0];
            double dL_dq_b;
            if (L.mass_model == 1) {
                gth[L.gamma] = -(0.69314718055994530942 * nat[NA_DTL] + nat[NA_DT2]);
                dL_dq_b = -(-nat[NA_D0] / (1 + q) - (t - 1) * q * nat[NA_D1] - nat[NA_D2] - 2.0 / ((1 + q) * (1 + q)) * nat[NA_D3]);
            } else {
                dL_dq_b = -nat[NA_DQS];
            }
            gth[L.mass] = dL_db * sqrt(q);
            double dq = dL_dq_b + dL_db * thE / (2 * sqrt(q));
            double dphi = -nat[NA_DPHI];
            ell_chain(e1, e2, E, dq, dphi, gth[L.ell], gth[L.ell + 1]);
            gth[L.ell + 2] = E.cphi * nat[NA_VX] - E.sphi * nat[NA_VY];
            gth[L.ell + 3] = E.sphi * nat[NA_VX] + E.cphi * nat[NA_VY];
            if (L.shear >= 0) { gth[L.shear] = nat[NA_G1]; gth[L.shear + 1] = nat[NA_G2]; }
            if (L.mp3 >= 0) { gth[L.mp3] = nat[NA_C3]; gth[L.mp3 + 1] = nat[NA_S3]; }
            if (L.mp4 >= 0) { gth[L.mp4] = nat[NA_C4]; gth[L.mp4 + 1] = nat[NA_S4]; }
            if (L.mp3 >= 0 || L.mp4 >= 0) { gth[L.ell + 2] += nat[NA_MCX]; gth[L.ell + 3] += nat[NA_MCY]; }
            if (L.eta2 >= 0) gth[L.eta2] = nat[NA_ETA];
        }
        if (lane >= 1 && lane <= 5 && valid) {
            const int blk_off[5] = {L.src, L.ll0, L.ll1, L.src1, L.ll2};
            const int blk_na[5] = {NA_SRC, NA_LL0, NA_LL1, NA_SRC1, NA_LL2};
            if (blk_off[lane - 1] >= 0) sersic_chain(th, blk_off[lane - 1], nat + blk_na[lane - 1], gth);
        }
        __syncwarp();
        if (lane == 0 && valid && L.shp >= 0) {
            double bs = theta_at(th, L.shp);
            gth[L.shp] = -nat[NA_SHB] / bs;
            gth[L.src + 4] -= nat[NA_SHX]; gth[L.src + 5] -= nat[NA_SHY];
        }
        __syncwarp();
        if (L.shp >= 0 && valid) {
            double bs = theta_at(th, L.shp);
            for (int k = lane; k < L.n_coef; k += 32) gth[L.shp + 1 + k] = nat[NA_SHA + k] * shp_scale(k) / bs;   // sums taken in the scaled basis
        }
        __syncwarp();
        // theta -> z, priors, log-det; a non-finite component invalidates the particle
        bool fin = true;
        for (int k = lane; k < L.n_params; k += 32) {
            Xform x = transform_one(pt, k, L.param_space, z_in(L, z, k));
            double g = (gth[k] + x.dlp_dth) * x.dth_dz + x.dlogdet_dz;
            if (L.amp_mode == 1 && is_amp(L, k)) g = 0;           // dL/da = 0 at the solved amplitudes (envelope theorem, S21)
            gth[k] = g; if (!isfinite(g)) fin = false;
        }
        fin = __all_sync(0xffffffffu, fin);
        good = good && fin;
        __syncwarp();
        for (int k = lane; k < L.n_params; k += 32)
            out_grad[(p_base + p) * L.n_params + k] = good ? (float)gth[k] : 0.f;
    }
    if (lane == 0) out_logp[p_base + p] = good ? (float)logp : -INFINITY;
}

// arg max over the particles (largest finite logp, lowest index on ties).  ONE block of 1024 threads:
// each thread scans a strided subset keeping (value, index), then a fixed tree in shared memory.
__global__ void __launch_bounds__(1024) gl_best_particle_kernel(const float* __restrict__ logp, int64_t n,
                                                                int64_t* __restrict__ out_index, float* __restrict__ out_logp) {
    __shared__ float sv[1024];
    __shared__ int64_t si[1024];
    float bv = -INFINITY; int64_t bi = -1;
    for (int64_t i = threadIdx.x; i < n; i += 1024) {
        const float v = logp[i];
        if (isfinite(v) && (bi < 0 || v > bv)) { bv = v; bi = i; }        // strided scan: indices increase, '>' keeps the first
    }
    sv[threadIdx.x] = bv; si[threadIdx.x] = bi;
    __syncthreads();
    for (int o = 512; o > 0; o >>= 1) {
        if (threadIdx.x < o) {
            const float v2 = sv[threadIdx.x + o]; const int64_t i2 = si[threadIdx.x + o];
            const float v1 = sv[threadIdx.x]; const int64_t i1 = si[threadIdx.x];
            const bool take = i2 >= 0 && (i1 < 0 || v2 > v1 || (v2 == v1 && i2 < i1));
            if (take) { sv[threadIdx.x] = v2; si[threadIdx.x] = i2; }
        }
        __syncthreads();
    }
    if (threadIdx.x == 0) { out_index[0] = si[0]; out_logp[0] = si[0] >= 0 ? sv[0] : -INFINITY; }
}

// Adam / AdaBelief update of every (particle, parameter), fp64 arithmetic on fp32 storage.
// One thread per element; a particle with a non-finite log-posterior or gradient row is left untouched (the
// gradient row of such a particle is all zero by construction of gl_finalize_kernel, its logp is -INF).
struct OptParams { int kind; double lr, b1, b2, eps, eps_root, c1, c2; };   // c1 = 1/(1-b1^t), c2 = 1/(1-b2^t)
// One bit per parameter (n_params <= 128): the solved amplitudes of backward modelling, which no optimiser may move.
struct DimMask {
    uint32_t w[4];
    __host__ __device__ bool test(int i) const { return (w[i >> 5] >> (i & 31)) & 1u; }
    __host__ __device__ int count(int n) const { int c = 0; for (int i = 0; i < n; ++i) c += test(i); return c; }
};

__global__ void gl_opt_update_kernel(const __grid_constant__ OptParams o, const __grid_constant__ DimMask dead, int64_t n_elem, int n_params,
                                     const float* __restrict__ logp, const float* __restrict__ grad,
                                     float* __restrict__ z, float* __restrict__ m, float* __restrict__ v) {
    const int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= n_elem) return;
    const int64_t p = e / n_params;
    if (dead.test((int)(e - p * n_params))) return;               // a solved amplitude: ignored on input, never updated
    const float lp = logp[p];
    const double g = -(double)grad[e];
    if (!isfinite(lp) || !isfinite(g)) return;
    const double m1 = o.b1 * (double)m[e] + (1.0 - o.b1) * g;
    const double d = o.kind == 1 ? g - m1 : g;
    const double v1 = o.b2 * (double)v[e] + (1.0 - o.b2) * d * d + (o.kind == 1 ? o.eps_root : 0.0);
    const double z1 = (double)z[e] - o.lr * (m1 * o.c1) / (sqrt(v1 * o.c2) + o.eps);
    m[e] = (float)m1; v[e] = (float)v1; z[e] = (float)z1;
}

}  // namespace gl
