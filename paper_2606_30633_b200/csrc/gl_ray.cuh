// gl_ray.cuh -- steps B + C (ray-trace + paint light) and the per-ray part of step F (adjoint).
//
// One CTA = one chunk of rays of one phase plane of ONE particle; the particle's derived scalars (PB) are staged in
// shared memory once per CTA and every per-ray quantity lives in registers.  Arithmetic type T = double (default mode:
// FP64 FMA pipe, MUFU results only as Newton seeds) or float (FP32 FMA pipe + MUFU rsqrt / lg2 / ex2 / rcp), see
// gl_math.cuh.  The 30-term EPL series (BASELINE.json configs[1]; reading S5) is a real-
// coefficient polynomial in w = -f e^{2 i phi}; because |w|^2 = f^2 is a per-particle constant it is
// evaluated by synthetic division by (x - w)(x - conj w) = x^2 - p x + f^2, p = 2 Re w:
//     b_k = a_k + p b_{k+1} - f^2 b_{k+2},   P(w) = b_1 w + (a_0 - f^2 b_2)
// i.e. 2 FMAs per term instead of the 4 of complex Horner; the recurrence is contractive for f < 1.
#pragma once
#include "gl_common.cuh"
#include "gl_math.cuh"
#include <type_traits>

namespace gl {


// Shapelet basis in the SCALED form psi_k = phi_k / c_k, c_k = sqrt(2^k / k!) (c_{k+1} = sqrt(2/(k+1)) c_k): the orthonormal
// Gauss-Hermite functions phi_{k+1} = sqrt(2/(k+1)) u phi_k - sqrt(k/(k+1)) phi_{k-1} become
//     psi_{k+1} = u psi_k - (k/2) psi_{k-1}          (2 operations per step instead of 3),
//     psi_k'    = (k/2) psi_{k-1} - psi_{k+1}        (1 operation: the product is the recurrence's own).
// The factors c_n1 c_n2 are per-coefficient constants: gl_unpack_kernel folds them into the coefficients in PB, and
// gl_finalize_kernel into the coefficient sums (shp_scale).  In fp64 the two Gaussians of phi_n1(u) phi_n2(v) are ONE
// exp2 of u^2 + v^2 carried by the u family (the v family is then the bare polynomial); fp32 keeps one Gaussian per
// family so that the polynomial cannot overflow where the Gaussian has already underflowed.
// (d_HC, shp_scale: gl_common.cuh)

// P(w) = sum_{k<=TOP} cf[k] w^k for real coefficients cf (shared memory, zero beyond the kept terms).
template <class T, int TOP>
__device__ __forceinline__ void knuth(const T* __restrict__ cf, T p, T nf2, T wr, T wi, T& Pr, T& Pi) {
    using R = Real<T>;
    T b1 = cf[TOP], b2 = T(0.);
#pragma unroll
    for (int k = TOP - 1; k >= 1; --k) {
        T bk = R::fma(p, b1, R::fma(nf2, b2, cf[k]));
        b2 = b1; b1 = bk;
    }
    T r0 = R::fma(nf2, b2, cf[0]);
    Pr = R::fma(b1, wr, r0); Pi = b1 * wi;
}

// K real-coefficient polynomials in the same w at once, in precision bands (all bounds are per-particle, hence
// CTA-uniform: no divergence).  Term k of the series is O(f^k) relative to the sum, so (gl_unpack_kernel picks M1, M2):
//   k > kt = 4(M1+M2)+1      dropped: 30 f^(kt+1) <= 1e-12 (fp64 mode, GL_SERIES_DROP) -- an order below the fp32 band's rounding;
//   4 M1 < k <= kt           recurrence steps in fp32 on the otherwise idle FP32 pipe: their rounding enters the sum
//                            scaled by f^k, 30 f^(4 M1 + 1) 1e-7 <= 1e-11;
//   k <= 4 M1                recurrence steps in T.
// cf: K coefficient arrays of T, cf32: fp32 copies (fp64 mode only); both in the SHIFTED shared-memory layout written by
// stage_series: coefficient idx of polynomial i sits at [SER_PITCH * i + idx + 3], so that the four coefficients
// k-3 .. k of one 4-step group (k a multiple of 4) are one aligned 16-byte (fp32) or two aligned 16-byte (fp64) loads.
constexpr int SER_PITCH = 36;

__device__ __forceinline__ void load_coef4(const float* __restrict__ c, int k, float (&v)[4]) {   // v[j] = coef[k - j]
    const float4 x = *reinterpret_cast<const float4*>(c + k);
    v[0] = x.w; v[1] = x.z; v[2] = x.y; v[3] = x.x;
}
__device__ __forceinline__ void load_coef4(const double* __restrict__ c, int k, double (&v)[4]) {
    const double2 lo = *reinterpret_cast<const double2*>(c + k), hi = *reinterpret_cast<const double2*>(c + k + 2);
    v[0] = hi.y; v[1] = hi.x; v[2] = lo.y; v[3] = lo.x;
}

// Stage the K_ALL = 3 coefficient arrays of a particle (PB_SER_A / _D / _E, stride 32 in PB) into the shifted layout.
template <class T>
__device__ __forceinline__ void stage_series(const T* __restrict__ src, T* __restrict__ cfs, float* __restrict__ cf32) {
    for (int e = threadIdx.x; e < 3 * SER_PITCH; e += blockDim.x) {
        const int i = e / SER_PITCH, pos = e - i * SER_PITCH, idx = pos - 3;
        const T v = (idx >= 0 && idx < 32) ? src[PB_SER_A + 32 * i + idx] : T(0.);
        cfs[e] = v;
        if constexpr (sizeof(T) == 8) cf32[e] = (float)v;
    }
}

// G groups of 4 recurrence steps, fully unrolled (G is a compile-time count: no loop control, immediate load offsets).
// c points at the shifted coefficient array position of index k_hi - 3 ... i.e. coefficient idx sits at c[idx + 3];
// the groups use indices k_hi, k_hi - 1, ..., k_hi - 4 G + 1 with k_hi a multiple of 4 (passed through the pointer).
template <class S, int K, int G>
__device__ __forceinline__ void knuth_groups(const S* __restrict__ c_at_khi, S p, S nf2, S (&b1)[K], S (&b2)[K]) {
#pragma unroll
    for (int g = 0; g < G; ++g) {
        S v[K][4];
#pragma unroll
        for (int i = 0; i < K; ++i) load_coef4(c_at_khi + SER_PITCH * i, -4 * g, v[i]);
#pragma unroll
        for (int j = 0; j < 4; ++j) {
#pragma unroll
            for (int i = 0; i < K; ++i) {
                S bk;
                if constexpr (sizeof(S) == 8) bk = fma(p, b1[i], fma(nf2, b2[i], v[i][j]));
                else bk = fmaf(p, b1[i], fmaf(nf2, b2[i], v[i][j]));
                b2[i] = b1[i]; b1[i] = bk;
            }
        }
    }
}
// run-time group count 0..7 -> the unrolled instance (one CTA-uniform switch per polynomial set instead of a loop)
// UNR = false: a plain loop over the groups instead (smaller code: measured better for the shapelet variants and for
// the fp32 adjoint, whose register budgets are tight).
template <class S, int K, bool UNR>
__device__ __forceinline__ void knuth_groups_n(int n, const S* __restrict__ c_base, int k_hi, S p, S nf2, S (&b1)[K], S (&b2)[K]) {
    const S* c_at_khi = c_base + k_hi;
    if constexpr (!UNR) {
        int k = k_hi;                                              // index form of the plain loop (measured faster than pointer steps)
        for (int g = 0; g < n; ++g, k -= 4) {
            S v[K][4];
#pragma unroll
            for (int i = 0; i < K; ++i) load_coef4(c_base + SER_PITCH * i, k, v[i]);
#pragma unroll
            for (int j = 0; j < 4; ++j) {
#pragma unroll
                for (int i = 0; i < K; ++i) {
                    S bk;
                    if constexpr (sizeof(S) == 8) bk = fma(p, b1[i], fma(nf2, b2[i], v[i][j]));
                    else bk = fmaf(p, b1[i], fmaf(nf2, b2[i], v[i][j]));
                    b2[i] = b1[i]; b1[i] = bk;
                }
            }
        }
        return;
    }
    switch (n) {
        case 1: knuth_groups<S, K, 1>(c_at_khi, p, nf2, b1, b2); break;
        case 2: knuth_groups<S, K, 2>(c_at_khi, p, nf2, b1, b2); break;
        case 3: knuth_groups<S, K, 3>(c_at_khi, p, nf2, b1, b2); break;
        case 4: knuth_groups<S, K, 4>(c_at_khi, p, nf2, b1, b2); break;
        case 5: knuth_groups<S, K, 5>(c_at_khi, p, nf2, b1, b2); break;
        case 6: knuth_groups<S, K, 6>(c_at_khi, p, nf2, b1, b2); break;
        case 7: knuth_groups<S, K, 7>(c_at_khi, p, nf2, b1, b2); break;
        default: break;
    }
}

template <class T, int K, bool UNR>
__device__ __forceinline__ void knuth_banded(const T* __restrict__ cf, const float* __restrict__ cf32, int m1, int m2,
                                             T p, T nf2, T wr, T wi, T (&Pr)[K], T (&Pi)[K]) {
    using R = Real<T>;
    T b1[K], b2[K];
    const int kt = 4 * (m1 + m2) + 1;
    bool seeded = false;
    if constexpr (sizeof(T) == 8) {
        if (m2 > 0) {
            const float pf = (float)p, nf = (float)nf2;
            float c1[K], c2[K];
#pragma unroll
            for (int i = 0; i < K; ++i) { c1[i] = cf32[SER_PITCH * i + kt + 3]; c2[i] = 0.f; }
            knuth_groups_n<float, K, UNR>(m2, cf32, kt - 1, pf, nf, c1, c2);
#pragma unroll
            for (int i = 0; i < K; ++i) { b1[i] = (T)c1[i]; b2[i] = (T)c2[i]; }
            seeded = true;
        }
    }
    if (!seeded) {
#pragma unroll
        for (int i = 0; i < K; ++i) { b1[i] = cf[SER_PITCH * i + kt + 3]; b2[i] = T(0.); }
    }
    knuth_groups_n<T, K, UNR>(m1, cf, 4 * m1, p, nf2, b1, b2);
#pragma unroll
    for (int i = 0; i < K; ++i) {
        const T r0 = R::fma(nf2, b2[i], cf[SER_PITCH * i + 3]);
        Pr[i] = R::fma(b1[i], wr, r0); Pi[i] = b1[i] * wi;
    }
}

// The two Gaussian factors of a ray (see above): gu multiplies the u family, gv the v family.
template <class T>
__device__ __forceinline__ void shp_gauss(const typename Real<T>::Tab& tb, T u, T v, T& gu, T& gv) {
    using R = Real<T>;
    if constexpr (sizeof(T) == 8) {      // pi^{-1/2} exp(-(u^2 + v^2)/2) = ex2(-0.5 log2(e) (u^2 + v^2) - 0.5 log2(pi))
        gu = R::ex2(tb, R::fma(-T(0.72134752044448170), R::fma(u, u, v * v), -T(0.82574806473615936)));
        gv = T(1.);
    } else {
        gu = R::ex2(tb, R::fma(-T(0.72134752044448170) * u, u, -T(0.41287403236807968)));
        gv = R::ex2(tb, R::fma(-T(0.72134752044448170) * v, v, -T(0.41287403236807968)));
    }
}
// f[k] = f0 psi-polynomial_k(x), k = 0..NMAX
template <class T, int NMAX>
__device__ __forceinline__ void hermite(T x, T f0, T* f) {
    using R = Real<T>;
    f[0] = f0;
    if constexpr (NMAX >= 1) f[1] = x * f0;
#pragma unroll
    for (int k = 1; k < NMAX; ++k) f[k + 1] = R::fma(x, f[k], T(-0.5 * k) * f[k - 1]);
}
// the same plus d[k] = d/dx of (f0(x) polynomial_k(x)) = (k/2) f[k-1] - f[k+1] (f0 a Gaussian in x, or constant times one)
template <class T, int NMAX>
__device__ __forceinline__ void hermite_d(T x, T f0, T* f, T* d) {
    using R = Real<T>;
    f[0] = f0;
    T nxt = x * f0;                      // f[k+1]
    d[0] = -nxt;
#pragma unroll
    for (int k = 1; k <= NMAX; ++k) {
        f[k] = nxt;
        const T t = T(0.5 * k) * f[k - 1];
        nxt = R::fma(x, f[k], -t);
        d[k] = t - nxt;
    }
}

template <class T> struct SersicOut { T I, xr, yr, u, lu, Iu_r2; };

// Sersic surface brightness at (px,py) = position - centre (lab frame); sb = the component's PB block.
template <class T, bool ADJ>
__device__ __forceinline__ SersicOut<T> sersic_eval(const typename Real<T>::Tab& tb, const T* __restrict__ sb, T px, T py) {
    using R = Real<T>;
    SersicOut<T> o;
    o.xr = R::fma(sb[SB_A11], px, sb[SB_A12] * py); o.yr = R::fma(sb[SB_A21], px, sb[SB_A22] * py);   // pre-scaled frame (x', y')
    T r2 = R::fma(o.xr, o.xr, o.yr * o.yr);
    r2 = R::max(r2, T(1e-16));
    T lr = R::lg2(tb, r2);
    o.lu = R::fma(sb[SB_K1], lr, sb[SB_K0]);
    o.u = R::ex2(tb, o.lu);
    const T c1 = sb[SB_C1];
    o.I = sb[SB_IE] * R::ex2(tb, R::fma(-c1, o.u, c1));
    if constexpr (ADJ) {                             // I u / r^2 (radial-derivative factor of the adjoint)
        if constexpr (sizeof(T) == 8) o.Iu_r2 = o.I * o.u * R::rcp(r2); else o.Iu_r2 = o.I * o.u * R::ex2(tb, -lr);
    } else o.Iu_r2 = T(0.);
    return o;
}

template <class T>
__device__ __forceinline__ void sersic_accum(const SersicOut<T>& o, T g, T* __restrict__ S) {
    using R = Real<T>;
    T gI = g * o.I, gIu = gI * o.u;
    S[SA_T0] += gI; S[SA_T1] += gIu; S[SA_T2] = R::fma(gIu, o.lu, S[SA_T2]);
    T W = g * o.Iu_r2;
    T Wx = W * o.xr, Wy = W * o.yr;
    S[SA_AX] += Wx; S[SA_AY] += Wy;
    S[SA_BXX] = R::fma(Wx, o.xr, S[SA_BXX]); S[SA_BYY] = R::fma(Wy, o.yr, S[SA_BYY]); S[SA_BXY] = R::fma(Wx, o.yr, S[SA_BXY]);
}

// Where the shapelet coefficient sums of the adjoint are taken: in the registers of gl_ray_adj_kernel, except in fp64 at
// n_max > 6, where 66 fp64 accumulators do not fit next to the 45 other sums.  Round 1 kept them in shared memory (66
// read-modify-writes per ray: top stall short_scoreboard at 8 warps per SM, profiles/r2a_cfg5_f64.md); now the adjoint
// kernel stores the shapelet coordinates (u, v) of every ray (16 bytes) and gl_shp_coef_kernel takes the sums from
// (gbar, u, v) with all 66 accumulators in registers and nothing else to hold.
template <class T, class V> __host__ __device__ constexpr bool coef_split() { return sizeof(T) == 8 && V::NMAX > 6; }

// Component slots of backward modelling (gl_linear.cuh): index of each light component among the amplitudes, -1 = absent.
struct CompIdx { int src, src1, shp0, n_coef, ll0, ll1, ll2; };

// Everything one ray needs.  ADJ = false: returns the surface brightness; ADJ = true: accumulates gbar * dI/d(natural).
// COMP (with ADJ = false; PB amplitudes all set to unity): also stores the surface brightness of every light component
// separately, component k at acc[k * cstride] (acc = this ray's element of component 0).
template <class T, class V, bool ADJ, bool COMP = false>
__device__ __forceinline__ T ray_eval(const typename Real<T>::Tab& tb, const T* __restrict__ pb,
                                      const T* __restrict__ cfs, const float* __restrict__ cf32, T fj, T fi, T gbar,
                                      T* __restrict__ acc,
                                      T* __restrict__ uvp = nullptr, size_t uvstride = 0,
                                      const CompIdx* ci = nullptr, size_t cstride = 0) {
    using R = Real<T>;
    const T step = pb[PB_STEP];
    const T cph = pb[PB_M_C], sph = pb[PB_M_S];
    const T dx = R::fma(fj, step, pb[PB_M_XOFF]), dy = R::fma(fi, step, pb[PB_M_YOFF]);
    const T xr = R::fma(cph, dx, sph * dy), yr = R::fma(cph, dy, -sph * dx);
    const T q = pb[PB_M_Q];
    const T qx = q * xr;
    const T R2 = R::max(R::fma(qx, qx, yr * yr), T(1e-30));
    const T rinv = R::rsqrt(R2);
    T axr, ayr;                                  // mass-frame deflection
    // adjoint-only pieces
    T S1r = 0, S1i = 0, S2r = 0, S2i = 0, S0r = 0, S0i = 0, S1fr = 0, S1fi = 0, amp = 0, lbr = 0, kap, dqx = 0, dqy = 0;
    if constexpr (V::MASS == 1) {
        const T ce = qx * rinv, se = yr * rinv;
        const T c2 = R::fma(ce, ce, -se * se), s2 = T(2.) * ce * se;
        const T f = pb[PB_M_F], nf2 = -pb[PB_M_F2];
        const T wr = -f * c2, wi = -f * s2, p = T(2.) * wr;
        const int m1 = (int)pb[PB_SER_M1], m2 = (int)pb[PB_SER_M2];
        T Pr[ADJ ? 3 : 1], Pi[ADJ ? 3 : 1];
        constexpr bool UNR = V::NMAX < 0 && (!ADJ || sizeof(T) == 8);      // where the unrolled band switch pays (measured)
        knuth_banded<T, (ADJ ? 3 : 1), UNR>(cfs, cf32, m1, m2, p, nf2, wr, wi, Pr, Pi);
        const T P0r = Pr[0], P0i = Pi[0];
        S0r = R::fma(ce, P0r, -se * P0i); S0i = R::fma(ce, P0i, se * P0r);
        const T lgR2 = R::lg2(tb, R2);
        amp = R::ex2(tb, R::fma(pb[PB_M_H1], lgR2, pb[PB_M_H0]));        // A (b/R)^(t-1) in one exp2
        if constexpr (ADJ) lbr = R::fma(-T(0.5), lgR2, pb[PB_M_L2B]);    // log2(b/R), needed by the slope derivative only
        axr = amp * S0r; ayr = amp * S0i;
        kap = pb[PB_M_KAPC] * amp * rinv;
        if constexpr (ADJ) {
            const T Q1r = Pr[ADJ ? 1 : 0], Q1i = Pi[ADJ ? 1 : 0], Q2r = Pr[ADJ ? 2 : 0], Q2i = Pi[ADJ ? 2 : 0];
            const T ewr = R::fma(ce, wr, -se * wi), ewi = R::fma(ce, wi, se * wr);       // E w
            S1r = R::fma(ewr, Q1r, -ewi * Q1i); S1i = R::fma(ewr, Q1i, ewi * Q1r);
            S2r = R::fma(ewr, Q2r, -ewi * Q2i); S2i = R::fma(ewr, Q2i, ewi * Q2r);
            const T e3r = R::fma(ce, c2, -se * s2), e3i = R::fma(ce, s2, se * c2);       // E^3
            S1fr = -R::fma(e3r, Q1r, -e3i * Q1i); S1fi = -R::fma(e3r, Q1i, e3i * Q1r);
        }
    } else {
        const T qp = pb[PB_M_QP], b = pb[PB_M_B];
        kap = T(0.5) * b * rinv;
        if (qp < T(1e-6)) {                            // SIS limit
            const T ri = R::rsqrt(R::max(R::fma(xr, xr, yr * yr), T(1e-30)));
            axr = b * xr * ri; ayr = b * yr * ri;
        } else {
            const T bqp = pb[PB_M_BQP];
            const T Aa = qp * xr * rinv, Bb = qp * yr * rinv;
            const T at = R::atan(Aa), ath = R::atanh(Bb);
            axr = bqp * at; ayr = bqp * ath;
            if constexpr (ADJ) {
                const T iqp = T(1.) / qp;
                const T common = -q * iqp * rinv - qp * q * xr * xr * rinv * rinv * rinv;
                const T k3 = q * iqp * iqp * iqp;
                dqx = b * R::fma(k3, at, xr * common * iqp / R::fma(Aa, Aa, T(1.)));
                dqy = b * R::fma(k3, ath, yr * common * iqp / R::fma(-Bb, Bb, T(1.)));
            }
        }
    }
    const T x = R::fma(fj, step, pb[PB_XFIRST]), y = R::fma(fi, step, pb[PB_XFIRST]);
    const T g1 = pb[PB_G1], g2 = pb[PB_G2];
    T ax = R::fma(cph, axr, R::fma(-sph, ayr, R::fma(g1, x, g2 * y)));      // rotate back + shear as one FMA chain
    T ay = R::fma(sph, axr, R::fma(cph, ayr, R::fma(g2, x, -g1 * y)));
    // multipoles about the mass centre, lab frame (S7)
    T ct = 0, st = 0, c3 = 0, s3 = 0, c4 = 0, s4 = 0, rinv_m = 0;
    if constexpr (V::MPMASK != 0) {
        rinv_m = R::rsqrt(R::max(R::fma(dx, dx, dy * dy), T(1e-30)));
        ct = dx * rinv_m; st = dy * rinv_m;
        const T cc2 = R::fma(ct, ct, -st * st), ss2 = T(2.) * ct * st;
        c3 = R::fma(cc2, ct, -ss2 * st); s3 = R::fma(ss2, ct, cc2 * st);
        c4 = R::fma(cc2, cc2, -ss2 * ss2); s4 = T(2.) * cc2 * ss2;
        if constexpr (V::MPMASK & 1) {
            const T Am = R::fma(pb[PB_C3], c3, pb[PB_S3] * s3), Bm = R::fma(pb[PB_S3], c3, -pb[PB_C3] * s3);
            ax += -T(0.125) * R::fma(ct, Am, -T(3.) * st * Bm); ay += -T(0.125) * R::fma(st, Am, T(3.) * ct * Bm);
        }
        if constexpr (V::MPMASK & 2) {
            const T Am = R::fma(pb[PB_C4], c4, pb[PB_S4] * s4), Bm = R::fma(pb[PB_S4], c4, -pb[PB_C4] * s4);
            ax += (-T(1.) / T(15.)) * R::fma(ct, Am, -T(4.) * st * Bm); ay += (-T(1.) / T(15.)) * R::fma(st, Am, T(4.) * ct * Bm);
        }
    }
    T Iray = T(0.), gbx = T(0.), gby = T(0.);          // surface brightness; source-plane gradient of the source light
    if constexpr (V::NSRC) {
        const T* sb = pb + PB_SRC;
        const T px = R::fma(fj, step, sb[SB_XOFF]) - ax, py = R::fma(fi, step, sb[SB_YOFF]) - ay;   // beta - centre
        SersicOut<T> o = sersic_eval<T, ADJ>(tb, sb, px, py);
        Iray += o.I;
        if constexpr (COMP) { if (ci->src >= 0) acc[(size_t)ci->src * cstride] = o.I; }
        if constexpr (ADJ) {
            sersic_accum(o, gbar, acc + NA_SRC);
            const T Ixr = -sb[SB_KQ] * o.Iu_r2 * o.xr, Iyr = -sb[SB_KQI] * o.Iu_r2 * o.yr;
            gbx = R::fma(sb[SB_C], Ixr, -sb[SB_S] * Iyr); gby = R::fma(sb[SB_S], Ixr, sb[SB_C] * Iyr);
        }
        if constexpr (V::NSRC >= 2) {                // second source on the same source plane (S1, S2)
            // second source: same plane (eta2 = 1, exactly the one-plane arithmetic) or its own plane, beta_2 = theta - eta2 alpha
            const T* s1 = pb + PB_SRC1;
            const T eta = s1[SB_ETA];
            const T qx1 = R::fma(-eta, ax, R::fma(fj, step, s1[SB_XOFF])), qy1 = R::fma(-eta, ay, R::fma(fi, step, s1[SB_YOFF]));
            SersicOut<T> o1 = sersic_eval<T, ADJ>(tb, s1, qx1, qy1);
            Iray += o1.I;
            if constexpr (COMP) { if (ci->src1 >= 0) acc[(size_t)ci->src1 * cstride] = o1.I; }
            if constexpr (ADJ) {
                sersic_accum(o1, gbar, acc + NA_SRC1);
                const T Ixr = -s1[SB_KQ] * o1.Iu_r2 * o1.xr, Iyr = -s1[SB_KQI] * o1.Iu_r2 * o1.yr;
                const T g1x = R::fma(s1[SB_C], Ixr, -s1[SB_S] * Iyr), g1y = R::fma(s1[SB_S], Ixr, s1[SB_C] * Iyr);
                gbx = R::fma(eta, g1x, gbx); gby = R::fma(eta, g1y, gby);             // d beta_2 / d(mass) = -eta2 d alpha / d(mass)
                acc[NA_ETA] = R::fma(-gbar, R::fma(g1x, ax, g1y * ay), acc[NA_ETA]);   // d beta_2 / d eta2 = -alpha
            }
        }
        if constexpr (V::NMAX >= 0) {
            constexpr int NM = V::NMAX >= 0 ? V::NMAX : 0;
            const T ibs = pb[PB_SHP];
            const T u = px * ibs, v = py * ibs;
            T gu, gv;
            shp_gauss<T>(tb, u, v, gu, gv);
            T fu[NM + 1], fv[NM + 1];
            const T* a = pb + PB_SHP_A;              // a_k c_n1 c_n2 / beta_s (scaled basis, see hermite)
            T Ish = T(0.);
            if constexpr (COMP) {                    // basis function k with unit coefficient: phi_n1(u) phi_n2(v) / beta_s
                hermite<T, NM>(u, gu, fu); hermite<T, NM>(v, gv, fv);
#pragma unroll
                for (int n2 = 0; n2 <= NM; ++n2) {
                    const T fvb = fv[n2] * ibs;
#pragma unroll
                    for (int n1 = 0; n1 <= NM - n2; ++n1) {
                        const int idx = (n1 + n2) * (n1 + n2 + 1) / 2 + n2;
                        if (idx < ci->n_coef) acc[(size_t)(ci->shp0 + idx) * cstride] = fu[n1] * fvb * (T)(d_HC[n1] * d_HC[n2]);
                    }
                }
            } else if constexpr (!ADJ) {
                hermite<T, NM>(u, gu, fu); hermite<T, NM>(v, gv, fv);
#pragma unroll
                for (int n2 = 0; n2 <= NM; ++n2) {
                    T row = T(0.);
#pragma unroll
                    for (int n1 = 0; n1 <= NM - n2; ++n1) row = R::fma(a[(n1 + n2) * (n1 + n2 + 1) / 2 + n2], fu[n1], row);
                    Ish = R::fma(row, fv[n2], Ish);
                }
            } else {
                // the N_coef coefficient sums gbar psi_n1(u) psi_n2(v) are taken here in registers, or (coef_split) by
                // gl_shp_coef_kernel from the (u, v) stored below.
                T dfu[NM + 1], dfv[NM + 1];
                hermite_d<T, NM>(u, gu, fu, dfu); hermite_d<T, NM>(v, gv, fv, dfv);
                if constexpr (coef_split<T, V>()) { uvp[0] = u; uvp[uvstride] = v; }
                T Iu = T(0.), Iv = T(0.);
#pragma unroll
                for (int n2 = 0; n2 <= NM; ++n2) {
                    T row = T(0.), drow = T(0.);
                    const T gfv = gbar * fv[n2];
#pragma unroll
                    for (int n1 = 0; n1 <= NM - n2; ++n1) {
                        const int idx = (n1 + n2) * (n1 + n2 + 1) / 2 + n2;
                        const T ak = a[idx];
                        row = R::fma(ak, fu[n1], row); drow = R::fma(ak, dfu[n1], drow);
                        if constexpr (!coef_split<T, V>()) acc[NA_SHA + idx] = R::fma(gfv, fu[n1], acc[NA_SHA + idx]);
                    }
                    Ish = R::fma(row, fv[n2], Ish); Iu = R::fma(drow, fv[n2], Iu); Iv = R::fma(row, dfv[n2], Iv);
                }
                acc[NA_SHB] = R::fma(gbar, Ish + R::fma(u, Iu, v * Iv), acc[NA_SHB]);
                const T Ibx = Iu * ibs, Iby = Iv * ibs;
                acc[NA_SHX] = R::fma(gbar, Ibx, acc[NA_SHX]); acc[NA_SHY] = R::fma(gbar, Iby, acc[NA_SHY]);
                gbx += Ibx; gby += Iby;
            }
            Iray += Ish;
        }
    }
    if constexpr (V::NLL >= 1) {
        const T* sb = pb + PB_LL0;
        SersicOut<T> o = sersic_eval<T, ADJ>(tb, sb, R::fma(fj, step, sb[SB_XOFF]), R::fma(fi, step, sb[SB_YOFF]));
        Iray += o.I; if constexpr (ADJ) sersic_accum(o, gbar, acc + NA_LL0);
        if constexpr (COMP) { if (ci->ll0 >= 0) acc[(size_t)ci->ll0 * cstride] = o.I; }
    }
    if constexpr (V::NLL >= 2) {
        const T* sb = pb + PB_LL1;
        SersicOut<T> o = sersic_eval<T, ADJ>(tb, sb, R::fma(fj, step, sb[SB_XOFF]), R::fma(fi, step, sb[SB_YOFF]));
        Iray += o.I; if constexpr (ADJ) sersic_accum(o, gbar, acc + NA_LL1);
        if constexpr (COMP) { if (ci->ll1 >= 0) acc[(size_t)ci->ll1 * cstride] = o.I; }
    }
    if constexpr (V::NLL >= 3) {
        const T* sb = pb + PB_LL2;
        SersicOut<T> o = sersic_eval<T, ADJ>(tb, sb, R::fma(fj, step, sb[SB_XOFF]), R::fma(fi, step, sb[SB_YOFF]));
        Iray += o.I; if constexpr (ADJ) sersic_accum(o, gbar, acc + NA_LL2);
        if constexpr (COMP) { if (ci->ll2 >= 0) acc[(size_t)ci->ll2 * cstride] = o.I; }
    }
    if constexpr (ADJ) {
        // mass parameters enter through beta only: d/dtheta_mass = -(gbar grad_beta I_src) . dalpha/dtheta_mass
        const T sx = gbar * gbx, sy = gbar * gby;
        const T srx = R::fma(cph, sx, sph * sy), sry = R::fma(cph, sy, -sph * sx);
        const T sa = R::fma(srx, axr, sry * ayr);
        const T tm1 = V::MASS == 1 ? pb[PB_M_TM1] : T(0.);
        const T izz = R::rcp(R::max(R::fma(xr, xr, yr * yr), T(1e-30)));
        const T hr = R::fma(-tm1, axr, -xr * kap), hi = R::fma(-tm1, ayr, -yr * kap);
        const T Gr = R::fma(xr, hr, -yr * hi) * izz, Gi = R::fma(xr, hi, yr * hr) * izz;
        const T Jxx = kap + Gr, Jyy = kap - Gr, Jxy = Gi;
        acc[NA_D0] += sa;
        if constexpr (V::MASS == 1) {
            const T rr2 = rinv * rinv;
            acc[NA_DTL] = R::fma(lbr, sa, acc[NA_DTL]);
            acc[NA_DT2] = R::fma(amp, R::fma(srx, S2r, sry * S2i), acc[NA_DT2]);
            acc[NA_D1] = R::fma(sa * xr, xr * rr2, acc[NA_D1]);
            const T Zr = R::fma(T(2.), S1r, S0r), Zi = R::fma(T(2.), S1i, S0i);
            acc[NA_D2] = R::fma(amp * xr * yr * rr2, R::fma(sry, Zr, -srx * Zi), acc[NA_D2]);
            acc[NA_D3] = R::fma(amp, R::fma(srx, S1fr, sry * S1fi), acc[NA_D3]);
        } else {
            acc[NA_DQS] += R::fma(srx, dqx, sry * dqy);
        }
        acc[NA_DPHI] += R::fma(srx, R::fma(Jxx, yr, -Jxy * xr) - ayr, sry * (R::fma(Jxy, yr, -Jyy * xr) + axr));
        acc[NA_VX] += R::fma(Jxx, srx, Jxy * sry); acc[NA_VY] += R::fma(Jxy, srx, Jyy * sry);
        acc[NA_G1] -= R::fma(sx, x, -sy * y); acc[NA_G2] -= R::fma(sx, y, sy * x);
        if constexpr (V::MPMASK != 0) {
            T Atot = T(0.);
            if constexpr (V::MPMASK & 1) {
                acc[NA_C3] += T(0.125) * R::fma(sx, R::fma(ct, c3, T(3.) * st * s3), sy * R::fma(st, c3, -T(3.) * ct * s3));
                acc[NA_S3] += T(0.125) * R::fma(sx, R::fma(ct, s3, -T(3.) * st * c3), sy * R::fma(st, s3, T(3.) * ct * c3));
                Atot += R::fma(pb[PB_C3], c3, pb[PB_S3] * s3);
            }
            if constexpr (V::MPMASK & 2) {
                acc[NA_C4] += (T(1.) / T(15.)) * R::fma(sx, R::fma(ct, c4, T(4.) * st * s4), sy * R::fma(st, c4, -T(4.) * ct * s4));
                acc[NA_S4] += (T(1.) / T(15.)) * R::fma(sx, R::fma(ct, s4, -T(4.) * st * c4), sy * R::fma(st, s4, T(4.) * ct * c4));
                Atot += R::fma(pb[PB_C4], c4, pb[PB_S4] * s4);
            }
            const T proj = Atot * rinv_m * R::fma(ct, sy, -st * sx);
            acc[NA_MCX] = R::fma(-st, proj, acc[NA_MCX]); acc[NA_MCY] = R::fma(ct, proj, acc[NA_MCY]);
        }
    }
    return Iray;
}

// ----------------------------------------------------------------------------- kernels
// Ray <-> thread mapping shared by both kernels: one CTA works on ONE phase plane (a, b) of one particle, so the
// plane shift (o_a, o_b) is CTA-uniform and consecutive threads touch consecutive addresses of a plane row.
// grid = (s*s*n_chunk, Pc); CTA (ph, ck) handles plane rays [ck*nt*RPT, (ck+1)*nt*RPT) of the N*N in plane ph.
// Ray coordinates are taken relative to the grid CENTRE (fj = j - (M-1)/2, exact in fp32), so that a position minus a
// component centre keeps its relative accuracy near that centre, where the light profiles are steepest.
struct PlaneIter {
    int ph, a, b, oa, ob, idx, j1, dj, off, doff, wrap_off;
    float fjf, fif, dfj, dfi, wrap_fj, wrap_fi;       // centre-relative ray coordinates, exact in fp32 (multiples of 1/2 below 2^12)
    // Everything a ray needs from its index -- element offset in the plane, (fj, fi) -- advances by additions: the products
    // and int -> float conversions per ray were ~5 % of the forward kernel's instructions on config 2.
    __device__ __forceinline__ PlaneIter(const Geom& G, int n_chunk, int RPT) {
        ph = blockIdx.x / n_chunk;
        const int ck = blockIdx.x - ph * n_chunk;
        a = ph / G.s; b = ph - a * G.s; oa = phase_shift(G, a); ob = phase_shift(G, b);
        idx = ck * (blockDim.x * RPT) + threadIdx.x;
        const int i1 = idx / G.N;
        j1 = idx - i1 * G.N;
        const int di = blockDim.x / G.N;
        dj = blockDim.x - di * G.N;
        const float half = 0.5f * (float)(G.M - 1);
        off = (i1 + oa) * G.Wp + (j1 + ob); doff = di * G.Wp + dj; wrap_off = G.Wp - G.N;
        fjf = (float)(G.s * j1 + b) - half; fif = (float)(G.s * i1 + a) - half;
        dfj = (float)(G.s * dj); dfi = (float)(G.s * di); wrap_fj = -(float)(G.s * G.N); wrap_fi = (float)G.s;
    }
    __device__ __forceinline__ void next(const Geom& G) {
        idx += blockDim.x; j1 += dj; off += doff; fjf += dfj; fif += dfi;
        if (j1 >= G.N) { j1 -= G.N; off += wrap_off; fjf += wrap_fj; fif += wrap_fi; }
    }
    template <class T> __device__ __forceinline__ T fj(const Geom&) const { return (T)fjf; }
    template <class T> __device__ __forceinline__ T fi(const Geom&) const { return (T)fif; }
    __device__ __forceinline__ size_t offset(const Geom&) const { return (size_t)off; }
};

// The same mapping with the smallest state (index, row, column; offset and coordinates computed per ray): for the adjoint
// variants that keep the shapelet coefficient sums in registers next to everything else (fp64, n_max <= 6: 254 registers), where
// the six more live values of PlaneIter cost more than the instructions they save (config 3: 17.5 against 18.2 ms).
struct PlaneIterLean {
    int ph, a, b, oa, ob, idx, i1, j1, di, dj;
    float half;
    __device__ __forceinline__ PlaneIterLean(const Geom& G, int n_chunk, int RPT) {
        ph = blockIdx.x / n_chunk;
        const int ck = blockIdx.x - ph * n_chunk;
        a = ph / G.s; b = ph - a * G.s; oa = phase_shift(G, a); ob = phase_shift(G, b);
        idx = ck * (blockDim.x * RPT) + threadIdx.x;
        i1 = idx / G.N; j1 = idx - i1 * G.N;
        di = blockDim.x / G.N; dj = blockDim.x - di * G.N;
        half = 0.5f * (float)(G.M - 1);
    }
    __device__ __forceinline__ void next(const Geom& G) {
        idx += blockDim.x; i1 += di; j1 += dj;
        if (j1 >= G.N) { j1 -= G.N; ++i1; }
    }
    template <class T> __device__ __forceinline__ T fj(const Geom& G) const { return (T)((float)(G.s * j1 + b) - half); }
    template <class T> __device__ __forceinline__ T fi(const Geom& G) const { return (T)((float)(G.s * i1 + a) - half); }
    __device__ __forceinline__ size_t offset(const Geom& G) const { return (size_t)(i1 + oa) * G.Wp + (j1 + ob); }
};

// Shared-memory copy of the fp64 exp2/log2 tables (double mode only; one dummy element in float mode).
template <class T> struct TabStage;
template <> struct TabStage<float> {
    static constexpr int N = 1;
    static __device__ __forceinline__ int make(double*, const double*) { return 0; }
};
template <> struct TabStage<double> {
    static constexpr int N = MATH_TAB_DOUBLES;
    static __device__ __forceinline__ MathTab make(double* sm, const double* g) { stage_math_tab(sm, g); return math_tab(sm); }
};

// Zero the border of one padded plane (everything outside the N x N interior at (oa, ob)); element e = first, first + stride, ...
// Row and column advance incrementally: one integer division per thread instead of one per element (the division loop was 7 % of
// the forward kernel's instructions on config 2).
template <class T>
__device__ __forceinline__ void zero_plane_border(const Geom& G, T* __restrict__ out, int oa, int ob, int first, int stride) {
    const int tot = G.Hp * G.Wp, dr = stride / G.Wp, dc = stride - dr * G.Wp;
    int r = first / G.Wp, cc = first - r * G.Wp;
    for (int e = first; e < tot; e += stride) {
        if (r < oa || r >= oa + G.N || cc < ob || cc >= ob + G.N) out[e] = T(0.);
        r += dr; cc += dc;
        if (cc >= G.Wp) { cc -= G.Wp; ++r; }
    }
}

// Steps B + C.  Writes the plane interior and zeroes this CTA's share of the plane border.
template <class T, class V, int NT, int RB>
__global__ void __launch_bounds__(NT) gl_ray_fwd_kernel(const __grid_constant__ Geom G, const T* __restrict__ pbg,
                                                        const double* __restrict__ tabg, T* __restrict__ ray, int RPT,
                                                        int n_chunk) {
    __shared__ __align__(16) T pb[PB_STRIDE];
    __shared__ __align__(128) double tabs[TabStage<T>::N];
    const int p = blockIdx.y;
    const T* src = pbg + (size_t)p * PB_STRIDE;
    for (int k = threadIdx.x; k < V::PB_NEED; k += blockDim.x) pb[k] = src[k];
    __shared__ __align__(16) T cfs[V::MASS == 1 ? 3 * SER_PITCH : 4];                          // series coefficients, shifted layout
    __shared__ __align__(16) float cf32[(sizeof(T) == 8 && V::MASS == 1) ? 3 * SER_PITCH : 4];  // their fp32 copies
    if constexpr (V::MASS == 1) stage_series<T>(src, cfs, cf32);
    const typename Real<T>::Tab tb = TabStage<T>::make(tabs, tabg);
    __syncthreads();
    PlaneIter it(G, n_chunk, RPT);
    T* out = ray + (size_t)p * ray_stride(G) + (size_t)it.ph * G.Hp * G.Wp;
    zero_plane_border(G, out, it.oa, it.ob, (blockIdx.x - it.ph * n_chunk) * blockDim.x + threadIdx.x, n_chunk * blockDim.x);
    const int NN = G.N * G.N;
    const bool valid = pb[PB_VALID] != T(0.);
    // RB rays per step, evaluated unconditionally in one basic block so that the scheduler interleaves their
    // dependency chains (the FP64 pipe needs ~4 independent DFMAs in flight per warp); only the store is predicated.
    for (int r = 0; r < RPT; r += RB) {
        int off = 0; asm volatile("" : "+r"(off));      // opaque: keeps the PB scalars in shared memory, not in registers
        T v[RB]; size_t o[RB]; bool ok[RB];
#pragma unroll
        for (int b = 0; b < RB; ++b) {
            ok[b] = it.idx < NN && r + b < RPT;
            o[b] = it.offset(G);
            v[b] = ray_eval<T, V, false>(tb, pb + off, cfs + off, cf32 + off, it.fj<T>(G), it.fi<T>(G), T(0.), nullptr);
            it.next(G);
        }
#pragma unroll
        for (int b = 0; b < RB; ++b)
            if (ok[b]) out[o[b]] = valid ? v[b] : T(0.);
    }
}

// Steps B + C on the dedicated psf_grid = 1 path (Geom.binned): that path convolves the BINNED image, the sum of the s*s
// phase planes, which all carry the same shift o there.  One thread evaluates the s*s rays of a detector pixel and adds them
// in the order of the bin pass (plane 0, 1, ..., s*s - 1: bit-identical to writing the planes and running
// gl_bin_planes_kernel), and only plane 0 is written: no bin pass (s*s + 1 plane-sized HBM transfers per particle) and s*s times
// fewer bytes stored here.  grid = (n_chunk, Pc); CTA ck handles pixels [ck nt RPT, (ck + 1) nt RPT) of the N*N.
template <class T, class V, int NT>
__global__ void __launch_bounds__(NT) gl_ray_fwd_binned_kernel(const __grid_constant__ Geom G, const T* __restrict__ pbg,
                                                               const double* __restrict__ tabg, T* __restrict__ ray, int RPT,
                                                               int n_chunk) {
    __shared__ __align__(16) T pb[PB_STRIDE];
    __shared__ __align__(128) double tabs[TabStage<T>::N];
    const int p = blockIdx.y, ck = blockIdx.x;
    const T* src = pbg + (size_t)p * PB_STRIDE;
    for (int k = threadIdx.x; k < V::PB_NEED; k += blockDim.x) pb[k] = src[k];
    __shared__ __align__(16) T cfs[V::MASS == 1 ? 3 * SER_PITCH : 4];
    __shared__ __align__(16) float cf32[(sizeof(T) == 8 && V::MASS == 1) ? 3 * SER_PITCH : 4];
    if constexpr (V::MASS == 1) stage_series<T>(src, cfs, cf32);
    const typename Real<T>::Tab tb = TabStage<T>::make(tabs, tabg);
    __syncthreads();
    T* out = ray + (size_t)p * ray_stride(G);                       // plane 0
    const int o = phase_shift(G, 0), N = G.N, s = G.s;
    zero_plane_border(G, out, o, o, ck * blockDim.x + threadIdx.x, n_chunk * blockDim.x);
    const int NN = N * N;
    const bool valid = pb[PB_VALID] != T(0.);
    const float half = 0.5f * (float)(G.M - 1);
    int idx = ck * (blockDim.x * RPT) + threadIdx.x;
    for (int r = 0; r < RPT; ++r, idx += blockDim.x) {
        if (idx >= NN) break;
        const int i1 = idx / N, j1 = idx - i1 * N;
        T sum = T(0.);
        for (int a = 0; a < s; ++a)
            for (int b = 0; b < s; ++b) {
                int off = 0; asm volatile("" : "+r"(off));      // opaque: keeps the PB scalars in shared memory, not in registers
                const T v = ray_eval<T, V, false>(tb, pb + off, cfs + off, cf32 + off, (T)((float)(s * j1 + b) - half),
                                                  (T)((float)(s * i1 + a) - half), T(0.), nullptr);
                sum = (a | b) == 0 ? v : sum + v;
            }
        out[(size_t)(i1 + o) * G.Wp + (j1 + o)] = valid ? sum : T(0.);
    }
}

// Component images of backward modelling: steps B-C once per ray (one deflection), every light component with unit
// amplitude stored in its own RAY buffer: comp_ray [n_amp][Pc][ray_stride].  Same grid as gl_ray_fwd_kernel.
template <class T, class V, int NT>
__global__ void __launch_bounds__(NT) gl_ray_comp_kernel(const __grid_constant__ Geom G, const __grid_constant__ CompIdx ci, int n_amp,
                                                         const T* __restrict__ pbg, const double* __restrict__ tabg,
                                                         T* __restrict__ comp_ray, size_t cstride, int RPT, int n_chunk) {
    __shared__ __align__(16) T pb[PB_STRIDE];
    __shared__ __align__(128) double tabs[TabStage<T>::N];
    const int p = blockIdx.y;
    const T* src = pbg + (size_t)p * PB_STRIDE;
    for (int k = threadIdx.x; k < V::PB_NEED; k += blockDim.x) pb[k] = src[k];
    __shared__ __align__(16) T cfs[V::MASS == 1 ? 3 * SER_PITCH : 4];
    __shared__ __align__(16) float cf32[(sizeof(T) == 8 && V::MASS == 1) ? 3 * SER_PITCH : 4];
    if constexpr (V::MASS == 1) stage_series<T>(src, cfs, cf32);
    const typename Real<T>::Tab tb = TabStage<T>::make(tabs, tabg);
    __syncthreads();
    PlaneIter it(G, n_chunk, RPT);
    T* out = comp_ray + (size_t)p * ray_stride(G) + (size_t)it.ph * G.Hp * G.Wp;
    for (int k = 0; k < n_amp; ++k)
        zero_plane_border(G, out + (size_t)k * cstride, it.oa, it.ob, (blockIdx.x - it.ph * n_chunk) * blockDim.x + threadIdx.x, n_chunk * blockDim.x);
    const int NN = G.N * G.N;
    const bool valid = pb[PB_VALID] != T(0.);
    for (int r = 0; r < RPT; ++r) {
        int off = 0; asm volatile("" : "+r"(off));
        if (it.idx < NN) {
            T* o = out + it.offset(G);
            if (valid) ray_eval<T, V, false, true>(tb, pb + off, cfs + off, cf32 + off, it.fj<T>(G), it.fi<T>(G), T(0.), o, nullptr, 0, &ci, cstride);
            else for (int k = 0; k < n_amp; ++k) o[(size_t)k * cstride] = T(0.);
        }
        it.next(G);
    }
}

// Per-ray part of step F.  gbar: plane layout; nap: [Pc][gridDim.x][V::NA].
#ifndef GL_ADJ_MINB
#define GL_ADJ_MINB 4
#endif
#ifndef GL_ADJ_MINB_X
#define GL_ADJ_MINB_X 3     // two sources / three lens blocks, no shapelets (61 fp64 sums): 168 registers
#endif
#ifndef GL_ADJ_MINB_S
#define GL_ADJ_MINB_S 1     // shapelet variants in fp64
#endif
template <class T, class V, int NT>
__global__ void __launch_bounds__(NT, (sizeof(T) == 8 && V::NMAX < 0 && V::NSRC < 2 && V::NLL < 3 ? GL_ADJ_MINB : (sizeof(T) == 8 && V::NMAX < 0 ? GL_ADJ_MINB_X : (sizeof(T) == 8 ? GL_ADJ_MINB_S : 1)))) gl_ray_adj_kernel(const __grid_constant__ Geom G, const T* __restrict__ pbg,
                                                        const double* __restrict__ tabg, const T* __restrict__ gbar,
                                                        T* __restrict__ nap, T* __restrict__ uv, int RPT, int n_chunk) {
    __shared__ __align__(16) T pb[PB_STRIDE];
    __shared__ __align__(128) double tabs[TabStage<T>::N];
    __shared__ T red[NT / 32][coef_split<T, V>() ? NA_SHA : V::NA];
    const int p = blockIdx.y;
    const T* src = pbg + (size_t)p * PB_STRIDE;
    for (int k = threadIdx.x; k < V::PB_NEED; k += blockDim.x) pb[k] = src[k];
    __shared__ __align__(16) T cfs[V::MASS == 1 ? 3 * SER_PITCH : 4];                          // series coefficients, shifted layout
    __shared__ __align__(16) float cf32[(sizeof(T) == 8 && V::MASS == 1) ? 3 * SER_PITCH : 4];  // their fp32 copies
    if constexpr (V::MASS == 1) stage_series<T>(src, cfs, cf32);
    const typename Real<T>::Tab tb = TabStage<T>::make(tabs, tabg);
    __syncthreads();
    using Iter = typename std::conditional<(sizeof(T) == 8 && V::NMAX >= 0 && !coef_split<T, V>()), PlaneIterLean, PlaneIter>::type;
    Iter it(G, n_chunk, RPT);
    const T* gb = gbar + (size_t)p * ray_stride(G) + (size_t)(G.binned ? 0 : it.ph) * G.Hp * G.Wp;   // binned: one gbar plane for all
    const int NN = G.N * G.N;
    constexpr bool CS = coef_split<T, V>();
    constexpr int NREG = CS ? NA_SHA : V::NA;                     // accumulators of this kernel (all in registers)
    const size_t rs = ray_stride(G);
    T* uvb = CS ? uv + (size_t)p * 2 * rs + (size_t)it.ph * G.Hp * G.Wp : nullptr;
    T acc[NREG];
#pragma unroll
    for (int k = 0; k < NREG; ++k) acc[k] = T(0.);
    if (pb[PB_VALID] != T(0.)) {
        for (int r = 0; r < RPT; ++r) {
            int off = 0; asm volatile("" : "+r"(off));      // opaque: keeps the PB scalars in shared memory, not in registers
            if (it.idx < NN) {
                const size_t o = it.offset(G);
                ray_eval<T, V, true>(tb, pb + off, cfs + off, cf32 + off, it.template fj<T>(G), it.template fi<T>(G), gb[o], acc, CS ? uvb + o : nullptr, rs);
            }
            it.next(G);
        }
    }
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5, nw = blockDim.x >> 5;
#pragma unroll
    for (int k = 0; k < NREG; ++k) {
        T v = warp_sum(acc[k]);
        if (lane == 0) red[w][k] = v;
    }
    __syncthreads();
    T* o = nap + ((size_t)p * gridDim.x + blockIdx.x) * V::NA;
    for (int k = threadIdx.x; k < NREG; k += blockDim.x) {
        T s = T(0.);
        for (int ww = 0; ww < nw; ++ww) s += red[ww][k];
        o[k] = s;
    }
}

#ifndef GL_COEF_NS
#define GL_COEF_NS 8
#endif
__device__ __forceinline__ void coef_cp8(void* smem_dst, const void* gsrc) {
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"((uint32_t)__cvta_generic_to_shared(smem_dst)), "l"(gsrc) : "memory");
}
// Shapelet coefficient sums of step F in the split form (coef_split): nap[..][NA_SHA + k] = sum_rays gbar phi_n1(u) phi_n2(v),
// k = (n1 + n2)(n1 + n2 + 1)/2 + n2, from the (u, v) gl_ray_adj_kernel stored.  Same grid, block and ray <-> thread mapping as
// that kernel, so both write the same partial slot of nap; fixed-order warp / CTA reduction, no atomics.
template <class T, int NMAX, int NA, int NT>
__global__ void __launch_bounds__(NT) gl_shp_coef_kernel(const __grid_constant__ Geom G, const T* __restrict__ pbg,
                                                         const double* __restrict__ tabg, const T* __restrict__ gbar,
                                                         const T* __restrict__ uv, T* __restrict__ nap, int RPT, int n_chunk) {
    constexpr int NC = (NMAX + 1) * (NMAX + 2) / 2;
    constexpr int NS = GL_COEF_NS;                              // cp.async ring depth (rays in flight per thread)
    __shared__ __align__(128) double tabs[TabStage<T>::N];
    __shared__ T red[NT / 32][NC];
    __shared__ __align__(16) T stg[NS][3][NT];
    const int p = blockIdx.y;
    const typename Real<T>::Tab tb = TabStage<T>::make(tabs, tabg);
    __syncthreads();
    PlaneIter it(G, n_chunk, RPT);
    const size_t rs = ray_stride(G), pl = (size_t)it.ph * G.Hp * G.Wp;
    const T* gb = gbar + (size_t)p * rs + (G.binned ? 0 : pl);
    const T* ub = uv + (size_t)p * 2 * rs + pl;
    const int NN = G.N * G.N;
    T acc[NC];
#pragma unroll
    for (int k = 0; k < NC; ++k) acc[k] = T(0.);
    if (pbg[(size_t)p * PB_STRIDE + PB_VALID] != T(0.)) {
        // (gbar, u, v) of the next NS rays of this thread are in flight as 8-byte cp.async copies into a shared-memory
        // ring of its own slots: the kernel holds ~230 registers (2 warps per scheduler), so the HBM latency has to be
        // covered by the thread itself (config 5, ms per step: 29.9 without prefetch, 21.6 / 18.5 with 4 / 8 register slots,
        // 17.9 with this ring at depth 8; depth 12 costs a resident CTA and is slower).  A thread reads only what it copied:
        // no CTA barrier.
        PlaneIter ld = it;
        auto fetch = [&](int k, int ray) {
            const bool ok = ld.idx < NN && ray < RPT;
            T* d = &stg[k][0][threadIdx.x];
            if (ok) {
                const size_t o = ld.offset(G);
                coef_cp8(d, gb + o); coef_cp8(d + NT, ub + o); coef_cp8(d + 2 * NT, ub + rs + o);
            } else { d[0] = T(0.); d[NT] = T(0.); d[2 * NT] = T(0.); }     // gbar = 0: such a ray adds nothing
            asm volatile("cp.async.commit_group;" ::: "memory");
            ld.next(G);
        };
#pragma unroll
        for (int k = 0; k < NS; ++k) fetch(k, k);
        for (int r0 = 0; r0 < RPT; r0 += NS) {
#pragma unroll
            for (int k = 0; k < NS; ++k) {
                asm volatile("cp.async.wait_group %0;" ::"n"(NS - 1) : "memory");
                const T* d = &stg[k][0][threadIdx.x];
                const T g = d[0], u = d[NT], v = d[2 * NT];
                fetch(k, r0 + k + NS);
                T gu, gv, fu[NMAX + 1], fv[NMAX + 1];
                shp_gauss<T>(tb, u, v, gu, gv);
                hermite<T, NMAX>(u, gu, fu); hermite<T, NMAX>(v, gv, fv);
#pragma unroll
                for (int n1 = 0; n1 <= NMAX; ++n1) {
                    const T gf = g * fu[n1];
#pragma unroll
                    for (int n2 = 0; n2 <= NMAX - n1; ++n2) {
                        const int idx = (n1 + n2) * (n1 + n2 + 1) / 2 + n2;
                        acc[idx] = Real<T>::fma(gf, fv[n2], acc[idx]);
                    }
                }
            }
        }
        asm volatile("cp.async.wait_group 0;" ::: "memory");
    }
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5, nw = blockDim.x >> 5;
#pragma unroll
    for (int k = 0; k < NC; ++k) {
        const T v = warp_sum(acc[k]);
        if (lane == 0) red[w][k] = v;
    }
    __syncthreads();
    T* o = nap + ((size_t)p * gridDim.x + blockIdx.x) * NA + NA_SHA;
    for (int k = threadIdx.x; k < NC; k += blockDim.x) {
        T s = T(0.);
        for (int ww = 0; ww < nw; ++ww) s += red[ww][k];
        o[k] = s;
    }
}

}  // namespace gl
