// gl_ray.cuh -- steps B + C (ray-trace + paint light) and the per-ray part of step F (adjoint).
//
// One CTA = one chunk of rays of one phase plane of ONE particle; the particle's derived scalars (PB) are staged in
// shared memory once per CTA and every per-ray quantity lives in registers.  FP32 FMA pipe + MUFU
// (rsqrt / lg2 / ex2 / rcp).  The 30-term EPL series (BASELINE.json configs[1]; reading S5) is a real-
// coefficient polynomial in w = -f e^{2 i phi}; because |w|^2 = f^2 is a per-particle constant it is
// evaluated by synthetic division by (x - w)(x - conj w) = x^2 - p x + f^2, p = 2 Re w:
//     b_k = a_k + p b_{k+1} - f^2 b_{k+2},   P(w) = b_1 w + (a_0 - f^2 b_2)
// i.e. 2 FMAs per term instead of the 4 of complex Horner; the recurrence is contractive for f < 1.
#pragma once
#include "gl_common.cuh"

namespace gl {

__device__ __forceinline__ float f_ex2(float x) { float y; asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ float f_lg2(float x) { float y; asm("lg2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ float f_rsqrt(float x) { float y; asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ float f_rcp(float x) { float y; asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }

// Gauss-Hermite recurrence constants: phi_{k+1} = HA[k] u phi_k - HB[k] phi_{k-1};  phi_k' = HD[k] phi_{k-1} - u phi_k
__constant__ float c_HA[12] = {1.41421356237309505f, 1.0f, 0.81649658092772603f, 0.70710678118654752f, 0.63245553203367587f,
                               0.57735026918962576f, 0.53452248382484879f, 0.5f, 0.47140452079103168f, 0.44721359549995794f,
                               0.42640143271122088f, 0.40824829046386302f};
__constant__ float c_HB[12] = {0.0f, 0.70710678118654752f, 0.81649658092772603f, 0.86602540378443865f, 0.89442719099991588f,
                               0.91287092917527686f, 0.92582009977255146f, 0.93541434669348535f, 0.94280904158206337f,
                               0.94868329805051380f, 0.95346258924559232f, 0.95742710775633811f};
__constant__ float c_HD[12] = {0.0f, 1.41421356237309505f, 2.0f, 2.44948974278317810f, 2.82842712474619010f, 3.16227766016837933f,
                               3.46410161513775459f, 3.74165738677394139f, 4.0f, 4.24264068711928515f, 4.47213595499957939f,
                               4.69041575982342955f};

// P(w) = sum_{k<=TOP} cf[k] w^k for real coefficients cf (shared memory, zero beyond the kept terms).
template <int TOP>
__device__ __forceinline__ void knuth(const float* __restrict__ cf, float p, float nf2, float wr, float wi, float& Pr, float& Pi) {
    float b1 = cf[TOP], b2 = 0.f;
#pragma unroll
    for (int k = TOP - 1; k >= 1; --k) {
        float bk = fmaf(p, b1, fmaf(nf2, b2, cf[k]));
        b2 = b1; b1 = bk;
    }
    float r0 = fmaf(nf2, b2, cf[0]);
    Pr = fmaf(b1, wr, r0); Pi = b1 * wi;
}

template <int NMAX>
__device__ __forceinline__ void hermite(float u, float* f) {
    // pi^{-1/4} exp(-u^2/2) = ex2(-0.5 log2(e) u^2 + log2(pi^{-1/4}))
    f[0] = f_ex2(fmaf(-0.72134752044448170f * u, u, -0.41287417812882825f));
    if constexpr (NMAX >= 1) f[1] = c_HA[0] * u * f[0];
#pragma unroll
    for (int k = 1; k < NMAX; ++k) f[k + 1] = fmaf(c_HA[k] * u, f[k], -c_HB[k] * f[k - 1]);
}

struct SersicOut { float I, xr, yr, u, lu, Iu_r2; };

// Sersic surface brightness at (px,py) = position - centre (lab frame); sb = the component's PB block.
__device__ __forceinline__ SersicOut sersic_eval(const float* __restrict__ sb, float px, float py) {
    SersicOut o;
    const float c = sb[SB_C], s = sb[SB_S];
    o.xr = fmaf(c, px, s * py); o.yr = fmaf(c, py, -s * px);
    float r2 = fmaf(sb[SB_Q] * o.xr, o.xr, sb[SB_QI] * o.yr * o.yr);
    r2 = fmaxf(r2, 1e-16f);
    float lr = f_lg2(r2);
    o.lu = fmaf(sb[SB_K1], lr, sb[SB_K0]);
    o.u = f_ex2(o.lu);
    const float c1 = sb[SB_C1];
    o.I = sb[SB_IE] * f_ex2(fmaf(-c1, o.u, c1));
    o.Iu_r2 = o.I * o.u * f_ex2(-lr);
    return o;
}

__device__ __forceinline__ void sersic_accum(const SersicOut& o, float g, float* __restrict__ T) {
    float gI = g * o.I, gIu = gI * o.u;
    T[SA_T0] += gI; T[SA_T1] += gIu; T[SA_T2] = fmaf(gIu, o.lu, T[SA_T2]);
    float W = g * o.Iu_r2;
    float Wx = W * o.xr, Wy = W * o.yr;
    T[SA_AX] += Wx; T[SA_AY] += Wy;
    T[SA_BXX] = fmaf(Wx, o.xr, T[SA_BXX]); T[SA_BYY] = fmaf(Wy, o.yr, T[SA_BYY]); T[SA_BXY] = fmaf(Wx, o.yr, T[SA_BXY]);
}

// Everything one ray needs.  ADJ = false: returns the surface brightness; ADJ = true: accumulates gbar * dI/d(natural).
template <class V, bool ADJ>
__device__ __forceinline__ float ray_eval(const float* __restrict__ pb, float fj, float fi, float gbar, float* __restrict__ acc) {
    const float step = pb[PB_STEP];
    const float cph = pb[PB_M_C], sph = pb[PB_M_S];
    const float dx = fmaf(fj, step, pb[PB_M_XOFF]), dy = fmaf(fi, step, pb[PB_M_YOFF]);
    const float xr = fmaf(cph, dx, sph * dy), yr = fmaf(cph, dy, -sph * dx);
    const float q = pb[PB_M_Q];
    const float qx = q * xr;
    const float R2 = fmaxf(fmaf(qx, qx, yr * yr), 1e-30f);
    const float rinv = f_rsqrt(R2);
    float axr, ayr;                                  // mass-frame deflection
    // adjoint-only pieces
    float S1r = 0, S1i = 0, S2r = 0, S2i = 0, S0r = 0, S0i = 0, S1fr = 0, S1fi = 0, amp = 0, lbr = 0, kap, dqx = 0, dqy = 0;
    if constexpr (V::MASS == 1) {
        const float ce = qx * rinv, se = yr * rinv;
        const float c2 = fmaf(ce, ce, -se * se), s2 = 2.f * ce * se;
        const float f = pb[PB_M_F], nf2 = -pb[PB_M_F2];
        const float wr = -f * c2, wi = -f * s2, p = 2.f * wr;
        float P0r, P0i;
        knuth<29>(pb + PB_SER_A, p, nf2, wr, wi, P0r, P0i);
        S0r = fmaf(ce, P0r, -se * P0i); S0i = fmaf(ce, P0i, se * P0r);
        lbr = fmaf(-0.5f, f_lg2(R2), pb[PB_M_L2B]);
        const float Pw = f_ex2(pb[PB_M_TM1] * lbr);
        amp = pb[PB_M_A] * Pw;
        axr = amp * S0r; ayr = amp * S0i;
        kap = pb[PB_M_KAPC] * Pw * rinv;
        if constexpr (ADJ) {
            float Q1r, Q1i, Q2r, Q2i;
            knuth<28>(pb + PB_SER_D, p, nf2, wr, wi, Q1r, Q1i);
            knuth<28>(pb + PB_SER_E, p, nf2, wr, wi, Q2r, Q2i);
            const float ewr = fmaf(ce, wr, -se * wi), ewi = fmaf(ce, wi, se * wr);       // E w
            S1r = fmaf(ewr, Q1r, -ewi * Q1i); S1i = fmaf(ewr, Q1i, ewi * Q1r);
            S2r = fmaf(ewr, Q2r, -ewi * Q2i); S2i = fmaf(ewr, Q2i, ewi * Q2r);
            const float e3r = fmaf(ce, c2, -se * s2), e3i = fmaf(ce, s2, se * c2);       // E^3
            S1fr = -fmaf(e3r, Q1r, -e3i * Q1i); S1fi = -fmaf(e3r, Q1i, e3i * Q1r);
        }
    } else {
        const float qp = pb[PB_M_QP], b = pb[PB_M_B];
        kap = 0.5f * b * rinv;
        if (qp < 1e-6f) {                            // SIS limit
            const float ri = f_rsqrt(fmaxf(fmaf(xr, xr, yr * yr), 1e-30f));
            axr = b * xr * ri; ayr = b * yr * ri;
        } else {
            const float bqp = pb[PB_M_BQP];
            const float Aa = qp * xr * rinv, Bb = qp * yr * rinv;
            const float at = atanf(Aa), ath = atanhf(Bb);
            axr = bqp * at; ayr = bqp * ath;
            if constexpr (ADJ) {
                const float iqp = 1.f / qp;
                const float common = -q * iqp * rinv - qp * q * xr * xr * rinv * rinv * rinv;
                const float k3 = q * iqp * iqp * iqp;
                dqx = b * fmaf(k3, at, xr * common * iqp / fmaf(Aa, Aa, 1.f));
                dqy = b * fmaf(k3, ath, yr * common * iqp / fmaf(-Bb, Bb, 1.f));
            }
        }
    }
    const float x = fmaf(fj, step, pb[PB_XFIRST]), y = fmaf(fi, step, pb[PB_XFIRST]);
    const float g1 = pb[PB_G1], g2 = pb[PB_G2];
    float ax = fmaf(cph, axr, -sph * ayr) + fmaf(g1, x, g2 * y);
    float ay = fmaf(sph, axr, cph * ayr) + fmaf(g2, x, -g1 * y);
    // multipoles about the mass centre, lab frame (S7)
    float ct = 0, st = 0, c3 = 0, s3 = 0, c4 = 0, s4 = 0, rinv_m = 0;
    if constexpr (V::MPMASK != 0) {
        rinv_m = f_rsqrt(fmaxf(fmaf(dx, dx, dy * dy), 1e-30f));
        ct = dx * rinv_m; st = dy * rinv_m;
        const float cc2 = fmaf(ct, ct, -st * st), ss2 = 2.f * ct * st;
        c3 = fmaf(cc2, ct, -ss2 * st); s3 = fmaf(ss2, ct, cc2 * st);
        c4 = fmaf(cc2, cc2, -ss2 * ss2); s4 = 2.f * cc2 * ss2;
        if constexpr (V::MPMASK & 1) {
            const float Am = fmaf(pb[PB_C3], c3, pb[PB_S3] * s3), Bm = fmaf(pb[PB_S3], c3, -pb[PB_C3] * s3);
            ax += -0.125f * fmaf(ct, Am, -3.f * st * Bm); ay += -0.125f * fmaf(st, Am, 3.f * ct * Bm);
        }
        if constexpr (V::MPMASK & 2) {
            const float Am = fmaf(pb[PB_C4], c4, pb[PB_S4] * s4), Bm = fmaf(pb[PB_S4], c4, -pb[PB_C4] * s4);
            ax += (-1.f / 15.f) * fmaf(ct, Am, -4.f * st * Bm); ay += (-1.f / 15.f) * fmaf(st, Am, 4.f * ct * Bm);
        }
    }
    float Iray = 0.f, gbx = 0.f, gby = 0.f;          // surface brightness; source-plane gradient of the source light
    if constexpr (V::NSRC) {
        const float* sb = pb + PB_SRC;
        const float px = fmaf(fj, step, sb[SB_XOFF]) - ax, py = fmaf(fi, step, sb[SB_YOFF]) - ay;   // beta - centre
        SersicOut o = sersic_eval(sb, px, py);
        Iray += o.I;
        if constexpr (ADJ) {
            sersic_accum(o, gbar, acc + NA_SRC);
            const float Ixr = -sb[SB_KQ] * o.Iu_r2 * o.xr, Iyr = -sb[SB_KQI] * o.Iu_r2 * o.yr;
            gbx = fmaf(sb[SB_C], Ixr, -sb[SB_S] * Iyr); gby = fmaf(sb[SB_S], Ixr, sb[SB_C] * Iyr);
        }
        if constexpr (V::NMAX >= 0) {
            constexpr int NM = V::NMAX >= 0 ? V::NMAX : 0;
            const float ibs = pb[PB_SHP];
            const float u = px * ibs, v = py * ibs;
            float fu[NM + 1], fv[NM + 1];
            hermite<NM>(u, fu); hermite<NM>(v, fv);
            const float* a = pb + PB_SHP_A;
            float Ish = 0.f;
            if constexpr (!ADJ) {
#pragma unroll
                for (int n2 = 0; n2 <= NM; ++n2) {
                    float row = 0.f;
#pragma unroll
                    for (int n1 = 0; n1 <= NM - n2; ++n1) row = fmaf(a[(n1 + n2) * (n1 + n2 + 1) / 2 + n2], fu[n1], row);
                    Ish = fmaf(row, fv[n2], Ish);
                }
            } else {
                float dfu[NM + 1], dfv[NM + 1];
                dfu[0] = -u * fu[0]; dfv[0] = -v * fv[0];
#pragma unroll
                for (int k = 1; k <= NM; ++k) { dfu[k] = fmaf(c_HD[k], fu[k - 1], -u * fu[k]); dfv[k] = fmaf(c_HD[k], fv[k - 1], -v * fv[k]); }
                float Iu = 0.f, Iv = 0.f;
#pragma unroll
                for (int n2 = 0; n2 <= NM; ++n2) {
                    float row = 0.f, drow = 0.f;
                    const float gfv = gbar * fv[n2];
#pragma unroll
                    for (int n1 = 0; n1 <= NM - n2; ++n1) {
                        const int idx = (n1 + n2) * (n1 + n2 + 1) / 2 + n2;
                        const float ak = a[idx];
                        row = fmaf(ak, fu[n1], row); drow = fmaf(ak, dfu[n1], drow);
                        acc[NA_SHA + idx] = fmaf(gfv, fu[n1], acc[NA_SHA + idx]);
                    }
                    Ish = fmaf(row, fv[n2], Ish); Iu = fmaf(drow, fv[n2], Iu); Iv = fmaf(row, dfv[n2], Iv);
                }
                acc[NA_SHB] = fmaf(gbar, Ish + fmaf(u, Iu, v * Iv), acc[NA_SHB]);
                const float Ibx = Iu * ibs, Iby = Iv * ibs;
                acc[NA_SHX] = fmaf(gbar, Ibx, acc[NA_SHX]); acc[NA_SHY] = fmaf(gbar, Iby, acc[NA_SHY]);
                gbx += Ibx; gby += Iby;
            }
            Iray += Ish;
        }
    }
    if constexpr (V::NLL >= 1) {
        const float* sb = pb + PB_LL0;
        SersicOut o = sersic_eval(sb, fmaf(fj, step, sb[SB_XOFF]), fmaf(fi, step, sb[SB_YOFF]));
        Iray += o.I; if constexpr (ADJ) sersic_accum(o, gbar, acc + NA_LL0);
    }
    if constexpr (V::NLL >= 2) {
        const float* sb = pb + PB_LL1;
        SersicOut o = sersic_eval(sb, fmaf(fj, step, sb[SB_XOFF]), fmaf(fi, step, sb[SB_YOFF]));
        Iray += o.I; if constexpr (ADJ) sersic_accum(o, gbar, acc + NA_LL1);
    }
    if constexpr (ADJ) {
        // mass parameters enter through beta only: d/dtheta_mass = -(gbar grad_beta I_src) . dalpha/dtheta_mass
        const float sx = gbar * gbx, sy = gbar * gby;
        const float srx = fmaf(cph, sx, sph * sy), sry = fmaf(cph, sy, -sph * sx);
        const float sa = fmaf(srx, axr, sry * ayr);
        const float tm1 = V::MASS == 1 ? pb[PB_M_TM1] : 0.f;
        const float izz = f_rcp(fmaxf(fmaf(xr, xr, yr * yr), 1e-30f));
        const float hr = fmaf(-tm1, axr, -xr * kap), hi = fmaf(-tm1, ayr, -yr * kap);
        const float Gr = fmaf(xr, hr, -yr * hi) * izz, Gi = fmaf(xr, hi, yr * hr) * izz;
        const float Jxx = kap + Gr, Jyy = kap - Gr, Jxy = Gi;
        acc[NA_D0] += sa;
        if constexpr (V::MASS == 1) {
            const float rr2 = rinv * rinv;
            acc[NA_DTL] = fmaf(lbr, sa, acc[NA_DTL]);
            acc[NA_DT2] = fmaf(amp, fmaf(srx, S2r, sry * S2i), acc[NA_DT2]);
            acc[NA_D1] = fmaf(sa * xr, xr * rr2, acc[NA_D1]);
            const float Zr = fmaf(2.f, S1r, S0r), Zi = fmaf(2.f, S1i, S0i);
            acc[NA_D2] = fmaf(amp * xr * yr * rr2, fmaf(sry, Zr, -srx * Zi), acc[NA_D2]);
            acc[NA_D3] = fmaf(amp, fmaf(srx, S1fr, sry * S1fi), acc[NA_D3]);
        } else {
            acc[NA_DQS] += fmaf(srx, dqx, sry * dqy);
        }
        acc[NA_DPHI] += fmaf(srx, fmaf(Jxx, yr, -Jxy * xr) - ayr, sry * (fmaf(Jxy, yr, -Jyy * xr) + axr));
        acc[NA_VX] += fmaf(Jxx, srx, Jxy * sry); acc[NA_VY] += fmaf(Jxy, srx, Jyy * sry);
        acc[NA_G1] -= fmaf(sx, x, -sy * y); acc[NA_G2] -= fmaf(sx, y, sy * x);
        if constexpr (V::MPMASK != 0) {
            float Atot = 0.f;
            if constexpr (V::MPMASK & 1) {
                acc[NA_C3] += 0.125f * fmaf(sx, fmaf(ct, c3, 3.f * st * s3), sy * fmaf(st, c3, -3.f * ct * s3));
                acc[NA_S3] += 0.125f * fmaf(sx, fmaf(ct, s3, -3.f * st * c3), sy * fmaf(st, s3, 3.f * ct * c3));
                Atot += fmaf(pb[PB_C3], c3, pb[PB_S3] * s3);
            }
            if constexpr (V::MPMASK & 2) {
                acc[NA_C4] += (1.f / 15.f) * fmaf(sx, fmaf(ct, c4, 4.f * st * s4), sy * fmaf(st, c4, -4.f * ct * s4));
                acc[NA_S4] += (1.f / 15.f) * fmaf(sx, fmaf(ct, s4, -4.f * st * c4), sy * fmaf(st, s4, 4.f * ct * c4));
                Atot += fmaf(pb[PB_C4], c4, pb[PB_S4] * s4);
            }
            const float proj = Atot * rinv_m * fmaf(ct, sy, -st * sx);
            acc[NA_MCX] = fmaf(-st, proj, acc[NA_MCX]); acc[NA_MCY] = fmaf(ct, proj, acc[NA_MCY]);
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
    int ph, a, b, oa, ob, idx, i1, j1, di, dj;
    float half;
    __device__ __forceinline__ PlaneIter(const Geom& G, int n_chunk, int RPT) {
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
    __device__ __forceinline__ float fj(const Geom& G) const { return (float)(G.s * j1 + b) - half; }
    __device__ __forceinline__ float fi(const Geom& G) const { return (float)(G.s * i1 + a) - half; }
    __device__ __forceinline__ size_t offset(const Geom& G) const { return (size_t)(i1 + oa) * G.Wp + (j1 + ob); }
};

// Steps B + C.  Writes the plane interior and zeroes this CTA's share of the plane border.
template <class V, int NT>
__global__ void __launch_bounds__(NT) gl_ray_fwd_kernel(const __grid_constant__ Geom G, const float* __restrict__ pbg,
                                                        float* __restrict__ ray, int RPT, int n_chunk) {
    __shared__ __align__(16) float pb[PB_STRIDE];
    const int p = blockIdx.y;
    const float* src = pbg + (size_t)p * PB_STRIDE;
    for (int k = threadIdx.x; k < V::PB_NEED; k += blockDim.x) pb[k] = src[k];
    __syncthreads();
    PlaneIter it(G, n_chunk, RPT);
    float* out = ray + (size_t)p * ray_stride(G) + (size_t)it.ph * G.Hp * G.Wp;
    {
        const int ck = blockIdx.x - it.ph * n_chunk, tot = G.Hp * G.Wp;
        for (int e = ck * blockDim.x + threadIdx.x; e < tot; e += n_chunk * blockDim.x) {
            const int r = e / G.Wp, cc = e - r * G.Wp;
            if (r < it.oa || r >= it.oa + G.N || cc < it.ob || cc >= it.ob + G.N) out[e] = 0.f;
        }
    }
    const int NN = G.N * G.N;
    const bool valid = pb[PB_VALID] != 0.f;
#pragma unroll 2
    for (int r = 0; r < RPT; ++r) {
        if (it.idx < NN) {
            float v = ray_eval<V, false>(pb, it.fj(G), it.fi(G), 0.f, nullptr);
            out[it.offset(G)] = valid ? v : 0.f;
        }
        it.next(G);
    }
}

// Per-ray part of step F.  gbar: plane layout; nap: [Pc][gridDim.x][V::NA].
template <class V, int NT>
__global__ void __launch_bounds__(NT) gl_ray_adj_kernel(const __grid_constant__ Geom G, const float* __restrict__ pbg,
                                                        const float* __restrict__ gbar, float* __restrict__ nap, int RPT,
                                                        int n_chunk) {
    __shared__ __align__(16) float pb[PB_STRIDE];
    __shared__ float red[NT / 32][V::NA];
    const int p = blockIdx.y;
    const float* src = pbg + (size_t)p * PB_STRIDE;
    for (int k = threadIdx.x; k < V::PB_NEED; k += blockDim.x) pb[k] = src[k];
    __syncthreads();
    PlaneIter it(G, n_chunk, RPT);
    const float* gb = gbar + (size_t)p * ray_stride(G) + (size_t)it.ph * G.Hp * G.Wp;
    const int NN = G.N * G.N;
    float acc[V::NA];
#pragma unroll
    for (int k = 0; k < V::NA; ++k) acc[k] = 0.f;
    if (pb[PB_VALID] != 0.f) {
        for (int r = 0; r < RPT; ++r) {
            if (it.idx < NN) ray_eval<V, true>(pb, it.fj(G), it.fi(G), gb[it.offset(G)], acc);
            it.next(G);
        }
    }
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5, nw = blockDim.x >> 5;
#pragma unroll
    for (int k = 0; k < V::NA; ++k) {
        float v = warp_sum(acc[k]);
        if (lane == 0) red[w][k] = v;
    }
    __syncthreads();
    float* o = nap + ((size_t)p * gridDim.x + blockIdx.x) * V::NA;
    for (int k = threadIdx.x; k < V::NA; k += blockDim.x) {
        float s = 0.f;
        for (int ww = 0; ww < nw; ++ww) s += red[ww][k];
        o[k] = s;
    }
}

}  // namespace gl
