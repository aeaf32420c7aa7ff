// gl_common.cuh -- layouts shared by the kernels of libgigalens (product path; shares nothing with oracle/).
//
// Data layout in HBM:
//   PB   [Pc][PB_STRIDE] fp32   per-particle block of derived scalars written by gl_unpack_kernel (step A)
//   RAY  [Pc][s*s][Hp][Wp] fp32 supersampled surface-brightness image (step B+C) as s*s PHASE PLANES: ray (i, j) =
//                               (s*i1 + a, s*j1 + b) lives in plane (a, b) at row i1 + o_a, column j1 + o_b with
//                               o_a = (a + c) div s; everything outside that N x N interior is ZERO.  The shift and
//                               the zero border turn step D into s*s plain "valid" stride-1 correlations that need no
//                               bounds checks and read 16-byte-aligned row segments.  Reused for gbar_ray (step F).
//   GPIX [Pc][Hg][Wg]    fp32   g_pix = -(model-obs)/sigma^2 (step E), zero-padded by U-1 on every side: input of the
//                               transposed step D
//   CHI  [Pc][n_ctile]   fp32   per-band chi-square partials, summed in fixed order by gl_finalize_kernel
//   NAP  [Pc][n_chunk][NA] fp32 per-chunk "natural" gradient accumulators of the adjoint (step F)
//   SYS  per system: kt (flipped pre-boxed PSF, phase-major), w = 1/sigma^2, sum(ln sigma)
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace gl {

// ----------------------------------------------------------------------------- particle block (PB)
enum : int {
    PB_VALID = 0,
    PB_M_XOFF = 1, PB_M_YOFF = 2,       // -x0, -y0 of the mass centre (ray coordinates are relative to the grid centre)
    PB_M_C = 3, PB_M_S = 4,             // cos phi, sin phi of the mass frame
    PB_M_Q = 5, PB_M_B = 6, PB_M_T = 7, PB_M_F = 8, PB_M_L2B = 9, PB_M_A = 10,
    PB_M_QP = 11, PB_M_BQP = 12,        // SIE: q' = sqrt(1-q^2), b/q'
    PB_M_F2 = 13, PB_M_TM1 = 14, PB_M_KAPC = 15,   // f^2, t-1, (2-t)/2 * b
    PB_G1 = 16, PB_G2 = 17, PB_C3 = 18, PB_S3 = 19, PB_C4 = 20, PB_S4 = 21,
    PB_XFIRST = 22, PB_STEP = 23,       // ray grid: x_j = x_first + fj*step with fj = j - (M-1)/2, x_first = 0
    PB_SRC = 24,                        // Sersic block, 16 floats
    PB_SHP = 40,                        // +0 1/beta_s ; coefficients a_k/beta_s from PB_SHP_A
    PB_SHP_A = 44,
    PB_LL0 = 112, PB_LL1 = 128,
    PB_SER_A = 144,                     // a_n, n = 0..31 (zero beyond epl_terms)
    PB_SER_D = 176,                     // d_m = (m+1) a_{m+1}
    PB_SER_E = 208,                     // e_m = L_{m+1} a_{m+1}
    PB_SER_M1 = 240, PB_SER_M2 = 241,   // series bands: 4*M1 steps in T, 4*M2 steps in fp32 above them, the rest skipped
    PB_M_H1 = 242, PB_M_H0 = 243,       // amplitude A (b/R)^(t-1) = 2^(H1 log2 R^2 + H0): H1 = -(t-1)/2, H0 = (t-1) log2 b + log2 A
    PB_SRC1 = 244,                      // second source Sersic block (same source plane), 16 floats
    PB_LL2 = 260,                       // third lens-light Sersic block, 16 floats
    PB_STRIDE = 276
};
// Sersic block offsets
// The component frame is stored PRE-SCALED: x' = sqrt(q) x_r = A11 px + A12 py, y' = y_r / sqrt(q) = A21 px + A22 py, so that
// r^2 = q x_r^2 + y_r^2 / q = x'^2 + y'^2 costs two FP64 operations instead of four.  KQ = (b_n/n) sqrt(q), KQI = (b_n/n)/sqrt(q);
// C, S (unscaled cos/sin phi) rotate source-plane gradients back.  The adjoint's moment sums are taken in (x', y') and
// unscaled per particle in gl_finalize_kernel (sersic_chain).
enum : int { SB_XOFF = 0, SB_YOFF = 1, SB_C = 2, SB_S = 3, SB_A11 = 4, SB_A12 = 5, SB_K1 = 6, SB_K0 = 7,
             SB_C1 = 8, SB_IE = 9, SB_KQ = 10, SB_KQI = 11, SB_A21 = 12, SB_A22 = 13,
             SB_ETA = 14 };             // PB_SRC1 only: eta2, the deflection scale of the second source's plane (1 on one plane)

// ----------------------------------------------------------------------------- natural accumulators (NA)
// Per-ray sums the adjoint kernel produces; gl_finalize_kernel applies the per-particle chain rule in fp64.
enum : int {
    NA_D0 = 0, NA_DTL = 1, NA_DT2 = 2, NA_D1 = 3, NA_D2 = 4, NA_D3 = 5, NA_DPHI = 6, NA_VX = 7, NA_VY = 8,
    NA_DQS = 9,                          // SIE only: sum s_r . dalpha/dq|b
    NA_G1 = 10, NA_G2 = 11,
    NA_C3 = 12, NA_S3 = 13, NA_C4 = 14, NA_S4 = 15, NA_MCX = 16, NA_MCY = 17,
    NA_SRC = 18,                         // 8: T0 T1 T2 AX AY BXX BYY BXY
    NA_SHB = 26, NA_SHX = 27, NA_SHY = 28,
    NA_LL0 = 29, NA_LL1 = 37,
    NA_SRC1 = 45, NA_LL2 = 53,           // second source / third lens-light block (8 each, like NA_SRC)
    NA_ETA = 61,                         // second source plane: -sum gbar grad_beta I_src2 . alpha  (= d logL / d eta2)
    NA_SHA = 62,                         // Nc coefficient sums
    NA_MAX = 62 + 66
};
enum : int { SA_T0 = 0, SA_T1 = 1, SA_T2 = 2, SA_AX = 3, SA_AY = 4, SA_BXX = 5, SA_BYY = 6, SA_BXY = 7 };

// ----------------------------------------------------------------------------- compile-time model variant
template <int MASS_, int MPMASK_, int NSRC_, int NMAX_, int NLL_>
struct Variant {
    static constexpr int MASS = MASS_;       // 0 SIE, 1 EPL
    static constexpr int MPMASK = MPMASK_;   // multipole bits
    static constexpr int NSRC = NSRC_;
    static constexpr int NMAX = NMAX_;       // -1: no shapelets
    static constexpr int NLL = NLL_;
    static constexpr int NCOEF = NMAX_ >= 0 ? (NMAX_ + 1) * (NMAX_ + 2) / 2 : 0;
    static constexpr int NA = NMAX_ >= 0 ? NA_SHA + NCOEF : NA_SHA;            // accumulators written per chunk
    static constexpr int PB_NEED = (MASS_ == 1 || NSRC_ > 1 || NLL_ > 2) ? PB_STRIDE : PB_SER_A;   // floats of PB a CTA stages
};

struct Geom {            // launch-invariant geometry, passed by value
    int N, s, M, K, c;   // pixels/side, supersample, rays/side, psf taps/side, half-width of the ray-level kernel
                         // ((K-1)/2 for psf_grid 0, s*(K-1)/2 for psf_grid 1)
    int KE, pgrid;       // ray-level taps per side of the effective kernel (K+s-1 or s*K); psf_grid
    int noise_model;     // 0 fixed sigma map, 1 variance sigma^2 + max(model,0) * inv_texp (SYS w then holds sigma^2)
    double inv_texp;
    int KEp, U;          // padded k_eff taps per side (multiple of s), taps per phase per side
    int n_terms;         // EPL series terms kept (2..30)
    double delta2;       // pix_scale^2 (fp64 product of the fp32 pix_scale)
    int UP;              // U rounded up to a multiple of the tap rows one conv thread handles
    int Hp, Wp;          // rows / row pitch of one padded phase plane of RAY
    int Hg, Wg, PADg;    // rows / row pitch / border of the padded GPIX image
    int binned;          // 1 (psf_grid 1, dedicated path): step D runs on the BINNED image held in phase plane 0 and the
                         // transpose writes plane 0 only; every plane's gbar is that plane (gl_ray_adj_kernel reads plane 0)
};
__host__ __device__ inline int phase_shift(const Geom& G, int a) { return (a + G.c) / G.s; }      // o_a
__host__ __device__ inline size_t ray_stride(const Geom& G) { return (size_t)G.s * G.s * G.Hp * G.Wp; }
__host__ __device__ inline size_t gpix_stride(const Geom& G) { return (size_t)G.Hg * G.Wg; }

// ----------------------------------------------------------------------------- scaled shapelet basis (gl_ray.cuh)
// psi_k = phi_k / c_k with c_k = sqrt(2^k / k!); the per-coefficient factor c_n1 c_n2 is folded into the coefficients of
// PB by step A and into the coefficient sums by the finalize.  Coefficient k = (n1 + n2)(n1 + n2 + 1)/2 + n2.
#define GL_HC_TABLE {1.0, 1.4142135623730951, 1.4142135623730951, 1.1547005383792515, 0.816496580927726, 0.5163977794943222, \
                     0.29814239699997197, 0.15936381457791915, 0.07968190728895957, 0.037562411321267405,                   \
                     0.01679842102263232, 0.007162870791336714}
__constant__ double d_HC[12] = GL_HC_TABLE;
__host__ __device__ inline void shp_orders(int k, int& n1, int& n2) {
    int o = 0;
    while ((o + 1) * (o + 2) / 2 <= k) ++o;
    n2 = k - o * (o + 1) / 2; n1 = o - n2;
}
__device__ __forceinline__ double shp_scale(int k) { int n1, n2; shp_orders(k, n1, n2); return d_HC[n1] * d_HC[n2]; }
inline double shp_scale_host(int k) { static const double hc[12] = GL_HC_TABLE; int n1, n2; shp_orders(k, n1, n2); return hc[n1] * hc[n2]; }

template <class T>
__device__ __forceinline__ T warp_sum(T v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

}  // namespace gl
