// gl_math.cuh -- scalar primitives of the per-ray kernels for the two arithmetic modes of libgigalens:
//   Real<float>   FP32 FMA pipe + MUFU (ex2 / lg2 / rsqrt / rcp approximations), the "fast" mode;
//   Real<double>  FP64 FMA pipe; MUFU and FP32 results are used only as SEEDS that a Newton step or a table +
//                 polynomial brings to ~1e-15 relative, so every per-ray value is fp64-accurate.  This is the
//                 mode that meets the north_star tolerances on every gradient component.
// Product path only; shares nothing with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace gl {

__device__ __forceinline__ float f_ex2(float x) { float y; asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ float f_lg2(float x) { float y; asm("lg2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ float f_rsqrt(float x) { float y; asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ float f_rcp(float x) { float y; asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }

// ----------------------------------------------------------------------------- fp64 exp2 / log2
// exp2(x) = 2^n * 2^(j/64) * P(r),  x = n + j/64 + r, |r| <= 1/128;  P = degree-5 Taylor of 2^r (error < 4e-17).
// log2(x) = e + log2(c_j) + log1p(r)/ln2,  x = 2^e m, m in [1,2), c_j = 1 + (j+0.5)/128, r = m/c_j - 1,
//           |r| <= 1/256 (+ rounding of the tabulated 1/c_j); log1p by a degree-7 alternating series (error < 1e-18).
// Tables are generated on the device in fp64 once per call by gl_prep_kernel (block 0) into the workspace and
// staged into shared memory by the kernels that use them (they are indexed per LANE): 64 + 2*128 doubles = 2.5 KB.
constexpr int EXP2_TAB = 64, LOG2_TAB = 128;
constexpr int MATH_TAB_DOUBLES = EXP2_TAB + 2 * LOG2_TAB;      // [2^(j/64)] [rc_j = fl(1/c_j)] [-log2 rc_j]

__device__ inline void fill_math_tab(double* g) {               // any block shape
    for (int k = threadIdx.x; k < EXP2_TAB; k += blockDim.x) g[k] = exp2((double)k / EXP2_TAB);
    for (int k = threadIdx.x; k < LOG2_TAB; k += blockDim.x) {
        const double rc = 1.0 / (1.0 + (k + 0.5) / LOG2_TAB);
        g[EXP2_TAB + k] = rc; g[EXP2_TAB + LOG2_TAB + k] = -log2(rc);
    }
}

struct MathTab {                       // pointers into the CTA's shared-memory copy
    const double* e2; const double* rc; const double* lc;
};
__device__ __forceinline__ void stage_math_tab(double* sm, const double* __restrict__ g) {
    for (int k = threadIdx.x; k < MATH_TAB_DOUBLES; k += blockDim.x) sm[k] = g[k];
}
__device__ __forceinline__ MathTab math_tab(const double* sm) { return MathTab{sm, sm + EXP2_TAB, sm + EXP2_TAB + LOG2_TAB}; }

__device__ __forceinline__ double d_exp2(const MathTab& tb, double x) {
    // clamp: 2^-1000 is 0 for every use here, 2^1000 never occurs for valid particles
    x = fmin(fmax(x, -1000.0), 1000.0);
    const double magic = 6755399441055744.0;                   // 1.5 * 2^52: adding it rounds to an integer in the low word
    const double kd = fma(x, 64.0, magic);
    const int k = __double2loint(kd);                          // k = rint(64 x)
    const double r = fma(kd - magic, -0.015625, x);            // x - k/64, exact
    const int j = k & 63, n = k >> 6;
    // 2^r = exp(r ln2), |r ln2| <= 0.0055: degree 5
    double p = 1.3333558146428443e-3;                          // ln2^5/120
    p = fma(p, r, 9.6181291076284772e-3);                      // ln2^4/24
    p = fma(p, r, 5.5504108664821580e-2);                      // ln2^3/6
    p = fma(p, r, 2.4022650695910071e-1);                      // ln2^2/2
    p = fma(p, r, 6.9314718055994531e-1);                      // ln2
    const double t = tb.e2[j];
    const double y = fma(t * r, p, t);
    // scale by 2^n through the exponent field (|n| <= 1001 keeps the result normal or flushes gracefully via two steps)
    const int hi = __double2hiint(y), lo = __double2loint(y);
    const int n1 = n >> 1, n2 = n - n1;
    const double y1 = __hiloint2double(hi + (n1 << 20), lo);
    return y1 * __hiloint2double((1023 + n2) << 20, 0);
}

__device__ __forceinline__ double d_log2(const MathTab& tb, double x) {
    // x > 0, normal (callers floor their arguments)
    const int hi = __double2hiint(x), lo = __double2loint(x);
    const int e = (hi >> 20) - 1023;
    const int j = (hi >> 13) & 127;                            // top 7 mantissa bits
    const double m = __hiloint2double((hi & 0x000fffff) | 0x3ff00000, lo);
    const double r = fma(m, tb.rc[j], -1.0);
    // log1p(r)/ln2 = r * (c1 + c2 r + ... ), c_k = (-1)^(k+1) / (k ln2)
    double p = 2.0609929155084896e-1;                          //  1/(7 ln2)
    p = fma(p, r, -2.4044917347599045e-1);                     // -1/(6 ln2)
    p = fma(p, r, 2.8853900817779268e-1);                      //  1/(5 ln2)
    p = fma(p, r, -3.6067376022224085e-1);                     // -1/(4 ln2)
    p = fma(p, r, 4.8089834696298783e-1);                      //  1/(3 ln2)
    p = fma(p, r, -7.2134752044448170e-1);                     // -1/(2 ln2)
    p = fma(p, r, 1.4426950408889634e+0);                      //  1/ln2
    return fma(p, r, tb.lc[j] + (double)e);
}

// 1/sqrt(x) and 1/x: MUFU seed (2^-22) + one Newton step in fp64 (-> ~2^-43) + a second cheap step (-> full).
__device__ __forceinline__ double d_rsqrt(double x) {
    const double y0 = (double)f_rsqrt((float)x);
    const double h = 0.5 * y0;
    double e = fma(-x * y0, y0, 1.0);
    double y = fma(h, e, y0);                                   // error ~ 3/8 e^2 ~ 2e-14
    e = fma(-x * y, y, 1.0);
    return fma(0.5 * y, e, y);
}
__device__ __forceinline__ double d_rcp(double x) {
    const double y0 = (double)f_rcp((float)x);
    double e = fma(-x, y0, 1.0);
    double y = fma(y0, e, y0);
    e = fma(-x, y, 1.0);
    return fma(y, e, y);
}

// ----------------------------------------------------------------------------- traits
template <class T> struct Real;

template <> struct Real<float> {
    using Tab = int;                                            // unused
    static __device__ __forceinline__ float ex2(const Tab&, float x) { return f_ex2(x); }
    static __device__ __forceinline__ float lg2(const Tab&, float x) { return f_lg2(x); }
    static __device__ __forceinline__ float rsqrt(float x) { return f_rsqrt(x); }
    static __device__ __forceinline__ float rcp(float x) { return f_rcp(x); }
    static __device__ __forceinline__ float fma(float a, float b, float c) { return fmaf(a, b, c); }
    static __device__ __forceinline__ float max(float a, float b) { return fmaxf(a, b); }
    static __device__ __forceinline__ float atan(float x) { return atanf(x); }
    static __device__ __forceinline__ float atanh(float x) { return atanhf(x); }
    static __device__ __forceinline__ float tiny() { return 1e-30f; }
};

template <> struct Real<double> {
    using Tab = MathTab;
    static __device__ __forceinline__ double ex2(const Tab& t, double x) { return d_exp2(t, x); }
    static __device__ __forceinline__ double lg2(const Tab& t, double x) { return d_log2(t, x); }
    static __device__ __forceinline__ double rsqrt(double x) { return d_rsqrt(x); }
    static __device__ __forceinline__ double rcp(double x) { return d_rcp(x); }
    static __device__ __forceinline__ double fma(double a, double b, double c) { return ::fma(a, b, c); }
    static __device__ __forceinline__ double max(double a, double b) { return fmax(a, b); }
    static __device__ __forceinline__ double atan(double x) { return ::atan(x); }
    static __device__ __forceinline__ double atanh(double x) { return ::atanh(x); }
    static __device__ __forceinline__ double tiny() { return 1e-300; }
};

}  // namespace gl
