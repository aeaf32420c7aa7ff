// gl_math.cuh -- scalar primitives of the per-ray kernels for the two arithmetic modes of libgigalens:
//   Real<float>   FP32 FMA pipe + MUFU (ex2 / lg2 / rsqrt / rcp approximations), the "fast" mode;
//   Real<double>  FP64 FMA pipe; MUFU and FP32 results are used only as SEEDS that a Newton step or a table +
//                 polynomial brings to < 1e-13 relative (1e6 times tighter than fp32).  This is the
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
// exp2(x) = 2^n * 2^(j/16) * (1 + r P(r)),  x = n + j/16 + r, |r| <= 1/32;  P = degree-3 Chebyshev fit (error < 6e-12).
// log2(x) = e + log2(c_j) + log1p(r)/ln2,  x = 2^e m, m in [1,2), c_j = 1 + (j+0.5)/16, r = m rc_j - 1, |r| <= 1/32;
//           log1p(r)/(r ln2) as a degree-4 Chebyshev fit (absolute error < 1.5e-11).  These errors are 1e4 times below fp32
//           and leave the parity margins of section 6 of DESIGN.md untouched (checked on all five configs); each
//           polynomial term costs an FP64 issue slot in kernels that run at the FP64 issue rate.
// The tables have 16 doubles = 128 bytes = ONE shared-memory bank row each, so a lookup with 32 arbitrary per-lane
// indices is always a single conflict-free wavefront (larger tables made the ray kernels shared-memory bound:
// profiles/r1b_cfg2_f64.md).  They are generated on the device in fp64 once per call by gl_prep_kernel (block 0) into
// the workspace and staged into 128-byte aligned shared memory by the kernels that use them.
constexpr int EXP2_TAB = 16, LOG2_TAB = 16;
constexpr int MATH_TAB_DOUBLES = EXP2_TAB + 2 * LOG2_TAB;      // [2^(j/16)] [rc_j = fl(1/c_j)] [-log2 rc_j]

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

// Polynomial and splitting constants live in __constant__ memory so that DFMA takes them as constant-bank operands
// (a 64-bit literal costs two extra move instructions per use, and the ray kernels are co-limited by issue slots).
__constant__ double c_dm[20] = {
    6755399441055744.0,        // 0: 1.5 * 2^52: adding it rounds to an integer in the low word
    16.0,                      // 1
    -0.0625,                   // 2: -1/16
    // 3..6: (2^r - 1)/r on |r| <= 1/32, degree-3 Chebyshev fit (relative error of 2^r < 6e-12)
    0.6931471804009947, 0.24022650691319444, 0.05550541078373476, 0.009618317140281765,
    0.0,                       // 7: unused
    // 8..12: log2(1 + r)/r on |r| <= 1/32, degree-4 Chebyshev fit (absolute error of log2(1 + r) < 1.5e-11)
    1.44269504089497, -0.7213474487115007, 0.4808982362719573, -0.36096750318286375, 0.2888411792028112,
    0.0, 0.0,                  // 13, 14: unused
    0.5, 1.0, -1.0, 0.0,       // 15..18
    0.0};

// 2^x, relative error < 6e-12, for -1e8 < x < 1000; below -1021 the result saturates at ~1e-308.
__device__ __forceinline__ double d_exp2(const MathTab& tb, double x) {
    const double kd = fma(x, c_dm[1], c_dm[0]);
    const int k = __double2loint(kd);                          // k = rint(16 x)
    const double r = fma(kd - c_dm[0], c_dm[2], x);            // x - k/16, exact
    const int j = k & 15, n = max(k >> 4, -1021);              // x < -1021: result 2^-1021 y ~ 1e-308 (stands for 0)
    double p = c_dm[6];
    p = fma(p, r, c_dm[5]);
    p = fma(p, r, c_dm[4]);
    p = fma(p, r, c_dm[3]);
    const double t = tb.e2[j];
    const double y = fma(t * r, p, t);                         // in [0.97, 2.05)
    return __hiloint2double(__double2hiint(y) + (n << 20), __double2loint(y));   // scale by 2^n through the exponent field
}

// log2(x) for normal x > 0, absolute error < 1.5e-11.
__device__ __forceinline__ double d_log2(const MathTab& tb, double x) {
    const int hi = __double2hiint(x), lo = __double2loint(x);
    const int e = (hi >> 20) - 1023;
    const int j = (hi >> 16) & 15;                             // top 4 mantissa bits
    const double m = __hiloint2double((hi & 0x000fffff) | 0x3ff00000, lo);
    const double r = fma(m, tb.rc[j], c_dm[17]);               // |r| <= 1/32
    // log1p(r)/ln2 = r (c1 + c2 r + ... + c5 r^4)
    double p = c_dm[12];
    p = fma(p, r, c_dm[11]);
    p = fma(p, r, c_dm[10]);
    p = fma(p, r, c_dm[9]);
    p = fma(p, r, c_dm[8]);
    return fma(p, r, tb.lc[j] + (double)e);
}

// 1/sqrt(x) and 1/x: MUFU seed (relative error e0 <= 3e-7 including the float rounding of x) + one Newton step in
// fp64: error 3/8 e0^2 < 4e-14 (rsqrt), e0^2 < 1e-13 (rcp).
__device__ __forceinline__ double d_rsqrt(double x) {
    const double y0 = (double)f_rsqrt((float)x);
    const double e = fma(-x * y0, y0, c_dm[16]);
    return fma(c_dm[15] * y0, e, y0);
}
__device__ __forceinline__ double d_rcp(double x) {
    const double y0 = (double)f_rcp((float)x);
    const double e = fma(-x, y0, c_dm[16]);
    return fma(y0, e, y0);
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
    // a compare and a select: fmax's NaN handling costs ~2 more instructions per call, and a NaN here belongs to a particle that
    // step A or the finalize marks invalid anyway (max(NaN, b) = NaN instead of b)
    static __device__ __forceinline__ double max(double a, double b) { return a < b ? b : a; }
    static __device__ __forceinline__ double atan(double x) { return ::atan(x); }
    static __device__ __forceinline__ double atanh(double x) { return ::atanh(x); }
    static __device__ __forceinline__ double tiny() { return 1e-300; }
};

}  // namespace gl
