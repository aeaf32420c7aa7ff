// gl_probe.cuh -- issue-rate probes of the SM pipes the path is bound by (FP32 FMA, FP64 FMA, MUFU), used by
// bench.py to put a MEASURED ALU peak beside the one derived from unit counts and clocks (SURVEY 8(d):
// MEASURED_PEAKS.json holds neither).  Measurement utility, not part of the hot path.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace gl {

constexpr int PROBE_CHAINS = 8;     // independent dependency chains per thread
constexpr int PROBE_INNER = 64;     // FMAs per chain per outer iteration

// kind 0: FP32 FMA;  1: FP64 FMA;  2: MUFU ex2;  3: FP32 and FP64 FMA interleaved 1:1 (counts both)
template <int KIND>
__global__ void __launch_bounds__(256) gl_probe_kernel(int n_outer, float seed, float* __restrict__ sink) {
    float a[PROBE_CHAINS]; double d[PROBE_CHAINS];
#pragma unroll
    for (int k = 0; k < PROBE_CHAINS; ++k) { a[k] = seed + k + threadIdx.x * 1e-3f; d[k] = (double)a[k]; }
    const float m = 0.999f + seed * 1e-6f, c = 1e-3f;
    const double md = (double)m, cd = (double)c;
    for (int o = 0; o < n_outer; ++o) {
#pragma unroll
        for (int i = 0; i < PROBE_INNER; ++i) {
#pragma unroll
            for (int k = 0; k < PROBE_CHAINS; ++k) {
                if constexpr (KIND == 0 || KIND == 3) a[k] = fmaf(a[k], m, c);
                if constexpr (KIND == 1 || KIND == 3) d[k] = fma(d[k], md, cd);
                if constexpr (KIND == 2) asm volatile("ex2.approx.ftz.f32 %0, %0;" : "+f"(a[k]));
            }
        }
    }
    float s = 0.f;
#pragma unroll
    for (int k = 0; k < PROBE_CHAINS; ++k) s += a[k] + (float)d[k];
    if (s == 12345.678f) sink[0] = s;       // never true in practice; keeps the chains alive
}

}  // namespace gl
