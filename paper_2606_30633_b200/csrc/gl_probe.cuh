// gl_probe.cuh -- issue-rate probes of the SM pipes the path is bound by (FP32 FMA, FP64 FMA, MUFU), used by
// bench.py to put a MEASURED ALU peak beside the one derived from unit counts and clocks (SURVEY 8(d):
// MEASURED_PEAKS.json holds neither).  Measurement utility, not part of the hot path.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace gl {

constexpr int PROBE_CHAINS = 8;     // independent dependency chains per thread
constexpr int PROBE_INNER = 64;     // FMAs per chain per outer iteration

// kind 0: FP32 FMA;  1: FP64 FMA;  2: MUFU ex2;  3: FP32 and FP64 FMA interleaved 1:1 (counts both);
// 4: FP64 FMA whose three operands are distinct registers in every chain (kinds 0-3 share multiplier and addend across
//    the chains, which lets the operand-reuse cache feed the pipe: kind 4 is what ordinary fp64 code can sustain)
// 5: FP64 tensor-core MMA (mma.sync.m8n8k4.f64, SASS DMMA), 8 independent accumulator pairs per thread; one warp
//    instruction is 8 x 8 x 4 = 256 FMAs = 8 lane-operations per lane (counted so);
// 7: FP64 FMA with two distinct vector-register operands and one warp-uniform operand (uniform register / constant);
// 8: FP64 FMA with three vector-register operands of which the multiplier is the same register in consecutive instructions
//    (what the operand-reuse cache can serve): 7 and 8 separate "three operands" from "three register-file reads";
// 6: kind 5 and kind 1 interleaved 1:1 (one DMMA, one DFMA, both counted): do the tensor and the vector FP64 paths add up?
template <int KIND>
__global__ void __launch_bounds__(256) gl_probe_kernel(int n_outer, float seed, float* __restrict__ sink) {
    float a[PROBE_CHAINS]; double d[PROBE_CHAINS], e[PROBE_CHAINS], f[PROBE_CHAINS];
    [[maybe_unused]] double t0[PROBE_CHAINS], t1[PROBE_CHAINS];
#pragma unroll
    for (int k = 0; k < PROBE_CHAINS; ++k) {
        a[k] = seed + k + threadIdx.x * 1e-3f; d[k] = (double)a[k];
        e[k] = 0.999 + 1e-12 * (double)(threadIdx.x + k) * (double)seed;          // per-thread values: not uniform registers
        f[k] = 1e-3 * (1.0 + 1e-6 * (double)threadIdx.x) * (double)seed * (k + 1);
        t0[k] = f[k]; t1[k] = -f[k];
    }
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
                if constexpr (KIND == 4) d[k] = fma(d[k], e[k], f[k]);
                if constexpr (KIND == 7) d[k] = fma(d[k], e[k], cd);            // two distinct vector registers + a uniform addend
                if constexpr (KIND == 8) d[k] = fma(d[k], e[0], f[k]);          // three vector registers, the multiplier shared by neighbours
                if constexpr (KIND == 5 || KIND == 6)
                    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0, %1}, {%2}, {%3}, {%0, %1};"
                                 : "+d"(t0[k]), "+d"(t1[k]) : "d"(e[k]), "d"(f[k]));
                if constexpr (KIND == 6) d[k] = fma(d[k], md, cd);
            }
        }
    }
    float s = 0.f;
#pragma unroll
    for (int k = 0; k < PROBE_CHAINS; ++k) {
        s += a[k] + (float)d[k];
        if constexpr (KIND == 5 || KIND == 6) s += (float)(t0[k] + t1[k]);
    }
    if (s == 12345.678f) sink[0] = s;       // never true in practice; keeps the chains alive
}

}  // namespace gl
