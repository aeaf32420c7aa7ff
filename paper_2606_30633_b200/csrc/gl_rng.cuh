// gl_rng.cuh -- counter-based draws for the SVI / HMC consumers (reading S22, DESIGN.md
// section 18): Philox4x32-10 bits (Salmon et al., SC'11), key = the 64-bit seed, counter = (step lo, step hi, row,
// stream_id << 24 | block); one counter yields four fp32 standard normals of a row (fp64 Box-Muller on the word pairs
// (0,1), (2,3)) or one ln u.  Stateless: any (seed, step, stream, row, element) can be regenerated in isolation, so the
// draws need no state buffer, no host round trip and are independent of the launch geometry.
// Product path only; shares nothing with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace gl {

struct Philox4 { uint32_t w[4]; };

__device__ __forceinline__ Philox4 philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, uint32_t k0, uint32_t k1) {
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        if (r > 0) { k0 += 0x9E3779B9u; k1 += 0xBB67AE85u; }
        const uint32_t hi0 = __umulhi(0xD2511F53u, c0), lo0 = 0xD2511F53u * c0;
        const uint32_t hi1 = __umulhi(0xCD9E8D57u, c2), lo1 = 0xCD9E8D57u * c2;
        const uint32_t n0 = hi1 ^ c1 ^ k0, n2 = hi0 ^ c3 ^ k1;
        c0 = n0; c1 = lo1; c2 = n2; c3 = lo0;
    }
    return Philox4{{c0, c1, c2, c3}};
}

__device__ __forceinline__ double rng_uniform(uint32_t w) { return ((double)w + 0.5) * 2.3283064365386963e-10; }   // 2^-32

// out [n_rows][n_cols] fp32 standard normals.  One thread per (row, block of 4 elements).
__global__ void gl_draw_normal_kernel(uint64_t seed, uint64_t step, uint32_t stream_id, int64_t n_rows, int n_cols,
                                      float* __restrict__ out) {
    const int nb = (n_cols + 3) >> 2;
    const int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= n_rows * nb) return;
    const int64_t i = e / nb; const int b = (int)(e - i * nb);
    const Philox4 p = philox4x32_10((uint32_t)step, (uint32_t)(step >> 32), (uint32_t)i, (stream_id << 24) + (uint32_t)b,
                                    (uint32_t)seed, (uint32_t)(seed >> 32));
    float v[4];
#pragma unroll
    for (int a = 0; a < 4; a += 2) {
        const double r = sqrt(-2.0 * log(rng_uniform(p.w[a]))), phi = 6.283185307179586477 * rng_uniform(p.w[a + 1]);
        double s, c; sincos(phi, &s, &c);
        v[a] = (float)(r * c); v[a + 1] = (float)(r * s);
    }
    float* o = out + i * n_cols + 4 * b;
#pragma unroll
    for (int a = 0; a < 4; ++a) if (4 * b + a < n_cols) o[a] = v[a];
}

// out [n_rows] fp32 = ln u, u uniform on (0, 1).
__global__ void gl_draw_log_uniform_kernel(uint64_t seed, uint64_t step, uint32_t stream_id, int64_t n_rows, float* __restrict__ out) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n_rows) return;
    const Philox4 p = philox4x32_10((uint32_t)step, (uint32_t)(step >> 32), (uint32_t)i, stream_id << 24, (uint32_t)seed, (uint32_t)(seed >> 32));
    out[i] = (float)log(rng_uniform(p.w[0]));
}

}  // namespace gl
