// gl_hmc.cuh -- SURVEY 8(f) NEXT-3: one HMC transition of many chains around the hot path.
// Leapfrog in the whitened momentum xi = L^T p (mass matrix M = Sigma^-1, Sigma = L L^T, L packed lower triangular or
// NULL = identity):  H = -log p~(z) + |xi|^2 / 2;  xi += (eps/2) L^T g;  z += eps L xi;  xi += (eps/2) L^T g.
// The trajectory (z, xi) is carried in fp64 in the workspace; the hot path is evaluated at the fp32-rounded position
// (its ABI).  Readings: DESIGN.md section 13.  One CTA per chain, n_params <= 128 threads do the two matvecs.
#pragma once
#include "gl_common.cuh"

namespace gl {

// xi += c * L^T g, then (if drift) z += eps * L xi and zf = fl32(z).  init: take z, xi from the fp32 inputs first.
// grid = n chains, block = 128.  g: [n][np] fp32 gradient of log p~ at the current z.
__global__ void __launch_bounds__(128) gl_hmc_kick_drift_kernel(int np, const float* __restrict__ Lp,
                                                                const float* __restrict__ g, double c, double eps,
                                                                int drift, int init, const float* __restrict__ z_in,
                                                                const float* __restrict__ xi_in, double* __restrict__ zd,
                                                                double* __restrict__ xid, float* __restrict__ zf) {
    __shared__ double sg[128], sx[128];
    const int64_t i = blockIdx.x;
    const int k = threadIdx.x;
    if (k < np) sg[k] = (double)g[i * np + k];
    __syncthreads();
    double x = 0.0, zz = 0.0;
    if (k < np) {
        x = init ? (double)xi_in[i * np + k] : xid[i * np + k];
        zz = init ? (double)z_in[i * np + k] : zd[i * np + k];
        double s = 0.0;                                            // (L^T g)_k = sum_{j >= k} L_jk g_j
        if (Lp) { for (int j = k; j < np; ++j) s = fma((double)Lp[(size_t)j * (j + 1) / 2 + k], sg[j], s); }
        else s = sg[k];
        x = fma(c, s, x);
        sx[k] = x;
        xid[i * np + k] = x;
    }
    __syncthreads();
    if (k < np) {
        if (drift) {
            double s = 0.0;                                        // (L xi)_k = sum_{j <= k} L_kj xi_j
            if (Lp) { const float* row = Lp + (size_t)k * (k + 1) / 2; for (int j = 0; j <= k; ++j) s = fma((double)row[j], sx[j], s); }
            else s = sx[k];
            zz = fma(eps, s, zz);
        }
        zd[i * np + k] = zz;
        zf[i * np + k] = (float)zz;
    }
}

// Accept / reject.  grid = n chains, block = 128.  State (z, logp, grad) is overwritten where the proposal is accepted.
__global__ void __launch_bounds__(128) gl_hmc_accept_kernel(int np, const float* __restrict__ xi0, const double* __restrict__ xid,
                                                            const double* __restrict__ zd, const float* __restrict__ lp1,
                                                            const float* __restrict__ g1, const float* __restrict__ log_u,
                                                            float* __restrict__ z, float* __restrict__ logp,
                                                            float* __restrict__ grad, int32_t* __restrict__ out_accept,
                                                            float* __restrict__ out_dh) {
    __shared__ double s0[128], s1[128];
    __shared__ int s_acc;
    const int64_t i = blockIdx.x;
    const int k = threadIdx.x;
    s0[k] = k < np ? (double)xi0[i * np + k] * (double)xi0[i * np + k] : 0.0;
    s1[k] = k < np ? xid[i * np + k] * xid[i * np + k] : 0.0;
    __syncthreads();
    if (k == 0) {
        double k0 = 0.0, k1 = 0.0;
        for (int j = 0; j < np; ++j) { k0 += s0[j]; k1 += s1[j]; }      // fixed order
        const double l0 = (double)logp[i], l1 = (double)lp1[i];
        const bool fin = isfinite(l1);
        const double dh = fin ? (-l0 + 0.5 * k0) - (-l1 + 0.5 * k1) : -INFINITY;
        const int acc = fin && (double)log_u[i] < dh;
        s_acc = acc;
        out_accept[i] = acc; out_dh[i] = (float)dh;
        if (acc) logp[i] = lp1[i];
    }
    __syncthreads();
    if (s_acc && k < np) { z[i * np + k] = (float)zd[i * np + k]; grad[i * np + k] = g1[i * np + k]; }
}

}  // namespace gl
