"""Shared builders for the parity tests: a seeded workload (workloads/), its observation rendered by the ORACLE
from the seeded truth, and the oracle's log-posterior / gradient on a subset of the particles.

Everything expected comes from oracle/ (fp64 CPU); nothing here touches the CUDA path.
"""
import functools

import numpy as np

import oracle
import workloads as W

# BASELINE.json north_star tolerances (SURVEY 8(c) "Tolerances")
RTOL_LOGP = 1e-4
RTOL_GRAD = 1e-3
ATOL_GRAD = 1e-5


@functools.lru_cache(maxsize=None)
def observation(k):
    """(workload at full size, obs, sigma) for BASELINE.json configs[k-1]; obs rendered by the oracle."""
    wl = W.make_workload(k)
    sp = wl.spec
    sid = np.arange(sp.n_systems, dtype=np.int32) if sp.n_systems > 1 else None
    truth = oracle.model_image(sp, wl.psf.astype(np.float64), wl.truth_theta, system_id=sid)
    obs, sig = W.finish_observation(wl, truth)
    return wl, obs, sig


def parity_subset(k, n=None):
    """Indices of the parity subset of config k inside the FULL batch (cfg 1 all 64; 2: 256;
    3: 128; 4: 4 per system; 5: 16).  Seeded, sorted."""
    n = W.PARITY_PARTICLES[k] if n is None else n
    full = W.FULL_PARTICLES[k]
    if k == 4:
        per = max(n // 100, 1)
        rng = np.random.default_rng(4004)
        idx = np.concatenate([s * 1024 + np.sort(rng.choice(1024, per, replace=False)) for s in range(100)])
        return idx.astype(np.int64)
    if n >= full:
        return np.arange(full, dtype=np.int64)
    rng = np.random.default_rng(9000 + k)
    return np.sort(rng.choice(full, n, replace=False)).astype(np.int64)


@functools.lru_cache(maxsize=None)
def oracle_subset(k, n=None):
    """Oracle logp / grad / gabs on the parity subset of config k.  Returns (idx, dict)."""
    wl, obs, sig = observation(k)
    idx = parity_subset(k, n)
    sid = wl.system_id[idx] if wl.system_id is not None else None
    out = oracle.logpost_grad(wl.spec, obs, sig, wl.psf, wl.params[idx].astype(np.float64), sid, want_gabs=True)
    return idx, out


def grad_report(g_gpu, g_ref, gabs=None):
    """Per-component pass mask under the north_star bar plus the summary numbers DESIGN.md section 7 reports."""
    g_gpu = np.asarray(g_gpu, dtype=np.float64); g_ref = np.asarray(g_ref, dtype=np.float64)
    err = np.abs(g_gpu - g_ref)
    ok = err <= np.maximum(RTOL_GRAD * np.abs(g_ref), ATOL_GRAD)
    rel = err / np.maximum(np.abs(g_ref), 1e-300)
    rep = dict(n=int(ok.size), n_fail=int((~ok).sum()), pass_frac=float(ok.mean()),
               worst_rel=float(rel[~ok].max()) if (~ok).any() else float(rel.max()),
               normwise=float(np.max(np.linalg.norm(g_gpu - g_ref, axis=1) / np.maximum(np.linalg.norm(g_ref, axis=1), 1e-300))))
    if gabs is not None:
        rep["cond_aware"] = float(np.max(err / np.maximum(np.asarray(gabs), 1e-300)))
    return ok, rep


def small_case(n_pix, s, K, mass_model, multipole_mask, shapelet_nmax, n_lens, seed, n_particles=6, epl_terms=30,
               psf_grid=0, with_truth=False):
    """A seeded small problem of arbitrary shape: spec with config-style priors, Gaussian PSF, oracle-rendered truth.
    Returns (spec, obs, sigma, psf, z [n_particles][n_params] prior draws) and, with_truth, the fp32 truth z [n_params]."""
    pri = W._default_priors(mass_model, multipoles=bool(multipole_mask), shapelet_nmax=shapelet_nmax, n_lens=n_lens)
    if multipole_mask and multipole_mask != 3:
        # _default_priors adds 4 multipole entries; keep 2 for a single order
        k0 = 1 + (1 if mass_model == 1 else 0) + 4 + 2
        pri = pri[:k0] + pri[k0 + 2:]
    sp = W.LensSpec(n_pix, s, K, W._r32(0.11 * 40 / n_pix * 2.4), mass_model=mass_model, epl_terms=epl_terms,
                    multipole_mask=multipole_mask, shapelet_nmax=shapelet_nmax, n_lens_sersic=n_lens, psf_grid=psf_grid,
                    priors=pri)
    sp.names = W.param_names(mass_model, 1, multipole_mask, 1, shapelet_nmax, n_lens)
    assert len(sp.names) == sp.n_params
    rng = np.random.default_rng(seed)
    step = sp.pix_scale / s if psf_grid == 0 else sp.pix_scale      # taps at ray spacing (S10) or pixel spacing (S10b)
    psf = W.gaussian_psf(K, 2.5 * step, step)[None].astype(np.float32)
    truth_z = W.z_of(pri, W.draw(rng, pri, 1)).astype(np.float32)
    truth = oracle.model_image(sp, psf.astype(np.float64), W.theta_of(pri, truth_z.astype(np.float64)))
    sigma = np.full((1, n_pix, n_pix), 0.05, np.float32)
    obs = (truth + 0.05 * rng.standard_normal(truth.shape)).astype(np.float32)
    z = W.z_of(pri, W.draw(rng, pri, n_particles)).astype(np.float32)
    if with_truth:
        return sp, obs, sigma, psf, z, truth_z[0]
    return sp, obs, sigma, psf, z
