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
