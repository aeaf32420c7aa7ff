"""Oracle of "backward" amplitude modelling ("we either model the light intensities as parameters
('forward' modeling) or solve for them by linear inversion ('backward' modeling)").

TEST INFRASTRUCTURE ONLY (see oracle/__init__.py).  Plain numpy on top of the C oracle's model images.

Reading S21 (the paper gives no formula).  The model image is linear in the light
amplitudes a = (I of the source Sersic, the shapelet coefficients, I of each lens Sersic), in the flat order S18:
    model = sum_k a_k A_k,     A_k = image of component k with unit amplitude, PSF-convolved and binned (O3-O6).
With the fixed noise map sigma (S12) the Gaussian likelihood is quadratic in a, and linear inversion is the weighted
least-squares solution
    a* = argmin_a sum_pix (obs - sum_k a_k A_k)^2 / sigma^2 = M^-1 b,   M_kl = sum A_k A_l / sigma^2,  b_k = sum A_k obs / sigma^2.
The log-posterior of the remaining ("non-linear") parameters is the joint density at a*:
    log p~_B(z) = log L(theta(z), a*) + sum over NON-amplitude parameters of (log prior + log-det)
(no prior on the amplitudes, no marginalisation term), and since dL/da = 0 at a*, its gradient with respect to the
non-linear parameters is the partial derivative at fixed a = a* (envelope theorem); the amplitude entries of z are
ignored on input and their gradient entries are zero.
"""
import copy
import numpy as np

import oracle

PRIOR_NONE_T = (oracle.PRIOR_NONE, 0.0, 1.0, 0.0, 0.0)


def amplitude_indices(spec):
    """Indices of the amplitude parameters in the flat order S18: mass block, shear, multipoles, source Sersic
    [R n e1 e2 x y I], shapelets [beta a_0..], lens Sersic blocks."""
    i = (6 if spec.mass_model == 1 else 5) + (2 if spec.has_shear else 0)
    i += 2 * bin(spec.multipole_mask & 3).count("1")
    idx = []
    for k in range(spec.n_source_sersic):
        idx.append(i + 6); i += 7
        if k == 1 and getattr(spec, "source2_plane", 0): i += 1       # eta2 follows the second source block (S23)
    if spec.shapelet_nmax >= 0:
        nc = (spec.shapelet_nmax + 1) * (spec.shapelet_nmax + 2) // 2
        idx += list(range(i + 1, i + 1 + nc)); i += 1 + nc
    for _ in range(spec.n_lens_sersic):
        idx.append(i + 6); i += 7
    assert i == spec.n_params
    return np.array(idx, dtype=np.int64)


def backward_spec(spec):
    """The same model with the amplitude parameters prior-free and untransformed (their z IS the amplitude)."""
    s = copy.copy(spec)
    s.priors = list(spec.priors)
    for k in amplitude_indices(spec):
        s.priors[k] = PRIOR_NONE_T
    return s


def _theta(spec, z):
    return np.array([oracle.transform_one(spec.priors[i], spec.param_space, z[i])["theta"] for i in range(spec.n_params)])


def component_images(spec, psf, theta, system=0, epl_terms=None):
    """A_k [n_amp][N][N]: the model image with amplitude k = 1 and every other amplitude 0."""
    amp = amplitude_indices(spec)
    rows = np.repeat(np.asarray(theta, dtype=np.float64)[None, :], len(amp), axis=0)
    rows[:, amp] = np.eye(len(amp))
    sid = np.full(len(amp), system, dtype=np.int32)
    return oracle.model_image(spec, psf, rows, epl_terms=epl_terms, system_id=sid)


def solve_amplitudes(spec, obs, sigma, psf, z, system=0, epl_terms=None):
    """a* = M^-1 b for one particle (normal equations, Cholesky in fp64).  Returns (a*, M, b); a* is None when M is
    not positive definite (a component that contributes nothing to the image)."""
    sb = backward_spec(spec)
    N = spec.n_pix
    th = _theta(sb, np.asarray(z, dtype=np.float64))
    A = component_images(sb, psf, th, system, epl_terms).reshape(-1, N * N)
    w = 1.0 / np.asarray(sigma, dtype=np.float64).reshape(-1, N * N)[system] ** 2
    d = np.asarray(obs, dtype=np.float64).reshape(-1, N * N)[system]
    M = (A * w) @ A.T
    b = (A * w) @ d
    try:
        Lc = np.linalg.cholesky(M)
    except np.linalg.LinAlgError:
        return None, M, b
    a = np.linalg.solve(Lc.T, np.linalg.solve(Lc, b))
    return a, M, b


def logpost_grad(spec, obs, sigma, psf, params, system_id=None, epl_terms=None, want_grad=True):
    """log p~_B and its gradient for each row of params (amplitude entries ignored, their gradient 0).
    Returns dict(logp [P], grad [P][n_params], amp [P][n_amp])."""
    assert int(getattr(spec, "noise_model", 0)) == 0, "linear inversion needs the fixed noise map (S21)"
    sb = backward_spec(spec)
    amp = amplitude_indices(spec)
    params = np.array(params, dtype=np.float64).reshape(-1, spec.n_params)
    P = params.shape[0]
    sid = np.zeros(P, dtype=np.int32) if system_id is None else np.asarray(system_id, dtype=np.int32)
    zs = params.copy(); zs[:, amp] = 1.0
    a_out = np.zeros((P, len(amp)))
    solved = np.zeros(P, dtype=bool)
    for p in range(P):
        th_ok = all(oracle.transform_one(sb.priors[i], sb.param_space, zs[p, i])["ok"] for i in range(spec.n_params))
        if not th_ok or not np.isfinite(oracle.logpost_grad(sb, obs, sigma, psf, zs[p], sid[p:p + 1], want_grad=False,
                                                           epl_terms=epl_terms)["logp"][0]):
            continue                                              # invalid non-linear parameters: logp = -inf below
        a, _, _ = solve_amplitudes(spec, obs, sigma, psf, zs[p], int(sid[p]), epl_terms)
        if a is None:
            continue
        a_out[p] = a; zs[p, amp] = a; solved[p] = True
    out = oracle.logpost_grad(sb, obs, sigma, psf, zs, sid, want_grad=want_grad, epl_terms=epl_terms)
    logp = np.where(solved, out["logp"], -np.inf)
    grad = None
    if want_grad:
        grad = out["grad"].copy(); grad[:, amp] = 0.0; grad[~solved] = 0.0
    return dict(logp=logp, grad=grad, amp=a_out, grad_at_amp=None if not want_grad else out["grad"][:, amp])
