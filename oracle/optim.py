"""fp64 ORACLE of the multi-start MAP optimiser step.  TEST INFRASTRUCTURE ONLY (see
oracle/gl_oracle.c): imported by tests/ only; shares nothing with the CUDA path.

What the paper fixes (PAPER.md = /root/reference/PAPER.md):
  * every MAP particle performs gradient descent independently (L72; fn 2, L83: descending the mean of all particles'
    losses is the same thing) on the loss  -log p~(I_obs, Theta~)  in the unconstrained space (L76, L89);
  * the optimiser is Adam by default for MAP, AdaBelief (Zhuang et al. 2020) gives the same result (L104-114);
    AdaBelief's hyperparameters are lr = 1e-4, b1 = 0.95, b2 = 0.99, no learning-rate schedule (L112).
What it leaves open, and the reading taken: the update formulas are the published ones, in the
form the paper's software (Optax, L225) documents them:
  Adam       m <- b1 m + (1-b1) g;  v <- b2 v + (1-b2) g^2;
             z <- z - lr * (m / (1 - b1^t)) / (sqrt(v / (1 - b2^t)) + eps)                    (eps 1e-8)
  AdaBelief  m <- b1 m + (1-b1) g;  s <- b2 s + (1-b2) (g - m)^2 + eps_root   (m already updated);
             z <- z - lr * (m / (1 - b1^t)) / (sqrt(s / (1 - b2^t)) + eps)                    (eps = eps_root = 1e-16)
with g = -grad log p~, t = 1, 2, ... the step index.  A particle whose log-posterior is not finite is left unchanged
(parameters and state).  Parameters and state are stored as fp32 by the interface; this oracle takes whatever it is
given, computes in fp64 and returns fp64.
"""
import numpy as np

ADAM, ADABELIEF = 0, 1


def update(kind, z, grad_logp, logp, m, v, t, lr, b1, b2, eps, eps_root=0.0):
    """One optimiser update for every row.  z, grad_logp, m, v: [P][n]; logp: [P]; t: 1-based step index.
    Returns (z_new, m_new, v_new) in fp64."""
    z = np.asarray(z, np.float64); m = np.asarray(m, np.float64); v = np.asarray(v, np.float64)
    g = -np.asarray(grad_logp, np.float64)
    ok = np.isfinite(np.asarray(logp, np.float64))[:, None] & np.all(np.isfinite(g), axis=1, keepdims=True)
    g = np.where(ok, g, 0.0)
    m1 = b1 * m + (1.0 - b1) * g
    if kind == ADAM:
        v1 = b2 * v + (1.0 - b2) * g * g
    elif kind == ADABELIEF:
        v1 = b2 * v + (1.0 - b2) * (g - m1) ** 2 + eps_root
    else:
        raise ValueError(kind)
    mhat = m1 / (1.0 - b1 ** t)
    vhat = v1 / (1.0 - b2 ** t)
    z1 = z - lr * mhat / (np.sqrt(vhat) + eps)
    return np.where(ok, z1, z), np.where(ok, m1, m), np.where(ok, v1, v)


def map_step(oracle_mod, spec, obs, sigma, psf, z, m, v, t, opt, system_id=None):
    """log p~ and its gradient at z (oracle.logpost_grad), then `update`.  opt = dict(kind, lr, b1, b2, eps, eps_root).
    Returns (logp, z_new, m_new, v_new)."""
    r = oracle_mod.logpost_grad(spec, obs, sigma, psf, np.asarray(z, np.float64), system_id)
    z1, m1, v1 = update(opt["kind"], z, r["grad"], r["logp"], m, v, t, opt["lr"], opt["b1"], opt["b2"], opt["eps"],
                        opt.get("eps_root", 0.0))
    return r["logp"], z1, m1, v1


# ------------------------------------------------------------------------------------------------ NEXT-2: SVI step
# a multivariate-normal surrogate q~(Theta~; mu~, Sigma~) is fitted by minimising the loss
#   ELBO = E_q[ log q~(Theta~) - log p~(I_obs, Theta~) ]                                   (Eq. 2; a LOSS, as printed)
# estimated at each iteration from n_VI draws (L91); the gradient with respect to (mu~, Sigma~) is obtained "with JAX's
# automatic differentiation" from the draws (L98) and an optimiser step is applied to (mu~, Sigma~) (L100); AdaBelief
# with lr 1e-4, b1 0.95, b2 0.99 is the default (L112).
# Readings: Sigma~ = L L^T with L lower triangular, positive diagonal, optimised entry by entry
# (packed row-major: L00, L10, L11, L20, ...); draws are reparameterised, z_i = mu + L xi_i with xi_i ~ N(0, I) supplied
# by the caller; differentiating the sampled loss through the draws gives the pathwise estimator
#   loss^   = -sum_j log L_jj - (n/2) log(2 pi e) + (1/N) sum_i [ -log p~(z_i) ]
#             (E_q[log q] = -entropy is taken in closed form; with xi fixed the sampled -1/2 |xi|^2 term has no gradient)
#   d/dmu_j   = -(1/N) sum_i g_ij                      g_i = grad log p~(z_i)
#   d/dL_jk   = -(1/N) sum_i g_ij xi_ik - delta_jk / L_jj          (k <= j)
# Eq. 3 as printed (L95) is the score-function form of the same gradient; both are unbiased, the text's autodiff of
# reparameterised draws yields the pathwise one, which is also the one that uses the hot path's gradient.
# Draws whose log p~ is not finite are left out of the averages (N = number of finite draws).

def tril_unpack(n, packed):
    L = np.zeros((n, n))
    L[np.tril_indices(n)] = np.asarray(packed, np.float64)
    return L


def tril_pack(L):
    return np.asarray(L, np.float64)[np.tril_indices(L.shape[0])]


def svi_draw(mu, L_packed, xi):
    mu = np.asarray(mu, np.float64); xi = np.asarray(xi, np.float64)
    return mu[None, :] + xi @ tril_unpack(mu.size, L_packed).T


def svi_loss_and_grad(mu, L_packed, xi, logp, grad_logp, active=None):
    """Sampled ELBO loss and its gradient w.r.t. (mu, packed L) from per-draw logp [N] and grad log p [N][n].
    active [n] bool (default all): the dimensions the surrogate lives on.  Backward modelling (
    DESIGN.md section 16) solves the light amplitudes inside every evaluation, so log p~ does not depend on their
    entries of z: the surrogate is the multivariate normal of the SAMPLED dimensions only -- entropy and gradient over
    the active block, zero gradient for mu_j and for every L entry in a row or column of an inactive dimension."""
    n = np.asarray(mu).size
    act = np.ones(n, bool) if active is None else np.asarray(active, bool)
    L = tril_unpack(n, L_packed)
    xi = np.asarray(xi, np.float64); g = np.asarray(grad_logp, np.float64); lp = np.asarray(logp, np.float64)
    ok = np.isfinite(lp) & np.all(np.isfinite(g), axis=1)
    N = int(ok.sum())
    d = np.diag(L)
    loss = -np.sum(np.log(np.abs(d[act]))) - 0.5 * int(act.sum()) * np.log(2.0 * np.pi * np.e) - lp[ok].sum() / N
    g_mu = -g[ok].sum(axis=0) / N
    g_L = -(g[ok].T @ xi[ok]) / N - np.diag(1.0 / d)
    g_mu = np.where(act, g_mu, 0.0)
    g_L = np.where(act[:, None] & act[None, :], g_L, 0.0)
    return loss, g_mu, tril_pack(g_L), N


# Score-function estimator: Eq. 3 AS PRINTED,
#   grad_phi ELBO = E_q[ (log q~(z) - log p~(z)) grad_phi log q~(z; phi) ],            phi = (mu~, L),  z held fixed,
# which needs log p~ only (no gradient of the model).  For the normal surrogate, with xi = L^-1 (z - mu) and s = L^-T xi:
#   log q~(z)       = -1/2 |xi|^2 - sum_j log L_jj - (n/2) log 2 pi
#   d log q~/d mu_j = s_j                      d log q~/d L_jk = s_j xi_k - delta_jk / L_jj         (k <= j)
# Sampled with N draws:  g^_phi = (1/N) sum_i c_i grad_phi log q~(z_i),  c_i = w_i - b_i,  w_i = log q~(z_i) - log p~(z_i).
# Reading: b_i = 0 is the estimator as printed; `baseline=True` takes the leave-one-out mean
# b_i = mean_{k != i} w_k, i.e. c_i = N/(N-1) (w_i - mean w) -- still unbiased (b_i is independent of draw i and
# E grad log q~ = 0) and the standard way to make the estimator usable (the paper prints no variance reduction).
# The loss reported is the same closed-entropy estimate as above.  Draws with a non-finite log p~ are left out.

def svi_score_terms(mu, L_packed, xi):
    """(log q~(z_i) [N], s_i = L^-T xi_i [N][n]) for the draws z_i = mu + L xi_i."""
    n = np.asarray(mu).size
    L = tril_unpack(n, L_packed)
    xi = np.asarray(xi, np.float64)
    logq = -0.5 * np.sum(xi * xi, axis=1) - np.sum(np.log(np.abs(np.diag(L)))) - 0.5 * n * np.log(2.0 * np.pi)
    s = np.linalg.solve(L.T, xi.T).T
    return logq, s


def svi_loss_and_grad_score(mu, L_packed, xi, logp, baseline=True):
    """Sampled ELBO loss (closed-form entropy) and the score-function estimate of its gradient w.r.t. (mu, packed L)
    from per-draw log p~ [N] alone.  Returns (loss, g_mu, g_L_packed, N_finite)."""
    n = np.asarray(mu).size
    L = tril_unpack(n, L_packed)
    xi = np.asarray(xi, np.float64); lp = np.asarray(logp, np.float64)
    ok = np.isfinite(lp)
    N = int(ok.sum())
    logq, s = svi_score_terms(mu, L_packed, xi)
    w = logq[ok] - lp[ok]
    c = (w - w.mean()) * (N / (N - 1.0)) if baseline else w
    d = np.diag(L)
    loss = -np.sum(np.log(np.abs(d))) - 0.5 * n * np.log(2.0 * np.pi * np.e) - lp[ok].sum() / N
    g_mu = (c[:, None] * s[ok]).sum(axis=0) / N
    g_L = (s[ok] * c[:, None]).T @ xi[ok] / N - np.diag(c.sum() / N / d)
    return loss, g_mu, tril_pack(np.tril(g_L)), N


def svi_step_score(logp_fn, mu, L_packed, xi, m, v, t, opt, baseline=True):
    """One SVI iteration with the score-function gradient.  logp_fn(z [N][n]) -> logp [N].
    Returns (loss, mu_new, L_new, m_new, v_new, logp)."""
    n = np.asarray(mu).size
    z = svi_draw(mu, L_packed, xi)
    lp = logp_fn(z)
    loss, g_mu, g_L, N = svi_loss_and_grad_score(mu, L_packed, xi, lp, baseline)
    theta = np.concatenate([np.asarray(mu, np.float64), np.asarray(L_packed, np.float64)])[None, :]
    grad_loss = np.concatenate([g_mu, g_L])[None, :]
    m0 = np.asarray(m, np.float64)[None, :]; v0 = np.asarray(v, np.float64)[None, :]
    th1, m1, v1 = update(opt["kind"], theta, -grad_loss, np.zeros(1), m0, v0, t, opt["lr"], opt["b1"], opt["b2"],
                         opt["eps"], opt.get("eps_root", 0.0))
    return loss, th1[0, :n], th1[0, n:], m1[0], v1[0], lp


def svi_step(logp_grad_fn, mu, L_packed, xi, m, v, t, opt, active=None):
    """One SVI iteration.  logp_grad_fn(z [N][n]) -> (logp [N], grad [N][n]).  State m, v over the concatenated
    parameter vector [mu; packed L].  Entries of inactive dimensions (see svi_loss_and_grad) keep their value and
    their optimiser state.  Returns (loss, mu_new, L_new, m_new, v_new, logp)."""
    n = np.asarray(mu).size
    act = np.ones(n, bool) if active is None else np.asarray(active, bool)
    z = svi_draw(mu, L_packed, xi)
    lp, g = logp_grad_fn(z)
    loss, g_mu, g_L, N = svi_loss_and_grad(mu, L_packed, xi, lp, g, act)
    theta = np.concatenate([np.asarray(mu, np.float64), np.asarray(L_packed, np.float64)])[None, :]
    grad_loss = np.concatenate([g_mu, g_L])[None, :]
    m0 = np.asarray(m, np.float64)[None, :]; v0 = np.asarray(v, np.float64)[None, :]
    th1, m1, v1 = update(opt["kind"], theta, -grad_loss, np.zeros(1), m0, v0, t, opt["lr"], opt["b1"], opt["b2"],
                         opt["eps"], opt.get("eps_root", 0.0))
    live = np.concatenate([act, tril_pack(act[:, None] & act[None, :]).astype(bool)])[None, :]
    th1 = np.where(live, th1, theta); m1 = np.where(live, m1, m0); v1 = np.where(live, v1, v0)
    return loss, th1[0, :n], th1[0, n:], m1[0], v1[0], lp


# ------------------------------------------------------------------------------------------------ NEXT-3: HMC transition
# every chain runs Hamiltonian Monte Carlo independently on log p~ in the unconstrained
# space; the surrogate covariance from SVI (or from the mass-matrix adaptation, L128) sets the scale of each dimension.
# The paper uses TFP's HMC and prints neither the integrator nor the step size or trajectory length.
# Readings: the standard leapfrog HMC transition (Neal 2011) with mass matrix M = Sigma^-1,
# Sigma = L L^T (L lower triangular, packed as for SVI), written in the whitened momentum xi = L^T p ~ N(0, I):
#   H(z, xi) = -log p~(z) + 1/2 |xi|^2
#   one leapfrog step:  xi <- xi + (eps/2) L^T g(z);  z <- z + eps L xi;  xi <- xi + (eps/2) L^T g(z)       g = grad log p~
#   accept the end point of n_leapfrog steps iff  log u < H(z0, xi0) - H(z1, xi1),  u ~ U(0, 1)
# xi0 and log u are INPUTS (both sides must see the same random numbers).  A proposal whose log p~ is not finite is
# rejected; the cached log p~ and gradient of the current state travel with it.

def _tril_matvecs(n, L_packed):
    L = tril_unpack(n, L_packed)
    return L, (lambda x: x @ L.T), (lambda g: g @ L)            # rows: L xi  and  L^T g


def hmc_leapfrog(logp_grad_fn, z, grad, L_packed, xi, eps, n_leapfrog):
    """n_leapfrog leapfrog steps from (z, xi) with grad = g(z).  Returns (z1, xi1, logp1, grad1)."""
    z = np.array(z, np.float64); xi = np.array(xi, np.float64); g = np.array(grad, np.float64)
    _, Lx, LTg = _tril_matvecs(z.shape[1], L_packed)
    lp = None
    for _ in range(n_leapfrog):
        xi = xi + 0.5 * eps * LTg(g)
        z = z + eps * Lx(xi)
        lp, g = logp_grad_fn(z)
        g = np.where(np.isfinite(lp)[:, None], g, 0.0)
        xi = xi + 0.5 * eps * LTg(g)
    return z, xi, lp, g


def hmc_transition(logp_grad_fn, z, logp, grad, L_packed, xi, log_u, eps, n_leapfrog):
    """One HMC transition for every chain (row).  Returns (z_new, logp_new, grad_new, accepted [bool], dH)."""
    z0 = np.asarray(z, np.float64); lp0 = np.asarray(logp, np.float64); g0 = np.asarray(grad, np.float64)
    xi0 = np.asarray(xi, np.float64)
    z1, xi1, lp1, g1 = hmc_leapfrog(logp_grad_fn, z0, g0, L_packed, xi0, eps, n_leapfrog)
    h0 = -lp0 + 0.5 * np.sum(xi0 * xi0, axis=1)
    h1 = np.where(np.isfinite(lp1), -lp1 + 0.5 * np.sum(xi1 * xi1, axis=1), np.inf)
    dH = h0 - h1
    acc = np.isfinite(lp1) & (np.asarray(log_u, np.float64) < dH)
    a = acc[:, None]
    return np.where(a, z1, z0), np.where(acc, lp1, lp0), np.where(a, g1, g0), acc, dH
