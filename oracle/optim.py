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
