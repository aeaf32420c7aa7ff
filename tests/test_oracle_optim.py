"""Pins of the optimiser oracle (oracle/optim.py) against what the published update rules fix in closed form."""
import numpy as np
import pytest

from oracle import optim


def _g(seed=0, shape=(5, 7)):
    return np.random.default_rng(seed).standard_normal(shape) * 3.0


def test_adam_first_step_is_lr_times_sign():
    """t = 1: m^ = g, v^ = g^2, so the step is lr * g / (|g| + eps): the textbook scale-invariance of Adam."""
    g = _g()                                         # gradient of the LOSS; the oracle takes grad log p = -g
    z = np.zeros_like(g)
    z1, m1, v1 = optim.update(optim.ADAM, z, -g, np.zeros(5), z, z, 1, 1e-3, 0.9, 0.999, 1e-8)
    assert np.allclose(z1, -1e-3 * g / (np.abs(g) + 1e-8), rtol=1e-13)
    assert np.allclose(m1, 0.1 * g) and np.allclose(v1, 0.001 * g * g)


def test_adam_constant_gradient_keeps_unit_steps():
    """A constant gradient: m^ = g and v^ = g^2 at every t, so every step is lr * sign(g) and z(t) = -t lr sign(g)."""
    g = _g(1)
    z = np.zeros_like(g); m = np.zeros_like(g); v = np.zeros_like(g)
    for t in range(1, 40):
        z, m, v = optim.update(optim.ADAM, z, -g, np.zeros(5), m, v, t, 1e-2, 0.9, 0.999, 0.0)
    assert np.allclose(z, -39 * 1e-2 * np.sign(g), rtol=1e-12)


def test_adabelief_first_step_closed_form():
    """t = 1 with eps = eps_root = 0: m = (1-b1) g, s = (1-b2) b1^2 g^2, so the step is lr * sign(g) / b1."""
    g = _g(2); z = np.zeros_like(g)
    z1, m1, s1 = optim.update(optim.ADABELIEF, z, -g, np.zeros(5), z, z, 1, 1e-4, 0.95, 0.99, 0.0, 0.0)
    assert np.allclose(z1, -1e-4 * np.sign(g) / 0.95, rtol=1e-12)
    assert np.allclose(s1, 0.01 * (0.95 * g) ** 2, rtol=1e-13)


def test_adabelief_belief_term_vanishes_for_constant_gradient():
    """Constant gradient: g - m -> 0 geometrically, so s decays like b2^t and the steps GROW (large belief)."""
    g = np.full((1, 1), 2.0); z = np.zeros((1, 1)); m = z.copy(); s = z.copy()
    steps = []
    for t in range(1, 200):
        z0 = z.copy()
        z, m, s = optim.update(optim.ADABELIEF, z, -g, np.zeros(1), m, s, t, 1e-4, 0.95, 0.99, 1e-16, 1e-16)
        steps.append(float((z0 - z)[0, 0]))
    assert abs(g - m).max() < 2.0 * 0.95 ** 199 * 1.0001
    assert steps[-1] > steps[0] > 0


@pytest.mark.parametrize("kind", [optim.ADAM, optim.ADABELIEF])
def test_descends_a_quadratic_bowl(kind):
    """loss = 1/2 sum a_i z_i^2 (log p = -loss): both rules bring every coordinate close to the minimum."""
    a = np.array([[0.5, 2.0, 10.0]])
    z = np.array([[1.0, -2.0, 0.5]]); m = np.zeros_like(z); v = np.zeros_like(z)
    for t in range(1, 3001):
        z, m, v = optim.update(kind, z, -(a * z), np.zeros(1), m, v, t, 5e-3, 0.9, 0.999, 1e-8, 1e-16)
    assert np.all(np.abs(z) < 2e-2)


def test_non_finite_rows_are_left_unchanged():
    g = _g(3); z = _g(4); m = _g(5) * 0.1; v = np.abs(_g(6))
    logp = np.array([0.0, -np.inf, 0.0, np.nan, 0.0])
    g2 = g.copy(); g2[2, 3] = np.nan
    z1, m1, v1 = optim.update(optim.ADAM, z, g2, logp, m, v, 3, 1e-3, 0.9, 0.999, 1e-8)
    for r in (1, 2, 3):
        assert np.array_equal(z1[r], z[r]) and np.array_equal(m1[r], m[r]) and np.array_equal(v1[r], v[r])
    for r in (0, 4):
        assert not np.array_equal(z1[r], z[r])
    assert np.all(np.isfinite(z1))


# ------------------------------------------------------------------------------------------------ SVI (NEXT-2)
def _toy_target(a, A):
    """A smooth non-Gaussian log density with closed-form gradient: -1/2 (z-a)^T A (z-a) - sum log cosh z."""
    def f(z):
        d = z - a
        return -0.5 * np.einsum("ij,jk,ik->i", d, A, d) - np.log(np.cosh(z)).sum(axis=1), -(d @ A.T) - np.tanh(z)
    return f


def _svi_setup(n=4, N=64, seed=3):
    rng = np.random.default_rng(seed)
    B = rng.standard_normal((n, n)); A = B @ B.T + n * np.eye(n)
    a = rng.standard_normal(n)
    L = np.tril(rng.standard_normal((n, n)) * 0.2) + np.diag(0.5 + rng.random(n))
    return rng.standard_normal(n), optim.tril_pack(L), rng.standard_normal((N, n)), _toy_target(a, A), a, A


def test_svi_gradient_is_the_derivative_of_the_sampled_loss():
    """With the draws xi held fixed, the assembled gradient must equal central finite differences of the sampled loss
    in every entry of mu and of the packed L (the pathwise estimator IS the derivative of the sampled objective)."""
    mu, Lp, xi, f, a, A = _svi_setup()

    def loss(mu_, Lp_):
        lp, g = f(optim.svi_draw(mu_, Lp_, xi))
        return optim.svi_loss_and_grad(mu_, Lp_, xi, lp, g)[0]

    lp, g = f(optim.svi_draw(mu, Lp, xi))
    _, g_mu, g_L, N = optim.svi_loss_and_grad(mu, Lp, xi, lp, g)
    assert N == 64
    h = 1e-6
    for j in range(mu.size):
        e = np.zeros_like(mu); e[j] = h
        assert abs((loss(mu + e, Lp) - loss(mu - e, Lp)) / (2 * h) - g_mu[j]) < 1e-6 * max(1, abs(g_mu[j]))
    for j in range(Lp.size):
        e = np.zeros_like(Lp); e[j] = h
        assert abs((loss(mu, Lp + e) - loss(mu, Lp - e)) / (2 * h) - g_L[j]) < 1e-6 * max(1, abs(g_L[j]))


def test_svi_gaussian_target_closed_form():
    """Quadratic log p: grad_mu = A (mu + L xbar - a), grad_L = tril(A (mu - a) xbar^T + A L S) - diag(1/L_jj) with the
    SAMPLE moments xbar, S of the draws; and the entropy term is the closed form of a Gaussian's."""
    mu, Lp, xi, _, a, A = _svi_setup(seed=8)
    L = optim.tril_unpack(mu.size, Lp)
    z = optim.svi_draw(mu, Lp, xi)
    assert np.allclose(z, mu + xi @ L.T)
    d = z - a
    lp = -0.5 * np.einsum("ij,jk,ik->i", d, A, d); g = -(d @ A.T)
    loss, g_mu, g_L, _ = optim.svi_loss_and_grad(mu, Lp, xi, lp, g)
    xbar = xi.mean(axis=0); S = xi.T @ xi / xi.shape[0]
    assert np.allclose(g_mu, A @ (mu + L @ xbar - a), rtol=1e-12)
    full = np.outer(A @ (mu - a), xbar) + A @ L @ S - np.diag(1 / np.diag(L))
    assert np.allclose(g_L, optim.tril_pack(full), rtol=1e-12, atol=1e-12)
    ent = 0.5 * np.linalg.slogdet(2 * np.pi * np.e * (L @ L.T))[1]
    assert np.isclose(loss, -ent - lp.mean(), rtol=1e-13)


def test_svi_fits_a_gaussian_target():
    """Minimising the loss on a Gaussian target recovers its mean and covariance (KL = 0 at the optimum, Eq. 1)."""
    rng = np.random.default_rng(0)
    n = 3
    A = np.array([[2.0, 0.3, 0.0], [0.3, 1.0, -0.2], [0.0, -0.2, 0.5]]); a = np.array([0.5, -1.0, 0.25])

    def f(z):
        d = z - a
        return -0.5 * np.einsum("ij,jk,ik->i", d, A, d), -(d @ A.T)

    mu = np.zeros(n); Lp = optim.tril_pack(np.eye(n)); m = np.zeros(n + 6); v = np.zeros(n + 6)
    opt = dict(kind=optim.ADAM, lr=2e-2, b1=0.9, b2=0.999, eps=1e-8)
    for t in range(1, 1501):
        _, mu, Lp, m, v, _ = optim.svi_step(f, mu, Lp, rng.standard_normal((256, n)), m, v, t, opt)
    L = optim.tril_unpack(n, Lp)
    assert np.allclose(mu, a, atol=0.05)
    assert np.allclose(L @ L.T, np.linalg.inv(A), atol=0.08)


def test_svi_non_finite_draws_are_left_out():
    mu, Lp, xi, f, a, A = _svi_setup(N=16)
    lp, g = f(optim.svi_draw(mu, Lp, xi))
    lp2 = lp.copy(); lp2[3] = -np.inf
    l1, gm1, gl1, N1 = optim.svi_loss_and_grad(mu, Lp, np.delete(xi, 3, 0), np.delete(lp, 3), np.delete(g, 3, 0))
    l2, gm2, gl2, N2 = optim.svi_loss_and_grad(mu, Lp, xi, lp2, g)
    assert N2 == 15 == N1 and np.isclose(l1, l2) and np.allclose(gm1, gm2) and np.allclose(gl1, gl2)


@pytest.mark.parametrize("kind", [optim.ADAM, optim.ADABELIEF])
def test_svi_inactive_dimensions_reduce_to_the_compact_problem(kind):
    """Backward modelling: log p~ ignores the solved-amplitude entries of z, so the surrogate is
    the normal of the sampled dimensions.  Three iterations with `active` on a 6-dimensional problem whose target ignores
    dimensions 1 and 4 equal the same iterations of the UNMASKED (already pinned) routine on the 4-dimensional compact
    problem: loss, mu, L and the optimiser state of the active block; the inactive entries never move; and the loss does
    not drift (the un-masked 6-dimensional run is the failure this guards against: -log L_jj of a dead dimension falls
    without bound)."""
    n, N = 6, 48
    act = np.array([True, False, True, True, False, True])
    ia = np.flatnonzero(act)
    mu4, Lp4, xi4, f4, a, A = _svi_setup(n=4, N=N, seed=5)

    def f6(z):                                                   # the target sees the active coordinates only
        lp, g = f4(z[:, ia])
        g6 = np.zeros_like(z); g6[:, ia] = g
        return lp, g6

    rng = np.random.default_rng(9)
    mu6 = rng.standard_normal(n); mu6[ia] = mu4
    L6 = np.tril(0.1 * rng.standard_normal((n, n))) + np.diag(0.7 + rng.random(n))
    L6[np.ix_(ia, ia)] = optim.tril_unpack(4, Lp4)
    L6[np.ix_(ia, ~act)] = 0.0                                   # active rows do not mix in the dead momenta
    Lp6 = optim.tril_pack(L6)
    opt = dict(kind=kind, lr=5e-3, b1=0.9, b2=0.99, eps=1e-8, eps_root=1e-16)
    m6 = np.zeros(n + 21); v6 = np.zeros(n + 21); m4 = np.zeros(4 + 10); v4 = np.zeros(4 + 10)
    keep = np.concatenate([act, optim.tril_pack(act[:, None] & act[None, :]).astype(bool)])
    mu6_0, Lp6_0 = mu6.copy(), Lp6.copy()
    for t in (1, 2, 3):
        xi6 = rng.standard_normal((N, n)); xi4 = xi6[:, ia]
        l6, mu6, Lp6, m6, v6, _ = optim.svi_step(f6, mu6, Lp6, xi6, m6, v6, t, opt, active=act)
        l4, mu4, Lp4, m4, v4, _ = optim.svi_step(f4, mu4, Lp4, xi4, m4, v4, t, opt)
        assert np.isclose(l6, l4, rtol=1e-13)
        assert np.allclose(mu6[ia], mu4, rtol=1e-13) and np.allclose(Lp6[keep[n:]], Lp4, rtol=1e-13, atol=1e-15)
        assert np.allclose(m6[keep], m4, rtol=1e-12, atol=1e-18) and np.allclose(v6[keep], v4, rtol=1e-12, atol=1e-30)
    dead = ~keep
    assert np.array_equal(np.concatenate([mu6, Lp6])[dead], np.concatenate([mu6_0, Lp6_0])[dead])
    assert np.all(m6[dead] == 0) and np.all(v6[dead] == 0)
    # without the mask the dead diagonal entries grow at every step and take the loss down with them
    muu, Lpu, mu_, vu = mu6_0.copy(), Lp6_0.copy(), np.zeros(n + 21), np.zeros(n + 21)
    d0 = np.diag(optim.tril_unpack(n, Lpu))[~act].copy()
    for t in (1, 2, 3):
        _, muu, Lpu, mu_, vu, _ = optim.svi_step(f6, muu, Lpu, rng.standard_normal((N, n)), mu_, vu, t, opt)
    assert np.all(np.diag(optim.tril_unpack(n, Lpu))[~act] > d0)


# ------------------------------------------------------------------------------------------------ HMC (NEXT-3)
def _gauss(a, A):
    def f(z):
        d = z - a
        return -0.5 * np.einsum("ij,jk,ik->i", d, A, d), -(d @ A.T)
    return f


def test_leapfrog_is_time_reversible():
    """Integrate, flip the momentum, integrate again: back at the start (the property that makes HMC valid)."""
    mu, Lp, xi, f, a, A = _svi_setup(n=5, N=7, seed=12)
    z0 = np.random.default_rng(1).standard_normal((7, 5))
    lp0, g0 = f(z0)
    z1, x1, lp1, g1 = optim.hmc_leapfrog(f, z0, g0, Lp, xi, 0.03, 25)
    z2, x2, _, _ = optim.hmc_leapfrog(f, z1, g1, Lp, -x1, 0.03, 25)
    assert np.allclose(z2, z0, atol=1e-11) and np.allclose(-x2, xi, atol=1e-11)


def test_leapfrog_energy_error_is_second_order():
    """Fixed trajectory length: halving the step size divides the energy error by ~4."""
    mu, Lp, xi, f, a, A = _svi_setup(n=4, N=32, seed=5)
    z0 = a + 0.3 * np.random.default_rng(2).standard_normal((32, 4))
    lp0, g0 = f(z0)
    errs = []
    for eps, n in ((0.04, 10), (0.02, 20), (0.01, 40)):
        z1, x1, lp1, _ = optim.hmc_leapfrog(f, z0, g0, Lp, xi, eps, n)
        errs.append(np.abs((-lp1 + 0.5 * (x1 ** 2).sum(1)) - (-lp0 + 0.5 * (xi ** 2).sum(1))).mean())
    assert 3.0 < errs[0] / errs[1] < 5.0 and 3.0 < errs[1] / errs[2] < 5.0


def test_whitened_dynamics_half_period_maps_to_mirror_point():
    """Gaussian target N(a, Sigma) with L = chol(Sigma): in whitened coordinates the flow is a rotation, so after time pi
    every chain sits at 2a - z0 whatever its momentum: pins the roles of L (position) and L^T (force)."""
    rng = np.random.default_rng(9)
    n = 4
    B = rng.standard_normal((n, n)); Sigma = B @ B.T + np.eye(n); a = rng.standard_normal(n)
    L = np.linalg.cholesky(Sigma)
    f = _gauss(a, np.linalg.inv(Sigma))
    z0 = a + rng.standard_normal((6, n)); xi = rng.standard_normal((6, n))
    lp0, g0 = f(z0)
    nstep = 2000
    z1, x1, _, _ = optim.hmc_leapfrog(f, z0, g0, optim.tril_pack(L), xi, np.pi / nstep, nstep)
    assert np.allclose(z1, 2 * a - z0, atol=1e-5) and np.allclose(x1, -xi, atol=1e-5)


def test_hmc_samples_a_gaussian_target():
    """2000 transitions of 64 chains reproduce mean and covariance of a correlated Gaussian within Monte-Carlo error;
    acceptance is high at this step size and rejected chains keep their state and cache."""
    rng = np.random.default_rng(3)
    a = np.array([1.0, -2.0, 0.5]); A = np.array([[2.0, 0.6, 0.0], [0.6, 1.0, -0.3], [0.0, -0.3, 0.8]])
    f = _gauss(a, A)
    Lp = optim.tril_pack(np.eye(3))
    z = rng.standard_normal((64, 3)); lp, g = f(z)
    acc_n = 0; samples = []
    for t in range(2000):
        z_old, lp_old = z.copy(), lp.copy()
        z, lp, g, acc, dH = optim.hmc_transition(f, z, lp, g, Lp, rng.standard_normal((64, 3)), np.log(rng.random(64)), 0.35, 5)
        assert np.array_equal(z[~acc], z_old[~acc]) and np.array_equal(lp[~acc], lp_old[~acc])
        lp_chk, g_chk = f(z)
        assert np.allclose(lp_chk, lp) and np.allclose(g_chk, g)
        acc_n += acc.sum()
        if t >= 200: samples.append(z.copy())
    s = np.concatenate(samples)
    assert acc_n / (2000 * 64) > 0.8
    assert np.allclose(s.mean(0), a, atol=0.03)
    assert np.allclose(np.cov(s.T), np.linalg.inv(A), atol=0.06)


def test_hmc_rejects_non_finite_proposals():
    def f(z):                                             # support z_0 < 1
        lp = np.where(z[:, 0] < 1.0, -0.5 * (z ** 2).sum(1), -np.inf)
        return lp, np.where(np.isfinite(lp)[:, None], -z, 0.0)
    z = np.array([[0.9, 0.0], [-0.5, 0.2]]); lp, g = f(z)
    xi = np.array([[3.0, 0.0], [0.1, 0.1]])
    z1, lp1, g1, acc, dH = optim.hmc_transition(f, z, lp, g, optim.tril_pack(np.eye(2)), xi, np.log([0.999, 1e-9]), 0.2, 3)
    assert not acc[0] and np.array_equal(z1[0], z[0]) and acc[1]


# ------------------------------------------------------------------------------------------------ score-function SVI (Eq. 3)
def test_svi_score_terms_are_log_q_and_its_derivatives():
    """log q~ against scipy's multivariate-normal log-density with covariance L L^T, and d log q~/d(mu, L) at FIXED z against
    central differences of that independent routine (this fixes which of L^-1, L^-T acts where, and the diagonal term)."""
    from scipy.stats import multivariate_normal
    mu, Lp, xi, _, _, _ = _svi_setup(n=4, N=5, seed=21)
    n = mu.size
    z = optim.svi_draw(mu, Lp, xi)
    logq, s = optim.svi_score_terms(mu, Lp, xi)

    def lq(mu_, Lp_):
        L_ = optim.tril_unpack(n, Lp_)
        return multivariate_normal(mean=mu_, cov=L_ @ L_.T).logpdf(z)

    assert np.allclose(logq, lq(mu, Lp), rtol=1e-12, atol=1e-12)
    h = 1e-6
    for j in range(n):
        e = np.zeros(n); e[j] = h
        assert np.allclose((lq(mu + e, Lp) - lq(mu - e, Lp)) / (2 * h), s[:, j], rtol=1e-6, atol=1e-7)
    L = optim.tril_unpack(n, Lp)
    rows, cols = np.tril_indices(n)
    for t, (j, k) in enumerate(zip(rows, cols)):
        e = np.zeros_like(Lp); e[t] = h
        want = s[:, j] * xi[:, k] - (1.0 / L[j, j] if j == k else 0.0)
        assert np.allclose((lq(mu, Lp + e) - lq(mu, Lp - e)) / (2 * h), want, rtol=1e-6, atol=1e-7)


@pytest.mark.parametrize("baseline", [True, False])
def test_svi_score_estimator_is_unbiased(baseline):
    """Gaussian target N(a, A^-1): the exact gradient of the loss is d/dmu = A (mu - a), d/dL = tril(A L) - diag(1/L_jj).
    Twenty independent estimates of 20,000 draws each scatter around it: their mean lies within 5 standard errors in
    every entry, with the leave-one-out baseline and (at a much larger scatter) as Eq. 3 prints it."""
    mu, Lp, _, _, a, A = _svi_setup(n=3, seed=5)
    n = mu.size
    L = optim.tril_unpack(n, Lp)
    exact = np.concatenate([A @ (mu - a), optim.tril_pack(np.tril(A @ L) - np.diag(1.0 / np.diag(L)))])
    rng = np.random.default_rng(77)
    est = []
    for _ in range(20):
        xi = rng.standard_normal((20000, n))
        d = optim.svi_draw(mu, Lp, xi) - a
        lp = -0.5 * np.einsum("ij,jk,ik->i", d, A, d) + 3.7             # an additive constant must not matter on average
        _, g_mu, g_L, N = optim.svi_loss_and_grad_score(mu, Lp, xi, lp, baseline)
        assert N == 20000
        est.append(np.concatenate([g_mu, g_L]))
    est = np.array(est)
    se = est.std(axis=0, ddof=1) / np.sqrt(est.shape[0])
    assert np.all(np.abs(est.mean(axis=0) - exact) < 5 * se + 1e-12), (est.mean(axis=0) - exact) / se
    if baseline:
        assert np.all(se < 0.05 * (1 + np.abs(exact)))                  # and it is tight enough to mean something


def test_svi_score_agrees_with_the_pathwise_estimator():
    """Both estimators estimate the same gradient: on the non-Gaussian toy target their averages over many draws agree
    within the score estimator's standard error."""
    mu, Lp, _, f, _, _ = _svi_setup(n=3, seed=9)
    rng = np.random.default_rng(4)
    sc, pw = [], []
    for _ in range(20):
        xi = rng.standard_normal((20000, mu.size))
        lp, g = f(optim.svi_draw(mu, Lp, xi))
        _, a1, b1, _ = optim.svi_loss_and_grad_score(mu, Lp, xi, lp, True)
        _, a2, b2, _ = optim.svi_loss_and_grad(mu, Lp, xi, lp, g)
        sc.append(np.concatenate([a1, b1])); pw.append(np.concatenate([a2, b2]))
    sc, pw = np.array(sc), np.array(pw)
    se = np.sqrt(sc.var(axis=0, ddof=1) + pw.var(axis=0, ddof=1)) / np.sqrt(sc.shape[0])
    assert np.all(np.abs(sc.mean(axis=0) - pw.mean(axis=0)) < 5 * se)


def test_svi_score_constant_weight_and_non_finite_draws():
    """w_i constant (log p~ = log q~ - const): the baseline form returns exactly zero, the printed form const * mean of
    grad log q~ (which is O(1/sqrt N)); draws with a non-finite log p~ are left out."""
    mu, Lp, xi, f, _, _ = _svi_setup(n=4, N=4000, seed=12)
    logq, s = optim.svi_score_terms(mu, Lp, xi)
    _, g_mu, g_L, _ = optim.svi_loss_and_grad_score(mu, Lp, xi, logq - 2.5, True)
    assert np.max(np.abs(g_mu)) < 1e-12 and np.max(np.abs(g_L)) < 1e-12
    _, g_mu, g_L, _ = optim.svi_loss_and_grad_score(mu, Lp, xi, logq - 2.5, False)
    assert np.allclose(g_mu, 2.5 * s.mean(axis=0)) and np.max(np.abs(g_mu)) < 2.5 * 5 / np.sqrt(4000) * np.abs(s).max()
    lp, _ = f(optim.svi_draw(mu, Lp, xi))
    lp2 = lp.copy(); lp2[7] = -np.inf
    r1 = optim.svi_loss_and_grad_score(mu, Lp, np.delete(xi, 7, 0), np.delete(lp, 7), True)
    r2 = optim.svi_loss_and_grad_score(mu, Lp, xi, lp2, True)
    assert r1[3] == r2[3] == 3999 and np.isclose(r1[0], r2[0]) and np.allclose(r1[1], r2[1]) and np.allclose(r1[2], r2[2])


def test_svi_score_fits_a_gaussian_target():
    """The score-function iteration (log p~ only) recovers mean and covariance of a Gaussian target."""
    rng = np.random.default_rng(1)
    n = 2
    A = np.array([[2.0, 0.4], [0.4, 1.0]]); a = np.array([0.5, -1.0])

    def logp(z):
        d = z - a
        return -0.5 * np.einsum("ij,jk,ik->i", d, A, d)

    mu = np.zeros(n); Lp = optim.tril_pack(np.eye(n)); m = np.zeros(n + 3); v = np.zeros(n + 3)
    opt = dict(kind=optim.ADAM, lr=2e-2, b1=0.9, b2=0.999, eps=1e-8)
    for t in range(1, 1201):
        _, mu, Lp, m, v, _ = optim.svi_step_score(logp, mu, Lp, rng.standard_normal((512, n)), m, v, t, opt, True)
    L = optim.tril_unpack(n, Lp)
    assert np.allclose(mu, a, atol=0.08)
    assert np.allclose(L @ L.T, np.linalg.inv(A), atol=0.12)
