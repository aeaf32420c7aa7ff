"""Pins for the oracle's hand-derived reverse-mode gradient (O9): central finite differences with one
Richardson step, in fp64, for every partial of every component and end to end on tiny grids.  CPU only.
"""
import math

import numpy as np
import pytest

import oracle
import workloads as W


def fd(f, x, h):
    """Richardson-extrapolated central difference, O(h^4)."""
    d1 = (f(x + h) - f(x - h)) / (2 * h)
    d2 = (f(x + h / 2) - f(x - h / 2)) / h
    return (4 * d2 - d1) / 3


def close(a, b, rtol=2e-7, atol=1e-9):
    return abs(a - b) <= atol + rtol * max(abs(a), abs(b))


# --------------------------------------------------------------------------- point-wise partials
@pytest.mark.parametrize("t", [0.6, 1.0, 1.4])
def test_epl_frame_partials(t):
    b, q, x, y = 1.1, 0.62, 0.8, -0.55
    r = oracle.epl_frame(b, t, q, x, y)
    A = lambda **k: oracle.epl_frame(**{**dict(b=b, t=t, q=q, x=x, y=y), **k})["alpha"]
    h = 1e-3
    for name, key in (("d_b", "b"), ("d_t", "t"), ("d_q", "q")):
        ref = fd(lambda v: A(**{key: v}), dict(b=b, t=t, q=q)[key], h)
        assert abs(r[name] - ref) < 3e-9 * max(1, abs(ref)), (name, r[name], ref)
    jx = fd(lambda v: A(x=v), x, h); jy = fd(lambda v: A(y=v), y, h)
    Jxx, Jyy, Jxy = r["J"]
    assert close(Jxx, jx.real, 1e-8) and close(Jxy, jx.imag, 1e-8) and close(Jxy, jy.real, 1e-8) and close(Jyy, jy.imag, 1e-8)


def test_epl_frame_q_derivative_near_circular():
    # f -> 0: the S1/f series must stay finite and correct
    b, t, x, y = 1.0, 1.3, 0.7, 0.4
    for q in (0.999999, 0.9999):
        r = oracle.epl_frame(b, t, q, x, y)
        ref = fd(lambda v: oracle.epl_frame(b, t, v, x, y)["alpha"], q, 5e-5 if q < 0.99999 else 5e-7)
        assert abs(r["d_q"] - ref) < 1e-6


def test_sie_frame_partials_and_agreement_with_epl():
    b, q, x, y = 0.9, 0.55, -0.7, 0.45
    r = oracle.sie_frame(b, q, x, y)
    A = lambda **k: oracle.sie_frame(**{**dict(b=b, q=q, x=x, y=y), **k})["alpha"]
    assert abs(r["d_b"] - fd(lambda v: A(b=v), b, 1e-3)) < 1e-9
    assert abs(r["d_q"] - fd(lambda v: A(q=v), q, 1e-3)) < 1e-9
    jx = fd(lambda v: A(x=v), x, 1e-3); jy = fd(lambda v: A(y=v), y, 1e-3)
    Jxx, Jyy, Jxy = r["J"]
    assert close(Jxx, jx.real, 1e-8) and close(Jxy, jx.imag, 1e-8) and close(Jyy, jy.imag, 1e-8)
    e = oracle.epl_frame(b, 1.0, q, x, y)                 # same function, two derivations
    for k in ("alpha", "d_b", "d_q"):
        assert abs(e[k] - r[k]) < 1e-13
    assert np.allclose(e["J"], r["J"], atol=1e-13)


@pytest.mark.parametrize("p", [[0.3, 1.7, 0.12, -0.2, 0.05, -0.04, 7.0], [0.9, 4.2, -0.05, 0.08, 0.01, 0.02, 3.0],
                               [0.25, 0.8, 0.3, 0.1, -0.1, 0.1, 1.0]])
def test_sersic_partials(p):
    x, y = 0.31, -0.22
    v, dp, dxy = oracle.sersic(p, x, y, want_grad=True)
    for k in range(7):
        def f(val, k=k):
            pp = list(p); pp[k] = val; return oracle.sersic(pp, x, y)
        assert close(dp[k], fd(f, p[k], 1e-3 * max(1, abs(p[k]))), 1e-8), k
    assert close(dxy[0], fd(lambda xx: oracle.sersic(p, xx, y), x, 1e-3), 1e-8)
    assert close(dxy[1], fd(lambda yy: oracle.sersic(p, x, yy), y, 1e-3), 1e-8)


def test_shapelet_partials():
    rng = np.random.default_rng(0)
    nmax = 4; nc = W.n_shapelet_coef(nmax)
    p = np.concatenate([[0.17], rng.normal(size=nc)])
    x0, y0, x, y = 0.03, -0.02, 0.21, 0.09
    v, da, dxy = oracle.shapelets(nmax, p, x0, y0, x, y, want_grad=True)
    for k in range(nc + 1):
        def f(val, k=k):
            pp = p.copy(); pp[k] = val; return oracle.shapelets(nmax, pp, x0, y0, x, y)
        assert close(da[k], fd(f, p[k], 1e-3), 1e-8), k
    assert close(dxy[0], fd(lambda xx: oracle.shapelets(nmax, p, x0, y0, xx, y), x, 1e-3), 1e-8)
    assert close(dxy[1], fd(lambda yy: oracle.shapelets(nmax, p, x0, y0, x, yy), y, 1e-3), 1e-8)
    assert close(-dxy[0], fd(lambda xx: oracle.shapelets(nmax, p, xx, y0, x, y), x0, 1e-3), 1e-8)


# --------------------------------------------------------------------------- end to end
def _tiny(kind, param_space):
    rng = np.random.default_rng(11)
    if kind == "sie":
        sp = W.LensSpec(6, 2, 3, 0.30, mass_model=0, param_space=param_space)
        pri = W._default_priors(0)
        th = [0.55, 0.10, -0.05, 0.02, -0.03, 0.03, -0.02, 0.20, 1.5, 0.10, 0.05, 0.05, -0.04, 8.0,
              0.60, 3.0, -0.05, 0.08, 0.01, 0.02, 4.0]
        # widen supports so the fixed theta above is inside them
        pri[0] = W.Uniform(0.3, 1.5)
    elif kind == "multi":
        # the component list of the paper's real-system model (env, L1, L2 lens light; S1, S2 sources)
        sp = W.LensSpec(8, 2, 5, 0.25, mass_model=1, n_source_sersic=2, n_lens_sersic=3, param_space=param_space)
        pri = W._default_priors(1, n_lens=3, n_src=2)
        pri[0] = W.Uniform(0.3, 1.5)
        th = [0.62, 2.1, 0.12, -0.07, 0.03, -0.02, 0.04, -0.03,
              0.22, 1.6, 0.1, 0.06, 0.06, -0.05, 9.0, 0.31, 2.2, -0.08, 0.05, 0.25, -0.21, 5.0,
              0.7, 3.1, -0.05, 0.08, 0.01, 0.02, 4.0, 1.2, 2.4, 0.04, -0.03, -0.01, 0.015, 1.5,
              0.9, 4.0, 0.06, 0.02, 0.012, -0.018, 2.5]
    else:
        sp = W.LensSpec(8, 2, 5, 0.25, mass_model=1, multipole_mask=3, shapelet_nmax=3, n_lens_sersic=2,
                        param_space=param_space)
        pri = W._default_priors(1, multipoles=True, shapelet_nmax=3, n_lens=2)
        pri[0] = W.LogNormal(math.log(0.6), 0.4)            # exercise every prior family
        th = ([0.62, 2.2, 0.12, -0.07, 0.03, -0.02, 0.04, -0.03, 0.012, -0.006, 0.004, 0.009,
               0.22, 1.6, 0.1, 0.06, 0.06, -0.05, 9.0, 0.15] + list(rng.normal(0, 1, 10)) +
              [0.7, 3.1, -0.05, 0.08, 0.01, 0.02, 4.0, 1.2, 2.4, 0.04, -0.03, -0.01, 0.015, 1.5])
    sp.priors = pri
    K = sp.psf_size
    psf = rng.uniform(0.2, 1.0, (1, K, K)); psf /= psf.sum()
    obs = rng.normal(0.5, 0.3, (1, sp.n_pix, sp.n_pix))
    sig = rng.uniform(0.05, 0.2, (1, sp.n_pix, sp.n_pix))
    th = np.array(th)
    assert len(th) == sp.n_params
    x = th if param_space == 1 else W.z_of(pri, th)[0]
    return sp, psf, obs, sig, x


@pytest.mark.parametrize("kind", ["sie", "epl_full", "multi"])
@pytest.mark.parametrize("param_space", [1, 0])
def test_gradient_vs_finite_differences(kind, param_space):
    sp, psf, obs, sig, x0 = _tiny(kind, param_space)
    o = oracle.logpost_grad(sp, obs, sig, psf, [x0], want_gabs=True)
    assert np.isfinite(o["logp"][0])
    g = o["grad"][0]

    def lp(x):
        return oracle.logpost_grad(sp, obs, sig, psf, [x], want_grad=False)["logp"][0]
    for k in range(sp.n_params):
        def f(v, k=k):
            x = x0.copy(); x[k] = v; return lp(x)
        h = 2e-4 * max(1.0, abs(x0[k]))
        ref = fd(f, x0[k], h)
        assert abs(g[k] - ref) < 2e-6 * abs(ref) + 1e-5, (k, g[k], ref)


@pytest.mark.parametrize("param_space", [1, 0])
def test_gradient_sis_branch_vs_finite_differences(param_space):
    """SIE with mass eps == 0 exactly (q' < 1e-6: the SIS branch of sie_frame, theta_E = 0.55 so the lens does deflect):
    every gradient component except the two mass ellipticities against central differences; the ellipticity
    components are the guard value 0 (O9: c < 1e-10)."""
    sp, psf, obs, sig, x0 = _tiny("sie", param_space)
    x0 = x0.copy(); x0[1] = 0.0; x0[2] = 0.0
    o = oracle.logpost_grad(sp, obs, sig, psf, [x0])
    g = o["grad"][0]
    assert np.isfinite(o["logp"][0])
    if param_space == 1:
        assert g[1] == 0.0 and g[2] == 0.0
    lp = lambda x: oracle.logpost_grad(sp, obs, sig, psf, [x], want_grad=False)["logp"][0]
    for k in [0] + list(range(3, sp.n_params)):
        def f(v, k=k):
            x = x0.copy(); x[k] = v; return lp(x)
        ref = fd(f, x0[k], 2e-4 * max(1.0, abs(x0[k])))
        assert abs(g[k] - ref) < 2e-6 * abs(ref) + 1e-5, (k, g[k], ref)
    # and the branch agrees with the EPL series at gamma = 2 on the same circular lens (same logp, same gradient)
    ep = W.LensSpec(6, 2, 3, 0.30, mass_model=1, param_space=1)
    ep.priors = [W.NoPrior()] * 22
    th = x0 if param_space == 1 else W.theta_of(sp.priors, x0[None])[0]
    sp1 = W.LensSpec(6, 2, 3, 0.30, mass_model=0, param_space=1); sp1.priors = [W.NoPrior()] * 21
    a = oracle.logpost_grad(sp1, obs, sig, psf, [th])
    b = oracle.logpost_grad(ep, obs, sig, psf, [np.concatenate([th[:1], [2.0], th[1:]])])
    assert abs(a["logp"][0] - b["logp"][0]) < 1e-9 * abs(a["logp"][0])
    gb = np.delete(b["grad"][0], 1)
    keep = [0] + list(range(3, 21))
    assert np.allclose(a["grad"][0][keep], gb[keep], rtol=1e-9, atol=1e-7)


def test_gradient_truncated_series_matches_its_own_finite_difference():
    """The epl_terms>0 (debug) mode differentiates the truncated sum term by term."""
    sp, psf, obs, sig, x0 = _tiny("epl_full", 1)
    o = oracle.logpost_grad(sp, obs, sig, psf, [x0], epl_terms=12)
    for k in (0, 1, 2, 3, 4, 5):
        def f(v, k=k):
            x = x0.copy(); x[k] = v
            return oracle.logpost_grad(sp, obs, sig, psf, [x], want_grad=False, epl_terms=12)["logp"][0]
        ref = fd(f, x0[k], 2e-4)
        assert abs(o["grad"][0][k] - ref) < 2e-6 * abs(ref) + 1e-5


def test_gradient_config1_prior_particles_fd_spotcheck():
    """Realistic scale (config 1, 40x40, s=2): a few parameters of a few prior-drawn particles."""
    wl = W.make_workload(1, n_particles=3)
    sp = wl.spec
    truth = oracle.model_image(sp, wl.psf.astype(np.float64), wl.truth_theta)
    obs, sig = W.finish_observation(wl, truth)
    z = wl.params.astype(np.float64)
    o = oracle.logpost_grad(sp, obs, sig, wl.psf, z, want_gabs=True)
    for p in range(3):
        for k in (0, 2, 4, 6, 7, 8, 11, 13, 15, 20):
            def f(v):
                x = z[p].copy(); x[k] = v
                return oracle.logpost_grad(sp, obs, sig, wl.psf, [x], want_grad=False)["logp"][0]
            ref = fd(f, z[p, k], 1e-4 * max(1, abs(z[p, k])))
            assert abs(o["grad"][p, k] - ref) < 1e-6 * abs(ref) + 1e-9 * o["gabs"][p, k] + 1e-4, (p, k, o["grad"][p, k], ref)


def test_two_sources_three_lens_blocks_add_up_from_single_component_models():
    """The model image is additive over light components: the 2-source, 3-lens-block model equals the
    sum of three renderings through the ONE-source, ONE-lens-block layout that every other pin exercises, and the
    parameter count follows S18 with the second source right after the first."""
    sp, psf, obs, sig, th = _tiny("multi", 1)
    full = oracle.model_image(sp, psf, th[None])[0]
    one = W.LensSpec(8, 2, 5, 0.25, mass_model=1, n_source_sersic=1, n_lens_sersic=1, param_space=1)
    one.priors = W._default_priors(1)
    mass = th[:8]
    s1, s2, l0, l1, l2 = th[8:15], th[15:22], th[22:29], th[29:36], th[36:43]
    dark = s1.copy(); dark[6] = 0.0
    parts = [np.concatenate([mass, a, b]) for a, b in ((s1, l0), (s2, l1), (dark, l2))]
    pieces = oracle.model_image(one, psf, np.array(parts))
    assert np.allclose(pieces.sum(axis=0), full, rtol=1e-13, atol=1e-13 * np.abs(full).max())
    assert sp.n_params == 43 and W.param_names(1, 1, 0, 2, -1, 3)[15] == "src2.R"
    # each piece carries light (the test would pass trivially on dark components)
    assert all(np.abs(p).max() > 1e-3 * np.abs(full).max() for p in pieces)


# --------------------------------------------------------------------------- two source planes (NEXT-4, reading S23)
def _two_plane(param_space, eta):
    """EPL + shear, two source Sersics (the second on its own plane, eta2 = `eta`), two lens-light blocks, 8x8, s = 2."""
    rng = np.random.default_rng(23)
    sp = W.LensSpec(8, 2, 5, 0.25, mass_model=1, n_source_sersic=2, n_lens_sersic=2, source2_plane=1, param_space=param_space)
    pri = W._default_priors(1, n_lens=2, n_src=2, src2_plane=True)
    pri[0] = W.Uniform(0.3, 1.5)
    sp.priors = pri
    th = np.array([0.62, 2.1, 0.12, -0.07, 0.03, -0.02, 0.04, -0.03,
                   0.22, 1.6, 0.1, 0.06, 0.06, -0.05, 9.0, 0.31, 2.2, -0.08, 0.05, 0.25, -0.21, 5.0, eta,
                   0.7, 3.1, -0.05, 0.08, 0.01, 0.02, 4.0, 1.2, 2.4, 0.04, -0.03, -0.01, 0.015, 1.5])
    assert len(th) == sp.n_params == 37 and W.param_names(1, 1, 0, 2, -1, 2, 1)[22] == "src2.eta"
    K = sp.psf_size
    psf = rng.uniform(0.2, 1.0, (1, K, K)); psf /= psf.sum()
    obs = rng.normal(0.5, 0.3, (1, 8, 8)); sig = rng.uniform(0.05, 0.2, (1, 8, 8))
    return sp, psf, obs, sig, th


def test_two_source_planes_end_points_and_shear_closed_form():
    """beta_2 = theta - eta2 alpha(theta) ("multi-source-plane systems"; reading S23).  eta2 = 1 IS the one-plane
    model, bit for bit; eta2 = 0 leaves the second source unlensed, i.e. it renders like a lens-plane Sersic block with
    the same parameters; under a pure external shear the total flux of the second source is F / (1 - eta2^2 |gamma|^2)
    (the shear-only magnification with the shear scaled by eta2: closed form at an intermediate eta2)."""
    import dataclasses
    sp, psf, obs, sig, th = _two_plane(1, 1.0)
    one = dataclasses.replace(sp, source2_plane=0, priors=sp.priors[:22] + sp.priors[23:])
    a = oracle.logpost_grad(sp, obs, sig, psf, [th], want_model=True)
    b = oracle.logpost_grad(one, obs, sig, psf, [np.delete(th, 22)], want_model=True)
    assert np.array_equal(a["model"], b["model"]) and a["logp"][0] == b["logp"][0]
    assert np.array_equal(np.delete(a["grad"][0], 22), b["grad"][0])
    # eta2 = 0: second source unlensed == (second source dark) + (a third lens-light block with its parameters)
    th0 = th.copy(); th0[22] = 0.0
    m0 = oracle.model_image(sp, psf, [th0])[0]
    three = W.LensSpec(8, 2, 5, 0.25, mass_model=1, n_source_sersic=2, n_lens_sersic=3, source2_plane=1, param_space=1)
    three.priors = sp.priors + W._default_priors(1)[-7:]
    dark = th0.copy(); dark[21] = 0.0
    m1 = oracle.model_image(three, psf, [np.concatenate([dark, th0[15:22]])])[0]
    assert np.allclose(m0, m1, rtol=1e-13, atol=1e-13 * np.abs(m0).max())
    assert np.abs(m0 - oracle.model_image(sp, psf, [th])[0]).max() > 1e-3 * np.abs(m0).max()      # eta2 matters
    # shear-only lens (theta_E -> 0), first source dark: flux of the second source = F / (1 - eta^2 (g1^2 + g2^2))
    g1, g2, R, n, Ie = 0.05, -0.03, 0.15, 1.0, 2.0
    bn = 1.9992 * n - 0.3271
    F = 2 * math.pi * n * Ie * R * R * math.exp(bn) * math.gamma(2 * n) / bn ** (2 * n)
    fl = W.LensSpec(200, 1, 3, 0.02, mass_model=0, has_shear=1, n_source_sersic=2, n_lens_sersic=0, source2_plane=1, param_space=1)
    fl.priors = [W.NoPrior()] * 22
    for eta in (0.6, 1.0, 1.4):
        ray = oracle.ray_image(fl, [1e-13, 0, 0, 0, 0, g1, g2, R, n, 0, 0, 0, 0, 0.0, R, n, 0.1, -0.05, 0.01, -0.02, Ie, eta])
        assert abs(ray.sum() * 0.02 ** 2 / (F / (1 - eta * eta * (g1 * g1 + g2 * g2))) - 1) < 2e-3, eta
    r1 = oracle.ray_image(fl, [1e-13, 0, 0, 0, 0, g1, g2, R, n, 0, 0, 0, 0, 0.0, R, n, 0.1, -0.05, 0.01, -0.02, Ie, 0.6]).sum()
    r2 = oracle.ray_image(fl, [1e-13, 0, 0, 0, 0, g1, g2, R, n, 0, 0, 0, 0, 0.0, R, n, 0.1, -0.05, 0.01, -0.02, Ie, 1.4]).sum()
    assert abs(r2 / r1 - (1 - 0.36 * (g1 * g1 + g2 * g2)) / (1 - 1.96 * (g1 * g1 + g2 * g2))) < 2e-5    # the eta dependence itself


@pytest.mark.parametrize("param_space", [1, 0])
@pytest.mark.parametrize("eta", [0.8, 1.35])
def test_two_source_planes_gradient_vs_finite_differences(param_space, eta):
    """Every component, eta2 included (d beta_2 / d eta2 = -alpha; the mass parameters see the second source through
    eta2 d alpha / d theta_mass)."""
    sp, psf, obs, sig, th = _two_plane(param_space, eta)
    x0 = th if param_space == 1 else W.z_of(sp.priors, th)[0]
    o = oracle.logpost_grad(sp, obs, sig, psf, [x0])
    assert np.isfinite(o["logp"][0])
    g = o["grad"][0]
    lp = lambda x: oracle.logpost_grad(sp, obs, sig, psf, [x], want_grad=False)["logp"][0]
    for k in range(sp.n_params):
        def f(v, k=k):
            x = x0.copy(); x[k] = v; return lp(x)
        ref = fd(f, x0[k], 2e-4 * max(1.0, abs(x0[k])))
        assert abs(g[k] - ref) < 2e-6 * abs(ref) + 1e-5, (k, g[k], ref)
    assert abs(g[22]) > 1e-2                                             # eta2 carries a real gradient
