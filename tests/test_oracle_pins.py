"""Pins for the fp64 oracle: each part is checked against something OTHER than itself -- closed forms,
direct numerical integration, scipy/mpmath special functions, invariants, survey golden values
(tests/golden/survey_appendix_b.json).  CPU only.  See SURVEY.md 8(c) "Pins" and DESIGN.md section 3.
"""
import json
import math
import os

import numpy as np
import pytest
from scipy import integrate, signal, special, stats

import oracle
import workloads as W

GOLD = json.load(open(os.path.join(os.path.dirname(__file__), "golden", "survey_appendix_b.json")))


def mass_spec(mass_model, has_shear=0, multipole_mask=0, n=8, s=1, K=3, scale=0.1):
    sp = W.LensSpec(n, s, K, scale, mass_model=mass_model, has_shear=has_shear, multipole_mask=multipole_mask,
                    n_source_sersic=0, n_lens_sersic=0, param_space=1)
    npar = (6 if mass_model == 1 else 5) + 2 * has_shear + 2 * bin(multipole_mask).count("1")
    sp.priors = [W.NoPrior()] * npar
    return sp


# --------------------------------------------------------------------------- deflection
def _kappa_epl(thE, gamma, q, xr, yr):
    """Convergence of the EPL, product-averaged normalisation (reading S3), typed from its definition."""
    return 0.5 * (3.0 - gamma) * (thE / math.sqrt(q * xr * xr + yr * yr / q)) ** (gamma - 1.0)


def _alpha_by_quadrature(thE, gamma, q, x, y, trunc):
    """alpha(theta) = (1/pi) Int kappa(theta') (theta-theta')/|theta-theta'|^2 d2theta' in the mass frame,
    polar about the field point, truncated on the homoeoid q x^2 + y^2/q = (trunc*m_theta)^2 (Newton's
    theorem: shells outside the point contribute nothing, so trunc = 1 and 2 must agree)."""
    m2 = (trunc ** 2) * (q * x * x + y * y / q)
    a0 = math.atan2(-y, -x)                       # direction towards the centre (log-singular inner integral)

    def rmax(a):
        ux, uy = math.cos(a), math.sin(a)
        A = q * ux * ux + uy * uy / q
        B = 2 * (q * x * ux + y * uy / q)
        Cc = q * x * x + y * y / q - m2
        disc = B * B - 4 * A * Cc
        if disc <= 0: return 0.0
        return max((-B + math.sqrt(disc)) / (2 * A), 0.0)

    def inner(a):
        rm = rmax(a)
        if rm <= 0: return 0.0
        ux, uy = math.cos(a), math.sin(a)
        rc = -(x * ux + y * uy)                   # closest approach to the centre
        pts = [rc] if 0 < rc < rm else None
        val, _ = integrate.quad(lambda r: _kappa_epl(thE, gamma, q, x + r * ux, y + r * uy), 0, rm,
                                points=pts, epsabs=1e-13, epsrel=1e-13, limit=400)
        return val

    out = []
    for comp in (math.cos, math.sin):
        lo, hi = a0 - math.pi, a0 + math.pi
        v1, _ = integrate.quad(lambda a: inner(a) * comp(a), lo, a0, epsabs=1e-11, epsrel=1e-11, limit=400)
        v2, _ = integrate.quad(lambda a: inner(a) * comp(a), a0, hi, epsabs=1e-11, epsrel=1e-11, limit=400)
        out.append(-(v1 + v2) / math.pi)          # (theta - theta') = -r u
    return out


@pytest.mark.filterwarnings("ignore::scipy.integrate.IntegrationWarning")
@pytest.mark.parametrize("gamma,tol", [(2.0, 2e-9), (1.7, 5e-7), (2.3, 5e-7)])
def test_deflection_vs_direct_integration_of_kappa(gamma, tol):
    thE, q = 1.2, 0.709401709402
    x, y = 0.62, -0.51                            # mass-frame point
    sp = mass_spec(1)
    c = (1 - q) / (1 + q)                         # eps along x => phi = 0, mass frame = lab frame
    ax, ay = oracle.deflection(sp, [thE, gamma, c, 0.0, 0.0, 0.0], x, y)
    for trunc in (1.0, 2.0):
        qx, qy = _alpha_by_quadrature(thE, gamma, q, x, y, trunc)
        assert abs(qx - ax) < tol and abs(qy - ay) < tol, (trunc, qx - ax, qy - ay)
    if gamma == 2.0:
        sx, sy = oracle.deflection(mass_spec(0), [thE, c, 0.0, 0.0, 0.0], x, y)
        qx, qy = _alpha_by_quadrature(thE, 2.0, q, x, y, 1.0)
        assert abs(qx - sx) < tol and abs(qy - sy) < tol


def test_epl_series_is_hyp2f1():
    mp = pytest.importorskip("mpmath")
    rng = np.random.default_rng(1)
    for _ in range(20):
        q = rng.uniform(0.3, 0.95); t = rng.uniform(0.3, 1.7); b = rng.uniform(0.5, 1.5)
        x, y = rng.uniform(-2, 2, 2)
        R = math.hypot(q * x, y); f = (1 - q) / (1 + q)
        E = complex(q * x, y) / R
        F = complex(mp.hyp2f1(1, t / 2, 2 - t / 2, -f * E * E))
        ref = 2 * b / (1 + q) * (b / R) ** (t - 1) * E * F
        got = oracle.epl_frame(b, t, q, x, y)["alpha"]
        assert abs(got - ref) < 1e-14 * abs(ref)
    # scipy's complex hyp2f1 as a second, independent library
    E = complex(0.6 * 0.7, -0.4) / math.hypot(0.6 * 0.7, 0.4)
    F = special.hyp2f1(1, 0.65, 2 - 0.65, -0.25 * E * E)
    ref = 2 * 1.1 / 1.6 * (1.1 / math.hypot(0.42, 0.4)) ** 0.3 * E * F
    assert abs(oracle.epl_frame(1.1, 1.3, 0.6, 0.7, -0.4)["alpha"] - ref) < 1e-12


def test_epl_at_gamma_2_is_sie_and_truncation_bound():
    rng = np.random.default_rng(2)
    for _ in range(50):
        thE = rng.uniform(0.5, 2); e1, e2 = rng.normal(0, 0.2, 2); x0, y0 = rng.normal(0, 0.1, 2)
        x, y = rng.uniform(-3, 3, 2)
        a = oracle.deflection(mass_spec(1), [thE, 2.0, e1, e2, x0, y0], x, y)
        b = oracle.deflection(mass_spec(0), [thE, e1, e2, x0, y0], x, y)
        assert np.allclose(a, b, rtol=0, atol=2e-14)
    # 30-term truncation (reading S5): relative error <= c^30/(1-c)
    for c in (0.3, 0.5, 0.6):
        full = np.array(oracle.deflection(mass_spec(1), [1.2, 2.2, c, 0.0, 0, 0], 0.9, 0.4))
        tr = np.array(oracle.deflection(mass_spec(1), [1.2, 2.2, c, 0.0, 0, 0], 0.9, 0.4, epl_terms=30))
        assert np.abs(full - tr).max() <= c ** 30 / (1 - c) * np.abs(full).max()


def test_golden_b1_deflection_and_geometry():
    for row in GOLD["B1"]["rows"]:
        ax, ay = oracle.deflection(mass_spec(1), [1.2, row["gamma"], 0.15, -0.08, 0.03, -0.02], 0.7, -0.45)
        assert abs(ax - row["ax"]) < 2e-12 and abs(ay - row["ay"]) < 2e-12
    c = math.hypot(0.15, -0.08)
    assert abs((1 - c) / (1 + c) - GOLD["B1"]["q"]) < 1e-12
    assert abs(0.5 * math.atan2(-0.08, 0.15) - GOLD["B1"]["phi"]) < 1e-12


@pytest.mark.parametrize("gamma", [1.7, 2.0, 2.3])
def test_divergence_is_2kappa_and_curl_free(gamma):
    sp = mass_spec(1); th = [1.2, gamma, 0.15, -0.08, 0.03, -0.02]
    x, y, h = 0.7, -0.45, 1e-5
    d = lambda xx, yy: np.array(oracle.deflection(sp, th, xx, yy))
    dax = (d(x + h, y) - d(x - h, y)) / (2 * h); day = (d(x, y + h) - d(x, y - h)) / (2 * h)
    c = math.hypot(0.15, -0.08); q = (1 - c) / (1 + c); phi = 0.5 * math.atan2(-0.08, 0.15)
    dx, dy = x - 0.03, y + 0.02
    xr, yr = math.cos(phi) * dx + math.sin(phi) * dy, -math.sin(phi) * dx + math.cos(phi) * dy
    kap = _kappa_epl(1.2, gamma, q, xr, yr)
    row = [r for r in GOLD["B1"]["rows"] if r["gamma"] == gamma][0]
    assert abs(kap - row["kappa"]) < 1e-11                       # the test's kappa is the survey's
    assert abs(0.5 * (dax[0] + day[1]) - kap) < 1e-8
    assert abs(dax[1] - day[0]) < 1e-8


@pytest.mark.parametrize("gamma", [1.5, 2.0, 2.6])
def test_circular_lens_ring_radius(gamma):
    thE = 1.1
    for ang in (0.0, 0.7, 2.9):
        ax, ay = oracle.deflection(mass_spec(1), [thE, gamma, 0.0, 0.0, 0.0, 0.0], thE * math.cos(ang), thE * math.sin(ang))
        assert abs(math.hypot(ax, ay) - thE) < 1e-13
        assert abs(ax * math.sin(ang) - ay * math.cos(ang)) < 1e-13          # radial
    # a centred compact source is imaged into a ring at theta_E (brightest ray within one ray spacing)
    sp = W.LensSpec(40, 2, 3, 0.1, mass_model=1, has_shear=0, n_lens_sersic=0, param_space=1)
    sp.priors = [W.NoPrior()] * 13
    ray = oracle.ray_image(sp, [thE, gamma, 0, 0, 0, 0, 0.02, 1.0, 0, 0, 0, 0, 1.0])
    i, j = np.unravel_index(np.argmax(ray), ray.shape)
    r = math.hypot(oracle.ray_coord(sp, j), oracle.ray_coord(sp, i))
    assert abs(r - thE) <= 0.1 / 2 * 0.75


@pytest.mark.parametrize("thE", [0.8, 1.3])
@pytest.mark.parametrize("ell", [0.0, 1e-13])
def test_sie_sis_branch_is_the_singular_isothermal_sphere(thE, ell):
    """The q' < 1e-6 branch of sie_frame (the SIS limit of O4; SIE named at PAPER.md L50) with a NON-trivial theta_E:
    |alpha| = theta_E on every ray and radial (closed form of the SIS); equal to the EPL series at t = 1; equal to the
    limit of the q' >= 1e-6 closed form (|eps| = 1e-5: O(eps) away); its Jacobian and d/db against central
    differences of the deflection itself (kappa = theta_E / 2r, pure tangential shear)."""
    e1, e2, x0, y0 = ell * math.cos(0.4), ell * math.sin(0.4), 0.07, -0.04
    th = [thE, e1, e2, x0, y0]
    for (x, y) in ((0.9, 0.3), (-0.2, 1.7), (0.11, -0.05), (-2.4, -0.6)):
        ax, ay = oracle.deflection(mass_spec(0), th, x, y)
        r = math.hypot(x - x0, y - y0)
        assert abs(math.hypot(ax, ay) - thE) < 1e-12
        assert abs(ax - thE * (x - x0) / r) < 1e-12 and abs(ay - thE * (y - y0) / r) < 1e-12
        bx, by = oracle.deflection(mass_spec(1), [thE, 2.0, e1, e2, x0, y0], x, y)
        assert abs(ax - bx) < 1e-12 and abs(ay - by) < 1e-12            # |eps| = 1e-13 itself moves the EPL by O(1e-13)
        cx, cy = oracle.deflection(mass_spec(0), [thE, 1e-5 * math.cos(0.4), 1e-5 * math.sin(0.4), x0, y0], x, y)
        assert abs(ax - cx) < 1e-4 * thE and abs(ay - cy) < 1e-4 * thE
    # frame-level outputs of the branch (b = theta_E at q = 1): alpha, d/db, Jacobian
    c = ell; q = (1 - c) / (1 + c); b = thE * math.sqrt(q)
    x, y, h = 0.6, -0.35, 1e-6
    o = oracle.sie_frame(b, q, x, y)
    assert math.sqrt(1 - q * q) < 1e-6                                   # this IS the SIS branch
    al = lambda xx, yy, bb=b: oracle.sie_frame(bb, q, xx, yy)["alpha"]
    assert abs(o["d_b"] - (al(x, y, b + h) - al(x, y, b - h)) / (2 * h)) < 1e-9
    dax = (al(x + h, y) - al(x - h, y)) / (2 * h); day = (al(x, y + h) - al(x, y - h)) / (2 * h)
    Jxx, Jyy, Jxy = o["J"]
    assert abs(Jxx - dax.real) < 1e-8 and abs(Jyy - day.imag) < 1e-8
    assert abs(Jxy - dax.imag) < 1e-8 and abs(Jxy - day.real) < 1e-8
    assert abs(0.5 * (Jxx + Jyy) - thE / (2 * math.hypot(x, y))) < 1e-9  # kappa of the SIS
    assert o["d_t"] == 0 and o["d_q"] == 0


def test_ray_grid_convention():
    b4 = GOLD["B4"]
    sp = W.LensSpec(6, 2, 3, 0.30)
    xs = [oracle.ray_coord(sp, j) for j in range(12)]
    assert abs(xs[0] - b4["ray_x_first"]) < 1e-15 and abs(xs[1] - b4["ray_x_second"]) < 1e-15
    assert abs(xs[-1] - b4["ray_x_last"]) < 1e-15
    assert np.allclose(np.array(xs) + np.array(xs[::-1]), 0, atol=1e-15)   # centred on the cutout
    # x <-> column, y <-> row: a source displaced to +x lights up larger column indices
    sp = W.LensSpec(10, 1, 3, 0.2, mass_model=0, has_shear=0, n_source_sersic=0, n_lens_sersic=1, param_space=1)
    sp.priors = [W.NoPrior()] * 12
    ray = oracle.ray_image(sp, [1e-12, 0, 0, 0, 0, 0.2, 1.0, 0, 0, 0.5, -0.3, 1.0])
    i, j = np.unravel_index(np.argmax(ray), ray.shape)
    assert abs(oracle.ray_coord(sp, j) - 0.5) <= 0.1 and abs(oracle.ray_coord(sp, i) + 0.3) <= 0.1


def test_shear_only_magnification():
    g1, g2 = 0.05, -0.03
    assert abs(1 / (1 - g1 * g1 - g2 * g2) - GOLD["B3"]["mu"]) < 1e-12
    sp = W.LensSpec(200, 1, 3, 0.02, mass_model=0, has_shear=1, n_lens_sersic=0, param_space=1)
    sp.priors = [W.NoPrior()] * 14
    R, n, Ie = 0.15, 1.0, 2.0
    ray = oracle.ray_image(sp, [1e-13, 0, 0, 0, 0, g1, g2, R, n, 0.1, -0.05, 0.01, -0.02, Ie])
    bn = 1.9992 * n - 0.3271
    Fsrc = 2 * math.pi * n * Ie * R * R * math.exp(bn) * math.gamma(2 * n) / bn ** (2 * n)
    assert abs(ray.sum() * 0.02 ** 2 / (Fsrc * GOLD["B3"]["mu"]) - 1) < 2e-3
    # and the deflection itself, against the potential 1/2 g1 (x^2-y^2) + g2 x y (reading S6)
    psi = lambda x, y: 0.5 * g1 * (x * x - y * y) + g2 * x * y
    x, y, h = 0.4, -0.9, 1e-5
    ax, ay = oracle.deflection(sp, [1e-13, 0, 0, 0, 0, g1, g2, R, n, 0, 0, 0, 0, Ie], x, y)
    assert abs(ax - (psi(x + h, y) - psi(x - h, y)) / (2 * h)) < 1e-9
    assert abs(ay - (psi(x, y + h) - psi(x, y - h)) / (2 * h)) < 1e-9


@pytest.mark.parametrize("mask,m", [(1, 3), (2, 4)])
def test_multipole_is_gradient_of_its_potential(mask, m):
    cm, sm, x0, y0 = 0.013, -0.008, 0.05, -0.02
    sp = mass_spec(1, multipole_mask=mask)
    th = [1e-13, 2.0, 0, 0, x0, y0, cm, sm]

    def psi(x, y):                                     # reading S7
        r = math.hypot(x - x0, y - y0); v = math.atan2(y - y0, x - x0)
        return r / (1 - m * m) * (cm * math.cos(m * v) + sm * math.sin(m * v))
    x, y, h = 0.8, 0.35, 1e-4
    ax, ay = oracle.deflection(sp, th, x, y)
    assert abs(ax - (psi(x + h, y) - psi(x - h, y)) / (2 * h)) < 1e-9
    assert abs(ay - (psi(x, y + h) - psi(x, y - h)) / (2 * h)) < 1e-9
    lap = (psi(x + h, y) + psi(x - h, y) + psi(x, y + h) + psi(x, y - h) - 4 * psi(x, y)) / (h * h)
    r = math.hypot(x - x0, y - y0); v = math.atan2(y - y0, x - x0)
    assert abs(0.5 * lap - (cm * math.cos(m * v) + sm * math.sin(m * v)) / (2 * r)) < 1e-6


# --------------------------------------------------------------------------- light
def test_sersic_total_flux_closed_form_and_half_light():
    for row in GOLD["B2"]["rows"]:
        n, Re, Ie = row["n"], 0.4, 3.0
        bn = 1.9992 * n - 0.3271
        closed = 2 * math.pi * n * Ie * Re * Re * math.exp(bn) * math.gamma(2 * n) / bn ** (2 * n)
        assert abs(closed - row["flux"]) < 1e-9
        for (e1, e2) in ((0.0, 0.0), (0.2, -0.1)):
            c = math.hypot(e1, e2); q = (1 - c) / (1 + c); phi = 0.5 * math.atan2(e2, e1)
            p = [Re, n, e1, e2, 0.07, -0.03, Ie]

            def f(m, psi):                            # elliptical polar coords, area element m dm dpsi
                xr, yr = m * math.cos(psi) / math.sqrt(q), m * math.sqrt(q) * math.sin(psi)
                x = 0.07 + math.cos(phi) * xr - math.sin(phi) * yr
                y = -0.03 + math.sin(phi) * xr + math.cos(phi) * yr
                return oracle.sersic(p, x, y) * m
            tot = sum(integrate.dblquad(f, 0, 2 * math.pi, a, b, epsabs=1e-10, epsrel=1e-10)[0]
                      for a, b in ((0, 0.05), (0.05, Re), (Re, 10 * Re), (10 * Re, 400 * Re)))
            assert abs(tot / closed - 1) < 1e-7, (n, e1, tot, closed)
            inner = sum(integrate.dblquad(f, 0, 2 * math.pi, a, b, epsabs=1e-10, epsrel=1e-10)[0]
                        for a, b in ((0, 0.05), (0.05, Re)))
            assert abs(inner / closed - 0.5) < 3e-3                          # b_n approximation
    # I = I_e on the ellipse r = R_e
    c = math.hypot(0.1, 0.05); q = (1 - c) / (1 + c); phi = 0.5 * math.atan2(0.05, 0.1)
    xr = 0.4 / math.sqrt(q)
    assert abs(oracle.sersic([0.4, 2.5, 0.1, 0.05, 0, 0, 3.0], math.cos(phi) * xr, math.sin(phi) * xr) - 3.0) < 1e-13


def test_shapelet_basis_orthonormal_and_hermite_form():
    nmax = 10
    us = np.linspace(-12, 12, 4801)
    B = np.array([oracle.shapelet_basis(nmax, u) for u in us])        # [u, k]
    G = integrate.simpson(B[:, :, None] * B[:, None, :], x=us, axis=0)
    assert np.abs(G - np.eye(nmax + 1)).max() < 1e-11
    for k in range(nmax + 1):
        ref = special.eval_hermite(k, us) * np.exp(-us * us / 2) / math.sqrt(2.0 ** k * math.sqrt(math.pi) * math.factorial(k))
        assert np.abs(B[:, k] - ref).max() < 5e-14
    assert W.n_shapelet_coef(6) == 28 and W.n_shapelet_coef(10) == 66


def test_shapelet_2d_order_prefactor_and_centre():
    nmax, bs, x0, y0, x, y = 3, 0.2, 0.05, -0.02, 0.17, 0.11
    pu = oracle.shapelet_basis(nmax, (x - x0) / bs); pv = oracle.shapelet_basis(nmax, (y - y0) / bs)
    order = [(0, 0), (1, 0), (0, 1), (2, 0), (1, 1), (0, 2), (3, 0), (2, 1), (1, 2), (0, 3)]   # (n1, n2), reading S9
    for idx, (n1, n2) in enumerate(order):
        a = np.zeros(10); a[idx] = 1.0
        v = oracle.shapelets(nmax, np.concatenate([[bs], a]), x0, y0, x, y)
        assert abs(v - pu[n1] * pv[n2] / bs) < 1e-14
    # total flux of the (0,0) mode: Int phi_0 phi_0 /bs dx dy = bs * (Int phi_0 du)^2 = bs * 2 sqrt(pi)
    g = np.linspace(-3, 3, 1201)
    a = np.zeros(10); a[0] = 1.0
    vals = np.array([[oracle.shapelets(nmax, np.concatenate([[bs], a]), 0, 0, xx, yy) for xx in g[::10]] for yy in g[::10]])
    assert abs(vals.sum() * (g[10] - g[0]) ** 2 / (bs * 2 * math.sqrt(math.pi)) - 1) < 1e-6


# --------------------------------------------------------------------------- image operator
def test_delta_psf_identity_and_flux_conservation():
    rng = np.random.default_rng(3)
    N, s, K, D = 7, 3, 5, 0.2
    ray = rng.uniform(0, 1, (N * s, N * s))
    delta = np.zeros((K, K)); delta[2, 2] = 1.0
    m = oracle.conv_bin(N, s, K, D, delta, ray)
    ref = D * D * ray.reshape(N, s, N, s).mean(axis=(1, 3))
    assert np.abs(m - ref).max() < 1e-16
    # interior source + unit-sum PSF: sum(model) = D^2 sum(ray)/s^2
    psf = rng.uniform(0, 1, (K, K)); psf /= psf.sum()
    ray2 = np.zeros_like(ray); ray2[6:15, 6:15] = rng.uniform(0, 1, (9, 9))
    m2 = oracle.conv_bin(N, s, K, D, psf, ray2)
    assert abs(m2.sum() - D * D * ray2.sum() / s ** 2) < 1e-15


def test_psf_orientation_true_convolution():
    N, s, K = 6, 1, 3
    ray = np.zeros((N, N)); ray[2, 3] = 1.0
    psf = np.zeros((K, K)); psf[2, 1] = 1.0                # tap (c+1, c): moves flux +1 ROW (reading S10)
    m = oracle.conv_bin(N, s, K, 1.0, psf, ray)
    assert m[3, 3] == 1.0 and m.sum() == 1.0
    psf = np.zeros((K, K)); psf[1, 0] = 1.0                # tap (c, c-1): moves flux -1 COLUMN
    m = oracle.conv_bin(N, s, K, 1.0, psf, ray)
    assert m[2, 2] == 1.0 and m.sum() == 1.0
    # zero padding: flux pushed off the edge is lost
    ray = np.zeros((N, N)); ray[5, 0] = 1.0
    psf = np.zeros((K, K)); psf[2, 1] = 1.0
    assert oracle.conv_bin(N, s, K, 1.0, psf, ray).sum() == 0.0


def test_conv_bin_vs_scipy_and_fused_keff_form():
    rng = np.random.default_rng(4)
    N, s, K, D = 12, 4, 7, 0.262
    M = N * s; c = (K - 1) // 2
    ray = rng.normal(size=(M, M)); psf = rng.uniform(size=(K, K))
    m = oracle.conv_bin(N, s, K, D, psf, ray)
    C = signal.convolve2d(ray, psf, mode="same")
    ref = D * D * C.reshape(N, s, N, s).mean(axis=(1, 3))
    assert np.abs(m - ref).max() < 1e-13
    # stride-s correlation with the flipped pre-boxed kernel
    keff = signal.convolve2d(psf, np.ones((s, s)), mode="full")
    kt = keff[::-1, ::-1] / s ** 2
    pad = np.zeros((M + 2 * (K + s), M + 2 * (K + s))); o = K + s
    pad[o:o + M, o:o + M] = ray
    fused = np.array([[D * D * (kt * pad[o + s * p - c:o + s * p - c + K + s - 1, o + s * q - c:o + s * q - c + K + s - 1]).sum()
                       for q in range(N)] for p in range(N)])
    assert np.abs(fused - m).max() < 1e-13


def test_conv_bin_transpose_is_the_adjoint():
    rng = np.random.default_rng(5)
    N, s, K, D = 6, 2, 5, 0.3
    ray = rng.normal(size=(N * s, N * s)); g = rng.normal(size=(N, N)); psf = rng.uniform(size=(K, K))
    lhs = (oracle.conv_bin(N, s, K, D, psf, ray) * g).sum()
    rhs = (ray * oracle.conv_bin_transpose(N, s, K, D, psf, g)).sum()
    assert abs(lhs - rhs) < 1e-12 * max(1, abs(lhs))


# --------------------------------------------------------------------------- likelihood, priors
def _b4_spec():
    sp = W.LensSpec(6, 2, 3, 0.30, mass_model=0, param_space=1)
    sp.priors = [W.NoPrior()] * 21
    k = np.array([0.25, 0.5, 0.25])
    return sp, np.outer(k, k)[None]


def test_likelihood_at_model_equals_obs_and_chi2_definition():
    sp, psf = _b4_spec(); th = GOLD["B4"]["theta"]
    sig = np.random.default_rng(6).uniform(0.05, 0.2, (1, 6, 6))
    m = oracle.model_image(sp, psf, th)
    lp = oracle.logpost_grad(sp, m, sig, psf, [th], want_grad=False)["logp"][0]
    assert abs(lp - (-np.log(sig).sum() - 18 * math.log(2 * math.pi))) < 1e-12
    obs = m + 0.3 * sig
    lp = oracle.logpost_grad(sp, obs, sig, psf, [th], want_grad=False)["logp"][0]
    assert abs(lp - (-0.5 * 36 * 0.09 - np.log(sig).sum() - 18 * math.log(2 * math.pi))) < 1e-11


def test_golden_b4_end_to_end():
    b4 = GOLD["B4"]; sp, psf = _b4_spec()
    o = oracle.logpost_grad(sp, np.zeros((1, 6, 6)), np.full((1, 6, 6), 0.1), psf, [b4["theta"]], want_model=True)
    m = o["model"][0]
    assert abs(m.sum() - b4["sum_model"]) < 1e-10
    assert abs(((m / 0.1) ** 2).sum() - b4["chi2"]) < 1e-8
    assert abs(o["logp"][0] - b4["logL"]) < 1e-9
    for (i, j) in ((0, 0), (2, 3), (3, 4), (5, 5)):
        assert abs(m[i, j] - b4["model_%d_%d" % (i, j)]) < 1e-11
    assert np.abs(o["grad"][0] - np.array(b4["grad"])).max() < 2e-6     # printed to 6 decimals


PRIORS = [W.Normal(0.3, 0.7), W.LogNormal(math.log(1.25), 0.4), W.Uniform(0.8, 1.5),
          W.TruncNormal(0.0, 0.1, -0.15, 0.15), W.TruncNormal(2, 0.5, 1, 3), W.LogUniform(1, 100)]


@pytest.mark.parametrize("prior", PRIORS)
def test_transformed_prior_integrates_to_one_and_matches_scipy(prior):
    k, a, b, lo, hi = prior
    dens = lambda z: math.exp(oracle.transform_one(prior, 0, z)["lp"] + oracle.transform_one(prior, 0, z)["logdet"])
    span = 40.0 if k in (W.PRIOR_UNIFORM, W.PRIOR_TRUNCNORMAL, W.PRIOR_LOGUNIFORM) else 12 * b
    mid = a if k in (W.PRIOR_NORMAL, W.PRIOR_LOGNORMAL) else 0.0
    tot, _ = integrate.quad(dens, mid - span, mid + span, epsabs=1e-13, epsrel=1e-13, limit=500, points=[mid])
    assert abs(tot - 1) < 1e-10
    dist = {W.PRIOR_NORMAL: lambda: stats.norm(a, b),
            W.PRIOR_LOGNORMAL: lambda: stats.lognorm(s=b, scale=math.exp(a)),
            W.PRIOR_UNIFORM: lambda: stats.uniform(lo, hi - lo),
            W.PRIOR_TRUNCNORMAL: lambda: stats.truncnorm((lo - a) / b, (hi - a) / b, loc=a, scale=b),
            W.PRIOR_LOGUNIFORM: lambda: stats.loguniform(lo, hi)}[k]()
    for z in (-2.0, -0.3, 0.0, 0.4, 1.7):
        t = oracle.transform_one(prior, 0, z)
        assert abs(t["lp"] - dist.logpdf(t["theta"])) < 1e-12
        h = 1e-6                                                         # log-det is log|dtheta/dz|
        dth = (oracle.transform_one(prior, 0, z + h)["theta"] - oracle.transform_one(prior, 0, z - h)["theta"]) / (2 * h)
        assert abs(t["logdet"] - math.log(abs(dth))) < 1e-8
        assert abs(t["dth_dz"] - dth) < 1e-8 * max(1, abs(dth))
        assert abs(float(W.to_unconstrained(prior, t["theta"])) - z) < 1e-9   # generator's inverse is the inverse
    if k == W.PRIOR_LOGNORMAL:                                           # LogNormal o exp is exactly Normal(mu, sigma) in z
        for z in (-1.0, 0.2, 0.9):
            t = oracle.transform_one(prior, 0, z)
            assert abs(t["lp"] + t["logdet"] - stats.norm(a, b).logpdf(z)) < 1e-13


def test_physical_space_support_and_invalid_particles():
    assert not oracle.transform_one(W.Uniform(0.8, 1.5), 1, 1.6)["ok"]
    assert oracle.transform_one(W.Uniform(0.8, 1.5), 1, 1.2)["ok"]
    sp, psf = _b4_spec(); th = np.array(GOLD["B4"]["theta"])
    bad = []
    for i, v in ((0, -0.5), (1, 0.9), (7, -0.1), (8, 0.0), (3, float("nan")), (15, float("inf"))):
        t = th.copy(); t[i] = v
        if i == 1: t[2] = 0.6                        # |eps| >= 1
        bad.append(t)
    o = oracle.logpost_grad(sp, np.zeros((1, 6, 6)), np.full((1, 6, 6), 0.1), psf, np.array(bad + [th]))
    assert np.all(np.isneginf(o["logp"][:-1])) and np.isfinite(o["logp"][-1])
    assert np.all(o["grad"][:-1] == 0)


def test_batch_composition_invariance():
    """PAPER.md L83 fn 2: particles are independent -- a particle's result cannot depend on its batch."""
    wl = W.make_workload(1, n_particles=6)
    sp = wl.spec
    truth = oracle.model_image(sp, wl.psf.astype(np.float64), wl.truth_theta)
    obs, sig = W.finish_observation(wl, truth)
    z = wl.params.astype(np.float64)
    a = oracle.logpost_grad(sp, obs, sig, wl.psf, z)
    perm = np.array([4, 0, 5])
    b = oracle.logpost_grad(sp, obs, sig, wl.psf, z[perm])
    assert np.array_equal(a["logp"][perm], b["logp"]) and np.array_equal(a["grad"][perm], b["grad"])
    # at the truth, chi^2 ~ N^2
    t = oracle.logpost_grad(sp, obs, sig, wl.psf, wl.truth_z.astype(np.float64), want_model=True)
    chi2 = (((t["model"][0] - obs[0]) / sig[0]) ** 2).sum()
    assert abs(chi2 / sp.n_pix ** 2 - 1) < 0.15


# ------------------------------------------------------------------------------------------------ NEXT-4: detector-grid PSF
def test_bin_conv_detector_grid_pins():
    """psf_grid = 1 (bin, then convolve at the pixel scale): equals scipy's zero-padded convolution of the binned image;
    coincides with the ray-grid operator at s = 1; a delta PSF gives the plain binned image; a shifted delta moves the
    image by one DETECTOR pixel; flux of an interior source is conserved; the transpose is the adjoint."""
    from scipy.signal import convolve2d
    rng = np.random.default_rng(42)
    N, s, K, D = 9, 3, 5, 0.2
    ray = rng.random((N * s, N * s)); psf = rng.random((K, K)); psf /= psf.sum()
    binned = D * D * ray.reshape(N, s, N, s).mean(axis=(1, 3))
    got = oracle.bin_conv(N, s, K, D, psf, ray)
    assert np.allclose(got, convolve2d(binned, psf, mode="same"), rtol=1e-13, atol=1e-15)
    ray1 = rng.random((N, N))
    assert np.allclose(oracle.bin_conv(N, 1, K, D, psf, ray1), oracle.conv_bin(N, 1, K, D, psf, ray1), rtol=1e-13)
    delta = np.zeros((K, K)); delta[2, 2] = 1.0
    assert np.allclose(oracle.bin_conv(N, s, K, D, delta, ray), binned, rtol=1e-14)
    sh = np.zeros((K, K)); sh[3, 2] = 1.0                                  # tap (c+1, c): +1 row
    moved = oracle.bin_conv(N, s, K, D, sh, ray)
    assert np.allclose(moved[1:], binned[:-1], rtol=1e-14) and np.allclose(moved[0], 0.0)
    src = np.zeros_like(ray); src[12:15, 12:15] = rng.random((3, 3))       # interior: nothing leaves the cutout
    assert np.isclose(oracle.bin_conv(N, s, K, D, psf, src).sum(), D * D * src.sum() / (s * s), rtol=1e-13)
    g = rng.standard_normal((N, N))
    assert np.isclose((oracle.bin_conv(N, s, K, D, psf, ray) * g).sum(),
                      (oracle.bin_conv_transpose(N, s, K, D, psf, g) * ray).sum(), rtol=1e-12)


def test_detector_grid_gradient_vs_finite_differences():
    """Full log-posterior gradient with psf_grid = 1 against central differences (every parameter, tiny grid)."""
    import dataclasses
    sp = dataclasses.replace(W.make_spec(2), n_pix=8, supersample=2, psf_size=3, psf_grid=1)
    rng = np.random.default_rng(6)
    psf = W.gaussian_psf(3, 0.4, sp.pix_scale)[None]
    z = W.z_of(sp.priors, W.draw(rng, sp.priors, 2))
    obs = rng.random((1, 8, 8)); sig = np.full((1, 8, 8), 0.3)
    r = oracle.logpost_grad(sp, obs, sig, psf, z)
    for j in range(sp.n_params):
        h = 1e-6 * max(1.0, abs(z[0, j]))
        zp, zm = z.copy(), z.copy(); zp[:, j] += h; zm[:, j] -= h
        fd = (oracle.logpost_grad(sp, obs, sig, psf, zp, want_grad=False)["logp"] -
              oracle.logpost_grad(sp, obs, sig, psf, zm, want_grad=False)["logp"]) / (2 * h)
        assert np.allclose(fd, r["grad"][:, j], rtol=2e-5, atol=1e-6 * np.abs(r["grad"]).max()), j


# ------------------------------------------------------------------------------------------------ NEXT-4: model-dependent variance
def _noise_case(noise_model, t_exp):
    import dataclasses
    sp = dataclasses.replace(W.make_spec(2), n_pix=8, supersample=2, psf_size=3, noise_model=noise_model, t_exp=t_exp)
    rng = np.random.default_rng(16)
    psf = W.gaussian_psf(3, 0.4, sp.pix_scale / 2)[None]
    z = W.z_of(sp.priors, W.draw(rng, sp.priors, 3))
    obs = 0.5 * rng.random((1, 8, 8)); sig = np.full((1, 8, 8), 0.2) + 0.1 * rng.random((1, 8, 8))
    return sp, psf, z, obs, sig


def test_model_variance_likelihood_definition_and_limits():
    """noise_model = 1: logL equals the written-out definition on the oracle's own model image; t_exp -> infinity gives
    the fixed-sigma likelihood; and it differs visibly at a finite exposure."""
    sp, psf, z, obs, sig = _noise_case(1, 50.0)
    r = oracle.logpost_grad(sp, obs, sig, psf, z, want_grad=False, want_model=True)
    sp0 = __import__("dataclasses").replace(sp, noise_model=0)
    r0 = oracle.logpost_grad(sp0, obs, sig, psf, z, want_grad=False, want_model=True)
    assert np.allclose(r["model"], r0["model"], rtol=1e-14)
    m = r["model"]; v = sig ** 2 + np.maximum(m, 0) / 50.0
    logL = -0.5 * (((m - obs) ** 2 / v) + np.log(v)).sum(axis=(1, 2)) - 32 * np.log(2 * np.pi)
    logL0 = -0.5 * (((m - obs) / sig) ** 2).sum(axis=(1, 2)) - np.log(sig).sum() - 32 * np.log(2 * np.pi)
    assert np.allclose(r["logp"] - r0["logp"], logL - logL0, rtol=1e-10)
    assert np.all(np.abs(logL - logL0) > 1e-3 * np.abs(logL0))
    rinf = oracle.logpost_grad(__import__("dataclasses").replace(sp, t_exp=1e30), obs, sig, psf, z, want_grad=False)
    assert np.allclose(rinf["logp"], r0["logp"], rtol=1e-13)


def test_model_variance_gradient_vs_finite_differences():
    sp, psf, z, obs, sig = _noise_case(1, 50.0)
    r = oracle.logpost_grad(sp, obs, sig, psf, z)
    for j in range(sp.n_params):
        h = 1e-6 * max(1.0, abs(z[0, j]))
        zp, zm = z.copy(), z.copy(); zp[:, j] += h; zm[:, j] -= h
        fd = (oracle.logpost_grad(sp, obs, sig, psf, zp, want_grad=False)["logp"] -
              oracle.logpost_grad(sp, obs, sig, psf, zm, want_grad=False)["logp"]) / (2 * h)
        assert np.allclose(fd, r["grad"][:, j], rtol=2e-5, atol=1e-6 * np.abs(r["grad"]).max()), j
