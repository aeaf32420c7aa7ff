"""Pins of the backward-modelling oracle (oracle/linear.py, reading S21) against what the mathematics
fixes: exact recovery of the amplitudes of noise-free data, optimality of a* (the C oracle's own amplitude gradient
vanishes there and no other amplitude vector has a lower chi^2), the envelope-theorem gradient against finite
differences of the PROFILED log-posterior (each difference re-solves the amplitudes), and indifference to the
amplitude entries of z.  CPU only."""
import numpy as np
import pytest

import oracle
import oracle.linear as OL
import workloads as W


def _case(shapelet_nmax=-1, n_lens=1, seed=5, n_pix=14, s=2, K=5, noise=0.05):
    pri = W._default_priors(1, shapelet_nmax=shapelet_nmax, n_lens=n_lens)
    sp = W.LensSpec(n_pix, s, K, W._r32(0.11 * 40 / n_pix * 2.4), mass_model=1, epl_terms=30, shapelet_nmax=shapelet_nmax,
                    n_lens_sersic=n_lens, priors=pri)
    rng = np.random.default_rng(seed)
    step = sp.pix_scale / s
    psf = W.gaussian_psf(K, 2.5 * step, step)[None]
    th_true = W.draw(rng, pri, 1)
    truth = oracle.model_image(sp, psf, th_true)
    sigma = np.full((1, n_pix, n_pix), 0.05)
    obs = truth + noise * rng.standard_normal(truth.shape)
    return sp, obs, sigma, psf, th_true, rng


def test_amplitude_indices_follow_the_names():
    for nmax, nl in [(-1, 1), (2, 1), (3, 2), (-1, 0)]:
        sp = _case(nmax, nl)[0]
        names = W.param_names(1, 1, 0, 1, nmax, nl)
        want = [i for i, n in enumerate(names) if n.endswith(".I") or n.startswith("shp.a")]
        assert list(OL.amplitude_indices(sp)) == want


@pytest.mark.parametrize("nmax,nl", [(-1, 1), (2, 1), (1, 2)])
def test_noise_free_data_return_the_true_amplitudes(nmax, nl):
    """obs = model(theta_true) exactly: the least-squares amplitudes at the true non-linear parameters are the true
    amplitudes and chi^2 = 0 (closed form of the inversion)."""
    sp, obs, sigma, psf, th_true, _ = _case(nmax, nl, noise=0.0)
    amp = OL.amplitude_indices(sp)
    z = W.z_of(sp.priors, th_true)[0]
    z[amp] = -7.0                                                  # garbage: must be ignored
    a, M, b = OL.solve_amplitudes(sp, obs, sigma, psf, z)
    assert np.allclose(a, th_true[0, amp], rtol=1e-7, atol=1e-9)
    out = OL.logpost_grad(sp, obs, sigma, psf, z[None])
    N = sp.n_pix
    non_amp = np.setdiff1d(np.arange(sp.n_params), amp)
    lp_prior = sum(oracle.transform_one(sp.priors[i], 0, z[i])["lp"] + oracle.transform_one(sp.priors[i], 0, z[i])["logdet"]
                   for i in non_amp)
    want = -np.sum(np.log(sigma)) - 0.5 * N * N * np.log(2 * np.pi) + lp_prior          # chi^2 = 0
    assert abs(out["logp"][0] - want) < 1e-8 * abs(want)


def test_solution_is_the_minimum_and_stationary():
    sp, obs, sigma, psf, th_true, rng = _case(2, 1)
    amp = OL.amplitude_indices(sp)
    z = W.z_of(sp.priors, W.draw(rng, sp.priors, 3))
    out = OL.logpost_grad(sp, obs, sigma, psf, z)
    assert np.isfinite(out["logp"]).all()
    # the C oracle's own gradient with respect to the (untransformed) amplitudes vanishes at a*
    g_amp = out["grad_at_amp"]
    a, M, b = OL.solve_amplitudes(sp, obs, sigma, psf, z[0])
    scale = np.abs(b).max()
    assert np.abs(g_amp[0]).max() < 1e-8 * scale
    # any other amplitude vector has a lower log-posterior by exactly 1/2 da^T M da
    sb = OL.backward_spec(sp)
    for _ in range(4):
        da = rng.standard_normal(len(amp)) * 0.3
        z2 = z[0].copy(); z2[amp] = a + da
        lp2 = oracle.logpost_grad(sb, obs, sigma, psf, z2[None], want_grad=False)["logp"][0]
        assert lp2 < out["logp"][0]
        assert abs((out["logp"][0] - lp2) - 0.5 * da @ M @ da) < 1e-7 * abs(0.5 * da @ M @ da)


def test_gradient_is_the_derivative_of_the_profiled_posterior():
    """Central differences of z -> log p~_B(z), re-solving a* at every displaced point, against the envelope gradient."""
    sp, obs, sigma, psf, th_true, rng = _case(1, 1, seed=9)
    amp = OL.amplitude_indices(sp)
    z = W.z_of(sp.priors, W.draw(rng, sp.priors, 1))[0]
    out = OL.logpost_grad(sp, obs, sigma, psf, z[None])
    g = out["grad"][0]
    assert np.all(g[amp] == 0)
    for i in np.setdiff1d(np.arange(sp.n_params), amp):
        h = 1e-5
        zp, zm = z.copy(), z.copy(); zp[i] += h; zm[i] -= h
        fp = OL.logpost_grad(sp, obs, sigma, psf, zp[None], want_grad=False)["logp"][0]
        fm = OL.logpost_grad(sp, obs, sigma, psf, zm[None], want_grad=False)["logp"][0]
        fd = (fp - fm) / (2 * h)
        assert abs(fd - g[i]) <= 2e-5 * max(abs(g[i]), 1.0) + 1e-6 * np.abs(g).max(), (i, fd, g[i])


def test_amplitude_entries_of_z_are_ignored_and_invalid_rows_flagged():
    sp, obs, sigma, psf, th_true, rng = _case(-1, 1)
    amp = OL.amplitude_indices(sp)
    z = W.z_of(sp.priors, W.draw(rng, sp.priors, 2))
    z2 = z.copy(); z2[:, amp] = rng.standard_normal((2, len(amp))) * 50
    a = OL.logpost_grad(sp, obs, sigma, psf, z); b = OL.logpost_grad(sp, obs, sigma, psf, z2)
    assert np.array_equal(a["logp"], b["logp"]) and np.array_equal(a["grad"], b["grad"])
    z3 = z.copy(); z3[0, 0] = np.nan
    c = OL.logpost_grad(sp, obs, sigma, psf, z3)
    assert c["logp"][0] == -np.inf and np.all(c["grad"][0] == 0) and np.isfinite(c["logp"][1])
