"""GPU parity of backward amplitude modelling (amplitude_mode 1, reading S21) against
oracle/linear.py: solved amplitudes, log-posterior at them and the envelope gradient, strict north_star bar in fp64
mode; the amplitude entries of params are ignored (NaN included) and their gradient entries are exactly zero."""
import copy

import numpy as np
import pytest

import workloads as W

pytestmark = pytest.mark.gpu

RTOL_LOGP = 1e-4


def _gl():
    import paper_2606_30633_b200 as gl
    return gl


def _case(n_pix, s, K, shapelet_nmax, n_lens, seed, n_particles, mass_model=1, multipoles=False):
    import oracle
    pri = W._default_priors(mass_model, multipoles=multipoles, shapelet_nmax=shapelet_nmax, n_lens=n_lens)
    sp = W.LensSpec(n_pix, s, K, W._r32(0.11 * 40 / n_pix * 2.4), mass_model=mass_model, epl_terms=30,
                    multipole_mask=3 if multipoles else 0, shapelet_nmax=shapelet_nmax, n_lens_sersic=n_lens, priors=pri,
                    amplitude_mode=1)
    rng = np.random.default_rng(seed)
    step = sp.pix_scale / s
    psf = W.gaussian_psf(K, 2.5 * step, step)[None].astype(np.float32)
    th_true = W.draw(rng, pri, 1)
    truth = oracle.model_image(sp, psf.astype(np.float64), th_true)
    sigma = np.full((1, n_pix, n_pix), 0.05, np.float32)
    obs = (truth + 0.05 * rng.standard_normal(truth.shape)).astype(np.float32)
    z = W.z_of(pri, W.draw(rng, pri, n_particles)).astype(np.float32)
    return sp, obs, sigma, psf, z


def _grad_ok(g, ref):
    tol = np.maximum(1e-3 * np.abs(ref), 1e-5)
    return np.abs(g - ref) <= tol


@pytest.mark.parametrize("shape", [(40, 2, 11, -1, 1), (24, 2, 5, 3, 1), (20, 3, 7, 2, 2), (16, 1, 5, -1, 0), (22, 2, 5, 7, 1)])
def test_backward_mode_matches_oracle(shape):
    import oracle.linear as OL
    import torch
    gl = _gl()
    n_pix, s, K, nmax, nl = shape
    sp, obs, sigma, psf, z = _case(n_pix, s, K, nmax, nl, seed=11 + n_pix, n_particles=6, multipoles=(nmax == 7))
    amp_idx = OL.amplitude_indices(sp)
    z[:, amp_idx] = np.float32(np.nan)                                   # ignored by contract
    z[1, amp_idx] = 3.0
    ref = OL.logpost_grad(sp, obs, sigma, psf, z.astype(np.float64))
    m = gl.LensModel(sp, obs, sigma, psf)
    assert gl.gl_config_n_amplitudes(m.h) == len(amp_idx)
    zt = torch.from_numpy(z).cuda()
    lp, g = m.logpost_grad(zt)
    amp, lp2 = m.linear_amplitudes(zt)
    lp0 = m.logpost(zt)
    lp, g, amp = lp.cpu().numpy().astype(np.float64), g.cpu().numpy().astype(np.float64), amp.cpu().numpy().astype(np.float64)
    assert np.array_equal(lp2.cpu().numpy(), lp0.cpu().numpy())
    fin = np.isfinite(ref["logp"])
    assert fin.sum() >= 4 and np.array_equal(np.isfinite(lp), fin)
    assert np.all(np.abs(lp[fin] - ref["logp"][fin]) <= RTOL_LOGP * np.abs(ref["logp"][fin]))
    assert np.all(np.abs(lp0.cpu().numpy()[fin] - ref["logp"][fin]) <= RTOL_LOGP * np.abs(ref["logp"][fin]))
    assert np.all(g[:, amp_idx] == 0)
    ok = _grad_ok(g[fin], ref["grad"][fin])
    assert ok.all(), (np.argwhere(~ok)[:5], g[fin][~ok][:5], ref["grad"][fin][~ok][:5])
    scale = np.abs(ref["amp"][fin]).max(axis=1, keepdims=True)
    assert np.all(np.abs(amp[fin] - ref["amp"][fin]) <= 1e-4 * scale + 1e-6)


def test_backward_mode_fp32_and_multi_system():
    """fp32 arithmetic mode: norm-wise agreement; two systems with a gather map: each particle is inverted against
    its own obs / sigma / PSF."""
    import oracle.linear as OL
    import torch
    gl = _gl()
    sp, obs, sigma, psf, z = _case(24, 2, 5, -1, 1, seed=3, n_particles=8)
    sp2 = copy.copy(sp); sp2.n_systems = 2
    rng = np.random.default_rng(0)
    obs2 = np.concatenate([obs, obs[:, ::-1].copy() * 0.7]); sig2 = np.concatenate([sigma, sigma * 1.5])
    psf2 = np.concatenate([psf, W.gaussian_psf(5, 3.5 * sp.pix_scale / 2, sp.pix_scale / 2)[None].astype(np.float32)])
    sid = np.array([0, 1, 1, 0, 1, 0, 0, 1], dtype=np.int32)
    ref = OL.logpost_grad(sp2, obs2, sig2, psf2, z.astype(np.float64), system_id=sid)
    for prec, tol in [(0, 1e-5), (1, 2e-2)]:
        spp = copy.copy(sp2); spp.precision = prec
        m = gl.LensModel(spp, obs2, sig2, psf2)
        lp, g = m.logpost_grad(torch.from_numpy(z).cuda(), system_id=sid)
        lp, g = lp.cpu().numpy().astype(np.float64), g.cpu().numpy().astype(np.float64)
        fin = np.isfinite(ref["logp"])
        assert np.array_equal(np.isfinite(lp), fin)
        assert np.all(np.abs(lp[fin] - ref["logp"][fin]) <= (1e-4 if prec == 0 else 1e-3) * np.abs(ref["logp"][fin]))
        num = np.linalg.norm(g[fin] - ref["grad"][fin], axis=1); den = np.linalg.norm(ref["grad"][fin], axis=1)
        assert np.all(num <= tol * den), (prec, num / den)


def test_backward_mode_config_errors_and_model_image():
    import torch
    gl = _gl()
    sp, obs, sigma, psf, z = _case(16, 2, 5, -1, 1, seed=2, n_particles=3)
    bad = copy.copy(sp); bad.noise_model = 1; bad.t_exp = 100.0
    with pytest.raises(gl.GLError):
        gl.gl_config_create(bad)
    fwd = copy.copy(sp); fwd.amplitude_mode = 0
    m0 = gl.LensModel(fwd, obs, sigma, psf)
    with pytest.raises(gl.GLError):
        m0.linear_amplitudes(torch.from_numpy(z).cuda())
    # gl_model_image in backward mode: the amplitude entries are the amplitudes -> image at a* has the solved chi^2
    m = gl.LensModel(sp, obs, sigma, psf)
    zt = torch.from_numpy(z).cuda()
    amp, lp = m.linear_amplitudes(zt)
    import oracle.linear as OL
    idx = OL.amplitude_indices(sp)
    z2 = zt.clone(); z2[:, torch.as_tensor(idx).cuda()] = amp
    img = m.model_image(z2).cpu().numpy().astype(np.float64)
    ref = OL.logpost_grad(sp, obs, sigma, psf, z.astype(np.float64), want_grad=False)
    import oracle
    sb = OL.backward_spec(sp)
    rows = z.astype(np.float64).copy(); rows[:, idx] = ref["amp"]
    theta = np.array([[oracle.transform_one(sb.priors[i], 0, v)["theta"] for i, v in enumerate(r)] for r in rows])
    ref_img = oracle.model_image(sb, psf.astype(np.float64), theta)
    assert np.allclose(img, ref_img, rtol=2e-4, atol=2e-4 * np.abs(ref_img).max())


def test_map_run_in_backward_mode_recovers_the_truth():
    """The MAP consumer on a backward-mode model (config-1 shape): the amplitude entries of z never move (zero
    gradient), every start improves, the best start reaches the truth's profiled log-posterior, and its solved
    amplitudes come out close to the amplitudes the observation was rendered with."""
    import copy as _copy
    import torch
    import oracle.linear as OL
    from _cases import observation
    gl = _gl()
    wl, obs, sig = observation(1)
    sp = _copy.copy(wl.spec); sp.amplitude_mode = 1
    idx = OL.amplitude_indices(sp)
    rng = np.random.default_rng(8)
    z0 = (wl.truth_z[0][None, :] + 0.05 * rng.standard_normal((32, sp.n_params))).astype(np.float32)
    z0[:, idx] = 123.0
    m = gl.LensModel(sp, obs, sig, wl.psf)
    lp_truth = float(m.logpost(torch.from_numpy(wl.truth_z[:1]).cuda())[0])
    z = torch.from_numpy(z0).cuda()
    lp0 = m.logpost(z).clone()
    m.map_run(z, dict(kind=0, lr=2e-3, b1=0.9, b2=0.999, eps=1e-8, eps_root=0.0), 300)
    lp1 = m.logpost(z)
    amp, _ = m.linear_amplitudes(z)
    torch.cuda.synchronize()
    assert torch.all(z[:, torch.as_tensor(idx).cuda()] == 123.0)
    assert torch.all(lp1 > lp0)
    assert float(lp1.max()) >= lp_truth - 25.0, (float(lp1.max()), lp_truth)
    best = int(torch.argmax(lp1))
    th_true = W.theta_of(wl.spec.priors, wl.truth_z[:1].astype(np.float64))[0]
    a_true = th_true[idx]
    assert np.all(np.abs(amp[best].cpu().numpy() - a_true) <= 0.2 * np.abs(a_true)), (amp[best], a_true)


def test_backward_mode_full_config2_batch_chunks_and_oracle_samples():
    """Config 2 in backward mode, the full batch of 4096 particles three times over (12288 rows: more than one chunk of
    the 16 GiB backward-mode workspace budget): every row is bit-identical to the same particle evaluated in a
    single-chunk call, and sampled rows of all three thirds meet the strict bar against the oracle."""
    import copy as _copy
    import torch
    import oracle.linear as OL
    from _cases import observation
    gl = _gl()
    wl, obs, sig = observation(2)
    sp = _copy.copy(wl.spec); sp.amplitude_mode = 1
    m = gl.LensModel(sp, obs, sig, wl.psf)
    z1 = torch.from_numpy(wl.params).cuda()
    P1 = z1.shape[0]
    z = torch.cat([z1, z1, z1]).contiguous()
    P = z.shape[0]
    assert gl.gl_workspace_bytes(m.h, P) < gl.gl_workspace_bytes(m.h, 1) * P * 0.8, "the batch should need several chunks"
    assert gl.gl_workspace_bytes(m.h, P1) > gl.gl_workspace_bytes(m.h, 1) * P1 * 0.8, "one third should fit one chunk"
    lp, g = m.logpost_grad(z)
    amp, _ = m.linear_amplitudes(z)
    lp1, g1 = m.logpost_grad(z1)
    assert float(torch.isfinite(lp).float().mean()) > 0.99
    for k in range(3):
        assert torch.equal(lp[k * P1:(k + 1) * P1], lp1) and torch.equal(g[k * P1:(k + 1) * P1], g1)
    lp, g, amp = lp.cpu().numpy(), g.cpu().numpy(), amp.cpu().numpy()
    idx = np.array([3, 1999, 4095, 4096 + 2345, 2 * 4096 + 2346, 3 * 4096 - 1])
    ref = OL.logpost_grad(sp, obs, sig, wl.psf, wl.params[idx % P1].astype(np.float64))
    assert np.isfinite(ref["logp"]).all()
    assert np.all(np.abs(lp[idx] - ref["logp"]) <= RTOL_LOGP * np.abs(ref["logp"]))
    assert _grad_ok(g[idx].astype(np.float64), ref["grad"]).all()
    assert np.all(np.abs(amp[idx] - ref["amp"]) <= 1e-4 * np.abs(ref["amp"]).max(axis=1, keepdims=True) + 1e-6)


def _multi_case(n_pix, s, K, seed, n_particles, nmax=-1, multipoles=False, mass_model=1, amplitude_mode=0):
    """Two sources on the source plane and three lens-plane Sersic blocks: the component list of the paper's
    real-system model (env, L1, L2, S1, S2)."""
    import oracle
    pri = W._default_priors(mass_model, multipoles=multipoles, shapelet_nmax=nmax, n_lens=3, n_src=2)
    sp = W.LensSpec(n_pix, s, K, W._r32(0.11 * 40 / n_pix * 2.4), mass_model=mass_model, epl_terms=30,
                    multipole_mask=3 if multipoles else 0, n_source_sersic=2, shapelet_nmax=nmax, n_lens_sersic=3,
                    priors=pri, amplitude_mode=amplitude_mode)
    assert sp.n_params == len(W.param_names(mass_model, 1, sp.multipole_mask, 2, nmax, 3))
    rng = np.random.default_rng(seed)
    step = sp.pix_scale / s
    psf = W.gaussian_psf(K, 2.5 * step, step)[None].astype(np.float32)
    truth = oracle.model_image(sp, psf.astype(np.float64), W.draw(rng, pri, 1))
    sigma = np.full((1, n_pix, n_pix), 0.05, np.float32)
    obs = (truth + 0.05 * rng.standard_normal(truth.shape)).astype(np.float32)
    z = W.z_of(pri, W.draw(rng, pri, n_particles)).astype(np.float32)
    return sp, obs, sigma, psf, z


@pytest.mark.parametrize("case", [(40, 2, 11, -1, False, 1), (20, 2, 5, -1, False, 0), (18, 3, 5, 3, True, 1), (16, 2, 5, 8, False, 0)])
def test_two_sources_three_lens_blocks_sampled_amplitudes(case):
    """Sampled ("forward") amplitudes, strict north_star bar in fp64 mode; fp32 mode norm-wise.  Kernel variants
    <.,0,2,-1,3> (the 43-parameter real-system list) and the superset <.,3,2,10,3>."""
    import copy as _copy
    import oracle
    import torch
    gl = _gl()
    n_pix, s, K, nmax, mp, mass = case
    sp, obs, sigma, psf, z = _multi_case(n_pix, s, K, seed=50 + n_pix, n_particles=6, nmax=nmax, multipoles=mp, mass_model=mass)
    ref = oracle.logpost_grad(sp, obs, sigma, psf, z.astype(np.float64), epl_terms=30 if mass == 1 else None)
    fin = np.isfinite(ref["logp"])
    assert fin.sum() >= 4
    for prec in (0, 1):
        spp = _copy.copy(sp); spp.precision = prec
        m = gl.LensModel(spp, obs, sigma, psf)
        lp, g = m.logpost_grad(torch.from_numpy(z).cuda())
        lp, g = lp.cpu().numpy().astype(np.float64), g.cpu().numpy().astype(np.float64)
        assert np.array_equal(np.isfinite(lp), fin)
        if prec == 0:
            assert np.all(np.abs(lp[fin] - ref["logp"][fin]) <= RTOL_LOGP * np.abs(ref["logp"][fin]))
            ok = _grad_ok(g[fin], ref["grad"][fin])
            assert ok.all(), (np.argwhere(~ok)[:5], g[fin][~ok][:5], ref["grad"][fin][~ok][:5])
        else:
            num = np.linalg.norm(g[fin] - ref["grad"][fin], axis=1); den = np.linalg.norm(ref["grad"][fin], axis=1)
            assert np.all(num <= 2e-2 * den), num / den
        img = m.model_image(torch.from_numpy(z[fin][:2]).cuda()).cpu().numpy()
        ref_img = oracle.model_image(sp, psf.astype(np.float64), W.theta_of(sp.priors, z[fin][:2].astype(np.float64)),
                                     epl_terms=30 if mass == 1 else None)
        assert np.allclose(img, ref_img, rtol=1e-3, atol=1e-4 * np.abs(ref_img).max())


@pytest.mark.parametrize("case", [(40, 2, 11, -1, False), (18, 2, 5, 2, True)])
def test_real_system_component_list_in_backward_mode(case):
    """The paper's real-system configuration: backward modelling of mass + shear, three lens-plane
    Sersic blocks and two sources -- 38 sampled parameters + 5 solved amplitudes -- against oracle/linear.py."""
    import oracle.linear as OL
    import torch
    gl = _gl()
    n_pix, s, K, nmax, mp = case
    sp, obs, sigma, psf, z = _multi_case(n_pix, s, K, seed=77, n_particles=6, nmax=nmax, multipoles=mp, amplitude_mode=1)
    idx = OL.amplitude_indices(sp)
    if nmax < 0:
        assert sp.n_params - len(idx) == 38 and len(idx) == 5
    z[:, idx] = np.float32(np.nan)
    ref = OL.logpost_grad(sp, obs, sigma, psf, z.astype(np.float64), epl_terms=30)
    m = gl.LensModel(sp, obs, sigma, psf)
    assert gl.gl_config_n_amplitudes(m.h) == len(idx)
    lp, g = m.logpost_grad(torch.from_numpy(z).cuda())
    amp, _ = m.linear_amplitudes(torch.from_numpy(z).cuda())
    lp, g, amp = lp.cpu().numpy().astype(np.float64), g.cpu().numpy().astype(np.float64), amp.cpu().numpy().astype(np.float64)
    fin = np.isfinite(ref["logp"])
    assert fin.sum() >= 4 and np.array_equal(np.isfinite(lp), fin)
    assert np.all(np.abs(lp[fin] - ref["logp"][fin]) <= RTOL_LOGP * np.abs(ref["logp"][fin]))
    assert np.all(g[:, idx] == 0)
    ok = _grad_ok(g[fin], ref["grad"][fin])
    assert ok.all(), (np.argwhere(~ok)[:5], g[fin][~ok][:5], ref["grad"][fin][~ok][:5])
    scale = np.abs(ref["amp"][fin]).max(axis=1, keepdims=True)
    assert np.all(np.abs(amp[fin] - ref["amp"][fin]) <= 1e-4 * scale + 1e-6)


def test_hmc_transition_in_backward_mode_matches_oracle():
    """The HMC consumer on a backward-mode model: one transition (3 leapfrog steps, identity mass matrix) of 12 chains
    near the config-1 truth against oracle/optim.py driven by oracle/linear.py: energy differences, accept decisions,
    positions and the cached log-posterior / gradient.  The amplitude coordinates feel no force (zero gradient)."""
    import copy as _copy
    import torch
    import oracle.linear as OL
    from oracle import optim
    from _cases import observation
    gl = _gl()
    wl, obs, sig = observation(1)
    sp = _copy.copy(wl.spec); sp.amplitude_mode = 1
    n = sp.n_params
    idx = OL.amplitude_indices(sp)
    rng = np.random.default_rng(41)
    z0 = (wl.truth_z[0][None, :] + 0.01 * rng.standard_normal((12, n))).astype(np.float32)
    xi = rng.standard_normal((12, n)).astype(np.float32)
    log_u = np.log(rng.random(12)).astype(np.float32)
    eps = 2e-5                                                          # stable for gradients of 1e5 (identity mass matrix)
    m = gl.LensModel(sp, obs, sig, wl.psf)
    d = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    zg = d(z0)
    lpg, gg = m.logpost_grad(zg)
    acc = torch.zeros(12, dtype=torch.int32, device="cuda"); dh = torch.zeros(12, device="cuda")
    ws = torch.empty(gl.gl_hmc_workspace_bytes(m.h, 12), dtype=torch.uint8, device="cuda")

    def f(z):
        r = OL.logpost_grad(sp, obs, sig, wl.psf, z.astype(np.float32).astype(np.float64))
        return r["logp"], np.where(np.isfinite(r["logp"])[:, None], r["grad"], 0.0)

    prev = [x.cpu().numpy().astype(np.float64) for x in (zg, lpg, gg)]
    z_o, lp_o, g_o, acc_o, dh_o = optim.hmc_transition(f, prev[0], prev[1], prev[2], optim.tril_pack(np.eye(n)),
                                                       xi.astype(np.float64), log_u.astype(np.float64),
                                                       float(np.float32(eps)), 3)
    gl.gl_hmc_step(m.h, m.obs, m.noise_sigma, m.psf, zg, lpg, gg, None, d(xi), d(log_u), None, eps, 3, acc, dh, ws)
    torch.cuda.synchronize()
    dh_g = dh.cpu().numpy().astype(np.float64); acc_g = acc.cpu().numpy().astype(bool)
    assert np.isfinite(dh_o).all() and np.isfinite(dh_g).all()
    assert np.all(np.abs(dh_g - dh_o) <= 1e-4 * np.abs(prev[1]) + 1e-6), np.max(np.abs(dh_g - dh_o))
    decided = np.abs(log_u.astype(np.float64) - dh_o) > 1e-3
    assert decided.sum() >= 9 and np.array_equal(acc_g[decided], acc_o[decided])
    same = acc_g == acc_o
    zz = zg.cpu().numpy().astype(np.float64)
    assert np.all(np.abs(zz[same] - z_o[same]) <= 2e-7 * np.abs(z_o[same]) + 1e-9)
    gn = gg.cpu().numpy().astype(np.float64)
    assert np.all(gn[:, idx] == 0)
    assert np.all(np.abs(gn[same] - g_o[same]) <= np.maximum(1e-3 * np.abs(g_o[same]), 1e-5))
    # the force-free amplitude coordinates of an accepted chain moved by exactly n_leapfrog * eps * xi
    a = same & acc_g
    assert a.any()
    want = z0[a][:, idx].astype(np.float64) + 3 * float(np.float32(eps)) * xi[a][:, idx].astype(np.float64)
    assert np.all(np.abs(zz[a][:, idx] - want) <= 4e-7 * np.abs(want) + 1e-7)
