"""the fused SVI iteration (gl_svi_step) against the SVI oracle (oracle/optim.py on top of the fp64
forward/gradient oracle)."""
import numpy as np
import pytest

from _cases import observation

pytestmark = pytest.mark.gpu

ADABELIEF = dict(kind=1, lr=1e-4, b1=0.95, b2=0.99, eps=1e-16, eps_root=1e-16)
ADAM = dict(kind=0, lr=1e-3, b1=0.9, b2=0.999, eps=1e-8, eps_root=0.0)


def _setup(k, n_draws, seed):
    import torch
    import paper_2606_30633_b200 as gl
    wl, obs, sig = observation(k)
    n = wl.spec.n_params
    rng = np.random.default_rng(seed)
    mu = wl.truth_z[0].astype(np.float32).copy()
    L = np.tril(0.002 * rng.standard_normal((n, n))) + np.diag(0.01 + 0.01 * rng.random(n))
    lt = L[np.tril_indices(n)].astype(np.float32)
    xi = rng.standard_normal((n_draws, n)).astype(np.float32)
    m = gl.LensModel(wl.spec, obs, sig, wl.psf)
    return gl, torch, wl, obs, sig, m, mu, lt, xi


@pytest.mark.parametrize("opt", [ADABELIEF, ADAM], ids=["adabelief", "adam"])
def test_svi_steps_match_oracle(opt):
    """Two consecutive iterations, 48 draws around the seeded truth of config 1 (one draw made invalid through an
    extreme xi): loss, mu, L and both state arrays follow the oracle."""
    import oracle
    from oracle import optim
    gl, torch, wl, obs, sig, m, mu, lt, xi = _setup(1, 48, 11)
    xi[7, 2] = 4.0e3                                                    # e1 far outside the unit disc: invalid draw
    n = wl.spec.n_params; nt = n * (n + 1) // 2
    opt_o = {k: (float(np.float32(x)) if k != "kind" else x) for k, x in opt.items()}
    d = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    mu_g, lt_g, xi_g = d(mu), d(lt), d(xi)
    mm, vv = torch.zeros(n + nt, device="cuda"), torch.zeros(n + nt, device="cuda")
    stats = torch.zeros(2, device="cuda")
    ws = torch.empty(gl.gl_svi_workspace_bytes(m.h, 48), dtype=torch.uint8, device="cuda")

    def f(z):
        r = oracle.logpost_grad(wl.spec, obs, sig, wl.psf, z.astype(np.float32).astype(np.float64), None)
        return r["logp"], r["grad"]

    for t in (1, 2):
        prev = [x.cpu().numpy().astype(np.float64) for x in (mu_g, lt_g, mm, vv)]
        loss_o, mu_o, lt_o, m_o, v_o, lp_o = optim.svi_step(f, prev[0], prev[1], xi.astype(np.float64), prev[2], prev[3], t, opt_o)
        gl.gl_svi_step(m.h, opt, m.obs, m.noise_sigma, m.psf, mu_g, lt_g, xi_g, None, mm, vv, t, stats, ws)
        torch.cuda.synchronize()
        assert int(stats[1]) == 47 == int(np.isfinite(lp_o).sum())
        assert abs(float(stats[0]) - loss_o) <= 1e-4 * abs(loss_o)
        th_prev = np.concatenate(prev[:2]); th_o = np.concatenate([mu_o, lt_o])
        th_g = np.concatenate([mu_g.cpu().numpy(), lt_g.cpu().numpy()]).astype(np.float64)
        # gradient sums of 47 draws cancel, and the draws themselves are stored in fp32 (the oracle evaluates the
        # fp32-rounded draws too): bar = the north_star gradient bar (1e-3) on the step, fp32 storage on the rest
        for got, want, old, c, name in ((th_g, th_o, th_prev, 1.0, "theta"), (mm.cpu().numpy().astype(np.float64), m_o, prev[2], opt_o["b1"], "m"),
                                        (vv.cpu().numpy().astype(np.float64), v_o, prev[3], opt_o["b2"], "v")):
            scale = np.abs(c * old) + np.abs(want - c * old)
            assert np.all(np.abs(got - want) <= 2e-3 * np.abs(want - c * old) + 4e-7 * scale + 1e-30), (name, t)
    assert gl.gl_last_launch_count() == 10                              # draw + 7 path kernels + reduce + update


def test_svi_loss_decreases_on_config1():
    """150 AdaBelief iterations (fresh draws each) from a surrogate centred 0.03 away from the truth: the loss estimate
    falls and the mean moves toward the posterior mode region (smoke test; P:L118 shows the paper's loss curves)."""
    gl, torch, wl, obs, sig, m, mu, lt, xi = _setup(1, 256, 21)
    n = wl.spec.n_params; nt = n * (n + 1) // 2
    rng = np.random.default_rng(22)
    mu0 = (mu + 0.03 * rng.standard_normal(n)).astype(np.float32)
    mu_g = torch.from_numpy(mu0).cuda(); lt_g = torch.from_numpy(lt).cuda()
    mm, vv = torch.zeros(n + nt, device="cuda"), torch.zeros(n + nt, device="cuda")
    stats = torch.zeros(2, device="cuda")
    ws = torch.empty(gl.gl_svi_workspace_bytes(m.h, 256), dtype=torch.uint8, device="cuda")
    gen = torch.Generator(device="cuda"); gen.manual_seed(5)
    losses = []
    opt = dict(ADABELIEF, lr=2e-3)
    for t in range(1, 151):
        x = torch.randn((256, n), device="cuda", generator=gen)
        gl.gl_svi_step(m.h, opt, m.obs, m.noise_sigma, m.psf, mu_g, lt_g, x, None, mm, vv, t, stats, ws)
        if t in (1, 150):
            losses.append(float(stats[0]))
    assert np.isfinite(losses).all() and losses[1] < losses[0], losses
    assert torch.all(torch.isfinite(mu_g)) and torch.all(torch.isfinite(lt_g))


def test_svi_argument_checks():
    gl, torch, wl, obs, sig, m, mu, lt, xi = _setup(1, 8, 1)
    n = wl.spec.n_params; nt = n * (n + 1) // 2
    d = lambda a: torch.from_numpy(a).cuda()
    mm, vv, stats = torch.zeros(n + nt, device="cuda"), torch.zeros(n + nt, device="cuda"), torch.zeros(2, device="cuda")
    small = torch.empty(256, dtype=torch.uint8, device="cuda")
    with pytest.raises(gl.GLError) as e:
        gl.gl_svi_step(m.h, ADAM, m.obs, m.noise_sigma, m.psf, d(mu), d(lt), d(xi), None, mm, vv, 1, stats, small)
    assert e.value.status == -5
    ws = torch.empty(gl.gl_svi_workspace_bytes(m.h, 8), dtype=torch.uint8, device="cuda")
    with pytest.raises(gl.GLError) as e:
        gl.gl_svi_step(m.h, dict(ADAM, b2=1.5), m.obs, m.noise_sigma, m.psf, d(mu), d(lt), d(xi), None, mm, vv, 1, stats, ws)
    assert e.value.status == -2


def _big_setup(n_draws, seed, amplitude_mode=0):
    """The config-3 parameter layout (EPL + shear, Sersic + shapelets n_max = 6, two lens Sersics: 58 parameters) on a
    16x16, s = 2, K = 5 geometry, so that the oracle evaluates EVERY draw in seconds; dense L."""
    import dataclasses
    import torch
    import paper_2606_30633_b200 as gl
    from _cases import small_case
    sp, obs, sig, psf, z, truth_z = small_case(16, 2, 5, 1, 0, 6, 2, seed=seed, n_particles=2, with_truth=True)
    sp = dataclasses.replace(sp, amplitude_mode=amplitude_mode)
    n = sp.n_params
    assert n == 58
    rng = np.random.default_rng(seed + 1)
    L = np.tril(0.001 * rng.standard_normal((n, n))) + np.diag(0.004 + 0.004 * rng.random(n))
    lt = L[np.tril_indices(n)].astype(np.float32)
    xi = rng.standard_normal((n_draws, n)).astype(np.float32)
    m = gl.LensModel(sp, obs, sig, psf)
    return gl, torch, sp, obs, sig, psf, m, truth_z.astype(np.float32).copy(), lt, xi


@pytest.mark.parametrize("opt", [ADABELIEF, ADAM], ids=["adabelief", "adam"])
def test_svi_step_58_params_2048_draws(opt):
    """gl_svi_reduce_kernel's 32-chunk two-level sums, tril_row and the update over 58 + 1711 surrogate parameters:
    two iterations of 2048 draws (3 of them thrown out of the model's domain) on the config-3 layout, the oracle
    evaluating every draw; loss, mu, L and the optimiser state against oracle/optim.py."""
    import oracle
    from oracle import optim
    gl, torch, sp, obs, sig, psf, m, mu, lt, xi = _big_setup(2048, 303)
    for r in (5, 700, 2047):
        xi[r, 2] = 5.0e4                                                # mass e1 far outside the unit disc
    n = sp.n_params; nt = n * (n + 1) // 2
    opt_o = {k: (float(np.float32(x)) if k != "kind" else x) for k, x in opt.items()}
    d = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    mu_g, lt_g, xi_g = d(mu), d(lt), d(xi)
    mm, vv = torch.zeros(n + nt, device="cuda"), torch.zeros(n + nt, device="cuda")
    stats = torch.zeros(2, device="cuda")
    ws = torch.empty(gl.gl_svi_workspace_bytes(m.h, 2048), dtype=torch.uint8, device="cuda")

    def f(z):
        r = oracle.logpost_grad(sp, obs, sig, psf, z.astype(np.float32).astype(np.float64), None)
        return r["logp"], r["grad"]

    for t in (1, 2):
        prev = [x.cpu().numpy().astype(np.float64) for x in (mu_g, lt_g, mm, vv)]
        loss_o, mu_o, lt_o, m_o, v_o, lp_o = optim.svi_step(f, prev[0], prev[1], xi.astype(np.float64), prev[2], prev[3], t, opt_o)
        gl.gl_svi_step(m.h, opt, m.obs, m.noise_sigma, m.psf, mu_g, lt_g, xi_g, None, mm, vv, t, stats, ws)
        torch.cuda.synchronize()
        assert int(stats[1]) == int(np.isfinite(lp_o).sum()) == 2045
        assert abs(float(stats[0]) - loss_o) <= 1e-4 * abs(loss_o)
        th_prev = np.concatenate(prev[:2]); th_o = np.concatenate([mu_o, lt_o])
        th_g = np.concatenate([mu_g.cpu().numpy(), lt_g.cpu().numpy()]).astype(np.float64)
        for got, want, old, c, name in ((th_g, th_o, th_prev, 1.0, "theta"), (mm.cpu().numpy().astype(np.float64), m_o, prev[2], opt_o["b1"], "m"),
                                        (vv.cpu().numpy().astype(np.float64), v_o, prev[3], opt_o["b2"], "v")):
            scale = np.abs(c * old) + np.abs(want - c * old)
            bad = np.abs(got - want) > 2e-3 * np.abs(want - c * old) + 4e-7 * scale + 1e-30
            assert not bad.any(), (name, t, int(bad.sum()), np.flatnonzero(bad)[:8])


def test_svi_backward_mode_surrogate_lives_on_the_sampled_dimensions():
    """amplitude_mode 1 (the combination of the paper's real-system run): the solved amplitudes have zero
    gradient, so their mu_j, the rows and columns j of L and their optimiser state must not move and log L_jj must stay out of
    the loss; everything else follows oracle/optim.py (active mask, pinned in tests/test_oracle_optim.py) on top of
    oracle/linear.py.  Three iterations; the loss must not drift downwards through the dead dimensions."""
    import oracle.linear as OL
    from oracle import optim
    gl, torch, sp, obs, sig, psf, m, mu, lt, xi = _big_setup(96, 411, amplitude_mode=1)
    n = sp.n_params; nt = n * (n + 1) // 2
    amp = np.asarray(OL.amplitude_indices(sp)); act = np.ones(n, bool); act[amp] = False
    assert (~act).sum() == 31
    opt = dict(ADAM, lr=2e-4)
    opt_o = {k: (float(np.float32(x)) if k != "kind" else x) for k, x in opt.items()}
    d = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    mu_g, lt_g = d(mu), d(lt)
    mm, vv = torch.zeros(n + nt, device="cuda"), torch.zeros(n + nt, device="cuda")
    stats = torch.zeros(2, device="cuda")
    ws = torch.empty(gl.gl_svi_workspace_bytes(m.h, 96), dtype=torch.uint8, device="cuda")

    def f(z):
        r = OL.logpost_grad(sp, obs, sig, psf, z.astype(np.float32).astype(np.float64))
        return r["logp"], r["grad"]

    live = np.concatenate([act, optim.tril_pack(act[:, None] & act[None, :]).astype(bool)])
    th0 = np.concatenate([mu, lt]).astype(np.float64)
    rng = np.random.default_rng(5)
    losses = []
    for t in (1, 2, 3):
        x = rng.standard_normal((96, n)).astype(np.float32)
        prev = [a.cpu().numpy().astype(np.float64) for a in (mu_g, lt_g, mm, vv)]
        loss_o, mu_o, lt_o, m_o, v_o, lp_o = optim.svi_step(f, prev[0], prev[1], x.astype(np.float64), prev[2], prev[3], t, opt_o, active=act)
        gl.gl_svi_step(m.h, opt, m.obs, m.noise_sigma, m.psf, mu_g, lt_g, d(x), None, mm, vv, t, stats, ws)
        torch.cuda.synchronize()
        assert int(stats[1]) == int(np.isfinite(lp_o).sum()) >= 90
        assert abs(float(stats[0]) - loss_o) <= 1e-4 * abs(loss_o)
        losses.append(float(stats[0]))
        th_g = np.concatenate([mu_g.cpu().numpy(), lt_g.cpu().numpy()]).astype(np.float64)
        th_o = np.concatenate([mu_o, lt_o]); th_p = np.concatenate(prev[:2])
        assert np.array_equal(th_g[~live], th0[~live])                   # dead entries: bit-identical to the start
        assert np.all(mm.cpu().numpy()[~live] == 0) and np.all(vv.cpu().numpy()[~live] == 0)
        step = np.abs(th_o - th_p)
        assert np.all(np.abs(th_g - th_o)[live] <= 2e-3 * step[live] + 4e-7 * (np.abs(th_p) + step)[live] + 1e-30)
    assert np.isfinite(losses).all()


# ------------------------------------------------------------------------------------------------ score-function estimator
def _score_compare(gl, torch, m, spec, obs, sig, psf, mu, lt, xi, opt, baseline, n_finite, n_launch=None):
    """Two iterations of gl_svi_step_score against oracle/optim.py::svi_step_score; the oracle's log p~ is rounded to fp32,
    the storage in which the interface hands it from the hot path to the estimator."""
    import oracle
    from oracle import optim
    n = spec.n_params; nt = n * (n + 1) // 2
    opt_o = {k: (float(np.float32(x)) if k != "kind" else x) for k, x in opt.items()}
    d = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    mu_g, lt_g, xi_g = d(mu), d(lt), d(xi)
    mm, vv = torch.zeros(n + nt, device="cuda"), torch.zeros(n + nt, device="cuda")
    stats = torch.zeros(2, device="cuda")
    ws = torch.empty(gl.gl_svi_workspace_bytes(m.h, xi.shape[0]), dtype=torch.uint8, device="cuda")

    def logp(z):
        r = oracle.logpost_grad(spec, obs, sig, psf, z.astype(np.float32).astype(np.float64), None, want_grad=False)
        return r["logp"].astype(np.float32).astype(np.float64)

    for t in (1, 2):
        prev = [x.cpu().numpy().astype(np.float64) for x in (mu_g, lt_g, mm, vv)]
        loss_o, mu_o, lt_o, m_o, v_o, lp_o = optim.svi_step_score(logp, prev[0], prev[1], xi.astype(np.float64), prev[2], prev[3], t,
                                                                  opt_o, bool(baseline))
        gl.gl_svi_step_score(m.h, opt, m.obs, m.noise_sigma, m.psf, mu_g, lt_g, xi_g, None, mm, vv, t, baseline, stats, ws)
        torch.cuda.synchronize()
        assert int(stats[1]) == n_finite == int(np.isfinite(lp_o).sum())
        assert abs(float(stats[0]) - loss_o) <= 1e-4 * abs(loss_o)
        th_prev = np.concatenate(prev[:2]); th_o = np.concatenate([mu_o, lt_o])
        th_g = np.concatenate([mu_g.cpu().numpy(), lt_g.cpu().numpy()]).astype(np.float64)
        for got, want, old, c, name in ((th_g, th_o, th_prev, 1.0, "theta"), (mm.cpu().numpy().astype(np.float64), m_o, prev[2], opt_o["b1"], "m"),
                                        (vv.cpu().numpy().astype(np.float64), v_o, prev[3], opt_o["b2"], "v")):
            scale = np.abs(c * old) + np.abs(want - c * old)
            bad = np.abs(got - want) > 2e-3 * np.abs(want - c * old) + 4e-7 * scale + 1e-30
            assert not bad.any(), (name, t, int(bad.sum()), np.flatnonzero(bad)[:8])
    if n_launch is not None:
        assert gl.gl_last_launch_count() == n_launch


@pytest.mark.parametrize("baseline", [1, 0], ids=["leave_one_out", "as_printed"])
@pytest.mark.parametrize("opt", [ADABELIEF, ADAM], ids=["adabelief", "adam"])
def test_svi_score_steps_match_oracle(opt, baseline):
    """Eq. 3 of the paper as printed (score-function gradient, log p~ only): two consecutive iterations, 48 draws around the
    seeded truth of config 1, one of them invalid; the hot path runs forward only (draw + 5 path kernels + 5 kernels of the
    estimator, reduction and update)."""
    gl, torch, wl, obs, sig, m, mu, lt, xi = _setup(1, 48, 13)
    xi[9, 2] = 4.0e3                                                    # e1 far outside the unit disc: invalid draw
    _score_compare(gl, torch, m, wl.spec, obs, sig, wl.psf, mu, lt, xi, opt, baseline, 47, n_launch=11)


def test_svi_score_step_58_params_2048_draws():
    """The same on the config-3 parameter layout with a dense L: 2048 draws x 58 parameters (back-substitution over 58 rows per
    draw, the 32-chunk reduction of the pseudo-gradient and its products with xi), three draws thrown out of the domain."""
    gl, torch, sp, obs, sig, psf, m, mu, lt, xi = _big_setup(2048, 307)
    for r in (11, 900, 2040):
        xi[r, 2] = 5.0e4
    _score_compare(gl, torch, m, sp, obs, sig, psf, mu, lt, xi, ADABELIEF, 1, 2045)


def test_svi_score_argument_checks_and_run_loop():
    """baseline outside {0, 1}, backward modelling (surrogate on a subset of the dimensions: pathwise only), and
    LensModel.svi_run with the score estimator: the loss estimate falls over 150 iterations of 1024 fresh draws."""
    import dataclasses
    gl, torch, wl, obs, sig, m, mu, lt, xi = _setup(1, 8, 2)
    n = wl.spec.n_params; nt = n * (n + 1) // 2
    d = lambda a: torch.from_numpy(a).cuda()
    mm, vv, stats = torch.zeros(n + nt, device="cuda"), torch.zeros(n + nt, device="cuda"), torch.zeros(2, device="cuda")
    ws = torch.empty(gl.gl_svi_workspace_bytes(m.h, 8), dtype=torch.uint8, device="cuda")
    with pytest.raises(gl.GLError) as e:
        gl.gl_svi_step_score(m.h, ADAM, m.obs, m.noise_sigma, m.psf, d(mu), d(lt), d(xi), None, mm, vv, 1, 2, stats, ws)
    assert e.value.status == -2
    mb = gl.LensModel(dataclasses.replace(wl.spec, amplitude_mode=1), obs, sig, wl.psf)
    with pytest.raises(gl.GLError) as e:
        gl.gl_svi_step_score(mb.h, ADAM, mb.obs, mb.noise_sigma, mb.psf, d(mu), d(lt), d(xi), None, mm, vv, 1, 1, stats, ws)
    assert e.value.status == -4
    rng = np.random.default_rng(23)
    mu_g = torch.from_numpy((mu + 0.03 * rng.standard_normal(n)).astype(np.float32)).cuda(); lt_g = torch.from_numpy(lt).cuda()
    st, _ = m.svi_run(mu_g, lt_g, dict(ADABELIEF, lr=1e-3), 150, 1024, seed=99, estimator="score")
    st = st.cpu().numpy()
    assert np.isfinite(st).all() and st[-10:, 0].mean() < st[:10, 0].mean(), (st[:3], st[-3:])
    assert torch.all(torch.isfinite(mu_g)) and torch.all(torch.isfinite(lt_g))
