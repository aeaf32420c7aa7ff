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
