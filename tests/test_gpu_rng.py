"""On-device counter-based draws (gl_draw_normal / gl_draw_log_uniform, reading S22) against oracle/rng.py, and the
device-resident SVI / HMC loops built on them."""
import numpy as np
import pytest

from _cases import observation

pytestmark = pytest.mark.gpu


def _ulp32(a, b):
    a = np.asarray(a, np.float32); b = np.asarray(b, np.float32)
    return np.abs(a.astype(np.float64) - b.astype(np.float64)) / np.spacing(np.maximum(np.abs(a), np.abs(b)).astype(np.float32)).astype(np.float64)


@pytest.mark.parametrize("shape", [(1, 1), (7, 22), (1000, 43), (3, 128), (257, 5)])
def test_draws_match_oracle(shape):
    """Same bits on both sides (Philox is integer work), fp64 Box-Muller on both: after rounding to fp32 the values
    agree to 1 ulp everywhere and are identical almost everywhere (libm's log/sincos differ from CUDA's by < 2 fp64 ulp)."""
    import torch
    import paper_2606_30633_b200 as gl
    from oracle import rng as R
    n, c = shape
    seed, step = 0xC0FFEE1234567, (3 << 32) + 17
    for sid in (0, 1, 255):
        x = gl.gl_draw_normal(seed, step, sid, torch.empty((n, c), device="cuda")).cpu().numpy()
        ref = R.draw_normal(seed, step, sid, n, c)
        assert np.all(_ulp32(x, ref) <= 1.0)
        assert (x == ref).mean() > 0.999 or x.size < 100
        lu = gl.gl_draw_log_uniform(seed, step, sid, torch.empty(n, device="cuda")).cpu().numpy()
        ref_u = R.draw_log_uniform(seed, step, sid, n)
        assert np.all(_ulp32(lu, ref_u) <= 1.0)
    assert gl.gl_last_launch_count() == 1


def test_draws_are_stateless_and_checked():
    import torch
    import paper_2606_30633_b200 as gl
    a = gl.gl_draw_normal(5, 9, 0, torch.empty((300, 22), device="cuda")).clone()
    b = gl.gl_draw_normal(5, 9, 0, torch.empty((100, 22), device="cuda"))
    assert torch.equal(a[:100], b)                                       # a smaller batch is a prefix: no hidden state
    c = gl.gl_draw_normal(5, 10, 0, torch.empty((300, 22), device="cuda"))
    assert not torch.any(a == c)
    with pytest.raises(gl.GLError):
        gl.gl_draw_normal(5, 9, 256, torch.empty((4, 4), device="cuda"))
    L = gl.lib()
    assert L.gl_draw_normal(1, 1, 0, 0, 4, None, None) == 0 and L.gl_draw_normal(1, 1, 0, 4, 4, None, None) == -1
    assert L.gl_draw_log_uniform(1, 1, 0, -1, None, None) == -3


def test_svi_run_with_device_draws_matches_oracle_driven_run():
    """Three SVI iterations on config 1 with the draws made on the device equal the same iterations fed with the
    oracle generator's draws through the xi argument (bit for bit where the draws are bit-identical, else to fp32
    rounding), and the loss follows oracle/optim.py driven by oracle/rng.py."""
    import torch
    import oracle
    from oracle import optim, rng as R
    import paper_2606_30633_b200 as gl
    wl, obs, sig = observation(1)
    n = wl.spec.n_params; nt = n * (n + 1) // 2
    rg = np.random.default_rng(3)
    mu0 = wl.truth_z[0].astype(np.float32).copy()
    L = np.tril(0.002 * rg.standard_normal((n, n))) + np.diag(0.01 + 0.01 * rg.random(n))
    lt0 = L[np.tril_indices(n)].astype(np.float32)
    opt = dict(kind=1, lr=1e-4, b1=0.95, b2=0.99, eps=1e-16, eps_root=1e-16)
    m = gl.LensModel(wl.spec, obs, sig, wl.psf)
    d = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    mu_a, lt_a = d(mu0), d(lt0)
    stats, _ = m.svi_run(mu_a, lt_a, opt, 3, 32, seed=99)
    # the same three iterations with host-made oracle draws
    mu_b, lt_b = d(mu0), d(lt0)
    mm, vv = torch.zeros(n + nt, device="cuda"), torch.zeros(n + nt, device="cuda")
    st = torch.zeros(2, device="cuda")
    ws = torch.empty(gl.gl_svi_workspace_bytes(m.h, 32), dtype=torch.uint8, device="cuda")
    opt_o = {k: (float(np.float32(x)) if k != "kind" else x) for k, x in opt.items()}
    mu_o, lt_o, m_o, v_o = mu0.astype(np.float64), lt0.astype(np.float64), np.zeros(n + nt), np.zeros(n + nt)

    def f(z):
        r = oracle.logpost_grad(wl.spec, obs, sig, wl.psf, z.astype(np.float32).astype(np.float64), None)
        return r["logp"], r["grad"]

    for t in (1, 2, 3):
        xi = R.draw_normal(99, t, 0, 32, n)
        gl.gl_svi_step(m.h, opt, m.obs, m.noise_sigma, m.psf, mu_b, lt_b, d(xi), None, mm, vv, t, st, ws)
        loss_o, mu_o, lt_o, m_o, v_o, _ = optim.svi_step(f, mu_o, lt_o, xi.astype(np.float64), m_o, v_o, t, opt_o)
        assert abs(float(stats[t - 1, 0]) - float(st[0])) <= 1e-5 * abs(float(st[0]))
        assert abs(float(st[0]) - loss_o) <= 1e-3 * abs(loss_o)
        assert int(stats[t - 1, 1]) == 32
    assert torch.allclose(mu_a, mu_b, rtol=0, atol=2e-6) and torch.allclose(lt_a, lt_b, rtol=0, atol=2e-6)


def test_hmc_run_with_device_draws_samples_near_the_mode():
    """64 chains, 20 transitions on config 1, every draw made on the device: acceptance in a sane band, the cached
    log-posterior stays consistent with a fresh evaluation, and a second run with the same seed is bit-identical."""
    import torch
    import paper_2606_30633_b200 as gl
    wl, obs, sig = observation(1)
    rg = np.random.default_rng(4)
    z0 = (wl.truth_z[0][None, :] + 0.002 * rg.standard_normal((64, wl.spec.n_params))).astype(np.float32)
    m = gl.LensModel(wl.spec, obs, sig, wl.psf)
    runs = []
    for _ in range(2):
        z = torch.from_numpy(z0).cuda()
        lp, g, acc = m.hmc_run(z, None, 2e-5, 4, 20, seed=7)
        torch.cuda.synchronize()
        runs.append((z.clone(), lp.clone(), acc.clone()))
    assert torch.equal(runs[0][0], runs[1][0]) and torch.equal(runs[0][2], runs[1][2])
    z, lp, acc = runs[0]
    rate = float(acc.float().mean())
    assert 0.3 < rate <= 1.0, rate
    lp2, _ = m.logpost_grad(z)
    assert torch.equal(lp, lp2)
    moved = (z != torch.from_numpy(z0).cuda()).any(dim=1)
    assert moved.float().mean() > 0.9
