"""the fused HMC transition (gl_hmc_step) against the HMC oracle (oracle/optim.py on top of the fp64
forward/gradient oracle)."""
import numpy as np
import pytest

from _cases import observation

pytestmark = pytest.mark.gpu


def _setup(n_chains, seed, dense):
    import torch
    import paper_2606_30633_b200 as gl
    wl, obs, sig = observation(1)
    n = wl.spec.n_params
    rng = np.random.default_rng(seed)
    z = (wl.truth_z[0][None, :] + 0.01 * rng.standard_normal((n_chains, n))).astype(np.float32)
    L = np.diag(0.004 + 0.004 * rng.random(n))
    if dense:
        L = L + np.tril(0.0008 * rng.standard_normal((n, n)), -1)
    lt = L[np.tril_indices(n)].astype(np.float32)
    xi = rng.standard_normal((n_chains, n)).astype(np.float32)
    log_u = np.log(rng.random(n_chains)).astype(np.float32)
    m = gl.LensModel(wl.spec, obs, sig, wl.psf)
    return gl, torch, wl, obs, sig, m, z, lt, xi, log_u


@pytest.mark.parametrize("dense", [True, False], ids=["dense_L", "identity_L"])
def test_hmc_transition_matches_oracle(dense):
    """Two consecutive transitions (4 leapfrog steps each) of 24 chains near the config-1 truth, one chain started with a
    momentum that throws it out of the model's domain: energy differences, accept flags, positions and the cached
    log-posterior / gradient follow the oracle."""
    import oracle
    from oracle import optim
    gl, torch, wl, obs, sig, m, z0, lt, xi, log_u = _setup(24, 31, dense)
    n = wl.spec.n_params
    if not dense:
        lt_o = optim.tril_pack(np.eye(n)); eps = 2e-5          # stable for config-1 gradients of 1e5
    else:
        lt_o = lt.astype(np.float64); eps = 0.004              # eps * L ~ 2e-5, as above
    xi[3, 1] = 6.0e4 if dense else 6.0e5                               # e1 leaves the unit disc along the trajectory
    d = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    zg = d(z0)
    lpg, gg = m.logpost_grad(zg)
    acc = torch.zeros(24, dtype=torch.int32, device="cuda"); dh = torch.zeros(24, device="cuda")
    ws = torch.empty(gl.gl_hmc_workspace_bytes(m.h, 24), dtype=torch.uint8, device="cuda")

    def f(z):                                                           # the hot path sees fp32 positions (its ABI)
        r = oracle.logpost_grad(wl.spec, obs, sig, wl.psf, z.astype(np.float32).astype(np.float64), None)
        return r["logp"], np.where(np.isfinite(r["logp"])[:, None], r["grad"], 0.0)

    rng = np.random.default_rng(77)
    for t in range(2):
        if t == 1:
            xi = rng.standard_normal(xi.shape).astype(np.float32); log_u = np.log(rng.random(24)).astype(np.float32)
        prev = [x.cpu().numpy().astype(np.float64) for x in (zg, lpg, gg)]
        z_o, lp_o, g_o, acc_o, dh_o = optim.hmc_transition(f, prev[0], prev[1], prev[2], lt_o, xi.astype(np.float64),
                                                           log_u.astype(np.float64), float(np.float32(eps)), 4)
        gl.gl_hmc_step(m.h, m.obs, m.noise_sigma, m.psf, zg, lpg, gg, d(lt) if dense else None, d(xi), d(log_u), None,
                       eps, 4, acc, dh, ws)
        torch.cuda.synchronize()
        dh_g = dh.cpu().numpy().astype(np.float64); acc_g = acc.cpu().numpy().astype(bool)
        fin = np.isfinite(dh_o)
        assert np.array_equal(fin, np.isfinite(dh_g))
        assert fin.sum() >= 20, fin.sum()                               # the trajectories stay inside the model's domain
        if t == 0:
            assert not fin[3] and not acc_g[3]                          # the thrown chain is rejected, state untouched
        # dH is a difference of log-posteriors of size |logp|: bar = the 1e-4 logp bar (far looser than observed)
        assert np.all(np.abs(dh_g[fin] - dh_o[fin]) <= 1e-4 * np.abs(prev[1][fin]) + 1e-6), np.max(np.abs(dh_g[fin] - dh_o[fin]))
        margin = np.abs(log_u.astype(np.float64) - dh_o)
        decided = ~fin | (margin > 1e-3)                                # a float decides an integer: compare where it is unambiguous
        assert decided.sum() >= 20 and np.array_equal(acc_g[decided], acc_o[decided])
        same = acc_g == acc_o
        zz = zg.cpu().numpy().astype(np.float64)
        assert np.all(np.abs(zz[same] - z_o[same]) <= 2e-7 * np.abs(z_o[same]) + 1e-9)
        lpn = lpg.cpu().numpy().astype(np.float64); gn = gg.cpu().numpy().astype(np.float64)
        assert np.all(np.abs(lpn[same] - lp_o[same]) <= 1e-4 * np.abs(lp_o[same]))
        assert np.all(np.abs(gn[same] - g_o[same]) <= np.maximum(1e-3 * np.abs(g_o[same]), 1e-5))
    assert gl.gl_last_launch_count() == 4 * 8 + 2                       # per leapfrog step: kick/drift + 7 path kernels


def test_hmc_chain_keeps_cache_consistent_and_accepts():
    """30 transitions with fresh momenta: the cached log-posterior and gradient stay those of the current positions,
    and with a step size well below the narrowest posterior width most proposals are accepted."""
    gl, torch, wl, obs, sig, m, z0, lt, xi, log_u = _setup(32, 5, False)
    n = wl.spec.n_params
    zg = torch.from_numpy(z0).cuda()
    lpg, gg = m.logpost_grad(zg)
    lpg, gg = lpg.clone(), gg.clone()
    acc = torch.zeros(32, dtype=torch.int32, device="cuda"); dh = torch.zeros(32, device="cuda")
    ws = torch.empty(gl.gl_hmc_workspace_bytes(m.h, 32), dtype=torch.uint8, device="cuda")
    gen = torch.Generator(device="cuda"); gen.manual_seed(9)
    n_acc = 0
    for t in range(30):
        x = torch.randn((32, n), device="cuda", generator=gen)
        lu = torch.log(torch.rand(32, device="cuda", generator=gen))
        gl.gl_hmc_step(m.h, m.obs, m.noise_sigma, m.psf, zg, lpg, gg, None, x, lu, None, 2e-5, 5, acc, dh, ws)
        n_acc += int(acc.sum())
    lp2, g2 = m.logpost_grad(zg)
    torch.cuda.synchronize()
    assert torch.equal(lp2, lpg) and torch.equal(g2, gg)
    assert n_acc / (30 * 32) > 0.5, n_acc


def test_hmc_argument_checks():
    gl, torch, wl, obs, sig, m, z0, lt, xi, log_u = _setup(4, 1, False)
    d = lambda a: torch.from_numpy(a).cuda()
    zg = d(z0); lpg, gg = m.logpost_grad(zg)
    acc = torch.zeros(4, dtype=torch.int32, device="cuda"); dh = torch.zeros(4, device="cuda")
    ws = torch.empty(gl.gl_hmc_workspace_bytes(m.h, 4), dtype=torch.uint8, device="cuda")
    for eps, nl in ((0.0, 3), (1e-3, 0)):
        with pytest.raises(gl.GLError) as e:
            gl.gl_hmc_step(m.h, m.obs, m.noise_sigma, m.psf, zg, lpg, gg, None, d(xi), d(log_u), None, eps, nl, acc, dh, ws)
        assert e.value.status == -2
    with pytest.raises(gl.GLError) as e:
        gl.gl_hmc_step(m.h, m.obs, m.noise_sigma, m.psf, zg, lpg, gg, None, d(xi), d(log_u), None, 1e-3, 2, acc, dh,
                       torch.empty(256, dtype=torch.uint8, device="cuda"))
    assert e.value.status == -5


@pytest.mark.parametrize("layout", [(58, 0, 6, 256), (100, 3, 10, 256)], ids=["cfg3_layout_58", "cfg5_layout_100"])
def test_hmc_transition_many_parameters_many_chains(layout):
    """gl_hmc_kick_drift_kernel / gl_hmc_accept_kernel beyond one warp of parameters: the 58-parameter layout of config 3
    and the 100-parameter layout of config 5 (multipoles, shapelets n_max = 10, two lens Sersics) on a 14x14, s = 2,
    K = 5 geometry where the oracle follows EVERY chain; 256 chains, dense L, 3 leapfrog steps, two transitions."""
    import oracle
    import torch
    import paper_2606_30633_b200 as gl
    from oracle import optim
    from _cases import small_case
    n_want, mp, nmax, nc = layout
    sp, obs, sig, psf, _, truth_z = small_case(14, 2, 5, 1, mp, nmax, 2, seed=600 + n_want, n_particles=2, with_truth=True)
    n = sp.n_params
    assert n == n_want
    rng = np.random.default_rng(n)
    z0 = (truth_z[None, :] + 0.003 * rng.standard_normal((nc, n))).astype(np.float32)
    L = np.diag(0.004 + 0.004 * rng.random(n)) + np.tril(0.0005 * rng.standard_normal((n, n)), -1)
    lt = L[np.tril_indices(n)].astype(np.float32)
    m = gl.LensModel(sp, obs, sig, psf)
    d = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    zg = d(z0)
    lpg, gg = m.logpost_grad(zg)
    lpg, gg = lpg.clone(), gg.clone()
    acc = torch.zeros(nc, dtype=torch.int32, device="cuda"); dh = torch.zeros(nc, device="cuda")
    ws = torch.empty(gl.gl_hmc_workspace_bytes(m.h, nc), dtype=torch.uint8, device="cuda")

    def f(z):
        r = oracle.logpost_grad(sp, obs, sig, psf, z.astype(np.float32).astype(np.float64), None)
        return r["logp"], np.where(np.isfinite(r["logp"])[:, None], r["grad"], 0.0)

    # step size from the largest gradient component: energy changes of order 0.1 .. 10 over 3 steps, nearly every
    # proposal inside the model's domain (checked against the oracle on the CPU when the test was written)
    eps = float(np.float32(1000.0 / max(float(np.abs(gg.cpu().numpy()).max()), 1.0)))
    for t in range(2):
        xi = rng.standard_normal((nc, n)).astype(np.float32)
        if t == 0:
            xi[9, 2] = 1.0e7                                            # thrown out of the model's domain
        log_u = np.log(rng.random(nc)).astype(np.float32)
        prev = [x.cpu().numpy().astype(np.float64) for x in (zg, lpg, gg)]
        z_o, lp_o, g_o, acc_o, dh_o = optim.hmc_transition(f, prev[0], prev[1], prev[2], lt.astype(np.float64), xi.astype(np.float64),
                                                           log_u.astype(np.float64), eps, 3)
        gl.gl_hmc_step(m.h, m.obs, m.noise_sigma, m.psf, zg, lpg, gg, d(lt), d(xi), d(log_u), None, eps, 3, acc, dh, ws)
        torch.cuda.synchronize()
        dh_g = dh.cpu().numpy().astype(np.float64); acc_g = acc.cpu().numpy().astype(bool)
        fin = np.isfinite(dh_o)
        assert np.array_equal(fin, np.isfinite(dh_g))
        assert fin.sum() >= nc - 8, fin.sum()
        if t == 0:
            assert not fin[9] and not acc_g[9]
        assert np.all(np.abs(dh_g[fin] - dh_o[fin]) <= 1e-4 * np.abs(prev[1][fin]) + 1e-6), np.max(np.abs(dh_g[fin] - dh_o[fin]))
        margin = np.abs(log_u.astype(np.float64) - dh_o)
        decided = ~fin | (margin > 1e-4 * np.abs(prev[1]) + 1e-3)       # a float decides an integer: compared where unambiguous
        assert decided.sum() >= nc * 0.9 and np.array_equal(acc_g[decided], acc_o[decided])
        assert acc_o[fin].any()                                         # the test exercises accepted moves
        same = acc_g == acc_o
        zz = zg.cpu().numpy().astype(np.float64)
        assert np.all(np.abs(zz[same] - z_o[same]) <= 2e-7 * np.abs(z_o[same]) + 1e-9)
        lpn = lpg.cpu().numpy().astype(np.float64); gn = gg.cpu().numpy().astype(np.float64)
        assert np.all(np.abs(lpn[same] - lp_o[same]) <= 1e-4 * np.abs(lp_o[same]))
        assert np.all(np.abs(gn[same] - g_o[same]) <= np.maximum(1e-3 * np.abs(g_o[same]), 1e-5))
