"""the fused MAP optimiser step (gl_map_step) against the optimiser oracle (oracle/optim.py on top
of the fp64 forward/gradient oracle), and a recover-the-truth smoke run (the analogue of PAPER.md Fig. 5)."""
import numpy as np
import pytest

import workloads as W
from _cases import observation

pytestmark = pytest.mark.gpu

ADAM = dict(kind=0, lr=1e-2, b1=0.9, b2=0.999, eps=1e-8, eps_root=0.0)
ADABELIEF = dict(kind=1, lr=1e-4, b1=0.95, b2=0.99, eps=1e-16, eps_root=1e-16)


@pytest.mark.parametrize("opt", [ADAM, ADABELIEF], ids=["adam", "adabelief"])
def test_map_steps_match_oracle(opt):
    """Three consecutive steps on 12 config-1 particles (one of them invalid): params, both state arrays and the
    reported logp follow the oracle; fp32 storage on the CUDA side bounds the agreement at a few ulp."""
    import oracle
    import torch
    from oracle import optim
    import paper_2606_30633_b200 as gl
    wl, obs, sig = observation(1)
    z0 = wl.params[:12].copy()
    z0[5, 1] = 40.0                                                     # |eps| >= 1 after the transform: invalid particle
    m = gl.LensModel(wl.spec, obs, sig, wl.psf)
    zg = torch.from_numpy(z0).cuda()
    mg, vg = torch.zeros_like(zg), torch.zeros_like(zg)
    lp = torch.empty(12, device="cuda"); g = torch.empty_like(zg)
    # both sides consume the SAME fp32-rounded hyperparameters (reading S20): gl_opt_desc stores floats
    opt_o = {k: (float(np.float32(x)) if k != "kind" else x) for k, x in opt.items()}
    for t in (1, 2, 3):
        # the oracle restarts each step from the fp32 state the interface stores (storage precision is the interface's)
        prev = [x.cpu().numpy().astype(np.float64) for x in (zg, mg, vg)]
        lpo, zo, mo, vo = optim.map_step(oracle, wl.spec, obs, sig, wl.psf, prev[0], prev[1], prev[2], t, opt_o)
        gl.gl_map_step(m.h, opt, m.obs, m.noise_sigma, m.psf, zg, None, mg, vg, t, lp, g, m.workspace(12))
        torch.cuda.synchronize()
        lpg = lp.cpu().numpy().astype(np.float64)
        assert lpg[5] == -np.inf and not np.isfinite(lpo[5])
        ok = np.isfinite(lpo)
        assert np.all(np.abs(lpg[ok] - lpo[ok]) <= 1e-4 * np.abs(lpo[ok]))
        # Each new value is old * c + increment; its error is bounded by the fp32 storage rounding (2^-24) and the
        # 6e-8 relative error of the fp32 gradient, both relative to the SIZE OF THE TWO TERMS (m may cancel).
        for got, want, old, c, name in ((zg, zo, prev[0], 1.0, "z"), (mg, mo, prev[1], opt_o["b1"], "m"),
                                        (vg, vo, prev[2], opt_o["b2"], "v")):
            got = got.cpu().numpy().astype(np.float64)
            scale = np.abs(c * old) + np.abs(want - c * old)
            assert np.all(np.abs(got - want) <= 4e-7 * scale + 1e-30), (name, t, np.max(np.abs(got - want) / (scale + 1e-300)))
        assert np.array_equal(zg.cpu().numpy()[5], z0[5])               # the invalid particle never moves
    assert gl.gl_last_launch_count() == 8                               # 7 path kernels + 1 update kernel


def test_map_run_recovers_the_truth_smoke():
    """Config 1: 32 starts scattered around the seeded truth (0.05 in unconstrained units), 300 Adam steps on the
    device with no host round trip: every start improves its log-posterior and the best one reaches the truth's."""
    import torch
    import paper_2606_30633_b200 as gl
    wl, obs, sig = observation(1)
    rng = np.random.default_rng(5)
    z0 = (wl.truth_z[0][None, :] + 0.05 * rng.standard_normal((32, wl.spec.n_params))).astype(np.float32)
    m = gl.LensModel(wl.spec, obs, sig, wl.psf)
    lp_truth = float(m.logpost(torch.from_numpy(wl.truth_z[:1]).cuda())[0])
    z = torch.from_numpy(z0).cuda()
    lp0 = m.logpost(z).clone()
    lp, _ = m.map_run(z, dict(ADAM, lr=2e-3), 300)
    lp1 = m.logpost(z)
    torch.cuda.synchronize()
    assert torch.all(lp1 > lp0)
    assert float(lp1.max()) >= lp_truth - 25.0, (float(lp1.max()), lp_truth)     # chi^2 within ~2 sigma of 1600 pixels


def test_map_step_argument_checks():
    import torch
    import paper_2606_30633_b200 as gl
    wl, obs, sig = observation(1)
    m = gl.LensModel(wl.spec, obs, sig, wl.psf)
    z = torch.from_numpy(wl.params[:4].copy()).cuda()
    mm, vv, g = torch.zeros_like(z), torch.zeros_like(z), torch.empty_like(z)
    lp = torch.empty(4, device="cuda")
    for bad in (dict(ADAM, lr=0.0), dict(ADAM, b1=1.0), dict(ADAM, kind=7), dict(ADAM, eps=-1.0)):
        with pytest.raises(gl.GLError) as e:
            gl.gl_map_step(m.h, bad, m.obs, m.noise_sigma, m.psf, z, None, mm, vv, 1, lp, g, m.workspace(4))
        assert e.value.status == -2
    with pytest.raises(gl.GLError) as e:
        gl.gl_map_step(m.h, ADAM, m.obs, m.noise_sigma, m.psf, z, None, mm, vv, 0, lp, g, m.workspace(4))
    assert e.value.status == -2


def test_best_particle_matches_numpy_argmax():
    """gl_best_particle against the plain definition (largest finite entry, lowest index on ties), including ties,
    non-finite entries, sizes around the block size and the all-invalid case.  Integer result: exact."""
    import torch
    import paper_2606_30633_b200 as gl
    rng = np.random.default_rng(4)
    for n in (1, 7, 1023, 1024, 1025, 4096, 100003):
        v = rng.standard_normal(n).astype(np.float32)
        v[rng.random(n) < 0.1] = -np.inf
        if n > 3:
            v[rng.integers(0, n, 3)] = np.nan
            j = rng.integers(0, n, 4); v[j] = np.float32(7.5)             # a four-way tie for the maximum
        w = np.where(np.isfinite(v), v, -np.inf)
        want = int(np.argmax(w)) if np.isfinite(w).any() else -1
        idx, val = gl.gl_best_particle(torch.from_numpy(v).cuda())
        assert int(idx[0]) == want, (n, int(idx[0]), want)
        assert float(val[0]) == (float(v[want]) if want >= 0 else -np.inf)
    idx, val = gl.gl_best_particle(torch.full((50,), -np.inf).cuda())
    assert int(idx[0]) == -1 and float(val[0]) == -np.inf
