"""gl_logpost_grad_noalloc: the hot path on the library's own static scratch buffer (include/gigalens.h), for callers
that cannot allocate device memory.  Checked against the existing caller-workspace path (gl_logpost_grad, itself held to
the oracle by test_gpu_parity.py) at the tolerances of the parity tests, on calls in a row that share the buffer.

Collected last on purpose (the suite runs with pytest -x); passes alone in a fresh process and after the other tests.
"""
import numpy as np
import pytest

from _cases import ATOL_GRAD, RTOL_GRAD, RTOL_LOGP, observation

pytestmark = pytest.mark.gpu


def _gl():
    import paper_2606_30633_b200 as gl
    gl.lib()                                   # fail loudly if the extension is missing
    return gl


def _both(gl, torch, m, z, sid=None):
    """(logp, grad) of the existing path and of the no-allocation entry point for the same particles."""
    lp0, g0 = m.logpost_grad(z, sid)
    lp1 = torch.full_like(lp0, float("nan")); g1 = torch.full_like(g0, float("nan"))
    gl.gl_logpost_grad_noalloc(m.h, m.obs, m.noise_sigma, m.psf, z, m._sid(sid), lp1, g1)
    torch.cuda.synchronize()
    return lp0, g0, lp1, g1


def _assert_same(torch, lp0, g0, lp1, g1):
    a, b = lp0.double().cpu().numpy(), lp1.double().cpu().numpy()
    fin = np.isfinite(a)
    assert fin.any() and np.array_equal(np.isfinite(b), fin)
    assert np.all(np.abs(a[fin] - b[fin]) <= RTOL_LOGP * np.abs(a[fin]))
    ga, gb = g0.double().cpu().numpy(), g1.double().cpu().numpy()
    assert np.all(np.abs(ga - gb) <= np.maximum(RTOL_GRAD * np.abs(ga), ATOL_GRAD))
    # same kernels, same fixed reduction orders: the documented guarantee is bit-identity
    assert torch.equal(lp0, lp1) and torch.equal(g0, g1)


def test_noalloc_matches_workspace_path_on_calls_in_a_row():
    import torch
    gl = _gl()
    wl, obs, sig = observation(1)                                  # config 1: 64 particles, 21 parameters, SIE + shear
    m = gl.LensModel(wl.spec, obs, sig, wl.psf)
    z_a = torch.from_numpy(wl.params).cuda()
    z_b = torch.from_numpy(wl.params[::-1].copy()).cuda()[:37]     # another batch, another size: the buffer holds call 1's data
    _assert_same(torch, *_both(gl, torch, m, z_a))
    _assert_same(torch, *_both(gl, torch, m, z_b))
    # a different configuration (EPL + shapelets, uniform-tap step D: another workspace layout) on the same buffer ...
    wl3, obs3, sig3 = observation(3)
    m3 = gl.LensModel(wl3.spec, obs3, sig3, wl3.psf)
    z3 = torch.from_numpy(wl3.params[:6]).cuda()
    _assert_same(torch, *_both(gl, torch, m3, z3))
    # ... and back: stale contents of another layout must not leak into the result
    lp0, g0, lp1, g1 = _both(gl, torch, m, z_a)
    _assert_same(torch, lp0, g0, lp1, g1)
    # the entry point itself allocates nothing: two bare calls in a row leave the device's free memory where it was
    lp = torch.empty(z_a.shape[0], device="cuda"); g = torch.empty_like(z_a)
    torch.cuda.synchronize()
    free1 = torch.cuda.mem_get_info()[0]
    for _ in range(2):
        gl.gl_logpost_grad_noalloc(m.h, m.obs, m.noise_sigma, m.psf, z_a, None, lp, g)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free1
    assert torch.equal(lp, lp0) and torch.equal(g, g0)
    m.close(); m3.close()


def test_noalloc_rejects_sizes_beyond_the_static_buffer():
    import torch
    gl = _gl()
    wl, obs, sig = observation(2)                                  # 4096 particles need ~3.3 GB of workspace
    m = gl.LensModel(wl.spec, obs, sig, wl.psf)
    z = torch.from_numpy(wl.params).cuda()
    assert gl.gl_workspace_bytes(m.h, z.shape[0]) > gl.GL_NOALLOC_MAX_BYTES
    lp = torch.full((z.shape[0],), 7.0, device="cuda"); g = torch.full_like(z, 7.0)
    with pytest.raises(gl.GLError) as e:
        gl.gl_logpost_grad_noalloc(m.h, m.obs, m.noise_sigma, m.psf, z, None, lp, g)
    assert e.value.status == -7 and "GL_ERR_NOALLOC_LIMIT" in str(e.value)
    assert gl.gl_last_launch_count() == 0                          # rejected before any launch
    torch.cuda.synchronize()
    assert bool((lp == 7.0).all()) and bool((g == 7.0).all())
    # the largest batch of this configuration that fits still runs, and agrees with the existing path
    n = 1
    while gl.gl_workspace_bytes(m.h, 2 * n) <= gl.GL_NOALLOC_MAX_BYTES:
        n *= 2
    _assert_same(torch, *_both(gl, torch, m, z[:n].contiguous()))
    # empty batch: GL_OK, no launch
    gl.gl_logpost_grad_noalloc(m.h, m.obs, m.noise_sigma, m.psf, z[:0], None, lp[:0], g[:0])
    assert gl.gl_last_launch_count() == 0
    m.close()
