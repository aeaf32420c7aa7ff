"""Host side of the C ABI without a GPU: libgigalens.so loads, exports every symbol include/gigalens.h declares,
and validates its arguments before any CUDA call (include/gigalens.h "Errors").  No compute call is made here."""
import ctypes as C
import dataclasses
import os
import re

import pytest

import workloads as W

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def gl():
    import __graft_entry__ as ge
    from paper_2606_30633_b200 import build as gl_build
    gl_build.build()
    import paper_2606_30633_b200 as gl
    gl.lib()
    return gl


def test_every_declared_symbol_is_exported(gl):
    hdr = open(os.path.join(ROOT, "include", "gigalens.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(gl_[a-z0-9_]+)\s*\(", hdr))
    assert len(declared) >= 17
    L = gl.lib()
    for name in sorted(declared):
        assert getattr(L, name) is not None, name
    assert declared == set(gl.EXPORTS), declared ^ set(gl.EXPORTS)
    assert L.gl_version().decode().count(".") == 1


@pytest.mark.parametrize("k, n_params", [(1, 21), (2, 22), (3, 58), (4, 22), (5, 100)])
def test_config_create_and_param_count(gl, k, n_params):
    sp = W.make_spec(k)
    for prec in (0, 1):
        h = gl.gl_config_create(dataclasses.replace(sp, precision=prec))
        assert gl.lib().gl_config_n_params(h) == n_params == sp.n_params
        w1, w2 = gl.gl_workspace_bytes(h, 1), gl.gl_workspace_bytes(h, 64)
        assert 0 < w1 < w2 and gl.gl_workspace_bytes(h, 0) == 0
        assert gl.gl_workspace_bytes(h, 10 ** 7) == gl.gl_workspace_bytes(h, 10 ** 8)     # flat beyond the chunk size
        assert gl.gl_workspace_bytes_host(h, 64) > w2
        gl.gl_config_destroy(h)
    h64 = gl.gl_config_create(dataclasses.replace(sp, precision=0))
    h32 = gl.gl_config_create(dataclasses.replace(sp, precision=1))
    assert gl.gl_workspace_bytes(h64, 16) > gl.gl_workspace_bytes(h32, 16)
    gl.gl_config_destroy(h64); gl.gl_config_destroy(h32)


@pytest.mark.parametrize("field, value, status", [
    ("psf_size", 10, -2), ("supersample", 0, -2), ("n_pix", 0, -2), ("pix_scale", 0.0, -2), ("mass_model", 2, -2),
    ("epl_terms", 31, -2), ("epl_terms", 1, -2), ("n_lens_sersic", 3, -2), ("shapelet_nmax", 11, -2),
    ("n_systems", 0, -2), ("precision", 2, -2), ("param_space", 2, -2), ("multipole_mask", 4, -2),
    ("psf_grid", 2, -4), ("n_pix", 5000, -4)])
def test_config_validation(gl, field, value, status):
    sp = W.make_spec(2)
    if field == "psf_grid":
        sp = dataclasses.replace(sp); sp.psf_grid = value
    else:
        sp = dataclasses.replace(sp, **{field: value})
    with pytest.raises(gl.GLError) as e:
        gl.gl_config_create(sp)
    assert e.value.status == status


def test_param_count_mismatch_and_bad_priors(gl):
    sp = W.make_spec(2)
    bad = dataclasses.replace(sp, priors=sp.priors[:-1])
    with pytest.raises(gl.GLError) as e:
        gl.gl_config_create(bad)
    assert e.value.status == -2
    pri = list(sp.priors); pri[0] = (W.PRIOR_UNIFORM, 0.0, 1.0, 2.0, 1.0)            # hi < lo
    with pytest.raises(gl.GLError):
        gl.gl_config_create(dataclasses.replace(sp, priors=pri))
    pri[0] = (W.PRIOR_NORMAL, 0.0, 0.0, 0.0, 0.0)                                     # sigma = 0
    with pytest.raises(gl.GLError):
        gl.gl_config_create(dataclasses.replace(sp, priors=pri))
    pri[0] = (W.PRIOR_LOGUNIFORM, 0.0, 1.0, 0.0, 1.0)                                 # lo = 0
    with pytest.raises(gl.GLError):
        gl.gl_config_create(dataclasses.replace(sp, priors=pri))


def test_argument_checks_precede_any_cuda_call(gl):
    """NULL handle, negative and zero particle counts are answered on the host (this box has no GPU)."""
    L = gl.lib()
    h = gl.gl_config_create(W.make_spec(1))
    null = C.c_void_p(0)
    assert L.gl_logpost(null, null, null, null, null, null, 4, null, null, 0, null) == -1
    assert L.gl_logpost(h, null, null, null, null, null, -1, null, null, 0, null) == -3
    assert L.gl_logpost(h, null, null, null, null, null, 0, null, null, 0, null) == 0
    assert L.gl_last_launch_count() == 0
    assert L.gl_logpost_grad(h, null, null, null, null, null, 4, null, null, null, 0, null) == -1     # NULL arrays
    assert L.gl_model_image(h, null, null, null, 0, null, null, 0, null) == 0
    assert L.gl_logpost_grad_host(h, null, null, null, null, null, 0, null, null, null, 0, null) == 0
    assert L.gl_workspace_bytes(null, 8) == 0 and L.gl_config_n_params(null) == 0
    # gl_logpost_grad_noalloc: the same checks, and the size limit, answered before any CUDA call
    assert L.gl_logpost_grad_noalloc(null, null, null, null, null, null, 4, null, null, null) == -1
    assert L.gl_logpost_grad_noalloc(h, null, null, null, null, null, -1, null, null, null) == -3
    assert L.gl_logpost_grad_noalloc(h, null, null, null, null, null, 0, null, null, null) == 0
    assert gl.gl_workspace_bytes(h, 10 ** 6) > gl.GL_NOALLOC_MAX_BYTES
    assert L.gl_logpost_grad_noalloc(h, null, null, null, null, null, 10 ** 6, null, null, null) == -7
    assert "GL_NOALLOC_MAX_BYTES" in L.gl_status_string(-7).decode()
    for s in range(0, -8, -1):
        assert L.gl_status_string(s).decode().startswith("GL_")
    assert L.gl_stage_count() == 8 and L.gl_stage_name(2).decode() == "ray_fwd" and L.gl_stage_name(7).decode() == "amplitude_solve"
    gl.gl_config_destroy(h)


def test_binding_refuses_to_compute_without_cuda(gl):
    import torch
    if torch.cuda.is_available():
        pytest.skip("CUDA present")
    with pytest.raises(RuntimeError):
        gl.LensModel(W.make_spec(1), None, None, None)


def test_amplitude_mode_is_validated_on_the_host(gl):
    """amplitude_mode 1 (backward modelling): accepted with the fixed noise map, refused with the model-dependent
    variance; gl_config_n_amplitudes counts I of each Sersic block and the shapelet coefficients."""
    sp = W.make_spec(3)
    h = gl.gl_config_create(sp)
    n_names = sum(1 for n in W.param_names(sp.mass_model, sp.has_shear, sp.multipole_mask, sp.n_source_sersic,
                                           sp.shapelet_nmax, sp.n_lens_sersic) if n.endswith(".I") or n.startswith("shp.a"))
    assert gl.gl_config_n_amplitudes(h) == n_names
    gl.gl_config_destroy(h)
    sp.amplitude_mode = 1
    h = gl.gl_config_create(sp)
    assert gl.gl_workspace_bytes(h, 16) > 0
    L = gl.lib()
    null = C.c_void_p(0)
    assert L.gl_linear_amplitudes(h, null, null, null, null, null, 0, null, null, null, 0, null) == 0
    assert L.gl_linear_amplitudes(h, null, null, null, null, null, 4, null, null, null, 0, null) == -1
    gl.gl_config_destroy(h)
    sp.noise_model = 1; sp.t_exp = 100.0
    with pytest.raises(gl.GLError):
        gl.gl_config_create(sp)
    sp.noise_model = 0; sp.amplitude_mode = 2
    with pytest.raises(gl.GLError):
        gl.gl_config_create(sp)


def test_optimiser_denominator_must_not_vanish_and_consumers_validate_on_the_host(gl):
    """An update 0 / (sqrt(0) + 0) would write NaN (an element whose gradient is exactly 0 from step 1 on): Adam needs
    eps > 0, AdaBelief eps > 0 or eps_root > 0.  And gl_svi_step / gl_hmc_step answer a NULL observation with
    GL_ERR_NULL on the host, before their first kernel (this box has no GPU: a launch would report GL_ERR_CUDA)."""
    L = gl.lib()
    h = gl.gl_config_create(W.make_spec(1))
    null = C.c_void_p(0)
    bad = [gl.gl_opt_desc(0, 1e-3, 0.9, 0.999, 0.0, 0.0), gl.gl_opt_desc(0, 1e-3, 0.9, 0.999, 0.0, 1e-8),
           gl.gl_opt_desc(1, 1e-4, 0.95, 0.99, 0.0, 0.0)]
    for o in bad:
        assert L.gl_map_step(h, C.byref(o), null, null, null, null, null, 4, null, null, 1, null, null, null, 0, null) == -2
        assert L.gl_svi_step(h, C.byref(o), null, null, null, null, null, null, null, 4, null, null, 1, null, null, 0, null) == -2
    ok = gl.gl_opt_desc(1, 1e-4, 0.95, 0.99, 0.0, 1e-16)
    assert L.gl_map_step(h, C.byref(ok), null, null, null, null, null, 0, null, null, 1, null, null, null, 0, null) == 0
    # consumers: every pointer of their own set is a (fake, never dereferenced on the host) non-NULL address, the
    # observation is NULL -> GL_ERR_NULL from the hot path's validation, no launch attempted
    fake = C.c_void_p(1 << 20)
    n = 4
    assert L.gl_svi_step(h, C.byref(ok), null, fake, fake, fake, fake, fake, null, n, fake, fake, 1, fake,
                         fake, L.gl_svi_workspace_bytes(h, n), null) == -1
    assert L.gl_hmc_step(h, null, fake, fake, fake, fake, fake, null, fake, fake, null, n, 1e-3, 2, fake, fake,
                         fake, L.gl_hmc_workspace_bytes(h, n), null) == -1
    assert L.gl_last_launch_count() == 0
    gl.gl_config_destroy(h)


@pytest.mark.parametrize("k", [1, 3, 4])
def test_config_shape(gl, k):
    sp = W.make_spec(k)
    h = gl.gl_config_create(sp)
    sh = gl.gl_config_shape(h)
    assert sh == dict(n_pix=sp.n_pix, psf_size=sp.psf_size, n_systems=sp.n_systems, n_params=sp.n_params,
                      n_amplitudes=gl.gl_config_n_amplitudes(h))
    assert gl.lib().gl_config_shape(C.c_void_p(0), (C.c_int32 * 5)()) == -1
    gl.gl_config_destroy(h)
