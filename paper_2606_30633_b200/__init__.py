"""paper_2606_30633_b200 -- thin Python binding of libgigalens (include/gigalens.h).

Argument marshalling only: every step of the path runs in the hand-written sm_100a kernels of
csrc/.  PyTorch is used for device memory and streams.  There is NO CPU fallback: importing works without
a GPU (so the symbol-export test can run), but every compute call raises if the shared library is missing or
CUDA is unavailable.  This package never imports oracle/.

Function names follow the C ABI: gl_config_create, gl_workspace_bytes, gl_logpost, gl_logpost_grad,
gl_model_image, gl_logpost_grad_host.  `LensModel` bundles a config handle with a cached workspace.
"""
import ctypes as C
import os

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(HERE, "libgigalens.so")

GL_OK = 0
GL_PRECISION_F64, GL_PRECISION_F32 = 0, 1
STATUS = {0: "GL_OK", -1: "GL_ERR_NULL", -2: "GL_ERR_BAD_CONFIG", -3: "GL_ERR_BAD_SHAPE", -4: "GL_ERR_UNSUPPORTED",
          -5: "GL_ERR_WORKSPACE", -6: "GL_ERR_CUDA", -7: "GL_ERR_NOALLOC_LIMIT"}
EXPORTS = ["gl_config_create", "gl_config_destroy", "gl_config_n_params", "gl_workspace_bytes", "gl_logpost",
           "gl_logpost_grad", "gl_model_image", "gl_workspace_bytes_host", "gl_logpost_grad_host",
           "gl_last_launch_count", "gl_status_string", "gl_version", "gl_stage_timing_enable", "gl_stage_count",
           "gl_stage_name", "gl_stage_times", "gl_probe_pipe", "gl_map_step",
           "gl_svi_workspace_bytes", "gl_svi_step", "gl_hmc_workspace_bytes", "gl_hmc_step",
           "gl_best_particle", "gl_config_n_amplitudes", "gl_linear_amplitudes", "gl_draw_normal", "gl_draw_log_uniform",
           "gl_config_shape", "gl_workspace_layout", "gl_logpost_grad_noalloc", "gl_svi_step_score"]
GL_NOALLOC_MAX_BYTES = 32 << 20      # include/gigalens.h


class GLError(RuntimeError):
    def __init__(self, status, where):
        self.status = status
        super().__init__("%s failed: %s (%d)" % (where, STATUS.get(status, "?"), status))


class gl_prior(C.Structure):
    _fields_ = [("kind", C.c_int32), ("a", C.c_float), ("b", C.c_float), ("lo", C.c_float), ("hi", C.c_float)]


class gl_opt_desc(C.Structure):
    _fields_ = [("kind", C.c_int32), ("lr", C.c_float), ("b1", C.c_float), ("b2", C.c_float), ("eps", C.c_float),
                ("eps_root", C.c_float)]


GL_OPT_ADAM, GL_OPT_ADABELIEF = 0, 1


class gl_config_desc(C.Structure):
    _fields_ = [("n_pix", C.c_int32), ("supersample", C.c_int32), ("psf_size", C.c_int32), ("pix_scale", C.c_float),
                ("psf_grid", C.c_int32), ("mass_model", C.c_int32), ("epl_terms", C.c_int32), ("has_shear", C.c_int32),
                ("multipole_mask", C.c_int32), ("n_source_sersic", C.c_int32), ("shapelet_nmax", C.c_int32),
                ("n_lens_sersic", C.c_int32), ("param_space", C.c_int32), ("n_systems", C.c_int32),
                ("n_params", C.c_int32), ("precision", C.c_int32), ("noise_model", C.c_int32),
                ("exposure_time", C.c_float), ("amplitude_mode", C.c_int32), ("source2_plane", C.c_int32),
                ("priors", C.POINTER(gl_prior))]


_lib = None


def lib():
    """Load libgigalens.so (built in-tree by paper_2606_30633_b200.build); fail loudly if it is missing."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError("libgigalens.so not built: run `python -m paper_2606_30633_b200.build` "
                               "(there is no CPU fallback)")
        L = C.CDLL(LIB_PATH)
        vp, i64, sz = C.c_void_p, C.c_int64, C.c_size_t
        L.gl_config_create.restype = C.c_int
        L.gl_config_create.argtypes = [C.POINTER(gl_config_desc), C.POINTER(vp)]
        L.gl_config_destroy.restype = None
        L.gl_config_destroy.argtypes = [vp]
        L.gl_config_n_params.restype = C.c_int32
        L.gl_config_n_params.argtypes = [vp]
        L.gl_config_shape.restype = C.c_int
        L.gl_config_shape.argtypes = [vp, C.POINTER(C.c_int32)]
        L.gl_workspace_bytes.restype = sz
        L.gl_workspace_bytes.argtypes = [vp, i64]
        L.gl_workspace_layout.restype = C.c_int
        L.gl_workspace_layout.argtypes = [vp, i64, C.POINTER(i64)]
        L.gl_workspace_bytes_host.restype = sz
        L.gl_workspace_bytes_host.argtypes = [vp, i64]
        L.gl_logpost.restype = C.c_int
        L.gl_logpost.argtypes = [vp, vp, vp, vp, vp, vp, i64, vp, vp, sz, vp]
        L.gl_logpost_grad.restype = C.c_int
        L.gl_logpost_grad.argtypes = [vp, vp, vp, vp, vp, vp, i64, vp, vp, vp, sz, vp]
        L.gl_logpost_grad_noalloc.restype = C.c_int
        L.gl_logpost_grad_noalloc.argtypes = [vp, vp, vp, vp, vp, vp, i64, vp, vp, vp]
        L.gl_logpost_grad_host.restype = C.c_int
        L.gl_logpost_grad_host.argtypes = [vp, vp, vp, vp, vp, vp, i64, vp, vp, vp, sz, vp]
        L.gl_map_step.restype = C.c_int
        L.gl_map_step.argtypes = [vp, C.POINTER(gl_opt_desc), vp, vp, vp, vp, vp, i64, vp, vp, i64, vp, vp, vp, sz, vp]
        L.gl_best_particle.restype = C.c_int
        L.gl_best_particle.argtypes = [vp, i64, vp, vp, vp]
        L.gl_hmc_workspace_bytes.restype = sz
        L.gl_hmc_workspace_bytes.argtypes = [vp, i64]
        L.gl_hmc_step.restype = C.c_int
        L.gl_hmc_step.argtypes = [vp, vp, vp, vp, vp, vp, vp, vp, vp, vp, vp, i64, C.c_float, C.c_int32, vp, vp, vp, sz, vp]
        L.gl_svi_workspace_bytes.restype = sz
        L.gl_svi_workspace_bytes.argtypes = [vp, i64]
        L.gl_svi_step.restype = C.c_int
        L.gl_svi_step.argtypes = [vp, C.POINTER(gl_opt_desc), vp, vp, vp, vp, vp, vp, vp, i64, vp, vp, i64, vp, vp, sz, vp]
        L.gl_svi_step_score.restype = C.c_int
        L.gl_svi_step_score.argtypes = [vp, C.POINTER(gl_opt_desc), vp, vp, vp, vp, vp, vp, vp, i64, vp, vp, i64, C.c_int32, vp, vp, sz, vp]
        L.gl_draw_normal.restype = C.c_int
        L.gl_draw_normal.argtypes = [C.c_uint64, C.c_uint64, C.c_uint32, i64, C.c_int32, vp, vp]
        L.gl_draw_log_uniform.restype = C.c_int
        L.gl_draw_log_uniform.argtypes = [C.c_uint64, C.c_uint64, C.c_uint32, i64, vp, vp]
        L.gl_config_n_amplitudes.restype = C.c_int32
        L.gl_config_n_amplitudes.argtypes = [vp]
        L.gl_linear_amplitudes.restype = C.c_int
        L.gl_linear_amplitudes.argtypes = [vp, vp, vp, vp, vp, vp, i64, vp, vp, vp, sz, vp]
        L.gl_model_image.restype = C.c_int
        L.gl_model_image.argtypes = [vp, vp, vp, vp, i64, vp, vp, sz, vp]
        L.gl_last_launch_count.restype = i64
        L.gl_status_string.restype = C.c_char_p
        L.gl_status_string.argtypes = [C.c_int]
        L.gl_version.restype = C.c_char_p
        L.gl_stage_timing_enable.restype = None
        L.gl_stage_timing_enable.argtypes = [C.c_int32]
        L.gl_stage_count.restype = C.c_int32
        L.gl_stage_name.restype = C.c_char_p
        L.gl_stage_name.argtypes = [C.c_int32]
        L.gl_stage_times.restype = C.c_int32
        L.gl_stage_times.argtypes = [C.POINTER(C.c_float), C.POINTER(C.c_int32), C.c_int32]
        L.gl_probe_pipe.restype = C.c_int
        L.gl_probe_pipe.argtypes = [C.c_int32, C.c_int32, vp, sz, vp, C.POINTER(C.c_double), C.POINTER(C.c_float)]
        _lib = L
    return _lib


def _check(status, where):
    if status != GL_OK:
        raise GLError(status, where)


def gl_config_create(spec):
    """spec: any object with the gl_config_desc field names (e.g. workloads.LensSpec) and
    priors = [(kind, a, b, lo, hi), ...].  Returns an opaque handle (c_void_p)."""
    n = len(spec.priors)
    pri = (gl_prior * max(n, 1))()
    for i, (k, a, b, lo, hi) in enumerate(spec.priors):
        pri[i] = gl_prior(int(k), float(a), float(b), float(lo), float(hi))
    d = gl_config_desc(spec.n_pix, spec.supersample, spec.psf_size, float(spec.pix_scale),
                       int(getattr(spec, "psf_grid", 0)), spec.mass_model, spec.epl_terms, spec.has_shear,
                       spec.multipole_mask, spec.n_source_sersic, spec.shapelet_nmax, spec.n_lens_sersic,
                       spec.param_space, spec.n_systems, int(getattr(spec, "n_params", n)),
                       int(getattr(spec, "precision", GL_PRECISION_F64)), int(getattr(spec, "noise_model", 0)),
                       float(getattr(spec, "t_exp", 1.0)), int(getattr(spec, "amplitude_mode", 0)),
                       int(getattr(spec, "source2_plane", 0)), pri)
    h = C.c_void_p()
    _check(lib().gl_config_create(C.byref(d), C.byref(h)), "gl_config_create")
    return h


def gl_config_destroy(h):
    _shape_cache.pop(h.value if isinstance(h, C.c_void_p) else h, None)
    lib().gl_config_destroy(h)


def gl_workspace_bytes(h, n):
    return lib().gl_workspace_bytes(h, int(n))


def gl_workspace_layout(h, n):
    """dict(off_pb, chunk, pb_stride, elem_bytes, idx_m1, idx_m2, idx_valid, last_chunk_first) -- include/gigalens.h."""
    out = (C.c_int64 * 8)()
    _check(lib().gl_workspace_layout(h, int(n), out), "gl_workspace_layout")
    return dict(zip(("off_pb", "chunk", "pb_stride", "elem_bytes", "idx_m1", "idx_m2", "idx_valid", "last_chunk_first"),
                    (int(x) for x in out)))


def gl_workspace_bytes_host(h, n):
    return lib().gl_workspace_bytes_host(h, int(n))


def gl_last_launch_count():
    return lib().gl_last_launch_count()


def gl_stage_timing_enable(on):
    lib().gl_stage_timing_enable(1 if on else 0)


def gl_stage_times():
    """{stage name: (milliseconds, launches)} of the most recent compute call of this thread (waits for it)."""
    L = lib()
    n = L.gl_stage_count()
    ms = (C.c_float * n)(); cnt = (C.c_int32 * n)()
    if L.gl_stage_times(ms, cnt, n) != n:
        raise RuntimeError("gl_stage_times failed")
    return {L.gl_stage_name(i).decode(): (float(ms[i]), int(cnt[i])) for i in range(n)}


def gl_probe_pipe(kind, n_outer=2048, stream=None):
    """(tera lane-ops/s, kernel ms) of one SM pipe: kind 0 FP32 FMA, 1 FP64 FMA, 2 MUFU ex2, 3 FP32+FP64 interleaved,
    4 FP64 FMA with distinct operands, 5 FP64 tensor MMA (m8n8k4), 6 FP64 MMA + FMA interleaved, 7 FP64 FMA with two vector
    operands + one uniform operand, 8 FP64 FMA with three vector operands, multiplier shared by neighbours."""
    torch = _torch()
    ws = torch.zeros(256, dtype=torch.uint8, device="cuda")
    rate = C.c_double(); ms = C.c_float()
    _check(lib().gl_probe_pipe(int(kind), int(n_outer), _ptr(ws), 256, _stream(stream), C.byref(rate), C.byref(ms)),
           "gl_probe_pipe")
    return rate.value, ms.value


def _torch():
    import torch
    if not torch.cuda.is_available():
        raise RuntimeError("CUDA device required: libgigalens has no CPU fallback")
    return torch


def _dev(t, dtype, name):
    torch = _torch()
    if t is None:
        return None
    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == dtype and t.is_contiguous()):
        raise TypeError("%s must be a contiguous CUDA tensor of dtype %s" % (name, dtype))
    return t


def _ptr(t):
    return C.c_void_p(t.data_ptr()) if t is not None else C.c_void_p(0)


def gl_config_shape(h):
    """dict(n_pix, psf_size, n_systems, n_params, n_amplitudes) of a handle."""
    out = (C.c_int32 * 5)()
    _check(lib().gl_config_shape(h, out), "gl_config_shape")
    return dict(zip(("n_pix", "psf_size", "n_systems", "n_params", "n_amplitudes"), (int(x) for x in out)))


_shape_cache = {}


def _extents(h, n, **arrays):
    """Element-count checks of the tensors of one call against the configuration (the C ABI sees plain pointers, so a
    wrongly sized tensor would otherwise be a silent out-of-bounds access on the device).  n = rows of the batch."""
    key = h.value if isinstance(h, C.c_void_p) else h
    sh = _shape_cache.get(key)
    if sh is None:
        sh = _shape_cache[key] = gl_config_shape(h)
    N2, K2, S, P, A = sh["n_pix"] ** 2, sh["psf_size"] ** 2, sh["n_systems"], sh["n_params"], sh["n_amplitudes"]
    T = P * (P + 1) // 2
    want = {"obs": S * N2, "noise_sigma": S * N2, "psf": S * K2, "params": n * P, "system_id": n, "out_logp": n,
            "out_grad": n * P, "out_image": n * N2, "out_amp": n * A, "opt_m": n * P, "opt_v": n * P, "mu": P, "l_tril": T,
            "xi": n * P, "svi_m": P + T, "svi_v": P + T, "out_stats": 2, "z": n * P, "logp": n, "grad": n * P, "log_u": n,
            "out_accept": n, "out_dh": n}
    for name, t in arrays.items():
        if t is not None and t.numel() != want[name]:
            raise ValueError("%s has %d elements, the configuration needs %d" % (name, t.numel(), want[name]))


def _stream(stream):
    torch = _torch()
    s = torch.cuda.current_stream() if stream is None else stream
    return C.c_void_p(s.cuda_stream)


def gl_logpost(h, obs, noise_sigma, psf, params, system_id, out_logp, workspace, stream=None):
    torch = _torch()
    f32 = torch.float32
    n = params.shape[0]
    _extents(h, n, obs=obs, noise_sigma=noise_sigma, psf=psf, params=params, system_id=system_id, out_logp=out_logp)
    _check(lib().gl_logpost(h, _ptr(_dev(obs, f32, "obs")), _ptr(_dev(noise_sigma, f32, "noise_sigma")),
                            _ptr(_dev(psf, f32, "psf")), _ptr(_dev(params, f32, "params")),
                            _ptr(_dev(system_id, torch.int32, "system_id")), n, _ptr(_dev(out_logp, f32, "out_logp")),
                            _ptr(workspace), workspace.numel() * workspace.element_size(), _stream(stream)), "gl_logpost")


def gl_draw_normal(seed, step, stream_id, out, stream=None):
    """Fill the fp32 CUDA tensor out [n_rows][n_cols] with counter-based standard normals (include/gigalens.h)."""
    torch = _torch()
    _dev(out, torch.float32, "out")
    assert out.dim() == 2
    _check(lib().gl_draw_normal(int(seed), int(step), int(stream_id), out.shape[0], out.shape[1], _ptr(out), _stream(stream)),
           "gl_draw_normal")
    return out


def gl_draw_log_uniform(seed, step, stream_id, out, stream=None):
    torch = _torch()
    _dev(out, torch.float32, "out")
    assert out.dim() == 1
    _check(lib().gl_draw_log_uniform(int(seed), int(step), int(stream_id), out.shape[0], _ptr(out), _stream(stream)),
           "gl_draw_log_uniform")
    return out


def gl_config_n_amplitudes(h):
    return int(lib().gl_config_n_amplitudes(h))


def gl_linear_amplitudes(h, obs, noise_sigma, psf, params, system_id, out_amp, out_logp, workspace, stream=None):
    torch = _torch()
    f32 = torch.float32
    n = params.shape[0]
    _extents(h, n, obs=obs, noise_sigma=noise_sigma, psf=psf, params=params, system_id=system_id, out_logp=out_logp, out_amp=out_amp)
    _check(lib().gl_linear_amplitudes(h, _ptr(_dev(obs, f32, "obs")), _ptr(_dev(noise_sigma, f32, "noise_sigma")),
                                      _ptr(_dev(psf, f32, "psf")), _ptr(_dev(params, f32, "params")),
                                      _ptr(_dev(system_id, torch.int32, "system_id")), n,
                                      _ptr(_dev(out_amp, f32, "out_amp")), _ptr(_dev(out_logp, f32, "out_logp")),
                                      _ptr(workspace), workspace.numel() * workspace.element_size(), _stream(stream)),
           "gl_linear_amplitudes")


def gl_logpost_grad(h, obs, noise_sigma, psf, params, system_id, out_logp, out_grad, workspace, stream=None):
    torch = _torch()
    f32 = torch.float32
    n = params.shape[0]
    _extents(h, n, obs=obs, noise_sigma=noise_sigma, psf=psf, params=params, system_id=system_id, out_logp=out_logp, out_grad=out_grad)
    _check(lib().gl_logpost_grad(h, _ptr(_dev(obs, f32, "obs")), _ptr(_dev(noise_sigma, f32, "noise_sigma")),
                                 _ptr(_dev(psf, f32, "psf")), _ptr(_dev(params, f32, "params")),
                                 _ptr(_dev(system_id, torch.int32, "system_id")), n,
                                 _ptr(_dev(out_logp, f32, "out_logp")), _ptr(_dev(out_grad, f32, "out_grad")),
                                 _ptr(workspace), workspace.numel() * workspace.element_size(), _stream(stream)),
           "gl_logpost_grad")


def gl_logpost_grad_noalloc(h, obs, noise_sigma, psf, params, system_id, out_logp, out_grad, stream=None):
    """gl_logpost_grad on the library's own static scratch buffer (no workspace argument, nothing allocated by the call;
    at most GL_NOALLOC_MAX_BYTES of workspace, else GLError GL_ERR_NOALLOC_LIMIT; calls must not overlap on the GPU)."""
    torch = _torch()
    f32 = torch.float32
    n = params.shape[0]
    _extents(h, n, obs=obs, noise_sigma=noise_sigma, psf=psf, params=params, system_id=system_id, out_logp=out_logp, out_grad=out_grad)
    _check(lib().gl_logpost_grad_noalloc(h, _ptr(_dev(obs, f32, "obs")), _ptr(_dev(noise_sigma, f32, "noise_sigma")),
                                         _ptr(_dev(psf, f32, "psf")), _ptr(_dev(params, f32, "params")),
                                         _ptr(_dev(system_id, torch.int32, "system_id")), n,
                                         _ptr(_dev(out_logp, f32, "out_logp")), _ptr(_dev(out_grad, f32, "out_grad")),
                                         _stream(stream)), "gl_logpost_grad_noalloc")


def gl_map_step(h, opt, obs, noise_sigma, psf, params, system_id, opt_m, opt_v, step, out_logp, out_grad, workspace,
                stream=None):
    """opt: dict(kind, lr, b1, b2, eps, eps_root) or a gl_opt_desc.  params / opt_m / opt_v are updated in place."""
    torch = _torch()
    f32 = torch.float32
    opt = _opt_desc(opt)
    n = params.shape[0]
    _extents(h, n, obs=obs, noise_sigma=noise_sigma, psf=psf, params=params, system_id=system_id, out_logp=out_logp, out_grad=out_grad,
             opt_m=opt_m, opt_v=opt_v)
    _check(lib().gl_map_step(h, C.byref(opt), _ptr(_dev(obs, f32, "obs")), _ptr(_dev(noise_sigma, f32, "noise_sigma")),
                             _ptr(_dev(psf, f32, "psf")), _ptr(_dev(params, f32, "params")),
                             _ptr(_dev(system_id, torch.int32, "system_id")), n, _ptr(_dev(opt_m, f32, "opt_m")),
                             _ptr(_dev(opt_v, f32, "opt_v")), int(step), _ptr(_dev(out_logp, f32, "out_logp")),
                             _ptr(_dev(out_grad, f32, "out_grad")), _ptr(workspace),
                             workspace.numel() * workspace.element_size(), _stream(stream)), "gl_map_step")


def _opt_desc(opt):
    if isinstance(opt, gl_opt_desc):
        return opt
    return gl_opt_desc(int(opt["kind"]), float(opt["lr"]), float(opt["b1"]), float(opt["b2"]), float(opt["eps"]),
                       float(opt.get("eps_root", 0.0)))


def gl_best_particle(logp, stream=None):
    """(index tensor [1] int64, value tensor [1] float32) of the largest finite log-posterior, on the device."""
    torch = _torch()
    idx = torch.empty(1, dtype=torch.int64, device=logp.device)
    val = torch.empty(1, dtype=torch.float32, device=logp.device)
    _check(lib().gl_best_particle(_ptr(_dev(logp, torch.float32, "logp")), logp.shape[0], _ptr(idx), _ptr(val),
                                  _stream(stream)), "gl_best_particle")
    return idx, val


def gl_hmc_workspace_bytes(h, n):
    return lib().gl_hmc_workspace_bytes(h, int(n))


def gl_hmc_step(h, obs, noise_sigma, psf, z, logp, grad, l_tril, xi, log_u, system_id, step_size, n_leapfrog,
                out_accept, out_dh, workspace, stream=None):
    """One HMC transition of every chain (row of z); z, logp, grad are updated in place where the proposal is accepted."""
    torch = _torch()
    f32 = torch.float32
    _extents(h, z.shape[0], obs=obs, noise_sigma=noise_sigma, psf=psf, z=z, logp=logp, grad=grad, l_tril=l_tril, xi=xi, log_u=log_u,
             system_id=system_id, out_accept=out_accept, out_dh=out_dh)
    _check(lib().gl_hmc_step(h, _ptr(_dev(obs, f32, "obs")), _ptr(_dev(noise_sigma, f32, "noise_sigma")),
                             _ptr(_dev(psf, f32, "psf")), _ptr(_dev(z, f32, "z")), _ptr(_dev(logp, f32, "logp")),
                             _ptr(_dev(grad, f32, "grad")), _ptr(_dev(l_tril, f32, "l_tril")), _ptr(_dev(xi, f32, "xi")),
                             _ptr(_dev(log_u, f32, "log_u")), _ptr(_dev(system_id, torch.int32, "system_id")), z.shape[0],
                             float(step_size), int(n_leapfrog), _ptr(_dev(out_accept, torch.int32, "out_accept")),
                             _ptr(_dev(out_dh, f32, "out_dh")), _ptr(workspace),
                             workspace.numel() * workspace.element_size(), _stream(stream)), "gl_hmc_step")


def gl_svi_workspace_bytes(h, n):
    return lib().gl_svi_workspace_bytes(h, int(n))


def gl_svi_step(h, opt, obs, noise_sigma, psf, mu, l_tril, xi, system_id, opt_m, opt_v, step, out_stats, workspace,
                stream=None):
    """One SVI iteration; mu, l_tril (packed lower triangle), opt_m, opt_v are updated in place; xi: [n_draws][n_params]."""
    torch = _torch()
    f32 = torch.float32
    opt = _opt_desc(opt)
    _extents(h, xi.shape[0], obs=obs, noise_sigma=noise_sigma, psf=psf, mu=mu, l_tril=l_tril, xi=xi, system_id=system_id, svi_m=opt_m,
             svi_v=opt_v, out_stats=out_stats)
    _check(lib().gl_svi_step(h, C.byref(opt), _ptr(_dev(obs, f32, "obs")), _ptr(_dev(noise_sigma, f32, "noise_sigma")),
                             _ptr(_dev(psf, f32, "psf")), _ptr(_dev(mu, f32, "mu")), _ptr(_dev(l_tril, f32, "l_tril")),
                             _ptr(_dev(xi, f32, "xi")), _ptr(_dev(system_id, torch.int32, "system_id")), xi.shape[0],
                             _ptr(_dev(opt_m, f32, "opt_m")), _ptr(_dev(opt_v, f32, "opt_v")), int(step),
                             _ptr(_dev(out_stats, f32, "out_stats")), _ptr(workspace),
                             workspace.numel() * workspace.element_size(), _stream(stream)), "gl_svi_step")


def gl_svi_step_score(h, opt, obs, noise_sigma, psf, mu, l_tril, xi, system_id, opt_m, opt_v, step, baseline, out_stats,
                      workspace, stream=None):
    """One SVI iteration with the score-function gradient (Eq. 3 of the paper as printed; log p~ only, forward pass only);
    baseline 0 / 1: as printed / leave-one-out control variate.  Arguments otherwise as gl_svi_step."""
    torch = _torch()
    f32 = torch.float32
    opt = _opt_desc(opt)
    _extents(h, xi.shape[0], obs=obs, noise_sigma=noise_sigma, psf=psf, mu=mu, l_tril=l_tril, xi=xi, system_id=system_id, svi_m=opt_m,
             svi_v=opt_v, out_stats=out_stats)
    _check(lib().gl_svi_step_score(h, C.byref(opt), _ptr(_dev(obs, f32, "obs")), _ptr(_dev(noise_sigma, f32, "noise_sigma")),
                                   _ptr(_dev(psf, f32, "psf")), _ptr(_dev(mu, f32, "mu")), _ptr(_dev(l_tril, f32, "l_tril")),
                                   _ptr(_dev(xi, f32, "xi")), _ptr(_dev(system_id, torch.int32, "system_id")), xi.shape[0],
                                   _ptr(_dev(opt_m, f32, "opt_m")), _ptr(_dev(opt_v, f32, "opt_v")), int(step), int(baseline),
                                   _ptr(_dev(out_stats, f32, "out_stats")), _ptr(workspace),
                                   workspace.numel() * workspace.element_size(), _stream(stream)), "gl_svi_step_score")


def gl_model_image(h, psf, params, system_id, out_image, workspace, stream=None):
    torch = _torch()
    f32 = torch.float32
    n = params.shape[0]
    _extents(h, n, psf=psf, params=params, system_id=system_id, out_image=out_image)
    _check(lib().gl_model_image(h, _ptr(_dev(psf, f32, "psf")), _ptr(_dev(params, f32, "params")),
                                _ptr(_dev(system_id, torch.int32, "system_id")), n,
                                _ptr(_dev(out_image, f32, "out_image")), _ptr(workspace),
                                workspace.numel() * workspace.element_size(), _stream(stream)), "gl_model_image")


def gl_logpost_grad_host(h, obs, noise_sigma, psf, params_host, system_id, out_logp_host, out_grad_host, workspace,
                         stream=None):
    """params_host / out_*_host: CPU tensors (pinned for asynchrony); the rest on the device."""
    torch = _torch()
    f32 = torch.float32
    for t, nm in ((params_host, "params_host"), (out_logp_host, "out_logp_host"), (out_grad_host, "out_grad_host")):
        if t is not None and not (isinstance(t, torch.Tensor) and (not t.is_cuda) and t.dtype == f32 and t.is_contiguous()):
            raise TypeError("%s must be a contiguous CPU float32 tensor" % nm)
    n = params_host.shape[0]
    _extents(h, n, obs=obs, noise_sigma=noise_sigma, psf=psf, params=params_host, system_id=system_id, out_logp=out_logp_host,
             out_grad=out_grad_host)
    _check(lib().gl_logpost_grad_host(h, _ptr(_dev(obs, f32, "obs")), _ptr(_dev(noise_sigma, f32, "noise_sigma")),
                                      _ptr(_dev(psf, f32, "psf")), _ptr(params_host),
                                      _ptr(_dev(system_id, torch.int32, "system_id")), n, _ptr(out_logp_host),
                                      _ptr(out_grad_host), _ptr(workspace),
                                      workspace.numel() * workspace.element_size(), _stream(stream)),
           "gl_logpost_grad_host")


class LensModel:
    """A config handle plus device-resident observation and a cached workspace (the call a user makes)."""

    def __init__(self, spec, obs, noise_sigma, psf, device="cuda:0"):
        torch = _torch()
        self.spec = spec
        self.h = gl_config_create(spec)
        self.device = torch.device(device)
        as_dev = lambda a: torch.as_tensor(a, dtype=torch.float32).contiguous().to(self.device) if a is not None else None
        self.obs, self.noise_sigma, self.psf = as_dev(obs), as_dev(noise_sigma), as_dev(psf)
        self.n_params = lib().gl_config_n_params(self.h)
        self._ws = None

    def close(self):
        if self.h is not None:
            gl_config_destroy(self.h); self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def workspace(self, n, host=False):
        torch = _torch()
        need = gl_workspace_bytes_host(self.h, n) if host else gl_workspace_bytes(self.h, n)
        if self._ws is None or self._ws.numel() < need:
            self._ws = torch.empty(max(need, 256), dtype=torch.uint8, device=self.device)
        return self._ws

    def _sid(self, system_id):
        torch = _torch()
        if system_id is None:
            return None
        if not (isinstance(system_id, torch.Tensor) and system_id.is_cuda):      # host ids: range-check before the copy
            t = torch.as_tensor(system_id, dtype=torch.int32)
            if t.numel() and (int(t.min()) < 0 or int(t.max()) >= self.spec.n_systems):
                raise ValueError("system_id outside [0, n_systems)")
            return t.contiguous().to(self.device)
        return system_id.to(torch.int32).contiguous()

    def logpost(self, params, system_id=None, stream=None):
        torch = _torch()
        out = torch.empty(params.shape[0], dtype=torch.float32, device=self.device)
        gl_logpost(self.h, self.obs, self.noise_sigma, self.psf, params, self._sid(system_id), out,
                   self.workspace(params.shape[0]), stream)
        return out

    def linear_amplitudes(self, params, system_id=None, stream=None):
        """Backward modelling (amplitude_mode 1): (solved amplitudes [n][n_amp], logp [n])."""
        torch = _torch()
        n = params.shape[0]
        amp = torch.empty((n, gl_config_n_amplitudes(self.h)), dtype=torch.float32, device=self.device)
        lp = torch.empty(n, dtype=torch.float32, device=self.device)
        gl_linear_amplitudes(self.h, self.obs, self.noise_sigma, self.psf, params, self._sid(system_id), amp, lp,
                             self.workspace(n), stream)
        return amp, lp

    def logpost_grad(self, params, system_id=None, stream=None, out_logp=None, out_grad=None):
        torch = _torch()
        n = params.shape[0]
        lp = out_logp if out_logp is not None else torch.empty(n, dtype=torch.float32, device=self.device)
        g = out_grad if out_grad is not None else torch.empty((n, self.n_params), dtype=torch.float32, device=self.device)
        gl_logpost_grad(self.h, self.obs, self.noise_sigma, self.psf, params, self._sid(system_id), lp, g,
                        self.workspace(n), stream)
        return lp, g

    def capture_logpost_grad(self, params, system_id=None):
        """Capture one gl_logpost_grad call on `params` (a CUDA tensor that the caller updates IN PLACE between replays)
        into a CUDA graph: returns (replay, logp, grad) with replay() re-running the seven kernels as one graph launch into
        the same logp / grad tensors.  For small batches, where the launch gaps of the seven dependent kernels are a visible
        share of the call (config 1, 64 particles: 0.137 -> 0.129 ms per call)."""
        torch = _torch()
        n = params.shape[0]
        lp = torch.empty(n, dtype=torch.float32, device=self.device)
        g = torch.empty((n, self.n_params), dtype=torch.float32, device=self.device)
        sid, ws = self._sid(system_id), self.workspace(n)
        side = torch.cuda.Stream(device=self.device)
        side.wait_stream(torch.cuda.current_stream(self.device))
        graph = torch.cuda.CUDAGraph()
        with torch.cuda.stream(side):
            gl_logpost_grad(self.h, self.obs, self.noise_sigma, self.psf, params, sid, lp, g, ws, side)     # warm-up (attributes, lazy init)
            side.synchronize()
            with torch.cuda.graph(graph, stream=side):
                gl_logpost_grad(self.h, self.obs, self.noise_sigma, self.psf, params, sid, lp, g, ws, side)
        torch.cuda.current_stream(self.device).wait_stream(side)
        self._graphs = getattr(self, "_graphs", []) + [(graph, ws, sid)]       # keep the captured buffers alive
        return graph.replay, lp, g

    def map_run(self, params, opt, n_steps, system_id=None, first_step=1, state=None, stream=None):
        """n_steps fused MAP steps (gl_map_step) on `params` IN PLACE; no host synchronisation between steps.
        Returns (logp at the last evaluated params, (m, v) optimiser state)."""
        torch = _torch()
        n = params.shape[0]
        m, v = state if state is not None else (torch.zeros_like(params), torch.zeros_like(params))
        lp = torch.empty(n, dtype=torch.float32, device=self.device)
        g = torch.empty((n, self.n_params), dtype=torch.float32, device=self.device)
        sid, ws = self._sid(system_id), self.workspace(n)
        for t in range(first_step, first_step + n_steps):
            gl_map_step(self.h, opt, self.obs, self.noise_sigma, self.psf, params, sid, m, v, t, lp, g, ws, stream)
        return lp, (m, v)

    def svi_run(self, mu, l_tril, opt, n_steps, n_draws, seed, first_step=1, state=None, stream=None, estimator="pathwise"):
        """n_steps SVI iterations (gl_svi_step) on (mu, l_tril) IN PLACE with the draws made on the device
        (gl_draw_normal, stream_id 0, step = the iteration number): nothing crosses the host between iterations.
        estimator: "pathwise" (gl_svi_step), "score" (gl_svi_step_score with the leave-one-out baseline) or "score_printed"
        (Eq. 3 as printed, no baseline).  Returns (stats [n_steps][2] = (loss, finite draws) per iteration, (m, v) optimiser state)."""
        torch = _torch()
        n = self.n_params
        nt = n * (n + 1) // 2
        m, v = state if state is not None else (torch.zeros(n + nt, dtype=torch.float32, device=self.device),
                                                torch.zeros(n + nt, dtype=torch.float32, device=self.device))
        xi = torch.empty((n_draws, n), dtype=torch.float32, device=self.device)
        stats = torch.zeros((n_steps, 2), dtype=torch.float32, device=self.device)
        need = gl_svi_workspace_bytes(self.h, n_draws)
        ws = torch.empty(max(need, 256), dtype=torch.uint8, device=self.device)
        for k, t in enumerate(range(first_step, first_step + n_steps)):
            gl_draw_normal(seed, t, 0, xi, stream)
            if estimator == "pathwise":
                gl_svi_step(self.h, opt, self.obs, self.noise_sigma, self.psf, mu, l_tril, xi, None, m, v, t, stats[k], ws, stream)
            else:
                gl_svi_step_score(self.h, opt, self.obs, self.noise_sigma, self.psf, mu, l_tril, xi, None, m, v, t,
                                  0 if estimator == "score_printed" else 1, stats[k], ws, stream)
        return stats, (m, v)

    def hmc_run(self, z, l_tril, step_size, n_leapfrog, n_transitions, seed, first_step=1, system_id=None, stream=None):
        """n_transitions HMC transitions (gl_hmc_step) of the chains `z` IN PLACE, momenta and acceptance uniforms drawn
        on the device (gl_draw_normal stream_id 1, gl_draw_log_uniform stream_id 2, step = the transition number).
        Returns (logp, grad, accepted [n_transitions][n_chains] int32)."""
        torch = _torch()
        nc = z.shape[0]
        sid = self._sid(system_id)
        lp, g = self.logpost_grad(z, system_id, stream)
        xi = torch.empty((nc, self.n_params), dtype=torch.float32, device=self.device)
        lu = torch.empty(nc, dtype=torch.float32, device=self.device)
        acc = torch.zeros((n_transitions, nc), dtype=torch.int32, device=self.device)
        dh = torch.zeros(nc, dtype=torch.float32, device=self.device)
        ws = torch.empty(max(gl_hmc_workspace_bytes(self.h, nc), 256), dtype=torch.uint8, device=self.device)
        for k, t in enumerate(range(first_step, first_step + n_transitions)):
            gl_draw_normal(seed, t, 1, xi, stream)
            gl_draw_log_uniform(seed, t, 2, lu, stream)
            gl_hmc_step(self.h, self.obs, self.noise_sigma, self.psf, z, lp, g, l_tril, xi, lu, sid, step_size, n_leapfrog,
                        acc[k], dh, ws, stream)
        return lp, g, acc

    def model_image(self, params, system_id=None, stream=None):
        torch = _torch()
        n = params.shape[0]
        out = torch.empty((n, self.spec.n_pix, self.spec.n_pix), dtype=torch.float32, device=self.device)
        gl_model_image(self.h, self.psf, params, self._sid(system_id), out, self.workspace(n), stream)
        return out
