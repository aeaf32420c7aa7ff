"""ctypes front-end of the fp64 CPU oracle (oracle/gl_oracle.c).

TEST INFRASTRUCTURE ONLY: imported by tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
--impl reference legs, never by the product package.  It imports nothing from the product package.

A "spec" below is any object with the attributes of workloads.LensSpec (duck-typed; this module does
not import it): n_pix, supersample, psf_size, pix_scale, mass_model, epl_terms, has_shear,
multipole_mask, n_source_sersic, shapelet_nmax, n_lens_sersic, param_space, n_systems, n_params,
priors = sequence of (kind, a, b, lo, hi).
"""
import ctypes as C
import numpy as np

from . import build as _build

PRIOR_NONE, PRIOR_NORMAL, PRIOR_LOGNORMAL, PRIOR_UNIFORM, PRIOR_TRUNCNORMAL, PRIOR_LOGUNIFORM = range(6)


class _Prior(C.Structure):
    _fields_ = [("kind", C.c_int32), ("a", C.c_double), ("b", C.c_double), ("lo", C.c_double), ("hi", C.c_double)]


class _Config(C.Structure):
    _fields_ = [("n_pix", C.c_int32), ("supersample", C.c_int32), ("psf_size", C.c_int32),
                ("pix_scale", C.c_double),
                ("mass_model", C.c_int32), ("epl_terms", C.c_int32), ("has_shear", C.c_int32),
                ("multipole_mask", C.c_int32), ("n_source_sersic", C.c_int32), ("shapelet_nmax", C.c_int32),
                ("n_lens_sersic", C.c_int32), ("param_space", C.c_int32), ("n_systems", C.c_int32),
                ("n_params", C.c_int32), ("psf_grid", C.c_int32), ("noise_model", C.c_int32), ("t_exp", C.c_double),
                ("source2_plane", C.c_int32), ("priors", C.POINTER(_Prior))]


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(_build.build())
        dp = C.POINTER(C.c_double)
        L.glo_n_params.restype = C.c_int
        L.glo_logpost_grad.restype = C.c_int
        L.glo_logpost_grad.argtypes = [C.POINTER(_Config), dp, dp, dp, dp, C.POINTER(C.c_int32), C.c_int64,
                                       dp, dp, dp, dp]
        L.glo_transform_one.restype = C.c_int
        L.glo_transform_one.argtypes = [C.POINTER(_Prior), C.c_int32, C.c_double] + [dp] * 6
        L.glo_deflection.argtypes = [C.POINTER(_Config), dp, C.c_double, C.c_double, dp, dp]
        L.glo_epl_frame.argtypes = [C.c_double] * 5 + [C.c_int, dp]
        L.glo_sie_frame.argtypes = [C.c_double] * 4 + [dp]
        L.glo_sersic.restype = C.c_double
        L.glo_sersic.argtypes = [dp, C.c_double, C.c_double, dp, dp]
        L.glo_shapelets.restype = C.c_double
        L.glo_shapelets.argtypes = [C.c_int, dp, C.c_double, C.c_double, C.c_double, C.c_double, dp, dp]
        L.glo_shapelet_basis.argtypes = [C.c_int, C.c_double, dp]
        L.glo_ray_image.argtypes = [C.POINTER(_Config), dp, dp]
        L.glo_ray_coord.restype = C.c_double
        L.glo_ray_coord.argtypes = [C.POINTER(_Config), C.c_int]
        L.glo_conv_bin.argtypes = [C.c_int, C.c_int, C.c_int, C.c_double, dp, dp, dp]
        L.glo_conv_bin_transpose.argtypes = [C.c_int, C.c_int, C.c_int, C.c_double, dp, dp, dp]
        L.glo_bin_conv.argtypes = [C.c_int, C.c_int, C.c_int, C.c_double, dp, dp, dp]
        L.glo_bin_conv_transpose.argtypes = [C.c_int, C.c_int, C.c_int, C.c_double, dp, dp, dp]
        L.glo_num_threads.restype = C.c_int
        L.glo_set_num_threads.argtypes = [C.c_int]
        _lib = L
    return _lib


def _dp(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def _f64(a):
    return np.ascontiguousarray(np.asarray(a, dtype=np.float64))


def _make_config(spec, epl_terms=None, param_space=None):
    pri = (_Prior * len(spec.priors))()
    for i, (k, a, b, lo, hi) in enumerate(spec.priors):
        pri[i] = _Prior(int(k), float(a), float(b), float(lo), float(hi))
    cfg = _Config(spec.n_pix, spec.supersample, spec.psf_size, float(spec.pix_scale), spec.mass_model,
                  0 if epl_terms is None else int(epl_terms), spec.has_shear, spec.multipole_mask,
                  spec.n_source_sersic, spec.shapelet_nmax, spec.n_lens_sersic,
                  spec.param_space if param_space is None else int(param_space),
                  spec.n_systems, spec.n_params, int(getattr(spec, "psf_grid", 0)),
                  int(getattr(spec, "noise_model", 0)), float(getattr(spec, "t_exp", 1.0)),
                  int(getattr(spec, "source2_plane", 0)), pri)
    cfg._keep = pri
    return cfg


def n_threads():
    return lib().glo_num_threads()


def set_num_threads(n):
    lib().glo_set_num_threads(int(n))


def logpost_grad(spec, obs, sigma, psf, params, system_id=None, want_grad=True, want_gabs=False,
                 want_model=False, epl_terms=None, param_space=None):
    """log p~ (Eq. 2) and d/dz for each row of params.  The series is summed to convergence
    unless epl_terms is given (reading S5).  Returns dict(logp, grad, gabs, model)."""
    L = lib()
    cfg = _make_config(spec, epl_terms, param_space)
    assert L.glo_n_params(C.byref(cfg)) == spec.n_params, "n_params does not match the layout"
    params = _f64(params).reshape(-1, spec.n_params)
    P = params.shape[0]
    N, K = spec.n_pix, spec.psf_size
    obs = _f64(obs).reshape(-1, N, N); sigma = _f64(sigma).reshape(-1, N, N); psf = _f64(psf).reshape(-1, K, K)
    assert obs.shape[0] == spec.n_systems == sigma.shape[0] == psf.shape[0]
    sid = None
    if system_id is not None:
        sid = np.ascontiguousarray(np.asarray(system_id, dtype=np.int32))
        assert sid.shape == (P,) and (P == 0 or (sid.min() >= 0 and sid.max() < spec.n_systems))
    logp = np.empty(P)
    grad = np.empty((P, spec.n_params)) if want_grad else None
    gabs = np.empty((P, spec.n_params)) if (want_grad and want_gabs) else None
    model = np.empty((P, N, N)) if want_model else None
    null = C.POINTER(C.c_double)()
    rc = L.glo_logpost_grad(C.byref(cfg), _dp(obs), _dp(sigma), _dp(psf), _dp(params),
                            sid.ctypes.data_as(C.POINTER(C.c_int32)) if sid is not None else None, P,
                            _dp(logp), _dp(grad) if grad is not None else null,
                            _dp(gabs) if gabs is not None else null,
                            _dp(model) if model is not None else null)
    assert rc == 0, rc
    return dict(logp=logp, grad=grad, gabs=gabs, model=model)


def model_image(spec, psf, theta, epl_terms=None, system_id=None):
    """Noise-free model image(s) for PHYSICAL parameter rows theta (O3-O6); row i uses the PSF of system
    system_id[i] (default: system 0)."""
    N = spec.n_pix
    theta = _f64(theta).reshape(-1, spec.n_params)
    obs = np.zeros((spec.n_systems, N, N)); sig = np.ones((spec.n_systems, N, N))
    class _S:  # physical-space, prior-free view of the same spec
        pass
    s = _S(); s.__dict__.update({k: getattr(spec, k) for k in (
        "n_pix supersample psf_size pix_scale mass_model epl_terms has_shear multipole_mask n_source_sersic "
        "shapelet_nmax n_lens_sersic n_systems n_params").split()})
    s.psf_grid = int(getattr(spec, "psf_grid", 0))
    s.source2_plane = int(getattr(spec, "source2_plane", 0))
    s.param_space = 1
    s.priors = [(PRIOR_NONE, 0, 1, 0, 1)] * spec.n_params
    out = logpost_grad(s, obs, sig, psf, theta, system_id, want_grad=False, want_model=True, epl_terms=epl_terms)
    return out["model"]


def transform_one(prior, param_space, z):
    k, a, b, lo, hi = prior
    p = _Prior(int(k), float(a), float(b), float(lo), float(hi))
    o = [C.c_double() for _ in range(6)]
    ok = lib().glo_transform_one(C.byref(p), int(param_space), float(z), *[C.byref(x) for x in o])
    names = ("theta", "lp", "logdet", "dth_dz", "dlp_dth", "dlogdet_dz")
    d = {n: x.value for n, x in zip(names, o)}
    d["ok"] = bool(ok)
    return d


def deflection(spec, theta, x, y, epl_terms=None):
    cfg = _make_config(spec, epl_terms)
    th = _f64(theta)
    ax, ay = C.c_double(), C.c_double()
    lib().glo_deflection(C.byref(cfg), _dp(th), float(x), float(y), C.byref(ax), C.byref(ay))
    return ax.value, ay.value


def epl_frame(b, t, q, x, y, n_terms=0):
    out = np.empty(11)
    lib().glo_epl_frame(b, t, q, x, y, int(n_terms), _dp(out))
    return dict(alpha=complex(out[0], out[1]), d_b=complex(out[2], out[3]), d_t=complex(out[4], out[5]),
                d_q=complex(out[6], out[7]), J=(out[8], out[9], out[10]))


def sie_frame(b, q, x, y):
    out = np.empty(11)
    lib().glo_sie_frame(b, q, x, y, _dp(out))
    return dict(alpha=complex(out[0], out[1]), d_b=complex(out[2], out[3]), d_t=complex(out[4], out[5]),
                d_q=complex(out[6], out[7]), J=(out[8], out[9], out[10]))


def sersic(p, x, y, want_grad=False):
    p = _f64(p)
    if not want_grad:
        return lib().glo_sersic(_dp(p), float(x), float(y), None, None)
    dp, dxy = np.empty(7), np.empty(2)
    v = lib().glo_sersic(_dp(p), float(x), float(y), _dp(dp), _dp(dxy))
    return v, dp, dxy


def shapelets(nmax, p, x0, y0, x, y, want_grad=False):
    p = _f64(p)
    if not want_grad:
        return lib().glo_shapelets(int(nmax), _dp(p), x0, y0, x, y, None, None)
    da, dxy = np.empty(len(p)), np.empty(2)
    v = lib().glo_shapelets(int(nmax), _dp(p), x0, y0, x, y, _dp(da), _dp(dxy))
    return v, da, dxy


def shapelet_basis(nmax, u):
    phi = np.empty(nmax + 1)
    lib().glo_shapelet_basis(int(nmax), float(u), _dp(phi))
    return phi


def ray_image(spec, theta, epl_terms=None):
    cfg = _make_config(spec, epl_terms)
    M = spec.n_pix * spec.supersample
    out = np.empty((M, M)); th = _f64(theta)
    lib().glo_ray_image(C.byref(cfg), _dp(th), _dp(out))
    return out


def ray_coord(spec, idx):
    cfg = _make_config(spec)
    return lib().glo_ray_coord(C.byref(cfg), int(idx))


def conv_bin(n_pix, s, K, pix_scale, psf, ray):
    psf = _f64(psf); ray = _f64(ray); out = np.empty((n_pix, n_pix))
    lib().glo_conv_bin(n_pix, s, K, float(pix_scale), _dp(psf), _dp(ray), _dp(out))
    return out


def bin_conv(n_pix, s, K, pix_scale, psf, ray):
    """psf_grid = 1: bin to detector pixels, then convolve with the PSF sampled at the pixel scale."""
    psf = _f64(psf); ray = _f64(ray); out = np.empty((n_pix, n_pix))
    lib().glo_bin_conv(n_pix, s, K, float(pix_scale), _dp(psf), _dp(ray), _dp(out))
    return out


def bin_conv_transpose(n_pix, s, K, pix_scale, psf, g):
    psf = _f64(psf); g = _f64(g); M = n_pix * s; out = np.empty((M, M))
    lib().glo_bin_conv_transpose(n_pix, s, K, float(pix_scale), _dp(psf), _dp(g), _dp(out))
    return out


def conv_bin_transpose(n_pix, s, K, pix_scale, psf, g):
    psf = _f64(psf); g = _f64(g); M = n_pix * s; out = np.empty((M, M))
    lib().glo_conv_bin_transpose(n_pix, s, K, float(pix_scale), _dp(psf), _dp(g), _dp(out))
    return out
