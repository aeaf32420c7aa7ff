"""Seeded synthetic inputs for the five BASELINE.json configs (recipe: DESIGN.md section 4, from
SURVEY.md 8(d)).  Serves BOTH the oracle-side tests and the CUDA-side tests/bench; holds none of the
method's arithmetic (no ray-tracing, no light profile, no convolution, no likelihood): it only draws
numbers, builds PSF tap tables, and lists the model configuration.  The observed image needs a renderer,
so it is finished by the caller (`finish_observation`) from a truth image the caller rendered with its
own side (tests: the oracle; bench GPU arm: gl_model_image; bench cpu_baseline: the oracle).

Stand-in statement: the paper measures on its own 100 simulated systems and on an
HST image (L305); neither is available, so these inputs take their shapes, sizes and value
distributions (Eq. 4) and stand in for them.

All draws are made in fp64 from numpy PCG64 streams spawned from SeedSequence(20260630 + k), in the order
truth / noise / particles / psf, then ROUNDED ONCE to fp32; the rounded arrays are the definition and are
what both sides consume (reading S20).
"""
from dataclasses import dataclass, field
import math
import numpy as np

PRIOR_NONE, PRIOR_NORMAL, PRIOR_LOGNORMAL, PRIOR_UNIFORM, PRIOR_TRUNCNORMAL, PRIOR_LOGUNIFORM = range(6)


def _r32(x):
    return float(np.float32(x))


def Normal(mu, sd):            return (PRIOR_NORMAL, _r32(mu), _r32(sd), 0.0, 0.0)
def LogNormal(mu, sd):         return (PRIOR_LOGNORMAL, _r32(mu), _r32(sd), 0.0, 0.0)
def Uniform(lo, hi):           return (PRIOR_UNIFORM, 0.0, 1.0, _r32(lo), _r32(hi))
def TruncNormal(mu, sd, lo, hi): return (PRIOR_TRUNCNORMAL, _r32(mu), _r32(sd), _r32(lo), _r32(hi))
def LogUniform(lo, hi):        return (PRIOR_LOGUNIFORM, 0.0, 1.0, _r32(lo), _r32(hi))
def NoPrior():                 return (PRIOR_NONE, 0.0, 1.0, 0.0, 0.0)


@dataclass
class LensSpec:
    """Model configuration; field names follow include/gigalens.h `gl_config_desc`."""
    n_pix: int
    supersample: int
    psf_size: int
    pix_scale: float
    mass_model: int = 1          # 0 SIE, 1 EPL
    epl_terms: int = 30
    has_shear: int = 1
    multipole_mask: int = 0      # bit0 m=3, bit1 m=4
    n_source_sersic: int = 1      # 0, 1 or 2 (same source plane)
    shapelet_nmax: int = -1
    n_lens_sersic: int = 1
    param_space: int = 0         # 0 unconstrained z, 1 physical theta
    n_systems: int = 1
    psf_grid: int = 0            # 0: PSF taps on the ray grid (S10); 1: on the detector grid (NEXT-4, S10b)
    noise_model: int = 0         # 0: fixed sigma map (S12); 1: variance sigma^2 + max(model,0)/t_exp (NEXT-4, S12b)
    t_exp: float = 1.0           # exposure time of noise_model 1
    amplitude_mode: int = 0      # 0: amplitudes sampled ("forward"); 1: solved by linear inversion ("backward", NEXT-4, S21)
    source2_plane: int = 0       # 1: the second source Sersic on its own source plane, one more parameter eta2 (NEXT-4, S23)
    precision: int = 0           # 0 GL_PRECISION_F64, 1 GL_PRECISION_F32 (CUDA path only; the oracle is always fp64)
    priors: list = field(default_factory=list)
    names: list = field(default_factory=list)

    @property
    def n_params(self):
        return len(self.priors)

    @property
    def n_rays(self):
        return self.n_pix * self.supersample


def n_shapelet_coef(nmax):
    return (nmax + 1) * (nmax + 2) // 2 if nmax >= 0 else 0


def param_names(mass_model, has_shear, multipole_mask, n_source_sersic, shapelet_nmax, n_lens_sersic, source2_plane=0):
    """Flat parameter order (reading S18)."""
    n = ["theta_E"] + (["gamma"] if mass_model == 1 else []) + ["e1", "e2", "x", "y"]
    n = ["mass." + s for s in n]
    if has_shear: n += ["shear.g1", "shear.g2"]
    if multipole_mask & 1: n += ["mp.c3", "mp.s3"]
    if multipole_mask & 2: n += ["mp.c4", "mp.s4"]
    ser = ["R", "n", "e1", "e2", "x", "y", "I"]
    if n_source_sersic: n += ["src." + s for s in ser]
    if n_source_sersic > 1: n += ["src2." + s for s in ser]          # second source (S1, S2)
    if n_source_sersic > 1 and source2_plane: n += ["src2.eta"]      # ... on its own plane: deflection scale eta2 (S23)
    if shapelet_nmax >= 0: n += ["shp.beta"] + ["shp.a%d" % i for i in range(n_shapelet_coef(shapelet_nmax))]
    for k in range(n_lens_sersic): n += ["ll%d." % k + s for s in ser]
    return n


# ------------------------------------------------------------------ priors of each config
def _default_priors(mass_model, multipoles=False, shapelet_nmax=-1, n_lens=1, n_src=1, src2_plane=False):
    """SURVEY 8(d) fill-ins for configs 1, 2, 3, 5 (BJ configs[0..2], [4])."""
    p = [Uniform(0.8, 1.5)]
    if mass_model == 1: p += [Uniform(1.6, 2.4)]
    p += [Normal(0, 0.1), Normal(0, 0.1), Normal(0, 0.05), Normal(0, 0.05)]
    p += [Normal(0, 0.05), Normal(0, 0.05)]
    if multipoles: p += [Normal(0, 0.01)] * 4
    p += [Uniform(0.1, 0.5), Uniform(1, 4), Normal(0, 0.15), Normal(0, 0.15), Normal(0, 0.2), Normal(0, 0.2),
          LogUniform(1, 100)]
    if n_src > 1:
        p += [Uniform(0.1, 0.5), Uniform(1, 4), Normal(0, 0.15), Normal(0, 0.15), Normal(0.3, 0.2), Normal(-0.2, 0.2),
              LogUniform(1, 100)]
        if src2_plane: p += [Uniform(0.6, 1.6)]                      # eta2: ratio of the lensing efficiencies of the two planes
    if shapelet_nmax >= 0: p += [Uniform(0.05, 0.3)] + [Normal(0, 1)] * n_shapelet_coef(shapelet_nmax)
    for _ in range(n_lens):
        p += [Uniform(0.5, 1.5), Uniform(2, 6), TruncNormal(0, 0.1, -0.15, 0.15), TruncNormal(0, 0.1, -0.15, 0.15),
              Normal(0, 0.02), Normal(0, 0.02), LogUniform(1, 100)]
    return p


def _eq4(which):
    """Eq. 4 of the paper, 'a / b' = simulation / modelling prior; which = 0 or 1.
    Garbled rows read as S17: the 'ln 300' row is I_l; R_s row lost -> exp N(ln 0.25, 0.15/0.25)."""
    w = which
    return [LogNormal(math.log(1.25), (0.25, 0.4)[w]), TruncNormal(2, (0.25, 0.5)[w], 1, 3),
            Normal(0, (0.1, 0.2)[w]), Normal(0, (0.1, 0.2)[w]), Normal(0, (0.03, 0.06)[w]), Normal(0, (0.03, 0.06)[w]),
            Normal(0, (0.05, 0.1)[w]), Normal(0, (0.05, 0.1)[w]),
            # source Sersic
            LogNormal(math.log(0.25), (0.15, 0.25)[w]), Uniform(0.5, (4, 8)[w]),
            TruncNormal(0, (0.15, 0.3)[w], -0.5, 0.5), TruncNormal(0, (0.15, 0.3)[w], -0.5, 0.5),
            Normal(0, (0.25, 0.5)[w]), Normal(0, (0.25, 0.5)[w]), LogNormal(math.log(150), (0.5, 0.9)[w]),
            # lens light Sersic
            LogNormal(math.log(1.6), (0.15, 0.25)[w]), Uniform((2, 0.5)[w], (6, 8)[w]),
            TruncNormal(0, (0.05, 0.1)[w], -0.15, 0.15), TruncNormal(0, (0.05, 0.1)[w], -0.15, 0.15),
            Normal(0, (0.01, 0.02)[w]), Normal(0, (0.01, 0.02)[w]), LogNormal(math.log(300), (0.3, 0.5)[w])]


def make_spec(k, **over):
    """LensSpec of BASELINE.json configs[k-1], k = 1..5; k = 6 (not a BASELINE.json config): the component list of the
    paper's real-system model (mass + shear, env / L1 / L2 lens light, S1 / S2 sources; 43 parameters,
    38 when the amplitudes are solved) on the geometry, PSF and noise recipe of config 2."""
    if k == 1:
        s = LensSpec(40, 2, 11, _r32(0.262), mass_model=0, priors=_default_priors(0))
    elif k == 2:
        s = LensSpec(60, 4, 21, _r32(0.262), priors=_default_priors(1))
    elif k == 3:
        s = LensSpec(100, 2, 31, _r32(0.065), shapelet_nmax=6, n_lens_sersic=2,
                     priors=_default_priors(1, shapelet_nmax=6, n_lens=2))
    elif k == 4:
        s = LensSpec(60, 4, 21, _r32(0.262), n_systems=100, priors=_eq4(1))
    elif k == 5:
        s = LensSpec(200, 4, 41, _r32(0.04), multipole_mask=3, shapelet_nmax=10, n_lens_sersic=2,
                     priors=_default_priors(1, multipoles=True, shapelet_nmax=10, n_lens=2))
    elif k == 6:
        s = LensSpec(60, 4, 21, _r32(0.262), n_source_sersic=2, n_lens_sersic=3,
                     priors=_default_priors(1, n_lens=3, n_src=2))
    else:
        raise ValueError(k)
    for a, v in over.items():
        setattr(s, a, v)
    s.names = param_names(s.mass_model, s.has_shear, s.multipole_mask, s.n_source_sersic, s.shapelet_nmax,
                          s.n_lens_sersic, s.source2_plane)
    assert len(s.names) == s.n_params, (len(s.names), s.n_params)
    return s


FULL_PARTICLES = {1: 64, 2: 4096, 3: 8192, 4: 102400, 5: 2048, 6: 4096}
PARITY_PARTICLES = {1: 64, 2: 256, 3: 128, 4: 400, 5: 16, 6: 64}     # SURVEY 8(d) parity subsets


# ------------------------------------------------------------------ sampling and the inverse bijector
def sample_prior(rng, prior, size=None):
    k, a, b, lo, hi = prior
    if k == PRIOR_NORMAL: return rng.normal(a, b, size)
    if k == PRIOR_LOGNORMAL: return np.exp(rng.normal(a, b, size))
    if k == PRIOR_UNIFORM: return rng.uniform(lo, hi, size)
    if k == PRIOR_LOGUNIFORM: return np.exp(rng.uniform(math.log(lo), math.log(hi), size))
    if k == PRIOR_TRUNCNORMAL:
        n = 1 if size is None else int(np.prod(size))
        out = np.empty(n); i = 0
        while i < n:                                   # plain rejection
            d = rng.normal(a, b, 2 * (n - i) + 8)
            d = d[(d > lo) & (d < hi)][: n - i]
            out[i:i + len(d)] = d; i += len(d)
        return out[0] if size is None else out.reshape(size)
    raise ValueError(k)


def to_unconstrained(prior, theta):
    """z = T^-1(theta) for the bijector family of `prior` (reading S13)."""
    k, a, b, lo, hi = prior
    theta = np.asarray(theta, dtype=np.float64)
    if k in (PRIOR_NONE, PRIOR_NORMAL): return theta
    if k == PRIOR_LOGNORMAL: return np.log(theta)
    if k in (PRIOR_UNIFORM, PRIOR_TRUNCNORMAL):
        u = (theta - lo) / (hi - lo); return np.log(u) - np.log1p(-u)
    if k == PRIOR_LOGUNIFORM:
        u = (np.log(theta) - math.log(lo)) / (math.log(hi) - math.log(lo)); return np.log(u) - np.log1p(-u)
    raise ValueError(k)


def to_physical(prior, z):
    """theta = T(z), fp64; used only to hand a physical truth vector to a renderer."""
    k, a, b, lo, hi = prior
    z = np.asarray(z, dtype=np.float64)
    sg = 1.0 / (1.0 + np.exp(-z))
    if k in (PRIOR_NONE, PRIOR_NORMAL): return z
    if k == PRIOR_LOGNORMAL: return np.exp(z)
    if k in (PRIOR_UNIFORM, PRIOR_TRUNCNORMAL): return lo + (hi - lo) * sg
    if k == PRIOR_LOGUNIFORM: return np.exp(math.log(lo) + (math.log(hi) - math.log(lo)) * sg)
    raise ValueError(k)


def draw(rng, priors, n):
    return np.stack([sample_prior(rng, p, n) for p in priors], axis=1)


def z_of(priors, theta):
    theta = np.atleast_2d(theta)
    return np.stack([to_unconstrained(p, theta[:, i]) for i, p in enumerate(priors)], axis=1)


def theta_of(priors, z):
    z = np.atleast_2d(z)
    return np.stack([to_physical(p, z[:, i]) for i, p in enumerate(priors)], axis=1)


# ------------------------------------------------------------------ PSF tap tables (taps at ray spacing, S10)
def _tap_grid(K, step):
    c = (K - 1) // 2
    ax = (np.arange(K) - c) * step
    return np.meshgrid(ax, ax, indexing="xy")


def gaussian_psf(K, fwhm, step):
    x, y = _tap_grid(K, step)
    sd = fwhm / 2.35482
    p = np.exp(-0.5 * (x * x + y * y) / (sd * sd))
    return p / p.sum()


def moffat_psf(K, fwhm, beta_m, step):
    x, y = _tap_grid(K, step)
    a = fwhm / (2.0 * math.sqrt(2.0 ** (1.0 / beta_m) - 1.0))
    p = (1.0 + (x * x + y * y) / (a * a)) ** (-beta_m)
    return p / p.sum()


# ------------------------------------------------------------------ workloads
@dataclass
class Workload:
    k: int
    spec: LensSpec
    psf: np.ndarray          # [n_systems, K, K] float32
    truth_z: np.ndarray      # [n_systems, n_params] float32 (unconstrained)
    truth_theta: np.ndarray  # [n_systems, n_params] float64 = T(float64(truth_z)), for a renderer
    params: np.ndarray       # [P, n_params] float32, unconstrained z
    system_id: np.ndarray    # [P] int32 or None
    noise_unit: np.ndarray   # [n_systems, N, N] float64 standard-normal draws
    sigma_bkg: float
    t_exp: float             # 0: constant sigma map; >0: sigma^2 = sigma_bkg^2 + max(truth,0)/t_exp


def make_workload(k, n_particles=None, per_system=None):
    """Config k at `n_particles` particles (default: the full BASELINE.json batch).  For config 4,
    `per_system` positions per system (default 1024), all 100 systems, system-major.  A smaller batch is
    a PREFIX of the full one for configs 1-3 and 5 (same stream), so parity subsets are bench inputs."""
    spec = make_spec(k)
    ss = np.random.SeedSequence(20260630 + k)
    s_truth, s_noise, s_part, s_psf = [np.random.Generator(np.random.PCG64(s)) for s in ss.spawn(4)]
    N, K, nsys = spec.n_pix, spec.psf_size, spec.n_systems
    step = spec.pix_scale / spec.supersample
    # truth
    truth_priors = _eq4(0) if k == 4 else spec.priors
    truth_theta = draw(s_truth, truth_priors, nsys)
    truth_z = z_of(spec.priors, truth_theta).astype(np.float32)
    truth_theta = theta_of(spec.priors, truth_z.astype(np.float64))          # T of the ROUNDED z
    noise_unit = s_noise.standard_normal((nsys, N, N))
    # psf
    if k == 1:   psf = gaussian_psf(K, 1.1, step)[None]
    elif k in (2, 6): psf = moffat_psf(K, 1.2, 3.0, step)[None]
    elif k == 3: psf = gaussian_psf(K, 0.1, step)[None]
    elif k == 4:
        fw = s_psf.uniform(1.0, 1.5, nsys); bm = s_psf.uniform(2.5, 4.0, nsys)
        psf = np.stack([moffat_psf(K, fw[i], bm[i], step) for i in range(nsys)])
    else:
        psf = (0.8 * gaussian_psf(K, 0.08, step) + 0.2 * moffat_psf(K, 0.16, 2.5, step))[None]
    psf = psf.astype(np.float32)
    # particles
    system_id = None
    if k in (1, 2, 5, 6):
        P = FULL_PARTICLES[k] if n_particles is None else n_particles
        z = z_of(spec.priors, draw(s_part, spec.priors, FULL_PARTICLES[k]))[:P]
    elif k == 3:
        P = FULL_PARTICLES[k] if n_particles is None else n_particles
        z = (truth_z[0].astype(np.float64) + 0.02 * s_part.standard_normal((FULL_PARTICLES[k], spec.n_params)))[:P]
    else:
        per = 1024 if per_system is None else per_system
        full = truth_z.astype(np.float64)[:, None, :] + 0.02 * s_part.standard_normal((nsys, 1024, spec.n_params))
        z = full[:, :per, :].reshape(nsys * per, spec.n_params)
        system_id = np.repeat(np.arange(nsys, dtype=np.int32), per)
    sigma_bkg = {1: 0.05, 2: 0.02, 3: 0.01, 4: 0.05, 5: 0.005, 6: 0.02}[k]
    t_exp = {1: 0.0, 2: 1000.0, 3: 0.0, 4: 1000.0, 5: 0.0, 6: 1000.0}[k]
    return Workload(k, spec, psf, truth_z, truth_theta, np.ascontiguousarray(z.astype(np.float32)), system_id,
                    noise_unit, sigma_bkg, t_exp)


def finish_observation(wl, truth_image):
    """(obs, noise_sigma), both [n_systems, N, N] float32, from the caller-rendered noise-free truth image(s).
    sigma^2 = sigma_bkg^2 + max(truth, 0)/t_exp (configs 2, 4: the 'Poisson-like variance term' baked into a
    FIXED map, reading S12); obs = truth + sigma * unit normal."""
    t = np.asarray(truth_image, dtype=np.float64).reshape(wl.noise_unit.shape)
    var = np.full_like(t, wl.sigma_bkg ** 2)
    if wl.t_exp > 0: var = var + np.maximum(t, 0.0) / wl.t_exp
    sigma = np.sqrt(var).astype(np.float32)
    obs = (t + sigma.astype(np.float64) * wl.noise_unit).astype(np.float32)
    return obs, sigma
