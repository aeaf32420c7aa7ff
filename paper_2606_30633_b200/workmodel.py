"""Frozen algorithmic work model of the hot path (SURVEY 8(d) "Algorithmic work per evaluation").

Counts are lane-operations with an FMA counted ONCE (add, mul and fma each count 1; min/max, selects, integer and
address arithmetic count 0) and MUFU operations separately, per ray, for the formulation the kernels implement
(csrc/gl_ray.cuh): the EPL series as a real-coefficient polynomial in w evaluated by synthetic division (2 FMA per
term, not the 6 of complex Horner that SURVEY 8(d) assumed), Sersic via lg2/ex2, shapelets by the three-term
recurrence.  They are hand counts of the formulas, frozen before timing.

Two things a reader must not confuse (round-1 review):
  * "ray_adjoint" is what the adjoint KERNEL must do: it recomputes steps B + C per ray (nothing is taped), so its
    count is forward + reverse sweep; the whole-step figure "total_fwd_grad" credits ONE forward and ONE reverse sweep
    (the recompute is not credited twice).
  * the series count comes in two forms.  `bands=None`: the fixed 30-term formulation, every term in the arithmetic
    type (the `frac_fixed30` of bench.py).  `bands=(m1, m2)` (batch means of what step A chose per particle, read back
    from the workspace): only the 4 m1 recurrence steps that DO run in the arithmetic type are credited to its pipe;
    the 4 m2 steps that the fp64 mode runs in fp32 on the FP32 pipe are returned separately ("*_fp32band") and the
    terms beyond 4 (m1 + m2) + 1, which are numerically zero and skipped, are credited to nobody.
This module holds no arithmetic of the method; bench.py uses it to turn a measured time into a roofline fraction.
"""

# primitive -> (fp32 lane-ops, mufu) per ray
FWD = {
    "frame":          (15, 1),    # centre, rotate, q x, R^2, 1/R, unit vector, cos/sin 2phi, w, p
    "epl_series":     (63, 0),    # 28 synthetic-division steps x 2 FMA + tail 3 + E * P(w) 4
    "epl_amp":        (6, 2),     # lg2 R^2, (b/R)^(t-1) via ex2, amplitude, 2 components
    "sie_closed":     (40, 4),    # atan + atanh (polynomial + rcp/lg2), prefactors
    "rotate_shear":   (12, 0),    # rotate back, shear, lab coordinates
    "multipoles":     (30, 1),    # m = 3 and 4 from the unit vector
    "sersic":         (15, 3),    # position, rotate, r^2, lg2, ex2 (u), ex2 (I)
    "shapelet_fixed": (8, 2),     # u, v, two Gaussians
    "sum":            (1, 0),
}
# extra work of the reverse sweep, per ray
ADJ = {
    "epl_series":     (134, 0),   # two more 27-step polynomials (S1, S2) and their rotations
    "mass_chain":     (77, 1),    # Jacobian from kappa/Gamma, projections onto the 9 natural mass sums
    "sie_chain":      (40, 0),
    "multipoles":     (40, 0),
    "sersic":         (15, 1),    # 8 natural sums + radial factor
    "sersic_src_grad": (8, 0),    # source-plane gradient of the source Sersic
    "shapelet_fixed": (20, 0),
}


# GL_PRECISION_F64: the same formulation on the FP64 pipe.  Counts are FP64 lane-operations (DFMA, DMUL and DADD
# count 1 each; compares, selects, integer and FP32/MUFU seed instructions count 0).  exp2 = 8 (split 3, degree-4
# polynomial 3, table product 2), log2 = 7, rsqrt = 4, rcp = 2 (csrc/gl_math.cuh).  Hand counts of csrc/gl_ray.cuh,
# cross-checked against the SASS loop bodies of the config-2 kernels; revised downward whenever the formulation got
# cheaper (round 1: 195 -> 187 forward operations per config-2 ray), never for work moved to the FP32 pipe.
FWD64 = {
    "frame":          (22, 0),    # 18 arithmetic + rsqrt 4
    "epl_series":     (63, 0),
    "epl_amp":        (20, 0),    # log2 7 + exp2 8 (A and b folded into the exponent) + 5
    "sie_closed":     (120, 0),   # libdevice atan + atanh (config 1 only; latency-bound, not rooflined)
    "rotate_shear":   (10, 0),    # two 4-FMA chains + the two lab coordinates
    "multipoles":     (34, 0),
    "sersic":         (36, 0),    # 13 arithmetic (pre-scaled frame) + log2 7 + 2 exp2 16
    "shapelet_fixed": (13, 0),    # u, v, ONE Gaussian of u^2 + v^2 through exp2 (scaled basis, round 2; was 22 with two Gaussians)
    "sum":            (0, 0),     # folded into the component counts
}
ADJ64 = {
    "epl_series":     (130, 0),
    "mass_chain":     (75, 0),    # includes rcp 2
    "sie_chain":      (45, 0),
    "multipoles":     (40, 0),
    "sersic":         (17, 0),    # 8 natural sums + radial factor + rcp
    "sersic_src_grad": (8, 0),
    "shapelet_fixed": (20, 0),
}


def shapelet_fwd(nmax):
    ncoef = (nmax + 1) * (nmax + 2) // 2
    return 4 * nmax + ncoef + (nmax + 1)          # two recurrences (2 ops/step each) + triangular contraction


def shapelet_adj(nmax):
    ncoef = (nmax + 1) * (nmax + 2) // 2
    # scaled basis (round 2): a derivative is ONE operation, (k/2) psi_{k-1} - psi_{k+1} with the product shared with the
    # recurrence, which runs one step further per family (4 operations); was 4 (nmax + 1) for the derivatives
    return 2 * (nmax + 1) + 4 + 2 * ncoef + 2 * (nmax + 1) + ncoef   # derivatives, d/du d/dv contractions, coefficient sums


# EPL series by band (csrc/gl_ray.cuh knuth_banded): one polynomial = 4 m recurrence steps of 2 FMA + a tail of 7 (fwd:
# 3 + the rotation E * P(w) 4); the reverse sweep adds two more polynomials (2 x 8 m) + 18 of tails and rotations.  The
# fixed 30-term figures above are m = 7: 8 * 7 + 7 = 63 and 2 * 56 + 18 = 130 (134 in fp32: 4 more in the rotations).
SERIES_M_FULL = 7


def series_ops(m, precision):
    """(forward, reverse-sweep extra) lane-ops of the series with 4 m recurrence steps per polynomial."""
    tail_adj = 18 if precision == "f64" else 22
    return 8.0 * m + 7.0, 16.0 * m + tail_adj


def per_ray(spec, precision="f32", bands=None):
    """(fwd lane-ops, fwd mufu, adjoint-sweep lane-ops, adjoint-sweep mufu, fwd fp32-band ops, adjoint fp32-band ops)
    per ray for a LensSpec-like object; precision "f32": FP32 lane-ops + MUFU, "f64": FP64 lane-ops (mufu = 0).
    bands = (mean m1, mean m2) or None for the fixed 30-term count (module docstring)."""
    f = m = a = am = 0
    F_, A_ = (FWD64, ADJ64) if precision == "f64" else (FWD, ADJ)

    def add(tab, key, times=1):
        nonlocal f, m, a, am
        if tab is FWD:
            f += F_[key][0] * times; m += F_[key][1] * times
        else:
            a += A_[key][0] * times; am += A_[key][1] * times

    add(FWD, "frame"); add(FWD, "rotate_shear"); add(FWD, "sum")
    if spec.mass_model == 1:
        add(FWD, "epl_series"); add(FWD, "epl_amp"); add(ADJ, "epl_series"); add(ADJ, "mass_chain")
    else:
        add(FWD, "sie_closed"); add(ADJ, "sie_chain"); add(ADJ, "mass_chain")
    if spec.multipole_mask:
        add(FWD, "multipoles"); add(ADJ, "multipoles")
    nser = spec.n_source_sersic + spec.n_lens_sersic
    add(FWD, "sersic", nser); add(ADJ, "sersic", nser)
    if spec.n_source_sersic:
        add(ADJ, "sersic_src_grad", spec.n_source_sersic)
    if spec.shapelet_nmax >= 0:
        add(FWD, "shapelet_fixed"); add(ADJ, "shapelet_fixed")
        f += shapelet_fwd(spec.shapelet_nmax); a += shapelet_adj(spec.shapelet_nmax)
    f32f = f32a = 0.0
    if bands is not None and spec.mass_model == 1:
        m1, m2 = bands
        full_f, full_a = series_ops(SERIES_M_FULL, precision)
        got_f, got_a = series_ops(m1, precision)
        f += got_f - full_f; a += got_a - full_a
        if precision == "f64":
            f32f, f32a = 8.0 * m2, 16.0 * m2
    return f, m, a, am, f32f, f32a


def per_eval(spec, precision="f32", bands=None):
    """Algorithmic lane-ops (FP32 or FP64, by `precision`) of one particle evaluation, by stage, for gl_logpost_grad.
    bands: see per_ray."""
    M = spec.n_pix * spec.supersample
    rays = M * M
    f, m, a, am, f32f, f32a = per_ray(spec, precision, bands)
    ke = spec.psf_size + spec.supersample - 1
    conv = spec.n_pix * spec.n_pix * ke * ke              # stride-s correlation with the pre-boxed kernel (step D)
    if getattr(spec, "psf_grid", 0) == 1:                 # bin (s^2 adds per pixel), then K x K taps at the pixel scale
        conv = spec.n_pix * spec.n_pix * (spec.psf_size ** 2 + spec.supersample ** 2)
    return {
        "rays": rays,
        "ray_fwd": f * rays, "ray_fwd_mufu": m * rays,
        "conv_chi2": conv + 4 * spec.n_pix * spec.n_pix,
        "conv_transpose": conv,
        "ray_adjoint": (f + a) * rays,                     # what the adjoint KERNEL must do (it recomputes B+C)
        "ray_adjoint_mufu": (m + am) * rays,
        "total_fwd": f * rays + conv,
        "total_fwd_grad": (f + a) * rays + 2 * conv,       # one forward + one reverse sweep; recompute not credited
        "total_fwd_grad_mufu": (m + am) * rays,
        # fp64 mode only: series steps that run in fp32 on the FP32 pipe (not part of the figures above)
        "ray_fwd_fp32band": f32f * rays, "ray_adjoint_fp32band": (f32f + f32a) * rays,
        "total_fwd_grad_fp32band": (f32f + f32a) * rays,
    }
