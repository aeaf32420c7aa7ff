"""Frozen algorithmic work model of the hot path (SURVEY 8(d) "Algorithmic work per evaluation").

Counts are FP32 lane-operations with an FMA counted ONCE (add, mul and fma each count 1; min/max, selects,
integer and address arithmetic count 0) and MUFU operations separately, per ray, for the formulation the
kernels implement (csrc/gl_ray.cuh): the EPL series as a real-coefficient polynomial in w evaluated by
synthetic division (2 FMA per term, not the 6 of complex Horner that SURVEY 8(d) assumed), Sersic via
lg2/ex2, shapelets by the three-term recurrence.  They are hand counts of the formulas, frozen before timing;
recomputation of the forward inside the adjoint kernel is NOT credited (one forward sweep + one reverse sweep).
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
    "shapelet_fixed": (22, 0),    # u, v, two Gaussians through exp2
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
    return 4 * (nmax + 1) + 2 * ncoef + 2 * (nmax + 1) + ncoef     # derivatives, d/du d/dv contractions, coefficient sums


def per_ray(spec, precision="f32"):
    """(fwd lane-ops, fwd mufu, adjoint-sweep lane-ops, adjoint-sweep mufu) per ray for a LensSpec-like object;
    precision "f32": FP32 lane-ops + MUFU, "f64": FP64 lane-ops (mufu = 0)."""
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
    return f, m, a, am


def per_eval(spec, precision="f32"):
    """Algorithmic lane-ops (FP32 or FP64, by `precision`) of one particle evaluation, by stage, for gl_logpost_grad."""
    M = spec.n_pix * spec.supersample
    rays = M * M
    f, m, a, am = per_ray(spec, precision)
    ke = spec.psf_size + spec.supersample - 1
    conv = spec.n_pix * spec.n_pix * ke * ke              # stride-s correlation with the pre-boxed kernel (step D)
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
    }
