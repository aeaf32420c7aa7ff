/*
 * gl_oracle.c -- fp64 CPU ORACLE for the GIGA-Lens batched log-posterior and its gradient.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and the
 * cpu_baseline / --impl reference legs of bench.py may build, link, import or call it.  It shares no
 * code, header, table or constant with the CUDA path (paper_2606_30633_b200/csrc) and never will.
 *
 * What it is: the plain definition, step by step, in double precision, of
 *   log p~(I_obs, Theta~)  (Eq. 2: the log joint in unconstrained space) and its
 *   gradient ("backpropagation for gradient evaluation", L62, L98)
 * for the model the paper names at PAPER.md L64 (EPL + external shear mass; Sersic / shapelet source
 * light; Sersic lens light; "forward" amplitudes), on the supersampled grid of PAPER.md L189 (fn 6).
 * The paper gives no formula for any ingredient (it defers to G22 / Birrer+15 / lenstronomy, none of
 * which is available); every formula below is the standard one for the named profile under the
 * readings S1-S20 of SURVEY.md section 8(c), restated in DESIGN.md section 3.  No blocking, fusion or
 * re-ordering: one particle at a time, one ray at a time, literal convolution, literal transpose.
 *
 * Pins (tests/test_oracle_pins.py, tests/test_oracle_grad.py): SIE deflection vs 2-D quadrature of its
 * convergence; EPL series vs scipy hyp2f1 and vs SIE at gamma=2; div/curl of alpha; ring radius; Sersic
 * total flux closed form; shapelet orthonormality and explicit Hermite form; delta-PSF identity, flux
 * conservation, shift orientation; likelihood at model==obs; transformed priors integrate to 1;
 * gradient vs central finite differences (Richardson) for every parameter of every component.
 * "parity unpinned" beyond those: no published logp / chi2 / gradient value exists.
 *
 * Build: gcc -O2 -fopenmp -shared -fPIC -o libgl_oracle.so gl_oracle.c -lm   (oracle/build.py)
 */
#include <complex.h>
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define GLO_PI 3.14159265358979323846264338327950288

enum { GLO_PRIOR_NONE = 0, GLO_PRIOR_NORMAL = 1, GLO_PRIOR_LOGNORMAL = 2, GLO_PRIOR_UNIFORM = 3,
       GLO_PRIOR_TRUNCNORMAL = 4, GLO_PRIOR_LOGUNIFORM = 5 };

typedef struct { int32_t kind; double a, b, lo, hi; } glo_prior;

typedef struct {
    int32_t n_pix, supersample, psf_size;
    double  pix_scale;
    int32_t mass_model;      /* 0 SIE (closed form), 1 EPL (series) */
    int32_t epl_terms;       /* <=0: sum the series to convergence (the model); >0: truncate (debug) */
    int32_t has_shear;
    int32_t multipole_mask;  /* bit0 m=3, bit1 m=4 */
    int32_t n_source_sersic; /* 0, 1 or 2 ("Sersic profiles and/or shapelets"; two lensed sources S1, S2) */
    int32_t shapelet_nmax;   /* -1 none */
    int32_t n_lens_sersic;   /* 0..3 ("one or more Sersic profiles"; env, L1, L2) */
    int32_t param_space;     /* 0: z (bijector + log-det); 1: physical theta */
    int32_t n_systems;
    int32_t n_params;
    int32_t psf_grid;        /* 0: PSF taps on the RAY grid, convolve then bin (S10); 1: taps on the DETECTOR grid,
                                bin then convolve (reading S10b) */
    int32_t noise_model;     /* 0: fixed sigma map (S12); 1: model-dependent variance
                                v_p = sigma_p^2 + max(model_p, 0) / t_exp (NEXT-4, reading S12b) */
    double  t_exp;           /* exposure time of noise_model 1 (> 0) */
    int32_t source2_plane;   /* 1: the second source Sersic sits on its OWN source plane ("multi-source-plane systems";
                                SURVEY 8(f) NEXT-4, reading S23): its rays are deflected by eta2 * alpha, with one more
                                sampled parameter eta2 right after its block; 0: both sources on one plane */
    const glo_prior* priors;
} glo_config;

/* ---------------------------------------------------------------- parameter layout (S18) -------- */
typedef struct {
    int mass, gamma, shear, mp3, mp4, src, src2, eta2, shp, ll[3], n;   /* offsets; -1 if absent */
    int n_coef;
} layout_t;

static void make_layout(const glo_config* c, layout_t* L) {
    int k = 0;
    L->mass = k; k += 1;                                   /* theta_E */
    if (c->mass_model == 1) { L->gamma = k; k += 1; } else L->gamma = -1;
    k += 4;                                                /* e1 e2 x y */
    if (c->has_shear) { L->shear = k; k += 2; } else L->shear = -1;
    if (c->multipole_mask & 1) { L->mp3 = k; k += 2; } else L->mp3 = -1;
    if (c->multipole_mask & 2) { L->mp4 = k; k += 2; } else L->mp4 = -1;
    if (c->n_source_sersic > 0) { L->src = k; k += 7; } else L->src = -1;
    if (c->n_source_sersic > 1) { L->src2 = k; k += 7; } else L->src2 = -1;   /* second source */
    if (c->n_source_sersic > 1 && c->source2_plane) { L->eta2 = k; k += 1; } else L->eta2 = -1;   /* its own plane: eta2 */
    L->n_coef = 0;
    if (c->shapelet_nmax >= 0) {
        L->n_coef = (c->shapelet_nmax + 1) * (c->shapelet_nmax + 2) / 2;
        L->shp = k; k += 1 + L->n_coef;
    } else L->shp = -1;
    for (int i = 0; i < 3; ++i) {
        if (i < c->n_lens_sersic) { L->ll[i] = k; k += 7; } else L->ll[i] = -1;
    }
    L->n = k;
}

int glo_n_params(const glo_config* c) { layout_t L; make_layout(c, &L); return L.n; }

/* ---------------------------------------------------------------- O1: bijectors and priors ------ */
static double softplus(double x) { return x > 0 ? x + log1p(exp(-x)) : log1p(exp(x)); }
static double sigmoid(double x)  { return x >= 0 ? 1.0 / (1.0 + exp(-x)) : exp(x) / (1.0 + exp(x)); }
static double norm_cdf(double x) { return 0.5 * erfc(-x / sqrt(2.0)); }

/* One parameter.  Outputs: theta, log prior density at theta, log|dtheta/dz|, dtheta/dz,
 * d(log prior)/dtheta, d(log-det)/dz.  Returns 0 if theta is outside the support (param_space=1). */
int glo_transform_one(const glo_prior* p, int32_t param_space, double z, double* theta, double* lp,
                      double* logdet, double* dth_dz, double* dlp_dth, double* dlogdet_dz) {
    const double HL2PI = 0.5 * log(2.0 * GLO_PI);
    double th = z, ld = 0.0, dth = 1.0, dld = 0.0;
    if (param_space == 0) {
        switch (p->kind) {
        case GLO_PRIOR_LOGNORMAL:
            th = exp(z); ld = z; dth = th; dld = 1.0; break;
        case GLO_PRIOR_UNIFORM:
        case GLO_PRIOR_TRUNCNORMAL: {
            double s = sigmoid(z), w = p->hi - p->lo;
            th = p->lo + w * s;
            ld = log(w) - softplus(-z) - softplus(z);
            dth = w * s * (1.0 - s); dld = 1.0 - 2.0 * s; break; }
        case GLO_PRIOR_LOGUNIFORM: {
            double s = sigmoid(z), w = log(p->hi) - log(p->lo);
            double u = log(p->lo) + w * s;
            th = exp(u);
            ld = u + log(w) - softplus(-z) - softplus(z);
            dth = th * w * s * (1.0 - s); dld = w * s * (1.0 - s) + 1.0 - 2.0 * s; break; }
        default: break;
        }
    }
    double l = 0.0, dl = 0.0; int ok = 1;
    switch (p->kind) {
    case GLO_PRIOR_NORMAL: {
        double r = (th - p->a) / p->b;
        l = -0.5 * r * r - log(p->b) - HL2PI; dl = -r / p->b; break; }
    case GLO_PRIOR_LOGNORMAL: {
        if (!(th > 0)) { ok = 0; break; }
        double r = (log(th) - p->a) / p->b;
        l = -0.5 * r * r - log(p->b) - HL2PI - log(th); dl = -r / (p->b * th) - 1.0 / th; break; }
    case GLO_PRIOR_UNIFORM:
        if (th < p->lo || th > p->hi) { ok = 0; break; }
        l = -log(p->hi - p->lo); dl = 0.0; break;
    case GLO_PRIOR_TRUNCNORMAL: {
        if (th < p->lo || th > p->hi) { ok = 0; break; }
        double r = (th - p->a) / p->b;
        double Z = norm_cdf((p->hi - p->a) / p->b) - norm_cdf((p->lo - p->a) / p->b);
        l = -0.5 * r * r - log(p->b) - HL2PI - log(Z); dl = -r / p->b; break; }
    case GLO_PRIOR_LOGUNIFORM:
        if (th < p->lo || th > p->hi) { ok = 0; break; }
        l = -log(th) - log(log(p->hi) - log(p->lo)); dl = -1.0 / th; break;
    default: break;
    }
    *theta = th; *lp = l; *logdet = ld; *dth_dz = dth; *dlp_dth = dl; *dlogdet_dz = dld;
    return ok;
}

/* ---------------------------------------------------------------- O2: ellipticity --------------- */
typedef struct { double c, q, phi, cphi, sphi; } ell_t;
static void make_ell(double e1, double e2, ell_t* E) {
    E->c = sqrt(e1 * e1 + e2 * e2);
    E->phi = 0.5 * atan2(e2, e1);
    E->q = (1.0 - E->c) / (1.0 + E->c);
    E->cphi = cos(E->phi); E->sphi = sin(E->phi);
}
/* chain (d/dq, d/dphi) -> (d/de1, d/de2); O9: zero for c < 1e-10 */
static void ell_chain(double e1, double e2, const ell_t* E, double dq, double dphi, double* de1, double* de2) {
    if (E->c < 1e-10) { *de1 = 0.0; *de2 = 0.0; return; }
    double dq_dc = -2.0 / ((1.0 + E->c) * (1.0 + E->c));
    *de1 = dq * dq_dc * e1 / E->c + dphi * (-e2 / (2.0 * E->c * E->c));
    *de2 = dq * dq_dc * e2 / E->c + dphi * ( e1 / (2.0 * E->c * E->c));
}

/* ---------------------------------------------------------------- O4: main deflector ------------ */
/* Mass-frame deflection of the EPL (Tessore & Metcalf 2015 series) and its partial derivatives.
 * Inputs: b = theta_E sqrt(q), t = gamma-1, q, mass-frame position (x,y), n_terms (<=0: converge).
 * d[] (if non-NULL) receives, each as a complex number alpha_x + i alpha_y:
 *   d[0] = dalpha/db, d[1] = dalpha/dt, d[2] = dalpha/dq at fixed b, and jac[0..2] = Jxx, Jyy, Jxy. */
static double complex epl_frame(double b, double t, double q, double x, double y, int n_terms,
                                double complex* d, double* jac) {
    double R = sqrt(q * q * x * x + y * y);
    if (R == 0.0) { if (d) { d[0] = d[1] = d[2] = 0; jac[0] = jac[1] = jac[2] = 0; } return 0.0; }
    double f = (1.0 - q) / (1.0 + q);
    double complex E = (q * x + I * y) / R;
    double complex E2 = E * E;
    double complex w = -f * E2;
    /* Omega_n = Omega_{n-1} w (2n-2+t)/(2n+2-t);  S0 = sum Omega_n, S1f = sum n Omega_n / f,
     * S2 = sum L_n Omega_n, L_n = sum_{k<=n} 4k/((2k+2-t)(2k-2+t)) */
    double complex Om = E, S0 = E, S1f = 0.0, S2 = 0.0;
    double complex Omf = 0.0;            /* Omega_n / f, valid for n >= 1 */
    double Ln = 0.0;
    int cap = n_terms > 0 ? n_terms : 2000;
    for (int n = 1; n < cap; ++n) {
        double ratio = (2.0 * n - 2.0 + t) / (2.0 * n + 2.0 - t);
        Omf = (n == 1) ? E * (-E2) * ratio : Omf * w * ratio;
        Om = Om * w * ratio;
        Ln += 4.0 * n / ((2.0 * n + 2.0 - t) * (2.0 * n - 2.0 + t));
        S0 += Om; S1f += n * Omf; S2 += Ln * Om;
        if (n_terms <= 0 && cabs(Om) < 1e-17 * cabs(S0) && n * cabs(Omf) <= 1e-17 * cabs(S1f) + 1e-300) break;
    }
    double A = 2.0 * b / (1.0 + q);
    double P = pow(b / R, t - 1.0);
    double complex alpha = A * P * S0;
    if (d) {
        double kappa = 0.5 * (2.0 - t) * pow(b / R, t);
        double complex zt = x + I * y;
        double complex G = (1.0 - t) * alpha / conj(zt) - (zt / conj(zt)) * kappa;
        jac[0] = kappa + creal(G); jac[1] = kappa - creal(G); jac[2] = cimag(G);
        d[0] = t * alpha / b;
        d[1] = log(b / R) * alpha + A * P * S2;
        double complex S1 = f * S1f;
        d[2] = -alpha / (1.0 + q) - (t - 1.0) * alpha / R * (q * x * x / R)
             + A * P * (I * (S0 + 2.0 * S1) * (-x * y / (R * R)) + S1f * (-2.0 / ((1.0 + q) * (1.0 + q))));
    }
    return alpha;
}

/* SIE closed form (Kormann et al. 1994), mass frame; same outputs (d[1], the slope derivative, = 0). */
static double complex sie_frame(double b, double q, double x, double y, double complex* d, double* jac) {
    double R = sqrt(q * q * x * x + y * y);
    if (R == 0.0) { if (d) { d[0] = d[1] = d[2] = 0; jac[0] = jac[1] = jac[2] = 0; } return 0.0; }
    double qp = sqrt(1.0 - q * q);
    double ax, ay;
    if (qp < 1e-6) {                       /* SIS limit: alpha = theta_E (x,y)/r, b = theta_E here */
        double r = sqrt(x * x + y * y);
        ax = b * x / r; ay = b * y / r;
        if (d) {
            d[0] = (ax + I * ay) / b; d[1] = 0; d[2] = 0;   /* eps-gradient is zero at c<1e-10 (O9) */
            double k = b / (2.0 * R);
            double complex zt = x + I * y, G = -(zt / conj(zt)) * k;
            jac[0] = k + creal(G); jac[1] = k - creal(G); jac[2] = cimag(G);
        }
        return ax + I * ay;
    }
    double Aa = qp * x / R, Bb = qp * y / R;
    ax = b / qp * atan(Aa); ay = b / qp * atanh(Bb);
    if (d) {
        double k = b / (2.0 * R);
        double complex zt = x + I * y, G = -(zt / conj(zt)) * k;
        jac[0] = k + creal(G); jac[1] = k - creal(G); jac[2] = cimag(G);
        d[0] = (ax + I * ay) / b; d[1] = 0;
        double common = (-q / qp) / R - qp * q * x * x / (R * R * R);   /* d(qp/R)/dq */
        double dA = x * common, dB = y * common;
        double dax = b * (q / (qp * qp * qp) * atan(Aa)  + dA / (qp * (1.0 + Aa * Aa)));
        double day = b * (q / (qp * qp * qp) * atanh(Bb) + dB / (qp * (1.0 - Bb * Bb)));
        d[2] = dax + I * day;
    }
    return ax + I * ay;
}

/* Lab-frame deflection of every mass component at (x,y); theta = physical parameter vector.
 * beta = (x,y) - alpha.  Exported for the pins. */
static void deflect(const glo_config* c, const layout_t* L, const double* th, double x, double y,
                    double* ax, double* ay) {
    int m = L->mass;
    double thE = th[m], t = (c->mass_model == 1) ? th[L->gamma] - 1.0 : 1.0;
    int o = (c->mass_model == 1) ? m + 2 : m + 1;
    double e1 = th[o], e2 = th[o + 1], x0 = th[o + 2], y0 = th[o + 3];
    ell_t E; make_ell(e1, e2, &E);
    double dx = x - x0, dy = y - y0;
    double xr = E.cphi * dx + E.sphi * dy, yr = -E.sphi * dx + E.cphi * dy;
    double b = thE * sqrt(E.q);
    double complex a = (c->mass_model == 1) ? epl_frame(b, t, E.q, xr, yr, c->epl_terms, NULL, NULL)
                                            : sie_frame(b, E.q, xr, yr, NULL, NULL);
    double sx = E.cphi * creal(a) - E.sphi * cimag(a);
    double sy = E.sphi * creal(a) + E.cphi * cimag(a);
    if (c->has_shear) {
        double g1 = th[L->shear], g2 = th[L->shear + 1];
        sx += g1 * x + g2 * y; sy += g2 * x - g1 * y;
    }
    for (int k = 0; k < 2; ++k) {
        int off = k == 0 ? L->mp3 : L->mp4; if (off < 0) continue;
        double mm = k == 0 ? 3.0 : 4.0, cm = th[off], sm = th[off + 1];
        double r = sqrt(dx * dx + dy * dy); if (r == 0.0) continue;
        double ct = dx / r, st = dy / r, vt = atan2(dy, dx);
        double Am = cm * cos(mm * vt) + sm * sin(mm * vt), Bm = -cm * sin(mm * vt) + sm * cos(mm * vt);
        sx += (ct * Am - mm * st * Bm) / (1.0 - mm * mm);
        sy += (st * Am + mm * ct * Bm) / (1.0 - mm * mm);
    }
    *ax = sx; *ay = sy;
}

/* ---------------------------------------------------------------- O5: light --------------------- */
/* Sersic surface brightness; p = [R, n, e1, e2, x0, y0, Ie].  If dp != NULL, dp[0..6] receives
 * dI/dp and dxy[0..1] receives dI/d(x,y). */
static double sersic(const double* p, double x, double y, double* dp, double* dxy) {
    double Re = p[0], n = p[1], Ie = p[6];
    ell_t E; make_ell(p[2], p[3], &E);
    double dx = x - p[4], dy = y - p[5];
    double xr = E.cphi * dx + E.sphi * dy, yr = -E.sphi * dx + E.cphi * dy;
    double r = sqrt(E.q * xr * xr + yr * yr / E.q);
    if (r < 1e-8) r = 1e-8;
    double bn = 1.9992 * n - 0.3271;
    double u = pow(r / Re, 1.0 / n);
    double Iv = Ie * exp(-bn * (u - 1.0));
    if (dp) {
        double dI_dr = -Iv * bn * u / (n * r);
        double dr_dxr = E.q * xr / r, dr_dyr = yr / (E.q * r);
        double dr_dq = (xr * xr - yr * yr / (E.q * E.q)) / (2.0 * r);
        double dI_dx = dI_dr * (dr_dxr * E.cphi - dr_dyr * E.sphi);
        double dI_dy = dI_dr * (dr_dxr * E.sphi + dr_dyr * E.cphi);
        double dI_dphi = dI_dr * (dr_dxr * yr - dr_dyr * xr);
        double dI_dq = dI_dr * dr_dq;
        dp[0] = Iv * bn * u / (n * Re);
        dp[1] = Iv * (-1.9992 * (u - 1.0) + bn * u * log(r / Re) / (n * n));
        ell_chain(p[2], p[3], &E, dI_dq, dI_dphi, &dp[2], &dp[3]);
        dp[4] = -dI_dx; dp[5] = -dI_dy;
        dp[6] = Iv / Ie;
        dxy[0] = dI_dx; dxy[1] = dI_dy;
    }
    return Iv;
}

/* 1-D orthonormal Gauss-Hermite functions phi_0..phi_nmax at u (S9). */
void glo_shapelet_basis(int nmax, double u, double* phi) {
    phi[0] = pow(GLO_PI, -0.25) * exp(-0.5 * u * u);
    if (nmax >= 1) phi[1] = sqrt(2.0) * u * phi[0];
    for (int k = 1; k < nmax; ++k)
        phi[k + 1] = sqrt(2.0 / (k + 1.0)) * u * phi[k] - sqrt(k / (k + 1.0)) * phi[k - 1];
}

/* Shapelet surface brightness at (x,y) about centre (x0,y0); p = [beta_s, a_0 ... a_{Nc-1}], order as O5.
 * If da != NULL: da[0] = dI/dbeta_s, da[1..Nc] = dI/da_k, dxy = dI/d(x,y) (= -dI/d(x0,y0)). */
static double shapelets(int nmax, const double* p, double x0, double y0, double x, double y,
                        double* da, double* dxy) {
    double bs = p[0], u = (x - x0) / bs, v = (y - y0) / bs;
    double pu[64], pv[64], dpu[64], dpv[64];
    glo_shapelet_basis(nmax, u, pu); glo_shapelet_basis(nmax, v, pv);
    for (int k = 0; k <= nmax; ++k) {
        dpu[k] = (k > 0 ? sqrt(2.0 * k) * pu[k - 1] : 0.0) - u * pu[k];
        dpv[k] = (k > 0 ? sqrt(2.0 * k) * pv[k - 1] : 0.0) - v * pv[k];
    }
    double Iv = 0.0, dIu = 0.0, dIv = 0.0; int idx = 0;
    for (int ord = 0; ord <= nmax; ++ord)
        for (int n2 = 0; n2 <= ord; ++n2, ++idx) {
            int n1 = ord - n2; double a = p[1 + idx];
            Iv += a * pu[n1] * pv[n2]; dIu += a * dpu[n1] * pv[n2]; dIv += a * pu[n1] * dpv[n2];
            if (da) da[1 + idx] = pu[n1] * pv[n2] / bs;
        }
    Iv /= bs; dIu /= bs; dIv /= bs;
    if (da) {
        da[0] = -Iv / bs - (u * dIu + v * dIv) / bs;
        dxy[0] = dIu / bs; dxy[1] = dIv / bs;
    }
    return Iv;
}

/* Surface brightness of one ray at image position (x,y): sources at beta, lens light at theta. */
static double ray_intensity(const glo_config* c, const layout_t* L, const double* th, double x, double y) {
    double ax, ay; deflect(c, L, th, x, y, &ax, &ay);
    double bx = x - ax, by = y - ay, Iv = 0.0;
    if (L->src >= 0) Iv += sersic(th + L->src, bx, by, NULL, NULL);
    /* S23: a source on another plane sees the same lens-plane deflection scaled by the ratio eta2 of the lensing
     * efficiencies D_ls/D_s of the two planes: beta_2 = theta - eta2 alpha(theta) (the first source carries no mass) */
    if (L->src2 >= 0) {
        double eta = L->eta2 >= 0 ? th[L->eta2] : 1.0;
        Iv += sersic(th + L->src2, x - eta * ax, y - eta * ay, NULL, NULL);
    }
    if (L->shp >= 0) Iv += shapelets(c->shapelet_nmax, th + L->shp, th[L->src + 4], th[L->src + 5], bx, by, NULL, NULL);
    for (int i = 0; i < 3; ++i) if (L->ll[i] >= 0) Iv += sersic(th + L->ll[i], x, y, NULL, NULL);
    return Iv;
}

/* O9: contribution of one ray to d(logL)/dtheta: out[j] = gbar * dI_ray/dtheta_j, j < n_params. */
static void ray_adjoint(const glo_config* c, const layout_t* L, const double* th, double x, double y,
                        double gbar, double* out) {
    memset(out, 0, sizeof(double) * (size_t)L->n);
    int m = L->mass;
    double thE = th[m], t = (c->mass_model == 1) ? th[L->gamma] - 1.0 : 1.0;
    int o = (c->mass_model == 1) ? m + 2 : m + 1;
    double e1 = th[o], e2 = th[o + 1], x0 = th[o + 2], y0 = th[o + 3];
    ell_t E; make_ell(e1, e2, &E);
    double dx = x - x0, dy = y - y0;
    double xr = E.cphi * dx + E.sphi * dy, yr = -E.sphi * dx + E.cphi * dy;
    double b = thE * sqrt(E.q);
    double complex d[3]; double J[3];
    double complex a = (c->mass_model == 1) ? epl_frame(b, t, E.q, xr, yr, c->epl_terms, d, J)
                                            : sie_frame(b, E.q, xr, yr, d, J);
    double ax, ay; deflect(c, L, th, x, y, &ax, &ay);
    double bx = x - ax, by = y - ay;

    /* source light and its source-plane gradient s = gbar * grad_beta I_src */
    double sx = 0.0, sy = 0.0;
    if (L->src >= 0) {
        double dp[7], dxy[2]; sersic(th + L->src, bx, by, dp, dxy);
        for (int k = 0; k < 7; ++k) out[L->src + k] += gbar * dp[k];
        sx += gbar * dxy[0]; sy += gbar * dxy[1];
    }
    if (L->src2 >= 0) {
        double eta = L->eta2 >= 0 ? th[L->eta2] : 1.0;
        double dp[7], dxy[2]; sersic(th + L->src2, x - eta * ax, y - eta * ay, dp, dxy);
        for (int k = 0; k < 7; ++k) out[L->src2 + k] += gbar * dp[k];
        sx += eta * gbar * dxy[0]; sy += eta * gbar * dxy[1];      /* d beta_2 / d(mass) = -eta2 d alpha / d(mass) */
        if (L->eta2 >= 0) out[L->eta2] += -gbar * (dxy[0] * ax + dxy[1] * ay);   /* d beta_2 / d eta2 = -alpha */
    }
    if (L->shp >= 0) {
        double da[1 + 66 + 8], dxy[2];
        shapelets(c->shapelet_nmax, th + L->shp, th[L->src + 4], th[L->src + 5], bx, by, da, dxy);
        for (int k = 0; k < 1 + L->n_coef; ++k) out[L->shp + k] += gbar * da[k];
        out[L->src + 4] += -gbar * dxy[0]; out[L->src + 5] += -gbar * dxy[1];
        sx += gbar * dxy[0]; sy += gbar * dxy[1];
    }
    for (int i = 0; i < 3; ++i) if (L->ll[i] >= 0) {
        double dp[7], dxy[2]; sersic(th + L->ll[i], x, y, dp, dxy);
        for (int k = 0; k < 7; ++k) out[L->ll[i] + k] += gbar * dp[k];
    }
    /* mass parameters enter only through beta: dI/dtheta_mass = -grad_beta I . dalpha/dtheta_mass */
    double srx = E.cphi * sx + E.sphi * sy, sry = -E.sphi * sx + E.cphi * sy;   /* s in the mass frame */
#define SDOT(zc) (srx * creal(zc) + sry * cimag(zc))
    double db = -SDOT(d[0]);
    double dq_fixed_b = -SDOT(d[2]);
    out[m] += db * sqrt(E.q);                                  /* b = theta_E sqrt(q) */
    if (c->mass_model == 1) out[L->gamma] += -SDOT(d[1]);      /* t = gamma - 1 */
    double dq = dq_fixed_b + db * thE / (2.0 * sqrt(E.q));
    /* angle: alpha_lab = Rot(phi) alpha_r(Rot(-phi)(theta-theta0)); d/dphi = i alpha_r + J (yr, -xr) */
    double dax = -cimag(a) + J[0] * yr + J[2] * (-xr);
    double day =  creal(a) + J[2] * yr + J[1] * (-xr);
    double dphi = -(srx * dax + sry * day);
    double de1, de2; ell_chain(e1, e2, &E, dq, dphi, &de1, &de2);
    out[o] += de1; out[o + 1] += de2;
    /* centre: dalpha/dx0 = -Rot J Rot^T e_x  =>  contribution = Rot (J s_r) */
    double vx = J[0] * srx + J[2] * sry, vy = J[2] * srx + J[1] * sry;
    out[o + 2] += E.cphi * vx - E.sphi * vy;
    out[o + 3] += E.sphi * vx + E.cphi * vy;
#undef SDOT
    if (c->has_shear) {
        out[L->shear]     += -(sx * x + sy * (-y));
        out[L->shear + 1] += -(sx * y + sy * x);
    }
    for (int k = 0; k < 2; ++k) {
        int off = k == 0 ? L->mp3 : L->mp4; if (off < 0) continue;
        double mm = k == 0 ? 3.0 : 4.0, cm = th[off], sm = th[off + 1];
        double r = sqrt(dx * dx + dy * dy); if (r == 0.0) continue;
        double ct = dx / r, st = dy / r, vt = atan2(dy, dx);
        double cmt = cos(mm * vt), smt = sin(mm * vt), inv = 1.0 / (1.0 - mm * mm);
        out[off]     += -(sx * (ct * cmt + mm * st * smt) * inv + sy * (st * cmt - mm * ct * smt) * inv);
        out[off + 1] += -(sx * (ct * smt - mm * st * cmt) * inv + sy * (st * smt + mm * ct * cmt) * inv);
        /* centre dependence: J_m = (A/r) tt^T with t = (-sin, cos); dalpha/dx0 = -J_m e_x */
        double Am = cm * cmt + sm * smt;
        double proj = (Am / r) * (-st * sx + ct * sy);
        out[o + 2] += proj * (-st);
        out[o + 3] += proj * ( ct);
    }
}

/* ---------------------------------------------------------------- O3, O6: grid and image operator */
static double ray_coord(const glo_config* c, int idx) {
    return ((idx + 0.5) / c->supersample - 0.5 * c->n_pix) * c->pix_scale;
}

/* model = Delta^2 * (s x s mean) of (psf (*) I_ray), true convolution, zero padding (O6). */
void glo_conv_bin(int n_pix, int s, int K, double pix_scale, const double* psf, const double* ray, double* model) {
    int M = n_pix * s, c = (K - 1) / 2;
    double* C = (double*)malloc(sizeof(double) * (size_t)M * M);
    for (int i = 0; i < M; ++i) for (int j = 0; j < M; ++j) {
        double acc = 0.0;
        for (int a = 0; a < K; ++a) { int ii = i - (a - c); if (ii < 0 || ii >= M) continue;
            for (int bb = 0; bb < K; ++bb) { int jj = j - (bb - c); if (jj < 0 || jj >= M) continue;
                acc += psf[a * K + bb] * ray[ii * M + jj]; } }
        C[i * M + j] = acc;
    }
    for (int p = 0; p < n_pix; ++p) for (int q = 0; q < n_pix; ++q) {
        double acc = 0.0;
        for (int di = 0; di < s; ++di) for (int dj = 0; dj < s; ++dj) acc += C[(s * p + di) * M + s * q + dj];
        model[p * n_pix + q] = pix_scale * pix_scale * acc / (s * s);
    }
    free(C);
}

/* Transpose of glo_conv_bin: gbar_ray = (d model / d ray)^T g_pix, written as the literal scatter. */
static void conv_bin_transpose(int n_pix, int s, int K, double pix_scale, const double* psf, const double* g, double* gbar) {
    int M = n_pix * s, c = (K - 1) / 2;
    double* gC = (double*)malloc(sizeof(double) * (size_t)M * M);
    for (int p = 0; p < n_pix; ++p) for (int q = 0; q < n_pix; ++q)
        for (int di = 0; di < s; ++di) for (int dj = 0; dj < s; ++dj)
            gC[(s * p + di) * M + s * q + dj] = pix_scale * pix_scale * g[p * n_pix + q] / (s * s);
    memset(gbar, 0, sizeof(double) * (size_t)M * M);
    for (int i = 0; i < M; ++i) for (int j = 0; j < M; ++j) {
        double gv = gC[i * M + j];
        for (int a = 0; a < K; ++a) { int ii = i - (a - c); if (ii < 0 || ii >= M) continue;
            for (int bb = 0; bb < K; ++bb) { int jj = j - (bb - c); if (jj < 0 || jj >= M) continue;
                gbar[ii * M + jj] += psf[a * K + bb] * gv; } }
    }
    free(gC);
}

/* psf_grid = 1 (reading S10b): bin first, B = Delta^2 * (s x s mean of I_ray), then a true convolution of the N x N
 * image B with the K x K PSF sampled at the DETECTOR pixel scale, zero padding. */
void glo_bin_conv(int n_pix, int s, int K, double pix_scale, const double* psf, const double* ray, double* model) {
    int M = n_pix * s, c = (K - 1) / 2;
    double* B = (double*)malloc(sizeof(double) * (size_t)n_pix * n_pix);
    for (int p = 0; p < n_pix; ++p) for (int q = 0; q < n_pix; ++q) {
        double acc = 0.0;
        for (int di = 0; di < s; ++di) for (int dj = 0; dj < s; ++dj) acc += ray[(s * p + di) * M + s * q + dj];
        B[p * n_pix + q] = pix_scale * pix_scale * acc / (s * s);
    }
    for (int p = 0; p < n_pix; ++p) for (int q = 0; q < n_pix; ++q) {
        double acc = 0.0;
        for (int a = 0; a < K; ++a) { int pp = p - (a - c); if (pp < 0 || pp >= n_pix) continue;
            for (int bb = 0; bb < K; ++bb) { int qq = q - (bb - c); if (qq < 0 || qq >= n_pix) continue;
                acc += psf[a * K + bb] * B[pp * n_pix + qq]; } }
        model[p * n_pix + q] = acc;
    }
    free(B);
}

/* Transpose of glo_bin_conv, as the literal scatter. */
void glo_bin_conv_transpose(int n_pix, int s, int K, double pix_scale, const double* psf, const double* g, double* gbar) {
    int M = n_pix * s, c = (K - 1) / 2;
    double* gB = (double*)calloc((size_t)n_pix * n_pix, sizeof(double));
    for (int p = 0; p < n_pix; ++p) for (int q = 0; q < n_pix; ++q) {
        double gv = g[p * n_pix + q];
        for (int a = 0; a < K; ++a) { int pp = p - (a - c); if (pp < 0 || pp >= n_pix) continue;
            for (int bb = 0; bb < K; ++bb) { int qq = q - (bb - c); if (qq < 0 || qq >= n_pix) continue;
                gB[pp * n_pix + qq] += psf[a * K + bb] * gv; } }
    }
    for (int p = 0; p < n_pix; ++p) for (int q = 0; q < n_pix; ++q)
        for (int di = 0; di < s; ++di) for (int dj = 0; dj < s; ++dj)
            gbar[(s * p + di) * M + s * q + dj] = pix_scale * pix_scale * gB[p * n_pix + q] / (s * s);
    free(gB);
}

/* ---------------------------------------------------------------- per-particle evaluation ------- */
static int theta_valid(const glo_config* c, const layout_t* L, const double* th) {
    for (int i = 0; i < L->n; ++i) if (!isfinite(th[i])) return 0;
    int m = L->mass, o = (c->mass_model == 1) ? m + 2 : m + 1;
    if (!(th[m] > 0)) return 0;
    if (c->mass_model == 1) { double t = th[L->gamma] - 1.0; if (!(t > 0 && t < 2)) return 0; }
    if (!(th[o] * th[o] + th[o + 1] * th[o + 1] < 1.0)) return 0;
    int blocks[5] = { L->src, L->src2, L->ll[0], L->ll[1], L->ll[2] };
    for (int k = 0; k < 5; ++k) { int s = blocks[k]; if (s < 0) continue;
        if (!(th[s] > 0) || !(th[s + 1] > 0)) return 0;
        if (!(th[s + 2] * th[s + 2] + th[s + 3] * th[s + 3] < 1.0)) return 0; }
    if (L->shp >= 0 && !(th[L->shp] > 0)) return 0;
    return 1;
}

/* theta -> ray image [M*M] */
static void render_rays(const glo_config* c, const layout_t* L, const double* th, double* ray) {
    int M = c->n_pix * c->supersample;
    for (int i = 0; i < M; ++i) { double y = ray_coord(c, i);
        for (int j = 0; j < M; ++j) { double x = ray_coord(c, j);
            ray[i * M + j] = ray_intensity(c, L, th, x, y); } }
}

/* One particle.  obs/sig/psf already point at this particle's system.  grad/gabs/model may be NULL.
 * grad is d logp / d z (param_space 0) or d logp / d theta (param_space 1). gabs[j] = sum over rays of
 * |contribution_j| * |dtheta_j/dz_j| (denominator of the condition-aware error, SURVEY 7 hard part 1). */
static void eval_particle(const glo_config* c, const layout_t* L, const double* obs, const double* sig,
                          const double* psf, const double* z, double* logp, double* grad, double* gabs,
                          double* model_out) {
    int n = L->n, N = c->n_pix, s = c->supersample, M = N * s;
    double th[128], dth[128], dlp[128], dld[128];
    double lp_sum = 0.0, ld_sum = 0.0; int ok = 1;
    for (int i = 0; i < n; ++i) {
        double lp, ld;
        if (!isfinite(z[i])) ok = 0;
        if (!glo_transform_one(&c->priors[i], c->param_space, z[i], &th[i], &lp, &ld, &dth[i], &dlp[i], &dld[i])) ok = 0;
        lp_sum += lp; ld_sum += ld;
    }
    if (ok) ok = theta_valid(c, L, th);
    if (!ok) { *logp = -INFINITY; if (grad) memset(grad, 0, sizeof(double) * (size_t)n);
               if (gabs) memset(gabs, 0, sizeof(double) * (size_t)n); return; }
    double* ray = (double*)malloc(sizeof(double) * (size_t)M * M);
    double* model = (double*)malloc(sizeof(double) * (size_t)N * N);
    render_rays(c, L, th, ray);
    if (c->psf_grid == 1) glo_bin_conv(N, s, c->psf_size, c->pix_scale, psf, ray, model);
    else glo_conv_bin(N, s, c->psf_size, c->pix_scale, psf, ray, model);
    if (model_out) memcpy(model_out, model, sizeof(double) * (size_t)N * N);
    double chi2 = 0.0, slog = 0.0;
    if (c->noise_model == 1) {
        /* S12b: Gaussian likelihood whose variance follows the MODEL: v = sigma_bkg^2 + max(model, 0) / t_exp;
         * log L = -1/2 sum [ (model - obs)^2 / v + ln v ] - (N^2/2) ln 2 pi */
        for (int p = 0; p < N * N; ++p) {
            double v = sig[p] * sig[p] + (model[p] > 0 ? model[p] : 0.0) / c->t_exp, r = model[p] - obs[p];
            chi2 += r * r / v; slog += 0.5 * log(v);
        }
    } else
        for (int p = 0; p < N * N; ++p) { double r = (model[p] - obs[p]) / sig[p]; chi2 += r * r; slog += log(sig[p]); }
    double logL = -0.5 * chi2 - slog - 0.5 * N * N * log(2.0 * GLO_PI);
    double lpv = logL + lp_sum + ld_sum;
    if (!isfinite(lpv)) { *logp = -INFINITY; if (grad) memset(grad, 0, sizeof(double) * (size_t)n);
        if (gabs) memset(gabs, 0, sizeof(double) * (size_t)n); free(ray); free(model); return; }
    *logp = lpv;
    if (grad) {
        double* g = (double*)malloc(sizeof(double) * (size_t)N * N);
        double* gbar = (double*)malloc(sizeof(double) * (size_t)M * M);
        if (c->noise_model == 1)
            for (int p = 0; p < N * N; ++p) {   /* d logL / d model with v' = [model > 0] / t_exp */
                double vp = model[p] > 0 ? 1.0 / c->t_exp : 0.0;
                double v = sig[p] * sig[p] + (model[p] > 0 ? model[p] : 0.0) / c->t_exp, r = model[p] - obs[p];
                g[p] = -r / v + 0.5 * r * r / (v * v) * vp - 0.5 * vp / v;
            }
        else
            for (int p = 0; p < N * N; ++p) g[p] = -(model[p] - obs[p]) / (sig[p] * sig[p]);
        if (c->psf_grid == 1) glo_bin_conv_transpose(N, s, c->psf_size, c->pix_scale, psf, g, gbar);
        else conv_bin_transpose(N, s, c->psf_size, c->pix_scale, psf, g, gbar);
        double dL[128], dA[128], contrib[128];
        memset(dL, 0, sizeof dL); memset(dA, 0, sizeof dA);
        for (int i = 0; i < M; ++i) { double y = ray_coord(c, i);
            for (int j = 0; j < M; ++j) { double x = ray_coord(c, j);
                ray_adjoint(c, L, th, x, y, gbar[i * M + j], contrib);
                for (int k = 0; k < n; ++k) { dL[k] += contrib[k]; dA[k] += fabs(contrib[k]); } } }
        int finite = 1;
        for (int k = 0; k < n; ++k) {
            grad[k] = (dL[k] + dlp[k]) * dth[k] + dld[k];
            if (gabs) gabs[k] = dA[k] * fabs(dth[k]);
            if (!isfinite(grad[k])) finite = 0;
        }
        if (!finite) { *logp = -INFINITY; memset(grad, 0, sizeof(double) * (size_t)n);
                       if (gabs) memset(gabs, 0, sizeof(double) * (size_t)n); }
        free(g); free(gbar);
    }
    free(ray); free(model);
}

/* ---------------------------------------------------------------- exported batch API ------------ */
/* obs, sig: [n_systems][N][N]; psf: [n_systems][K][K]; params: [P][n_params]; system_id: [P] or NULL.
 * out_logp: [P]; out_grad, out_gabs: [P][n_params] or NULL; out_model: [P][N][N] or NULL.
 * Returns 0, or -2 if n_params does not match the layout. OpenMP over particles only. */
int glo_logpost_grad(const glo_config* c, const double* obs, const double* sig, const double* psf,
                     const double* params, const int32_t* system_id, int64_t P,
                     double* out_logp, double* out_grad, double* out_gabs, double* out_model) {
    layout_t L; make_layout(c, &L);
    if (L.n != c->n_params || L.n > 128) return -2;
    int N = c->n_pix, K = c->psf_size;
#pragma omp parallel for schedule(dynamic, 1)
    for (int64_t p = 0; p < P; ++p) {
        int sys = system_id ? system_id[p] : 0;
        eval_particle(c, &L, obs + (size_t)sys * N * N, sig + (size_t)sys * N * N, psf + (size_t)sys * K * K,
                      params + (size_t)p * L.n, &out_logp[p],
                      out_grad ? out_grad + (size_t)p * L.n : NULL,
                      out_gabs ? out_gabs + (size_t)p * L.n : NULL,
                      out_model ? out_model + (size_t)p * N * N : NULL);
    }
    return 0;
}

int glo_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
void glo_set_num_threads(int n) {
#ifdef _OPENMP
    omp_set_num_threads(n);
#else
    (void)n;
#endif
}

/* ---------------------------------------------------------------- point-wise exports (pins) ----- */
/* Lab-frame total deflection of the configured mass model at (x,y) for PHYSICAL parameters theta. */
int glo_deflection(const glo_config* c, const double* theta, double x, double y, double* ax, double* ay) {
    layout_t L; make_layout(c, &L);
    deflect(c, &L, theta, x, y, ax, ay); return 0;
}
/* Mass-frame EPL series pieces, for pinning the partials one by one. out = [Re a, Im a, Re d0, Im d0,
 * Re d1, Im d1, Re d2, Im d2, Jxx, Jyy, Jxy] */
void glo_epl_frame(double b, double t, double q, double x, double y, int n_terms, double* out) {
    double complex d[3]; double J[3];
    double complex a = epl_frame(b, t, q, x, y, n_terms, d, J);
    out[0] = creal(a); out[1] = cimag(a);
    for (int k = 0; k < 3; ++k) { out[2 + 2 * k] = creal(d[k]); out[3 + 2 * k] = cimag(d[k]); }
    out[8] = J[0]; out[9] = J[1]; out[10] = J[2];
}
void glo_sie_frame(double b, double q, double x, double y, double* out) {
    double complex d[3]; double J[3];
    double complex a = sie_frame(b, q, x, y, d, J);
    out[0] = creal(a); out[1] = cimag(a);
    for (int k = 0; k < 3; ++k) { out[2 + 2 * k] = creal(d[k]); out[3 + 2 * k] = cimag(d[k]); }
    out[8] = J[0]; out[9] = J[1]; out[10] = J[2];
}
/* Sersic with p = [R, n, e1, e2, x0, y0, Ie] at (x,y); dp[7], dxy[2] may be NULL together. */
double glo_sersic(const double* p, double x, double y, double* dp, double* dxy) { return sersic(p, x, y, dp, dxy); }
double glo_shapelets(int nmax, const double* p, double x0, double y0, double x, double y, double* da, double* dxy) {
    return shapelets(nmax, p, x0, y0, x, y, da, dxy);
}
/* Ray image [M][M] for PHYSICAL parameters theta. */
int glo_ray_image(const glo_config* c, const double* theta, double* ray) {
    layout_t L; make_layout(c, &L);
    render_rays(c, &L, theta, ray); return 0;
}
double glo_ray_coord(const glo_config* c, int idx) { return ray_coord(c, idx); }
void glo_conv_bin_transpose(int n_pix, int s, int K, double pix_scale, const double* psf, const double* g, double* gbar) {
    conv_bin_transpose(n_pix, s, K, pix_scale, psf, g, gbar);
}
