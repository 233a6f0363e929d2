/*
 * chim_oracle.c -- plain, slow, fp64 CPU oracle for the hierarchical-likelihood hot path of
 * arXiv:2504.02034 (CHIMERA 2.0).  THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
 * build, load or call it.  It shares no code, header, table or constant generator with the CUDA
 * library under paper_2504_02034_b200/csrc/, and neither imports the other.
 *
 * The method is an estimator (KDE + quadrature + Monte-Carlo sum), so the oracle follows the
 * algorithm step by step in the paper's order; every sub-quantity with a plain definition (the
 * distance integral, its inverse, the mass-function normalisations) is computed from that
 * definition by high-order quadrature / root finding, NOT from interpolation tables, so that the
 * CUDA path's tables are checked rather than shared.  No blocking, truncation or reordering:
 * the KDE is the full N_s x N_z sum.
 *
 * Citations are PAPER.md:<line> (section / equation).  Readings R1..R23 and the mass-model
 * reading M1..M4 are SURVEY.md sec. 8(c), restated in DESIGN.md.
 *
 * Pins (tests/test_oracle_pins.py): every function below is pinned except the *choices*
 * "bandwidth rule = Scott" (R3), "placement default = on samples" (R1), "u(z) in xi" (R6),
 * "m_low fiducial" (R11), "Epanechnikov bandwidth h_E = sqrt(5) h" (R19), "per-pixel bandwidth of
 * many-1d" (R20), "binning recipe" (R23) and "sparse pixels are left out" (R24), which the paper does not fix: for those, parity is unpinned by the paper and pinned only by DESIGN.md.
 *
 * lambda layout (15 doubles): H0, Om, Xi0, n, alpha, beta, delta_m, m_low, m_high, mu_g,
 * sigma_g, lambda_g, gamma, kappa, z_p   (Table 1; m_low per R11).
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define CHIMO_C_KMS 299792.458
#define CHIMO_NLAM 15
#define CHIMO_PLACE_SAMPLES 0 /* N: psi/J in the per-sample weights (default)          */
#define CHIMO_PLACE_GRID 1    /* P: psi/J on the grid, paper eq. (14) literally        */
#define CHIMO_BW_SCOTT 0
#define CHIMO_BW_FIXED 1

/* flag bits (same meaning as include/chim.h; values restated, not shared) */
#define CHIMO_F_LAMBDA_DOMAIN 1u
#define CHIMO_F_DL_NONMONOTONE 2u
#define CHIMO_F_EVENT_ZERO 4u
#define CHIMO_F_XI_ZERO 8u
#define CHIMO_F_NEFF_LOW 16u
#define CHIMO_F_TABLE_RANGE 32u
#define CHIMO_F_BW_DEGENERATE 64u

typedef struct {
    double H0, Om, Xi0, n, alpha, beta, delta_m, m_low, m_high, mu_g, sigma_g, lambda_g, gamma,
        kappa, z_p;
} lam_t;

/* ------------------------------------------------------------------ Gauss-Legendre nodes ---- */
#define GLN 32
static double gl_x[GLN], gl_w[GLN];
static int gl_ready = 0;

/* nodes/weights of the GLN-point Gauss-Legendre rule on [-1,1]: Newton iteration on P_n(x),
 * the textbook construction (roots of the Legendre polynomial, w = 2/((1-x^2) P_n'(x)^2)). */
static void gl_init(void) {
    if (gl_ready) return;
    for (int i = 0; i < GLN; ++i) {
        double x = cos(M_PI * (i + 0.75) / (GLN + 0.5));
        double dp = 1.0;
        for (int it = 0; it < 100; ++it) {
            double p0 = 1.0, p1 = x;
            for (int k = 2; k <= GLN; ++k) {
                double p2 = ((2.0 * k - 1.0) * x * p1 - (k - 1.0) * p0) / k;
                p0 = p1;
                p1 = p2;
            }
            dp = GLN * (x * p1 - p0) / (x * x - 1.0);
            double dx = p1 / dp;
            x -= dx;
            if (fabs(dx) < 1e-16) break;
        }
        {
            double p0 = 1.0, p1 = x;
            for (int k = 2; k <= GLN; ++k) {
                double p2 = ((2.0 * k - 1.0) * x * p1 - (k - 1.0) * p0) / k;
                p0 = p1;
                p1 = p2;
            }
            dp = GLN * (x * p1 - p0) / (x * x - 1.0);
        }
        gl_x[i] = x;
        gl_w[i] = 2.0 / ((1.0 - x * x) * dp * dp);
    }
    gl_ready = 1;
}

void chimo_init(void) { gl_init(); }

/* composite GL: integral of f over [a,b] with `panels` equal panels of GLN nodes each */
typedef double (*fn1)(double, const void *);
static double gl_integrate(fn1 f, const void *ctx, double a, double b, int panels) {
    if (!(b > a)) return 0.0;
    double sum = 0.0, hw = 0.5 * (b - a) / panels;
    for (int p = 0; p < panels; ++p) {
        double mid = a + (2 * p + 1) * hw;
        double s = 0.0;
        for (int i = 0; i < GLN; ++i) s += gl_w[i] * f(mid + hw * gl_x[i], ctx);
        sum += s * hw;
    }
    return sum;
}

/* ------------------------------------------------------------------------ O1 distances ------ */
/* E(z) of flat LCDM, matter + Lambda only (R4; "flat geometry" PAPER.md:19, "flat LCDM" :193) */
static double E_of_z(double z, const lam_t *L) {
    double a = 1.0 + z;
    return sqrt(L->Om * a * a * a + 1.0 - L->Om);
}
static double inv_E(double z, const void *ctx) { return 1.0 / E_of_z(z, (const lam_t *)ctx); }

/* comoving distance d_C = (c/H0) int_0^z dz'/E  [Mpc]  (eq. 1, without the (1+z)) */
static double d_C(double z, const lam_t *L) {
    if (z <= 0.0) return 0.0;
    int panels = (int)ceil(z / 0.25);
    if (panels < 1) panels = 1;
    return (CHIMO_C_KMS / L->H0) * gl_integrate(inv_E, L, 0.0, z, panels);
}
/* Xi(z) = Xi0 + (1-Xi0)/(1+z)^n   (eq. 2) */
static double Xi_of_z(double z, const lam_t *L) { return L->Xi0 + (1.0 - L->Xi0) * pow(1.0 + z, -L->n); }
static double dXi_dz(double z, const lam_t *L) { return -L->n * (1.0 - L->Xi0) * pow(1.0 + z, -L->n - 1.0); }
/* d_L^gw = Xi(z) (1+z) d_C(z)   (PAPER.md:17 eq. 1, :23 eq. 2) */
static double dL_gw(double z, const lam_t *L) { return Xi_of_z(z, L) * (1.0 + z) * d_C(z, L); }
/* d d_L^gw / dz = Xi'(1+z) d_C + Xi [ d_C + (1+z) c/(H0 E) ] */
static double ddL_gw_dz(double z, const lam_t *L) {
    double dc = d_C(z, L);
    return dXi_dz(z, L) * (1.0 + z) * dc +
           Xi_of_z(z, L) * (dc + (1.0 + z) * CHIMO_C_KMS / (L->H0 * E_of_z(z, L)));
}
/* Jacobian of eq. (11): J(z) = (1+z)^3 |d d_L^gw/dz| */
static double jac(double z, const lam_t *L) {
    double a = 1.0 + z;
    return a * a * a * fabs(ddL_gw_dz(z, L));
}
/* full-sky dV_c/dz = 4 pi d_C^2 c/(H0 E)  [Mpc^3] and V_c(z) = 4 pi/3 d_C^3  (eq. 8-9, 23) */
static double dVc_dz(double z, const lam_t *L) {
    double dc = d_C(z, L);
    return 4.0 * M_PI * dc * dc * CHIMO_C_KMS / (L->H0 * E_of_z(z, L));
}
static double V_c(double z, const lam_t *L) {
    double dc = d_C(z, L);
    return 4.0 * M_PI / 3.0 * dc * dc * dc;
}

void chimo_distances(const double *lam, int n, const double *z, double *dc, double *dl_em,
                     double *dl_gw, double *ddl_gw_dz) {
    gl_init();
    const lam_t *L = (const lam_t *)lam;
    for (int i = 0; i < n; ++i) {
        double d = d_C(z[i], L);
        if (dc) dc[i] = d;
        if (dl_em) dl_em[i] = (1.0 + z[i]) * d;
        if (dl_gw) dl_gw[i] = dL_gw(z[i], L);
        if (ddl_gw_dz) ddl_gw_dz[i] = ddL_gw_dz(z[i], L);
    }
}
void chimo_volume(const double *lam, int n, const double *z, double *dvdz, double *vc) {
    gl_init();
    const lam_t *L = (const lam_t *)lam;
    for (int i = 0; i < n; ++i) {
        if (dvdz) dvdz[i] = dVc_dz(z[i], L);
        if (vc) vc[i] = V_c(z[i], L);
    }
}

/* per-lambda validity: parameter domain */
static int lambda_in_domain(const lam_t *L) {
    if (!(L->H0 > 0.0) || !(L->Om > 0.0 && L->Om <= 1.0) || !(L->Xi0 > 0.0)) return 0;
    if (!(L->delta_m > 0.0) || !(L->sigma_g > 0.0)) return 0;
    if (!(L->lambda_g >= 0.0 && L->lambda_g <= 1.0)) return 0;
    if (!(L->m_low > 0.0) || !(L->m_high > L->m_low)) return 0;
    if (!(L->z_p > -1.0)) return 0;
    for (int k = 0; k < CHIMO_NLAM; ++k)
        if (!isfinite(((const double *)L)[k])) return 0;
    return 1;
}
/* R16: d_L^gw must be increasing; rule = analytic derivative > 0 at z_k = k z_max/n, k=0..n */
static int dl_monotone(const lam_t *L, double z_table_max, int n_table) {
    for (int k = 0; k <= n_table; ++k) {
        double z = z_table_max * k / n_table;
        if (!(ddL_gw_dz(z, L) > 0.0)) return 0;
    }
    return 1;
}
int chimo_dl_monotone(const double *lam, double z_table_max, int n_table) {
    gl_init();
    return dl_monotone((const lam_t *)lam, z_table_max, n_table);
}

/* ------------------------------------------------------------------------ O2 inversion ------ */
/* z solving d_L^gw(z) = dl: bracket by doubling, safeguarded Newton to 1e-13.
 * Returns NaN if dl > d_L^gw(z_table_max) (the TABLE_RANGE rule: such a sample gets weight 0). */
static double z_of_dL(double dl, const lam_t *L, double z_table_max) {
    if (!(dl > 0.0)) return 0.0;
    double lo = 0.0, hi = (z_table_max < 0.5) ? z_table_max : 0.5;
    while (dL_gw(hi, L) < dl) {
        if (hi >= z_table_max) return NAN;
        lo = hi;
        hi = fmin(2.0 * hi, z_table_max);
    }
    double z = 0.5 * (lo + hi);
    for (int it = 0; it < 200; ++it) {
        double f = dL_gw(z, L) - dl;
        if (f > 0.0) hi = z; else lo = z;
        double dz = -f / ddL_gw_dz(z, L);
        double zn = z + dz;
        if (!(zn > lo && zn < hi)) { /* Newton left the bracket: bisect */
            zn = 0.5 * (lo + hi);
            dz = zn - z;
        }
        z = zn;
        if (fabs(dz) < 1e-13 || hi - lo < 1e-14) break;
    }
    return z;
}
void chimo_z_of_dl(const double *lam, double z_table_max, int n, const double *dl, double *z) {
    gl_init();
    for (int i = 0; i < n; ++i) z[i] = z_of_dL(dl[i], (const lam_t *)lam, z_table_max);
}

/* --------------------------------------------------------------------- O4 mass function ----- */
/* The mass function is evaluated in LOG space (ln S, ln p(m1), ln C, ln p(m1,m2)) and the linear-valued functions the
 * pins call are exp() of these: deep in the smoothing window S(m) = e^(-delta/m') leaves the fp64 range (m' < delta/709)
 * although ln S is an ordinary number, and an event whose only supported samples sit there has a well-defined log I
 * (R21: with linear weights the oracle used to return I = 0 there -- an fp64 artefact, not the definition). */
static double logaddexp(double a, double b) {
    if (a == -INFINITY) return b;
    if (b == -INFINITY) return a;
    double mx = a > b ? a : b, mn = a > b ? b : a;
    return mx + log1p(exp(mn - mx));
}
/* M1: low-mass smoothing S(m) ("smoothed using delta_m"; form: the published
 * power-law+peak definition the paper cites at :224):  S = 1/(1 + e^f), f = delta/m' + delta/(m' - delta), m' = m - m_low;
 * ln S = -ln(1 + e^f) = -f - ln(1 + e^-f) for f > 0. */
static double ln_smooth_S(double m, const lam_t *L) {
    if (m < L->m_low) return -INFINITY;
    if (m >= L->m_low + L->delta_m) return 0.0;
    double mp = m - L->m_low;
    if (mp <= 0.0) return -INFINITY;
    double f = L->delta_m / mp + L->delta_m / (mp - L->delta_m);
    return (f > 0.0) ? -(f + log1p(exp(-f))) : -log1p(exp(f));
}
static double smooth_S(double m, const lam_t *L) { return exp(ln_smooth_S(m, L)); }
/* normalised truncated power law m^-alpha on [m_low, m_high] (closed interval, R15) */
static double ln_powerlaw_pdf(double m, const lam_t *L) {
    if (m < L->m_low || m > L->m_high) return -INFINITY;
    double norm;
    if (fabs(L->alpha - 1.0) < 1e-12) norm = log(L->m_high / L->m_low);
    else norm = (pow(L->m_high, 1.0 - L->alpha) - pow(L->m_low, 1.0 - L->alpha)) / (1.0 - L->alpha);
    return -L->alpha * log(m) - log(norm);
}
static double ln_gauss_pdf(double m, double mu, double sig) {
    double d = (m - mu) / sig;
    return -0.5 * d * d - log(sig * sqrt(2.0 * M_PI));
}
/* M2: un-normalised primary density [ (1-lg) PL + lg N ] S */
static double ln_p1_unnorm(double m, const lam_t *L) {
    double a = (L->lambda_g < 1.0) ? log(1.0 - L->lambda_g) + ln_powerlaw_pdf(m, L) : -INFINITY;
    double b = (L->lambda_g > 0.0) ? log(L->lambda_g) + ln_gauss_pdf(m, L->mu_g, L->sigma_g) : -INFINITY;
    double s = ln_smooth_S(m, L);
    if (s == -INFINITY) return -INFINITY;
    return logaddexp(a, b) + s;
}
static double p1_unnorm(double m, const void *ctx) { return exp(ln_p1_unnorm(m, (const lam_t *)ctx)); }
/* Z1 = int_{m_low}^{inf} p1_unnorm dm.  Pieces: the smoothing window (split at m_high if the
 * power law ends inside it), the plateau up to m_high, and the Gaussian beyond (to +40 sigma). */
static double Z1_norm(const lam_t *L) {
    double a = L->m_low, c = L->m_low + L->delta_m, b = L->m_high;
    double top = fmax(fmax(b, c), L->mu_g + 40.0 * L->sigma_g);
    double z = 0.0;
    if (b < c) {
        z += gl_integrate(p1_unnorm, L, a, b, 16);
        z += gl_integrate(p1_unnorm, L, b, c, 16);
        z += gl_integrate(p1_unnorm, L, c, top, 64);
    } else {
        z += gl_integrate(p1_unnorm, L, a, c, 16);
        z += gl_integrate(p1_unnorm, L, c, b, 64);
        z += gl_integrate(p1_unnorm, L, b, top, 64);
    }
    return z;
}
/* integrand of C(m1) with S(m1') factored out: m^beta S(m)/S(m_ref), S(m)/S(m_ref) = exp(ln S(m) - ln S(m_ref)) <= 1 */
typedef struct { const lam_t *L; double ln_s_ref; } m2_ctx;
static double m2_kernel(double m, const void *ctx) {
    const m2_ctx *c = (const m2_ctx *)ctx;
    double ls = ln_smooth_S(m, c->L);
    if (ls == -INFINITY) return 0.0;
    return pow(m, c->L->beta) * exp(ls - c->ln_s_ref);
}
/* M3/M4: C(m1) = int_{m_low}^{m1} m^beta S(m) dm, returned as ln C.  Above the window S = 1 and the integrand is a pure power
 * (closed form, beta = -1 -> log) on top of the full-window integral.  Inside the window S(m1) is factored out (it may be
 * e^-1000) and the rest -- which piles up at the upper end over a width ~ m1'^2/delta -- is integrated on panels that halve
 * towards m1 (13 panels of GLN nodes: resolves m1'/delta down to ~1e-4). */
static double ln_C_norm(double m1, const lam_t *L) {
    double a = L->m_low, c = L->m_low + L->delta_m;
    if (m1 <= a) return -INFINITY;
    if (m1 < c) {
        m2_ctx k = {L, ln_smooth_S(m1, L)};
        if (k.ln_s_ref == -INFINITY) return -INFINITY;
        double sum = 0.0, lo = a, w = m1 - a;
        for (int p = 0; p <= 12; ++p) {            /* panels [a, m1 - w/2], [m1 - w/2, m1 - w/4], ..., [m1 - w/4096, m1] */
            double hi = (p < 12) ? m1 - w / (double)(2 << p) : m1;
            sum += gl_integrate(m2_kernel, &k, lo, hi, 1);
            lo = hi;
        }
        return k.ln_s_ref + log(sum);
    }
    m2_ctx k = {L, 0.0};
    double w = gl_integrate(m2_kernel, &k, a, c, 8);
    double bp = L->beta + 1.0;
    if (fabs(bp) < 1e-12) return log(w + log(m1 / c));
    return log(w + (pow(m1, bp) - pow(c, bp)) / bp);
}
/* ln p(m1,m2), p(m1,m2) = p(m1) p(m2|m1)  (eq. 20); ln_Z1 = ln of Z1_norm */
static double ln_mass_pdf(double m1, double m2, const lam_t *L, double ln_Z1) {
    if (m2 < L->m_low || m2 > m1) return -INFINITY;
    double lp1 = ln_p1_unnorm(m1, L);
    if (lp1 == -INFINITY) return -INFINITY;
    double ls2 = ln_smooth_S(m2, L);
    if (ls2 == -INFINITY) return -INFINITY;
    double lC = ln_C_norm(m1, L);
    if (lC == -INFINITY) return -INFINITY;
    return lp1 - ln_Z1 + L->beta * log(m2) + ls2 - lC;
}
static double mass_pdf(double m1, double m2, const lam_t *L, double Z1) { return exp(ln_mass_pdf(m1, m2, L, log(Z1))); }

void chimo_smoothing(const double *lam, int n, const double *m, double *out) {
    for (int i = 0; i < n; ++i) out[i] = smooth_S(m[i], (const lam_t *)lam);
}
void chimo_p_m1(const double *lam, int n, const double *m, double *out) {
    gl_init();
    const lam_t *L = (const lam_t *)lam;
    double Z1 = Z1_norm(L);
    for (int i = 0; i < n; ++i) out[i] = p1_unnorm(m[i], L) / Z1;
}
void chimo_p_m2_given_m1(const double *lam, int n, const double *m1, const double *m2, double *out) {
    gl_init();
    const lam_t *L = (const lam_t *)lam;
    for (int i = 0; i < n; ++i) {
        if (m2[i] < L->m_low || m2[i] > m1[i]) { out[i] = 0.0; continue; }
        double lC = ln_C_norm(m1[i], L), ls = ln_smooth_S(m2[i], L);
        out[i] = (lC > -INFINITY && ls > -INFINITY) ? exp(L->beta * log(m2[i]) + ls - lC) : 0.0;
    }
}
/* log-valued entries (finite where the linear ones underflow) */
void chimo_ln_smoothing(const double *lam, int n, const double *m, double *out) {
    for (int i = 0; i < n; ++i) out[i] = ln_smooth_S(m[i], (const lam_t *)lam);
}
void chimo_ln_p_m2_given_m1(const double *lam, int n, const double *m1, const double *m2, double *out) {
    gl_init();
    const lam_t *L = (const lam_t *)lam;
    for (int i = 0; i < n; ++i) {
        double lC = ln_C_norm(m1[i], L), ls = ln_smooth_S(m2[i], L);
        out[i] = (m2[i] >= L->m_low && m2[i] <= m1[i] && lC > -INFINITY && ls > -INFINITY) ? L->beta * log(m2[i]) + ls - lC : -INFINITY;
    }
}
void chimo_ln_mass_pdf(const double *lam, int n, const double *m1, const double *m2, double *out) {
    gl_init();
    const lam_t *L = (const lam_t *)lam;
    double ln_Z1 = log(Z1_norm(L));
    for (int i = 0; i < n; ++i) out[i] = ln_mass_pdf(m1[i], m2[i], L, ln_Z1);
}
void chimo_mass_pdf(const double *lam, int n, const double *m1, const double *m2, double *out) {
    gl_init();
    const lam_t *L = (const lam_t *)lam;
    double Z1 = Z1_norm(L);
    for (int i = 0; i < n; ++i) out[i] = mass_pdf(m1[i], m2[i], L, Z1);
}

/* ----------------------------------------------------------------------------- O5 rate ------ */
/* Madau-Dickinson, eq. (21) PAPER.md:226 with proportionality constant 1 (R5) */
static double psi_rate(double z, const lam_t *L) {
    double a = 1.0 + z;
    return pow(a, L->gamma) / (1.0 + pow(a / (1.0 + L->z_p), L->gamma + L->kappa));
}
void chimo_psi(const double *lam, int n, const double *z, double *out) {
    for (int i = 0; i < n; ++i) out[i] = psi_rate(z[i], (const lam_t *)lam);
}

/* -------------------------------------------------------------------------- O6 weights ------ */
/* Per-sample redshift and LOG weight (PAPER.md:52; :112 eq. 16 weights; :75 eq. 11; R1, R10).
 *   placement N: w = p_m(m1,m2) psi(z)/J(z) / pi ;  placement P: w = p_m / pi.
 * ln w = -inf where the weight is 0 (R15).  Samples beyond the table range (z = NaN) get z = z_table_max, w = 0 and
 * raise *range_flag. */
void chimo_sample_log_weights(const double *lam, int placement, double z_table_max, int n,
                              const double *dl, const double *m1d, const double *m2d,
                              const double *ln_prior, double *z_out, double *lw_out, int *range_flag) {
    gl_init();
    const lam_t *L = (const lam_t *)lam;
    double ln_Z1 = log(Z1_norm(L));
    int rf = 0;
    for (int j = 0; j < n; ++j) {
        double z = z_of_dL(dl[j], L, z_table_max);
        if (isnan(z)) { z_out[j] = z_table_max; lw_out[j] = -INFINITY; rf = 1; continue; }
        double m1 = m1d[j] / (1.0 + z), m2 = m2d[j] / (1.0 + z);
        double lw = ln_mass_pdf(m1, m2, L, ln_Z1);
        if (lw > -INFINITY) {
            lw -= ln_prior[j];
            if (placement == CHIMO_PLACE_SAMPLES) lw += log(psi_rate(z, L)) - log(jac(z, L));
        }
        z_out[j] = z;
        lw_out[j] = lw;
    }
    if (range_flag) *range_flag = rf;
}
/* the same as linear weights w = exp(ln w) (may underflow to 0 for ln w < -745: the step-by-step pins use it) */
void chimo_sample_weights(const double *lam, int placement, double z_table_max, int n,
                          const double *dl, const double *m1d, const double *m2d,
                          const double *ln_prior, double *z_out, double *w_out, int *range_flag) {
    chimo_sample_log_weights(lam, placement, z_table_max, n, dl, m1d, m2d, ln_prior, z_out, w_out, range_flag);
    for (int j = 0; j < n; ++j) w_out[j] = exp(w_out[j]);
}

/* ------------------------------------------------------------------------ O7 bandwidth ------ */
/* Scott's rule on the weighted sample (R3): w^ = w/sum w, n_eff = 1/sum w^^2,
 * var = sum w^(z-zbar)^2 / (1 - sum w^^2), h = sqrt(var) n_eff^(-1/5).
 *
 * Input: LOG weights.  The rule is evaluated in an algebraically identical form that neither cancels nor underflows when one
 * sample d carries (almost) the whole event -- both sums of the definition then tend to 0 together (R21).  With
 * d = argmax ln w, l2 = the largest ln w among the others, s = exp(l2 - ln w_d) in (0, 1], e_j = exp(ln w_j - l2),
 * u_j = z_j - z_d and, over j != d,  W = sum e_j, Q = sum e_j^2, A = sum e_j u_j^2, B = sum e_j u_j:
 *     sum w / w_d = 1 + sW,     1 - sum w^^2 = [2sW + s^2 (W^2 - Q)] / (1 + sW)^2,
 *     sum w^(z-zbar)^2 = [sA(1 + sW) - s^2 B^2] / (1 + sW)^2
 *  => var = [A(1 + sW) - s B^2] / [2W + s (W^2 - Q)],   n_eff = (1 + sW)^2 / (1 + s^2 Q).
 * Undefined (NaN, BW_DEGENERATE) iff fewer than two samples have non-zero weight -- then 1 - sum w^^2 = 0 exactly -- or
 * var = 0 (all weighted samples at one redshift).  Two samples d apart give var = d^2/2 for every weight ratio. */
double chimo_scott_bw_log(int n, const double *z, const double *lw) {
    int d = -1;
    for (int j = 0; j < n; ++j)
        if (lw[j] > -INFINITY && (d < 0 || lw[j] > lw[d])) d = j;
    if (d < 0) return NAN;
    double l2 = -INFINITY;
    for (int j = 0; j < n; ++j)
        if (j != d && lw[j] > l2) l2 = lw[j];
    if (l2 == -INFINITY) return NAN;
    long double s = expl((long double)l2 - (long double)lw[d]);
    long double W = 0.0L, Q = 0.0L, A = 0.0L, B = 0.0L;
    for (int j = 0; j < n; ++j) {
        if (j == d || lw[j] == -INFINITY) continue;
        long double e = expl((long double)lw[j] - (long double)l2), u = (long double)z[j] - (long double)z[d];
        W += e;
        Q += e * e;
        A += e * u * u;
        B += e * u;
    }
    long double var = (A * (1.0L + s * W) - s * B * B) / (2.0L * W + s * (W * W - Q));
    if (!(var > 0.0L)) return NAN;
    long double neff = (1.0L + s * W) * (1.0L + s * W) / (1.0L + s * s * Q);
    return sqrt((double)var) * pow((double)neff, -0.2);
}
/* linear-weight entry (w >= 0): ln w = log(w), log(0) = -inf */
double chimo_scott_bw(int n, const double *z, const double *w) {
    double *lw = (double *)malloc(sizeof(double) * (n > 0 ? n : 1));
    for (int j = 0; j < n; ++j) lw[j] = (w[j] > 0.0) ? log(w[j]) : -INFINITY;
    double h = chimo_scott_bw_log(n, z, lw);
    free(lw);
    return h;
}

/* ------------------------------------------------------------------------------ O8 KDE ------ */
/* K(z_g) = (1/N_s) sum_j w_j exp(-(z_g-z_j)^2/(2h^2)) / (h sqrt(2 pi)): full sum, no cut-off
 * (eq. 19; R2 normalisation by N_s; R9 no truncation). */
void chimo_kde(int n, const double *z, const double *w, double h, int ng, const double *zg, double *K) {
    double norm = 1.0 / ((double)n * h * sqrt(2.0 * M_PI));
    for (int g = 0; g < ng; ++g) {
        long double s = 0.0L;
        for (int j = 0; j < n; ++j) {
            double d = (zg[g] - z[j]) / h;
            s += w[j] * exp(-0.5 * d * d);
        }
        K[g] = (double)s * norm;
    }
}

/* O8' Epanechnikov variant ("Epanechnikov kernel", no formula given; reading R19 of DESIGN.md):
 * K(z_g) = (1/N_s) sum_j w_j (3/(4 h_E)) max(0, 1 - ((z_g - z_j)/h_E)^2),  h_E = sqrt(5) h,
 * so that the kernel has the same standard deviation h as the Gaussian one (the bandwidth rule is unchanged). */
void chimo_kde_epan(int n, const double *z, const double *w, double h, int ng, const double *zg, double *K) {
    double hE = sqrt(5.0) * h, norm = 0.75 / ((double)n * hE);
    for (int g = 0; g < ng; ++g) {
        long double s = 0.0L;
        for (int j = 0; j < n; ++j) {
            double u = (zg[g] - z[j]) / hE, k = 1.0 - u * u;
            if (k > 0.0) s += w[j] * k;
        }
        K[g] = (double)s * norm;
    }
}

/* Sample binning ("the weighted PE samples ... are binned" to a fixed-size dataset; no recipe given;
 * reading R23 of DESIGN.md): n_bins equal-width bins on [min_j z_j, max_j z_j]; every bin becomes one pseudo-sample at the
 * weighted mean redshift of its members carrying the sum of their weights (an empty bin: weight 0).  The bandwidth is the one
 * of the ORIGINAL samples and the KDE keeps its 1/N_s, so binning approximates the unbinned estimator to O((bin width / h)^2).
 * zb, wb: [n_bins].  Returns the number of bins written (n_bins; 1 if all z_j coincide). */
int chimo_bin_samples(int n, const double *z, const double *w, int n_bins, double *zb, double *wb) {
    double lo = INFINITY, hi = -INFINITY;
    for (int j = 0; j < n; ++j) { if (z[j] < lo) lo = z[j]; if (z[j] > hi) hi = z[j]; }
    if (!(hi > lo)) n_bins = 1;
    double width = (hi - lo) / n_bins;
    for (int b = 0; b < n_bins; ++b) { zb[b] = 0.0; wb[b] = 0.0; }
    for (int j = 0; j < n; ++j) {
        int b = (hi > lo) ? (int)((z[j] - lo) / width) : 0;
        if (b > n_bins - 1) b = n_bins - 1;
        wb[b] += w[j];
        zb[b] += w[j] * (z[j] - lo);
    }
    for (int b = 0; b < n_bins; ++b) zb[b] = (wb[b] > 0.0) ? lo + zb[b] / wb[b] : lo + (b + 0.5) * width;
    return n_bins;
}

static int chimo_n_bins = 0; /* 0 = no binning (default) */
void chimo_set_bins(int n_bins) { chimo_n_bins = n_bins; }

static int chimo_kernel_kind = 0; /* 0 Gaussian (default), 1 Epanechnikov: selects O8 / O8' in chimo_event_logI */
void chimo_set_kernel(int kind) { chimo_kernel_kind = kind; }
int chimo_get_kernel(void) { return chimo_kernel_kind; }

/* -------------------------------------------------------------------- O9 event integral ----- */
/* I_i = composite trapezoid of y_g = K(z_g) G(z_g) p_gal(z_g) on the given grid (PAPER.md:97,
 * eq. 14 with N_pix = 1, R13).  G = 1 (placement N) or psi/J at the grid point (placement P). */
double chimo_event_integral(const double *lam, int placement, int ng, const double *zg,
                            const double *K, const double *pgal) {
    gl_init();
    const lam_t *L = (const lam_t *)lam;
    long double I = 0.0L;
    double yprev = 0.0;
    for (int g = 0; g < ng; ++g) {
        double G = 1.0;
        if (placement == CHIMO_PLACE_GRID) G = psi_rate(zg[g], L) / jac(zg[g], L);
        double y = K[g] * G * pgal[g];
        if (g > 0) I += 0.5L * ((long double)y + yprev) * (zg[g] - zg[g - 1]);
        yprev = y;
    }
    return (double)I;
}

/* One event end to end: O2..O9.  Returns log I_i; optional outputs h, flags.
 * The weights are carried as ln w_j and enter O8-O9 as w_j / w_max (P10: w -> c w gives I -> c I with the same h), ln w_max
 * is added back to log I: an event whose weights all lie below the fp64 range is small, not empty. */
double chimo_event_logI(const double *lam, int placement, int bw_rule, double fixed_bw,
                        double z_table_max, int ns, const double *dl, const double *m1d,
                        const double *m2d, const double *ln_prior, int ng, const double *zg,
                        const double *pgal, double *h_out, uint32_t *flags) {
    double *z = (double *)malloc(sizeof(double) * ns), *lw = (double *)malloc(sizeof(double) * ns);
    double *w = (double *)malloc(sizeof(double) * ns);
    double *K = (double *)malloc(sizeof(double) * ng);
    int rf = 0;
    uint32_t fl = 0;
    chimo_sample_log_weights(lam, placement, z_table_max, ns, dl, m1d, m2d, ln_prior, z, lw, &rf);
    if (rf) fl |= CHIMO_F_TABLE_RANGE;
    double lmax = -INFINITY, h, logI;
    for (int j = 0; j < ns; ++j) if (lw[j] > lmax) lmax = lw[j];
    if (lmax == -INFINITY) { /* all-zero event: I = 0 (R15) */
        fl |= CHIMO_F_EVENT_ZERO;
        h = NAN;
        logI = -INFINITY;
    } else {
        for (int j = 0; j < ns; ++j) w[j] = exp(lw[j] - lmax);
        h = (bw_rule == CHIMO_BW_FIXED) ? fixed_bw : chimo_scott_bw_log(ns, z, lw);
        if (!(h > 0.0) || !isfinite(h)) {
            fl |= CHIMO_F_BW_DEGENERATE;
            logI = NAN;
        } else {
            int nk = ns;
            const double *zk = z, *wk = w;
            double *zb = NULL, *wb = NULL;
            if (chimo_n_bins > 0) {   /* R23: pseudo-samples; h stays the one of the original samples, 1/N_s stays */
                zb = (double *)malloc(sizeof(double) * chimo_n_bins);
                wb = (double *)malloc(sizeof(double) * chimo_n_bins);
                nk = chimo_bin_samples(ns, z, w, chimo_n_bins, zb, wb);
                zk = zb; wk = wb;
            }
            if (chimo_kernel_kind == 1) chimo_kde_epan(nk, zk, wk, h, ng, zg, K);
            else chimo_kde(nk, zk, wk, h, ng, zg, K);
            if (nk != ns) { double f = (double)nk / (double)ns; for (int g = 0; g < ng; ++g) K[g] *= f; }   /* keep 1/N_s */
            free(zb); free(wb);
            double I = chimo_event_integral(lam, placement, ng, zg, K, pgal);
            if (I > 0.0) logI = log(I) + lmax;
            else { fl |= CHIMO_F_EVENT_ZERO; logI = -INFINITY; }
        }
    }
    if (h_out) *h_out = h;
    if (flags) *flags |= fl;
    free(z); free(lw); free(w); free(K);
    return logI;
}

/* ------------------------------------------------------------------------ O10 selection ----- */
/* s_j = p_m psi(z_j) u(z_j) / J(z_j) / p_draw,j ; u = (dVc/dz)/Vc(z_cat_max) on [0,z_cat_max]
 * (PAPER.md:87 eq. 12; :65 eq. 9 with P_compl -> 0; R6, R7).  Returns sum s, sum s^2. */
void chimo_selection_sums(const double *lam, double z_cat_max, double z_table_max, int64_t n_det,
                          const double *dl, const double *m1d, const double *m2d,
                          const double *ln_pdraw, double *sum_s, double *sum_s2, double *s_out,
                          int *range_flag) {
    gl_init();
    const lam_t *L = (const lam_t *)lam;
    double ln_Z1 = log(Z1_norm(L));
    double Vmax = V_c(z_cat_max, L);
    long double S1 = 0.0L, S2 = 0.0L;
    int rf = 0;
#pragma omp parallel for schedule(dynamic, 1024) reduction(+ : S1, S2) reduction(| : rf)
    for (int64_t j = 0; j < n_det; ++j) {
        double s = 0.0;
        double z = z_of_dL(dl[j], L, z_table_max);
        if (isnan(z)) rf |= 1;
        else if (z <= z_cat_max) {
            double m1 = m1d[j] / (1.0 + z), m2 = m2d[j] / (1.0 + z);
            double lpm = ln_mass_pdf(m1, m2, L, ln_Z1);
            if (lpm > -INFINITY) s = exp(lpm - ln_pdraw[j]) * psi_rate(z, L) * (dVc_dz(z, L) / Vmax) / jac(z, L);
        }
        if (s_out) s_out[j] = s;
        S1 += s;
        S2 += (long double)s * s;
    }
    *sum_s = (double)S1;
    *sum_s2 = (double)S2;
    if (range_flag) *range_flag = rf;
}
/* eq. (13) */
double chimo_neff(double sum_s, double sum_s2, double n_inj_total) {
    return sum_s * sum_s / (sum_s2 - sum_s * sum_s / n_inj_total);
}

/* -------------------------------------------------------------- p_cat from a galaxy list ---- */
/* PAPER.md:62 eq. 8 for one line of sight (the step before the hot path; reading R22 of DESIGN.md):
 *   p_cat(z) = (1/sum_g w_g) sum_g w_g N(z; zt_g, st_g) dVc/dz(z) / Z_g,   Z_g = int_0^inf N(z; zt_g, st_g) dVc/dz dz,
 * dV_c/dz at the fixed cosmology lam (computed once, fixed for the whole inference); Z_g by Gauss-Legendre on
 * [max(0, zt - 10 st), zt + 10 st].  w == NULL: unit weights. */
typedef struct { const lam_t *L; double zt, st; } pcat_ctx;
static double pcat_integrand(double z, const void *ctx) {
    const pcat_ctx *c = (const pcat_ctx *)ctx;
    double u = (z - c->zt) / c->st;
    return exp(-0.5 * u * u) / (c->st * sqrt(2.0 * M_PI)) * dVc_dz(z, c->L);
}
void chimo_pcat(const double *lam, int n_gal, const double *zt, const double *st, const double *w, int ng,
                const double *zg, double *out) {
    gl_init();
    const lam_t *L = (const lam_t *)lam;
    double *coef = (double *)malloc(sizeof(double) * (n_gal > 0 ? n_gal : 1));
    long double sw = 0.0L;
    for (int g = 0; g < n_gal; ++g) {
        pcat_ctx c = {L, zt[g], st[g]};
        double lo = zt[g] - 10.0 * st[g], hi = zt[g] + 10.0 * st[g];
        if (lo < 0.0) lo = 0.0;
        double Z = gl_integrate(pcat_integrand, &c, lo, hi, 8);
        double wg = w ? w[g] : 1.0;
        coef[g] = wg / Z;
        sw += wg;
    }
    for (int i = 0; i < ng; ++i) {
        long double acc = 0.0L;
        for (int g = 0; g < n_gal; ++g) {
            double u = (zg[i] - zt[g]) / st[g];
            acc += coef[g] * exp(-0.5 * u * u) / (st[g] * sqrt(2.0 * M_PI));
        }
        out[i] = (double)(acc / sw) * dVc_dz(zg[i], L);
    }
    free(coef);
}

/* ---------------------------------------------------- p_gal with the completeness terms ---- */
/* PAPER.md:58 eq. 7, :65 eq. 9, :67 eq. 10 for one line of sight (reading R25 of DESIGN.md):
 *   p_gal(z) = f_R p_cat(z) + (1 - f_R) p_miss(z),   (1 - f_R) p_miss(z) = [1 - P_compl(z)] u(z),
 *   u(z) = (dV_c/dz)(z) / V_c(z_max) on [0, z_max], 0 beyond (the homogeneous density of eq. 9; the same u as in xi, R6),
 *   f_R = (1/V_c(z_max)) int dV_c P_compl = int_0^{z_max} P_compl(z) u(z) dz                                   (eq. 10)
 * The completeness P_compl(z) of the line of sight is given at nc nodes zc (increasing), linear in between and constant
 * beyond the first / last node.  f_R: Gauss-Legendre on every stretch between consecutive nodes (and 0, z_max).
 * p_cat: chimo_pcat (eq. 8).  Returns f_R. */
typedef struct { const lam_t *L; int nc; const double *zc, *pc; double vmax; } compl_ctx;
static double compl_at(const compl_ctx *c, double z) {
    if (z <= c->zc[0]) return c->pc[0];
    if (z >= c->zc[c->nc - 1]) return c->pc[c->nc - 1];
    int k = 0;
    while (k + 2 < c->nc && z >= c->zc[k + 1]) ++k;
    double t = (z - c->zc[k]) / (c->zc[k + 1] - c->zc[k]);
    return c->pc[k] + t * (c->pc[k + 1] - c->pc[k]);
}
static double compl_integrand(double z, const void *ctx) {
    const compl_ctx *c = (const compl_ctx *)ctx;
    return compl_at(c, z) * dVc_dz(z, c->L) / c->vmax;
}
double chimo_pgal(const double *lam, double z_max, int n_gal, const double *zt, const double *st, const double *w, int nc,
                  const double *zc, const double *pc, int ng, const double *zg, double *out) {
    gl_init();
    const lam_t *L = (const lam_t *)lam;
    compl_ctx c = {L, nc, zc, pc, V_c(z_max, L)};
    double fR = 0.0, a = 0.0;
    for (int k = 0; k <= nc; ++k) {   /* stretches [0, zc_0], [zc_0, zc_1], ..., [zc_last, z_max], clipped to [0, z_max] */
        double b = (k < nc) ? zc[k] : z_max;
        if (b > z_max) b = z_max;
        if (b > a) { fR += gl_integrate(compl_integrand, &c, a, b, 1 + (int)((b - a) / 0.25)); a = b; }
    }
    chimo_pcat(lam, n_gal, zt, st, w, ng, zg, out);
    for (int i = 0; i < ng; ++i) {
        double u = (zg[i] <= z_max) ? dVc_dz(zg[i], L) / c.vmax : 0.0;
        out[i] = fR * out[i] + (1.0 - compl_at(&c, zg[i])) * u;
    }
    return fR;
}

/* ------------------------------------------------------------------------- O11 log L -------- */
void chimo_loglike_batch_grouped(int n_lambda, const double *lam, int placement, int bw_rule,
                         double z_cat_max, double z_table_max, int n_table, double neff_factor,
                         int n_events, const int64_t *sample_off, const double *dl,
                         const double *m1d, const double *m2d, const double *ln_prior,
                         const int64_t *grid_off, const double *zg, const double *pgal,
                         const double *fixed_bw, int64_t n_det, double n_inj_total,
                         const double *inj_dl, const double *inj_m1d, const double *inj_m2d,
                         const double *inj_ln_pdraw, int n_groups, const int64_t *group_off,
                         const double *ln_factor, double *out_loglike, double *out_event_logI,
                         double *out_logxi, double *out_neff, double *out_h, uint32_t *out_flags);

/* log L = sum_i log I_i - N_e log xi   (eq. 3) for a batch of lambda.
 * event_lo/hi select a sub-range of events (for bounded timing samples); out arrays may be NULL. */
void chimo_loglike_batch(int n_lambda, const double *lam, int placement, int bw_rule,
                         double z_cat_max, double z_table_max, int n_table, double neff_factor,
                         int n_events, const int64_t *sample_off, const double *dl,
                         const double *m1d, const double *m2d, const double *ln_prior,
                         const int64_t *grid_off, const double *zg, const double *pgal,
                         const double *fixed_bw, int64_t n_det, double n_inj_total,
                         const double *inj_dl, const double *inj_m1d, const double *inj_m2d,
                         const double *inj_ln_pdraw, double *out_loglike, double *out_event_logI,
                         double *out_logxi, double *out_neff, double *out_h, uint32_t *out_flags) {
    chimo_loglike_batch_grouped(n_lambda, lam, placement, bw_rule, z_cat_max, z_table_max, n_table, neff_factor,
                                n_events, sample_off, dl, m1d, m2d, ln_prior, grid_off, zg, pgal, fixed_bw, n_det,
                                n_inj_total, inj_dl, inj_m1d, inj_m2d, inj_ln_pdraw, 0, NULL, NULL, out_loglike,
                                out_event_logI, out_logxi, out_neff, out_h, out_flags);
}

/* "many-1d" kernel (eq. 18; eq. 14's sum over pixels; reading R20 of DESIGN.md): the n_events
 * entries are (event, pixel) SUB-events -- the N_k PE samples that fall in pixel k, the pixel's own grid and p_gal --
 * and physical event g owns the sub-events [group_off[g], group_off[g+1]):
 *     I_g = sum_k F_k I_k,   I_k = int KDE[{z_j | w_j}_{j in pixel k}](z) p_gal,k(z) dz  (O8-O9 per pixel, 1/N_k, own Scott h),
 * F_k = exp(ln_factor[k]) the hyperparameter-independent factor of eq. 18 (2-d sky KDE at the pixel centre x pixel area).
 * log L = sum_g log I_g - N_groups log xi.  n_groups = 0: every sub-event is its own event (single-1d).
 * Sparse pixels (reading R24 of DESIGN.md; PAPER.md:167-169 notes "less populated pixels" but gives no rule): a pixel whose
 * Scott bandwidth is undefined under this lambda (fewer than two samples with non-zero weight) is left out of the sum. */
void chimo_loglike_batch_grouped(int n_lambda, const double *lam, int placement, int bw_rule,
                         double z_cat_max, double z_table_max, int n_table, double neff_factor,
                         int n_events, const int64_t *sample_off, const double *dl,
                         const double *m1d, const double *m2d, const double *ln_prior,
                         const int64_t *grid_off, const double *zg, const double *pgal,
                         const double *fixed_bw, int64_t n_det, double n_inj_total,
                         const double *inj_dl, const double *inj_m1d, const double *inj_m2d,
                         const double *inj_ln_pdraw, int n_groups, const int64_t *group_off,
                         const double *ln_factor, double *out_loglike, double *out_event_logI,
                         double *out_logxi, double *out_neff, double *out_h, uint32_t *out_flags) {
    gl_init();
    const int n_phys = (n_groups > 0) ? n_groups : n_events;   /* N_obs of eq. 3 */
    for (int l = 0; l < n_lambda; ++l) {
        const double *la = lam + (size_t)l * CHIMO_NLAM;
        const lam_t *L = (const lam_t *)la;
        uint32_t fl = 0;
        double total = 0.0, logxi = 0.0, neff = NAN;
        int bad = 0;
        if (!lambda_in_domain(L)) { fl |= CHIMO_F_LAMBDA_DOMAIN; bad = 1; }
        else if (!dl_monotone(L, z_table_max, n_table)) { fl |= CHIMO_F_DL_NONMONOTONE; bad = 1; }
        if (bad) {
            out_loglike[l] = NAN;
            if (out_logxi) out_logxi[l] = NAN;
            if (out_neff) out_neff[l] = NAN;
            if (out_event_logI) for (int i = 0; i < n_events; ++i) out_event_logI[(size_t)l * n_events + i] = NAN;
            if (out_h) for (int i = 0; i < n_events; ++i) out_h[(size_t)l * n_events + i] = NAN;
            if (out_flags) out_flags[l] = fl;
            continue;
        }
        double *li = (double *)malloc(sizeof(double) * (n_events > 0 ? n_events : 1));
        uint32_t efl = 0;
#pragma omp parallel for schedule(dynamic, 1) reduction(| : efl)
        for (int i = 0; i < n_events; ++i) {
            uint32_t f = 0;
            double h;
            int64_t s0 = sample_off[i], g0 = grid_off[i];
            li[i] = chimo_event_logI(la, placement, bw_rule, fixed_bw ? fixed_bw[i] : NAN, z_table_max,
                                     (int)(sample_off[i + 1] - s0), dl + s0, m1d + s0, m2d + s0,
                                     ln_prior + s0, (int)(grid_off[i + 1] - g0), zg + g0, pgal + g0, &h, &f);
            efl |= f;
            if (out_event_logI) out_event_logI[(size_t)l * n_events + i] = li[i];
            if (out_h) out_h[(size_t)l * n_events + i] = h;
        }
        if (n_groups > 0) {   /* pixel sum of eq. 14 in log space; a pixel with I = 0 is not an empty event */
            efl &= ~CHIMO_F_EVENT_ZERO;
            for (int g = 0; g < n_groups; ++g) {
                /* R24: a pixel whose bandwidth is undefined (log I_k = NaN, BW_DEGENERATE stays raised) is left out of the
                 * pixel sum; an event none of whose pixels has I_k > 0 is NaN if a pixel was left out, else empty (-inf) */
                double mx = -INFINITY, acc = 0.0;
                int nan = 0;
                for (int64_t k = group_off[g]; k < group_off[g + 1]; ++k) {
                    double v = li[k] + ln_factor[k];
                    if (isnan(v)) nan = 1;
                    else if (v > mx) mx = v;
                }
                if (mx == -INFINITY) {
                    if (nan) total = NAN;
                    else { efl |= CHIMO_F_EVENT_ZERO; total += -INFINITY; }
                    continue;
                }
                for (int64_t k = group_off[g]; k < group_off[g + 1]; ++k) {
                    double v = li[k] + ln_factor[k];
                    if (!isnan(v)) acc += exp(v - mx);
                }
                total += mx + log(acc);
            }
        } else {
            for (int i = 0; i < n_events; ++i) total += li[i];
        }
        fl |= efl;
        free(li);
        if (n_det > 0) {
            double S1, S2;
            int rf = 0;
            chimo_selection_sums(la, z_cat_max, z_table_max, n_det, inj_dl, inj_m1d, inj_m2d,
                                 inj_ln_pdraw, &S1, &S2, NULL, &rf);
            if (rf) fl |= CHIMO_F_TABLE_RANGE;
            double xi = S1 / n_inj_total;
            neff = chimo_neff(S1, S2, n_inj_total);
            if (!(xi > 0.0)) { fl |= CHIMO_F_XI_ZERO; logxi = NAN; total = NAN; }
            else {
                logxi = log(xi);
                if (neff < neff_factor * n_phys) fl |= CHIMO_F_NEFF_LOW; /* R8: report only */
                total -= n_phys * logxi;
            }
        }
        out_loglike[l] = total;
        if (out_logxi) out_logxi[l] = logxi;
        if (out_neff) out_neff[l] = neff;
        if (out_flags) out_flags[l] = fl;
    }
}

int chimo_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
