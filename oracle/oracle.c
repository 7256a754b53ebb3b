/*
 * oracle.c -- see oracle.h.  TEST INFRASTRUCTURE ONLY; shares nothing with the CUDA path.
 *
 * Build: gcc -O2 -std=c11 -mfma -ffp-contract=off -fopenmp -shared -fPIC oracle.c -o liboracle.so -lm
 *   -ffp-contract=off : no a*b+c is fused unless written as fma(); the only fma() calls are the
 *                       two in orc_escale(), whose rounding sequence is normative (R8).
 *   -mfma             : fma() compiles to one vfmadd instead of the (equally correctly rounded)
 *                       libm software routine.
 *
 * Steps follow SURVEY.md 8(c) O1-O5, which restate PAPER.md:34-39 (Eq. 1-2), :67-83 (Eq. 3-6),
 * :119-125 (Eq. 9) and :177 (signal step 1).
 */
#include "oracle.h"

#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

/* phase = 1.267 * dm2[eV^2] * L[m] / E[MeV]  (R1: the literal 1.267, as north_star states) */
static const double K_PHASE = 1.267;

static double par(const orc_model *m, const double *theta, int slot)
{
    int idx = m->idx_osc[slot];
    return idx >= 0 ? theta[idx] : m->fixed_osc[slot];
}

/* first-octant branch theta < pi/4 (R4): cos 2theta = +sqrt(1 - sin^2 2theta) */
static void mixing(double s22, double *cos2, double *sin2, double *cos4)
{
    double c2t = sqrt(1.0 - s22);
    *cos2 = (1.0 + c2t) / 2.0;
    *sin2 = (1.0 - c2t) / 2.0;
    *cos4 = (*cos2) * (*cos2);
}

int orc_terms(const orc_model *m, const double *theta, double A[ORC_MAX_TERMS], double dm2[ORC_MAX_TERMS])
{
    double s13 = par(m, theta, 0), mee = par(m, theta, 1);
    double s12 = par(m, theta, 2), m21 = par(m, theta, 3);
    double c2_13, s2_13, c4_13, c2_12, s2_12, c4_12;
    mixing(s13, &c2_13, &s2_13, &c4_13);
    mixing(s12, &c2_12, &s2_12, &c4_12);
    (void)s2_13; (void)c4_12;

    switch (m->osc_model) {
    case ORC_EQ1:
        /* PAPER.md:34 Eq. 1:  1 - sin^2(2th13) sin^2(D_ee) - cos^4(th13) sin^2(2th12) sin^2(D_21) */
        A[0] = s13;          dm2[0] = mee;
        A[1] = c4_13 * s12;  dm2[1] = m21;
        return 2;
    case ORC_FULL3: {
        /* exact 3-flavour vacuum P_ee (BASELINE.json config 4 "with dm2_31, dm2_32"):
         *   1 - cos^4(th13) sin^2(2th12) sin^2(D_21)
         *     - sin^2(2th13) [cos^2(th12) sin^2(D_31) + sin^2(th12) sin^2(D_32)]
         * with |dm2_31|, |dm2_32| from inverting PAPER.md:39 Eq. 2 under dm2_31 - dm2_32 = dm2_21:
         *   normal   (o=+1): dm31 = mee + sin^2(th12) m21,  dm32 = mee - cos^2(th12) m21
         *   inverted (o=-1): |dm31| = mee - sin^2(th12) m21, |dm32| = mee + cos^2(th12) m21     */
        double o = m->ordering >= 0 ? 1.0 : -1.0;
        A[0] = c4_13 * s12;  dm2[0] = m21;
        A[1] = s13 * c2_12;  dm2[1] = mee + o * s2_12 * m21;
        A[2] = s13 * s2_12;  dm2[2] = mee - o * c2_12 * m21;
        return 3;
    }
    case ORC_STERILE4: {
        /* BASELINE.json config 5 (the paper prints no 3+1 formula):
         *   1 - cos^4(th14) sin^2(2th13) sin^2(D_ee) - sin^2(2th14) sin^2(D_41)
         *     - cos^4(th13) sin^2(2th12) sin^2(D_21)                                             */
        double s14 = par(m, theta, 4), m41 = par(m, theta, 5);
        double c2_14, s2_14, c4_14;
        mixing(s14, &c2_14, &s2_14, &c4_14);
        (void)c2_14; (void)s2_14;
        A[0] = c4_14 * s13;  dm2[0] = mee;
        A[1] = s14;          dm2[1] = m41;
        A[2] = c4_13 * s12;  dm2[2] = m21;
        return 3;
    }
    default:
        return -1;
    }
}

double orc_pee(int S, const double *A, const double *dm2, double L_m, double E_MeV)
{
    double x = L_m / E_MeV;
    double p = 1.0;
    for (int k = 0; k < S; ++k) {
        double c = K_PHASE * dm2[k];
        double s = sin(c * x);
        p -= A[k] * (s * s);
    }
    return p;
}

double orc_escale(double a0, double a1, double a2, double e_vis)
{
    return fma(fma(a2, e_vis, a1), e_vis, a0);
}

int32_t orc_bin(const double *edges, int32_t n_bins, double e)
{
    if (e < edges[0] || !(e < edges[n_bins])) return -1;   /* also drops NaN */
    /* upper_bound(edges, e) - 1 : last j with edges[j] <= e */
    int32_t lo = 0, hi = n_bins;                            /* invariant edges[lo] <= e < edges[hi] */
    while (hi - lo > 1) {
        int32_t mid = lo + (hi - lo) / 2;
        if (edges[mid] <= e) lo = mid; else hi = mid;
    }
    return lo;
}

/* Neumaier-compensated running sum: keeps the oracle's own rounding << 1e-9 of a bin. */
static inline void nsum(double *s, double *c, double y)
{
    double t = *s + y;
    if (!isfinite(t)) { *s = t; return; }        /* inf / NaN: nothing to compensate */
    if (fabs(*s) >= fabs(y)) *c += (*s - t) + y;
    else                     *c += (y - t) + *s;
    *s = t;
}

static int64_t total_bins(const orc_model *m)
{
    int64_t t = 0;
    for (int d = 0; d < m->n_datasets; ++d) t += m->datasets[d].n_bins;
    return t;
}

static void get_a(const orc_dataset *ds, const double *theta, double a[3])
{
    static const double dflt[3] = {0.0, 1.0, 0.0};
    for (int j = 0; j < 3; ++j) a[j] = ds->idx_a[j] >= 0 ? theta[ds->idx_a[j]] : dflt[j];
}

static int check(const orc_model *m, const orc_events *ev)
{
    if (!m || !ev || m->n_datasets <= 0) return -1;
    for (int d = 0; d < m->n_datasets; ++d)
        if (m->datasets[d].n_bins != ev[d].n_bins || ev[d].n_bins <= 0) return -2;
    return 0;
}

/* one point: signal step 1 of PAPER.md:177 -- weight every MC event with P_ee and sum per bin */
static void spectra_point(const orc_model *m, const orc_events *ev, const double *theta,
                          double *hist, double *comp, int32_t *bins_out)
{
    double A[ORC_MAX_TERMS], dm2[ORC_MAX_TERMS];
    int S = orc_terms(m, theta, A, dm2);
    int64_t off = 0, ev_off = 0;
    for (int d = 0; d < m->n_datasets; ++d) {
        const orc_events *e = &ev[d];
        const orc_dataset *ds = &m->datasets[d];
        double a[3];
        get_a(ds, theta, a);
        if (m->energy_correction == 1) { a[0] = 0.0; a[1] = 1.0; a[2] = 0.0; }    /* step 3 acts on the bins instead */
        for (int b = 0; b < e->n_bins; ++b) { hist[off + b] = 0.0; comp[off + b] = 0.0; }
        for (int64_t i = 0; i < e->n; ++i) {
            double E = (double)e->e_nu[i];
            double L = e->L_m[e->core ? e->core[i] : 0];
            double p = orc_pee(S, A, dm2, L, E);
            double v = (double)e->e_vis[i];
            double ep = orc_escale(a[0], a[1], a[2], v);
            int32_t b = orc_bin(e->edges, e->n_bins, ep);
            if (bins_out) bins_out[ev_off + i] = b;
            if (b < 0) continue;
            double wi = e->w ? (double)e->w[i] : 1.0;
            nsum(&hist[off + b], &comp[off + b], wi * p);
        }
        for (int b = 0; b < e->n_bins; ++b) hist[off + b] += comp[off + b];
        off += e->n_bins;
        ev_off += e->n;
    }
}

int orc_max_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

int orc_spectra(const orc_model *m, const orc_events *ev, int32_t P, const double *params,
                double *hist, int n_threads)
{
    int rc = check(m, ev);
    if (rc) return rc;
    int64_t TB = total_bins(m);
    int nt = n_threads > 0 ? n_threads : orc_max_threads();
    (void)nt;
#pragma omp parallel num_threads(nt)
    {
        double *comp = (double *)malloc(sizeof(double) * (size_t)TB);
#pragma omp for schedule(dynamic, 1)
        for (int32_t p = 0; p < P; ++p)
            spectra_point(m, ev, params + (int64_t)p * m->n_params, hist + (int64_t)p * TB, comp, NULL);
        free(comp);
    }
    return 0;
}

int orc_event_bins(const orc_model *m, const orc_events *ev, int32_t P, const double *params,
                   int32_t *bins)
{
    int rc = check(m, ev);
    if (rc) return rc;
    int64_t TB = total_bins(m), NE = 0;
    for (int d = 0; d < m->n_datasets; ++d) NE += ev[d].n;
    double *h = (double *)malloc(sizeof(double) * (size_t)TB * 2);
    for (int32_t p = 0; p < P; ++p)
        spectra_point(m, ev, params + (int64_t)p * m->n_params, h, h + TB, bins + (int64_t)p * NE);
    free(h);
    return 0;
}

/* ---- PAPER.md:177 steps 2-3 on the binned spectrum (R27, R28) -------------------------------------- */
double orc_escale_inverse(double a0, double a1, double a2, double t)
{
    const double c = t - a0;
    if (a2 == 0.0) return c / a1;
    return (2.0 * c) / (a1 + sqrt(a1 * a1 + 4.0 * a2 * c));
}

/* cumulative integral, from src_edges[t0], of the smoothed density that belongs to source bin b */
static double cumulative(int32_t n, const double *e, const double *h, int32_t b, double E)
{
    if (n == 1) return h[0] / (e[1] - e[0]) * (E - e[0]);
    int32_t t0 = b - 1;
    if (t0 < 0) t0 = 0;
    if (t0 > n - 3) t0 = n - 3;
    if (n == 2) {
        /* quadratic cumulative through (e0, 0), (e1, h0), (e2, h0 + h1): a straight-line density */
        const double d1 = h[0] / (e[1] - e[0]);
        const double d1b = h[1] / (e[2] - e[1]);
        const double d2 = (d1b - d1) / (e[2] - e[0]);
        return d1 * (E - e[0]) + d2 * (E - e[0]) * (E - e[1]);
    }
    /* Newton form of the cubic through the four cumulative points of bins t0, t0+1, t0+2 */
    const double *x = e + t0, *y = h + t0;
    const double f01 = y[0] / (x[1] - x[0]), f12 = y[1] / (x[2] - x[1]), f23 = y[2] / (x[3] - x[2]);
    const double f012 = (f12 - f01) / (x[2] - x[0]), f123 = (f23 - f12) / (x[3] - x[1]);
    const double f0123 = (f123 - f012) / (x[3] - x[0]);
    return f01 * (E - x[0]) + f012 * (E - x[0]) * (E - x[1]) + f0123 * (E - x[0]) * (E - x[1]) * (E - x[2]);
}

int orc_rebin_quadratic(int32_t n_src, const double *e, const double *h, int32_t n_tgt, const double *x, double *out)
{
    if (n_src < 1 || n_tgt < 0) return -1;
    for (int32_t c = 0; c < n_tgt; ++c) {
        const double lo = x[c], hi = x[c + 1];
        if (isnan(lo) || isnan(hi)) { out[c] = NAN; continue; }
        double s = 0.0;
        for (int32_t b = 0; b < n_src; ++b) {
            const double a = lo > e[b] ? lo : e[b], z = hi < e[b + 1] ? hi : e[b + 1];
            if (a < z) s += cumulative(n_src, e, h, b, z) - cumulative(n_src, e, h, b, a);
        }
        out[c] = s;
    }
    return 0;
}

/* pre-images of the bin edges under the energy scale of dataset ds at theta */
static void preimages(const orc_dataset *ds, const double *edges, const double *theta, double *x)
{
    double a[3];
    get_a(ds, theta, a);
    for (int32_t b = 0; b <= ds->n_bins; ++b) x[b] = orc_escale_inverse(a[0], a[1], a[2], edges[b]);
}

int orc_flux_scales(const orc_dataset *ds, const double *edges, const double *theta, double *f)
{
    const int32_t B = ds->n_bins, n = ds->n_flux_par;
    if (n <= 0) {
        for (int32_t b = 0; b < B; ++b) f[b] = (ds->idx_flux && ds->idx_flux[b] >= 0) ? theta[ds->idx_flux[b]] : 1.0;
        return 0;
    }
    /* the n parameters are bin averages on the uniform fine grid; "area conserving spline ... energy
     * corrected and later transformed into the original binning" (R28) */
    double *fe = (double *)malloc(sizeof(double) * (size_t)(2 * n + 1 + 2 * (B + 1)));
    if (!fe) return -3;
    double *fi = fe + n + 1, *x = fi + n, *in = x + B + 1;
    for (int32_t j = 0; j <= n; ++j) fe[j] = ds->flux_lo + ds->flux_width * (double)j;
    for (int32_t j = 0; j < n; ++j) fi[j] = theta[ds->idx_flux_par[j]] * ds->flux_width;
    preimages(ds, edges, theta, x);
    orc_rebin_quadratic(n, fe, fi, B, x, in);
    for (int32_t b = 0; b < B; ++b) {
        /* average over the pre-image: the part inside the fine grid from the spline, the rest at the nominal 1 */
        const double lo = x[b], hi = x[b + 1];
        const double a = lo > fe[0] ? lo : fe[0], z = hi < fe[n] ? hi : fe[n];
        const double inside = a < z ? z - a : 0.0;
        f[b] = (in[b] + ((hi - lo) - inside)) / (hi - lo);
    }
    free(fe);
    return 0;
}

int orc_correct_spectra(const orc_model *m, const double *const *edges, int32_t P, const double *params,
                        const double *hist, double *out)
{
    int64_t TB = total_bins(m);
    for (int32_t p = 0; p < P; ++p) {
        const double *theta = params + (int64_t)p * m->n_params;
        int64_t off = 0;
        for (int d = 0; d < m->n_datasets; ++d) {
            const orc_dataset *ds = &m->datasets[d];
            double *x = (double *)malloc(sizeof(double) * (size_t)(ds->n_bins + 1));
            if (!x) return -3;
            preimages(ds, edges[d], theta, x);
            orc_rebin_quadratic(ds->n_bins, edges[d], hist + p * TB + off, ds->n_bins, x, out + p * TB + off);
            free(x);
            off += ds->n_bins;
        }
    }
    return 0;
}

int orc_expectation(const orc_model *m, const double *const *edges, int32_t P, const double *params,
                    const double *hist, double *mu)
{
    int64_t TB = total_bins(m);
    for (int32_t p = 0; p < P; ++p) {
        const double *theta = params + (int64_t)p * m->n_params;
        int64_t off = 0;
        for (int d = 0; d < m->n_datasets; ++d) {
            const orc_dataset *ds = &m->datasets[d];
            const int32_t B = ds->n_bins;
            double eps = ds->idx_signorm >= 0 ? theta[ds->idx_signorm] : 1.0;
            double *f = (double *)malloc(sizeof(double) * (size_t)(3 * B + 1));
            if (!f) return -3;
            double *g = f + B, *x = g + B;
            if ((ds->n_flux_par > 0 || m->energy_correction == 1) && !edges) { free(f); return -4; }
            orc_flux_scales(ds, edges ? edges[d] : NULL, theta, f);
            if (m->energy_correction == 1) {
                /* step 2 (bin re-scaling) on the raw spectrum, then step 3 (energy correction of the bins) */
                for (int32_t b = 0; b < B; ++b) g[b] = f[b] * hist[p * TB + off + b];
                preimages(ds, edges[d], theta, x);
                double *gc = (double *)malloc(sizeof(double) * (size_t)B);
                if (!gc) { free(f); return -3; }
                orc_rebin_quadratic(B, edges[d], g, B, x, gc);
                for (int32_t b = 0; b < B; ++b) g[b] = gc[b];
                free(gc);
            }
            for (int b = 0; b < B; ++b) {
                double v = m->energy_correction == 1 ? eps * ds->norm * g[b]
                                                     : eps * ds->norm * f[b] * hist[p * TB + off + b];   /* signal */
                for (int k = 0; k < ds->n_bkg; ++k) {                        /* + backgrounds */
                    const orc_bkg *bk = &ds->bkg[k];
                    double r = bk->idx_rate >= 0 ? theta[bk->idx_rate] : 1.0;
                    double s = (bk->idx_shape && bk->idx_shape[b] >= 0) ? theta[bk->idx_shape[b]] : 1.0;
                    v += r * s * bk->tmpl[b];
                }
                mu[p * TB + off + b] = v;
            }
            free(f);
            off += B;
        }
    }
    return 0;
}

double orc_dev(double n, double mu)
{
    /* -ln L + ln L_saturated for one Poisson bin (Eq. 3 over PAPER.md:96 Eq. 8's
     * saturated model mu = n): the n! cancels.  DESIGN.md R9 (normalisation), R10 (edge cases). */
    if (isnan(n) || isnan(mu)) return NAN;
    if (mu < 0.0) return INFINITY;
    if (n > 0.0) {
        if (mu == 0.0) return INFINITY;
        return mu - n + n * log(n / mu);
    }
    if (n == 0.0) return mu;
    return NAN;                                  /* negative counts are not data */
}

/* a constrained quantity b(theta) that is a function of the fitted parameters (R29) */
double orc_function_value(const orc_function *f, const double *theta)
{
    double v = f->offset;
    for (int32_t m = 0; m < f->n_terms; ++m) {
        const orc_monomial *t = &f->terms[m];
        double term = t->coef;
        for (int32_t i = 0; i < t->n_factors; ++i) {
            const double x = theta[t->idx[i]];
            const int32_t pw = t->power[i], n = pw < 0 ? -pw : pw;
            if (n == 0) continue;
            double q = x;
            for (int32_t r = 1; r < n; ++r) q *= x;
            if (pw > 0) term *= q; else term /= q;
        }
        v += term;
    }
    return v;
}

/* value of entry idx of a prior block: a parameter, or a function of the parameters */
static double constrained_value(const orc_model *m, const double *theta, int32_t idx)
{
    if (idx < m->n_params) return theta[idx];
    return orc_function_value(&m->functions[idx - m->n_params], theta);
}

int orc_nll_from_mu(const orc_model *m, int32_t P, const double *params, const double *mu,
                    const double *data, double *nll)
{
    int64_t TB = total_bins(m);
    for (int32_t p = 0; p < P; ++p) {
        const double *theta = params + (int64_t)p * m->n_params;
        double s = 0.0, c = 0.0;
        for (int64_t i = 0; i < TB; ++i) nsum(&s, &c, orc_dev(data[i], mu[p * TB + i]));
        if (m->prior_mean && m->prior_sigma) {
            /* uncorrelated Gaussian priors G(b - b_bar, sigma) (Eq. 6):
             * -ln G = 1/2 ((b - b_bar)/sigma)^2 + const, constant dropped (R9) */
            for (int j = 0; j < m->n_params; ++j) {
                double sg = m->prior_sigma[j];
                if (!(sg > 0.0) || isinf(sg)) continue;
                double z = (theta[j] - m->prior_mean[j]) / sg;
                nsum(&s, &c, 0.5 * z * z);
            }
        }
        /* correlated constraints G((b - b0)^T V^-1 (b - b0)) (Eq. 9):
         * -ln G = 1/2 (b - b0)^T V^-1 (b - b0) + const, the plain double sum over i, j */
        for (int32_t k = 0; k < m->n_prior_blocks; ++k) {
            const orc_prior_block *B = &m->prior_blocks[k];
            for (int32_t i = 0; i < B->n; ++i) {
                double di = constrained_value(m, theta, B->idx[i]) - B->mean[i];
                for (int32_t j = 0; j < B->n; ++j) {
                    double dj = constrained_value(m, theta, B->idx[j]) - B->mean[j];
                    nsum(&s, &c, 0.5 * di * B->inv_cov[(int64_t)i * B->n + j] * dj);
                }
            }
        }
        nll[p] = s + c;
    }
    return 0;
}

int orc_nll(const orc_model *m, const orc_events *ev, int32_t P, const double *params,
            const double *data, double *nll, int n_threads)
{
    int64_t TB = total_bins(m);
    double *hist = (double *)malloc(sizeof(double) * (size_t)TB * (size_t)P * 2);
    if (!hist) return -3;
    double *mu = hist + (size_t)TB * (size_t)P;
    int rc = orc_spectra(m, ev, P, params, hist, n_threads);
    const double **edges = (const double **)malloc(sizeof(double *) * (size_t)m->n_datasets);
    if (!edges) { free(hist); return -3; }
    for (int d = 0; d < m->n_datasets; ++d) edges[d] = ev[d].edges;
    if (!rc) rc = orc_expectation(m, edges, P, params, hist, mu);
    free(edges);
    if (!rc) rc = orc_nll_from_mu(m, P, params, mu, data, nll);
    free(hist);
    return rc;
}

/* the affine map written out; the sum over j in index order with fma (the same
 * correctly rounded sequence on any machine). */
int orc_transform(int32_t n_params, int32_t n_u, const int32_t *copy_src, const double *copy_const,
                  int32_t n_blocks, const orc_transform_block *blocks, int32_t P, const double *u, double *theta)
{
    for (int32_t p = 0; p < P; ++p) {
        const double *up = u + (int64_t)p * n_u;
        double *tp = theta + (int64_t)p * n_params;
        for (int32_t j = 0; j < n_params; ++j) {
            if (copy_src[j] >= n_u) return -1;
            tp[j] = copy_src[j] >= 0 ? up[copy_src[j]] : (copy_const ? copy_const[j] : 0.0);
        }
        for (int32_t k = 0; k < n_blocks; ++k) {
            const orc_transform_block *B = &blocks[k];
            for (int32_t i = 0; i < B->n_out; ++i) {
                double acc = B->offset[i];
                for (int32_t j = 0; j < B->n_in; ++j)
                    acc = fma(B->matrix[(int64_t)i * B->n_in + j], up[B->idx_in[j]] - B->centre[j], acc);
                tp[B->idx_out[i]] = acc;
            }
        }
    }
    return 0;
}

/* ---- pseudo-experiments (section 4.1: "test statistics derived from large ensembles of
 * pseudo-experiments"): Poisson-fluctuated counts n[e][i] ~ Poisson(mu[i]).  The paper names no generator and no
 * sampler; R26 fixes both so that the counts are a function of (seed, experiment, bin, mu) alone:
 *
 *   uniform   Philox4x32-10 (Salmon et al., SC'11), counter (bin, experiment, 0, 0), key = the 64-bit seed;
 *             u = (x0 * 2^21 + (x1 >> 11)) * 2^-53 in [0, 1), x0, x1 the first two output words;
 *   sampler   exact inversion of the Poisson distribution from its mode outwards, using only +, *, / (every
 *             operation correctly rounded, hence the same bits on any IEEE machine):
 *               weights relative to the mode m = floor(mu):  w_m = 1,  w_{k+1} = w_k * (mu / (k+1)),
 *                                                            w_{k-1} = w_k * (k / mu)     (pmf ratios)
 *               Z = (sum of the left weights, outwards until a term no longer changes the sum)
 *                   + 1 + (the same to the right)                                  [orc_poisson_norm]
 *               the interval [0, Z) is cut into pieces of length w_k in the order m, m+1, m-1, m+2, m-2, ...;
 *               the count is the k whose piece holds u * Z                          [orc_poisson_inv]
 *             P(k) = w_k / Z = the Poisson pmf up to the rounding of ~10 sqrt(mu) additions (1e-13).
 * Cost O(sqrt(mu)) per draw. */
static void mulhilo32(uint32_t a, uint32_t b, uint32_t *hi, uint32_t *lo)
{
    uint64_t p = (uint64_t)a * (uint64_t)b;
    *hi = (uint32_t)(p >> 32);
    *lo = (uint32_t)p;
}

void orc_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4])
{
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3], k0 = key[0], k1 = key[1];
    for (int r = 0; r < 10; ++r) {
        uint32_t hi0, lo0, hi1, lo1;
        mulhilo32(0xD2511F53u, c0, &hi0, &lo0);
        mulhilo32(0xCD9E8D57u, c2, &hi1, &lo1);
        uint32_t n0 = hi1 ^ c1 ^ k0, n1 = lo1, n2 = hi0 ^ c3 ^ k1, n3 = lo0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        k0 += 0x9E3779B9u;                       /* golden-ratio Weyl sequence on the key */
        k1 += 0xBB67AE85u;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

double orc_uniform53(uint64_t seed, uint32_t bin, uint32_t experiment)
{
    uint32_t ctr[4] = {bin, experiment, 0u, 0u}, key[2] = {(uint32_t)seed, (uint32_t)(seed >> 32)}, x[4];
    orc_philox4x32_10(ctr, key, x);
    return (double)(((uint64_t)x[0] << 21) | (uint64_t)(x[1] >> 11)) * 0x1p-53;
}

double orc_poisson_norm(double mu)
{
    if (!(mu > 0.0) || isinf(mu) || mu > 1e9) return 1.0;     /* outside the domain (R26): Z is not used */
    const double m = floor(mu);
    double L = 0.0, R = 0.0, t = 1.0;
    for (double k = m; k >= 1.0; k -= 1.0) {     /* w_{k-1} = w_k * (k / mu) */
        t = t * (k / mu);
        if (L + t == L) break;
        L += t;
    }
    t = 1.0;
    for (double k = m + 1.0;; k += 1.0) {        /* w_k = w_{k-1} * (mu / k) */
        t = t * (mu / k);
        if (R + t == R) break;
        R += t;
    }
    return (L + 1.0) + R;
}

double orc_poisson_inv(double mu, double Z, double u)
{
    if (mu > 1e9 && !isinf(mu)) return NAN;      /* DESIGN.md R26: a finite mu above 1e9 is outside the domain */
    if (!(mu > 0.0) || isinf(mu)) return 0.0;
    const double m = floor(mu), target = u * Z;
    double acc = 1.0, tr = 1.0, tl = 1.0, kr = m, kl = m;
    if (target < acc) return m;
    for (;;) {
        kr += 1.0;
        tr = tr * (mu / kr);
        acc += tr;
        if (target < acc) return kr;
        int left_done = 1;
        if (kl >= 1.0) {
            tl = tl * (kl / mu);
            kl -= 1.0;
            const double before = acc;
            acc += tl;
            if (target < acc) return kl;
            left_done = acc == before;
        }
        /* both tails exhausted and u * Z still not reached (it can sit within rounding of Z): the last piece */
        if (acc + tr == acc && left_done) return kr;
    }
}

int orc_draw_pseudo_data(int64_t total_bins_, const double *mu, int32_t E, uint64_t seed, double *data)
{
    for (int64_t i = 0; i < total_bins_; ++i) {
        const double Z = orc_poisson_norm(mu[i]);
        for (int32_t e = 0; e < E; ++e)
            data[(int64_t)e * total_bins_ + i] = orc_poisson_inv(mu[i], Z, orc_uniform53(seed, (uint32_t)i, (uint32_t)e));
    }
    return 0;
}


/* PAPER.md:155; R30: one variable-metric (MIGRAD-type) step: rank-two update of the inverse Hessian estimate,
 * Newton direction, estimated distance to the minimum */
int orc_variable_metric_step(int32_t N, double *V, const double *dx, const double *dg, const double *grad,
                             double *direction, double *edm)
{
    int skipped = 0;
    if (dx && dg) {
        double *vg = (double *)malloc(sizeof(double) * (size_t)(N > 0 ? N : 1));
        if (!vg) return -3;
        double a = 0.0, b = 0.0;
        for (int32_t i = 0; i < N; ++i) {
            double s = 0.0;
            for (int32_t j = 0; j < N; ++j) s += V[(int64_t)i * N + j] * dg[j];
            vg[i] = s;
        }
        for (int32_t i = 0; i < N; ++i) a += dx[i] * dg[i];
        for (int32_t i = 0; i < N; ++i) b += dg[i] * vg[i];
        if (a > 0.0 && b > 0.0) {
            for (int32_t i = 0; i < N; ++i)
                for (int32_t j = 0; j < N; ++j) {
                    double v = V[(int64_t)i * N + j];
                    v += dx[i] * dx[j] / a;
                    v -= vg[i] * vg[j] / b;
                    if (a > b) {
                        const double ui = dx[i] / a - vg[i] / b, uj = dx[j] / a - vg[j] / b;
                        v += b * ui * uj;
                    }
                    V[(int64_t)i * N + j] = v;
                }
        } else {
            skipped = 1;
        }
        free(vg);
    }
    double e = 0.0;
    for (int32_t i = 0; i < N; ++i) {
        double s = 0.0;
        for (int32_t j = 0; j < N; ++j) s += V[(int64_t)i * N + j] * grad[j];
        direction[i] = -s;
        e += grad[i] * s;
    }
    *edm = 0.5 * e;
    return skipped;
}
