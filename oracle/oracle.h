/*
 * oracle.h -- plain CPU oracle for the oscillation-weighted event spectrum and the binned
 * Poisson negative log-likelihood of arXiv 2502.15253 (PhyLiNO).
 *
 * TEST INFRASTRUCTURE ONLY.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may build, load or call this.  It shares no code, header, table or
 * constant with the CUDA path under paper_2502_15253_b200/ and neither includes the other.
 *
 * Everything is straight double-precision loops in the caller's event order, libm sin/log/sqrt,
 * std fma() where the rounding sequence is normative.  Citations are PAPER.md line numbers
 * and DESIGN.md reading numbers (R1...).
 *
 * Pins (tests/test_oracle_*.py): every function below is pinned by closed forms, invariants,
 * mpmath / exact-rational brute force, textbook identities, published known-answer vectors (Philox) and
 * goodness of fit against scipy.stats (Poisson sampler); none is "parity unpinned".
 * End-to-end numeric values are NOT pinned against the paper: it prints no spectrum or
 * likelihood value and its inputs are not public ("What pins the oracle").
 */
#ifndef PHYLINO_ORACLE_H
#define PHYLINO_ORACLE_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

enum { ORC_EQ1 = 0, ORC_FULL3 = 1, ORC_STERILE4 = 2 };
enum { ORC_MAX_TERMS = 3 };

/* MC events of one dataset, caller order. */
typedef struct {
    int64_t        n;
    const float   *e_nu;     /* [n] true neutrino energy, MeV */
    const float   *e_vis;    /* [n] reconstructed energy, MeV */
    const float   *w;        /* [n] MC weight, NULL => 1 */
    const int32_t *core;     /* [n] reactor-core index, NULL => 0 */
    int32_t        n_cores;
    const double  *L_m;      /* [n_cores] baselines, metres */
    int32_t        n_bins;
    const double  *edges;    /* [n_bins+1] strictly ascending */
} orc_events;

typedef struct {
    int32_t        idx_rate;   /* -1 => 1 */
    const double  *tmpl;       /* [n_bins] */
    const int32_t *idx_shape;  /* [n_bins] or NULL => 1 */
} orc_bkg;

typedef struct {
    int32_t        n_bins;
    int32_t        idx_a[3];     /* -1 => (0,1,0) */
    int32_t        idx_signorm;  /* -1 => 1 */
    double         norm;
    const int32_t *idx_flux;     /* [n_bins] or NULL => 1 */
    int32_t        n_bkg;
    const orc_bkg *bkg;
    /* reactor-flux model on a uniform fine grid (R28): n_flux_par > 0 replaces idx_flux.
     * theta[idx_flux_par[j]] is the average flux correction on [flux_lo + j flux_width, flux_lo + (j+1) flux_width) */
    int32_t        n_flux_par;
    const int32_t *idx_flux_par; /* [n_flux_par] */
    double         flux_lo, flux_width;
} orc_dataset;

/* One correlated Gaussian constraint: (b - b0)^T V^-1 (b - b0) over the parameters idx
 * (third factor of Eq. 9; "multiple parameters with correlations"). */
typedef struct {
    int32_t        n;
    const int32_t *idx;        /* [n] indices into theta */
    const double  *mean;       /* [n] b0 */
    const double  *inv_cov;    /* [n*n] V^-1, row-major */
} orc_prior_block;

/* A constrained quantity that is a FUNCTION of the fitted parameters ("a generalized parametrization
 * where the constrained parameters b_i(theta) are functions of the actually fitted nuisance parameters"; the paper
 * names no function family -- DESIGN.md R29: polynomials with integer powers,
 *     b(theta) = offset + sum_m coef_m prod_i theta[idx_mi]^power_mi,
 * which covers affine maps, products (rate x efficiency) and ratios).  A prior block refers to function f through the
 * index n_params + f. */
typedef struct {
    double         coef;
    int32_t        n_factors;
    const int32_t *idx;        /* [n_factors] indices into theta */
    const int32_t *power;      /* [n_factors] integer powers, negative = divide */
} orc_monomial;

typedef struct {
    double              offset;
    int32_t             n_terms;
    const orc_monomial *terms;
} orc_function;

typedef struct {
    int32_t            osc_model;    /* ORC_EQ1 / ORC_FULL3 / ORC_STERILE4 */
    int32_t            ordering;     /* +1 normal, -1 inverted (FULL3) */
    int32_t            n_params;
    int32_t            n_datasets;
    int32_t            idx_osc[6];   /* s13, mee, s12, m21, s14, m41; -1 => fixed_osc */
    double             fixed_osc[6];
    const orc_dataset *datasets;
    const double      *prior_mean;   /* [n_params] or NULL */
    const double      *prior_sigma;  /* [n_params] or NULL; <=0, inf or NaN => unconstrained */
    int32_t                n_prior_blocks;
    const orc_prior_block *prior_blocks; /* [n_prior_blocks] or NULL */
    int32_t            energy_correction; /* 0: per event before binning (north_star; R8);
                                             1: on the binned spectrum (PAPER.md:177 step 3; R27) */
    int32_t             n_functions;  /* constrained functions of theta (R29); prior blocks reach function f */
    const orc_function *functions;    /* through the index n_params + f */
} orc_model;

/* b(theta) of one function: offset + sum over the terms, in order, of coef x the factors in order, a factor being
 * theta^|power| by repeated multiplication, multiplied in (power > 0) or divided out (power < 0); power 0 is 1. */
double orc_function_value(const orc_function *f, const double *theta);

/* O1-O2: amplitudes A_k and mass splittings m_k [eV^2] of the oscillation terms at one point.
 * Returns the number of terms S (2 or 3).  PAPER.md:34 (Eq. 1), :39 (Eq. 2), BASELINE.json config 5. */
int orc_terms(const orc_model *m, const double *theta, double A[ORC_MAX_TERMS], double dm2[ORC_MAX_TERMS]);

/* P_ee = 1 - sum_k A_k sin^2(1.267 dm2_k L/E)   (Eq. 1; phase constant: DESIGN.md R1). */
double orc_pee(int S, const double *A, const double *dm2, double L_m, double E_MeV);

/* Energy-scale map E' = fma(fma(a2,v,a1),v,a0)  (R8). */
double orc_escale(double a0, double a1, double a2, double e_vis);

/* Bin of E' in half-open bins [edges[b], edges[b+1]); -1 if outside or NaN (R7). */
int32_t orc_bin(const double *edges, int32_t n_bins, double e);

/* O3: hist[p][off_d + b] = sum_i w_i P_ee(i,p) over events of dataset d landing in bin b.
 * hist is [P][total_bins] row-major, dataset-major inside a point.  n_threads <= 0 => all cores
 * (parallel over points only; each point sums its events sequentially in input order). */
int orc_spectra(const orc_model *m, const orc_events *ev, int32_t P, const double *params,
                double *hist, int n_threads);

/* Same, additionally writing the bin index of every event of every dataset at point p
 * (bins[p][i] over the concatenated events, -1 = dropped).  For bit-exact bin-assignment parity. */
int orc_event_bins(const orc_model *m, const orc_events *ev, int32_t P, const double *params,
                   int32_t *bins);

/* O4: mu[p][off_d+b] = eps_d norm_d f_db H + sum_k r_dk s_dkb T_dkb.
 * energy_correction = 1: hist is the RAW (identity-binned) step-1 spectrum, and the signal part is
 * eps_d norm_d C_a(f_d . H)_b with C_a the bin-level correction above (step 2, then step 3).
 * edges: per dataset [n_bins + 1]; needed only with energy_correction = 1 or a flux model, else may be NULL. */
int orc_expectation(const orc_model *m, const double *const *edges, int32_t P, const double *params,
                    const double *hist, double *mu);

/* Half-deviance of one bin, mu - n + n ln(n/mu)  (PAPER.md:67 Eq. 3, :96 Eq. 8; R9-R10). */
double orc_dev(double n, double mu);

/* O5: nll[p] = sum_bins dev(n, mu) + 1/2 sum_j ((theta_j - mean_j)/sigma_j)^2
 *             + 1/2 sum_blocks (b - b0)^T V^-1 (b - b0)            (PAPER.md:82 Eq. 6, :119-123 Eq. 9),
 * b_i = theta[idx_i], or the function idx_i - n_params of theta where idx_i >= n_params (R29). */
int orc_nll_from_mu(const orc_model *m, int32_t P, const double *params, const double *mu,
                    const double *data, double *nll);

/* O3+O4+O5 in one call. */
int orc_nll(const orc_model *m, const orc_events *ev, int32_t P, const double *params,
            const double *data, double *nll, int n_threads);

/* Transformation layer between the minimiser's parameters u and the model parameters theta (PAPER.md:171
 * "A transformation layer applies the covariance of any changed model parameter"; "the 9 polynomial
 * coefficients can be expressed by 7 independent parameters"):
 *   theta_j = u[copy_src[j]]  (or copy_const[j] where copy_src[j] < 0), then for every block, in order,
 *   theta[idx_out[i]] = offset[i] + sum_j matrix[i][j] (u[idx_in[j]] - centre[j]). */
typedef struct {
    int32_t        n_out, n_in;
    const int32_t *idx_out;
    const int32_t *idx_in;
    const double  *offset;     /* [n_out] */
    const double  *centre;     /* [n_in] */
    const double  *matrix;     /* [n_out * n_in] row-major */
} orc_transform_block;

int orc_transform(int32_t n_params, int32_t n_u, const int32_t *copy_src, const double *copy_const,
                  int32_t n_blocks, const orc_transform_block *blocks, int32_t P, const double *u, double *theta);

/* ---- the paper's own signal steps 2-3 on the BINNED spectrum (R27, R28) --------------
 * "The expectation is smoothed using a second-degree polynomial function.  These corrected bins entries are then
 * integrated over the original binning" -- the paper gives no formula; the reading taken (R27):
 *   smoothing   inside source bin b the density is the parabola whose integrals over three consecutive bins
 *               (b-1, b, b+1; the first / last three at the ends) equal their contents, i.e. the derivative of the
 *               cubic through the four cumulative points of that triple (2 bins: straight line; 1 bin: constant);
 *   correction  content arriving in [t_c, t_c+1) of the corrected energy E' = a0 + a1 E + a2 E^2 is the integral
 *               of that density over the pre-image [x_c, x_c+1), x = E'^-1(t) on the branch through (t - a0)/a1.
 * orc_escale_inverse: x with a0 + a1 x + a2 x^2 = t, as 2 (t - a0) / (a1 + sqrt(a1^2 + 4 a2 (t - a0))).
 * orc_rebin_quadratic: out[c] = integral over [x[c], x[c+1]) of the smoothed density of (src_edges, src_int);
 *   x ascending, n_tgt + 1 values; nothing outside the source range; NaN in x gives NaN out.
 * orc_correct_spectra: applies the correction of the point's energy-scale parameters to every dataset of raw
 *   (identity-binned) spectra hist [P x total_bins] -> out: what the product's spectra call returns in mode 1.
 * orc_flux_scales: f[b] of dataset d at theta (R28): the fine-grid flux parameters, smoothed the same way, averaged
 *   over the pre-image of analysis bin b under the dataset's energy scale; 1 outside the fine grid. */
double orc_escale_inverse(double a0, double a1, double a2, double t);
int    orc_rebin_quadratic(int32_t n_src, const double *src_edges, const double *src_int, int32_t n_tgt,
                           const double *x, double *out);
int    orc_correct_spectra(const orc_model *m, const double *const *edges, int32_t P, const double *params,
                           const double *hist, double *out);
int    orc_flux_scales(const orc_dataset *ds, const double *edges, const double *theta, double *f);

/* Pseudo-experiments (R26): Philox4x32-10 counter-based uniforms and the exact
 * mode-outward inversion of the Poisson distribution built from +, *, / only (see oracle.c).
 *   orc_philox4x32_10   one block of the generator (Random123 reference algorithm)
 *   orc_uniform53       u in [0,1) of (seed, bin, experiment): counter (bin, experiment, 0, 0), key = seed
 *   orc_poisson_norm    Z(mu) = sum of the pmf weights relative to the mode
 *   orc_poisson_inv     the count for uniform u
 *   orc_draw_pseudo_data  data[e][i] = orc_poisson_inv(mu[i], Z(mu[i]), orc_uniform53(seed, i, e)) */
void   orc_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]);
double orc_uniform53(uint64_t seed, uint32_t bin, uint32_t experiment);
double orc_poisson_norm(double mu);
double orc_poisson_inv(double mu, double Z, double u);
int    orc_draw_pseudo_data(int64_t total_bins, const double *mu, int32_t E, uint64_t seed, double *data);

/* One variable-metric step of the minimiser's loop ("This function is minimized by iteratively modifying
 * the model parameters until the estimated distance to the minimum is smaller than a predefined threshold"; the
 * minimiser is Minuit2's MIGRAD [28], a variable-metric method -- the paper prints no formula; R30 takes the
 * published rule).  V [N x N] is the current estimate of the INVERSE Hessian of the NLL (symmetric), updated in place
 * from the last move dx = x_new - x_old and the change of the gradient dg = g_new - g_old (both NULL: no update):
 *     vg = V dg,  a = dx.dg,  b = dg.vg
 *     V += dx dx^T / a - vg vg^T / b                                  (Davidon-Fletcher-Powell)
 *     V += b u u^T,  u = dx / a - vg / b          where a > b        (the rank-one term that makes it BFGS)
 * skipped (V unchanged, return value 1) unless a > 0 and b > 0.  Then
 *     direction = -V grad,   edm = 1/2 grad^T V grad   (the estimated distance to the minimum).
 * All sums run in index order in plain double arithmetic. */
int orc_variable_metric_step(int32_t N, double *V, const double *dx, const double *dg, const double *grad,
                             double *direction, double *edm);

/* Number of threads orc_spectra would use for n_threads <= 0. */
int orc_max_threads(void);

#ifdef __cplusplus
}
#endif
#endif
