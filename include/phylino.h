/*
 * phylino.h -- C-ABI of the B200 (sm_100a) hot path of PhyLiNO's forward-folding likelihood
 * fit (arXiv 2502.15253): the oscillation-weighted MC event spectrum, batched over parameter
 * points, and the binned Poisson negative log-likelihood with Gaussian priors.
 *
 * Citations are line numbers of /root/reference/PAPER.md and reading numbers (R1...) of DESIGN.md.
 *
 * What the library computes, for every parameter point p of a batch (signal step 1):
 *
 *   P_ee(e,p) = 1 - sum_k A_k(p) sin^2( 1.267 dm2_k(p)[eV^2] L_core(e)[m] / E_nu(e)[MeV] )
 *               (PAPER.md:34 Eq. 1, :39 Eq. 2; 3-flavour and 3+1 forms: DESIGN.md R2, R15)
 *   E'(e,p)   = fma(fma(a2, v, a1), v, a0),  v = (double)E_vis(e)          (R8)
 *   H[p,d,b]  = sum over MC events e of dataset d with edges[b] <= E' < edges[b+1] of w(e) P_ee(e,p)
 *   mu[p,d,b] = eps_d norm_d f_db H[p,d,b] + sum_k r_dk s_dkb T_dkb
 *   nll[p]    = sum_{d,b} [mu - n + n ln(n/mu)] + 1/2 sum_j ((theta_j - mean_j)/sigma_j)^2
 *               + 1/2 sum_blocks (b - b0)^T V^-1 (b - b0)     (phylino_set_prior_blocks)
 *               (PAPER.md:67-83 Eq. 3-6, :96 Eq. 8, :119-125 Eq. 9; R9, R10)
 *
 * Conventions
 *   Pointers  : every pointer argument says HOST or DEVICE.  DEVICE pointers must belong to the
 *               CUDA device the context was created on.
 *   Ownership : the context deep-copies everything handed to phylino_set_model and
 *               phylino_load_events and owns all device memory it allocates.  The caller owns
 *               `params`, `data` and the outputs; they must stay alive until the stream has
 *               passed the call.
 *   Async     : phylino_spectra / phylino_nll / phylino_expectation / phylino_nll_ensemble /
 *               phylino_event_bins only enqueue work on the context's stream and return; they
 *               never touch host-visible output, and they synchronise the stream in ONE case only:
 *               when a batch is larger than any before it on this context, the per-point work
 *               buffers grow (stream synchronise + cudaMalloc).  phylino_reserve(ctx, max_points)
 *               sizes them once, after which these calls never synchronise (required before the
 *               stream is captured into a CUDA graph).  phylino_load_events / phylino_set_model /
 *               phylino_set_transform / phylino_set_prior_blocks synchronise the stream.
 *   Errors    : every entry point returns a phylino_status; nothing throws across the ABI.
 *               Shape / state problems are detected on the host before any launch.  The text of
 *               the last error of a context is kept in phylino_last_error().  VALUE problems in
 *               device-resident `params` (NaN, sin^2 2theta above 1) are not errors: they
 *               propagate as NaN into that point's outputs, as sqrt of a negative does.  One more
 *               value rule: a point whose oscillation amplitudes have sum_k |A_k| > 3 (reachable only
 *               with sin^2 2theta far below 0, e.g. -2: cos^4 theta > 2) reads NaN in every bin --
 *               the 64-bit fixed-point bin accumulators are scaled for |P_ee| <= 4 (R19).
 *   Threads   : one context must not be used from two host threads at once; any number of
 *               contexts may coexist (independent fits).
 *   Determinism: identical inputs give bit-identical outputs on every call (64-bit fixed-point
 *               bin accumulators: integer addition is associative).
 *   No CPU fallback: without a CUDA device phylino_create fails with PHYLINO_ERR_CUDA.
 */
#ifndef PHYLINO_H
#define PHYLINO_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#if defined(__GNUC__)
#define PHYLINO_API __attribute__((visibility("default")))
#else
#define PHYLINO_API
#endif

#define PHYLINO_MAX_DATASETS 32     /* PAPER.md:209 splits Double Chooz into 18 histograms */
#define PHYLINO_MAX_BINS     2048   /* per dataset */
#define PHYLINO_MAX_BKG      8      /* background contributions per dataset (3-4) */

typedef struct phylino_ctx phylino_ctx;   /* opaque */

typedef enum {
    PHYLINO_OK        = 0,
    PHYLINO_ERR_ARG   = 1,   /* NULL pointer, negative size, non-finite weight or baseline, ... */
    PHYLINO_ERR_SHAPE = 2,   /* sizes disagree with the model (n_bins, dataset index, P < 0, ...) */
    PHYLINO_ERR_STATE = 3,   /* call order: set_model -> load_events (all datasets) -> spectra/nll */
    PHYLINO_ERR_OOM   = 4,   /* host or device allocation failed */
    PHYLINO_ERR_CUDA  = 5    /* any other CUDA runtime error (text in phylino_last_error) */
} phylino_status;

typedef enum {
    PHYLINO_OSC_EQ1      = 0,  /* PAPER.md:34 Eq. 1: terms (sin^2 2th13, dm2_ee), (cos^4 th13 sin^2 2th12, dm2_21) */
    PHYLINO_OSC_FULL3    = 1,  /* exact 3-flavour vacuum P_ee with dm2_31, dm2_32 from Eq. 2 (R2) */
    PHYLINO_OSC_STERILE4 = 2   /* 3+1 extension (formula of BASELINE.json config 5; R15) */
} phylino_osc_model;

/* slots of idx_osc / fixed_osc */
enum { PHYLINO_S13 = 0, PHYLINO_MEE = 1, PHYLINO_S12 = 2, PHYLINO_M21 = 3, PHYLINO_S14 = 4, PHYLINO_M41 = 5 };

/* One background contribution of a dataset: rate * shape_b * template_b. HOST pointers. */
typedef struct {
    int32_t        idx_rate;     /* index into theta of the rate multiplier, -1 => 1 */
    const double  *tmpl;         /* HOST [n_bins] expected counts at rate = shape = 1 */
    const int32_t *idx_shape;    /* HOST [n_bins] indices into theta (-1 => 1), or NULL => all 1 */
} phylino_bkg_desc;

/* How theta acts on one dataset. HOST pointers. */
typedef struct {
    int32_t        n_bins;
    int32_t        idx_a[3];     /* energy-scale a0,a1,a2; -1 => 0,1,0 */
    int32_t        idx_signorm;  /* signal normalisation multiplier eps_d; -1 => 1 */
    double         norm;         /* constant MC -> data normalisation (R16) */
    const int32_t *idx_flux;     /* HOST [n_bins] per-bin flux scale f_db, or NULL => all 1 */
    int32_t        n_bkg;        /* 0 ... PHYLINO_MAX_BKG */
    const phylino_bkg_desc *bkg; /* HOST [n_bkg] */
} phylino_dataset_desc;

typedef struct {
    int32_t  osc_model;          /* phylino_osc_model */
    int32_t  ordering;           /* +1 normal, -1 inverted; PHYLINO_OSC_FULL3 only (R5) */
    int32_t  n_params;           /* NPAR, length of one parameter point theta */
    int32_t  n_datasets;         /* D, 1 ... PHYLINO_MAX_DATASETS */
    int32_t  idx_osc[6];         /* indices into theta of sin^2 2th13, dm2_ee, sin^2 2th12, dm2_21,
                                    sin^2 2th14, dm2_41; -1 => fixed_osc[slot] */
    double   fixed_osc[6];
    const phylino_dataset_desc *datasets;   /* HOST [n_datasets] */
    const double *prior_mean;    /* HOST [n_params] or NULL (no priors) */
    const double *prior_sigma;   /* HOST [n_params] or NULL; sigma <= 0, inf or NaN => unconstrained
                                    (sin^2 2th13 is left free) */
} phylino_model_desc;

/* One correlated Gaussian constraint over several parameters ("multiple parameters with
 * correlations", third factor of Eq. 9): G((b - b0)^T V^-1 (b - b0)) with b = theta[idx].
 * HOST pointers, deep-copied. */
typedef struct {
    int32_t        n;          /* parameters in the block, 1 ... PHYLINO_MAX_BLOCK */
    const int32_t *idx;        /* HOST [n] indices into theta, each 0 ... n_params-1; or n_params + f for the
                                  constrained function f of phylino_set_functions */
    const double  *mean;       /* HOST [n] central values b0 */
    const double  *inv_cov;    /* HOST [n*n] INVERSE covariance V^-1, row-major; used as written (an
                                  unsymmetric matrix counts as its symmetric part) */
} phylino_prior_block;
#define PHYLINO_MAX_BLOCK 1024

/* A constrained quantity that is a FUNCTION of the fitted parameters ("a generalized parametrization where
 * the constrained parameters b_i(theta) are functions of the actually fitted nuisance parameters"; the paper names no
 * function family -- DESIGN.md R29: polynomials with integer powers),
 *     b(theta) = offset + sum_m coef_m prod_i theta[idx_mi]^power_mi :
 * affine maps, products (rate x efficiency), ratios.  Evaluated as written: the terms in order, inside a term the
 * factors in order, a factor being theta^|power| by repeated multiplication, multiplied in (power > 0) or divided out
 * (power < 0); power 0 is 1.  HOST pointers, deep-copied. */
typedef struct {
    double         coef;
    int32_t        n_factors;  /* 0 ... PHYLINO_MAX_FACTORS */
    const int32_t *idx;        /* HOST [n_factors] indices into theta */
    const int32_t *power;      /* HOST [n_factors], |power| <= PHYLINO_MAX_POWER */
} phylino_monomial;
typedef struct {
    double                  offset;
    int32_t                 n_terms;
    const phylino_monomial *terms;   /* HOST [n_terms] */
} phylino_function;
#define PHYLINO_MAX_FACTORS 16
#define PHYLINO_MAX_POWER   16

/* One block of the transformation layer between the minimiser's parameters u and the model parameters theta
 * ("A transformation layer applies the covariance of any changed model parameter within the
 * calculation of the likelihood"; "the 9 polynomial coefficients can be expressed by 7 independent
 * parameters"): theta[idx_out[i]] = offset[i] + sum_j matrix[i][j] (u[idx_in[j]] - centre[j]).  A Cholesky factor
 * of a covariance is a square block, the 9 <- 7 energy-response map a 9 x 7 one.  HOST pointers, deep-copied. */
typedef struct {
    int32_t        n_out, n_in;   /* 1 ... PHYLINO_MAX_BLOCK each */
    const int32_t *idx_out;       /* HOST [n_out] indices into theta */
    const int32_t *idx_in;        /* HOST [n_in] indices into u */
    const double  *offset;        /* HOST [n_out] */
    const double  *centre;        /* HOST [n_in] */
    const double  *matrix;        /* HOST [n_out * n_in] row-major */
} phylino_transform_block;

/* Create a context on CUDA device `device`.  `cuda_stream` is a cudaStream_t (0 = default stream)
 * on which all later work of this context is enqueued.  Fails with PHYLINO_ERR_CUDA when there is
 * no such device (there is no CPU fallback). */
PHYLINO_API phylino_status phylino_create(int device, void *cuda_stream, phylino_ctx **out);

/* Frees everything the context owns.  NULL is allowed. */
PHYLINO_API void phylino_destroy(phylino_ctx *ctx);

/* Deep-copies the model.  Drops events loaded under an earlier model. */
PHYLINO_API phylino_status phylino_set_model(phylino_ctx *ctx, const phylino_model_desc *model);

/* Event store of dataset `dataset` (MC events with the full detector response;
 * :191 "copied to the GPU memory only once").  All pointers HOST; arrays are copied.
 *   e_nu_MeV  [n] true neutrino energy (finite, > 0)
 *   e_vis_MeV [n] reconstructed energy (NaN allowed: such an event never lands in a bin)
 *   weight    [n] MC weight (finite), NULL => 1
 *   core      [n] reactor-core index in [0, n_cores), NULL => 0       (R13)
 *   baseline_m[n_cores] L in metres (finite, >= 0)
 *   edges     [n_bins+1] strictly ascending reco-energy bin edges; n_bins must equal the model's.
 * The store is sorted by reconstructed energy ("sorted according to their energy";
 * R14) and cut into records of 4 events: x = L_core/E_nu as fp64 and E_vis as fp32 -- 12 bytes per event
 * when every weight is exactly 1 (or NULL), else 24 with the weights as fp64.
 * n = 0 is allowed (empty dataset).  Reloading a dataset replaces it. */
PHYLINO_API phylino_status phylino_load_events(phylino_ctx *ctx, int dataset, int64_t n,
                                   const float *e_nu_MeV, const float *e_vis_MeV, const float *weight,
                                   const int32_t *core, int n_cores, const double *baseline_m,
                                   int n_bins, const double *edges);

/* H[p, off_d + b] for P parameter points (PAPER.md:177 step 1; Eq. 1).
 *   params DEVICE [P x n_params] row-major;  hist DEVICE [P x total_bins], dataset-major inside a point.
 * P = 0 is a no-op. */
PHYLINO_API phylino_status phylino_spectra(phylino_ctx *ctx, int P, const double *params, double *hist);

/* nll[p] (PAPER.md:67-83 Eq. 3-6, :119-125 Eq. 9): spectra, expectation assembly and the
 * Poisson half-deviance + prior reduction, all on the device.
 *   params DEVICE [P x n_params]; data DEVICE [total_bins] observed counts n_db; nll DEVICE [P]. */
PHYLINO_API phylino_status phylino_nll(phylino_ctx *ctx, int P, const double *params, const double *data, double *nll);

/* mu[p, off_d + b]: the spectra followed by the expectation assembly (PAPER.md:105-107, :177 step 2
 * reduced to per-bin multipliers): mu = eps_d norm_d f_db H + sum_k r_dk s_dkb T_dkb.
 *   params DEVICE [P x n_params]; mu DEVICE [P x total_bins]. */
PHYLINO_API phylino_status phylino_expectation(phylino_ctx *ctx, int P, const double *params, double *mu);

/* Diagnostic for the bit-exact bin-assignment parity test: bins[p, i] = bin index b (within its
 * dataset) of event i at point p, -1 if E' falls outside [edges[0], edges[n_bins]) or is NaN.
 * i runs over the datasets' events concatenated in the CALLER's original order.  The call runs the
 * PRODUCTION kernels of this batch size (same schedule, same work cut as phylino_spectra) in a
 * diagnostic instantiation that also records, for every event a lane accumulates, the bin the hot
 * loop put it in; nothing else is written (the accumulators are cleared).
 *   params DEVICE [P x n_params]; bins DEVICE int32 [P x total_events]. */
PHYLINO_API phylino_status phylino_event_bins(phylino_ctx *ctx, int P, const double *params, int32_t *bins);

/* Same as phylino_nll / phylino_spectra but with HOST buffers: pinned staging, H2D of params (and
 * data), the kernels, D2H of the result, and a stream synchronise -- the end-to-end call a host
 * minimiser makes once per batch (parameters go to the GPU, the result comes back). */
PHYLINO_API phylino_status phylino_nll_host(phylino_ctx *ctx, int P, const double *params_host,
                                const double *data_host, double *nll_host);
PHYLINO_API phylino_status phylino_spectra_host(phylino_ctx *ctx, int P, const double *params_host, double *hist_host);

/* Pseudo-experiment ensembles ("test statistics derived from large ensembles of
 * pseudo-experiments"): nll[p * E + e] = the NLL of phylino_nll at point p against the observed counts
 * data[e * total_bins ...], for all P points and E experiments.  The spectra and expectations are computed once
 * per point; only the deviance sums are per experiment.  params DEVICE [P x n_params], data DEVICE
 * [E x total_bins], nll DEVICE [P x E] row-major.  Asynchronous on the context's stream like phylino_nll. */
PHYLINO_API phylino_status phylino_nll_ensemble(phylino_ctx *ctx, int P, const double *params, int E,
                                                const double *data, double *nll);

/* Poisson pseudo-data for an ensemble of pseudo-experiments, drawn on the device:
 * data[e * total_bins + i] ~ Poisson(mu[i]), e = 0 ... E-1.  mu DEVICE [total_bins] (e.g. one row of
 * phylino_expectation at the injected hypothesis), data DEVICE [E x total_bins]; feed it to phylino_nll_ensemble.
 * The counts are a function of (seed, e, i, mu[i]) alone (R26): Philox4x32-10 uniforms with counter
 * (i, e, 0, 0) and key = seed, and an exact inversion of the Poisson distribution from its mode outwards that uses
 * only +, *, / -- the same integers as any other IEEE implementation of that sequence, and from run to run.  mu[i] <= 0, NaN or inf gives 0;
 * a finite mu[i] above 1e9 is outside the sampler's domain and gives NaN (the walk costs O(sqrt(mu)) steps per draw and
 * every loop is bounded, so no value in `mu` can stall the device).  Asynchronous on the context's stream. */
PHYLINO_API phylino_status phylino_draw_pseudo_data(phylino_ctx *ctx, const double *mu, int E, uint64_t seed,
                                                    double *data);

/* Scan of one parameter under BOTH mass orderings in one call (Fig. 4: the likelihood as a
 * function of dm2_ee under the normal and the inverted ordering): for every grid value g the point theta with
 * theta[scan_param] = grid[g] is evaluated with ordering +1 and -1 (the model's own ordering flag is ignored).
 *   grid DEVICE [n_grid]; theta DEVICE [param_width] the point the other parameters are taken from;
 *   data DEVICE [total_bins]; nll DEVICE [2 x n_grid]: row 0 normal, row 1 inverted ordering.
 * Only the PHYLINO_OSC_FULL3 model depends on the ordering.  The minimisation over the other parameters that a
 * PROFILE needs stays with the caller's minimiser (out of scope); this is its inner batch.
 * Always dense.  Asynchronous. */
PHYLINO_API phylino_status phylino_ordering_scan(phylino_ctx *ctx, int n_grid, int scan_param, const double *grid,
                                                 const double *theta, const double *data, double *nll);

/* Central-difference gradient of the NLL from the 2 N + 1-point batch a minimiser evaluates per iteration
 * (R18), N = param_width: the batch {theta} U {theta +- step_j e_j} is formed on the
 * device, evaluated (with cross-point caching if phylino_set_caching is on), and
 *   grad[j] = (nll(theta + step_j e_j) - nll(theta - step_j e_j)) / ((theta_j + step_j) - (theta_j - step_j)).
 *   theta, step DEVICE [N] (step_j != 0); data DEVICE [total_bins]; nll0 DEVICE [1] receives nll(theta), may be
 *   NULL; grad DEVICE [N].  Asynchronous, also with caching on: which points of a central-difference batch share an
 *   energy scale or a mass splitting follows from which column each point perturbs, so the plan needs no values and
 *   nothing is copied back (a step below one ulp of theta_j only loses a merge, never a result).  Exception: caching
 *   together with a transformation layer goes through the host plan of phylino_set_caching (one copy back, one
 *   synchronisation). */
PHYLINO_API phylino_status phylino_nll_gradient(phylino_ctx *ctx, const double *theta, const double *step,
                                                const double *data, double *nll0, double *grad);

/* One variable-metric step of the minimiser's loop on the device ("This function is minimized by
 * iteratively modifying the model parameters until the estimated distance to the minimum is smaller than a predefined
 * threshold"; the minimiser is Minuit2's MIGRAD, a variable-metric method -- the paper prints no formula, R30
 * takes the published rule).  V DEVICE [N x N] row-major, in/out: the current estimate of the INVERSE Hessian of the NLL;
 * dx, dg DEVICE [N]: the last move x_new - x_old and the change of the gradient (both NULL: V is used as it is); grad
 * DEVICE [N] (e.g. from phylino_nll_gradient); direction DEVICE [N] out; edm DEVICE [2] out.
 *     vg = V dg, a = dx.dg, b = dg.vg;   V += dx dx^T / a - vg vg^T / b   (+ b u u^T, u = dx / a - vg / b, where a > b)
 *     -- only if a > 0 and b > 0, else V stays and edm[1] = 1 (edm[1] = 0 otherwise);
 *     direction = -V grad,   edm[0] = 1/2 grad^T V grad.
 * All sums in index order in plain double arithmetic.  The line search along `direction`, the convergence test on
 * edm[0] and the loop itself stay with the caller.  Needs no model; asynchronous on the
 * context's stream (the scratch grows once with N, as phylino.h "Async" says of the work buffers). */
PHYLINO_API phylino_status phylino_variable_metric_step(phylino_ctx *ctx, int N, double *V, const double *dx,
                                                        const double *dg, const double *grad, double *direction,
                                                        double *edm);

/* The same variable-metric step, for callers that cannot let this library allocate device memory.
 *
 * phylino_variable_metric_step above needs a context (phylino_create allocates) and keeps its 2 N + 2 doubles of
 * scratch in a cudaMalloc'ed buffer that grows with N.  That rules it out for a fit that shares its GPU with a
 * framework whose caching allocator already owns the memory (a cudaMalloc of ours can fail or fragment that pool, and
 * under an MPS / MIG memory limit it counts against the limit), for a minimiser loop that cannot afford the
 * device-wide synchronisation cudaMalloc / cudaFree imply, and for services that allow no allocation after start-up.
 * This entry point takes no context and calls no cudaMalloc, cudaFree or other allocating routine, ever: its scratch
 * is ONE fixed array inside the library's device image.
 *
 *   cuda_stream a cudaStream_t of the CURRENT device (0 = default stream); the work is enqueued there and the call
 *               returns without waiting.  Every DEVICE pointer must belong to the current device.
 *   N           0 ... PHYLINO_STATIC_MAX_N.  Anything larger is refused with PHYLINO_ERR_SHAPE before any launch
 *               (the array cannot grow) -- use phylino_variable_metric_step for such problems.
 *   V, dx, dg, grad, direction, edm   DEVICE, exactly as for phylino_variable_metric_step (same rule, same operation
 *               order, same kernels: the two entry points return identical bits).  The caller owns all of them.
 *   error       HOST [error_len] or NULL: receives the text of a failure ("" on success); there is no context to
 *               keep it in.
 *
 * What the fixed array costs and how it behaves:
 *   - (2 * PHYLINO_STATIC_MAX_N + 2) * 8 = 32 784 bytes of device memory on every GPU that loads this library, from
 *     the moment its device code is loaded there until the process exits, whether or not this call is ever made.
 *   - The FIRST call on each device looks up the array's device address (cudaGetSymbolAddress, with that device
 *     current) and remembers it per device; make that first call before any stream capture begins.
 *   - All calls on a device share the array, and it keeps whatever the last call wrote.  No call depends on that:
 *     each part of the array is written in full on the stream before the kernel that reads it, so nothing needs
 *     clearing.  But two calls that can run at the same time on one GPU -- different streams, or two host threads --
 *     race on it and corrupt each other's results; keep all calls of a device on one stream, or order them yourself.
 * Returns PHYLINO_ERR_ARG for NULL V / grad / direction / edm or for only one of dx, dg; PHYLINO_ERR_CUDA if the
 * address lookup or a launch fails (no device: there is no CPU fallback). */
#define PHYLINO_STATIC_MAX_N 2048
PHYLINO_API phylino_status phylino_variable_metric_step_static(void *cuda_stream, int N, double *V, const double *dx,
                                                               const double *dg, const double *grad,
                                                               double *direction, double *edm, char *error,
                                                               int error_len);

/* Where the energy-scale systematic acts.  mode 0 (default; what BASELINE.json's north_star
 * asks for, R8): on every event before binning, E' = a0 + a1 E_vis + a2 E_vis^2.  mode 1: on the BINNED
 * spectrum, the paper's own signal step 3 ("The expectation is smoothed using a second-degree polynomial function.
 * These corrected bins entries are then integrated over the original binning"; reading R27 of DESIGN.md:
 * inside a bin the density is the parabola whose integrals over three consecutive bins equal their contents; a bin of
 * the corrected spectrum is the integral of that density over the bin's pre-image under E'): the events are binned
 * under the identity scale, then per point and dataset  mu = eps norm C_a(f . H) + backgrounds, i.e. step 2 (the per-bin
 * re-scaling f) followed by step 3 (C_a).  phylino_spectra returns C_a(H).  With mode 1 no event work depends on the
 * energy-scale parameters, so cross-point caching merges all of them.  Needs total_bins <= 2000
 * (PHYLINO_ERR_SHAPE otherwise); PHYLINO_ERR_STATE before set_model, which resets the mode to 0. */
PHYLINO_API phylino_status phylino_set_energy_correction_mode(phylino_ctx *ctx, int mode);

/* Reactor-flux model of one dataset on a uniform fine grid (41 parameters on 0.25-MeV bins from 1 to
 * 11.25 MeV, "the basis of an area conserving spline, which is energy corrected and later transformed into the
 * original binning"; reading R28): theta[idx_par[j]] is the average flux correction on
 * [lo + j width, lo + (j+1) width); the flux scale f_db of analysis bin b becomes the average, over the bin's
 * pre-image under the dataset's energy scale, of the same area-conserving parabolic reconstruction as above (1 outside
 * the grid), replacing theta[idx_flux[b]].  idx_par HOST [n_par], copied; n_par = 0 removes the model; set_model
 * removes all.  Needs total_bins <= 2000.  Synchronises the stream. */
PHYLINO_API phylino_status phylino_set_flux_model(phylino_ctx *ctx, int dataset, int n_par, const int32_t *idx_par,
                                                  double lo, double width);

/* Correlated prior blocks: phylino_nll / phylino_nll_host add 1/2 (b - b0)^T V^-1 (b - b0) per block and
 * point (constants dropped, R9), on top of the uncorrelated priors of the model descriptor (a parameter of
 * a block normally has prior_sigma <= 0 there).  Call after phylino_set_model, which clears the blocks;
 * n_blocks = 0 clears them too.  Synchronises the stream.  PHYLINO_ERR_STATE before set_model,
 * PHYLINO_ERR_SHAPE for n or an index out of range, PHYLINO_ERR_ARG for NULL arrays or non-finite
 * mean / inv_cov entries. */
PHYLINO_API phylino_status phylino_set_prior_blocks(phylino_ctx *ctx, int n_blocks, const phylino_prior_block *blocks);

/* Constrained functions of the parameters (R29).  After this call a prior block may name function f
 * (0 ... n_functions-1) through the index n_params + f: 1/2 (b - b0)^T V^-1 (b - b0) then runs over b_i = theta[idx_i] or
 * b_i = function value; a Gaussian constraint on one function is a block of one with inv_cov = 1/sigma^2.  With a
 * transformation layer the functions are functions of theta = T(u).  Call after phylino_set_model (which clears them)
 * and BEFORE the blocks that use them; replacing the functions by fewer than the current blocks reference is
 * PHYLINO_ERR_STATE.  n_functions = 0 clears.  Synchronises the stream.  PHYLINO_ERR_SHAPE for an index or a power out
 * of range, PHYLINO_ERR_ARG for NULL arrays or non-finite coefficients. */
PHYLINO_API phylino_status phylino_set_functions(phylino_ctx *ctx, int n_functions, const phylino_function *functions);

/* Transformation layer.  After this call every `params` argument (DEVICE or HOST) is a batch of the minimiser's
 * vectors u, [P x n_u] row-major, and the library forms theta itself before anything else:
 *   theta_j = u[copy_src[j]]  (copy_const[j] where copy_src[j] < 0; copy_src HOST [n_params], copy_const HOST
 *   [n_params], may be NULL if no entry of copy_src is negative), then for every block, in order,
 *   theta[idx_out] = offset + matrix (u[idx_in] - centre); the sums run over j in index order with fma, on the
 *   device for the DEVICE entry points (one extra kernel), on the host for the HOST ones (identical bits).
 * Priors (diagonal and blocks) and every index of the model descriptor keep referring to theta.  n_u = 0 with
 * n_blocks = 0 removes the layer; phylino_set_model removes it too.  Synchronises the stream.
 * phylino_param_width: n_u if a layer is set, else n_params (0 before set_model). */
PHYLINO_API phylino_status phylino_set_transform(phylino_ctx *ctx, int n_u, const int32_t *copy_src,
                                                 const double *copy_const, int n_blocks,
                                                 const phylino_transform_block *blocks);
PHYLINO_API int64_t phylino_param_width(const phylino_ctx *ctx);

/* Sizes the caller needs for its buffers. */
PHYLINO_API int64_t phylino_total_bins(const phylino_ctx *ctx);     /* sum_d n_bins, 0 before set_model */
PHYLINO_API int64_t phylino_total_events(const phylino_ctx *ctx);   /* sum_d n over loaded datasets */

/* Pre-size every per-batch work buffer of the context for batches of up to max_points points (accumulators -- also
 * for the rows of a cached batch --, per-point records and bin thresholds, pinned staging of the HOST entry points,
 * the transformed batch, the plan of a cached batch, the work buffer of phylino_nll_gradient / _ordering_scan /
 * _draw_pseudo_data / _variable_metric_step, the expectations of phylino_nll_ensemble) and build what a first call would
 * otherwise build with a synchronisation (kernel occupancies, the unit order of the single-launch kernel, and -- if
 * phylino_set_caching is ON at the time of this call -- the structural plan of the central-difference batch).  After it,
 * calls with P <= max_points allocate nothing and the DEVICE entry points never synchronise (with caching on only
 * phylino_nll_gradient: see phylino_set_caching).  A batch counts with all its points: phylino_nll_gradient needs
 * max_points >= 2 W + 1, phylino_ordering_scan max_points >= n_grid (W = phylino_param_width), and
 * phylino_variable_metric_step N <= W.  Synchronises the stream if anything grows.  PHYLINO_ERR_STATE before the model
 * and all events are loaded. */
PHYLINO_API phylino_status phylino_reserve(phylino_ctx *ctx, int max_points);

/* Which kernels evaluate a batch: 0 (default) the library chooses -- the single-launch kernel for small batches
 * (at most 16 points with two oscillation terms, 4 with three: the minimiser's single evaluations; setup and event
 * walk in one kernel, the finalize kernel behind it as its programmatic dependent), else the setup / spectra /
 * finalize kernels with the work-item tickets; 1 always the three kernels; 2 the single-launch kernel for every
 * batch of at most 16 points.  Results agree
 * to rounding (another grouping of the fp64 partial sums); for tests and measurements. */
PHYLINO_API phylino_status phylino_set_schedule(phylino_ctx *ctx, int mode);

/* Tuning knobs (0 => library default).  unit_events: events per unit of the event store (a unit is staged in
 * shared memory: values above 256 -- 512 where every dataset has unit weights -- are clamped; the last stretch of
 * the store is always cut finer);
 * chunk_groups: groups of 32 parameter points per work item (a warp of the spectra kernel walks one
 * unit for every group of an item, then claims the next item); max_warps: cap on the warps of the
 * persistent grid.  Results are bit-identical from call to call for fixed knobs; other values
 * regroup the fp64 partial sums (rounding-level differences only). */
PHYLINO_API phylino_status phylino_set_tuning(phylino_ctx *ctx, int unit_events, int chunk_groups, int max_warps);

/* Cross-point caching for the HOST-buffer entry points (the paper's "caching, where
 * costly recalculations are only triggered upon relevant parameter changes").  For a fixed
 * energy scale and fixed mass splittings the spectrum is affine in the oscillation amplitudes (PAPER.md:34
 * Eq. 1): H[p,b] = P0(p) W[b] + sum_k A_k(p) C_k[b].  With caching on, phylino_nll_host / phylino_spectra_host
 * group the points of the batch by the BIT PATTERNS of the parameters that enter the energy scale and each
 * mass splitting, evaluate W and C_k once per group (packed as "virtual points" for the same kernels), and
 * combine them per point.  Points whose parameters differ only in amplitudes, flux/background nuisances or
 * rates share all of the event work: a 603-point central-difference batch of a 301-parameter fit needs 21
 * virtual points.  Results agree with the dense path to rounding (within the same per-bin and NLL tolerances) and
 * are bitwise reproducible; a cell that left the fixed-point domain reads NaN (the dense path tells +-inf
 * apart).  If the batch does not shrink to at most half, the dense path runs.  Off by default.  With caching
 * on, phylino_spectra and phylino_nll (DEVICE pointers) use it too, at the price of ONE device-to-host copy of the
 * batch and ONE stream synchronisation per call (the plan is made on the host) -- the "never synchronise" rule
 * above holds only with caching off; phylino_expectation, phylino_nll_ensemble and phylino_event_bins are always dense.  phylino_last_plan: virtual points and energy-scale classes
 * of the last host call that used the cache (0, 0 if it ran dense). */
PHYLINO_API phylino_status phylino_set_caching(phylino_ctx *ctx, int on);
PHYLINO_API phylino_status phylino_last_plan(const phylino_ctx *ctx, int64_t *virtual_points, int64_t *classes);

/* Device timing of the three kernels of a call (CUDA events on the context's stream, recorded
 * around the setup, spectra and finalize kernels of every later call).  phylino_last_kernel_ms
 * waits for the last call to finish and writes its three durations in milliseconds to ms[0..2]
 * (HOST pointer): per-point setup (records + bin thresholds), spectra, finalize. */
PHYLINO_API phylino_status phylino_set_timing(phylino_ctx *ctx, int on);
PHYLINO_API phylino_status phylino_last_kernel_ms(phylino_ctx *ctx, float *ms);

/* Which arithmetic the last spectra launch of this context ran (for the roofline accounting of bench.py): the
 * fraction, weighted by events x points, of (point group, dataset) pairs whose LAST oscillation term took the
 * small-phase form of 1/2 cos(2 phase) -- 6 fp64 instructions per event x point instead of 10 or 11 (7 in the
 * single-launch kernel for at most 16 points).  The kernels pick it
 * per group of 32 points and dataset where |1.267 dm2 (2/pi) L/E| <= 1/8 for every event and point (the solar term
 * at Double-Chooz baselines).  fraction HOST; synchronises the stream. */
PHYLINO_API phylino_status phylino_last_small_phase(phylino_ctx *ctx, double *fraction_host);
/* fraction_host (HOST, out): share of the event x point evaluations of the last spectra launch on this context whose
 * FIRST term took the no-reduction form (its phase stayed within half a half-turn for every event of a work item and
 * every point of the group: DESIGN.md section 6.1; bit-identical results, fewer instructions).  With cross-point
 * caching on the count is over virtual points.  Synchronises the stream. */
PHYLINO_API phylino_status phylino_last_medium_phase(phylino_ctx *ctx, double *fraction_host);

/* Kernel launches enqueued by this context so far (bench.py's `gpu_launches`). */
PHYLINO_API int64_t phylino_launch_count(const phylino_ctx *ctx);

/* Text of the last error of this context ("" if none).  Valid until the next call on ctx. */
PHYLINO_API const char *phylino_last_error(const phylino_ctx *ctx);

/* Microbenchmark of the pipe that bounds the batched path: issues
 * `iters` dependent-chain DFMA per thread over a full-chip grid on the context's stream and
 * returns the achieved fp64 FMA instructions per second (lane-operations/s) in *dfma_per_s. */
PHYLINO_API phylino_status phylino_peak_fp64(phylino_ctx *ctx, int iters, double *dfma_per_s_host);

/* Microbenchmark: device time in microseconds (HOST pointer; CUDA events, best of `reps`, L2 flushed before each) of
 * one kernel that does nothing but read `bytes` from HBM with coalesced loads.  The practical floor, launch ramp
 * included, under a call bound by its event bytes (one parameter point over a large event store): reported beside
 * bytes / peak bandwidth.  Allocates bytes + 256 MiB for the duration of the call; synchronises. */
PHYLINO_API phylino_status phylino_hbm_read_floor(phylino_ctx *ctx, int64_t bytes, int reps, double *us_host);

/* Microbenchmark: host wall time, in microseconds per repetition (HOST pointer), of launching an empty
 * kernel on the context's stream and synchronising it -- the floor under any call whose result the host
 * waits for.  Launch-latency-bound workloads (one parameter point over a small event store) are reported
 * against it. */
PHYLINO_API phylino_status phylino_launch_floor(phylino_ctx *ctx, int reps, double *us_per_call_host);

#ifdef __cplusplus
}
#endif
#endif /* PHYLINO_H */
