/*
 * internal.h -- host/device structures shared by the translation units of libphylino.so.
 * Not part of the ABI (include/phylino.h is); private to the CUDA path.
 */
#ifndef PHYLINO_INTERNAL_H
#define PHYLINO_INTERNAL_H

#include <cuda_runtime.h>
#include <stdint.h>

#include <string>
#include <utility>
#include <vector>

#include "phylino.h"

namespace phylino {

/* ---- layout of the event store and of a launch -------------------------------------------------
 * The events of a dataset, sorted by E_vis, are cut into batches of EB consecutive events, one record
 * each (48 bytes when every MC weight of the dataset is exactly 1, else 96); `unit_batches` consecutive
 * batches form a unit.  Large batches of points: a work item is one unit x `chunk_groups` groups of 32
 * parameter points; the warps of a persistent grid claim items from a global counter and walk the unit
 * once per group, ONE POINT PER LANE.  Small batches: every warp owns one contiguous range of batches and
 * setup, walk and likelihood run in ONE launch (spectra.cu). */
constexpr int EB          = 4;                      /* events per batch; every dataset is padded to a multiple */
#ifndef PHYLINO_WARPS
#define PHYLINO_WARPS 4
#endif
#ifndef PHYLINO_CTAS_PER_SM
#define PHYLINO_CTAS_PER_SM 4
#endif
constexpr int WARPS       = PHYLINO_WARPS;          /* warps per CTA of the spectra kernels */
constexpr int CTAS_PER_SM = PHYLINO_CTAS_PER_SM;    /* ... and CTAs per SM their register budget is set for */
constexpr int STAGE_BUF_BYTES = 6144;               /* one staging buffer of a warp: a unit is at most this long */
constexpr int HINT_BATCHES = 16;                    /* one bin hint per this many batches of a dataset */
constexpr int MAX_TERMS   = 3;
constexpr int SETUP_THREADS = 128;
constexpr int FIN_THREADS = 128;                    /* = WARPS * 32: the last CTA of the fused kernel runs the likelihood stage */
constexpr int FUSED_MAX_POINTS = 16;                /* largest batch the single-launch kernel takes */
constexpr int FIN_STAGE_MAX_BINS = 2000;            /* 3 doubles per bin of shared memory in the finalize kernel */

/* flag bits of a (point, bin) accumulator whose value left the fixed-point domain */
enum : unsigned { FLAG_NAN = 1u, FLAG_PINF = 2u, FLAG_NINF = 4u };

/* EB consecutive events of the E_vis-sorted store: everything the hot loop reads, behind one pointer.
 * Weighted datasets (some w != 1): */
struct __align__(16) EventBatchW {
    double x[EB];           /* L_core/E_nu  [m/MeV], fp64 (phase range reduction needs it) */
    double w[EB];           /* MC weight as fp64 (exact copy of the fp32 input); padding = 0 */
    float  v[EB];           /* E_vis [MeV]; padding = NaN */
    double wsum;            /* w[0] + ... + w[EB-1], summed in that order */
    int32_t reserved[2];
};
/* Unit-weight datasets (every BASELINE.json config): 12 bytes per event */
struct __align__(16) EventBatchU {
    double x[EB];
    float  v[EB];
};
static_assert(sizeof(EventBatchW) == 96 && sizeof(EventBatchU) == 48, "records are read with fixed 16-byte offsets");
template <bool UW> struct RecOf { typedef EventBatchW type; };
template <> struct RecOf<true> { typedef EventBatchU type; };

/* One entry per HINT_BATCHES batches of a dataset's store, read once per work item and lane. */
struct HintEntry {
    int32_t bin;            /* bin of the first event of batch HINT_BATCHES i under the identity energy scale (-1 below the
                               first edge, n_bins above the last / NaN): where a lane starts looking for its bin, never
                               trusted */
    float   x_env;          /* >= L/E_nu of every event of the batches HINT_BATCHES i, ... to the end of the dataset
                               (rounded up): decides per item whether the first term's phase can wrap at all */
};

/* Per-dataset entry of the table that travels by value in the kernel parameters. */
struct DatasetDev {
    const void *ev;         /* [n_batches] EventBatchU if unit_w else EventBatchW */
    const double *edges;    /* [n_bins+1] */
    const HintEntry *hint;  /* [ceil(n_batches / HINT_BATCHES)] */
    const int32_t *perm;    /* [n] caller's index of sorted event i (diagnostic instantiation only) */
    long long ev_off;       /* events of the datasets before this one (diagnostic instantiation only) */
    int32_t n_events;       /* events before padding */
    int32_t n_bins;
    int32_t bin_off;        /* offset of this dataset inside a point's total_bins */
    int32_t thr_off;        /* offset of this dataset inside a threshold row: sum of (n_bins+1) before it */
    int32_t per_point;      /* the energy scale of this dataset depends on theta */
    int32_t unit_w;         /* every event weight of the dataset is exactly 1 */
    int32_t n_batches;
    int32_t unit_begin;     /* first global unit of this dataset (units never straddle datasets) */
    int32_t idx_a[3];       /* energy-scale indices into theta, -1 => (0,1,0) */
    float   v_pos_min;      /* smallest positive finite E_vis of the dataset (+inf if none) */
    float   v_max;          /* largest finite E_vis (-inf if none) */
    double  fx_scale;       /* 2^e: fixed-point scale of the bin accumulators */
    double  x_max;          /* largest L/E_nu of the dataset (0 if empty) */
};

struct OscDev {
    int32_t osc_model, ordering;
    int32_t idx_osc[6];
    double  fixed_osc[6];
};

/* per-point record written by the setup kernel, structure-of-arrays: rec[field * P + p] */
constexpr int rec_fields(int S) { return 2 * S + 2; }       /* h_k, A_k, P0, bad */

struct SpectraArgs {
    DatasetDev ds[PHYLINO_MAX_DATASETS];
    OscDev  osc;
    int32_t n_datasets;
    int32_t n_params;
    int32_t P;              /* points in the batch */
    int32_t n_units;        /* units over all datasets */
    int32_t unit_batches;   /* U: batches per unit (the last unit of a dataset may be shorter) */
    int32_t chunk_groups;   /* G: point groups per work item */
    int32_t n_chunks;       /* ceil(n_groups / G) */
    int32_t n_items;        /* n_units x n_chunks; item = unit * n_chunks + chunk */
    /* fine tail: the last stretch of the last dataset is cut into shorter units, so that the warps of
     * the persistent grid run out of work within a fraction of a full item of each other */
    int32_t tail_unit;      /* first global unit of the fine tail (= n_units if there is none) */
    int32_t tail_b0;        /* its first batch inside the last dataset */
    int32_t tail_batches;   /* batches per unit of the fine tail */
    int32_t n_warps;        /* warps of the persistent grid (a multiple of WARPS) */
    int32_t sched;          /* 0: items claimed from the counter; 1: one contiguous range of batches per warp, single launch */
    unsigned *counter;      /* DEVICE work counter of the ticket kernel; the setup kernel zeroes it */
    unsigned *done;         /* DEVICE work counter of the single-launch kernel; the finalize kernel behind it zeroes it */
    const int32_t *unit_order;  /* DEVICE [n_units] single-launch kernel: item -> unit, the units nearest a bin edge
                                   first (api.cu build_unit_order); NULL: item = unit */
    unsigned long long *med_count;  /* DEVICE event x point evaluations whose first term took the no-reduction form
                                       (phylino_last_medium_phase); the setup kernel zeroes it */
    int32_t  *dbg_bins;     /* DEVICE [P x total_events] diagnostic instantiation: bin the hot loop gave every event */
    long long total_events;
    int32_t thr_stride;     /* floats per threshold row: total_bins + n_datasets */
    int32_t thr_rows;       /* P if some dataset's energy scale depends on theta, else 1 */
    int32_t total_bins;
    const double *params;   /* DEVICE [P x n_params]; NULL: the batch is in the ParamBlob argument (small-batch kernel) */
    double       *rec;      /* DEVICE [rec_fields x P] per-point records (setup kernel) */
    float        *thr;      /* DEVICE [thr_rows x thr_stride] fp32 bin thresholds (setup kernel) */
    float2       *safe;     /* DEVICE [thr_rows x n_datasets] fp32 interval on which a row holds */
    unsigned char *small;   /* DEVICE [n_groups x n_datasets] small-phase flag of the last term (setup kernel) */
    long long    *acc;      /* DEVICE [P x total_bins] fixed-point accumulators (zero on entry) */
    unsigned     *flags;    /* DEVICE [P x total_bins] FLAG_* (zero on entry) */
    /* component mode (cross-point caching; api.cu plan_components): the P
     * "points" of this launch are VIRTUAL points -- an energy-scale class (threshold row) plus S
     * half-turn coefficients, each taken from (real point, term) of the caller's batch -- and a run
     * is flushed as S + 1 separate sums (W, C_1..C_S) into acc[(p (S+1) + j) x total_bins + bin]. */
    int32_t comp;
    const int32_t *vp_class;    /* DEVICE [P] threshold row of a virtual point */
    const int32_t *vp_src;      /* DEVICE [P x S] source of slot s: real point * 4 + term */
    const int32_t *class_rep;   /* DEVICE [thr_rows] real point whose energy scale defines the row */
};

/* a small batch of parameter points travelling BY VALUE with the arguments of the small-batch kernel */
constexpr int PARAM_BLOB_DOUBLES = 448;
struct ParamBlob { double v[PARAM_BLOB_DOUBLES]; };

/* Model tables of the expectation / NLL stage, all DEVICE pointers. */
struct FinalizeArgs {
    int32_t P, n_params, total_bins, n_datasets, max_bkg;
    int32_t staged;               /* total_bins <= FIN_STAGE_MAX_BINS: per-bin model values staged in shared memory */
    unsigned *reset_counter;      /* DEVICE word zeroed at the end (the work counter of the single-launch kernel), or NULL */
    const double  *params;        /* [P x n_params] */
    long long     *acc;           /* [P x total_bins]; re-zeroed by the kernel */
    unsigned      *flags;         /* [P x total_bins]; re-zeroed by the kernel */
    const int32_t *bin_ds;        /* [total_bins] dataset of a global bin */
    const int32_t *idx_flux;      /* [total_bins] */
    const double  *inv_scale;     /* [n_datasets] 2^-e */
    const double  *norm;          /* [n_datasets] */
    const int32_t *idx_signorm;   /* [n_datasets] */
    const int32_t *n_bkg;         /* [n_datasets] */
    const int32_t *idx_rate;      /* [n_datasets x max_bkg] */
    const int32_t *idx_shape;     /* [max_bkg x total_bins] */
    const double  *tmpl;          /* [max_bkg x total_bins] */
    const double  *prior_mean;    /* [n_params] or NULL */
    const double  *prior_sigma;   /* [n_params] or NULL */
    /* correlated prior blocks (phylino_set_prior_blocks), flattened */
    int32_t        n_blocks;
    const int32_t *blk_off;       /* [n_blocks + 1] offsets into blk_idx / blk_mean */
    const int64_t *blk_moff;      /* [n_blocks] offsets into blk_inv */
    const int32_t *blk_idx;
    const double  *blk_mean;
    const double  *blk_inv;
    /* constrained functions of theta (phylino_set_functions, R29), flattened; a block index
     * >= n_params names function idx - n_params */
    int32_t        n_functions;
    const double  *fn_offset;     /* [n_functions] */
    const int32_t *fn_term_off;   /* [n_functions + 1] offsets into term_coef / term_fac_off */
    const double  *term_coef;     /* [terms] */
    const int32_t *term_fac_off;  /* [terms + 1] offsets into fac_idx / fac_pow */
    const int32_t *fac_idx;
    const int32_t *fac_pow;
    const double  *data;          /* [total_bins] (NLL mode) */
    double        *hist;          /* [P x total_bins] (spectra / expectation mode) */
    double        *nll;           /* [P] (NLL mode) */
    /* the paper's bin-level steps (PAPER.md:177 steps 2-3, :129; R27, R28) */
    int32_t        ec_mode;       /* 1: the energy correction acts on the binned spectrum (the events were binned under
                                     the identity scale); 0: it acted per event */
    int32_t        have_fm;       /* some dataset takes its flux scales from a fine-grid flux model */
    const double  *edges_all;     /* [total_bins + n_datasets] bin edges, dataset d at ds_bin_off[d] + d */
    const int32_t *ds_bin_off;    /* [n_datasets + 1] */
    const int32_t *ds_idx_a;      /* [n_datasets x 3] energy-scale indices into theta, -1 => (0,1,0) */
    const int32_t *fm_off;        /* [n_datasets + 1] offsets into fm_idx (equal => no flux model for the dataset) */
    const int32_t *fm_idx;        /* indices into theta of the fine-grid parameters */
    const double  *fm_grid;       /* [n_datasets x 2] lower end and bin width of the fine grid */
    /* component mode: H[p,b] = P0(p) W[b] + sum_k A_k(p) C_k[b] from the cells pt_comp names */
    int32_t comp, n_terms;
    OscDev  osc;
    const int32_t *pt_comp;       /* [P x (n_terms + 1)] accumulator rows: W, then the row of each term's C */
};

/* transformation layer (transform.cu), all DEVICE pointers except P-dependent u / theta set per call */
struct TransformArgs {
    int32_t P, n_params, n_u, n_blocks;
    const int32_t *copy_src;      /* [n_params] */
    const double  *copy_const;    /* [n_params] */
    const int32_t *row_off;       /* [n_blocks + 1] offsets into idx_out / offset */
    const int32_t *col_off;       /* [n_blocks + 1] offsets into idx_in / centre */
    const int64_t *mat_off;       /* [n_blocks] offsets into matrix */
    const int32_t *idx_out, *idx_in;
    const double  *offset, *centre, *matrix;
    const double  *u;             /* [P x n_u] */
    double        *theta;         /* [P x n_params] */
};

/* cross-point caching: the plan of a batch (api.cu plan_components) */
struct ComponentPlan {
    int V = 0, C = 0;               /* virtual points, energy-scale classes */
    std::vector<int32_t> vp_class, vp_src, class_rep, pt_comp;
};

/* kernel launchers (spectra.cu, finalize.cu, transform.cu, peaks.cu) */
cudaError_t launch_transform(const TransformArgs &a, cudaStream_t st);
cudaError_t launch_setup(const SpectraArgs &a, int S, cudaStream_t st);
size_t      fused_table_bytes(int S, int P, int thr_rows, int thr_stride, int n_datasets);
bool        fused_fits(size_t table_bytes);
cudaError_t allow_stage_all();      /* shared-memory opt-in of every spectra kernel on the current device (phylino_create) */
cudaError_t spectra_max_warps(int S, int sm_count, bool fused, size_t table_bytes, int *warps);
cudaError_t launch_spectra(const SpectraArgs &a, int S, cudaStream_t st, bool pdl, bool dbg);
cudaError_t launch_fused(const SpectraArgs &a, const ParamBlob &blob, int S, cudaStream_t st, bool pdl, bool dbg);
cudaError_t launch_finalize(const FinalizeArgs &a, int mode /*0 H, 1 mu, 2 nll, 3 clear*/, cudaStream_t st, bool pdl);
cudaError_t launch_ensemble(const FinalizeArgs &a, int E, int sm_count, cudaStream_t st);
cudaError_t launch_pseudo_data(const double *mu, double *Z, int n, int E, unsigned long long seed, double *data,
                               cudaStream_t st);
cudaError_t launch_scan_batch(const double *theta, int width, int col, const double *grid, int n_grid, double *batch,
                              cudaStream_t st);
cudaError_t launch_gradient_batch(const double *theta, const double *h, int width, double *batch, cudaStream_t st);
cudaError_t launch_gradient(const double *theta, const double *h, const double *nll, int width, double *nll0,
                            double *grad, cudaStream_t st);
cudaError_t launch_variable_metric_step(int N, double *V, const double *dx, const double *dg, const double *grad,
                                        double *direction, double *out, double *work, cudaStream_t st);
cudaError_t run_peak_fp64(int iters, cudaStream_t st, double *dfma_per_s);
cudaError_t run_launch_floor(int reps, cudaStream_t st, double *us_per_call);
cudaError_t run_hbm_read_floor(size_t bytes, int reps, cudaStream_t st, double *us_best);

} // namespace phylino

/* ---- host-side context ---------------------------------------------------------------------- */
struct phylino_dataset_host {
    /* model */
    int32_t n_bins = 0;
    int32_t idx_a[3] = {-1, -1, -1};
    int32_t idx_signorm = -1;
    double  norm = 1.0;
    std::vector<int32_t> idx_flux;                 /* empty => all -1 */
    struct Bkg { int32_t idx_rate; std::vector<double> tmpl; std::vector<int32_t> idx_shape; };
    std::vector<Bkg> bkg;
    /* events */
    bool     loaded = false;
    int64_t  n = 0, n_pad = 0;
    double   wsum_abs = 0.0;
    float    v_pos_min = 0.f, v_max = 0.f;
    bool     unit_w = false;
    int      fx_exp = 0;
    double   x_max = 0.0;
    void    *d_ev = nullptr;                        /* EventBatchU[] if unit_w else EventBatchW[] */
    phylino::HintEntry *d_hint = nullptr;
    std::vector<float>  v_blk;                     /* E_vis of the first event of every block of HINT_BATCHES batches */
    std::vector<double> edges;                     /* host copy of the bin edges */
    double  *d_edges = nullptr;
    int32_t *d_perm = nullptr;
};

struct phylino_ctx {
    int device = 0;
    int sm_count = 0;
    cudaStream_t stream = nullptr;
    std::string err;
    bool have_model = false;
    int32_t osc_model = 0, ordering = 1, n_params = 0, n_datasets = 0, n_terms = 2;
    int32_t idx_osc[6] = {-1, -1, -1, -1, -1, -1};
    double  fixed_osc[6] = {0, 0, 0, 0, 0, 0};
    bool    per_point_binning = false;
    int32_t total_bins = 0, max_bkg = 0, max_bins = 0;
    std::vector<phylino_dataset_host> ds;
    /* device model tables */
    void *d_tables = nullptr;                      /* one allocation, carved up below */
    phylino::FinalizeArgs fin{};                   /* table pointers filled by set_model */
    /* accumulators and per-call point tables */
    int64_t   acc_capacity = 0;                    /* in (point, bin) cells */
    long long *d_acc = nullptr;
    unsigned  *d_flags = nullptr;
    int64_t   point_capacity = 0;                  /* points the tables below hold */
    double   *d_rec = nullptr;                     /* [rec_fields x point_capacity] */
    float    *d_thr = nullptr;                     /* [thr_rows x (total_bins + n_datasets)] */
    float2   *d_safe = nullptr;                    /* [thr_rows x n_datasets] */
    unsigned char *d_small = nullptr;              /* [ceil(point_capacity / 32) x n_datasets] */
    /* cross-point caching of the host-buffer entry points (phylino_set_caching) */
    bool caching = false;
    int32_t *d_plan = nullptr;                     /* vp_class | vp_src | class_rep | pt_comp */
    int64_t plan_capacity = 0;                     /* int32 entries */
    int64_t last_virtual_points = 0, last_classes = 0;
    phylino::ComponentPlan grad_plan;              /* structural plan of the central-difference batch (phylino_nll_gradient) */
    int grad_plan_state = 0;                       /* 0: not made for this model yet, 1: made, -1: does not pay */
    int32_t max_block_idx = -1;                    /* largest index any prior block names (functions must cover it) */
    int32_t *d_grad_plan = nullptr;                /* ... on the device: vp_class | vp_src | class_rep | pt_comp */
    /* transformation layer (phylino_set_transform): host copy for the host entry points, device tables */
    bool have_tf = false;
    int32_t n_u = 0;
    std::vector<int32_t> tf_src, tf_row_off, tf_col_off, tf_idx_out, tf_idx_in;
    std::vector<int64_t> tf_mat_off;
    std::vector<double>  tf_const, tf_offset, tf_centre, tf_matrix;
    phylino::TransformArgs tf{};                   /* device table pointers */
    double *d_theta = nullptr;                     /* [theta_capacity] transformed batch of a device call */
    int64_t theta_capacity = 0;
    double *d_mu = nullptr;                        /* [mu_capacity] expectations of an ensemble call */
    int64_t mu_capacity = 0;
    double *d_work = nullptr;                      /* [work_capacity] batches / NLLs / Poisson norms of the consumers */
    int64_t work_capacity = 0;
    int ordering_override = 0;                     /* +-1 while an ordering scan runs, else 0 */
    int ec_mode = 0;                               /* phylino_set_energy_correction_mode */
    int last_points = 0;                           /* launch points of the last spectra launch (phylino_last_small_phase) */
    std::vector<std::vector<int32_t>> fm_idx;      /* per dataset: fine-grid flux parameters (phylino_set_flux_model) */
    std::vector<double> fm_lo, fm_width;
    /* host-buffer entry points: pinned + device staging */
    double *h_pin = nullptr, *d_stage = nullptr, *d_pin = nullptr;   /* d_pin: device alias of h_pin */
    int64_t stage_capacity = 0;                    /* doubles */
    unsigned *d_counter = nullptr;                 /* work counter of the spectra kernel */
    /* tuning knobs, 0 => default (phylino_set_tuning) */
    int unit_events = 0, chunk_groups = 0, max_warps = 0;
    int resident_warps = 0;                        /* warps of the ticket kernel the chip holds at once */
    int fused_warps = 0;                           /* ... of the single-launch kernel with fused_tables bytes of tables */
    size_t fused_tables = 0;
    std::vector<std::pair<size_t, int>> fused_cache;   /* (table bytes, warps) of every table size asked so far */
    int schedule = 0;                              /* phylino_set_schedule: 0 auto, 1 tickets, 2 single launch */
    unsigned *d_done = nullptr;                    /* work counter of the small-batch kernel */
    int32_t  *d_unit_order = nullptr;              /* its item -> unit table for units of order_U batches */
    int64_t   order_U = 0, order_units = 0;
    unsigned long long *d_med = nullptr;           /* medium-phase evaluations of the last ticket launch */
    bool last_fused = false;                       /* the last spectra launch was the single-launch kernel */
    phylino::ParamBlob blob{};                     /* a small host batch on its way into the kernel arguments */
    /* optional device timing of the three kernels of a call (phylino_set_timing) */
    bool timing = false;
    cudaEvent_t ev[4] = {nullptr, nullptr, nullptr, nullptr};
    int64_t launches = 0;
};

#endif
