/*
 * spectra.cu -- the batched oscillation-weight + histogram kernels (
 * PAPER.md:177 signal step 1, :183 "the most time-demanding computational step").
 *
 * Layout of the work: ONE PARAMETER POINT PER LANE.  The E_vis-sorted events of a dataset are cut
 * into batches of EB events (48-byte records when every MC weight is 1, else 96-byte ones) and the
 * batches into units.
 *
 * Large batches of points (spectra_kernel, "tickets").  A work item is one unit x a chunk of point
 * groups (32 points each).  The warps of a persistent grid claim items from a global counter (dynamic
 * balance: units that contain bin edges cost more; the last stretch of the store is cut into
 * quarter-size units so the warps run out of work together) and walk the unit once per group.
 *
 * Small batches (spectra_fused_kernel: at most FUSED_MAX_POINTS points -- the minimiser's single
 * evaluations).  ONE launch does rows a1-a5: every CTA derives the per-point records and the
 * bin thresholds it needs into its own shared memory, then the same ticket loop runs over units as long as a
 * staging buffer holds, the lanes of a warp split into 32 / PL sub-streams (PL = points rounded up to a power of
 * two) that are dealt the batches of a unit in turn.  No setup launch and no host copy of the parameters (a small
 * host batch rides with the kernel arguments); the finalize kernel behind it is a programmatic dependent that
 * does its table work while the events are walked.  The call is bound by the event bytes over HBM (12 B/event
 * for unit-weight datasets) and by latency -- launch, per-CTA setup, the instruction lines of everything that is
 * not the hot loop -- not by arithmetic.
 *
 * Staging.  Each warp owns two unit-sized buffers in shared memory and one mbarrier per buffer; lane 0
 * starts ONE bulk async copy (cp.async.bulk global -> shared, completion on the mbarrier) of the NEXT
 * unit while the current one is walked.  The hot loop reads warp-uniform LDS.128 broadcasts;
 * everything that depends on the point (half-turn coefficients h_k, the run accumulators, the current
 * bin, its fp32 upper threshold and the one after it) lives in the lane's registers.  No shuffles in
 * the loop, no block barriers.
 *
 * Oscillation weight (row a2).  P_ee = P0 + sum_k A_k g_k with g = 1/2 cos(2 phase) (devmath.cuh):
 * the lane accumulates C_k = sum_e w_e g_k(e) and W = sum_e w_e over a run of events that share a
 * bin; the run's total is P0 W + sum_k A_k C_k, formed once per run.  Per event x point and term that is
 * 11 fp64 instructions and one integer instruction in the general form; unit-weight datasets take cheaper
 * forms where they are exact: the run sum formed by the last Horner step itself (10 + 2 integer; two-term
 * model), no range reduction where the first term's phase cannot wrap within a work item (8), a cubic for a
 * last term that stays below an eighth of a half-turn over a dataset (6): see folded() below.
 *
 * Binning (row a3).  For one point the map v -> E' = fma(fma(a2,v,a1),v,a0) is non-decreasing over
 * the fp32 values of a dataset (checked per point), so bin(E'(v)) >= b <=> v >= T[b] with T[b] the
 * smallest fp32 value whose E' reaches edges[b].  T is found with the SAME fp64 fma sequence and the
 * SAME fp64 edges, hence the fp32 comparison decides exactly what the fp64 comparison E' >= edges[b]
 * decides: bit-exact bins.  Events are sorted, so 4, 2 or 1 batches lie inside the lane's current bin
 * iff the LAST event of the last one is below the bin's upper threshold: one fp32 compare, then a
 * straight-line stretch of rows a2 + a4 (unit-weight datasets carry no weights at all).  A lane opens its
 * run at its first event from a load-time hint (one per HINT_BATCHES batches).  Events outside the
 * interval on which a table is proven (and points that fail the monotonicity check) take the per-event
 * fp64 map.
 *
 * Histogram (rows a4, a5).  When a run ends (bin edge, end of the unit or range) its fp64 total is
 * converted once to 64-bit fixed point and added to the (point, bin) accumulator with an integer RED.
 * Integer addition is associative: the result depends neither on which warp walks an item nor on
 * the order of arrival, i.e. bitwise reproducible with no float atomics anywhere (the cut of the
 * events into items is a function of the sizes only).
 *
 * Component mode (cross-point caching): the launch's points are virtual points (an energy-scale class
 * plus S splittings) and a run is flushed as S + 1 separate sums; finalize.cu combines them per point.
 *
 * Diagnostic instantiation (template flag DBG, phylino_event_bins): the SAME kernels additionally write,
 * for every event a lane accumulates, the bin it put it in -- through the hint walk, the forward scan, the
 * whole-batch test, the 2-/4-batch paths and the sub-stream split -- for the bit-exact bin parity test.
 *
 * Launch.  The ticket kernel is a programmatic dependent of the setup kernel: barriers and the first
 * event copy are set up while the setup kernel runs; griddepcontrol.wait precedes the first read of a
 * record, a threshold or the work counter.
 */
#include "devmath.cuh"

namespace phylino {

namespace {

__device__ __forceinline__ float pos_inf() { return __int_as_float(0x7f800000); }

/* -DPHYLINO_TRACE (never in the shipped build): phase timestamps of the single-launch kernel for timeline work */
#ifdef PHYLINO_TRACE
__device__ unsigned long long g_trace[8];
__device__ unsigned long long g_wtrace[4][256];     /* per-unit timestamps of four sample warps */
__device__ int g_wn[4];
__device__ long long g_sub[64][4];                 /* walk_unit sub-phases of the first 64 lanes-0 */
__device__ unsigned long long g_wend[4096];
__device__ int g_wunits[4096];
__device__ __forceinline__ unsigned long long gtime()
{
    unsigned long long t;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
    return t;
}
#define TRACE_MIN(i) do { if (threadIdx.x == 0) atomicMin(&g_trace[i], gtime()); } while (0)
#define TRACE_MAX(i) do { if (threadIdx.x == 0) atomicMax(&g_trace[i], gtime()); } while (0)
#else
#define TRACE_MIN(i) do { } while (0)
#define TRACE_MAX(i) do { } while (0)
#endif

/* ---- per-warp staging of a unit in shared memory: one bulk async copy (TMA engine, no tensor map),
 * completion signalled on an mbarrier that the 32 lanes poll.  (PTX ISA cp.async.bulk / mbarrier.) */
__device__ __forceinline__ unsigned smem_u32(const void *p) { return (unsigned)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(unsigned long long *bar, unsigned count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}

/* lane 0 of the warp: expect `bytes` on `bar` and start the copy global -> shared */
__device__ __forceinline__ void bulk_load(void *dst, const void *src, unsigned bytes, unsigned long long *bar)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(smem_u32(dst)), "l"(src), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}

__device__ __forceinline__ void mbar_wait(unsigned long long *bar, unsigned parity)
{
    unsigned done;
    do {
        asm volatile("{\n\t.reg .pred p;\n\t"
                     "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
                     "selp.u32 %0, 1, 0, p;\n\t}"
                     : "=r"(done) : "r"(smem_u32(bar)), "r"(parity) : "memory");
    } while (!done);
}

__device__ __forceinline__ unsigned rec_bytes(const DatasetDev &ds)
{
    return ds.unit_w ? (unsigned)sizeof(EventBatchU) : (unsigned)sizeof(EventBatchW);
}

/* address of batch b of the dataset's store */
__device__ __forceinline__ const void *batch_ptr(const DatasetDev &ds, int b)
{
    return static_cast<const char *>(ds.ev) + (size_t)b * rec_bytes(ds);
}

/* run total -> fixed point; values outside the domain become flag bits */
__device__ __forceinline__ long long to_fixed(double s, double scale, bool bad, unsigned &fl)
{
    double y = s * scale;                                   /* scale = 2^e: exact */
    if (bad || !(fabs(y) < 4.0e18)) {
        fl = (bad || s != s) ? FLAG_NAN : (s > 0.0 ? FLAG_PINF : FLAG_NINF);
        return 0;
    }
    fl = 0;
    return __double2ll_rn(y);
}

/* smallest fp32 v in [safe_lo, safe_hi] (positive, normal) with E'(v) >= edge, +inf if none.  E' is
 * non-decreasing over the fp32 values of the interval (the caller checked), so the answer is unique and any
 * bracketing search finds it: a Newton guess of the root in fp64, a galloping bracket around it, bisection
 * inside (a handful of evaluations instead of the ~30 of a bisection over the whole interval). */
__device__ float threshold_search(double a0, double a1, double a2, double edge, float safe_lo, float safe_hi)
{
    if (!(safe_lo <= safe_hi)) return pos_inf();
    if (!(escale(a0, a1, a2, (double)safe_hi) >= edge)) return pos_inf();
    if (escale(a0, a1, a2, (double)safe_lo) >= edge) return safe_lo;
    int lo = __float_as_int(safe_lo), hi = __float_as_int(safe_hi);   /* E'(lo) < edge <= E'(hi) */
    double g = (edge - a0) / a1;
#pragma unroll
    for (int it = 0; it < 2; ++it) g -= (escale(a0, a1, a2, g) - edge) / fma(2.0 * a2, g, a1);
    if (g > (double)safe_lo && g < (double)safe_hi) {
        const int gi = min(max(__float_as_int(__double2float_rn(g)), lo + 1), hi);
        int step = 1;
        if (escale(a0, a1, a2, (double)__int_as_float(gi)) >= edge) {
            hi = gi;
            for (;;) {
                const int c = hi - step;
                if (c <= lo) break;
                if (escale(a0, a1, a2, (double)__int_as_float(c)) >= edge) { hi = c; step <<= 1; } else { lo = c; break; }
            }
        } else {
            lo = gi;
            for (;;) {
                const int c = lo + step;
                if (c >= hi) break;
                if (escale(a0, a1, a2, (double)__int_as_float(c)) >= edge) { hi = c; break; } else { lo = c; step <<= 1; }
            }
        }
    }
    while (hi - lo > 1) {
        int mid = lo + ((hi - lo) >> 1);
        if (escale(a0, a1, a2, (double)__int_as_float(mid)) >= edge) hi = mid; else lo = mid;
    }
    return __int_as_float(hi);
}

__device__ __forceinline__ void energy_scale_of(const DatasetDev &ds, const double *theta, double &a0, double &a1,
                                                double &a2)
{
    a0 = ds.idx_a[0] >= 0 ? theta[ds.idx_a[0]] : 0.0;
    a1 = ds.idx_a[1] >= 0 ? theta[ds.idx_a[1]] : 1.0;
    a2 = ds.idx_a[2] >= 0 ? theta[ds.idx_a[2]] : 0.0;
}

/* threshold row of launch point p, and the parameter vector its energy scale comes from */
__device__ __forceinline__ int row_of(const SpectraArgs &a, int p)
{
    return a.comp ? a.vp_class[p] : (a.thr_rows > 1 ? p : 0);
}

__device__ __forceinline__ const double *theta_of(const SpectraArgs &a, const double *params, int p)
{
    return params + (size_t)(a.comp ? a.class_rep[a.vp_class[p]] : p) * a.n_params;
}

/* The per-call tables the walk reads: in global memory behind the setup kernel (tickets), in the CTA's own
 * shared memory in the single-launch kernel. */
struct Tables {
    const double *params;   /* [P x n_params]: a.params, or the copy that came with the kernel arguments */
    const double *rec;      /* [rec_fields x P]: h_k, A_k, P0, bad */
    const float  *thr;      /* [thr_rows x thr_stride] */
    const float2 *safe;     /* [thr_rows x n_datasets] */
    const unsigned char *small;     /* [n_groups x n_datasets] the last term takes half_cos_small for this group and dataset */
};

/* row a1: record of launch point p -> rec[field * P + p] */
/* returns the half-turn coefficient of the point's last term */
template <int S>
__device__ __forceinline__ double point_record(const SpectraArgs &a, const double *params, int p, double *rec)
{
    if (a.comp) {
        /* virtual point: slot s computes the half-turn coefficient of (real point, term) vp_src */
#pragma unroll
        for (int k = 0; k < S; ++k) {
            const int src = a.vp_src[(size_t)p * S + k];
            double A[MAX_TERMS], dm2[MAX_TERMS];
            osc_terms(a.osc, params + (size_t)(src >> 2) * a.n_params, A, dm2);
            rec[(size_t)k * a.P + p] = halfturn_coeff(dm2[src & 3]);
        }
        return rec[(size_t)(S - 1) * a.P + p];
    }
    const double *theta = params + (size_t)p * a.n_params;
    double A[MAX_TERMS], dm2[MAX_TERMS];
    osc_terms(a.osc, theta, A, dm2);
    double asum = 0.0, half = 0.0;
#pragma unroll
    for (int k = 0; k < S; ++k) {
        rec[(size_t)k * a.P + p] = halfturn_coeff(dm2[k]);
        rec[(size_t)(S + k) * a.P + p] = A[k];
        asum += fabs(A[k]);
        half += A[k];
    }
    rec[(size_t)(2 * S) * a.P + p] = 1.0 - 0.5 * half;            /* P0 */
    /* |P0| + 1/2 sum|A_k| <= 1 + sum|A_k| <= 4 keeps every run total inside the fixed-point range
     * (phylino.h "Errors": a point beyond this bound reads NaN) */
    rec[(size_t)(2 * S + 1) * a.P + p] = (asum <= 3.0) ? 0.0 : 1.0;
    return rec[(size_t)(S - 1) * a.P + p];
}

/* One warp, its lane's last coefficient (0 for a lane without a point): small[d] = the phase of the last term stays
 * within SMALL_PHASE over dataset d for all 32 lanes.  A NaN coefficient compares false and lands on the cheap form,
 * where it is as much a NaN as on the other. */
__device__ __forceinline__ void group_flags(const SpectraArgs &a, double h_last, unsigned char *small)
{
    for (int d = 0; d < a.n_datasets; ++d) {
        const bool big = __any_sync(0xffffffffu, fabs(h_last) * a.ds[d].x_max > SMALL_PHASE);
        if ((threadIdx.x & 31) == 0) small[d] = big ? 0 : 1;
    }
}

/* tables of row a3: entry e of threshold row `row` (and the row's validity interval per dataset) */
__device__ __forceinline__ void threshold_entry(const SpectraArgs &a, const double *params, int row, int e, float *thr,
                                                float2 *safe)
{
    /* only read where idx_a >= 0 */
    const double *theta = params + (size_t)(a.comp ? a.class_rep[row] : row) * a.n_params;
    int d = 0;
    for (int i = 1; i < a.n_datasets; ++i)
        if (e >= a.ds[i].thr_off) d = i;
    const DatasetDev &ds = a.ds[d];
    const int b = e - ds.thr_off;
    const double edge = ds.edges[b];
    float slo, shi, t;
    if (!ds.per_point) {
        slo = -pos_inf(); shi = pos_inf();      /* E' = v exactly: the table holds for every float */
        t = __double2float_ru(edge);            /* v >= edge <=> v >= ru(edge) */
    } else {
        /* E'(v) computed with the two fma is non-decreasing over the fp32 values of
         * [v_pos_min, v_max] if the Horner inner value t = a2 v + a1 is positive and the
         * derivative a1 + 2 a2 v exceeds 2^-20 t at both ends (both are linear in v): between
         * fp32 neighbours the exact increase then outweighs the rounding of t 2^8-fold
         * (DESIGN.md "Bit-exact binning with fp32 thresholds"). */
        double a0, a1, a2;
        energy_scale_of(ds, theta, a0, a1, a2);
        double vl = (double)ds.v_pos_min, vh = (double)ds.v_max;
        double t_lo = fma(a2, vl, a1), t_hi = fma(a2, vh, a1);
        double g_lo = fma(2.0 * a2, vl, a1), g_hi = fma(2.0 * a2, vh, a1);
        double tm = fmax(t_lo, t_hi) * 0x1p-20;
        bool ok = t_lo > 0.0 && t_hi > 0.0 && g_lo >= tm && g_hi >= tm && fabs(a0) < 1.0e300 &&
                  t_hi < 1.0e300 && ds.v_pos_min >= 1.17549435e-38f && ds.v_pos_min <= ds.v_max;
        slo = ok ? ds.v_pos_min : pos_inf();
        shi = ok ? ds.v_max : -pos_inf();
        t = threshold_search(a0, a1, a2, edge, slo, shi);
    }
    thr[(size_t)row * a.thr_stride + e] = t;
    if (b == 0) safe[(size_t)row * a.n_datasets + d] = make_float2(slo, shi);
}

/* threshold row entry with the conventions thr[-1] = -inf, thr[B + 1] = +inf */
__device__ __forceinline__ float thr_at(const float *thr, int B, int i)
{
    PHYLINO_ASSERT(i >= -2 && i <= B + 3);
    return i < 0 ? -pos_inf() : (i > B ? pos_inf() : thr[i]);
}

/* Bin of one event of dataset ds at one point, and the fp32 bound `hi` below which later (larger)
 * events are known to stay in that bin (-inf: not known, ask again).
 *   table : thr[b] <= v decides E'(v) >= edges[b] for v in [safe.x, safe.y]; the result is the number
 *           of thresholds <= v, minus one: -1 below the first edge, n_bins at or above the last;
 *   else  : the fp64 map and the fp64 edges (R7, R8); -1 outside the histogram or NaN. */
__device__ __forceinline__ int locate_bin(const DatasetDev &ds, const float *thr, float2 safe, const double *theta,
                                          float v, float &hi)
{
    const int B = ds.n_bins;
    if (v >= safe.x && v <= safe.y) {
        int lo = -1, up = B + 1;                    /* thr[lo] <= v < thr[up], thr[-1] = -inf, thr[B+1] = +inf */
        while (up - lo > 1) {
            int mid = (lo + up) >> 1;
            if (thr[mid] <= v) lo = mid; else up = mid;
        }
        hi = lo < B ? thr[lo + 1] : pos_inf();
        return lo;
    }
    double a0, a1, a2;
    energy_scale_of(ds, theta, a0, a1, a2);
    hi = -pos_inf();
    return bin_search(ds.edges, B, escale(a0, a1, a2, (double)v));
}

/* ---- setup kernel (tickets): per-point records and threshold rows (row a1 and the tables of row a3) ----
 * blocks [0, rec_blocks): one thread per point writes its record;
 * blocks [rec_blocks, rec_blocks + thr_rows): one CTA per threshold row. */
template <int S>
__global__ void __launch_bounds__(SETUP_THREADS) setup_kernel(const __grid_constant__ SpectraArgs a, int rec_blocks)
{
    /* programmatic dependent launch: the spectra kernel may start its prologue (barriers, first copy of
     * event data) now; it waits for this grid to finish before it reads anything written here */
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    if ((int)blockIdx.x < rec_blocks) {
        const int p = blockIdx.x * SETUP_THREADS + threadIdx.x;
        if (p == 0) {
            *a.counter = 0u;                                    /* the work counter of ticket_loop */
            *a.med_count = 0ull;                                /* phylino_last_medium_phase */
        }
        const double h_last = p < a.P ? point_record<S>(a, a.params, p, a.rec) : 0.0;
        group_flags(a, h_last, a.small + (size_t)(p >> 5) * a.n_datasets);      /* SETUP_THREADS is a multiple of 32 */
        return;
    }
    const int row = blockIdx.x - rec_blocks;
    for (int e = threadIdx.x; e < a.thr_stride; e += SETUP_THREADS) threshold_entry(a, a.params, row, e, a.thr, a.safe);
}

/* ---- the hot loop ------------------------------------------------------------------------------ */

/* the lane's open run: events of ONE bin seen since the last flush */
template <int S> struct Run {
    double C[S];    /* sum of w g_k over the run; a FOLDED term (see folded()) holds only its oscillating part C'
                     * (devmath.cuh, half_cos_accumulate), the rest is 1/2 W - odd[k] */
    int    odd[S];  /* folded GENERAL terms (two-term model only): events of the run whose half-turn count n_k is odd;
                     * the small-phase and the no-reduction form have n = 0, so three-term models never touch it */
    bool   sm;      /* the run's last term takes the small-phase form (fixed per group and dataset) */
    bool   med;     /* the run's first term takes the no-reduction form (fixed per work item and group) */
    bool   fo;      /* the kernel folds at all (the large-batch kernel does, the single-launch one does not) */
    double W;       /* sum of w over the run */
    int    cur;     /* its bin; < 0 or >= n_bins: events that land in no bin (never flushed) */
    float  hi;      /* later events below hi stay in the run (-inf: re-locate at the next event) */
    float  hi2;     /* threshold after hi (+inf past the last edge), loaded when the run opened so that the
                     * end of the run does not wait for it; meaningful only while hi is a table threshold */
};

template <int S> __device__ __forceinline__ void run_reset(Run<S> &r)
{
#pragma unroll
    for (int k = 0; k < S; ++k) { r.C[k] = 0.0; r.odd[k] = 0; }
    r.W = 0.0;
    r.cur = -1;
    r.hi = -pos_inf();
    r.hi2 = pos_inf();
    r.sm = false;
    r.med = false;
    r.fo = false;
}

/* Which terms of a UNIT-WEIGHT run are accumulated in the folded form (devmath.cuh, half_cos_accumulate): the
 * small-phase last term always (no sign, so the fold costs nothing: 6 fp64 instructions instead of 7); the general
 * terms of the two-term model (10 + 2 integer instead of 11 + 1: config 3 +4 %).  Not the general terms of the
 * three-term models: measured in round 2, config 4 lost 5.6 % (128 registers, fp64 pipe 91.7 -> 78.8 % busy, top stall
 * "wait": the two extra integer instructions per term sit in the dependency chains of three terms at once).
 * Not in the single-launch kernel for at most 16 points either (fo = false): that call is bound by latency and by the
 * instruction lines it has to fetch, not by the fp64 pipe, and was 3 us slower per call with the folded flush. */
template <int S> __device__ __forceinline__ bool folded(bool fo, bool sm, bool med, int k)
{
    return fo && (S == 2 || (sm && k == S - 1) || (med && k == 0));     /* the no-reduction form has no sign either */
}

/* sum of w g_k over the run, whichever way it was accumulated */
template <int S>
__device__ __forceinline__ double run_sum(const DatasetDev &ds, const Run<S> &r, int k)
{
    return (ds.unit_w && folded<S>(r.fo, r.sm, r.med, k)) ? r.C[k] + (0.5 * r.W - (S == 2 ? (double)r.odd[k] : 0.0)) : r.C[k];
}

/* diagnostic instantiation: the bin the hot loop gave event j of dataset batch gb at point p */
template <bool DBG>
__device__ __forceinline__ void dbg_mark(const SpectraArgs &a, const DatasetDev &ds, int p, bool active, int gb, int j,
                                         int cur)
{
    if (!DBG) return;
    const long long i = (long long)gb * EB + j;
    if (!active || i >= ds.n_events) return;
    PHYLINO_ASSERT(ds.perm[i] >= 0 && ds.perm[i] < ds.n_events && ds.ev_off + ds.perm[i] < a.total_events);
    a.dbg_bins[(size_t)p * a.total_events + ds.ev_off + ds.perm[i]] = (cur >= 0 && cur < ds.n_bins) ? cur : -1;
}

template <int S>
__device__ __forceinline__ void flush_run(const SpectraArgs &a, const Tables &T, const DatasetDev &ds, int p,
                                          bool active, Run<S> &r)
{
    if (a.comp && active && r.cur >= 0 && r.cur < ds.n_bins) {
        /* component mode: W and every C_k go to cells of their own (the amplitudes come later) */
        const size_t cell = (size_t)p * (S + 1) * a.total_bins + ds.bin_off + r.cur;
        PHYLINO_ASSERT(cell + (size_t)S * a.total_bins < (size_t)a.P * (S + 1) * a.total_bins);
#pragma unroll
        for (int j = 0; j <= S; ++j) {
            unsigned fl;
            const long long q = to_fixed(j == 0 ? r.W : run_sum<S>(ds, r, j - 1), ds.fx_scale, false, fl);
            if (q) atomicAdd((unsigned long long *)a.acc + cell + (size_t)j * a.total_bins, (unsigned long long)q);
            if (fl) atomicOr(a.flags + cell + (size_t)j * a.total_bins, fl);
        }
    } else if (active && r.cur >= 0 && r.cur < ds.n_bins) {
        double tot = T.rec[(size_t)(2 * S) * a.P + p] * r.W;                 /* P0 W */
#pragma unroll
        for (int k = 0; k < S; ++k) tot = fma(T.rec[(size_t)(S + k) * a.P + p], run_sum<S>(ds, r, k), tot);
        const bool bad = T.rec[(size_t)(2 * S + 1) * a.P + p] != 0.0;
        unsigned fl;
        const long long q = to_fixed(tot, ds.fx_scale, bad, fl);
        const size_t cell = (size_t)p * a.total_bins + ds.bin_off + r.cur;
        PHYLINO_ASSERT(cell < (size_t)a.P * a.total_bins);
        if (q) atomicAdd((unsigned long long *)a.acc + cell, (unsigned long long)q);
        if (fl) atomicOr(a.flags + cell, fl);
    }
#pragma unroll
    for (int k = 0; k < S; ++k) { r.C[k] = 0.0; r.odd[k] = 0; }
    r.W = 0.0;
}

/* The flush at the end of a unit / range when the group has at most 16 points: the 32 / PL sub-streams of a
 * point usually end in the same bin, and 32 lanes of every resident warp adding to the same one or two cells
 * would queue at the L2 atomic unit (same-address atomics: a 6e6-event, 1-point call spent 0.45 ms there).
 * Every lane converts its run to fixed point as usual; the integers of the lanes that share a cell are
 * summed over the sub-streams with shuffles (exact, so the bits are those of the separate REDs) and the
 * first lane of each cell issues one RED.  All 32 lanes call this together. */
template <int S>
__device__ __forceinline__ void flush_run_substreams(const SpectraArgs &a, const Tables &T, const DatasetDev &ds, int p,
                                                     bool active, int lg, int lane, Run<S> &r)
{
    const bool live = active && r.cur >= 0 && r.cur < ds.n_bins;
    const bool comp = a.comp != 0;                              /* warp-uniform */
    const int pl = lane & ((1 << lg) - 1);
    /* the usual case: the sub-streams of every point end in the same bin (the cell is a function of point and bin) */
    const int my_bin = live ? r.cur : -1;
    const bool uniform = __all_sync(0xffffffffu, my_bin == __shfl_sync(0xffffffffu, my_bin, pl));
    long long q[S + 1];
    unsigned fl[S + 1];
#pragma unroll
    for (int j = 0; j <= S; ++j) { q[j] = 0; fl[j] = 0; }
    unsigned long long cell = ~0ull;
    if (live) {
        if (comp) {
            cell = (unsigned long long)p * (S + 1) * a.total_bins + ds.bin_off + r.cur;
#pragma unroll
            for (int j = 0; j <= S; ++j) q[j] = to_fixed(j == 0 ? r.W : run_sum<S>(ds, r, j - 1), ds.fx_scale, false, fl[j]);
        } else {
            double tot = T.rec[(size_t)(2 * S) * a.P + p] * r.W;
#pragma unroll
            for (int k = 0; k < S; ++k) tot = fma(T.rec[(size_t)(S + k) * a.P + p], run_sum<S>(ds, r, k), tot);
            cell = (unsigned long long)p * a.total_bins + ds.bin_off + r.cur;
            q[0] = to_fixed(tot, ds.fx_scale, T.rec[(size_t)(2 * S + 1) * a.P + p] != 0.0, fl[0]);
        }
    }
    bool first = true;
    if (uniform) {
        /* a butterfly over the sub-stream bits of the lane index (exact integers: any order gives the same bits) */
        for (int o = 16; o >= (1 << lg); o >>= 1) {
            q[0] += __shfl_xor_sync(0xffffffffu, q[0], o);
            if (comp) {
#pragma unroll
                for (int j = 1; j <= S; ++j) q[j] += __shfl_xor_sync(0xffffffffu, q[j], o);
            }
        }
        first = lane == pl;
    }
    /* else: a bin edge inside the unit -- the sub-streams of a point end in different cells.  Rare (one unit per
     * edge and point), so every lane simply adds its own total: the same integers in another order, and nothing
     * cold to fetch on the way (the shuffle loop that used to sort the lanes by cell was a second cold function
     * behind the event-by-event path: a warp with an edge ended 5 us after the others in a one-point call) */
    if (live) {
#pragma unroll
        for (int j = 0; j <= S; ++j) {
            if (j == 0 || comp) {
                if (first && q[j]) atomicAdd((unsigned long long *)a.acc + cell + (size_t)j * a.total_bins, (unsigned long long)q[j]);
                if (fl[j]) atomicOr(a.flags + cell + (size_t)j * a.total_bins, fl[j]);
            }
        }
    }
#pragma unroll
    for (int k = 0; k < S; ++k) { r.C[k] = 0.0; r.odd[k] = 0; }
    r.W = 0.0;
}

/* Open the lane's run at its first event v0 (dataset batch gb): start from the load-time hint (the bin, under
 * the identity energy scale, of an event at most HINT_BATCHES batches earlier; loaded by the caller one item
 * ahead, off the critical path) and step to the bin the lane's
 * own thresholds give -- the same decision as the binary search of locate_bin, usually with two independent
 * loads and no dependent one; a lane whose bin lies far from the hint falls back to the search. */
template <int S>
__device__ __forceinline__ void open_run(const DatasetDev &ds, const float *thr, float2 safe, float v0, int hint,
                                         Run<S> &r)
{
    if (!(v0 >= safe.x && v0 <= safe.y)) return;        /* the first walk_batch locates it in fp64 */
    const int B = ds.n_bins;
    int b = max(-1, min(hint, B));
    float lo = thr_at(thr, B, b), hi = thr_at(thr, B, b + 1);
    int steps = 0;
    while (b >= 0 && v0 < lo && steps < 8) { --b; hi = lo; lo = thr_at(thr, B, b); ++steps; }
    while (b < B && !(v0 < hi) && steps < 8) { ++b; hi = thr_at(thr, B, b + 1); ++steps; }
    if (steps >= 8) b = locate_bin(ds, thr, safe, nullptr, v0, hi);     /* inside the table's interval: theta unused */
    r.cur = b;
    r.hi = hi;
    r.hi2 = thr_at(thr, B, b + 2);
}

/* K batches of the lane's stream (bp, bp + st, ...; dataset batches gb, gb + st, ...) known to lie inside the lane's
 * open run (the store is sorted: the last event of the last batch is below r.hi): rows a2 + a4 only, straight-line. */
template <int S, bool UW, int K, bool DBG, bool SM, bool MED, bool FO>
__device__ __forceinline__ void walk_inside(const SpectraArgs &a, const DatasetDev &ds,
                                            const typename RecOf<UW>::type *bp, int gb, int st, const double (&h)[S],
                                            int p, bool active, Run<S> &r)
{
    unsigned parity[S];                             /* unit weights: parity bits of this stretch's events, per term */
#pragma unroll
    for (int k = 0; k < S; ++k) parity[k] = 0u;
    static_assert(EB * K <= 32, "one parity register per term and stretch");
#pragma unroll
    for (int u = 0; u < K; ++u) {
        const double2 *q = reinterpret_cast<const double2 *>(bp + u * st);
#pragma unroll
        for (int j = 0; j < EB / 2; ++j) {
            const double2 t = q[j];
            if (UW) {
                /* every weight of the dataset is exactly 1 (the padding sits behind a NaN E_vis and never
                 * reaches this path): no weight is stored, and the run sum takes the accumulating form */
#pragma unroll
                for (int k = 0; k < S; ++k) {
                    if (folded<S>(FO, SM, MED, k)) half_cos_term_accumulate<S, SM, MED>(k, h[k], t.x, r.C[k], parity[k]);
                    else                       r.C[k] += half_cos_term<S, SM>(k, h[k], t.x);    /* 1 * g + C == g + C bit for bit */
                }
#pragma unroll
                for (int k = 0; k < S; ++k) {
                    if (folded<S>(FO, SM, MED, k)) half_cos_term_accumulate<S, SM, MED>(k, h[k], t.y, r.C[k], parity[k]);
                    else                       r.C[k] += half_cos_term<S, SM>(k, h[k], t.y);
                }
            } else {
                const double2 w = q[EB / 2 + j];
#pragma unroll
                for (int k = 0; k < S; ++k) r.C[k] = fma(w.x, half_cos_term<S, SM>(k, h[k], t.x), r.C[k]);
#pragma unroll
                for (int k = 0; k < S; ++k) r.C[k] = fma(w.y, half_cos_term<S, SM>(k, h[k], t.y), r.C[k]);
            }
        }
        if (!UW) r.W += reinterpret_cast<const EventBatchW *>(bp + u * st)->wsum;
        if (DBG)
            for (int j = 0; j < EB; ++j) dbg_mark<DBG>(a, ds, p, active, gb + u * st, j, r.cur);
    }
    if (UW) {
        r.W += (double)(EB * K);                    /* whole numbers: the same bits as K separate adds */
#pragma unroll
        for (int k = 0; k < S; ++k)
            if (FO && S == 2 && !(SM && k == S - 1) && !(MED && k == 0)) r.odd[k] += __popc(parity[k]);
    }
}

/* the half-turn coefficients of the lane's point, by value (they travel to the non-inlined slow path) */
template <int S> struct Coef { double h[S]; };

/* A batch in which a run ends (or none is open yet): its events one by one (rows a2-a4).  Rare -- once per
 * bin edge and lane -- and therefore NOT inlined and not unrolled: the hot loop stays small, and a warp that
 * meets an edge fetches few instruction lines it has not seen before (a cold instruction line costs as much as
 * a DRAM access; round 2 timeline: warps that met an edge finished 20 us late).  Everything by value: the run
 * must stay in registers in the caller. */
template <int S, bool UW, bool DBG>
__device__ __noinline__ Run<S> walk_batch_slow(const SpectraArgs &a, Tables T, const DatasetDev &ds,
                                               const typename RecOf<UW>::type *bp, int gb, Coef<S> c,
                                               const float *thr, float2 safe, int p, bool active, Run<S> r)
{
    const int B = ds.n_bins;
#pragma unroll 1
    for (int j = 0; j < EB; ++j) {
        const float v = bp->v[j];
        if (!(v < r.hi)) {
            int b;
            float nhi;
            if (r.hi > -pos_inf() && r.hi < pos_inf() && v <= safe.y) {
                /* r.hi = thr[cur + 1] <= v inside the table's interval: scan forward */
                b = r.cur + 1;
                nhi = r.hi2;
                while (b < B && !(v < nhi)) { ++b; nhi = thr_at(thr, B, b + 1); }
            } else {
                b = locate_bin(ds, thr, safe, theta_of(a, T.params, p), v, nhi);
            }
            if (b != r.cur) {
                flush_run<S>(a, T, ds, p, active, r);
                r.cur = b;
            }
            r.hi = nhi;
            r.hi2 = thr_at(thr, B, b + 2);
        }
        /* the padding of the last batch (E_vis = NaN, so it is in no bin): weight 0 in a weighted store,
         * skipped by index in a unit-weight one */
        const bool pad = UW && (long long)gb * EB + j >= ds.n_events;
        const double x = bp->x[j];
        double w = 1.0;
        if (!UW) w = reinterpret_cast<const EventBatchW *>(bp)->w[j];
#pragma unroll
        for (int k = 0; k < S; ++k) {
            if (UW) {
                if (pad) continue;
                if (folded<S>(r.fo, r.sm, r.med, k)) {        /* the accumulating form of walk_inside, one event at a time */
                    unsigned parity = 0u;               /* (n = 0 wherever a three-term model folds a term) */
                    half_cos_accumulate(c.h[k], x, r.C[k], parity);
                    if (S == 2) r.odd[k] += (int)(parity >> 31);
                } else {
                    r.C[k] += half_cos_halfturns(c.h[k], x);
                }
            } else {
                r.C[k] = fma(w, half_cos_halfturns(c.h[k], x), r.C[k]);
            }
        }
        if (UW) { if (!pad) r.W += 1.0; }
        else    r.W += w;
        dbg_mark<DBG>(a, ds, p, active, gb, j, r.cur);
    }
    return r;
}

/* One batch of the lane's stream (rows a2-a4); gb: its index in the dataset. */
template <int S, bool UW, bool DBG, bool SM, bool MED, bool FO>
__device__ __forceinline__ void walk_batch(const SpectraArgs &a, const Tables &T, const DatasetDev &ds,
                                           const typename RecOf<UW>::type *bp, int gb, const double (&h)[S],
                                           const float *thr, float2 safe, int p, bool active, Run<S> &r)
{
    if (bp->v[EB - 1] < r.hi) {
        /* rows a3 + a4: the store is sorted, so the whole batch lies in the run's bin (a padding event has
         * E_vis = NaN and fails the test: it never comes here) */
        walk_inside<S, UW, 1, DBG, SM, MED, FO>(a, ds, bp, gb, 1, h, p, active, r);
    } else {
        Coef<S> c;
#pragma unroll
        for (int k = 0; k < S; ++k) c.h[k] = h[k];
        r = walk_batch_slow<S, UW, DBG>(a, T, ds, bp, gb, c, thr, safe, p, active, r);
    }
}

/* `mine` batches of the lane's stream, bp, bp + st, bp + 2 st, ... (dataset batches gb, gb + st, ...): 4, 2 or 1 at a
 * time.  st = 1: every lane walks the whole unit; st = NS: the lane's sub-stream of a small batch of points. */
template <int S, bool UW, bool DBG, bool SM, bool MED, bool FO>
__device__ __forceinline__ void walk_stretch(const SpectraArgs &a, const Tables &T, const DatasetDev &ds,
                                             const typename RecOf<UW>::type *bp, int gb, int mine, int st,
                                             const double (&h)[S], const float *thr, float2 safe, int p, bool active,
                                             Run<S> &r)
{
    int i = 0;
#pragma unroll 1
    while (i < mine) {
        if (i + 4 <= mine && bp[3 * st].v[EB - 1] < r.hi) {
            walk_inside<S, UW, 4, DBG, SM, MED, FO>(a, ds, bp, gb + i * st, st, h, p, active, r);
            i += 4;
            bp += 4 * st;
        } else if (i + 2 <= mine && bp[st].v[EB - 1] < r.hi) {
            walk_inside<S, UW, 2, DBG, SM, MED, FO>(a, ds, bp, gb + i * st, st, h, p, active, r);
            i += 2;
            bp += 2 * st;
        } else {
            walk_batch<S, UW, DBG, SM, MED, FO>(a, T, ds, bp, gb + i * st, h, thr, safe, p, active, r);
            ++i;
            bp += st;
        }
    }
}

/* One warp, the nb batches [b0, b0 + nb) of dataset ds staged at `unit` (SHARED memory), point group g
 * (points 32 g ... 32 g + 31).  FULL: the group has more than 16 points, every lane walks all batches. */
/* lane -> (point, sub-stream) for a group of np <= 16 points: PL = 2^lg >= np point lanes, the nb batches of a unit
 * dealt out to NS = 32 / PL sub-streams in turn: this lane's are my0, my0 + NS, my0 + 2 NS, ... (`mine` of them).
 * Dealt out, not cut into contiguous pieces: the lanes of a warp then read NEIGHBOURING 48-byte records of the staged
 * unit with every 128-bit load -- eight lanes of a quarter-warp, eight different 16-byte bank groups -- where the
 * contiguous pieces (4 records = 192 bytes apart for one point) put four lanes on each group: ncu counted 1.49e6
 * bank-conflict wavefronts of 2.23e6 in a one-point call over 6e6 events.  A lane's events stay sorted, which is all
 * the run logic needs. */
__device__ __forceinline__ void substream_of(int np, int lane, int nb, int &lg, int &pl, int &my0, int &mine, int &st)
{
    lg = np <= 1 ? 0 : 32 - __clz(np - 1);
    pl = lane & ((1 << lg) - 1);
    st = 32 >> lg;
    my0 = lane >> lg;
    mine = my0 < nb ? (nb - my0 + st - 1) >> (5 - lg) : 0;
}

/* the hint a lane needs to open its run in unit [b0, b0 + nb) of dataset ds (group of np points; np > 16: all
 * lanes start at b0) */
__device__ __forceinline__ HintEntry load_hint(const DatasetDev &ds, int np, int lane, int b0, int nb)
{
    int my0 = 0;
    if (np <= 16) {
        int lg, pl, mine, st;
        substream_of(np, lane, nb, lg, pl, my0, mine, st);
        if (mine == 0) my0 = 0;                         /* a lane without a batch opens no run */
    }
    PHYLINO_ASSERT(b0 + my0 >= 0 && (b0 + my0 < ds.n_batches || (nb == 0 && b0 + my0 <= ds.n_batches)));
    const int2 e = __ldg(reinterpret_cast<const int2 *>(ds.hint + (b0 + my0) / HINT_BATCHES));
    HintEntry he;
    he.bin = e.x;
    he.x_env = __int_as_float(e.y);
    return he;
}

/* One warp, the nb batches [b0, b0 + nb) of dataset ds staged at `unit` (SHARED memory), point group g
 * (points 32 g ... 32 g + 31).  FULL: the group has more than 16 points, every lane walks all batches; lanes past
 * the last point shadow point 32 g and never flush.  hint: load_hint() of this lane for this unit and group. */
template <int S, bool FULL, bool UW, bool DBG, bool FO>
__device__ __forceinline__ void walk_unit(const SpectraArgs &a, const Tables &T, const DatasetDev &ds, int d,
                                          const void *unit, int b0, int nb, int g, int lane, HintEntry hint)
{
    typedef typename RecOf<UW>::type Rec;
    int my0 = 0, mine = nb, lg = 5, st = 1;
    bool active = 32 * g + lane < a.P;
    int p = 32 * g + (active ? lane : 0);
    if (!FULL) {
        const int np = min(32, a.P - 32 * g);
        int pl;
        substream_of(np, lane, nb, lg, pl, my0, mine, st);
        active = pl < np;
        p = 32 * g + (active ? pl : 0);
    }

    double h[S];
#pragma unroll
    for (int k = 0; k < S; ++k) h[k] = T.rec[(size_t)k * a.P + p];
    const int row = row_of(a, p);
    const float *thr = T.thr + (size_t)row * a.thr_stride + ds.thr_off;
    const float2 safe = T.safe[(size_t)row * a.n_datasets + d];

#ifdef PHYLINO_TRACE
    const long long q0 = clock64();
#endif
    Run<S> r;
    run_reset<S>(r);
    r.sm = T.small[g * a.n_datasets + d] != 0;
    r.fo = FO;
    PHYLINO_ASSERT(my0 >= 0 && mine >= 0 && (mine == 0 || my0 + (mine - 1) * st < nb) && p >= 0 && p < a.P);
    PHYLINO_ASSERT(row >= 0 && row < a.thr_rows);
    const Rec *bp = static_cast<const Rec *>(unit) + my0;
    if (mine > 0) open_run<S>(ds, thr, safe, bp->v[0], hint.bin, r);
#ifdef PHYLINO_TRACE
    const long long q1 = clock64();
#endif
    /* the last term's phase stays small over this dataset for every point of the group: its cheap form */
    /* the first term's phase cannot wrap for any event this lane meets in this item (unit-weight stores only: the
     * weighted ones keep the one form; neither does the single-launch kernel); a NaN coefficient compares false */
    constexpr bool ME = UW && FO;
    r.med = ME && __all_sync(0xffffffffu, fabs(h[0]) * (double)hint.x_env <= MEDIUM_PHASE);
    if (ME && r.med) {
        if (lane == 0) atomicAdd(a.med_count, (unsigned long long)nb * EB * (unsigned)min(32, a.P - 32 * g));
        if (r.sm) walk_stretch<S, UW, DBG, true, ME, FO>(a, T, ds, bp, b0 + my0, mine, st, h, thr, safe, p, active, r);
        else      walk_stretch<S, UW, DBG, false, ME, FO>(a, T, ds, bp, b0 + my0, mine, st, h, thr, safe, p, active, r);
    } else {
        if (r.sm) walk_stretch<S, UW, DBG, true, false, FO>(a, T, ds, bp, b0 + my0, mine, st, h, thr, safe, p, active, r);
        else      walk_stretch<S, UW, DBG, false, false, FO>(a, T, ds, bp, b0 + my0, mine, st, h, thr, safe, p, active, r);
    }
#ifdef PHYLINO_TRACE
    const long long q2 = clock64();
#endif
    if (FULL) flush_run<S>(a, T, ds, p, active, r);
    else      flush_run_substreams<S>(a, T, ds, p, active, lg, lane, r);
#ifdef PHYLINO_TRACE
    const long long q3 = clock64();
    const unsigned wid = blockIdx.x * WARPS + (threadIdx.x >> 5);
    if (lane == 0 && wid < 64) { g_sub[wid][0] += q1 - q0; g_sub[wid][1] += q2 - q1; g_sub[wid][2] += q3 - q2; g_sub[wid][3] += 1; }
#endif
}

/* lane 0 takes the next ticket of the work counter; the value is needed one item later */
__device__ __forceinline__ unsigned take_ticket(unsigned *counter, int lane)
{
    unsigned t = 0;
    /* atom.inc with a limit the counter never reaches (items + tickets stay below 2^31, fill_batch):
     * ptxas turns a uniform-address atom.add into its warp-aggregated form, whose shuffle would wait
     * for the atomic right here instead of one item later */
    if (lane == 0) asm volatile("atom.global.inc.u32 %0, [%1], 0x7fffffff;" : "=r"(t) : "l"(counter) : "memory");
    return t;
}

/* item -> (dataset, batches [b0, b1), chunk); SMALL: one chunk, no fine tail (an item is a unit) */
template <bool SMALL>
__device__ __forceinline__ void decode_item(const SpectraArgs &a, unsigned item, int &d, int &b0, int &b1, int &chunk)
{
    /* SMALL: the units nearest a bin edge are handed out first (api.cu build_unit_order) */
    const int unit = SMALL ? (a.unit_order ? __ldg(a.unit_order + item) : (int)item) : (int)(item / (unsigned)a.n_chunks);
    chunk = SMALL ? 0 : (int)(item - (unsigned)unit * (unsigned)a.n_chunks);
    if (!SMALL && unit >= a.tail_unit) {
        d = a.n_datasets - 1;
        b0 = a.tail_b0 + (unit - a.tail_unit) * a.tail_batches;
        b1 = min(b0 + a.tail_batches, a.ds[d].n_batches);
        PHYLINO_ASSERT(b0 >= 0 && b0 < b1 && (unsigned)(b1 - b0) * rec_bytes(a.ds[d]) <= (unsigned)STAGE_BUF_BYTES);
        return;
    }
    d = 0;
    for (int i = 1; i < a.n_datasets; ++i)
        if (unit >= a.ds[i].unit_begin) d = i;
    b0 = (unit - a.ds[d].unit_begin) * a.unit_batches;
    b1 = min(b0 + a.unit_batches, a.ds[d].n_batches);
    PHYLINO_ASSERT(item < (unsigned)a.n_items && d >= 0 && d < a.n_datasets);
    PHYLINO_ASSERT(b0 >= 0 && b0 < b1 && b1 <= a.ds[d].n_batches);
    PHYLINO_ASSERT((unsigned)(b1 - b0) * rec_bytes(a.ds[d]) <= (unsigned)STAGE_BUF_BYTES);
}

/* The persistent warp: its first two items are static (warp index, + number of warps), later ones come from
 * the counter (zero at kernel start; ticket t is item 2 nW + t): warps that meet expensive units (bin edges) or
 * slow memory simply claim fewer.  The unit of item i + 1 is copied into the warp's other buffer while item i
 * is walked.  first_item_loading(): the copy of the first item was started before the tables were ready. */
struct WarpPipe {
    unsigned char *buf0;            /* the warp's two unit buffers */
    unsigned long long *bars;       /* its two mbarriers */
};

struct Item { int d, b0, b1, chunk; };

template <bool SMALL>
__device__ __forceinline__ void start_first_item(const SpectraArgs &a, const WarpPipe &wp, unsigned cur, int lane)
{
    if (lane == 0) {
        mbar_init(wp.bars, 1);
        mbar_init(wp.bars + 1, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        if (cur < (unsigned)a.n_items) {
            Item it;
            decode_item<SMALL>(a, cur, it.d, it.b0, it.b1, it.chunk);
            bulk_load(wp.buf0, batch_ptr(a.ds[it.d], it.b0), (unsigned)(it.b1 - it.b0) * rec_bytes(a.ds[it.d]), wp.bars);
        }
    }
    __syncwarp();
}

/* the hint of the item's first group (its other groups, and the short last group of a large batch, load theirs
 * when they get there) */
__device__ __forceinline__ HintEntry item_hint(const SpectraArgs &a, const Item &it, int lane)
{
    const int np = min(32, a.P - 32 * it.chunk * a.chunk_groups);
    return load_hint(a.ds[it.d], np, lane, it.b0, it.b1 - it.b0);
}

/* SMALL: at most 16 points (one group of sub-streams): the full-group code is not even instantiated */
template <int S, bool DBG, bool SMALL>
__device__ __forceinline__ void ticket_loop(const SpectraArgs &a, const Tables &T, unsigned *counter, const WarpPipe &wp,
                                            unsigned cur, unsigned nW, int lane)
{
    const int n_groups = (a.P + 31) >> 5;
    const unsigned n_items = (unsigned)a.n_items;
    unsigned nxt = cur + nW;
    unsigned phase = 0u;                                /* bit b: parity of the next completion of buffer b */
    int b = 0;
#ifdef PHYLINO_TRACE
    const unsigned wme = cur;
    int wcount = 0;
    long long kacc[4] = {0, 0, 0, 0};
#endif
    Item it, nit;
    HintEntry hint, nhint;
    hint.bin = 0; hint.x_env = pos_inf();
    nhint = hint;
    if (cur < n_items) {
        decode_item<SMALL>(a, cur, it.d, it.b0, it.b1, it.chunk);
        hint = item_hint(a, it, lane);
    }
#pragma unroll 1
    while (cur < n_items) {
#ifdef PHYLINO_TRACE
        const long long k0 = clock64();
#endif
        const unsigned ticket = take_ticket(counter, lane);
        if (nxt < n_items) {
            /* the other buffer was last read one item ago; every lane has passed the shuffle below */
            decode_item<SMALL>(a, nxt, nit.d, nit.b0, nit.b1, nit.chunk);
            if (lane == 0)
                bulk_load(wp.buf0 + (b ^ 1) * STAGE_BUF_BYTES, batch_ptr(a.ds[nit.d], nit.b0),
                          (unsigned)(nit.b1 - nit.b0) * rec_bytes(a.ds[nit.d]), wp.bars + (b ^ 1));
            nhint = item_hint(a, nit, lane);            /* needed one item from now */
        }
#ifdef PHYLINO_TRACE
        const long long k1 = clock64();
#endif
        mbar_wait(wp.bars + b, (phase >> b) & 1u);
#ifdef PHYLINO_TRACE
        const long long k2 = clock64();
#endif
        phase ^= 1u << b;
        const DatasetDev &ds = a.ds[it.d];
        const int nb = it.b1 - it.b0;
        const int g0 = it.chunk * a.chunk_groups, g1 = min(g0 + a.chunk_groups, n_groups);
#pragma unroll 1
        for (int g = g0; g < g1; ++g) {
            const void *unit = wp.buf0 + b * STAGE_BUF_BYTES;
            const bool full = !SMALL && 32 * g + 16 < a.P;
            /* the prefetched hint fits the item's first group, and every full group (all lanes start at b0) */
            HintEntry hg = hint;
            if (!SMALL && g > g0 && !full) hg = load_hint(ds, a.P - 32 * g, lane, it.b0, nb);
            if (ds.unit_w) {
                if (full) { if (!SMALL) walk_unit<S, true, true, DBG, !SMALL>(a, T, ds, it.d, unit, it.b0, nb, g, lane, hg); }
                else      walk_unit<S, false, true, DBG, !SMALL>(a, T, ds, it.d, unit, it.b0, nb, g, lane, hg);
            } else {
                if (full) { if (!SMALL) walk_unit<S, true, false, DBG, !SMALL>(a, T, ds, it.d, unit, it.b0, nb, g, lane, hg); }
                else      walk_unit<S, false, false, DBG, !SMALL>(a, T, ds, it.d, unit, it.b0, nb, g, lane, hg);
            }
        }
#ifdef PHYLINO_TRACE
        const long long k3 = clock64();
        ++wcount;
#endif
        cur = nxt;
        it = nit;
        hint = nhint;
        nxt = 2u * nW + __shfl_sync(0xffffffffu, ticket, 0);    /* also orders this item's reads before the next copy */
#ifdef PHYLINO_TRACE
        const long long k4 = clock64();
        kacc[0] += k1 - k0; kacc[1] += k2 - k1; kacc[2] += k3 - k2; kacc[3] += k4 - k3;
#endif
        b ^= 1;
    }
#ifdef PHYLINO_TRACE
    if (lane == 0 && wme < 4096) {
        g_wend[wme] = gtime(); g_wunits[wme] = wcount;
        if (wme < 64) for (int i = 0; i < 4; ++i) g_wtrace[0][4 * wme + i] = (unsigned long long)kacc[i];
    }
#endif
}

template <int S, bool DBG>
__global__ void __launch_bounds__(WARPS * 32, CTAS_PER_SM) spectra_kernel(const __grid_constant__ SpectraArgs a)
{
    static_assert(EB == 4, "the batch loads are written for EB = 4");
    extern __shared__ __align__(128) unsigned char stage[];       /* [WARPS][2][STAGE_BUF_BYTES] */
    __shared__ unsigned long long bars[WARPS][2];
    const int lane = threadIdx.x & 31, wib = threadIdx.x >> 5;
    const unsigned nW = gridDim.x * WARPS, cur = blockIdx.x * WARPS + wib;
    WarpPipe wp;
    wp.buf0 = stage + (size_t)(2 * wib) * STAGE_BUF_BYTES;
    wp.bars = &bars[wib][0];
    start_first_item<false>(a, wp, cur, lane);
    /* everything above touched only kernel parameters and the event store; the records, thresholds
     * and the work counter come from the setup kernel (no-op unless launched as its dependent) */
    asm volatile("griddepcontrol.wait;" ::: "memory");
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    Tables T;
    T.params = a.params;
    T.rec = a.rec;
    T.thr = a.thr;
    T.safe = a.safe;
    T.small = a.small;
    ticket_loop<S, DBG, false>(a, T, a.counter, wp, cur, nW, lane);
}

/* ---- small batches (at most FUSED_MAX_POINTS points: one group of sub-streams) ----
 * Rows a1 and the tables of a3 per CTA in shared memory -- no setup launch -- then the same ticket loop over the
 * units.  The finalize kernel behind it is its programmatic dependent and does its table work meanwhile; it also
 * zeroes the work counter a.done again.  A batch of at most PARAM_BLOB_DOUBLES parameters may travel by value
 * with the kernel arguments (blob): a host call then needs no copy engine at all. */
template <int S, bool DBG>
__global__ void __launch_bounds__(WARPS * 32, CTAS_PER_SM) spectra_fused_kernel(const __grid_constant__ SpectraArgs a,
                                                                      const __grid_constant__ ParamBlob blob)
{
    /* [WARPS][2][STAGE_BUF_BYTES] stage | rec [rec_fields x P] | safe [thr_rows x D] | thr [thr_rows x thr_stride] */
    extern __shared__ __align__(128) unsigned char stage[];
    __shared__ unsigned long long bars[WARPS][2];
    __shared__ unsigned char small_s[PHYLINO_MAX_DATASETS];
    const int lane = threadIdx.x & 31, wib = threadIdx.x >> 5;
    const unsigned nW = gridDim.x * WARPS, cur = blockIdx.x * WARPS + wib;
    TRACE_MIN(0);
    TRACE_MAX(1);
    WarpPipe wp;
    wp.buf0 = stage + (size_t)(2 * wib) * STAGE_BUF_BYTES;
    wp.bars = &bars[wib][0];
    start_first_item<true>(a, wp, cur, lane);
    /* the event copy above touched only the event store; the parameters may come from a kernel before us, and
     * the accumulators and the work counter must have been left clean by the finalize kernel of the call before */
    asm volatile("griddepcontrol.wait;" ::: "memory");
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");

    double *rec_s = reinterpret_cast<double *>(stage + (size_t)WARPS * 2 * STAGE_BUF_BYTES);
    float2 *safe_s = reinterpret_cast<float2 *>(rec_s + (size_t)(2 * S + 2) * a.P);
    float *thr_s = reinterpret_cast<float *>(safe_s + (size_t)a.thr_rows * a.n_datasets);
#ifdef PHYLINO_CHECKED
    {
        unsigned dyn;
        asm volatile("mov.u32 %0, %%dynamic_smem_size;" : "=r"(dyn));
        PHYLINO_ASSERT((size_t)((unsigned char *)(thr_s + (size_t)a.thr_rows * a.thr_stride) - stage) <= dyn);
        PHYLINO_ASSERT(a.P >= 1 && a.P <= FUSED_MAX_POINTS && a.n_chunks == 1 && a.tail_unit == a.n_units);
    }
#endif
    /* a.params == NULL: the batch came by value with the kernel arguments (host entry points, small batches) */
    const double *params = a.params ? a.params : blob.v;
    if (threadIdx.x < 32) {             /* at most FUSED_MAX_POINTS <= 32 points: the first warp */
        const double h_last = (int)threadIdx.x < a.P ? point_record<S>(a, params, threadIdx.x, rec_s) : 0.0;
        group_flags(a, h_last, small_s);
    }
    for (int e = threadIdx.x; e < a.thr_rows * a.thr_stride; e += WARPS * 32)
        threshold_entry(a, params, e / a.thr_stride, e % a.thr_stride, thr_s, safe_s);
    __syncthreads();
    TRACE_MAX(2);
    if (blockIdx.x == 0 && (int)threadIdx.x < a.n_datasets) a.small[threadIdx.x] = small_s[threadIdx.x];   /* for phylino_last_small_phase */
    Tables T;
    T.params = params;
    T.rec = rec_s;
    T.thr = thr_s;
    T.safe = safe_s;
    T.small = small_s;
    ticket_loop<S, DBG, true>(a, T, a.done, wp, cur, nW, lane);
    TRACE_MIN(3);
    TRACE_MAX(4);
}

/* dynamic shared memory of one CTA: two unit buffers per warp */
constexpr size_t STAGE_BYTES = (size_t)WARPS * 2 * STAGE_BUF_BYTES;
/* records + thresholds of the small-batch kernel: what 227 KB of shared memory per CTA leave beside the staging */
constexpr size_t FUSED_TABLE_MAX = (227 * 1024 - 1024 - STAGE_BYTES) < 160 * 1024 ? (227 * 1024 - 1024 - STAGE_BYTES) : 160 * 1024;

template <int S, bool DBG> cudaError_t launch_t(const SpectraArgs &a, cudaStream_t st, bool pdl)
{
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(a.n_warps / WARPS);
    cfg.blockDim = dim3(WARPS * 32);
    cfg.dynamicSmemBytes = STAGE_BYTES;
    cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = pdl ? 1 : 0;
    return cudaLaunchKernelEx(&cfg, spectra_kernel<S, DBG>, a);
}

template <int S, bool DBG>
cudaError_t launch_fused_t(const SpectraArgs &a, const ParamBlob &blob, cudaStream_t st, bool pdl)
{
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(a.n_warps / WARPS);
    cfg.blockDim = dim3(WARPS * 32);
    cfg.dynamicSmemBytes = STAGE_BYTES + fused_table_bytes(S, a.P, a.thr_rows, a.thr_stride, a.n_datasets);
    cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = pdl ? 1 : 0;
    return cudaLaunchKernelEx(&cfg, spectra_fused_kernel<S, DBG>, a, blob);
}

/* the dynamic shared memory sits above the 48 KB default: opt every instantiation in (the attribute is per
 * function, so a context that changes its oscillation model finds the other S ready too) */
template <int S, bool DBG> cudaError_t allow_stage_t()
{
    cudaError_t e = cudaFuncSetAttribute(spectra_kernel<S, DBG>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                         (int)STAGE_BYTES);
    if (e != cudaSuccess) return e;
    return cudaFuncSetAttribute(spectra_fused_kernel<S, DBG>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                (int)(STAGE_BYTES + FUSED_TABLE_MAX));
}

} // namespace

cudaError_t allow_stage_all()
{
    cudaError_t e = allow_stage_t<2, false>();
    if (e == cudaSuccess) e = allow_stage_t<3, false>();
    if (e == cudaSuccess) e = allow_stage_t<2, true>();
    if (e == cudaSuccess) e = allow_stage_t<3, true>();
    return e;
}

#ifdef PHYLINO_TRACE
extern "C" __attribute__((visibility("default"))) int phylino_debug_trace(unsigned long long *out, int reset)
{
    if (out && cudaMemcpyFromSymbol(out, g_trace, sizeof(unsigned long long) * 8) != cudaSuccess) return 1;
    if (out && reset == 2) {        /* out: [8 + 4 * 256 + 4] */
        if (cudaMemcpyFromSymbol(out + 8, g_wtrace, sizeof(unsigned long long) * 1024) != cudaSuccess) return 1;
        int n[4];
        if (cudaMemcpyFromSymbol(n, g_wn, sizeof n) != cudaSuccess) return 1;
        for (int i = 0; i < 4; ++i) out[8 + 1024 + i] = (unsigned long long)n[i];
        return 0;
    }
    if (out && reset == 4) return cudaMemcpyFromSymbol(out, g_sub, sizeof(long long) * 256) != cudaSuccess;
    if (out && reset == 3) {        /* out: [4096 end times | 4096 unit counts] */
        if (cudaMemcpyFromSymbol(out, g_wend, sizeof(unsigned long long) * 4096) != cudaSuccess) return 1;
        static int u[4096];
        if (cudaMemcpyFromSymbol(u, g_wunits, sizeof u) != cudaSuccess) return 1;
        for (int i = 0; i < 4096; ++i) out[4096 + i] = (unsigned long long)u[i];
        return 0;
    }
    if (reset) {
        static long long zs[256];
        if (cudaMemcpyToSymbol(g_sub, zs, sizeof zs) != cudaSuccess) return 1;
        int zn[4] = {0, 0, 0, 0};
        if (cudaMemcpyToSymbol(g_wn, zn, sizeof zn) != cudaSuccess) return 1;
        unsigned long long z[8] = {~0ull, 0, 0, ~0ull, 0, 0, 0, 0};
        if (cudaMemcpyToSymbol(g_trace, z, sizeof z) != cudaSuccess) return 1;
    }
    return 0;
}
#endif

size_t fused_table_bytes(int S, int P, int thr_rows, int thr_stride, int n_datasets)
{
    const size_t b = (size_t)rec_fields(S) * P * sizeof(double) + (size_t)thr_rows * n_datasets * sizeof(float2) +
                     (size_t)thr_rows * thr_stride * sizeof(float);
    return (b + 15) / 16 * 16;
}

bool fused_fits(size_t table_bytes) { return table_bytes <= FUSED_TABLE_MAX; }

/* warps of a persistent grid the chip holds at once: the ticket kernel (fused = false) or the single-launch
 * kernel with `table_bytes` of tables */
cudaError_t spectra_max_warps(int S, int sm_count, bool fused, size_t table_bytes, int *warps)
{
    int per_sm = 0;
    cudaError_t e = cudaSuccess;
    if (fused) {
        e = S == 2 ? cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, spectra_fused_kernel<2, false>, WARPS * 32,
                                                                   STAGE_BYTES + table_bytes)
                   : cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, spectra_fused_kernel<3, false>, WARPS * 32,
                                                                   STAGE_BYTES + table_bytes);
    } else {
        e = S == 2 ? cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, spectra_kernel<2, false>, WARPS * 32, STAGE_BYTES)
                   : cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, spectra_kernel<3, false>, WARPS * 32, STAGE_BYTES);
    }
    if (e != cudaSuccess) return e;
    if (per_sm < 1) return cudaErrorLaunchOutOfResources;
    *warps = sm_count * per_sm * WARPS;
    return cudaSuccess;
}

cudaError_t launch_setup(const SpectraArgs &a, int S, cudaStream_t st)
{
    if (a.P <= 0) return cudaSuccess;
    const int rec_blocks = (a.P + SETUP_THREADS - 1) / SETUP_THREADS;
    if (S == 2) setup_kernel<2><<<rec_blocks + a.thr_rows, SETUP_THREADS, 0, st>>>(a, rec_blocks);
    else        setup_kernel<3><<<rec_blocks + a.thr_rows, SETUP_THREADS, 0, st>>>(a, rec_blocks);
    return cudaGetLastError();
}

/* persistent grid of a.n_warps warps (a multiple of WARPS) that claim the a.n_items work items */
cudaError_t launch_spectra(const SpectraArgs &a, int S, cudaStream_t st, bool pdl, bool dbg)
{
    if (a.n_items <= 0 || a.P <= 0 || a.n_warps < WARPS) return cudaSuccess;
    if (dbg) return S == 2 ? launch_t<2, true>(a, st, pdl) : launch_t<3, true>(a, st, pdl);
    return S == 2 ? launch_t<2, false>(a, st, pdl) : launch_t<3, false>(a, st, pdl);
}

/* the kernel for at most FUSED_MAX_POINTS points (setup fused in): a.n_warps warps */
cudaError_t launch_fused(const SpectraArgs &a, const ParamBlob &blob, int S, cudaStream_t st, bool pdl, bool dbg)
{
    if (a.P <= 0 || a.n_warps < WARPS) return cudaSuccess;
    if (dbg) return S == 2 ? launch_fused_t<2, true>(a, blob, st, pdl) : launch_fused_t<3, true>(a, blob, st, pdl);
    return S == 2 ? launch_fused_t<2, false>(a, blob, st, pdl) : launch_fused_t<3, false>(a, blob, st, pdl);
}

} // namespace phylino
