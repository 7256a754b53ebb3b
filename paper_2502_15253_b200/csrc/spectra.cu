/*
 * spectra.cu -- the batched oscillation-weight + histogram kernels (
 * PAPER.md:177 signal step 1, :183 "the most time-demanding computational step").
 *
 * Layout of the work: ONE PARAMETER POINT PER LANE.  The E_vis-sorted events of a dataset are cut
 * into 96-byte batches of EB events and the batches into units; a work item is one unit x a chunk
 * of point groups (32 points each).  The warps of a persistent grid claim items from a global
 * counter (dynamic balance: units that contain bin edges cost more; the last stretch of the store is
 * cut into quarter-size units so the warps run out of work together) and walk the unit once per group.
 *
 * Staging.  Each warp owns two unit-sized buffers in shared memory and one mbarrier per buffer; lane 0
 * starts ONE bulk async copy (cp.async.bulk global -> shared, completion on the mbarrier) of the NEXT
 * item's unit while the current one is walked.  The hot loop reads warp-uniform LDS.128 broadcasts;
 * everything that depends on the point (half-turn coefficients h_k, the run accumulators, the current
 * bin, its fp32 upper threshold and the one after it) lives in the lane's registers.  No shuffles in
 * the loop, no block barriers.  A group of fewer than 17 points splits the unit into 32/PL sub-streams
 * (PL = points rounded up to a power of two), so that a batch of 1 point still uses all 32 lanes.
 *
 * Oscillation weight (row a2).  P_ee = P0 + sum_k A_k g_k with g = 1/2 cos(2 phase) (devmath.cuh):
 * the lane accumulates C_k = sum_e w_e g_k(e) and W = sum_e w_e over a run of events that share a
 * bin; the run's total is P0 W + sum_k A_k C_k, formed once per run.  Per event x point that is
 * 11 fp64 instructions and one integer instruction per oscillation term.
 *
 * Binning (row a3).  For one point the map v -> E' = fma(fma(a2,v,a1),v,a0) is non-decreasing over
 * the fp32 values of a dataset (checked per point by the setup kernel), so bin(E'(v)) >= b <=>
 * v >= T[b] with T[b] the smallest fp32 value whose E' reaches edges[b].  T is found by bisection
 * with the SAME fp64 fma sequence, hence the fp32 comparison decides exactly what the fp64
 * comparison E' >= edges[b] decides: bit-exact bins.  Events are sorted, so 4, 2 or 1 batches lie
 * inside the lane's current bin iff the LAST event of the last one is below the bin's upper threshold:
 * one fp32 compare, then a straight-line stretch of rows a2 + a4 (datasets whose weights are all exactly
 * 1 skip the weight loads).  A lane opens its run at the first event of a unit from the load-time hint
 * bin0 of the batch.  Events outside the interval on which a table is proven (and points that fail the
 * monotonicity check) take the per-event fp64 map.
 *
 * Histogram (rows a4, a5).  When a run ends (bin edge, end of the unit) its fp64 total is converted
 * once to 64-bit fixed point and added to the (point, bin) accumulator with an integer RED.
 * Integer addition is associative: the result depends neither on which warp walks an item nor on
 * the order of arrival, i.e. bitwise reproducible with no float atomics anywhere (the cut of the
 * events into items is a function of the sizes only).
 *
 * Component mode (cross-point caching): the launch's points are virtual points (an energy-scale class
 * plus S splittings) and a run is flushed as S + 1 separate sums; finalize.cu combines them per point.
 *
 * Launch.  The spectra kernel is a programmatic dependent of the setup kernel: barriers and the first
 * event copy are set up while the setup kernel runs; griddepcontrol.wait precedes the first read of a
 * record, a threshold or the work counter.
 */
#include "devmath.cuh"

namespace phylino {

namespace {

__device__ __forceinline__ float pos_inf() { return __int_as_float(0x7f800000); }

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

/* smallest fp32 v in [safe_lo, safe_hi] (positive, normal) with E'(v) >= edge, +inf if none */
__device__ float threshold_search(double a0, double a1, double a2, double edge, float safe_lo, float safe_hi)
{
    if (!(safe_lo <= safe_hi)) return pos_inf();
    if (!(escale(a0, a1, a2, (double)safe_hi) >= edge)) return pos_inf();
    if (escale(a0, a1, a2, (double)safe_lo) >= edge) return safe_lo;
    int lo = __float_as_int(safe_lo), hi = __float_as_int(safe_hi);   /* E'(lo) < edge <= E'(hi) */
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

__device__ __forceinline__ const double *theta_of(const SpectraArgs &a, int p)
{
    return a.params + (size_t)(a.comp ? a.class_rep[a.vp_class[p]] : p) * a.n_params;
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
            if (__ldg(thr + mid) <= v) lo = mid; else up = mid;
        }
        hi = lo < B ? __ldg(thr + lo + 1) : pos_inf();
        return lo;
    }
    double a0, a1, a2;
    energy_scale_of(ds, theta, a0, a1, a2);
    hi = -pos_inf();
    return bin_search(ds.edges, B, escale(a0, a1, a2, (double)v));
}

/* ---- setup kernel: per-point records and threshold rows (row a1 and the tables of row a3) ---------
 * blocks [0, rec_blocks): one thread per point writes rec[field * P + p] = h_k, A_k, P0, bad;
 * blocks [rec_blocks, rec_blocks + thr_rows): one CTA per threshold row. */
template <int S>
__global__ void __launch_bounds__(SETUP_THREADS) setup_kernel(const __grid_constant__ SpectraArgs a, int rec_blocks)
{
    /* programmatic dependent launch: the spectra kernel may start its prologue (barriers, first copy of
     * event data) now; it waits for this grid to finish before it reads anything written here */
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    if ((int)blockIdx.x < rec_blocks) {
        const int p = blockIdx.x * SETUP_THREADS + threadIdx.x;
        if (p == 0) *a.counter = 2u * (unsigned)a.n_warps;     /* see spectra_kernel */
        if (p >= a.P) return;
        if (a.comp) {
            /* virtual point: slot s computes the half-turn coefficient of (real point, term) vp_src */
#pragma unroll
            for (int k = 0; k < S; ++k) {
                const int src = a.vp_src[(size_t)p * S + k];
                double A[MAX_TERMS], dm2[MAX_TERMS];
                osc_terms(a.osc, a.params + (size_t)(src >> 2) * a.n_params, A, dm2);
                a.rec[(size_t)k * a.P + p] = halfturn_coeff(dm2[src & 3]);
            }
            return;
        }
        const double *theta = a.params + (size_t)p * a.n_params;
        double A[MAX_TERMS], dm2[MAX_TERMS];
        osc_terms(a.osc, theta, A, dm2);
        double asum = 0.0, half = 0.0;
#pragma unroll
        for (int k = 0; k < S; ++k) {
            a.rec[(size_t)k * a.P + p] = halfturn_coeff(dm2[k]);
            a.rec[(size_t)(S + k) * a.P + p] = A[k];
            asum += fabs(A[k]);
            half += A[k];
        }
        a.rec[(size_t)(2 * S) * a.P + p] = 1.0 - 0.5 * half;            /* P0 */
        /* |P0| + 1/2 sum|A_k| <= 1 + sum|A_k| <= 4 keeps every run total inside the fixed-point range */
        a.rec[(size_t)(2 * S + 1) * a.P + p] = (asum <= 3.0) ? 0.0 : 1.0;
        return;
    }
    const int row = blockIdx.x - rec_blocks;
    /* only read where idx_a >= 0 */
    const double *theta = a.params + (size_t)(a.comp ? a.class_rep[row] : row) * a.n_params;
    for (int e = threadIdx.x; e < a.thr_stride; e += SETUP_THREADS) {
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
        a.thr[(size_t)row * a.thr_stride + e] = t;
        if (b == 0) a.safe[(size_t)row * a.n_datasets + d] = make_float2(slo, shi);
    }
}

/* ---- the hot kernel ---------------------------------------------------------------------------- */

/* the lane's open run: events of ONE bin seen since the last flush */
template <int S> struct Run {
    double C[S];    /* sum of w g_k over the run */
    double W;       /* sum of w over the run */
    int    cur;     /* its bin; < 0 or >= n_bins: events that land in no bin (never flushed) */
    float  hi;      /* later events below hi stay in the run (-inf: re-locate at the next event) */
    float  hi2;     /* threshold after hi (+inf past the last edge), loaded when the run opened so that the
                     * end of the run does not wait for it; meaningful only while hi is a table threshold */
};

template <int S>
__device__ __forceinline__ void flush_run(const SpectraArgs &a, const DatasetDev &ds, int p, bool active, Run<S> &r)
{
    if (a.comp && active && r.cur >= 0 && r.cur < ds.n_bins) {
        /* component mode: W and every C_k go to cells of their own (the amplitudes come later) */
        const size_t cell = (size_t)p * (S + 1) * a.total_bins + ds.bin_off + r.cur;
#pragma unroll
        for (int j = 0; j <= S; ++j) {
            unsigned fl;
            const long long q = to_fixed(j == 0 ? r.W : r.C[j - 1], ds.fx_scale, false, fl);
            if (q) atomicAdd((unsigned long long *)a.acc + cell + (size_t)j * a.total_bins, (unsigned long long)q);
            if (fl) atomicOr(a.flags + cell + (size_t)j * a.total_bins, fl);
        }
    } else if (active && r.cur >= 0 && r.cur < ds.n_bins) {
        double tot = a.rec[(size_t)(2 * S) * a.P + p] * r.W;                 /* P0 W */
#pragma unroll
        for (int k = 0; k < S; ++k) tot = fma(a.rec[(size_t)(S + k) * a.P + p], r.C[k], tot);
        const bool bad = a.rec[(size_t)(2 * S + 1) * a.P + p] != 0.0;
        unsigned fl;
        const long long q = to_fixed(tot, ds.fx_scale, bad, fl);
        const size_t cell = (size_t)p * a.total_bins + ds.bin_off + r.cur;
        if (q) atomicAdd((unsigned long long *)a.acc + cell, (unsigned long long)q);
        if (fl) atomicOr(a.flags + cell, fl);
    }
#pragma unroll
    for (int k = 0; k < S; ++k) r.C[k] = 0.0;
    r.W = 0.0;
}

/* The flush at the end of a unit when the group has at most 16 points: the 32 / PL sub-streams of a point
 * usually end in the same bin, and 32 lanes of every resident warp adding to the same one or two cells
 * would queue at the L2 atomic unit (same-address atomics: a 6e6-event, 1-point call spent 0.45 ms there).
 * Every lane converts its run to fixed point as usual; the integers of the lanes that share a cell are
 * summed over the sub-streams with shuffles (exact, so the bits are those of the separate REDs) and the
 * first lane of each cell issues one RED.  All 32 lanes call this together. */
template <int S>
__device__ __forceinline__ void flush_run_substreams(const SpectraArgs &a, const DatasetDev &ds, int p, bool active,
                                                     int lg, int lane, Run<S> &r)
{
    const bool live = active && r.cur >= 0 && r.cur < ds.n_bins;
    const int nq = a.comp ? S + 1 : 1;
    long long q[S + 1];
    unsigned fl[S + 1];
#pragma unroll
    for (int j = 0; j <= S; ++j) { q[j] = 0; fl[j] = 0; }
    unsigned long long cell = ~0ull;
    if (live) {
        if (a.comp) {
            cell = (unsigned long long)p * (S + 1) * a.total_bins + ds.bin_off + r.cur;
#pragma unroll
            for (int j = 0; j <= S; ++j) q[j] = to_fixed(j == 0 ? r.W : r.C[j - 1], ds.fx_scale, false, fl[j]);
        } else {
            double tot = a.rec[(size_t)(2 * S) * a.P + p] * r.W;
#pragma unroll
            for (int k = 0; k < S; ++k) tot = fma(a.rec[(size_t)(S + k) * a.P + p], r.C[k], tot);
            cell = (unsigned long long)p * a.total_bins + ds.bin_off + r.cur;
            q[0] = to_fixed(tot, ds.fx_scale, a.rec[(size_t)(2 * S + 1) * a.P + p] != 0.0, fl[0]);
        }
    }
    long long sum[S + 1];
#pragma unroll
    for (int j = 0; j <= S; ++j) sum[j] = 0;
    bool first = true;
    const int pl = lane & ((1 << lg) - 1);
    for (int src = pl; src < 32; src += 1 << lg) {              /* the sub-streams of this lane's point */
        const unsigned long long c = __shfl_sync(0xffffffffu, cell, src);
        const bool same = live && c == cell;
        if (same && src < lane) first = false;
#pragma unroll
        for (int j = 0; j <= S; ++j) {
            const long long v = __shfl_sync(0xffffffffu, q[j], src);
            if (same && j < nq) sum[j] += v;
        }
    }
    if (live) {
        for (int j = 0; j < nq; ++j) {
            if (first && sum[j]) atomicAdd((unsigned long long *)a.acc + cell + (size_t)j * a.total_bins, (unsigned long long)sum[j]);
            if (fl[j]) atomicOr(a.flags + cell + (size_t)j * a.total_bins, fl[j]);
        }
    }
#pragma unroll
    for (int k = 0; k < S; ++k) r.C[k] = 0.0;
    r.W = 0.0;
}

/* threshold row entry with the conventions thr[-1] = -inf, thr[B + 1] = +inf */
__device__ __forceinline__ float thr_at(const float *thr, int B, int i)
{
    return i < 0 ? -pos_inf() : (i > B ? pos_inf() : __ldg(thr + i));
}

/* One batch of the lane's stream (rows a2-a4). */
template <int S>
__device__ __forceinline__ void walk_batch(const SpectraArgs &a, const DatasetDev &ds, const EventBatch *bp,
                                           const double (&h)[S], const float *thr, float2 safe, int p, bool active,
                                           Run<S> &r)
{
    const int B = ds.n_bins;
    double x[EB], w[EB];
    {
        const double2 *q = reinterpret_cast<const double2 *>(bp);
#pragma unroll
        for (int j = 0; j < EB / 2; ++j) {
            double2 t = q[j], u = q[EB / 2 + j];
            x[2 * j] = t.x; x[2 * j + 1] = t.y;
            w[2 * j] = u.x; w[2 * j + 1] = u.y;
        }
    }
    const float v_last = bp->v[EB - 1];

    /* row a2: g_k of every event of the batch */
    double gk[S][EB];
#pragma unroll
    for (int j = 0; j < EB; ++j)
#pragma unroll
        for (int k = 0; k < S; ++k) gk[k][j] = half_cos_halfturns(h[k], x[j]);

    if (v_last < r.hi) {
        /* rows a3 + a4: the store is sorted, so the whole batch lies in the run's bin */
#pragma unroll
        for (int j = 0; j < EB; ++j)
#pragma unroll
            for (int k = 0; k < S; ++k) r.C[k] = fma(w[j], gk[k][j], r.C[k]);
        r.W += bp->wsum;
    } else {
        /* a run ends inside the batch (or none is open yet): walk its events one by one */
        const float4 v4 = *reinterpret_cast<const float4 *>(bp->v);
        const float v[EB] = {v4.x, v4.y, v4.z, v4.w};
#pragma unroll
        for (int j = 0; j < EB; ++j) {
            if (!(v[j] < r.hi)) {
                int b;
                float nhi;
                if (r.hi > -pos_inf() && r.hi < pos_inf() && v[j] <= safe.y) {
                    /* r.hi = thr[cur + 1] <= v inside the table's interval: scan forward */
                    b = r.cur + 1;
                    nhi = r.hi2;
                    while (b < B && !(v[j] < nhi)) { ++b; nhi = thr_at(thr, B, b + 1); }
                } else {
                    b = locate_bin(ds, thr, safe, theta_of(a, p), v[j], nhi);
                }
                if (b != r.cur) {
                    flush_run<S>(a, ds, p, active, r);
                    r.cur = b;
                }
                r.hi = nhi;
                r.hi2 = thr_at(thr, B, b + 2);
            }
#pragma unroll
            for (int k = 0; k < S; ++k) r.C[k] = fma(w[j], gk[k][j], r.C[k]);
            r.W += w[j];
        }
    }
}

/* K consecutive batches known to lie inside the lane's open run (the store is sorted: the last
 * event of the last batch is below r.hi): rows a2 + a4 only, straight-line. */
template <int S, bool UW, int K>
__device__ __forceinline__ void walk_inside(const EventBatch *bp, const double (&h)[S], Run<S> &r)
{
#pragma unroll
    for (int u = 0; u < K; ++u) {
        const double2 *q = reinterpret_cast<const double2 *>(bp + u);
#pragma unroll
        for (int j = 0; j < EB / 2; ++j) {
            const double2 t = q[j];
            if (UW) {
                /* every weight of the dataset is exactly 1 (the padding, weight 0, sits behind a NaN E_vis
                 * and never reaches this path): 1 * g + C == g + C bit for bit, and w is not loaded */
#pragma unroll
                for (int k = 0; k < S; ++k) r.C[k] += half_cos_halfturns(h[k], t.x);
#pragma unroll
                for (int k = 0; k < S; ++k) r.C[k] += half_cos_halfturns(h[k], t.y);
            } else {
                const double2 w = q[EB / 2 + j];
#pragma unroll
                for (int k = 0; k < S; ++k) r.C[k] = fma(w.x, half_cos_halfturns(h[k], t.x), r.C[k]);
#pragma unroll
                for (int k = 0; k < S; ++k) r.C[k] = fma(w.y, half_cos_halfturns(h[k], t.y), r.C[k]);
            }
        }
        if (!UW) r.W += bp[u].wsum;
    }
    if (UW) r.W += (double)(EB * K);                /* whole numbers: the same bits as K separate adds */
}

/* One warp, the nb batches of one unit of dataset ds staged at `unit` (SHARED memory), point group g
 * (points 32 g ... 32 g + 31).  FULL: the group has more than 16 points, every lane walks all batches. */
template <int S, bool FULL, bool UW>
__device__ __forceinline__ void walk_unit(const SpectraArgs &a, const DatasetDev &ds, int d, const EventBatch *unit,
                                          int nb, int g, int lane)
{
    /* lane -> (point, sub-stream): a group of np < 32 points uses PL = 2^ceil(log2 np) point lanes
     * and splits the batches into NS = 32 / PL contiguous sub-streams */
    /* FULL: more than 16 points, so every lane walks all batches; lanes past the last point shadow point
     * 32 g and never flush */
    int my0 = 0, mine = nb, iters = nb, lg = 5;
    bool active = 32 * g + lane < a.P;
    int p = 32 * g + (active ? lane : 0);
    if (!FULL) {
        const int np = min(32, a.P - 32 * g);
        int PL = 1;
        lg = 0;
        while (PL < np) { PL <<= 1; ++lg; }
        const int NS = 32 / PL;
        const int pl = lane & (PL - 1), s = lane / PL;
        active = pl < np;
        p = 32 * g + (active ? pl : 0);
        my0 = nb * s / NS;
        mine = nb * (s + 1) / NS - my0;
        iters = (nb + NS - 1) / NS;                        /* >= mine for every lane */
    }

    double h[S];
#pragma unroll
    for (int k = 0; k < S; ++k) h[k] = a.rec[(size_t)k * a.P + p];
    const int row = row_of(a, p);
    const float *thr = a.thr + (size_t)row * a.thr_stride + ds.thr_off;
    const float2 safe = a.safe[(size_t)row * a.n_datasets + d];
    const int B = ds.n_bins;

    Run<S> r;
#pragma unroll
    for (int k = 0; k < S; ++k) r.C[k] = 0.0;
    r.W = 0.0;
    r.cur = -1;
    r.hi = -pos_inf();
    r.hi2 = pos_inf();

    const EventBatch *bp = unit + my0;
    if (mine > 0) {
        /* open the run at the lane's first event: start from the load-time hint (its bin under the
         * identity energy scale) and step to the bin the lane's own thresholds give -- the same
         * decision as the binary search of locate_bin, usually without a single dependent load */
        const float v0 = bp->v[0];
        if (v0 >= safe.x && v0 <= safe.y) {
            int b = max(-1, min(bp->bin0, B));
            float lo = thr_at(thr, B, b), hi = thr_at(thr, B, b + 1);
            while (b >= 0 && v0 < lo) { --b; hi = lo; lo = thr_at(thr, B, b); }
            while (b < B && !(v0 < hi)) { ++b; hi = thr_at(thr, B, b + 1); }
            r.cur = b;
            r.hi = hi;
            r.hi2 = thr_at(thr, B, b + 2);
        }
    }
    if (FULL) {
        int i = 0;
#pragma unroll 1
        while (i < nb) {
            if (i + 4 <= nb && bp[3].v[EB - 1] < r.hi) {
                walk_inside<S, UW, 4>(bp, h, r);
                i += 4;
                bp += 4;
            } else if (i + 2 <= nb && bp[1].v[EB - 1] < r.hi) {
                walk_inside<S, UW, 2>(bp, h, r);
                i += 2;
                bp += 2;
            } else {
                walk_batch<S>(a, ds, bp, h, thr, safe, p, active, r);
                ++i;
                ++bp;
            }
        }
    } else {
#pragma unroll 1
        for (int i = 0; i < iters; ++i, ++bp) {
            if (i >= mine) continue;
            walk_batch<S>(a, ds, bp, h, thr, safe, p, active, r);
        }
    }
    if (FULL) flush_run<S>(a, ds, p, active, r);
    else      flush_run_substreams<S>(a, ds, p, active, lg, lane, r);
}

/* ---- static schedule: ONE contiguous range of batches per warp, runs carried across units ------------
 * A run is "the events of one bin at one point", not "adjacent events": a lane may keep its run open
 * across consecutive units (its events stay sorted), so a warp that owns a contiguous range pays the
 * group prologue and the flush once per (range, group) instead of once per (unit, group), and there is
 * no ticket, no tail of unequal items: every warp holds the same number of batches.  The units of the
 * range stream through the warp's two buffers; the copy of the next unit (of this range, or the first
 * unit of what the warp walks next) is in flight while a unit is walked. */
struct Pipe {
    EventBatch *buf0;               /* the warp's two unit buffers */
    unsigned long long *bars;       /* its two mbarriers */
    int b;                          /* buffer that holds (or will hold) the unit walked next */
    unsigned phase;
};

/* one segment [B0, B1) of dataset d for point group g; (nd, n0, n1): the unit to copy when the last unit of
 * this segment is being walked (n0 < 0: nothing follows) */
template <int S, bool FULL, bool UW>
__device__ __forceinline__ void walk_range(const SpectraArgs &a, int d, int B0, int B1, int g, int lane, Pipe &pp,
                                           int nd, int n0, int n1)
{
    const DatasetDev &ds = a.ds[d];
    int lg = 5;
    bool active = 32 * g + lane < a.P;
    int p = 32 * g + (active ? lane : 0), s = 0;
    if (!FULL) {
        const int np = min(32, a.P - 32 * g);
        lg = np <= 1 ? 0 : 32 - __clz(np - 1);
        const int pl = lane & ((1 << lg) - 1);
        s = lane >> lg;
        active = pl < np;
        p = 32 * g + (active ? pl : 0);
    }
    double h[S];
#pragma unroll
    for (int k = 0; k < S; ++k) h[k] = a.rec[(size_t)k * a.P + p];
    const int row = row_of(a, p);
    const float *thr = a.thr + (size_t)row * a.thr_stride + ds.thr_off;
    const float2 safe = a.safe[(size_t)row * a.n_datasets + d];
    const int B = ds.n_bins, U = a.unit_batches;

    Run<S> r;
#pragma unroll
    for (int k = 0; k < S; ++k) r.C[k] = 0.0;
    r.W = 0.0;
    r.cur = -1;
    r.hi = -pos_inf();
    r.hi2 = pos_inf();

#pragma unroll 1
    for (int off = B0; off < B1; off += U) {
        const int nb = min(U, B1 - off);
        if (lane == 0) {
            /* the other buffer was last read one unit ago (every lane has passed the __syncwarp below) */
            int cd = d, c0 = off + U, c1 = min(off + 2 * U, B1);
            if (c0 >= B1) { cd = nd; c0 = n0; c1 = n1; }
            if (c0 >= 0)
                bulk_load(pp.buf0 + (pp.b ^ 1) * U, a.ds[cd].ev + c0, (unsigned)(c1 - c0) * (unsigned)sizeof(EventBatch),
                          pp.bars + (pp.b ^ 1));
        }
        mbar_wait(pp.bars + pp.b, (pp.phase >> pp.b) & 1u);
        pp.phase ^= 1u << pp.b;
        int my0 = 0, mine = nb;
        if (!FULL) {
            my0 = (nb * s) >> (5 - lg);
            mine = ((nb * (s + 1)) >> (5 - lg)) - my0;
        }
        const EventBatch *bp = pp.buf0 + pp.b * U + my0;
        if (off == B0 && mine > 0) {
            /* open the run at the lane's first event from the load-time hint (see walk_unit) */
            const float v0 = bp->v[0];
            if (v0 >= safe.x && v0 <= safe.y) {
                int bb = max(-1, min(bp->bin0, B));
                float lo = thr_at(thr, B, bb), hi = thr_at(thr, B, bb + 1);
                while (bb >= 0 && v0 < lo) { --bb; hi = lo; lo = thr_at(thr, B, bb); }
                while (bb < B && !(v0 < hi)) { ++bb; hi = thr_at(thr, B, bb + 1); }
                r.cur = bb;
                r.hi = hi;
                r.hi2 = thr_at(thr, B, bb + 2);
            }
        }
        int i = 0;
#pragma unroll 1
        while (i < mine) {
            if (i + 4 <= mine && bp[3].v[EB - 1] < r.hi) {
                walk_inside<S, UW, 4>(bp, h, r);
                i += 4;
                bp += 4;
            } else if (i + 2 <= mine && bp[1].v[EB - 1] < r.hi) {
                walk_inside<S, UW, 2>(bp, h, r);
                i += 2;
                bp += 2;
            } else {
                walk_batch<S>(a, ds, bp, h, thr, safe, p, active, r);
                ++i;
                ++bp;
            }
        }
        __syncwarp();                                   /* this unit's reads are over before its buffer is refilled */
        pp.b ^= 1;
    }
    if (FULL) flush_run<S>(a, ds, p, active, r);
    else      flush_run_substreams<S>(a, ds, p, active, lg, lane, r);
}

/* first (dataset, segment) at or after dataset d0 that the global batch range [G0, G1) touches */
__device__ __forceinline__ bool next_segment(const SpectraArgs &a, long long G0, long long G1, int d0, int &d, int &B0,
                                             int &B1)
{
    long long off = 0;
    for (int i = 0; i < a.n_datasets; ++i) {
        const long long nb = a.ds[i].n_batches;
        if (i >= d0) {
            const long long lo = max(G0, off), hi = min(G1, off + nb);
            if (lo < hi) { d = i; B0 = (int)(lo - off); B1 = (int)(hi - off); return true; }
        }
        off += nb;
    }
    return false;
}

template <int S>
__global__ void __launch_bounds__(WARPS * 32, 4) spectra_static_kernel(const __grid_constant__ SpectraArgs a)
{
    extern __shared__ __align__(128) unsigned char stage[];       /* [WARPS][2][unit_batches] EventBatch */
    __shared__ unsigned long long bars[WARPS][2];
    const int lane = threadIdx.x & 31, wib = threadIdx.x >> 5;
    const long long nW = (long long)gridDim.x * WARPS, w = (long long)blockIdx.x * WARPS + wib;
    const int n_groups = (a.P + 31) >> 5, U = a.unit_batches;
    long long total = 0;
    for (int i = 0; i < a.n_datasets; ++i) total += a.ds[i].n_batches;
    const long long G0 = total * w / nW, G1 = total * (w + 1) / nW;       /* this warp's batches, all datasets */
    Pipe pp;
    pp.buf0 = reinterpret_cast<EventBatch *>(stage) + (size_t)(2 * wib) * U;
    pp.bars = &bars[wib][0];
    pp.b = 0;
    pp.phase = 0u;
    if (lane == 0) {
        mbar_init(&bars[wib][0], 1);
        mbar_init(&bars[wib][1], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncwarp();
    int fd, f0, f1;
    const bool any = next_segment(a, G0, G1, 0, fd, f0, f1);
    if (any && lane == 0)
        bulk_load(pp.buf0, a.ds[fd].ev + f0, (unsigned)(min(f0 + U, f1) - f0) * (unsigned)sizeof(EventBatch), pp.bars);
    asm volatile("griddepcontrol.wait;" ::: "memory");
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    if (!any) return;
#pragma unroll 1
    for (int g = 0; g < n_groups; ++g) {
        int d, B0, B1;
        bool more = next_segment(a, G0, G1, 0, d, B0, B1);
#pragma unroll 1
        while (more) {
            /* what follows this segment: the next dataset's segment, else the first segment again for the
             * next group, else nothing */
            int nd, n0, n1, e1;
            const bool nxt = next_segment(a, G0, G1, d + 1, nd, n0, e1);
            if (!nxt) {
                if (g + 1 < n_groups) { nd = fd; n0 = f0; e1 = f1; } else { nd = 0; n0 = -1; e1 = -1; }
            }
            n1 = n0 < 0 ? -1 : min(n0 + U, e1);
            const DatasetDev &ds = a.ds[d];
            if (32 * g + 16 >= a.P) walk_range<S, false, false>(a, d, B0, B1, g, lane, pp, nd, n0, n1);
            else if (ds.unit_w)    walk_range<S, true, true>(a, d, B0, B1, g, lane, pp, nd, n0, n1);
            else                   walk_range<S, true, false>(a, d, B0, B1, g, lane, pp, nd, n0, n1);
            more = nxt;
            if (nxt) { d = nd; B0 = n0; B1 = e1; }
        }
    }
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

/* item -> (dataset, batches [b0, b1), chunk) */
__device__ __forceinline__ void decode_item(const SpectraArgs &a, unsigned item, int &d, int &b0, int &b1, int &chunk)
{
    const int unit = (int)(item / (unsigned)a.n_chunks);
    chunk = (int)(item - (unsigned)unit * (unsigned)a.n_chunks);
    if (unit >= a.tail_unit) {
        d = a.n_datasets - 1;
        b0 = a.tail_b0 + (unit - a.tail_unit) * a.tail_batches;
        b1 = min(b0 + a.tail_batches, a.ds[d].n_batches);
        return;
    }
    d = 0;
    for (int i = 1; i < a.n_datasets; ++i)
        if (unit >= a.ds[i].unit_begin) d = i;
    b0 = (unit - a.ds[d].unit_begin) * a.unit_batches;
    b1 = min(b0 + a.unit_batches, a.ds[d].n_batches);
}

template <int S>
__global__ void __launch_bounds__(WARPS * 32, 4) spectra_kernel(const __grid_constant__ SpectraArgs a)
{
    static_assert(EB == 4, "the batch loads are written for EB = 4");
    extern __shared__ __align__(128) unsigned char stage[];       /* [WARPS][2][unit_batches] EventBatch */
    __shared__ unsigned long long bars[WARPS][2];
    const int lane = threadIdx.x & 31, wib = threadIdx.x >> 5;
    const unsigned nW = gridDim.x * WARPS;
    const int n_groups = (a.P + 31) >> 5;
    const unsigned n_items = (unsigned)a.n_items;
    EventBatch *const buf0 = reinterpret_cast<EventBatch *>(stage) + (size_t)(2 * wib) * a.unit_batches;
    if (lane == 0) {
        mbar_init(&bars[wib][0], 1);
        mbar_init(&bars[wib][1], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncwarp();
    /* the first two items of a warp are static, later ones come from the counter (which the setup
     * kernel left at 2 nW): warps that meet expensive units (bin edges) simply claim fewer.  The
     * unit of item i + 1 is copied into the warp's other buffer while item i is walked. */
    unsigned cur = blockIdx.x * WARPS + wib, nxt = cur + nW;
    unsigned phase = 0u;                                /* bit b: parity of the next completion of buffer b */
    int b = 0;
    if (cur < n_items && lane == 0) {
        int d, b0, b1, chunk;
        decode_item(a, cur, d, b0, b1, chunk);
        bulk_load(buf0, a.ds[d].ev + b0, (unsigned)(b1 - b0) * (unsigned)sizeof(EventBatch), &bars[wib][0]);
    }
    /* everything above touched only kernel parameters and the event store; the records, thresholds
     * and the work counter come from the setup kernel (no-op unless launched as its dependent) */
    asm volatile("griddepcontrol.wait;" ::: "memory");
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
#pragma unroll 1
    while (cur < n_items) {
        const unsigned ticket = take_ticket(a.counter, lane);
        int d, b0, b1, chunk;
        decode_item(a, cur, d, b0, b1, chunk);
        if (nxt < n_items && lane == 0) {
            /* the other buffer was last read one item ago; every lane has passed the __syncwarp below */
            int nd, nb0, nb1, nc;
            decode_item(a, nxt, nd, nb0, nb1, nc);
            bulk_load(buf0 + (b ^ 1) * a.unit_batches, a.ds[nd].ev + nb0, (unsigned)(nb1 - nb0) * (unsigned)sizeof(EventBatch),
                      &bars[wib][b ^ 1]);
        }
        mbar_wait(&bars[wib][b], (phase >> b) & 1u);
        phase ^= 1u << b;
        const DatasetDev &ds = a.ds[d];
        const int g1 = min((chunk + 1) * a.chunk_groups, n_groups);
#pragma unroll 1
        for (int g = chunk * a.chunk_groups; g < g1; ++g) {
            const EventBatch *unit = buf0 + b * a.unit_batches;
            if (32 * g + 16 >= a.P) walk_unit<S, false, false>(a, ds, d, unit, b1 - b0, g, lane);
            else if (ds.unit_w)    walk_unit<S, true, true>(a, ds, d, unit, b1 - b0, g, lane);
            else                   walk_unit<S, true, false>(a, ds, d, unit, b1 - b0, g, lane);
        }
        cur = nxt;
        nxt = __shfl_sync(0xffffffffu, ticket, 0);      /* also orders this item's reads before the next copy */
        b ^= 1;
    }
}

/* dynamic shared memory of one CTA: two unit buffers per warp, sized for the largest unit */
constexpr size_t STAGE_BYTES = (size_t)WARPS * 2 * MAX_UNIT_BATCHES * sizeof(EventBatch);

template <int S> cudaError_t launch_t(const SpectraArgs &a, cudaStream_t st, bool pdl)
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
    if (a.sched == 1) return cudaLaunchKernelEx(&cfg, spectra_static_kernel<S>, a);
    return cudaLaunchKernelEx(&cfg, spectra_kernel<S>, a);
}

template <int S> cudaError_t max_warps_t(int sm_count, int *warps)
{
    int per_sm = 0;
    cudaError_t e = cudaFuncSetAttribute(spectra_kernel<S>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                         (int)STAGE_BYTES);
    if (e != cudaSuccess) return e;
    e = cudaFuncSetAttribute(spectra_static_kernel<S>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)STAGE_BYTES);
    if (e != cudaSuccess) return e;
    e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, spectra_kernel<S>, WARPS * 32, STAGE_BYTES);
    if (e != cudaSuccess) return e;
    if (per_sm < 1) return cudaErrorLaunchOutOfResources;
    *warps = sm_count * per_sm * WARPS;
    return cudaSuccess;
}

} // namespace

cudaError_t spectra_max_warps(int S, int sm_count, int *warps)
{
    return S == 2 ? max_warps_t<2>(sm_count, warps) : max_warps_t<3>(sm_count, warps);
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
cudaError_t launch_spectra(const SpectraArgs &a, int S, cudaStream_t st, bool pdl)
{
    if (a.n_items <= 0 || a.P <= 0 || a.n_warps < WARPS) return cudaSuccess;
    return S == 2 ? launch_t<2>(a, st, pdl) : launch_t<3>(a, st, pdl);
}

/* ---- diagnostic: bin index of every event at every point (bit-exact parity of row a3) ----
 * Reads the threshold rows the setup kernel wrote and assigns bins with the same locate_bin() as
 * the hot kernel, so the test covers the production binning. */
namespace {
__global__ void __launch_bounds__(256) event_bins_kernel(const __grid_constant__ SpectraArgs a, int d,
                                                         const int32_t *perm, long long n, long long ev_off,
                                                         long long total_events, int32_t *bins)
{
    const DatasetDev &ds = a.ds[d];
    const int p = blockIdx.y;
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const int row = row_of(a, p);
    float hi;
    int b = locate_bin(ds, a.thr + (size_t)row * a.thr_stride + ds.thr_off, a.safe[(size_t)row * a.n_datasets + d],
                       theta_of(a, p), ds.ev[i / EB].v[i % EB], hi);
    bins[(size_t)p * total_events + ev_off + perm[i]] = (b >= 0 && b < ds.n_bins) ? b : -1;
}
} // namespace

cudaError_t launch_event_bins(const SpectraArgs &a, int d, const int32_t *perm, long long n, long long ev_off,
                              long long total_events, int32_t *bins, cudaStream_t st)
{
    if (n <= 0 || a.P <= 0) return cudaSuccess;
    dim3 grid((unsigned)((n + 255) / 256), a.P);
    event_bins_kernel<<<grid, 256, 0, st>>>(a, d, perm, n, ev_off, total_events, bins);
    return cudaGetLastError();
}

} // namespace phylino
