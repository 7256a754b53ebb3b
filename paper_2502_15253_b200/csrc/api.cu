/*
 * api.cu -- the C-ABI of include/phylino.h: context, model tables, event store, launches.
 * Host logic only; the arithmetic of the path lives in spectra.cu / finalize.cu.
 */
#include <algorithm>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <new>
#include <numeric>
#include <vector>

#include "internal.h"

using namespace phylino;

namespace {

struct DeviceGuard {
    int prev = -1;
    bool ok = true;
    explicit DeviceGuard(int dev)
    {
        if (cudaGetDevice(&prev) != cudaSuccess) { prev = -1; ok = false; return; }
        if (prev != dev && cudaSetDevice(dev) != cudaSuccess) ok = false;
    }
    ~DeviceGuard() { if (prev >= 0) cudaSetDevice(prev); }
};

phylino_status fail(phylino_ctx *c, phylino_status s, const char *fmt, ...)
{
    char buf[512];
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(buf, sizeof buf, fmt, ap);
    va_end(ap);
    if (c) c->err = buf;
    return s;
}

phylino_status cuda_fail(phylino_ctx *c, cudaError_t e, const char *what)
{
    cudaGetLastError();     /* clear the sticky-less error state */
    return fail(c, e == cudaErrorMemoryAllocation ? PHYLINO_ERR_OOM : PHYLINO_ERR_CUDA, "%s: %s", what,
                cudaGetErrorString(e));
}

#define CU(call)                                                    \
    do {                                                            \
        cudaError_t e_ = (call);                                    \
        if (e_ != cudaSuccess) return cuda_fail(ctx, e_, #call);    \
    } while (0)

template <class T> cudaError_t upload(T **dst, const std::vector<T> &src, cudaStream_t st)
{
    *dst = nullptr;
    size_t n = std::max<size_t>(src.size(), 1);
    cudaError_t e = cudaMalloc((void **)dst, n * sizeof(T));
    if (e != cudaSuccess) return e;
    if (!src.empty()) e = cudaMemcpyAsync(*dst, src.data(), src.size() * sizeof(T), cudaMemcpyHostToDevice, st);
    return e;
}

void free_events(phylino_dataset_host &d)
{
    cudaFree(d.d_ev); cudaFree(d.d_edges); cudaFree(d.d_perm); cudaFree(d.d_hint);
    d.d_ev = nullptr; d.d_edges = nullptr; d.d_perm = nullptr; d.d_hint = nullptr;
    d.loaded = false; d.n = d.n_pad = 0;
}

void free_tables(phylino_ctx *c)
{
    FinalizeArgs &f = c->fin;
    cudaFree((void *)f.bin_ds); cudaFree((void *)f.idx_flux); cudaFree((void *)f.inv_scale);
    cudaFree((void *)f.norm); cudaFree((void *)f.idx_signorm); cudaFree((void *)f.n_bkg);
    cudaFree((void *)f.idx_rate); cudaFree((void *)f.idx_shape); cudaFree((void *)f.tmpl);
    cudaFree((void *)f.prior_mean); cudaFree((void *)f.prior_sigma);
    cudaFree((void *)f.blk_off); cudaFree((void *)f.blk_moff); cudaFree((void *)f.blk_idx);
    cudaFree((void *)f.blk_mean); cudaFree((void *)f.blk_inv);
    cudaFree((void *)f.edges_all); cudaFree((void *)f.ds_bin_off); cudaFree((void *)f.ds_idx_a);
    cudaFree((void *)f.fm_off); cudaFree((void *)f.fm_idx); cudaFree((void *)f.fm_grid);
    cudaFree((void *)f.fn_offset); cudaFree((void *)f.fn_term_off); cudaFree((void *)f.term_coef);
    cudaFree((void *)f.term_fac_off); cudaFree((void *)f.fac_idx); cudaFree((void *)f.fac_pow);
    f = FinalizeArgs{};
    c->max_block_idx = -1;
}

void free_transform(phylino_ctx *c)
{
    TransformArgs &t = c->tf;
    cudaFree((void *)t.copy_src); cudaFree((void *)t.copy_const); cudaFree((void *)t.row_off);
    cudaFree((void *)t.col_off); cudaFree((void *)t.mat_off); cudaFree((void *)t.idx_out);
    cudaFree((void *)t.idx_in); cudaFree((void *)t.offset); cudaFree((void *)t.centre); cudaFree((void *)t.matrix);
    t = TransformArgs{};
    c->have_tf = false;
    c->n_u = 0;
}

void free_all(phylino_ctx *c)
{
    for (auto &d : c->ds) free_events(d);
    c->ds.clear();
    free_tables(c);
    cudaFree(c->d_acc); cudaFree(c->d_flags);
    c->d_acc = nullptr; c->d_flags = nullptr; c->acc_capacity = 0;
    cudaFree(c->d_rec); cudaFree(c->d_thr); cudaFree(c->d_safe); cudaFree(c->d_counter); cudaFree(c->d_done); cudaFree(c->d_med); cudaFree(c->d_grad_plan); cudaFree(c->d_unit_order);
    cudaFree(c->d_small);
    c->d_rec = nullptr; c->d_thr = nullptr; c->d_safe = nullptr; c->d_counter = nullptr; c->d_done = nullptr; c->d_med = nullptr; c->d_grad_plan = nullptr; c->grad_plan_state = 0; c->d_unit_order = nullptr; c->order_U = c->order_units = 0;
    c->d_small = nullptr;
    c->point_capacity = 0;
    cudaFree(c->d_plan); c->d_plan = nullptr; c->plan_capacity = 0;
    cudaFree(c->d_mu); c->d_mu = nullptr; c->mu_capacity = 0;
    cudaFree(c->d_work); c->d_work = nullptr; c->work_capacity = 0;
    free_transform(c);
    cudaFree(c->d_theta); c->d_theta = nullptr; c->theta_capacity = 0;
    cudaFree(c->d_stage); c->d_stage = nullptr;
    if (c->h_pin) cudaFreeHost(c->h_pin);
    c->h_pin = nullptr; c->stage_capacity = 0;
    c->resident_warps = c->fused_warps = 0;     /* occupancy of the kernels of the model's n_terms: asked again */
    c->fused_tables = 0;
    c->fused_cache.clear();
    c->have_model = false;
}

void free_events_timing(phylino_ctx *c)
{
    for (auto &e : c->ev) { if (e) cudaEventDestroy(e); e = nullptr; }
    c->timing = false;
}

bool idx_ok(int32_t i, int32_t n) { return i >= -1 && i < n; }

phylino_status check_ready(phylino_ctx *ctx, int P, const void *params, const void *out)
{
    if (!ctx) return PHYLINO_ERR_ARG;
    if (!ctx->have_model) return fail(ctx, PHYLINO_ERR_STATE, "phylino_set_model has not been called");
    for (int d = 0; d < ctx->n_datasets; ++d)
        if (!ctx->ds[d].loaded) return fail(ctx, PHYLINO_ERR_STATE, "dataset %d has no events loaded", d);
    if (P < 0) return fail(ctx, PHYLINO_ERR_SHAPE, "P = %d is negative", P);
    if ((int64_t)P * ctx->total_bins > (int64_t)1 << 40) return fail(ctx, PHYLINO_ERR_SHAPE, "P x total_bins too large");
    if (P > 0 && (!params || !out)) return fail(ctx, PHYLINO_ERR_ARG, "NULL params or output pointer");
    return PHYLINO_OK;
}

phylino_status ensure_acc(phylino_ctx *ctx, int P)
{
    int64_t need = (int64_t)P * ctx->total_bins;
    if (need > ctx->acc_capacity) {
        /* the stream may still use the old buffers */
        CU(cudaStreamSynchronize(ctx->stream));
        cudaFree(ctx->d_acc); cudaFree(ctx->d_flags);
        ctx->d_acc = nullptr; ctx->d_flags = nullptr; ctx->acc_capacity = 0;
        CU(cudaMalloc((void **)&ctx->d_acc, need * sizeof(long long)));
        CU(cudaMalloc((void **)&ctx->d_flags, need * sizeof(unsigned)));
        CU(cudaMemsetAsync(ctx->d_acc, 0, need * sizeof(long long), ctx->stream));
        CU(cudaMemsetAsync(ctx->d_flags, 0, need * sizeof(unsigned), ctx->stream));
        ctx->acc_capacity = need;
    }
    if (!ctx->d_counter) {
        CU(cudaMalloc((void **)&ctx->d_counter, sizeof(unsigned)));
        CU(cudaMemsetAsync(ctx->d_counter, 0, sizeof(unsigned), ctx->stream));
    }
    if (!ctx->d_done) {
        CU(cudaMalloc((void **)&ctx->d_done, sizeof(unsigned)));
        CU(cudaMemsetAsync(ctx->d_done, 0, sizeof(unsigned), ctx->stream));
    }
    if (!ctx->d_med) {
        CU(cudaMalloc((void **)&ctx->d_med, sizeof(unsigned long long)));
        CU(cudaMemsetAsync(ctx->d_med, 0, sizeof(unsigned long long), ctx->stream));
    }
    if (P > ctx->point_capacity) {
        /* per-point records and threshold rows written by the setup kernel of every call */
        CU(cudaStreamSynchronize(ctx->stream));
        cudaFree(ctx->d_rec); cudaFree(ctx->d_thr); cudaFree(ctx->d_safe); cudaFree(ctx->d_small);
        ctx->d_rec = nullptr; ctx->d_thr = nullptr; ctx->d_safe = nullptr; ctx->d_small = nullptr; ctx->point_capacity = 0;
        const int64_t rows = ctx->per_point_binning ? P : 1;      /* (sized for mode 0 even while mode 1 is on) */
        CU(cudaMalloc((void **)&ctx->d_rec, (size_t)rec_fields(ctx->n_terms) * P * sizeof(double)));
        CU(cudaMalloc((void **)&ctx->d_thr, (size_t)rows * (ctx->total_bins + ctx->n_datasets) * sizeof(float)));
        CU(cudaMalloc((void **)&ctx->d_safe, (size_t)rows * ctx->n_datasets * sizeof(float2)));
        CU(cudaMalloc((void **)&ctx->d_small, (size_t)((P + 31) / 32 + 4) * ctx->n_datasets));
        ctx->point_capacity = P;
    }
    return PHYLINO_OK;
}

/* fill the by-value kernel arguments that do not depend on the batch */
void fill_datasets(const phylino_ctx *ctx, SpectraArgs &a)
{
    for (int d = 0; d < ctx->n_datasets; ++d) {
        const phylino_dataset_host &h = ctx->ds[d];
        DatasetDev &v = a.ds[d];
        v.ev = h.d_ev; v.edges = h.d_edges; v.hint = h.d_hint; v.perm = h.d_perm;
        v.ev_off = d == 0 ? 0 : a.ds[d - 1].ev_off + a.ds[d - 1].n_events;
        v.n_events = (int32_t)h.n;
        v.n_bins = h.n_bins;
        v.bin_off = d == 0 ? 0 : a.ds[d - 1].bin_off + a.ds[d - 1].n_bins;
        v.thr_off = v.bin_off + d;
        /* bin-level energy correction (phylino_set_energy_correction_mode): the events are binned under the
         * identity scale, the finalize stage corrects the bins */
        v.per_point = (!ctx->ec_mode && (h.idx_a[0] >= 0 || h.idx_a[1] >= 0 || h.idx_a[2] >= 0)) ? 1 : 0;
        v.n_batches = (int32_t)(h.n_pad / EB);
        for (int j = 0; j < 3; ++j) v.idx_a[j] = ctx->ec_mode ? -1 : h.idx_a[j];
        v.unit_w = h.unit_w ? 1 : 0;
        v.v_pos_min = h.v_pos_min;
        v.v_max = h.v_max;
        v.fx_scale = std::ldexp(1.0, h.fx_exp);
        v.x_max = h.x_max;
    }
    a.osc.osc_model = ctx->osc_model;
    a.osc.ordering = ctx->ordering_override ? ctx->ordering_override : ctx->ordering;
    for (int j = 0; j < 6; ++j) { a.osc.idx_osc[j] = ctx->idx_osc[j]; a.osc.fixed_osc[j] = ctx->fixed_osc[j]; }
    a.n_datasets = ctx->n_datasets;
    a.n_params = ctx->n_params;
    a.total_bins = ctx->total_bins;
    a.thr_stride = ctx->total_bins + ctx->n_datasets;
    a.rec = ctx->d_rec;
    a.thr = ctx->d_thr;
    a.safe = ctx->d_safe;
    a.small = ctx->d_small;
    a.acc = ctx->d_acc;
    a.flags = ctx->d_flags;
    a.counter = ctx->d_counter;
    a.done = ctx->d_done;
    a.med_count = ctx->d_med;
}

/* Cut of the batch into work items (spectra.cu): U batches per unit, G point groups per item.
 * Aim: at least 12 items per resident warp (dynamic balance, short tail) of at least 16 batch-groups
 * each (the per-item cost -- first bin search, one flush per point -- stays a few percent). */
/* small batches (the minimiser's single evaluations) are bound by launch latency and HBM bytes, not by
 * arithmetic: they take ONE launch of the single-launch kernel (spectra.cu, spectra_fused_kernel).  Measured in
 * round 1 with the then separate static-range kernel on 6e6 events: 1 / 4 / 16 points 0.098 / 0.123 / 0.204 ms
 * (tickets) -> 0.062 / 0.082 / 0.178 ms (two-term models); on config 4's store (three terms, 410 bins) 1 / 2 points
 * 0.142 / 0.143 -> 0.084 / 0.114 ms, even at 4, slower from 8.  Larger batches are faster with the tickets
 * (config 2: 0.21 ms against 0.29 ms static). */
/* Order in which the single-launch kernel hands out its units: those nearest a bin edge FIRST, those in the middle of
 * a bin last.  A call for a few points is as long as its slowest warp, and a warp that meets a bin edge is 1-2.5 us
 * late (the event-by-event path through cold instruction lines; round-2 timeline: median warp done at 20 us, the last
 * at 27-30 us, all of the late ones had met an edge).  Met early, the delay is absorbed by the tickets -- a late warp
 * claims fewer units; met in a warp's last unit, it is the end of the call.  "Nearest" under the identity energy scale,
 * in units of the local bin width: the real edges move with the energy-scale parameters, by far less than half a bin.
 * The order changes no result (the accumulators are integers).  One table per (store, unit length), built at the
 * first small-batch call and kept on the device. */
phylino_status build_unit_order(phylino_ctx *ctx, int64_t U, int64_t units)
{
    std::vector<std::pair<float, int32_t>> key;
    key.reserve((size_t)units);
    int32_t unit = 0;
    for (int d = 0; d < ctx->n_datasets; ++d) {
        const phylino_dataset_host &h = ctx->ds[d];
        const int64_t nb = h.n_pad / EB;
        const int B = h.n_bins;
        const int64_t n_blk = (int64_t)h.v_blk.size();
        for (int64_t b0 = 0; b0 < nb; b0 += U, ++unit) {
            const int64_t b1 = std::min(b0 + U, nb);
            /* [va, vb] contains every E_vis of the unit: first event of the block b0 falls in, first event of the first
             * block at or after b1 (the store is sorted; the largest value of the dataset past the last block) */
            const float va = h.v_blk[(size_t)(b0 / HINT_BATCHES)];
            const int64_t kb = (b1 + HINT_BATCHES - 1) / HINT_BATCHES;
            float vb = kb < n_blk ? h.v_blk[(size_t)kb] : h.v_max;
            if (!(vb == vb)) vb = h.v_max;              /* a block of padding / NaN events */
            float dist = 1.0e30f;                       /* no finite event: never at an edge */
            if (va == va && vb == vb) {
                const double *e = h.edges.data();
                const int i = (int)(std::upper_bound(e, e + B + 1, (double)va) - e) - 1;     /* -1 ... B */
                if (i < 0)       dist = (float)((e[0] - (double)vb) / (e[1] - e[0]));
                else if (i >= B) dist = (float)(((double)va - e[B]) / (e[B] - e[B - 1]));
                else             dist = (float)(std::min((double)va - e[i], e[i + 1] - (double)vb) / (e[i + 1] - e[i]));
                if (!(dist > 0.0f)) dist = 0.0f;        /* an edge inside the unit */
            }
            key.emplace_back(dist, unit);
        }
    }
    if ((int64_t)key.size() != units) return fail(ctx, PHYLINO_ERR_STATE, "unit order: %lld units expected, %lld found", (long long)units, (long long)key.size());
    std::stable_sort(key.begin(), key.end(), [](const std::pair<float, int32_t> &x, const std::pair<float, int32_t> &y) { return x.first < y.first; });
    std::vector<int32_t> order((size_t)units);
    for (int64_t i = 0; i < units; ++i) order[(size_t)i] = key[(size_t)i].second;
    CU(cudaStreamSynchronize(ctx->stream));             /* a launch in flight may still read the old table */
    cudaFree(ctx->d_unit_order);
    ctx->d_unit_order = nullptr;
    ctx->order_U = ctx->order_units = 0;
    CU(cudaMalloc((void **)&ctx->d_unit_order, (size_t)std::max<int64_t>(units, 1) * sizeof(int32_t)));
    CU(cudaMemcpy(ctx->d_unit_order, order.data(), (size_t)units * sizeof(int32_t), cudaMemcpyHostToDevice));
    ctx->order_U = U;
    ctx->order_units = units;
    return PHYLINO_OK;
}

bool wants_single_launch(const phylino_ctx *ctx, int P)
{
    if (ctx->schedule == 1) return false;
    if (ctx->schedule == 2) return P <= FUSED_MAX_POINTS;
    return P <= (ctx->n_terms == 2 ? FUSED_MAX_POINTS : 4);
}

phylino_status fill_batch(phylino_ctx *ctx, SpectraArgs &a, int P, const double *params, int thr_rows = 0)
{
    if (ctx->resident_warps == 0)
        CU(spectra_max_warps(ctx->n_terms, ctx->sm_count, false, 0, &ctx->resident_warps));
    a.P = P;
    a.params = params;
    a.thr_rows = thr_rows > 0 ? thr_rows : (ctx->per_point_binning && !ctx->ec_mode ? P : 1);
    const int64_t n_groups = (P + 31) / 32;
    int streams = 1;                                    /* sub-streams per warp when P < 32 */
    if (P < 32) { int pl = 1; while (pl < P) pl <<= 1; streams = 32 / pl; }
    int64_t batches = 0;
    bool all_slim = true;
    for (int d = 0; d < ctx->n_datasets; ++d) {
        batches += ctx->ds[d].n_pad / EB;
        all_slim = all_slim && (ctx->ds[d].unit_w || ctx->ds[d].n_pad == 0);
    }
    const int last = ctx->n_datasets - 1;
    const int64_t nb_last = ctx->ds[last].n_pad / EB;

    a.sched = 0;
    if (wants_single_launch(ctx, P)) {
        const size_t tables = fused_table_bytes(ctx->n_terms, P, a.thr_rows, a.thr_stride, ctx->n_datasets);
        if (fused_fits(tables)) {
            /* one occupancy query per distinct table size (the size depends on P): a minimiser that alternates
             * single evaluations with small line-search batches finds both in the list */
            int found = 0;
            for (const auto &kv : ctx->fused_cache) if (kv.first == tables) { found = kv.second; break; }
            if (found == 0) {
                CU(spectra_max_warps(ctx->n_terms, ctx->sm_count, true, tables, &found));
                ctx->fused_cache.emplace_back(tables, found);
            }
            ctx->fused_warps = found;
            ctx->fused_tables = tables;
            a.sched = 1;
        }
    }
    if (a.sched == 1) {
        /* single launch: bound by the event bytes over HBM, so units as long as a staging buffer holds (6 KB: 128
         * slim or 64 weighted batches), shorter only where the store is too small to give every SM a few of them */
        /* the finalize CTAs (one per point) must find room beside the persistent grid to work ahead */
        int fcap = std::max(ctx->fused_warps - WARPS * P, WARPS);
        if (ctx->max_warps > 0) fcap = std::max(WARPS, std::min(fcap, ctx->max_warps / WARPS * WARPS));
        int64_t U = STAGE_BUF_BYTES / (int64_t)(all_slim ? sizeof(EventBatchU) : sizeof(EventBatchW));
        while (U > 32 && (batches + U - 1) / U < 4ll * ctx->sm_count) U /= 2;
        if (ctx->unit_events > 0)
            U = std::max<int64_t>(1, std::min<int64_t>(ctx->unit_events / EB, STAGE_BUF_BYTES / (int64_t)sizeof(EventBatchW)));
        U = std::max<int64_t>(U, streams);              /* every sub-stream of a unit holds a batch */
        int64_t units = 0;
        for (int d = 0; d < ctx->n_datasets; ++d) {
            a.ds[d].unit_begin = (int32_t)units;
            units += (ctx->ds[d].n_pad / EB + U - 1) / U;
        }
        a.tail_unit = (int32_t)units;                   /* no fine tail */
        a.tail_b0 = (int32_t)nb_last;
        a.tail_batches = (int32_t)U;
        a.unit_batches = (int32_t)U;
        a.chunk_groups = 1;
        a.n_units = (int32_t)units;
        a.n_chunks = 1;
        a.n_items = (int32_t)units;
        a.n_warps = (int32_t)std::max<int64_t>(WARPS, std::min<int64_t>(fcap, (units + WARPS - 1) / WARPS * WARPS));
        /* edge-first order of the units -- where there are tickets at all: with at most two units per warp every
         * unit is a static first item, the order buys nothing and its look-up sits in front of the first copy */
        a.unit_order = nullptr;
        if (units > 2ll * a.n_warps) {
            if (!ctx->d_unit_order || ctx->order_U != U || ctx->order_units != units) {
                const phylino_status so = build_unit_order(ctx, U, units);
                if (so != PHYLINO_OK) return so;
            }
            a.unit_order = ctx->d_unit_order;
        }
        return PHYLINO_OK;
    }

    /* Cut of the batch into work items (spectra.cu): U batches per unit, G point groups per item.
     * Aim: at least 6 items per resident warp (dynamic balance; the fine tail below evens out the end) of at least
     * 16 batch-groups each, units as long as the staging buffer allows: an item costs about 500 instructions that
     * the hot loop keeps evicting from the instruction cache (ticket, decode, opening and flushing the run),
     * against 300 per 16 events x 32 points of work -- round 2, ncu source view of config 2: 22 % of all warp
     * instructions with units of 32 batches.  Measured (unit batches x groups per item): config 2 32 x 1 7.3e11,
     * 64 x 1 7.7e11, 128 x 1 6.8e11 event x point/s; config 3 64 x 2 0.997e12, 128 x 1 1.014e12; config 5 64 x 2
     * 6.21e11, 128 x 2 6.27e11, 128 x 1 6.25e11. */
    int cap = std::max(ctx->resident_warps, WARPS);
    if (ctx->max_warps > 0) cap = std::max(WARPS, std::min(cap, ctx->max_warps / WARPS * WARPS));
    const int64_t work = std::max<int64_t>(1, batches * n_groups / (6ll * cap));
    /* a unit must fit the warp's staging buffer: 64 weighted or 128 unit-weight batches */
    const int64_t u_max = STAGE_BUF_BYTES / (int64_t)(all_slim ? sizeof(EventBatchU) : sizeof(EventBatchW));
    int64_t U = 16;
    while (U < u_max && U * 2 <= work) U *= 2;
    U = std::max<int64_t>(U, 4 * streams);
    if (ctx->unit_events > 0) U = std::max(1, ctx->unit_events / EB);
    U = std::min<int64_t>(U, u_max);
    /* point groups per item: one once the units are long; chunks of equal size */
    int64_t G = std::max<int64_t>(1, std::min<int64_t>(std::min<int64_t>(work, 128) / U, n_groups));
    G = (n_groups + (n_groups + G - 1) / G - 1) / ((n_groups + G - 1) / G);
    if (ctx->chunk_groups > 0) G = std::min<int64_t>(ctx->chunk_groups, n_groups);
    int64_t units, chunks, tail_unit, tail_b0, Us;
    for (;;) {
        chunks = (n_groups + G - 1) / G;
        /* fine tail: about the last 1.5 items of every warp's share, at most a quarter of the work and
         * never more than the last dataset, in units of U/4 */
        const int64_t per_warp = std::max<int64_t>(1, (batches + U - 1) / U * chunks / cap);
        int64_t fine = std::min<int64_t>(batches / 4, batches * 3 / (2 * per_warp));
        fine = std::min(fine, nb_last);
        Us = std::max<int64_t>(std::max<int64_t>(4, streams), U / 4);
        if (Us >= U || fine < 2 * U) fine = 0;
        tail_b0 = (nb_last - fine) / U * U;
        if (fine == 0) tail_b0 = nb_last;
        units = 0;
        for (int d = 0; d < ctx->n_datasets; ++d) {
            a.ds[d].unit_begin = (int32_t)units;
            const int64_t nb = d == last ? tail_b0 : ctx->ds[d].n_pad / EB;
            units += (nb + U - 1) / U;
        }
        tail_unit = units;
        units += (nb_last - tail_b0 + Us - 1) / Us;
        if (units * chunks < (1ll << 31) - 2ll * cap) break;
        if (G < n_groups) G *= 2; else U *= 2;          /* keep items and tickets inside 32 bits */
    }
    a.tail_unit = (int32_t)tail_unit;
    a.tail_b0 = (int32_t)tail_b0;
    a.tail_batches = (int32_t)Us;
    a.unit_batches = (int32_t)U;
    a.chunk_groups = (int32_t)G;
    a.n_units = (int32_t)units;
    a.n_chunks = (int32_t)chunks;
    a.n_items = (int32_t)(units * chunks);
    const int64_t warps = std::min<int64_t>(cap, (a.n_items + WARPS - 1) / WARPS * WARPS);
    a.n_warps = (int32_t)std::max<int64_t>(warps, WARPS);
    return PHYLINO_OK;
}

/* enqueue rows a1-a7 for P points: one launch of the single-launch kernel for small batches, else the
 * setup, spectra (tickets) and finalize kernels.  mode: 0 spectra H -> hist, 1 expectation mu -> hist, 2 NLL -> nll;
 * bins != NULL: the diagnostic instantiation (bin of every event), accumulators cleared, no other output. */
phylino_status enqueue_eval(phylino_ctx *ctx, int P, const double *params, const double *data, double *hist,
                            double *nll, int mode, int32_t *bins = nullptr, const double *host_copy = nullptr)
{
    SpectraArgs a{};
    fill_datasets(ctx, a);
    phylino_status s = fill_batch(ctx, a, P, params);
    if (s != PHYLINO_OK) return s;
    const bool dbg = bins != nullptr;
    ctx->last_points = P;
    ctx->last_fused = a.sched == 1;
    a.dbg_bins = bins;
    a.total_events = phylino_total_events(ctx);
    FinalizeArgs f = ctx->fin;
    f.P = P;
    f.params = params;
    f.acc = ctx->d_acc;
    f.flags = ctx->d_flags;
    f.data = data;
    f.hist = hist;
    f.nll = nll;
    f.ec_mode = ctx->ec_mode;
    if (dbg) mode = 3;
    const bool pdl = !ctx->timing;
    if (ctx->timing) { CU(cudaEventRecord(ctx->ev[0], ctx->stream)); }
    if (a.sched == 1) {
        /* small batch: setup fused into the spectra kernel, the finalize kernel (its programmatic dependent, one
         * CTA per point) does its table work while the events are walked and zeroes the work counter */
        if (ctx->timing) CU(cudaEventRecord(ctx->ev[1], ctx->stream));
        /* host_copy: the same batch in host memory, small enough to ride with the kernel arguments -- the walk then
         * never touches `params` (which may be the device alias of pinned host memory: only the few finalize CTAs
         * read it, in their prologue) */
        ParamBlob &blob = ctx->blob;                    /* contents matter only when a.params == NULL */
        if (host_copy && (int64_t)P * ctx->n_params <= PARAM_BLOB_DOUBLES) {
            std::memcpy(blob.v, host_copy, (size_t)P * ctx->n_params * sizeof(double));
            a.params = nullptr;
        }
        CU(launch_fused(a, blob, ctx->n_terms, ctx->stream, pdl, dbg));
        ctx->launches += 1;
        if (ctx->timing) CU(cudaEventRecord(ctx->ev[2], ctx->stream));
        f.reset_counter = ctx->d_done;
        CU(launch_finalize(f, mode, ctx->stream, pdl));
        ctx->launches += 1;
        if (ctx->timing) CU(cudaEventRecord(ctx->ev[3], ctx->stream));
        return PHYLINO_OK;
    }
    if (a.n_items > 0 && P > 0) {
        CU(launch_setup(a, ctx->n_terms, ctx->stream));
        ctx->launches += 1;
    }
    if (ctx->timing) CU(cudaEventRecord(ctx->ev[1], ctx->stream));
    if (a.n_items > 0 && P > 0) {
        CU(launch_spectra(a, ctx->n_terms, ctx->stream, pdl, dbg));
        ctx->launches += 1;
    }
    if (ctx->timing) CU(cudaEventRecord(ctx->ev[2], ctx->stream));
    /* the finalize prologue reads params and data BEFORE its griddepcontrol.wait, which is safe only behind a spectra
     * kernel of this call (that kernel waited for its own predecessor before releasing dependents).  With nothing to
     * walk (every dataset empty) no such kernel was launched: the finalize kernel then follows the caller's
     * producer of params / data directly and must be an ordinary, fully ordered launch. */
    CU(launch_finalize(f, mode, ctx->stream, pdl && a.n_items > 0 && P > 0));
    ctx->launches += 1;
    if (ctx->timing) CU(cudaEventRecord(ctx->ev[3], ctx->stream));
    return PHYLINO_OK;
}

phylino_status ensure_stage(phylino_ctx *ctx, int64_t doubles)
{
    if (doubles <= ctx->stage_capacity) return PHYLINO_OK;
    CU(cudaStreamSynchronize(ctx->stream));
    cudaFree(ctx->d_stage); ctx->d_stage = nullptr;
    if (ctx->h_pin) cudaFreeHost(ctx->h_pin);
    ctx->h_pin = nullptr; ctx->stage_capacity = 0;
    CU(cudaMalloc((void **)&ctx->d_stage, doubles * sizeof(double)));
    CU(cudaHostAlloc((void **)&ctx->h_pin, doubles * sizeof(double), cudaHostAllocMapped));
    CU(cudaHostGetDevicePointer((void **)&ctx->d_pin, ctx->h_pin, 0));      /* the kernels' view of the pinned block */
    ctx->stage_capacity = doubles;
    return PHYLINO_OK;
}

/* width of one row of the caller's parameter batch: the minimiser's vector if a transformation layer is set */
int64_t param_width(const phylino_ctx *ctx) { return ctx->have_tf ? ctx->n_u : ctx->n_params; }

/* the transformation layer on the host: the same fma sequence as transform.cu */
void host_transform(const phylino_ctx *ctx, int P, const double *u, double *theta)
{
    const int NP = ctx->n_params, NU = ctx->n_u;
    const int n_blocks = (int)ctx->tf_mat_off.size();
    for (int p = 0; p < P; ++p) {
        const double *up = u + (size_t)p * NU;
        double *tp = theta + (size_t)p * NP;
        for (int j = 0; j < NP; ++j) tp[j] = ctx->tf_src[j] >= 0 ? up[ctx->tf_src[j]] : ctx->tf_const[j];
        for (int k = 0; k < n_blocks; ++k) {
            const int ro = ctx->tf_row_off[k], n_out = ctx->tf_row_off[k + 1] - ro;
            const int co = ctx->tf_col_off[k], n_in = ctx->tf_col_off[k + 1] - co;
            const double *M = ctx->tf_matrix.data() + ctx->tf_mat_off[k];
            for (int i = 0; i < n_out; ++i) {
                double acc = ctx->tf_offset[ro + i];
                for (int j = 0; j < n_in; ++j)
                    acc = std::fma(M[(size_t)i * n_in + j], up[ctx->tf_idx_in[co + j]] - ctx->tf_centre[co + j], acc);
                tp[ctx->tf_idx_out[ro + i]] = acc;
            }
        }
    }
}

/* DEVICE batch of a device entry point -> model parameters: the caller's pointer, or the transformed copy */
phylino_status resolve_params(phylino_ctx *ctx, int P, const double *params, const double **theta)
{
    *theta = params;
    if (!ctx->have_tf || P == 0) return PHYLINO_OK;
    const int64_t need = (int64_t)P * ctx->n_params;
    if (need > ctx->theta_capacity) {
        CU(cudaStreamSynchronize(ctx->stream));
        cudaFree(ctx->d_theta); ctx->d_theta = nullptr; ctx->theta_capacity = 0;
        CU(cudaMalloc((void **)&ctx->d_theta, need * sizeof(double)));
        ctx->theta_capacity = need;
    }
    TransformArgs t = ctx->tf;
    t.P = P; t.u = params; t.theta = ctx->d_theta;
    CU(launch_transform(t, ctx->stream));
    ctx->launches += 1;
    *theta = ctx->d_theta;
    return PHYLINO_OK;
}

/* ---- cross-point caching ("costly recalculations are only
 * triggered upon relevant parameter changes") ---------------------------------------------------
 * For a fixed energy scale and fixed mass splittings the histogram is affine in the amplitudes:
 *   H[p,b] = P0(p) W[b] + sum_k A_k(p) C_k[b],  W[b] = sum_e w_e,  C_k[b] = sum_e w_e g(h_k x_e),
 * so a batch needs one W per distinct energy-scale tuple ("class") and one C per distinct
 * (class, splitting).  The plan groups the caller's points by the BIT PATTERNS of the parameters
 * these depend on (never by value tolerance), packs the distinct (class, splitting) pairs S at a
 * time into virtual points for the spectra kernel, and tells the finalize kernel which cells each
 * real point combines.  A 603-point central-difference batch of config 3 becomes 21 virtual
 * points, the 4096-point grid of config 5 becomes 22. */
/* parameters the half-turn coefficient of term k depends on (devmath.cuh osc_terms) */
int term_deps(int osc_model, int k, int slots[3])
{
    if (osc_model == PHYLINO_OSC_EQ1) { slots[0] = k == 0 ? PHYLINO_MEE : PHYLINO_M21; return 1; }
    if (osc_model == PHYLINO_OSC_STERILE4) { slots[0] = k == 0 ? PHYLINO_MEE : (k == 1 ? PHYLINO_M41 : PHYLINO_M21); return 1; }
    if (k == 2) { slots[0] = PHYLINO_M21; return 1; }            /* FULL3: (31, 32, 21) */
    slots[0] = PHYLINO_MEE; slots[1] = PHYLINO_S12; slots[2] = PHYLINO_M21;
    return 3;
}

uint64_t bits_of(double x) { uint64_t u; std::memcpy(&u, &x, sizeof u); return u; }

/* tags of the symbolic batch of gradient_plan: two disjoint families of bit patterns */
constexpr uint64_t kSymbolTag = 0xfff8000000000000ull, kFixedTag = 0xfff9000000000000ull;

uint64_t mix64(uint64_t h, uint64_t x)
{
    h ^= x + 0x9e3779b97f4a7c15ull + (h << 6) + (h >> 2);
    h *= 0xff51afd7ed558ccdull;
    return h ^ (h >> 32);
}

/* open-addressing set of ids; equality is decided by the caller on the ACTUAL key bits (the hash only
 * picks the probe start), so two different keys are never merged */
struct IdTable {
    std::vector<int32_t> slot;
    uint64_t mask;
    explicit IdTable(size_t n) { size_t c = 16; while (c < 2 * n + 2) c <<= 1; slot.assign(c, -1); mask = c - 1; }
    template <class Eq> int32_t find_or_insert(uint64_t h, int32_t fresh, Eq same, bool &inserted)
    {
        for (uint64_t i = h & mask;; i = (i + 1) & mask) {
            if (slot[i] < 0) { slot[i] = fresh; inserted = true; return fresh; }
            if (same(slot[i])) { inserted = false; return slot[i]; }
        }
    }
};

/* false: caching would not pay (more than half as many virtual points as points) -- use the dense path.
 * symbolic: `params` holds the symbols of gradient_plan (tags, not values); a FIXED oscillation parameter then
 * enters the comparison as a tag of its own (fixed slots with equal bits share one) that no symbol can equal, so a
 * fixed splitting is never merged with a fitted one because its value happens to look like a symbol. */
bool plan_components(const phylino_ctx *ctx, int P, const double *params, ComponentPlan &pl, bool symbolic = false)
{
    const int S = ctx->n_terms, NP = ctx->n_params;
    if (P >= (1 << 29)) return false;                   /* (point, term) is packed as p * 4 + k in an int32 */
    /* columns of the parameter vector that enter the energy scale of any dataset */
    std::vector<int32_t> acols;
    for (int d = 0; d < ctx->n_datasets && !ctx->ec_mode; ++d)     /* bin-level correction: the walk ignores the scale */
        for (int j = 0; j < 3; ++j)
            if (ctx->ds[d].idx_a[j] >= 0) acols.push_back(ctx->ds[d].idx_a[j]);
    std::vector<int32_t> cls((size_t)P);
    {
        IdTable tab((size_t)P);
        for (int p = 0; p < P; ++p) {
            const double *th = params + (size_t)p * NP;
            uint64_t h = 0x243f6a8885a308d3ull;
            for (int32_t c : acols) h = mix64(h, bits_of(th[c]));
            bool ins;
            const int32_t id = tab.find_or_insert(h, (int32_t)pl.class_rep.size(), [&](int32_t other) {
                const double *to = params + (size_t)pl.class_rep[other] * NP;
                for (int32_t c : acols) if (bits_of(th[c]) != bits_of(to[c])) return false;
                return true;
            }, ins);
            if (ins) pl.class_rep.push_back(p);
            cls[p] = id;
        }
    }
    pl.C = (int)pl.class_rep.size();
    /* distinct (class, formula, dependency bits) -> pair id, in order of first appearance */
    std::vector<int32_t> pair_class, pair_src, pt_pair((size_t)P * S);
    {
        IdTable tab((size_t)P * S);
        auto dep = [&](int p, int k, int j, int n_slots, const int *slots) -> uint64_t {
            (void)k; (void)n_slots;
            const int idx = ctx->idx_osc[slots[j]];
            if (idx >= 0) return bits_of(params[(size_t)p * NP + idx]);
            if (!symbolic) return bits_of(ctx->fixed_osc[slots[j]]);
            int first = slots[j];                           /* lowest fixed slot with the same bits */
            for (int q = 0; q < slots[j]; ++q)
                if (ctx->idx_osc[q] < 0 && bits_of(ctx->fixed_osc[q]) == bits_of(ctx->fixed_osc[slots[j]])) { first = q; break; }
            return kFixedTag | (uint64_t)first;
        };
        for (int p = 0; p < P; ++p) {
            for (int k = 0; k < S; ++k) {
                int slots[3];
                const int n = term_deps(ctx->osc_model, k, slots);
                const int formula = n == 1 ? 0 : k;             /* single-parameter terms share one formula */
                uint64_t h = mix64(mix64(0x13198a2e03707344ull, (uint64_t)cls[p]), (uint64_t)formula);
                for (int j = 0; j < n; ++j) h = mix64(h, dep(p, k, j, n, slots));
                bool ins;
                const int32_t id = tab.find_or_insert(h, (int32_t)pair_src.size(), [&](int32_t other) {
                    const int op = pair_src[other] >> 2, ok = pair_src[other] & 3;
                    int oslots[3];
                    const int on = term_deps(ctx->osc_model, ok, oslots);
                    if (pair_class[other] != cls[p] || on != n || (on == 1 ? 0 : ok) != formula) return false;
                    for (int j = 0; j < n; ++j) if (dep(p, k, j, n, slots) != dep(op, ok, j, on, oslots)) return false;
                    return true;
                }, ins);
                if (ins) { pair_class.push_back(cls[p]); pair_src.push_back(p * 4 + k); }
                pt_pair[(size_t)p * S + k] = id;
            }
        }
    }
    /* Pack the pairs of a class into virtual points of S slots.  Two ways, both exact: by TERM -- slot k holds only
     * pairs that first appeared as term k, so that a virtual point looks like a real one (the slow splitting in the
     * last slot, dm2_ee in the first) and the kernel's cheaper forms of those terms apply to the whole group -- or
     * S at a time in order of appearance, which needs fewer virtual points when one term has many more distinct
     * splittings than the others (config 5's grid: 64 values of dm2_41, one of each other: 22 against 64).  By term
     * where that costs no extra virtual point (config 3's gradient batch: 21 either way). */
    const int n_pairs = (int)pair_class.size();
    std::vector<int32_t> cnt_c((size_t)pl.C, 0), cnt_ck((size_t)pl.C * S, 0), pair_cell((size_t)n_pairs);
    for (int q = 0; q < n_pairs; ++q) {
        ++cnt_c[pair_class[q]];
        ++cnt_ck[(size_t)pair_class[q] * S + (pair_src[q] & 3)];
    }
    int64_t v_free = 0, v_term = 0;
    for (int c = 0; c < pl.C; ++c) {
        v_free += (cnt_c[c] + S - 1) / S;
        int m = 0;
        for (int k = 0; k < S; ++k) m = std::max(m, (int)cnt_ck[(size_t)c * S + k]);
        v_term += m;
    }
    if (v_term <= v_free) {
        std::vector<int32_t> base((size_t)pl.C, 0), first_c((size_t)pl.C, -1), first_ck((size_t)pl.C * S, -1);
        for (int q = n_pairs - 1; q >= 0; --q) {
            first_c[pair_class[q]] = pair_src[q];
            first_ck[(size_t)pair_class[q] * S + (pair_src[q] & 3)] = pair_src[q];
        }
        for (int c = 0; c < pl.C; ++c) {
            int m = 0;
            for (int k = 0; k < S; ++k) m = std::max(m, (int)cnt_ck[(size_t)c * S + k]);
            base[c] = pl.V;
            for (int j = 0; j < m; ++j) {
                pl.vp_class.push_back(c);
                for (int k = 0; k < S; ++k)         /* unused slots repeat the first pair of their term (or class) */
                    pl.vp_src.push_back(first_ck[(size_t)c * S + k] >= 0 ? first_ck[(size_t)c * S + k] : first_c[c]);
            }
            pl.V += m;
        }
        std::vector<int32_t> seen((size_t)pl.C * S, 0);
        for (int q = 0; q < n_pairs; ++q) {
            const int c = pair_class[q], k = pair_src[q] & 3;
            const int vp = base[c] + seen[(size_t)c * S + k]++;
            pl.vp_src[(size_t)vp * S + k] = pair_src[q];
            pair_cell[q] = vp * (S + 1) + 1 + k;
        }
    } else {
        std::vector<int32_t> fill((size_t)pl.C, 0), open_vp((size_t)pl.C, -1);
        for (int q = 0; q < n_pairs; ++q) {
            const int c = pair_class[q];
            if (open_vp[c] < 0 || fill[c] == S) {
                open_vp[c] = pl.V++;
                fill[c] = 0;
                pl.vp_class.push_back(c);
                for (int s2 = 0; s2 < S; ++s2) pl.vp_src.push_back(pair_src[q]);   /* unused slots repeat the first pair */
            }
            pl.vp_src[(size_t)open_vp[c] * S + fill[c]] = pair_src[q];
            pair_cell[q] = open_vp[c] * (S + 1) + 1 + fill[c];
            ++fill[c];
        }
    }
    if (2 * (int64_t)pl.V > P) return false;
    pl.pt_comp.resize((size_t)P * (S + 1));
    for (int p = 0; p < P; ++p) {
        int32_t *row = &pl.pt_comp[(size_t)p * (S + 1)];
        for (int k = 0; k < S; ++k) row[k + 1] = pair_cell[pt_pair[(size_t)p * S + k]];
        row[0] = (row[1] - 1) / (S + 1) * (S + 1);          /* W of the virtual point that holds term 0 */
    }
    return true;
}

/* the plan as the kernels read it: vp_class | vp_src | class_rep | pt_comp */
std::vector<int32_t> plan_blob(const ComponentPlan &pl)
{
    std::vector<int32_t> blob;
    blob.reserve(pl.vp_class.size() + pl.vp_src.size() + pl.class_rep.size() + pl.pt_comp.size());
    blob.insert(blob.end(), pl.vp_class.begin(), pl.vp_class.end());
    blob.insert(blob.end(), pl.vp_src.begin(), pl.vp_src.end());
    blob.insert(blob.end(), pl.class_rep.begin(), pl.class_rep.end());
    blob.insert(blob.end(), pl.pt_comp.begin(), pl.pt_comp.end());
    return blob;
}

/* enqueue rows a1-a7 for a host-resident batch already copied to d_params, through the component
 * plan; hist xor nll as in enqueue_finalize */
phylino_status enqueue_cached(phylino_ctx *ctx, int P, const double *h_params, const double *d_params,
                              const double *d_data, double *d_hist, double *d_nll, bool *used,
                              const ComponentPlan *given = nullptr, const int32_t *d_given = nullptr)
{
    *used = false;
    ctx->last_virtual_points = ctx->last_classes = 0;
    ComponentPlan made;
    if (!given && !plan_components(ctx, P, h_params, made)) return PHYLINO_OK;
    const ComponentPlan &pl = given ? *given : made;
    const int S = ctx->n_terms, V = pl.V;
    phylino_status s;
    /* accumulator rows: V (S + 1); threshold rows and records: sized by ensure_acc for max(P, .) points */
    if ((s = ensure_acc(ctx, std::max(P, V * (S + 1)))) != PHYLINO_OK) return s;
    const int64_t n_int = (int64_t)V + (int64_t)V * S + pl.C + (int64_t)P * (S + 1);
    const int32_t *d_plan = d_given;            /* a plan that already sits on the device (gradient_plan) */
    if (!d_plan) {
        if (n_int > ctx->plan_capacity) {
            CU(cudaStreamSynchronize(ctx->stream));
            cudaFree(ctx->d_plan); ctx->d_plan = nullptr; ctx->plan_capacity = 0;
            CU(cudaMalloc((void **)&ctx->d_plan, n_int * sizeof(int32_t)));
            ctx->plan_capacity = n_int;
        }
        const std::vector<int32_t> blob = plan_blob(pl);
        /* pageable source: the copy is staged by the driver before the call returns */
        CU(cudaMemcpyAsync(ctx->d_plan, blob.data(), n_int * sizeof(int32_t), cudaMemcpyHostToDevice, ctx->stream));
        d_plan = ctx->d_plan;
    }

    SpectraArgs a{};
    fill_datasets(ctx, a);
    a.comp = 1;
    if ((s = fill_batch(ctx, a, V, d_params, pl.C)) != PHYLINO_OK) return s;
    ctx->last_points = V;
    ctx->last_fused = a.sched == 1;
    a.vp_class = d_plan;
    a.vp_src = d_plan + V;
    a.class_rep = d_plan + V + (int64_t)V * S;
    FinalizeArgs f = ctx->fin;
    f.P = P; f.params = d_params; f.acc = ctx->d_acc; f.flags = ctx->d_flags;
    f.data = d_data; f.hist = d_hist; f.nll = d_nll;
    f.comp = 1; f.n_terms = S; f.osc = a.osc;
    f.ec_mode = ctx->ec_mode;
    f.pt_comp = d_plan + V + (int64_t)V * S + pl.C;
    if (ctx->timing) CU(cudaEventRecord(ctx->ev[0], ctx->stream));
    if (a.sched == 1) {
        /* few virtual points: setup and walk in one launch; the per-point combination stays a launch of its own */
        if (ctx->timing) CU(cudaEventRecord(ctx->ev[1], ctx->stream));
        CU(launch_fused(a, ctx->blob, S, ctx->stream, !ctx->timing, false));
        ctx->launches += 1;
        f.reset_counter = ctx->d_done;
    } else {
        if (a.n_items > 0) { CU(launch_setup(a, S, ctx->stream)); ctx->launches += 1; }
        if (ctx->timing) CU(cudaEventRecord(ctx->ev[1], ctx->stream));
        if (a.n_items > 0) { CU(launch_spectra(a, S, ctx->stream, !ctx->timing, false)); ctx->launches += 1; }
    }
    if (ctx->timing) CU(cudaEventRecord(ctx->ev[2], ctx->stream));
    CU(launch_finalize(f, d_nll ? 2 : 0, ctx->stream, !ctx->timing && (a.sched == 1 || a.n_items > 0)));
    ctx->launches += 1;
    if (ctx->timing) CU(cudaEventRecord(ctx->ev[3], ctx->stream));
    /* the cells are shared between points: cleared here, not by the finalize kernel */
    const size_t cells = (size_t)V * (S + 1) * ctx->total_bins;
    CU(cudaMemsetAsync(ctx->d_acc, 0, cells * sizeof(long long), ctx->stream));
    CU(cudaMemsetAsync(ctx->d_flags, 0, cells * sizeof(unsigned), ctx->stream));
    ctx->last_virtual_points = V;
    ctx->last_classes = pl.C;
    *used = true;
    return PHYLINO_OK;
}

/* The plan of a central-difference batch {theta} U {theta +- step_j e_j} needs no values: which points share an
 * energy-scale tuple or a mass splitting follows from WHICH column a point perturbs.  plan_components only compares
 * bit patterns, so it is run once per model on a symbolic batch with that equality structure (column j holds the
 * tag 4 j, perturbed entries 4 j + 1 / 4 j + 2; fixed oscillation parameters get tags of another family, see
 * plan_components) and the plan is kept.  Points that are structurally different but equal in value (a step below
 * one ulp, a fixed splitting equal to a fitted one) are merely not merged; structurally equal points ARE equal in
 * value, so nothing is merged wrongly.  Not with a transformation layer (a step in u_j moves several columns of theta by amounts the symbols do
 * not know).  With this phylino_nll_gradient plans without seeing the batch: no copy back, no synchronisation. */
const ComponentPlan *gradient_plan(phylino_ctx *ctx, int width)
{
    if (ctx->grad_plan_state == 0) {
        cudaFree(ctx->d_grad_plan);
        ctx->d_grad_plan = nullptr;
        const int P = 2 * width + 1;
        std::vector<double> sym((size_t)P * width);
        for (int r = 0; r < P; ++r)
            for (int j = 0; j < width; ++j) {
                const uint64_t tag = kSymbolTag | (4ull * (uint64_t)j + ((r > 0 && (r - 1) / 2 == j) ? ((r & 1) ? 1u : 2u) : 0u));
                std::memcpy(&sym[(size_t)r * width + j], &tag, sizeof tag);
            }
        ctx->grad_plan = ComponentPlan();
        ctx->grad_plan_state = plan_components(ctx, P, sym.data(), ctx->grad_plan, true) ? 1 : -1;
        if (ctx->grad_plan_state > 0) {
            /* once per model, outside any capture: the plan stays on the device */
            const std::vector<int32_t> blob = plan_blob(ctx->grad_plan);
            if (cudaMalloc((void **)&ctx->d_grad_plan, blob.size() * sizeof(int32_t)) != cudaSuccess ||
                cudaMemcpy(ctx->d_grad_plan, blob.data(), blob.size() * sizeof(int32_t), cudaMemcpyHostToDevice) != cudaSuccess) {
                cudaGetLastError();
                cudaFree(ctx->d_grad_plan);
                ctx->d_grad_plan = nullptr;
                ctx->grad_plan_state = -1;
            }
        }
    }
    return ctx->grad_plan_state > 0 ? &ctx->grad_plan : nullptr;
}

/* Caching for a DEVICE-resident batch: the plan is made on the host, so theta comes back once (one
 * device -> host copy of the batch and one stream synchronisation per call -- the price stated in phylino.h). */
phylino_status cached_from_device(phylino_ctx *ctx, int P, const double *d_theta, const double *d_data,
                                  double *d_hist, double *d_nll, bool *used)
{
    *used = false;
    const int64_t np = (int64_t)P * ctx->n_params;
    phylino_status s;
    if ((s = ensure_stage(ctx, np)) != PHYLINO_OK) return s;
    CU(cudaMemcpyAsync(ctx->h_pin, d_theta, np * sizeof(double), cudaMemcpyDeviceToHost, ctx->stream));
    CU(cudaStreamSynchronize(ctx->stream));
    return enqueue_cached(ctx, P, ctx->h_pin, d_theta, d_data, d_hist, d_nll, used);
}

} // namespace

extern "C" {

phylino_status phylino_create(int device, void *cuda_stream, phylino_ctx **out)
{
    if (!out) return PHYLINO_ERR_ARG;
    *out = nullptr;
    int n = 0;
    cudaError_t e = cudaGetDeviceCount(&n);
    if (e != cudaSuccess || device < 0 || device >= n) { cudaGetLastError(); return PHYLINO_ERR_CUDA; }
    phylino_ctx *c = new (std::nothrow) phylino_ctx;
    if (!c) return PHYLINO_ERR_OOM;
    c->device = device;
    c->stream = (cudaStream_t)cuda_stream;
    DeviceGuard g(device);
    /* allow_stage_all: the shared-memory opt-in of the spectra kernels, once per context (it is a per-device setting) */
    if (!g.ok || cudaFree(0) != cudaSuccess ||
        cudaDeviceGetAttribute(&c->sm_count, cudaDevAttrMultiProcessorCount, device) != cudaSuccess ||
        allow_stage_all() != cudaSuccess) {
        cudaGetLastError();
        delete c;
        return PHYLINO_ERR_CUDA;
    }
    *out = c;
    return PHYLINO_OK;
}

void phylino_destroy(phylino_ctx *ctx)
{
    if (!ctx) return;
    DeviceGuard g(ctx->device);
    cudaStreamSynchronize(ctx->stream);
    free_all(ctx);
    free_events_timing(ctx);
    delete ctx;
}

phylino_status phylino_set_model(phylino_ctx *ctx, const phylino_model_desc *m)
{
    if (!ctx) return PHYLINO_ERR_ARG;
    if (!m || !m->datasets) return fail(ctx, PHYLINO_ERR_ARG, "NULL model");
    if (m->osc_model < PHYLINO_OSC_EQ1 || m->osc_model > PHYLINO_OSC_STERILE4)
        return fail(ctx, PHYLINO_ERR_ARG, "unknown osc_model %d", m->osc_model);
    if (m->n_params < 0) return fail(ctx, PHYLINO_ERR_SHAPE, "n_params = %d", m->n_params);
    if (m->n_datasets < 1 || m->n_datasets > PHYLINO_MAX_DATASETS)
        return fail(ctx, PHYLINO_ERR_SHAPE, "n_datasets = %d not in 1..%d", m->n_datasets, PHYLINO_MAX_DATASETS);
    const int n_used_osc = m->osc_model == PHYLINO_OSC_STERILE4 ? 6 : 4;
    for (int j = 0; j < n_used_osc; ++j)
        if (!idx_ok(m->idx_osc[j], m->n_params)) return fail(ctx, PHYLINO_ERR_SHAPE, "idx_osc[%d] = %d out of range", j, m->idx_osc[j]);
    int64_t tb = 0;
    int max_bkg = 0, max_bins = 0;
    bool perpoint = false;
    for (int d = 0; d < m->n_datasets; ++d) {
        const phylino_dataset_desc &s = m->datasets[d];
        if (s.n_bins < 1 || s.n_bins > PHYLINO_MAX_BINS)
            return fail(ctx, PHYLINO_ERR_SHAPE, "dataset %d: n_bins = %d not in 1..%d", d, s.n_bins, PHYLINO_MAX_BINS);
        if (s.n_bkg < 0 || s.n_bkg > PHYLINO_MAX_BKG || (s.n_bkg > 0 && !s.bkg))
            return fail(ctx, PHYLINO_ERR_SHAPE, "dataset %d: n_bkg = %d", d, s.n_bkg);
        for (int j = 0; j < 3; ++j) {
            if (!idx_ok(s.idx_a[j], m->n_params)) return fail(ctx, PHYLINO_ERR_SHAPE, "dataset %d: idx_a[%d] out of range", d, j);
            perpoint |= s.idx_a[j] >= 0;
        }
        if (!idx_ok(s.idx_signorm, m->n_params)) return fail(ctx, PHYLINO_ERR_SHAPE, "dataset %d: idx_signorm out of range", d);
        if (s.idx_flux)
            for (int b = 0; b < s.n_bins; ++b)
                if (!idx_ok(s.idx_flux[b], m->n_params)) return fail(ctx, PHYLINO_ERR_SHAPE, "dataset %d: idx_flux[%d] out of range", d, b);
        for (int k = 0; k < s.n_bkg; ++k) {
            const phylino_bkg_desc &bk = s.bkg[k];
            if (!bk.tmpl) return fail(ctx, PHYLINO_ERR_ARG, "dataset %d bkg %d: NULL template", d, k);
            if (!idx_ok(bk.idx_rate, m->n_params)) return fail(ctx, PHYLINO_ERR_SHAPE, "dataset %d bkg %d: idx_rate out of range", d, k);
            if (bk.idx_shape)
                for (int b = 0; b < s.n_bins; ++b)
                    if (!idx_ok(bk.idx_shape[b], m->n_params)) return fail(ctx, PHYLINO_ERR_SHAPE, "dataset %d bkg %d: idx_shape[%d] out of range", d, k, b);
        }
        tb += s.n_bins;
        max_bkg = std::max(max_bkg, s.n_bkg);
        max_bins = std::max(max_bins, s.n_bins);
    }

    DeviceGuard g(ctx->device);
    CU(cudaStreamSynchronize(ctx->stream));
    free_all(ctx);

    ctx->osc_model = m->osc_model;
    ctx->ordering = m->ordering >= 0 ? 1 : -1;
    ctx->n_params = m->n_params;
    ctx->n_datasets = m->n_datasets;
    ctx->n_terms = m->osc_model == PHYLINO_OSC_EQ1 ? 2 : 3;
    for (int j = 0; j < 6; ++j) { ctx->idx_osc[j] = j < n_used_osc ? m->idx_osc[j] : -1; ctx->fixed_osc[j] = m->fixed_osc[j]; }
    ctx->per_point_binning = perpoint;
    ctx->total_bins = (int32_t)tb;
    ctx->max_bkg = max_bkg;
    ctx->max_bins = max_bins;
    ctx->ds.resize(m->n_datasets);

    std::vector<int32_t> bin_ds(tb), idx_flux(tb, -1), idx_signorm(m->n_datasets), n_bkg(m->n_datasets);
    std::vector<int32_t> idx_rate((size_t)m->n_datasets * std::max(max_bkg, 1), -1);
    std::vector<int32_t> idx_shape((size_t)std::max(max_bkg, 1) * tb, -1);
    std::vector<double> tmpl((size_t)std::max(max_bkg, 1) * tb, 0.0), norm(m->n_datasets), inv_scale(m->n_datasets, 1.0);
    int64_t off = 0;
    for (int d = 0; d < m->n_datasets; ++d) {
        const phylino_dataset_desc &s = m->datasets[d];
        phylino_dataset_host &h = ctx->ds[d];
        h.n_bins = s.n_bins;
        for (int j = 0; j < 3; ++j) h.idx_a[j] = s.idx_a[j];
        h.idx_signorm = s.idx_signorm;
        h.norm = s.norm;
        idx_signorm[d] = s.idx_signorm;
        norm[d] = s.norm;
        n_bkg[d] = s.n_bkg;
        for (int b = 0; b < s.n_bins; ++b) {
            bin_ds[off + b] = d;
            if (s.idx_flux) idx_flux[off + b] = s.idx_flux[b];
        }
        for (int k = 0; k < s.n_bkg; ++k) {
            const phylino_bkg_desc &bk = s.bkg[k];
            idx_rate[(size_t)d * max_bkg + k] = bk.idx_rate;
            for (int b = 0; b < s.n_bins; ++b) {
                tmpl[(size_t)k * tb + off + b] = bk.tmpl[b];
                if (bk.idx_shape) idx_shape[(size_t)k * tb + off + b] = bk.idx_shape[b];
            }
        }
        off += s.n_bins;
    }
    FinalizeArgs &f = ctx->fin;
    f.n_params = m->n_params;
    f.total_bins = (int32_t)tb;
    f.staged = tb <= FIN_STAGE_MAX_BINS ? 1 : 0;
    ctx->ec_mode = 0;
    ctx->grad_plan_state = 0;
    ctx->fm_idx.assign(m->n_datasets, std::vector<int32_t>());
    ctx->fm_lo.assign(m->n_datasets, 0.0);
    ctx->fm_width.assign(m->n_datasets, 0.0);
    {
        std::vector<int32_t> ds_off(m->n_datasets + 1, 0), ds_a((size_t)m->n_datasets * 3, -1);
        for (int d = 0; d < m->n_datasets; ++d) {
            ds_off[d + 1] = ds_off[d] + m->datasets[d].n_bins;
            for (int j = 0; j < 3; ++j) ds_a[(size_t)3 * d + j] = m->datasets[d].idx_a[j];
        }
        std::vector<double> edges0((size_t)tb + m->n_datasets, 0.0);
        std::vector<int32_t> fm_off(m->n_datasets + 1, 0);
        CU(upload((int32_t **)&f.ds_bin_off, ds_off, ctx->stream));
        CU(upload((int32_t **)&f.ds_idx_a, ds_a, ctx->stream));
        CU(upload((double **)&f.edges_all, edges0, ctx->stream));
        CU(upload((int32_t **)&f.fm_off, fm_off, ctx->stream));
        CU(cudaStreamSynchronize(ctx->stream));
    }
    f.n_datasets = m->n_datasets;
    f.max_bkg = max_bkg;
    cudaStream_t st = ctx->stream;
    CU(upload((int32_t **)&f.bin_ds, bin_ds, st));
    CU(upload((int32_t **)&f.idx_flux, idx_flux, st));
    CU(upload((double **)&f.inv_scale, inv_scale, st));
    CU(upload((double **)&f.norm, norm, st));
    CU(upload((int32_t **)&f.idx_signorm, idx_signorm, st));
    CU(upload((int32_t **)&f.n_bkg, n_bkg, st));
    CU(upload((int32_t **)&f.idx_rate, idx_rate, st));
    CU(upload((int32_t **)&f.idx_shape, idx_shape, st));
    CU(upload((double **)&f.tmpl, tmpl, st));
    if (m->prior_mean && m->prior_sigma && m->n_params > 0) {
        std::vector<double> pm(m->prior_mean, m->prior_mean + m->n_params);
        std::vector<double> ps(m->prior_sigma, m->prior_sigma + m->n_params);
        CU(upload((double **)&f.prior_mean, pm, st));
        CU(upload((double **)&f.prior_sigma, ps, st));
    }
    CU(cudaStreamSynchronize(st));      /* the host vectors above die here */
    ctx->have_model = true;
    ctx->err.clear();
    return PHYLINO_OK;
}

phylino_status phylino_load_events(phylino_ctx *ctx, int dataset, int64_t n, const float *e_nu,
                                   const float *e_vis, const float *weight, const int32_t *core,
                                   int n_cores, const double *baseline_m, int n_bins, const double *edges)
{
    if (!ctx) return PHYLINO_ERR_ARG;
    if (!ctx->have_model) return fail(ctx, PHYLINO_ERR_STATE, "phylino_set_model must come before phylino_load_events");
    if (dataset < 0 || dataset >= ctx->n_datasets) return fail(ctx, PHYLINO_ERR_SHAPE, "dataset %d not in 0..%d", dataset, ctx->n_datasets - 1);
    phylino_dataset_host &h = ctx->ds[dataset];
    if (n_bins != h.n_bins) return fail(ctx, PHYLINO_ERR_SHAPE, "dataset %d: n_bins = %d, model says %d", dataset, n_bins, h.n_bins);
    if (n < 0 || n > 0x7fff0000ll) return fail(ctx, PHYLINO_ERR_SHAPE, "n = %lld out of range", (long long)n);
    if (!edges || n_cores < 1 || !baseline_m || (n > 0 && (!e_nu || !e_vis)))
        return fail(ctx, PHYLINO_ERR_ARG, "NULL array or n_cores < 1");
    for (int b = 0; b <= n_bins; ++b)
        if (!std::isfinite(edges[b]) || (b > 0 && !(edges[b] > edges[b - 1])))
            return fail(ctx, PHYLINO_ERR_ARG, "edges must be finite and strictly ascending (at %d)", b);
    for (int c = 0; c < n_cores; ++c)
        if (!std::isfinite(baseline_m[c]) || baseline_m[c] < 0.0) return fail(ctx, PHYLINO_ERR_ARG, "baseline %d is not finite >= 0", c);
    for (int64_t i = 0; i < n; ++i) {
        if (!(e_nu[i] > 0.0f) || !std::isfinite(e_nu[i])) return fail(ctx, PHYLINO_ERR_ARG, "e_nu[%lld] is not finite > 0", (long long)i);
        if (weight && !std::isfinite(weight[i])) return fail(ctx, PHYLINO_ERR_ARG, "weight[%lld] is not finite", (long long)i);
        if (core && (core[i] < 0 || core[i] >= n_cores)) return fail(ctx, PHYLINO_ERR_ARG, "core[%lld] = %d out of range", (long long)i, core[i]);
    }

    /* sort by reconstructed energy (R14), NaN last, stable */
    std::vector<int32_t> perm((size_t)n);
    std::iota(perm.begin(), perm.end(), 0);
    std::stable_sort(perm.begin(), perm.end(), [e_vis](int32_t a, int32_t b) {
        float x = e_vis[a], y = e_vis[b];
        if (x != x) return false;
        if (y != y) return true;
        return x < y;
    });
    const int64_t n_pad = (n + EB - 1) / EB * EB, n_batches = n_pad / EB;
    double wsum = 0.0;
    bool unit_w = true;
    float v_pos_min = INFINITY, v_max = -INFINITY;
    for (int64_t i = 0; i < n; ++i) {
        const float vi = e_vis[i];
        const double wi = weight ? (double)weight[i] : 1.0;
        wsum += std::fabs(wi);
        unit_w = unit_w && wi == 1.0;
        if (std::isfinite(vi)) {
            if (vi > 0.0f && vi < v_pos_min) v_pos_min = vi;
            if (vi > v_max) v_max = vi;
        }
    }
    /* records of EB consecutive sorted events: 48 bytes (x, v) when every weight is exactly 1, else 96 (x, w, v,
     * batch weight sum); padding: x = 0, w = 0, v = NaN (lands in no bin) */
    std::vector<EventBatchU> ev_u;
    std::vector<EventBatchW> ev_w;
    {
        EventBatchU bu{};
        EventBatchW bw{};
        for (int j = 0; j < EB; ++j) { bu.v[j] = std::nanf(""); bw.v[j] = std::nanf(""); }
        if (unit_w) ev_u.assign((size_t)n_batches, bu); else ev_w.assign((size_t)n_batches, bw);
    }
    /* where a lane starts looking for its bin (a hint, never trusted): the bin of the first event of every
     * HINT_BATCHES-th batch under the identity energy scale */
    std::vector<HintEntry> hint((size_t)((n_batches + HINT_BATCHES - 1) / HINT_BATCHES), HintEntry{n_bins, 0.0f});
    std::vector<double> x_blk(hint.size(), 0.0);       /* largest L/E_nu of each block of HINT_BATCHES batches */
    std::vector<float> v_blk(hint.size(), std::nanf(""));
    double x_max = 0.0;
    for (int64_t i = 0; i < n; ++i) {
        const int32_t s = perm[i];
        const int64_t b = i / EB;
        const int j = (int)(i % EB);
        const float vi = e_vis[s];
        const double xi = baseline_m[core ? core[s] : 0] / (double)e_nu[s];
        x_max = std::max(x_max, xi);
        x_blk[(size_t)(b / HINT_BATCHES)] = std::max(x_blk[(size_t)(b / HINT_BATCHES)], xi);
        if (unit_w) {
            ev_u[(size_t)b].x[j] = xi;
            ev_u[(size_t)b].v[j] = vi;
        } else {
            EventBatchW &r = ev_w[(size_t)b];
            r.x[j] = xi;
            r.v[j] = vi;
            r.w[j] = (double)weight[s];
            r.wsum += r.w[j];                   /* in event order: the batch total the hot kernel adds */
        }
        if (j == 0 && b % HINT_BATCHES == 0) v_blk[(size_t)(b / HINT_BATCHES)] = vi;
        if (j == 0 && b % HINT_BATCHES == 0)
            hint[(size_t)(b / HINT_BATCHES)].bin =
                vi == vi ? (int32_t)(std::upper_bound(edges, edges + n_bins + 1, (double)vi) - edges) - 1 : n_bins;
    }
    /* envelope of L/E_nu from a block to the end of the store, as a float rounded up: the store is sorted by E_vis, and
     * L/E_nu falls with it, so the envelope stays close to the block's own largest value */
    {
        double env = 0.0;
        for (size_t i = hint.size(); i-- > 0;) {
            env = std::max(env, x_blk[i]);
            float f = (float)env;
            if ((double)f < env) f = std::nextafter(f, INFINITY);
            hint[i].x_env = f;
        }
    }
    /* fixed-point scale 2^e with 8 * sum|w| * 2^e <= 2^62 (|P_ee| <= 4 is enforced per point) */
    int ex = 0;
    if (wsum > 0.0) std::frexp(wsum, &ex);
    int fx = std::max(-1000, std::min(1000, 59 - ex));

    DeviceGuard g(ctx->device);
    CU(cudaStreamSynchronize(ctx->stream));
    free_events(h);
    cudaStream_t st = ctx->stream;
    std::vector<double> ed(edges, edges + n_bins + 1);
    if (unit_w) { EventBatchU *d = nullptr; CU(upload(&d, ev_u, st)); h.d_ev = d; }
    else        { EventBatchW *d = nullptr; CU(upload(&d, ev_w, st)); h.d_ev = d; }
    CU(upload(&h.d_edges, ed, st));
    CU(upload(&h.d_perm, perm, st));
    CU(upload(&h.d_hint, hint, st));
    double inv = std::ldexp(1.0, -fx);
    CU(cudaMemcpyAsync((void *)(ctx->fin.inv_scale + dataset), &inv, sizeof(double), cudaMemcpyHostToDevice, st));
    {
        int64_t off = dataset;                  /* dataset d's edges start at (bins before it) + d */
        for (int d = 0; d < dataset; ++d) off += ctx->ds[d].n_bins;
        CU(cudaMemcpyAsync((void *)(ctx->fin.edges_all + off), ed.data(), ed.size() * sizeof(double), cudaMemcpyHostToDevice, st));
    }
    CU(cudaStreamSynchronize(st));
    h.n = n; h.n_pad = n_pad; h.wsum_abs = wsum; h.fx_exp = fx; h.loaded = true;
    h.v_pos_min = v_pos_min; h.v_max = v_max; h.unit_w = unit_w; h.x_max = x_max;
    h.v_blk.swap(v_blk);
    h.edges = ed;
    cudaFree(ctx->d_unit_order);                /* the single-launch kernel's unit order belongs to the old store */
    ctx->d_unit_order = nullptr;
    ctx->order_U = ctx->order_units = 0;
    ctx->err.clear();
    return PHYLINO_OK;
}

phylino_status phylino_spectra(phylino_ctx *ctx, int P, const double *params, double *hist)
{
    phylino_status s = check_ready(ctx, P, params, hist);
    if (s != PHYLINO_OK || P == 0) return s;
    DeviceGuard g(ctx->device);
    if ((s = resolve_params(ctx, P, params, &params)) != PHYLINO_OK) return s;
    if (ctx->caching && !wants_single_launch(ctx, P)) {
        bool cached = false;
        if ((s = cached_from_device(ctx, P, params, nullptr, hist, nullptr, &cached)) != PHYLINO_OK || cached) return s;
    } else {
        ctx->last_virtual_points = ctx->last_classes = 0;
    }
    if ((s = ensure_acc(ctx, P)) != PHYLINO_OK) return s;
    return enqueue_eval(ctx, P, params, nullptr, hist, nullptr, 0);
}

phylino_status phylino_nll(phylino_ctx *ctx, int P, const double *params, const double *data, double *nll)
{
    phylino_status s = check_ready(ctx, P, params, nll);
    if (s != PHYLINO_OK || P == 0) return s;
    if (!data) return fail(ctx, PHYLINO_ERR_ARG, "NULL data pointer");
    DeviceGuard g(ctx->device);
    if ((s = resolve_params(ctx, P, params, &params)) != PHYLINO_OK) return s;
    if (ctx->caching && !wants_single_launch(ctx, P)) {
        bool cached = false;
        if ((s = cached_from_device(ctx, P, params, data, nullptr, nll, &cached)) != PHYLINO_OK || cached) return s;
    } else {
        ctx->last_virtual_points = ctx->last_classes = 0;
    }
    if ((s = ensure_acc(ctx, P)) != PHYLINO_OK) return s;
    return enqueue_eval(ctx, P, params, data, nullptr, nll, 2);
}

phylino_status phylino_nll_ensemble(phylino_ctx *ctx, int P, const double *params, int E, const double *data,
                                    double *nll)
{
    phylino_status s = check_ready(ctx, P, params, nll);
    if (s != PHYLINO_OK) return s;
    if (E < 0) return fail(ctx, PHYLINO_ERR_SHAPE, "E = %d is negative", E);
    if (P == 0 || E == 0) return PHYLINO_OK;
    if (!data) return fail(ctx, PHYLINO_ERR_ARG, "NULL data pointer");
    DeviceGuard g(ctx->device);
    if ((s = resolve_params(ctx, P, params, &params)) != PHYLINO_OK) return s;
    if ((s = ensure_acc(ctx, P)) != PHYLINO_OK) return s;
    const int64_t need = (int64_t)P * ctx->total_bins;
    if (need > ctx->mu_capacity) {
        CU(cudaStreamSynchronize(ctx->stream));
        cudaFree(ctx->d_mu); ctx->d_mu = nullptr; ctx->mu_capacity = 0;
        CU(cudaMalloc((void **)&ctx->d_mu, need * sizeof(double)));
        ctx->mu_capacity = need;
    }
    if ((s = enqueue_eval(ctx, P, params, nullptr, ctx->d_mu, nullptr, 1)) != PHYLINO_OK) return s;
    FinalizeArgs f = ctx->fin;
    f.P = P; f.params = params; f.data = data; f.hist = ctx->d_mu; f.nll = nll;
    f.ec_mode = ctx->ec_mode;
    CU(launch_ensemble(f, E, ctx->sm_count, ctx->stream));
    ctx->launches += 1;
    return PHYLINO_OK;
}

/* work buffer of the consumers below (grown with a stream synchronise, like the other per-batch buffers) */
static phylino_status ensure_work(phylino_ctx *ctx, int64_t doubles)
{
    if (doubles <= ctx->work_capacity) return PHYLINO_OK;
    CU(cudaStreamSynchronize(ctx->stream));
    cudaFree(ctx->d_work); ctx->d_work = nullptr; ctx->work_capacity = 0;
    CU(cudaMalloc((void **)&ctx->d_work, doubles * sizeof(double)));
    ctx->work_capacity = doubles;
    return PHYLINO_OK;
}

phylino_status phylino_draw_pseudo_data(phylino_ctx *ctx, const double *mu, int E, uint64_t seed, double *data)
{
    if (!ctx) return PHYLINO_ERR_ARG;
    if (!ctx->have_model) return fail(ctx, PHYLINO_ERR_STATE, "phylino_set_model has not been called");
    if (E < 0) return fail(ctx, PHYLINO_ERR_SHAPE, "E = %d is negative", E);
    if (E == 0) return PHYLINO_OK;
    if (!mu || !data) return fail(ctx, PHYLINO_ERR_ARG, "NULL mu or data pointer");
    DeviceGuard g(ctx->device);
    phylino_status s;
    if ((s = ensure_work(ctx, ctx->total_bins)) != PHYLINO_OK) return s;
    CU(launch_pseudo_data(mu, ctx->d_work, ctx->total_bins, E, (unsigned long long)seed, data, ctx->stream));
    ctx->launches += 2;
    return PHYLINO_OK;
}

phylino_status phylino_ordering_scan(phylino_ctx *ctx, int n_grid, int scan_param, const double *grid,
                                     const double *theta, const double *data, double *nll)
{
    phylino_status s = check_ready(ctx, n_grid, theta, nll);
    if (s != PHYLINO_OK || n_grid == 0) return s;
    if (!grid || !data) return fail(ctx, PHYLINO_ERR_ARG, "NULL grid or data pointer");
    const int64_t width = param_width(ctx);
    if (scan_param < 0 || scan_param >= width) return fail(ctx, PHYLINO_ERR_SHAPE, "scan_param = %d not in 0..%lld", scan_param, (long long)width - 1);
    DeviceGuard g(ctx->device);
    if ((s = ensure_work(ctx, (int64_t)n_grid * width)) != PHYLINO_OK) return s;
    if ((s = ensure_acc(ctx, n_grid)) != PHYLINO_OK) return s;
    double *batch = ctx->d_work;
    CU(launch_scan_batch(theta, (int)width, scan_param, grid, n_grid, batch, ctx->stream));
    ctx->launches += 1;
    const double *params = batch;
    if ((s = resolve_params(ctx, n_grid, batch, &params)) != PHYLINO_OK) return s;
    for (int o = 0; o < 2 && s == PHYLINO_OK; ++o) {
        ctx->ordering_override = o == 0 ? +1 : -1;
        s = enqueue_eval(ctx, n_grid, params, data, nullptr, nll + (size_t)o * n_grid, 2);
    }
    ctx->ordering_override = 0;
    ctx->last_virtual_points = ctx->last_classes = 0;
    return s;
}

phylino_status phylino_nll_gradient(phylino_ctx *ctx, const double *theta, const double *step, const double *data,
                                    double *nll0, double *grad)
{
    if (!ctx) return PHYLINO_ERR_ARG;
    const int64_t width = ctx->have_model ? param_width(ctx) : 0;
    if (width > (1 << 20)) return fail(ctx, PHYLINO_ERR_SHAPE, "too many parameters for a gradient batch");
    const int P = (int)(2 * width + 1);
    phylino_status s = check_ready(ctx, P, theta, grad);
    if (s != PHYLINO_OK) return s;
    if (!step || !data) return fail(ctx, PHYLINO_ERR_ARG, "NULL step or data pointer");
    if (width == 0) return PHYLINO_OK;
    DeviceGuard g(ctx->device);
    if ((s = ensure_work(ctx, (int64_t)P * width + P)) != PHYLINO_OK) return s;
    if ((s = ensure_acc(ctx, P)) != PHYLINO_OK) return s;
    double *batch = ctx->d_work, *nll = ctx->d_work + (int64_t)P * width;
    CU(launch_gradient_batch(theta, step, (int)width, batch, ctx->stream));
    ctx->launches += 1;
    bool done = false;
    if (ctx->caching && !ctx->have_tf && !wants_single_launch(ctx, P)) {
        /* cached through the structural plan of the batch: asynchronous like the dense call */
        if (const ComponentPlan *pl = gradient_plan(ctx, (int)width))
            if ((s = enqueue_cached(ctx, P, nullptr, batch, data, nullptr, nll, &done, pl, ctx->d_grad_plan)) != PHYLINO_OK) return s;
    }
    if (!done && (s = phylino_nll(ctx, P, batch, data, nll)) != PHYLINO_OK) return s;   /* dense, or cached via the host plan */
    CU(launch_gradient(theta, step, nll, (int)width, nll0, grad, ctx->stream));
    ctx->launches += 1;
    return PHYLINO_OK;
}

phylino_status phylino_variable_metric_step(phylino_ctx *ctx, int N, double *V, const double *dx, const double *dg,
                                            const double *grad, double *direction, double *edm)
{
    if (!ctx) return PHYLINO_ERR_ARG;
    if (N < 0 || N > (1 << 14)) return fail(ctx, PHYLINO_ERR_SHAPE, "N = %d not in 0..%d", N, 1 << 14);
    if (N == 0) return PHYLINO_OK;
    if (!V || !grad || !direction || !edm) return fail(ctx, PHYLINO_ERR_ARG, "NULL V, grad, direction or edm");
    if ((dx == nullptr) != (dg == nullptr)) return fail(ctx, PHYLINO_ERR_ARG, "dx and dg must both be given or both be NULL");
    DeviceGuard g(ctx->device);
    phylino_status s;
    if ((s = ensure_work(ctx, 2 * (int64_t)N + 2)) != PHYLINO_OK) return s;
    CU(launch_variable_metric_step(N, V, dx, dg, grad, direction, edm, ctx->d_work, ctx->stream));
    ctx->launches += (dx && dg) ? 5 : 2;
    return PHYLINO_OK;
}

phylino_status phylino_expectation(phylino_ctx *ctx, int P, const double *params, double *mu)
{
    phylino_status s = check_ready(ctx, P, params, mu);
    if (s != PHYLINO_OK || P == 0) return s;
    DeviceGuard g(ctx->device);
    if ((s = resolve_params(ctx, P, params, &params)) != PHYLINO_OK) return s;
    if ((s = ensure_acc(ctx, P)) != PHYLINO_OK) return s;
    return enqueue_eval(ctx, P, params, nullptr, mu, nullptr, 1);
}

phylino_status phylino_event_bins(phylino_ctx *ctx, int P, const double *params, int32_t *bins)
{
    phylino_status s = check_ready(ctx, P, params, bins);
    if (s != PHYLINO_OK || P == 0) return s;
    DeviceGuard g(ctx->device);
    if ((s = resolve_params(ctx, P, params, &params)) != PHYLINO_OK) return s;
    if ((s = ensure_acc(ctx, P)) != PHYLINO_OK) return s;
    /* the production kernels of this batch size in their diagnostic instantiation */
    CU(cudaMemsetAsync(bins, 0xff, (size_t)P * phylino_total_events(ctx) * sizeof(int32_t), ctx->stream));
    return enqueue_eval(ctx, P, params, nullptr, nullptr, nullptr, 3, bins);
}

phylino_status phylino_nll_host(phylino_ctx *ctx, int P, const double *params_host, const double *data_host,
                                double *nll_host)
{
    phylino_status s = check_ready(ctx, P, params_host, nll_host);
    if (s != PHYLINO_OK || P == 0) return s;
    if (!data_host) return fail(ctx, PHYLINO_ERR_ARG, "NULL data pointer");
    DeviceGuard g(ctx->device);
    const int64_t np = (int64_t)P * ctx->n_params, tb = ctx->total_bins;
    if ((s = ensure_stage(ctx, np + tb + P)) != PHYLINO_OK) return s;
    if ((s = ensure_acc(ctx, P)) != PHYLINO_OK) return s;
    if (ctx->have_tf) host_transform(ctx, P, params_host, ctx->h_pin);
    else std::memcpy(ctx->h_pin, params_host, np * sizeof(double));
    std::memcpy(ctx->h_pin + np, data_host, tb * sizeof(double));
    /* the likelihood stage writes nll[P] straight into the pinned block (8 P bytes over PCIe): no copy back */
    double *d_out = ctx->d_pin + np + tb;
    if (wants_single_launch(ctx, P) && np <= PARAM_BLOB_DOUBLES) {
        /* a single evaluation: no copy engine.  The parameters ride with the kernel arguments of the walk; the
         * finalize CTAs read parameters and data from the pinned block through its device alias while the events
         * are walked, and write nll[P] into it */
        ctx->last_virtual_points = ctx->last_classes = 0;
        if ((s = enqueue_eval(ctx, P, ctx->d_pin, ctx->d_pin + np, nullptr, d_out, 2, nullptr, ctx->h_pin)) != PHYLINO_OK)
            return s;
    } else {
        CU(cudaMemcpyAsync(ctx->d_stage, ctx->h_pin, (np + tb) * sizeof(double), cudaMemcpyHostToDevice, ctx->stream));
        bool cached = false;
        if (ctx->caching && !wants_single_launch(ctx, P) &&
            (s = enqueue_cached(ctx, P, ctx->h_pin, ctx->d_stage, ctx->d_stage + np, nullptr, d_out, &cached)) != PHYLINO_OK)
            return s;
        if (!cached) {
            ctx->last_virtual_points = ctx->last_classes = 0;
            if ((s = enqueue_eval(ctx, P, ctx->d_stage, ctx->d_stage + np, nullptr, d_out, 2)) != PHYLINO_OK) return s;
        }
    }
    CU(cudaStreamSynchronize(ctx->stream));
    std::memcpy(nll_host, ctx->h_pin + np + tb, P * sizeof(double));
    return PHYLINO_OK;
}

phylino_status phylino_spectra_host(phylino_ctx *ctx, int P, const double *params_host, double *hist_host)
{
    phylino_status s = check_ready(ctx, P, params_host, hist_host);
    if (s != PHYLINO_OK || P == 0) return s;
    DeviceGuard g(ctx->device);
    const int64_t np = (int64_t)P * ctx->n_params, nh = (int64_t)P * ctx->total_bins;
    if ((s = ensure_stage(ctx, np + nh)) != PHYLINO_OK) return s;
    if ((s = ensure_acc(ctx, P)) != PHYLINO_OK) return s;
    if (ctx->have_tf) host_transform(ctx, P, params_host, ctx->h_pin);
    else std::memcpy(ctx->h_pin, params_host, np * sizeof(double));
    CU(cudaMemcpyAsync(ctx->d_stage, ctx->h_pin, np * sizeof(double), cudaMemcpyHostToDevice, ctx->stream));
    bool cached = false;
    if (ctx->caching && !wants_single_launch(ctx, P) &&
        (s = enqueue_cached(ctx, P, ctx->h_pin, ctx->d_stage, nullptr, ctx->d_stage + np, nullptr, &cached)) != PHYLINO_OK)
        return s;
    if (!cached) {
        ctx->last_virtual_points = ctx->last_classes = 0;
        if ((s = enqueue_eval(ctx, P, ctx->d_stage, nullptr, ctx->d_stage + np, nullptr, 0)) != PHYLINO_OK) return s;
    }
    CU(cudaMemcpyAsync(ctx->h_pin + np, ctx->d_stage + np, nh * sizeof(double), cudaMemcpyDeviceToHost, ctx->stream));
    CU(cudaStreamSynchronize(ctx->stream));
    std::memcpy(hist_host, ctx->h_pin + np, nh * sizeof(double));
    return PHYLINO_OK;
}

phylino_status phylino_set_transform(phylino_ctx *ctx, int n_u, const int32_t *copy_src, const double *copy_const,
                                     int n_blocks, const phylino_transform_block *blocks)
{
    if (!ctx) return PHYLINO_ERR_ARG;
    if (!ctx->have_model) return fail(ctx, PHYLINO_ERR_STATE, "phylino_set_model must come before phylino_set_transform");
    DeviceGuard g(ctx->device);
    CU(cudaStreamSynchronize(ctx->stream));
    if (n_u == 0 && n_blocks == 0) { free_transform(ctx); ctx->err.clear(); return PHYLINO_OK; }
    if (n_u < 1 || n_blocks < 0) return fail(ctx, PHYLINO_ERR_SHAPE, "n_u = %d, n_blocks = %d", n_u, n_blocks);
    if (!copy_src || (n_blocks > 0 && !blocks)) return fail(ctx, PHYLINO_ERR_ARG, "NULL copy_src or blocks");
    const int NP = ctx->n_params;
    std::vector<int32_t> src(copy_src, copy_src + NP), row_off(1, 0), col_off(1, 0), idx_out, idx_in;
    std::vector<double> cst(NP, 0.0), offset, centre, matrix;
    std::vector<int64_t> mat_off;
    for (int j = 0; j < NP; ++j) {
        if (src[j] >= n_u) return fail(ctx, PHYLINO_ERR_SHAPE, "copy_src[%d] = %d out of range", j, src[j]);
        if (src[j] < 0) {
            if (!copy_const || !std::isfinite(copy_const[j])) return fail(ctx, PHYLINO_ERR_ARG, "copy_const[%d] missing or not finite", j);
            cst[j] = copy_const[j];
        }
    }
    for (int k = 0; k < n_blocks; ++k) {
        const phylino_transform_block &b = blocks[k];
        if (b.n_out < 1 || b.n_in < 1 || b.n_out > PHYLINO_MAX_BLOCK || b.n_in > PHYLINO_MAX_BLOCK)
            return fail(ctx, PHYLINO_ERR_SHAPE, "transform block %d: %d x %d not in 1..%d", k, b.n_out, b.n_in, PHYLINO_MAX_BLOCK);
        if (!b.idx_out || !b.idx_in || !b.offset || !b.centre || !b.matrix) return fail(ctx, PHYLINO_ERR_ARG, "transform block %d: NULL array", k);
        for (int i = 0; i < b.n_out; ++i)
            if (b.idx_out[i] < 0 || b.idx_out[i] >= NP || !std::isfinite(b.offset[i])) return fail(ctx, PHYLINO_ERR_SHAPE, "transform block %d: idx_out/offset[%d]", k, i);
        for (int j = 0; j < b.n_in; ++j)
            if (b.idx_in[j] < 0 || b.idx_in[j] >= n_u || !std::isfinite(b.centre[j])) return fail(ctx, PHYLINO_ERR_SHAPE, "transform block %d: idx_in/centre[%d]", k, j);
        for (int64_t i = 0; i < (int64_t)b.n_out * b.n_in; ++i)
            if (!std::isfinite(b.matrix[i])) return fail(ctx, PHYLINO_ERR_ARG, "transform block %d: matrix[%lld] is not finite", k, (long long)i);
        mat_off.push_back((int64_t)matrix.size());
        idx_out.insert(idx_out.end(), b.idx_out, b.idx_out + b.n_out);
        offset.insert(offset.end(), b.offset, b.offset + b.n_out);
        idx_in.insert(idx_in.end(), b.idx_in, b.idx_in + b.n_in);
        centre.insert(centre.end(), b.centre, b.centre + b.n_in);
        matrix.insert(matrix.end(), b.matrix, b.matrix + (size_t)b.n_out * b.n_in);
        row_off.push_back((int32_t)idx_out.size());
        col_off.push_back((int32_t)idx_in.size());
    }
    free_transform(ctx);
    TransformArgs &t = ctx->tf;
    cudaStream_t st = ctx->stream;
    CU(upload((int32_t **)&t.copy_src, src, st));
    CU(upload((double **)&t.copy_const, cst, st));
    CU(upload((int32_t **)&t.row_off, row_off, st));
    CU(upload((int32_t **)&t.col_off, col_off, st));
    CU(upload((int64_t **)&t.mat_off, mat_off, st));
    CU(upload((int32_t **)&t.idx_out, idx_out, st));
    CU(upload((int32_t **)&t.idx_in, idx_in, st));
    CU(upload((double **)&t.offset, offset, st));
    CU(upload((double **)&t.centre, centre, st));
    CU(upload((double **)&t.matrix, matrix, st));
    CU(cudaStreamSynchronize(st));
    t.n_params = NP; t.n_u = n_u; t.n_blocks = n_blocks;
    ctx->tf_src = src; ctx->tf_const = cst; ctx->tf_row_off = row_off; ctx->tf_col_off = col_off;
    ctx->tf_mat_off = mat_off; ctx->tf_idx_out = idx_out; ctx->tf_idx_in = idx_in;
    ctx->tf_offset = offset; ctx->tf_centre = centre; ctx->tf_matrix = matrix;
    ctx->n_u = n_u;
    ctx->have_tf = true;
    ctx->err.clear();
    return PHYLINO_OK;
}

int64_t phylino_param_width(const phylino_ctx *ctx) { return ctx && ctx->have_model ? param_width(ctx) : 0; }

static void free_functions(phylino_ctx *ctx)
{
    FinalizeArgs &f = ctx->fin;
    cudaFree((void *)f.fn_offset); cudaFree((void *)f.fn_term_off); cudaFree((void *)f.term_coef);
    cudaFree((void *)f.term_fac_off); cudaFree((void *)f.fac_idx); cudaFree((void *)f.fac_pow);
    f.fn_offset = nullptr; f.fn_term_off = nullptr; f.term_coef = nullptr;
    f.term_fac_off = nullptr; f.fac_idx = nullptr; f.fac_pow = nullptr;
    f.n_functions = 0;
}

phylino_status phylino_set_functions(phylino_ctx *ctx, int n_functions, const phylino_function *functions)
{
    if (!ctx) return PHYLINO_ERR_ARG;
    if (!ctx->have_model) return fail(ctx, PHYLINO_ERR_STATE, "phylino_set_model must come before phylino_set_functions");
    if (n_functions < 0 || (n_functions > 0 && !functions)) return fail(ctx, PHYLINO_ERR_ARG, "n_functions = %d with NULL functions", n_functions);
    if (ctx->max_block_idx >= ctx->n_params + n_functions)
        return fail(ctx, PHYLINO_ERR_STATE, "a prior block names function %d: clear the blocks before removing functions", ctx->max_block_idx - ctx->n_params);
    std::vector<double> offset, coef;
    std::vector<int32_t> term_off(1, 0), fac_off(1, 0), fidx, fpow;
    for (int k = 0; k < n_functions; ++k) {
        const phylino_function &fn = functions[k];
        if (!std::isfinite(fn.offset)) return fail(ctx, PHYLINO_ERR_ARG, "function %d: offset is not finite", k);
        if (fn.n_terms < 0 || (fn.n_terms > 0 && !fn.terms)) return fail(ctx, PHYLINO_ERR_ARG, "function %d: n_terms = %d with NULL terms", k, fn.n_terms);
        offset.push_back(fn.offset);
        for (int m = 0; m < fn.n_terms; ++m) {
            const phylino_monomial &t = fn.terms[m];
            if (!std::isfinite(t.coef)) return fail(ctx, PHYLINO_ERR_ARG, "function %d term %d: coef is not finite", k, m);
            if (t.n_factors < 0 || t.n_factors > PHYLINO_MAX_FACTORS) return fail(ctx, PHYLINO_ERR_SHAPE, "function %d term %d: n_factors = %d not in 0..%d", k, m, t.n_factors, PHYLINO_MAX_FACTORS);
            if (t.n_factors > 0 && (!t.idx || !t.power)) return fail(ctx, PHYLINO_ERR_ARG, "function %d term %d: NULL idx or power", k, m);
            for (int i = 0; i < t.n_factors; ++i) {
                if (t.idx[i] < 0 || t.idx[i] >= ctx->n_params) return fail(ctx, PHYLINO_ERR_SHAPE, "function %d term %d: idx[%d] = %d out of range", k, m, i, t.idx[i]);
                if (t.power[i] < -PHYLINO_MAX_POWER || t.power[i] > PHYLINO_MAX_POWER) return fail(ctx, PHYLINO_ERR_SHAPE, "function %d term %d: power[%d] = %d out of range", k, m, i, t.power[i]);
                fidx.push_back(t.idx[i]);
                fpow.push_back(t.power[i]);
            }
            coef.push_back(t.coef);
            fac_off.push_back((int32_t)fidx.size());
        }
        term_off.push_back((int32_t)coef.size());
    }
    DeviceGuard g(ctx->device);
    CU(cudaStreamSynchronize(ctx->stream));
    free_functions(ctx);
    if (n_functions > 0) {
        FinalizeArgs &f = ctx->fin;
        cudaStream_t st = ctx->stream;
        /* never empty: a function without terms, a term without factors are legal */
        if (coef.empty()) coef.push_back(0.0);
        if (fidx.empty()) { fidx.push_back(0); fpow.push_back(0); }
        CU(upload((double **)&f.fn_offset, offset, st));
        CU(upload((int32_t **)&f.fn_term_off, term_off, st));
        CU(upload((double **)&f.term_coef, coef, st));
        CU(upload((int32_t **)&f.term_fac_off, fac_off, st));
        CU(upload((int32_t **)&f.fac_idx, fidx, st));
        CU(upload((int32_t **)&f.fac_pow, fpow, st));
        CU(cudaStreamSynchronize(st));
        f.n_functions = n_functions;
    }
    ctx->err.clear();
    return PHYLINO_OK;
}

phylino_status phylino_set_prior_blocks(phylino_ctx *ctx, int n_blocks, const phylino_prior_block *blocks)
{
    if (!ctx) return PHYLINO_ERR_ARG;
    if (!ctx->have_model) return fail(ctx, PHYLINO_ERR_STATE, "phylino_set_model must come before phylino_set_prior_blocks");
    if (n_blocks < 0 || (n_blocks > 0 && !blocks)) return fail(ctx, PHYLINO_ERR_ARG, "n_blocks = %d with NULL blocks", n_blocks);
    std::vector<int32_t> off(1, 0), idx;
    std::vector<int64_t> moff;
    std::vector<double> mean, inv;
    for (int k = 0; k < n_blocks; ++k) {
        const phylino_prior_block &b = blocks[k];
        if (b.n < 1 || b.n > PHYLINO_MAX_BLOCK) return fail(ctx, PHYLINO_ERR_SHAPE, "block %d: n = %d not in 1..%d", k, b.n, PHYLINO_MAX_BLOCK);
        if (!b.idx || !b.mean || !b.inv_cov) return fail(ctx, PHYLINO_ERR_ARG, "block %d: NULL array", k);
        for (int i = 0; i < b.n; ++i) {
            if (b.idx[i] < 0 || b.idx[i] >= ctx->n_params + ctx->fin.n_functions)
                return fail(ctx, PHYLINO_ERR_SHAPE, "block %d: idx[%d] = %d out of range (%d parameters, %d functions)", k, i, b.idx[i], ctx->n_params, ctx->fin.n_functions);
            if (!std::isfinite(b.mean[i])) return fail(ctx, PHYLINO_ERR_ARG, "block %d: mean[%d] is not finite", k, i);
        }
        for (int64_t i = 0; i < (int64_t)b.n * b.n; ++i)
            if (!std::isfinite(b.inv_cov[i])) return fail(ctx, PHYLINO_ERR_ARG, "block %d: inv_cov[%lld] is not finite", k, (long long)i);
        moff.push_back((int64_t)inv.size());
        idx.insert(idx.end(), b.idx, b.idx + b.n);
        mean.insert(mean.end(), b.mean, b.mean + b.n);
        inv.insert(inv.end(), b.inv_cov, b.inv_cov + (size_t)b.n * b.n);
        off.push_back((int32_t)idx.size());
    }
    DeviceGuard g(ctx->device);
    CU(cudaStreamSynchronize(ctx->stream));
    FinalizeArgs &f = ctx->fin;
    cudaFree((void *)f.blk_off); cudaFree((void *)f.blk_moff); cudaFree((void *)f.blk_idx);
    cudaFree((void *)f.blk_mean); cudaFree((void *)f.blk_inv);
    f.blk_off = nullptr; f.blk_moff = nullptr; f.blk_idx = nullptr; f.blk_mean = nullptr; f.blk_inv = nullptr;
    f.n_blocks = 0;
    ctx->max_block_idx = -1;
    if (n_blocks > 0) {
        for (int32_t i : idx) ctx->max_block_idx = std::max(ctx->max_block_idx, i);
        cudaStream_t st = ctx->stream;
        CU(upload((int32_t **)&f.blk_off, off, st));
        CU(upload((int64_t **)&f.blk_moff, moff, st));
        CU(upload((int32_t **)&f.blk_idx, idx, st));
        CU(upload((double **)&f.blk_mean, mean, st));
        CU(upload((double **)&f.blk_inv, inv, st));
        CU(cudaStreamSynchronize(st));
        f.n_blocks = n_blocks;
    }
    ctx->err.clear();
    return PHYLINO_OK;
}

int64_t phylino_total_bins(const phylino_ctx *ctx) { return ctx && ctx->have_model ? ctx->total_bins : 0; }

int64_t phylino_total_events(const phylino_ctx *ctx)
{
    int64_t t = 0;
    if (ctx) for (const auto &d : ctx->ds) if (d.loaded) t += d.n;
    return t;
}

phylino_status phylino_set_tuning(phylino_ctx *ctx, int unit_events, int chunk_groups, int max_warps)
{
    if (!ctx) return PHYLINO_ERR_ARG;
    if (unit_events < 0 || chunk_groups < 0 || max_warps < 0) return fail(ctx, PHYLINO_ERR_ARG, "negative tuning value");
    ctx->unit_events = unit_events;
    ctx->chunk_groups = chunk_groups;
    ctx->max_warps = max_warps;
    return PHYLINO_OK;
}

phylino_status phylino_set_energy_correction_mode(phylino_ctx *ctx, int mode)
{
    if (!ctx) return PHYLINO_ERR_ARG;
    if (!ctx->have_model) return fail(ctx, PHYLINO_ERR_STATE, "phylino_set_model must come before phylino_set_energy_correction_mode");
    if (mode != 0 && mode != 1) return fail(ctx, PHYLINO_ERR_ARG, "mode %d not 0 or 1", mode);
    if (mode == 1 && !ctx->fin.staged)
        return fail(ctx, PHYLINO_ERR_SHAPE, "the bin-level correction needs total_bins <= %d", FIN_STAGE_MAX_BINS);
    ctx->ec_mode = mode;
    ctx->grad_plan_state = 0;
    ctx->fused_warps = 0;               /* the threshold tables of the small-batch kernel change size */
    ctx->fused_cache.clear();
    return PHYLINO_OK;
}

phylino_status phylino_set_flux_model(phylino_ctx *ctx, int dataset, int n_par, const int32_t *idx_par, double lo,
                                      double width)
{
    if (!ctx) return PHYLINO_ERR_ARG;
    if (!ctx->have_model) return fail(ctx, PHYLINO_ERR_STATE, "phylino_set_model must come before phylino_set_flux_model");
    if (dataset < 0 || dataset >= ctx->n_datasets) return fail(ctx, PHYLINO_ERR_SHAPE, "dataset %d not in 0..%d", dataset, ctx->n_datasets - 1);
    if (n_par < 0 || n_par > PHYLINO_MAX_BLOCK) return fail(ctx, PHYLINO_ERR_SHAPE, "n_par = %d not in 0..%d", n_par, PHYLINO_MAX_BLOCK);
    if (n_par > 0) {
        if (!idx_par) return fail(ctx, PHYLINO_ERR_ARG, "NULL idx_par");
        if (!std::isfinite(lo) || !(width > 0.0) || !std::isfinite(width)) return fail(ctx, PHYLINO_ERR_ARG, "fine grid: lo must be finite, width finite > 0");
        if (!ctx->fin.staged) return fail(ctx, PHYLINO_ERR_SHAPE, "a flux model needs total_bins <= %d", FIN_STAGE_MAX_BINS);
        for (int j = 0; j < n_par; ++j)
            if (idx_par[j] < 0 || idx_par[j] >= ctx->n_params) return fail(ctx, PHYLINO_ERR_SHAPE, "idx_par[%d] = %d out of range", j, idx_par[j]);
    }
    ctx->fm_idx[dataset].assign(idx_par, idx_par + n_par);
    ctx->fm_lo[dataset] = lo;
    ctx->fm_width[dataset] = width;
    std::vector<int32_t> off(ctx->n_datasets + 1, 0), idx;
    std::vector<double> grid((size_t)ctx->n_datasets * 2, 0.0);
    for (int d = 0; d < ctx->n_datasets; ++d) {
        idx.insert(idx.end(), ctx->fm_idx[d].begin(), ctx->fm_idx[d].end());
        off[d + 1] = (int32_t)idx.size();
        grid[2 * d] = ctx->fm_lo[d];
        grid[2 * d + 1] = ctx->fm_width[d];
    }
    DeviceGuard g(ctx->device);
    CU(cudaStreamSynchronize(ctx->stream));
    FinalizeArgs &f = ctx->fin;
    cudaFree((void *)f.fm_off); cudaFree((void *)f.fm_idx); cudaFree((void *)f.fm_grid);
    f.fm_off = nullptr; f.fm_idx = nullptr; f.fm_grid = nullptr;
    CU(upload((int32_t **)&f.fm_off, off, ctx->stream));
    CU(upload((int32_t **)&f.fm_idx, idx, ctx->stream));
    CU(upload((double **)&f.fm_grid, grid, ctx->stream));
    CU(cudaStreamSynchronize(ctx->stream));
    f.have_fm = idx.empty() ? 0 : 1;
    ctx->err.clear();
    return PHYLINO_OK;
}

phylino_status phylino_set_schedule(phylino_ctx *ctx, int mode)
{
    if (!ctx) return PHYLINO_ERR_ARG;
    if (mode < 0 || mode > 2) return fail(ctx, PHYLINO_ERR_ARG, "schedule %d not in 0..2", mode);
    ctx->schedule = mode;
    return PHYLINO_OK;
}

phylino_status phylino_reserve(phylino_ctx *ctx, int max_points)
{
    phylino_status s = check_ready(ctx, max_points, nullptr, nullptr);
    if (s != PHYLINO_OK && !(s == PHYLINO_ERR_ARG && ctx && max_points > 0)) return s;   /* no buffers to check here */
    if (max_points == 0) return PHYLINO_OK;
    DeviceGuard g(ctx->device);
    if ((s = ensure_acc(ctx, max_points)) != PHYLINO_OK) return s;
    const int64_t width = std::max<int64_t>(ctx->n_params, param_width(ctx));
    if ((s = ensure_stage(ctx, (int64_t)max_points * (width + ctx->total_bins) + ctx->total_bins)) != PHYLINO_OK) return s;
    const int64_t need = (int64_t)max_points * ctx->n_params;
    if (ctx->have_tf && need > ctx->theta_capacity) {
        CU(cudaStreamSynchronize(ctx->stream));
        cudaFree(ctx->d_theta); ctx->d_theta = nullptr; ctx->theta_capacity = 0;
        CU(cudaMalloc((void **)&ctx->d_theta, need * sizeof(double)));
        ctx->theta_capacity = need;
    }
    /* the buffers of the consumers and of the cached path, so that "allocates nothing, never synchronises" holds for
     * every DEVICE entry point and not only for spectra / nll / expectation:
     *   d_work   batch + NLLs of phylino_nll_gradient (2 W + 1 <= max_points) and phylino_ordering_scan
     *            (n_grid <= max_points), the Poisson norms of phylino_draw_pseudo_data, the 2 W + 2 doubles of
     *            phylino_variable_metric_step (N <= W);
     *   d_mu     the expectations of phylino_nll_ensemble;
     *   d_plan   the largest plan a cached batch of max_points points can have, V + V S + C + P (S + 1) <= P (2 S + 3);
     *   accumulators for the V (S + 1) <= P (S + 1) / 2 rows of a cached batch (V <= P / 2 or the batch runs dense);
     *   the structural plan of the central-difference batch, if caching is on now and the batch fits. */
    {
        const int64_t W = param_width(ctx), S = ctx->n_terms;
        const int64_t work = std::max<int64_t>((int64_t)max_points * (W + 1), std::max<int64_t>(ctx->total_bins, 2 * W + 2));
        if ((s = ensure_work(ctx, work)) != PHYLINO_OK) return s;
        const int64_t mu_need = (int64_t)max_points * ctx->total_bins;
        if (mu_need > ctx->mu_capacity) {
            CU(cudaStreamSynchronize(ctx->stream));
            cudaFree(ctx->d_mu); ctx->d_mu = nullptr; ctx->mu_capacity = 0;
            CU(cudaMalloc((void **)&ctx->d_mu, mu_need * sizeof(double)));
            ctx->mu_capacity = mu_need;
        }
        const int64_t plan_need = (int64_t)max_points * (2 * S + 3);
        if (plan_need > ctx->plan_capacity) {
            CU(cudaStreamSynchronize(ctx->stream));
            cudaFree(ctx->d_plan); ctx->d_plan = nullptr; ctx->plan_capacity = 0;
            CU(cudaMalloc((void **)&ctx->d_plan, plan_need * sizeof(int32_t)));
            ctx->plan_capacity = plan_need;
        }
        const int64_t rows = ((int64_t)max_points * (S + 1) + 1) / 2;
        if (rows > max_points && rows < (1ll << 30) && (s = ensure_acc(ctx, (int)rows)) != PHYLINO_OK) return s;
        if (ctx->caching && !ctx->have_tf && W > 0 && 2 * W + 1 <= max_points) gradient_plan(ctx, (int)W);
    }
    /* everything else a first call would set up with a synchronisation: the occupancy of the kernels, and the
     * single-launch kernel's edge-first unit order (a function of the store alone at the default unit length) */
    for (int P = 1; P <= std::min(max_points, FUSED_MAX_POINTS); P *= 2) {
        SpectraArgs a{};
        fill_datasets(ctx, a);
        if ((s = fill_batch(ctx, a, P, nullptr)) != PHYLINO_OK) return s;
    }
    {
        SpectraArgs a{};
        fill_datasets(ctx, a);
        if ((s = fill_batch(ctx, a, max_points, nullptr)) != PHYLINO_OK) return s;
    }
    ctx->err.clear();
    return PHYLINO_OK;
}

phylino_status phylino_set_caching(phylino_ctx *ctx, int on)
{
    if (!ctx) return PHYLINO_ERR_ARG;
    ctx->caching = on != 0;
    return PHYLINO_OK;
}

phylino_status phylino_last_plan(const phylino_ctx *ctx, int64_t *virtual_points, int64_t *classes)
{
    if (!ctx || !virtual_points || !classes) return PHYLINO_ERR_ARG;
    *virtual_points = ctx->last_virtual_points;
    *classes = ctx->last_classes;
    return PHYLINO_OK;
}

phylino_status phylino_last_small_phase(phylino_ctx *ctx, double *fraction_host)
{
    if (!ctx || !fraction_host) return PHYLINO_ERR_ARG;
    *fraction_host = 0.0;
    const int P = ctx->last_points;
    if (!ctx->have_model || P <= 0 || !ctx->d_small) return PHYLINO_OK;
    DeviceGuard g(ctx->device);
    const int n_groups = (P + 31) / 32, D = ctx->n_datasets;
    std::vector<unsigned char> flags((size_t)n_groups * D);
    CU(cudaMemcpyAsync(flags.data(), ctx->d_small, flags.size(), cudaMemcpyDeviceToHost, ctx->stream));
    CU(cudaStreamSynchronize(ctx->stream));
    double small = 0.0, total = 0.0;
    for (int gi = 0; gi < n_groups; ++gi) {
        const double np = std::min(32, P - 32 * gi);
        for (int d = 0; d < D; ++d) {
            const double w = np * (double)ctx->ds[d].n;
            total += w;
            if (flags[(size_t)gi * D + d]) small += w;
        }
    }
    *fraction_host = total > 0.0 ? small / total : 0.0;
    return PHYLINO_OK;
}

phylino_status phylino_last_medium_phase(phylino_ctx *ctx, double *fraction_host)
{
    if (!ctx || !fraction_host) return PHYLINO_ERR_ARG;
    *fraction_host = 0.0;
    const int P = ctx->last_points;
    if (!ctx->have_model || P <= 0 || !ctx->d_med || ctx->last_fused) return PHYLINO_OK;   /* the single-launch kernel has no such form */
    DeviceGuard g(ctx->device);
    unsigned long long n = 0;
    CU(cudaMemcpyAsync(&n, ctx->d_med, sizeof n, cudaMemcpyDeviceToHost, ctx->stream));
    CU(cudaStreamSynchronize(ctx->stream));
    double total = 0.0;
    for (int d = 0; d < ctx->n_datasets; ++d) total += (double)ctx->ds[d].n_pad * P;
    *fraction_host = total > 0.0 ? std::min(1.0, (double)n / total) : 0.0;
    return PHYLINO_OK;
}

phylino_status phylino_set_timing(phylino_ctx *ctx, int on)
{
    if (!ctx) return PHYLINO_ERR_ARG;
    DeviceGuard g(ctx->device);
    if (on && !ctx->ev[0])
        for (auto &e : ctx->ev) CU(cudaEventCreate(&e));
    ctx->timing = on != 0;
    return PHYLINO_OK;
}

phylino_status phylino_last_kernel_ms(phylino_ctx *ctx, float *ms)
{
    if (!ctx || !ms) return PHYLINO_ERR_ARG;
    if (!ctx->timing) return fail(ctx, PHYLINO_ERR_STATE, "phylino_set_timing(ctx, 1) has not been called");
    DeviceGuard g(ctx->device);
    CU(cudaEventSynchronize(ctx->ev[3]));
    for (int i = 0; i < 3; ++i) CU(cudaEventElapsedTime(ms + i, ctx->ev[i], ctx->ev[i + 1]));
    return PHYLINO_OK;
}

int64_t phylino_launch_count(const phylino_ctx *ctx) { return ctx ? ctx->launches : 0; }

const char *phylino_last_error(const phylino_ctx *ctx) { return ctx ? ctx->err.c_str() : ""; }

phylino_status phylino_launch_floor(phylino_ctx *ctx, int reps, double *us_per_call_host)
{
    if (!ctx || !us_per_call_host || reps < 1) return PHYLINO_ERR_ARG;
    DeviceGuard g(ctx->device);
    CU(cudaStreamSynchronize(ctx->stream));
    CU(run_launch_floor(reps, ctx->stream, us_per_call_host));
    ctx->launches += reps + 1;
    return PHYLINO_OK;
}

phylino_status phylino_hbm_read_floor(phylino_ctx *ctx, int64_t bytes, int reps, double *us_host)
{
    if (!ctx || !us_host || reps < 1 || bytes < 16 || bytes > ((int64_t)1 << 36)) return PHYLINO_ERR_ARG;
    DeviceGuard g(ctx->device);
    CU(cudaStreamSynchronize(ctx->stream));
    CU(run_hbm_read_floor((size_t)bytes, reps, ctx->stream, us_host));
    ctx->launches += reps + 2;
    return PHYLINO_OK;
}

phylino_status phylino_peak_fp64(phylino_ctx *ctx, int iters, double *dfma_per_s_host)
{
    if (!ctx || !dfma_per_s_host || iters < 1) return PHYLINO_ERR_ARG;
    DeviceGuard g(ctx->device);
    CU(run_peak_fp64(iters, ctx->stream, dfma_per_s_host));
    ctx->launches += 2;
    return PHYLINO_OK;
}

} // extern "C"
