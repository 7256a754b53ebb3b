/*
 * spectra.cu -- the batched oscillation-weight + histogram kernel (
 * PAPER.md:177 signal step 1, :183 "the most time-demanding computational step").
 *
 * Work split.  The event store of every dataset is cut into tiles of EV_PER_CTA consecutive
 * E_vis-sorted events, the batch into chunks of `points_per_cta` parameter points.  The
 * (chunk, tile) units, chunk-major, are dealt out as equal contiguous ranges to a persistent
 * grid of (#SM x resident CTAs) CTAs: no tail wave, and a CTA stays inside one (chunk, dataset)
 * "context" for many tiles.  Inside a context thread t owns a contiguous slice of the events,
 * keeps K_EV of them at a time in registers (x = L/E in fp64, E_vis, w) and walks the chunk's
 * points over them; the per-point quantities come from shared memory as warp-wide broadcasts.
 *
 * Binning (row a3).  For one point the map v -> E' = fma(fma(a2,v,a1),v,a0) is non-decreasing over
 * the fp32 values of a dataset (checked per point, see build_context), so bin(E'(v)) >= b  <=>
 * v >= T[b] with T[b] the smallest fp32 value whose E' reaches edges[b].  T is found by bisection
 * with the SAME fp64 fma sequence, hence the fp32 comparison v >= T[b] decides exactly what the
 * fp64 comparison E' >= edges[b] decides: bit-exact bins for 2 fp32 compares per thread and tile
 * instead of 2 DFMA + 2 DSETP per event and point.  Points that fail the monotonicity check take
 * the per-event fp64 path.
 *
 * Histogram (rows a4, a5).  Events are sorted, so a thread's K_EV events -- and its events in the
 * following tiles -- stay in ONE bin for a long run.  The thread keeps (bin, fp64 run total, the
 * fp32 interval of that bin) per point in shared memory and only adds to it while the run lasts.
 * When the run ends (or the context does) the total is converted once to 64-bit fixed point and
 * added to the (point, bin) accumulator with an integer RED -- warp-aggregated by shuffles at
 * context end.  Integer addition is associative: the result does not depend on which CTA or
 * warp arrives first, i.e. bitwise reproducible with no float atomics anywhere.
 */
#include "devmath.cuh"

namespace phylino {

namespace {

constexpr unsigned FULL = 0xffffffffu;

template <int S> struct RecLayout {
    static constexpr int H = 0;              /* half-turn coefficients h_k                       */
    static constexpr int A = S;              /* amplitudes A_k                                   */
    static constexpr int E = 2 * S;          /* energy scale a0, a1, a2                          */
    static constexpr int BAD = 2 * S + 3;    /* 1.0: point left the fixed-point domain           */
    static constexpr int SAFE_LO = 2 * S + 4;/* fp32 interval on which the threshold table holds */
    static constexpr int SAFE_HI = 2 * S + 5;
    static constexpr int SIZE = 2 * S + 6;
};

/* per (point, thread) run state */
struct __align__(16) Run {
    double acc;     /* fp64 total of the current run                                   */
    float  lo, hi;  /* the run's bin as an fp32 interval [lo, hi) of E_vis; lo=+inf: none */
};

__device__ __forceinline__ long long warp_sum_ll(long long v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(FULL, v, o);
    return v;
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

__device__ __forceinline__ void red_add(const SpectraArgs &a, int p, int cell_bin, long long q, unsigned fl)
{
    size_t cell = (size_t)p * a.total_bins + cell_bin;
    if (q) atomicAdd((unsigned long long *)a.acc + cell, (unsigned long long)q);
    if (fl) atomicOr(a.flags + cell, fl);
}

/* Add every lane's (key, q) to the accumulators of point p, one RED per distinct key. */
__device__ __forceinline__ void warp_flush(const SpectraArgs &a, int p, int key, long long q, unsigned fl,
                                           int lane)
{
    int key0 = __shfl_sync(FULL, key, 0);
    if (__all_sync(FULL, key == key0)) {
        if (key0 < 0) return;
        q = warp_sum_ll(q);
        fl = __reduce_or_sync(FULL, fl);
        if (lane == 0) red_add(a, p, key0, q, fl);
        return;
    }
    unsigned todo = __ballot_sync(FULL, key >= 0);
    while (todo) {
        int leader = __ffs(todo) - 1;
        int kk = __shfl_sync(FULL, key, leader);
        bool mine = key == kk;
        unsigned grp = __ballot_sync(FULL, mine);
        long long s = warp_sum_ll(mine ? q : 0ll);
        unsigned f = __reduce_or_sync(FULL, mine ? fl : 0u);
        if (lane == leader) red_add(a, p, kk, s, f);
        todo &= ~grp;
    }
}

/* largest b with thr[b] <= v, -1 unless thr[0] <= v < thr[B] (thr non-decreasing) */
__device__ __forceinline__ int table_bin(const float *thr, int B, float v)
{
    if (!(v >= thr[0]) || !(v < thr[B])) return -1;
    int lo = 0, hi = B;
    while (hi - lo > 1) {
        int mid = (lo + hi) >> 1;
        if (thr[mid] <= v) lo = mid; else hi = mid;
    }
    return lo;
}

/* smallest fp32 v in [safe_lo, safe_hi] (positive, normal) with E'(v) >= edge, +inf if none */
__device__ float threshold_search(double a0, double a1, double a2, double edge, float safe_lo, float safe_hi)
{
    const float inf = __int_as_float(0x7f800000);
    if (!(safe_lo <= safe_hi)) return inf;
    if (!(escale(a0, a1, a2, (double)safe_hi) >= edge)) return inf;
    if (escale(a0, a1, a2, (double)safe_lo) >= edge) return safe_lo;
    int lo = __float_as_int(safe_lo), hi = __float_as_int(safe_hi);   /* E'(lo) < edge <= E'(hi) */
    while (hi - lo > 1) {
        int mid = lo + ((hi - lo) >> 1);
        if (escale(a0, a1, a2, (double)__int_as_float(mid)) >= edge) hi = mid; else lo = mid;
    }
    return __int_as_float(hi);
}

/* bin of one event at one point: the threshold table where it is proven, else the fp64 map */
template <int S>
__device__ __forceinline__ int event_bin(const double *rec, const float *thr, const double *edges, int B, float v)
{
    using R = RecLayout<S>;
    if (v >= (float)rec[R::SAFE_LO] && v <= (float)rec[R::SAFE_HI]) return table_bin(thr, B, v);
    return bin_search(edges, B, escale(rec[R::E], rec[R::E + 1], rec[R::E + 2], (double)v));
}

template <int S> __device__ __forceinline__ double survival(const double *h, const double *A, double x)
{
    double p = 1.0;
#pragma unroll
    for (int k = 0; k < S; ++k) p = fma(-A[k], sin2_halfturns(h[k], x), p);
    return p;
}

/* shared-memory carve-up, identical for every context of a launch */
template <int S> struct Smem {
    double *edges;   /* [max_bins + 1]                */
    double *recs;    /* [ppc][RecLayout<S>::SIZE]      */
    Run    *run;     /* [ppc][CTA_THREADS]             */
    int    *key;     /* [ppc][CTA_THREADS]             */
    float  *thr;     /* [n_tables][max_bins + 1]       */
    __device__ Smem(unsigned char *base, int max_bins, int ppc)
    {
        edges = reinterpret_cast<double *>(base);
        recs = edges + ((max_bins + 2) & ~1);
        run = reinterpret_cast<Run *>(recs + ppc * RecLayout<S>::SIZE);
        key = reinterpret_cast<int *>(run + ppc * CTA_THREADS);
        thr = reinterpret_cast<float *>(key + ppc * CTA_THREADS);
    }
    static size_t bytes(int max_bins, int ppc, int n_tables)
    {
        return (size_t)((max_bins + 2) & ~1) * 8 + (size_t)ppc * RecLayout<S>::SIZE * 8 +
               (size_t)ppc * CTA_THREADS * (sizeof(Run) + sizeof(int)) + (size_t)n_tables * (max_bins + 1) * 4;
    }
};

/* Per-point records, threshold tables and empty run states of one (chunk, dataset) context. */
template <int S>
__device__ void build_context(const SpectraArgs &a, const DatasetDev &ds, const Smem<S> &sm, int p_begin, int np)
{
    using R = RecLayout<S>;
    const int B = ds.n_bins, tid = threadIdx.x;
    const float inf = __int_as_float(0x7f800000);
    for (int i = tid; i <= B; i += CTA_THREADS) sm.edges[i] = ds.edges[i];
    if (tid < np) {
        const double *theta = a.params + (size_t)(p_begin + tid) * a.n_params;
        double A[MAX_TERMS], dm2[MAX_TERMS];
        osc_terms(a.osc, theta, A, dm2);
        double *r = sm.recs + tid * R::SIZE;
        double asum = 0.0;
#pragma unroll
        for (int k = 0; k < S; ++k) {
            r[R::H + k] = halfturn_coeff(dm2[k]);
            r[R::A + k] = A[k];
            asum += fabs(A[k]);
        }
        /* |P_ee| <= 1 + sum|A_k| <= 4 keeps every partial sum inside the fixed-point range */
        r[R::BAD] = (asum <= 3.0) ? 0.0 : 1.0;
        double a0 = ds.idx_a[0] >= 0 ? theta[ds.idx_a[0]] : 0.0;
        double a1 = ds.idx_a[1] >= 0 ? theta[ds.idx_a[1]] : 1.0;
        double a2 = ds.idx_a[2] >= 0 ? theta[ds.idx_a[2]] : 0.0;
        r[R::E] = a0; r[R::E + 1] = a1; r[R::E + 2] = a2;
        float slo, shi;
        if (!a.per_point_binning) {
            slo = -inf; shi = inf;          /* E' = v exactly: the table holds for every float */
        } else {
            /* E'(v) computed with the two fma is non-decreasing over the fp32 values of
             * [v_pos_min, v_max] if the Horner inner value t = a2 v + a1 is positive and the
             * derivative a1 + 2 a2 v exceeds 2^-20 t at both ends (both are linear in v): between
             * fp32 neighbours the exact increase then outweighs the rounding of t 2^8-fold
             * (DESIGN.md "Bit-exact binning with fp32 thresholds"). */
            double vl = (double)ds.v_pos_min, vh = (double)ds.v_max;
            double t_lo = fma(a2, vl, a1), t_hi = fma(a2, vh, a1);
            double g_lo = fma(2.0 * a2, vl, a1), g_hi = fma(2.0 * a2, vh, a1);
            double tm = fmax(t_lo, t_hi) * 0x1p-20;
            bool ok = t_lo > 0.0 && t_hi > 0.0 && g_lo >= tm && g_hi >= tm && fabs(a0) < 1.0e300 &&
                      t_hi < 1.0e300 && ds.v_pos_min >= 1.17549435e-38f && ds.v_pos_min <= ds.v_max;
            slo = ok ? ds.v_pos_min : inf;
            shi = ok ? ds.v_max : -inf;
        }
        r[R::SAFE_LO] = (double)slo;
        r[R::SAFE_HI] = (double)shi;
    }
    __syncthreads();
    const int n_tab = a.per_point_binning ? np : 1;
    for (int e = tid; e < n_tab * (B + 1); e += CTA_THREADS) {
        int tab = e / (B + 1), b = e - tab * (B + 1);
        const double *r = sm.recs + tab * R::SIZE;
        float t;
        if (!a.per_point_binning) t = __double2float_ru(sm.edges[b]);    /* v >= edge <=> v >= ru(edge) */
        else t = threshold_search(r[R::E], r[R::E + 1], r[R::E + 2], sm.edges[b], (float)r[R::SAFE_LO],
                                  (float)r[R::SAFE_HI]);
        sm.thr[tab * (a.max_bins + 1) + b] = t;
    }
    __syncthreads();
}

template <int S>
__device__ void flush_context(const SpectraArgs &a, const DatasetDev &ds, const Smem<S> &sm, int p_begin, int np)
{
    using R = RecLayout<S>;
    const int tid = threadIdx.x, lane = tid & 31;
    for (int pi = 0; pi < np; ++pi) {
        int k = sm.key[pi * CTA_THREADS + tid];
        double s = sm.run[pi * CTA_THREADS + tid].acc;
        bool bad = sm.recs[pi * R::SIZE + R::BAD] != 0.0;
        unsigned fl = 0;
        long long q = k >= 0 ? to_fixed(s, ds.fx_scale, bad, fl) : 0ll;
        warp_flush(a, p_begin + pi, k >= 0 ? ds.bin_off + k : -1, q, fl, lane);
    }
}

template <int S>
__global__ void __launch_bounds__(CTA_THREADS, 2) spectra_kernel(const __grid_constant__ SpectraArgs a)
{
    using R = RecLayout<S>;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const Smem<S> sm(smem_raw, a.max_bins, a.points_per_cta);
    const int tid = threadIdx.x;
    const float inf = __int_as_float(0x7f800000);

    /* This CTA's contiguous range of virtual (chunk, tile) units, chunk-major.  Virtual tiles are the
     * real ones with blocks of TILE_BLOCK tiles dealt out in a stride permutation, so that a
     * CTA's range is made of blocks from all over the energy range: the sparse high-energy tail
     * (many short runs, the slower general path below) is shared by many CTAs instead of ending
     * up in one.  A context never leaves its block, so results do not depend on the grid size. */
    const int nb = (a.n_tiles + TILE_BLOCK - 1) / TILE_BLOCK;
    const long long per_chunk = (long long)nb * TILE_BLOCK;
    const long long U = per_chunk * a.n_chunks;
    long long u = (long long)blockIdx.x * U / gridDim.x;
    const long long u_end = (long long)(blockIdx.x + 1) * U / gridDim.x;
    int ctx_c = -1, ctx_d = -1;

#pragma unroll 1
    while (u < u_end) {
        /* ---- one context: chunk c, dataset d, tiles [tile0, tile0 + n_iter) ---- */
        const int c = (int)(u / per_chunk);
        const int vt = (int)(u - (long long)c * per_chunk);
        const int off = vt % TILE_BLOCK;
        const int tile0 = (int)(((long long)(vt / TILE_BLOCK) * a.block_stride) % nb) * TILE_BLOCK + off;
        if (tile0 >= a.n_tiles) {               /* the ragged last block has no such tile */
            u += TILE_BLOCK - off;
            continue;
        }
        int d = 0;
#pragma unroll 1
        for (int i = 1; i < a.n_datasets; ++i)
            if (tile0 >= a.ds[i].tile_begin) d = i;
        const DatasetDev &ds = a.ds[d];
        const int ds_tile_end = d + 1 < a.n_datasets ? a.ds[d + 1].tile_begin : a.n_tiles;
        const int n_iter = (int)min((long long)min(ds_tile_end - tile0, TILE_BLOCK - off), u_end - u);
        const int p_begin = c * a.points_per_cta;
        const int np = min(a.points_per_cta, a.P - p_begin);
        const int B = ds.n_bins;
        if (c != ctx_c || d != ctx_d) {        /* records and threshold tables of (chunk, dataset) */
            __syncthreads();                   /* everybody is done with the previous tables */
            build_context<S>(a, ds, sm, p_begin, np);
            ctx_c = c;
            ctx_d = d;
        }

        /* Thread t owns the contiguous slice [t * K_EV * n_iter, (t+1) * K_EV * n_iter) of the
         * context's events and walks it K_EV events per iteration: a bin edge then ends the run of
         * ONE thread (the one whose slice it falls in), not of all 256. */
        const size_t slice0 = ((size_t)(tile0 - ds.tile_begin) * CTA_THREADS + (size_t)tid * n_iter) * K_EV;

        /* open every point's run at the bin of the slice's first event */
        {
            const float vf = __ldg(ds.v + slice0);
            for (int pi = 0; pi < np; ++pi) {
                const double *r = sm.recs + pi * R::SIZE;
                const float *thr = sm.thr + (a.per_point_binning ? pi : 0) * (a.max_bins + 1);
                const bool safe = vf >= (float)r[R::SAFE_LO] && vf <= (float)r[R::SAFE_HI];
                const int b = safe ? table_bin(thr, B, vf) : -1;
                Run z;
                z.acc = 0.0;
                z.lo = b >= 0 ? thr[b] : inf;
                z.hi = b >= 0 ? thr[b + 1] : inf;
                sm.run[pi * CTA_THREADS + tid] = z;
                sm.key[pi * CTA_THREADS + tid] = b;
            }
        }

#pragma unroll 1
        for (int it = 0; it < n_iter; ++it) {
            /* ---- K_EV consecutive events of the slice ---- */
            const size_t e0 = slice0 + (size_t)it * K_EV;
            double x[K_EV], w[K_EV];
            float v[K_EV];
            {
                const double2 *xp = reinterpret_cast<const double2 *>(ds.x + e0);
                const float4 *vp = reinterpret_cast<const float4 *>(ds.v + e0);
                const float4 *wp = reinterpret_cast<const float4 *>(ds.w + e0);
#pragma unroll
                for (int j = 0; j < K_EV / 2; ++j) {
                    double2 t = __ldg(xp + j);
                    x[2 * j] = t.x; x[2 * j + 1] = t.y;
                }
#pragma unroll
                for (int j = 0; j < K_EV / 4; ++j) {
                    float4 tv = __ldg(vp + j), tw = __ldg(wp + j);
                    v[4 * j] = tv.x; v[4 * j + 1] = tv.y; v[4 * j + 2] = tv.z; v[4 * j + 3] = tv.w;
                    w[4 * j] = tw.x; w[4 * j + 1] = tw.y; w[4 * j + 2] = tw.z; w[4 * j + 3] = tw.w;
                }
            }

#pragma unroll 1
            for (int pi = 0; pi < np; ++pi) {
                const double *r = sm.recs + pi * R::SIZE;
                double h[S], A[S];
#pragma unroll
                for (int k = 0; k < S; ++k) { h[k] = r[R::H + k]; A[k] = r[R::A + k]; }
                Run st = sm.run[pi * CTA_THREADS + tid];

                /* the store is sorted: v[0] <= ... <= v[K_EV-1] (NaN padding, last, fails the test) */
                if (v[0] >= st.lo && v[K_EV - 1] < st.hi) {
                    /* rows a2 + a4: all K_EV events inside the current run's bin */
                    double s = 0.0;
#pragma unroll
                    for (int j = 0; j < K_EV; ++j) s = fma(w[j], survival<S>(h, A, x[j]), s);
                    sm.run[pi * CTA_THREADS + tid].acc = st.acc + s;
                } else {
                    /* A run ends inside these events (or none is open, or events are out of range).
                     * Same arithmetic with the same instruction-level parallelism first, then a
                     * light sequential walk over the sorted events that closes runs as bin edges
                     * go by; finished runs go straight to the accumulators. */
                    const float *thr = sm.thr + (a.per_point_binning ? pi : 0) * (a.max_bins + 1);
                    const bool bad = r[R::BAD] != 0.0;
                    const float safe_lo = (float)r[R::SAFE_LO], safe_hi = (float)r[R::SAFE_HI];
                    double pee[K_EV];
#pragma unroll
                    for (int j = 0; j < K_EV; ++j) pee[j] = survival<S>(h, A, x[j]);
                    int cur = sm.key[pi * CTA_THREADS + tid];
                    double s = st.acc;
                    float lo = st.lo, hi = st.hi;
#pragma unroll
                    for (int j = 0; j < K_EV; ++j) {
                        if (!(v[j] >= lo && v[j] < hi)) {
                            /* leave the current run: close it, open the one of this event's bin */
                            if (cur >= 0) {
                                unsigned fl;
                                long long q = to_fixed(s, ds.fx_scale, bad, fl);
                                red_add(a, p_begin + pi, ds.bin_off + cur, q, fl);
                            }
                            s = 0.0;
                            if (cur >= 0 && cur + 1 < B && v[j] >= hi && v[j] < thr[cur + 2]) {
                                /* sorted events: nearly always the next bin; hi < +inf here means the
                                 * run was on the table, and v[j] < thr[cur+2] <= safe_hi keeps it there */
                                cur += 1;
                                lo = hi;
                                hi = thr[cur + 1];
                            } else {
                                cur = event_bin<S>(r, thr, sm.edges, B, v[j]);
                                const bool on_table = cur >= 0 && v[j] >= safe_lo && v[j] <= safe_hi;
                                lo = on_table ? thr[cur] : inf;     /* lo = +inf: re-examined at the next event */
                                hi = on_table ? thr[cur + 1] : inf;
                            }
                        }
                        if (cur >= 0) s = fma(w[j], pee[j], s);
                    }
                    Run nw;
                    nw.acc = s; nw.lo = lo; nw.hi = hi;
                    sm.run[pi * CTA_THREADS + tid] = nw;
                    sm.key[pi * CTA_THREADS + tid] = cur;
                }
            }
        }
        flush_context<S>(a, ds, sm, p_begin, np);
        u += n_iter;
    }
}

template <int S>
cudaError_t launch_t(const SpectraArgs &a, int sm_count, cudaStream_t st)
{
    size_t smem = Smem<S>::bytes(a.max_bins, a.points_per_cta, a.per_point_binning ? a.points_per_cta : 1);
    cudaError_t e = cudaFuncSetAttribute(spectra_kernel<S>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    /* ask for the full shared-memory carve-out so that two CTAs of up to ~110 KB are resident */
    e = cudaFuncSetAttribute(spectra_kernel<S>, cudaFuncAttributePreferredSharedMemoryCarveout,
                             cudaSharedmemCarveoutMaxShared);
    if (e != cudaSuccess) return e;
    int per_sm = 0;
    e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, spectra_kernel<S>, CTA_THREADS, smem);
    if (e != cudaSuccess) return e;
    if (per_sm < 1) return cudaErrorLaunchOutOfResources;
    /* persistent grid: exactly the CTAs that are resident at once, each with an equal range of units */
    const long long units = (long long)a.n_tiles * a.n_chunks;
    const int grid = (int)(units < (long long)sm_count * per_sm ? units : (long long)sm_count * per_sm);
    spectra_kernel<S><<<grid, CTA_THREADS, smem, st>>>(a);
    return cudaGetLastError();
}

} // namespace

size_t spectra_smem_bytes(int S, int max_bins, int ppc, bool per_point)
{
    return S == 2 ? Smem<2>::bytes(max_bins, ppc, per_point ? ppc : 1)
                  : Smem<3>::bytes(max_bins, ppc, per_point ? ppc : 1);
}

cudaError_t launch_spectra(const SpectraArgs &a, int S, int sm_count, cudaStream_t st)
{
    if (a.n_tiles <= 0 || a.P <= 0 || sm_count <= 0) return cudaSuccess;
    return S == 2 ? launch_t<2>(a, sm_count, st) : launch_t<3>(a, sm_count, st);
}

/* ---- diagnostic: bin index of every event at every point (bit-exact parity of row a3) ----
 * One CTA per (256 events, point): it builds the point's threshold table exactly as the hot kernel
 * does and assigns bins with the same event_bin(), so the test covers the production binning. */
namespace {
__global__ void __launch_bounds__(CTA_THREADS) event_bins_kernel(const __grid_constant__ SpectraArgs a, int d,
                                                                 const int32_t *perm, long long n,
                                                                 long long ev_off, long long total_events,
                                                                 int32_t *bins)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const Smem<2> sm(smem_raw, a.max_bins, 1);
    const DatasetDev &ds = a.ds[d];
    const int p = blockIdx.y;
    build_context<2>(a, ds, sm, p, 1);
    long long i = (long long)blockIdx.x * CTA_THREADS + threadIdx.x;
    if (i >= n) return;
    bins[(size_t)p * total_events + ev_off + perm[i]] = event_bin<2>(sm.recs, sm.thr, sm.edges, ds.n_bins, ds.v[i]);
}
} // namespace

cudaError_t launch_event_bins(const SpectraArgs &a, int d, const int32_t *perm, long long n, long long ev_off,
                              long long total_events, int32_t *bins, cudaStream_t st)
{
    if (n <= 0 || a.P <= 0) return cudaSuccess;
    dim3 grid((unsigned)((n + CTA_THREADS - 1) / CTA_THREADS), a.P);
    size_t smem = Smem<2>::bytes(a.max_bins, 1, 1);
    cudaError_t e = cudaFuncSetAttribute(event_bins_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    event_bins_kernel<<<grid, CTA_THREADS, smem, st>>>(a, d, perm, n, ev_off, total_events, bins);
    return cudaGetLastError();
}

} // namespace phylino
