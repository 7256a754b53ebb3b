/*
 * spectra.cu -- the batched oscillation-weight + histogram kernel (
 * PAPER.md:177 signal step 1, :183 "the most time-demanding computational step").
 *
 * Work split: blockIdx.x = a tile of EV_PER_CTA consecutive E_vis-sorted events of one dataset,
 * blockIdx.y = a chunk of parameter points.  Each thread keeps K_EV consecutive events in
 * registers (x = L/E in fp64, E_vis, w) and walks the chunk's points over them, so the event
 * bytes are read once per chunk and the per-point quantities come from shared memory as
 * warp-wide broadcasts.
 *
 * Histogram stage: the events are sorted by E_vis, so the K_EV events of a thread -- and almost
 * always the 256 events of a warp -- fall into ONE bin at a given point.  A thread sums its run
 * in an fp64 register (fixed order), converts the run total once to 64-bit fixed point, the warp
 * adds the lanes' integers with shuffles when they share a bin, and one lane issues one 64-bit
 * integer RED to the (point, bin) accumulator.  Integer addition is associative, so the result
 * does not depend on the order in which warps and CTAs arrive: bitwise reproducible with no
 * float atomics anywhere.
 */
#include "devmath.cuh"

namespace phylino {

namespace {

constexpr unsigned FULL = 0xffffffffu;

template <int S> struct RecLayout {
    static constexpr int H = 0;          /* half-turn coefficients h_k          */
    static constexpr int A = S;          /* amplitudes A_k                      */
    static constexpr int E = 2 * S;      /* energy scale a0, a1, a2             */
    static constexpr int BAD = 2 * S + 3;/* 1.0 if the point left the fixed-point domain */
    static constexpr int SIZE = 2 * S + 4;
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

__device__ __forceinline__ void red_add(const SpectraArgs &a, int p, int key, long long q, unsigned fl)
{
    size_t cell = (size_t)p * a.total_bins + key;
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

template <int S, bool PERPOINT>
__global__ void __launch_bounds__(CTA_THREADS, 2) spectra_kernel(const __grid_constant__ SpectraArgs a)
{
    using R = RecLayout<S>;
    extern __shared__ double smem[];

    /* dataset of this tile (tiles of a dataset are contiguous in blockIdx.x) */
    int d = 0;
#pragma unroll 1
    for (int i = 1; i < a.n_datasets; ++i)
        if ((int)blockIdx.x >= a.ds[i].tile_begin) d = i;
    const DatasetDev &ds = a.ds[d];
    const int B = ds.n_bins;
    double *edges = smem;
    double *recs = smem + ((B + 2) & ~1);

    const int p_begin = blockIdx.y * a.points_per_cta;
    const int np = min(a.points_per_cta, a.P - p_begin);

    /* ---- prologue: edges and per-point records to shared memory ---- */
    for (int i = threadIdx.x; i <= B; i += CTA_THREADS) edges[i] = ds.edges[i];
    if ((int)threadIdx.x < np) {
        const double *theta = a.params + (size_t)(p_begin + threadIdx.x) * a.n_params;
        double A[MAX_TERMS], dm2[MAX_TERMS];
        osc_terms(a.osc, theta, A, dm2);
        double *r = recs + threadIdx.x * R::SIZE;
        double asum = 0.0;
#pragma unroll
        for (int k = 0; k < S; ++k) {
            r[R::H + k] = halfturn_coeff(dm2[k]);
            r[R::A + k] = A[k];
            asum += fabs(A[k]);
        }
        r[R::E + 0] = ds.idx_a[0] >= 0 ? theta[ds.idx_a[0]] : 0.0;
        r[R::E + 1] = ds.idx_a[1] >= 0 ? theta[ds.idx_a[1]] : 1.0;
        r[R::E + 2] = ds.idx_a[2] >= 0 ? theta[ds.idx_a[2]] : 0.0;
        /* |P_ee| <= 1 + sum|A_k| <= 4 keeps every partial sum inside the fixed-point range */
        r[R::BAD] = (asum <= 3.0) ? 0.0 : 1.0;
    }

    /* ---- this thread's K_EV consecutive events ---- */
    const int lane = threadIdx.x & 31;
    const size_t e0 = ((size_t)(blockIdx.x - ds.tile_begin) * CTA_THREADS + threadIdx.x) * K_EV;
    double x[K_EV], v[K_EV], w[K_EV];
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
    __syncthreads();

    /* bins that do not depend on the point (energy scale fixed at (0,1,0): E' = v exactly) */
    int bj[K_EV];
    bool hoisted_same = true;
    if (!PERPOINT) {
#pragma unroll
        for (int j = 0; j < K_EV; ++j) {
            bj[j] = bin_search(edges, B, v[j]);
            hoisted_same &= bj[j] == bj[0];
        }
    }
    /* cached bin of the thread's first event and its edges (PERPOINT) */
    int bcur = -1;
    double lo = 0.0, hi = 0.0;

    const double scale = ds.fx_scale;

#pragma unroll 1
    for (int pi = 0; pi < np; ++pi) {
        const double *r = recs + pi * R::SIZE;
        double h[S], A[S];
#pragma unroll
        for (int k = 0; k < S; ++k) { h[k] = r[R::H + k]; A[k] = r[R::A + k]; }
        const bool bad = r[R::BAD] != 0.0;

        /* survival probability of every event at this point */
        double pee[K_EV];
#pragma unroll
        for (int j = 0; j < K_EV; ++j) {
            double p = 1.0;
#pragma unroll
            for (int k = 0; k < S; ++k) p = fma(-A[k], sin2_halfturns(h[k], x[j]), p);
            pee[j] = p;
        }

        /* SURVEY 8(a) a3 + a4: bin of every event, run total of the thread */
        int key;
        double acc = 0.0;
        bool same;
        double a0 = 0.0, a1 = 1.0, a2 = 0.0;
        if (PERPOINT) {
            a0 = r[R::E + 0]; a1 = r[R::E + 1]; a2 = r[R::E + 2];
            double e = escale(a0, a1, a2, v[0]);
            if (bcur < 0 || !(e >= lo) || !(e < hi)) {
                bcur = bin_search(edges, B, e);
                if (bcur >= 0) { lo = edges[bcur]; hi = edges[bcur + 1]; }
            }
            same = bcur >= 0;
#pragma unroll
            for (int j = 0; j < K_EV; ++j) {
                double ej = escale(a0, a1, a2, v[j]);
                same &= (ej >= lo) & (ej < hi);
            }
            key = ds.bin_off + bcur;
        } else {
            same = hoisted_same;
            key = bj[0] >= 0 ? ds.bin_off + bj[0] : -1;
        }

        if (same) {
#pragma unroll
            for (int j = 0; j < K_EV; ++j) acc = fma(w[j], pee[j], acc);
        } else {
            /* the thread's events straddle a bin edge (or some are out of range): run-length
             * accumulate, earlier runs go straight to the accumulators */
            int cur = -1;
#pragma unroll
            for (int j = 0; j < K_EV; ++j) {
                int b = PERPOINT ? bin_search(edges, B, escale(a0, a1, a2, v[j])) : bj[j];
                if (b != cur) {
                    if (cur >= 0) {
                        unsigned fl;
                        long long q = to_fixed(acc, scale, bad, fl);
                        red_add(a, p_begin + pi, ds.bin_off + cur, q, fl);
                    }
                    cur = b;
                    acc = 0.0;
                }
                acc = fma(w[j], pee[j], acc);
            }
            key = cur >= 0 ? ds.bin_off + cur : -1;
        }

        unsigned fl = 0;
        long long q = key >= 0 ? to_fixed(acc, scale, bad, fl) : 0ll;
        warp_flush(a, p_begin + pi, key, q, fl, lane);
    }
}

template <int S, bool PERPOINT>
cudaError_t launch_t(const SpectraArgs &a, int n_tiles, int max_bins, cudaStream_t st)
{
    using R = RecLayout<S>;
    size_t smem = (size_t)(((max_bins + 2) & ~1) + a.points_per_cta * R::SIZE) * sizeof(double);
    dim3 grid(n_tiles, (a.P + a.points_per_cta - 1) / a.points_per_cta);
    if (smem > 48 * 1024) {
        cudaError_t e = cudaFuncSetAttribute(spectra_kernel<S, PERPOINT>,
                                             cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
    }
    spectra_kernel<S, PERPOINT><<<grid, CTA_THREADS, smem, st>>>(a);
    return cudaGetLastError();
}

} // namespace

cudaError_t launch_spectra(const SpectraArgs &a, int n_tiles, int S, bool per_point_binning,
                           int max_bins, cudaStream_t st)
{
    if (n_tiles <= 0 || a.P <= 0) return cudaSuccess;
    if (S == 2) return per_point_binning ? launch_t<2, true>(a, n_tiles, max_bins, st)
                                         : launch_t<2, false>(a, n_tiles, max_bins, st);
    return per_point_binning ? launch_t<3, true>(a, n_tiles, max_bins, st)
                             : launch_t<3, false>(a, n_tiles, max_bins, st);
}

/* ---- diagnostic: bin index of every event at every point (bit-exact parity of a3) ---- */
namespace {
__global__ void event_bins_kernel(const __grid_constant__ EventBinsArgs a)
{
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    int p = blockIdx.y;
    if (i >= a.n) return;
    const double *theta = a.params + (size_t)p * a.n_params;
    double a0 = a.ds.idx_a[0] >= 0 ? theta[a.ds.idx_a[0]] : 0.0;
    double a1 = a.ds.idx_a[1] >= 0 ? theta[a.ds.idx_a[1]] : 1.0;
    double a2 = a.ds.idx_a[2] >= 0 ? theta[a.ds.idx_a[2]] : 0.0;
    double e = escale(a0, a1, a2, (double)a.ds.v[i]);
    a.bins[(size_t)p * a.total_events + a.ev_off + a.perm[i]] = bin_search(a.ds.edges, a.ds.n_bins, e);
}
} // namespace

cudaError_t launch_event_bins(const EventBinsArgs &a, cudaStream_t st)
{
    if (a.n <= 0 || a.P <= 0) return cudaSuccess;
    dim3 grid((unsigned)((a.n + 255) / 256), a.P);
    event_bins_kernel<<<grid, 256, 0, st>>>(a);
    return cudaGetLastError();
}

} // namespace phylino
