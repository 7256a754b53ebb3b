/*
 * finalize.cu -- SURVEY.md 8(a) rows a5-a7: fixed-point accumulators -> fp64 spectra, expectation
 * assembly, and the Poisson half-deviance + Gaussian-prior reduction.
 *
 *   mu[p,d,b] = eps_d norm_d f_db H[p,d,b] + sum_k r_dk s_dkb T_dkb
 *   nll[p]    = sum_{d,b} dev(n, mu) + 1/2 sum_j ((theta_j - mean_j)/sigma_j)^2
 *   dev(n,mu) = mu - n + n ln(n/mu)   (Eq. 3 over the saturated model of :96 Eq. 8; R9, R10)
 *
 * One CTA per parameter point, launched as a programmatic dependent of the spectra kernel: everything that
 * does not need the histograms (signal multipliers, background sums, priors -- most of the table look-ups and
 * of the instruction footprint) is done BEFORE the wait for the spectra grid, while the events are still being
 * walked; after it only the accumulators are read, one log per bin taken and the sums formed (finalize.cuh).
 * Every thread sums a fixed strided subset of the bins and of the priors, the warps combine by a fixed shuffle
 * tree and warp 0 adds the warp totals in index order: the result is bitwise reproducible.  The kernel
 * re-zeroes the accumulators it reads so the next call needs no memset launch.
 *
 * Component mode (cross-point caching): the spectra kernel summed, per
 * energy-scale class and distinct mass splitting, W[b] = sum_e w_e and C[b] = sum_e w_e g(h x_e);
 * here H[p,b] = P0(p) W[b] + sum_k A_k(p) C_k[b] -- the histogram is affine in the amplitudes
 * (Eq. 1; the paper's own "caching").  Cells are shared between points, so
 * the caller clears them after this kernel.
 */
#include <algorithm>

#include "finalize.cuh"

namespace phylino {

namespace {

template <int MODE>   /* 0 = spectra H, 1 = expectation mu, 2 = NLL, 3 = clear only */
__global__ void __launch_bounds__(FIN_THREADS) finalize_kernel(const __grid_constant__ FinalizeArgs a)
{
    extern __shared__ double stage[];                   /* [3 x total_bins] if a.staged */
    __shared__ double wsum[FIN_THREADS / 32];
    FinPre pre;
    /* a programmatic dependent of the spectra kernel: this part runs while the events are still being walked
     * (the parameters and model tables were complete before the spectra kernel let its dependents go) */
    finalize_pre<MODE>(a, blockIdx.x, a.staged ? stage : nullptr, pre);
    if (a.staged) __syncthreads();
    asm volatile("griddepcontrol.wait;" ::: "memory");  /* the accumulators of the whole spectra grid are in */
    finalize_post<MODE>(a, blockIdx.x, a.staged ? stage : nullptr, pre, wsum);   /* ec_mode implies staged (api.cu) */
    if (a.reset_counter && blockIdx.x == 0 && threadIdx.x == 0) *a.reset_counter = 0u;
}

/* Pseudo-experiment ensembles: nll[p, e] for E observed-count vectors
 * against the SAME expectations mu[p, .] (written by finalize_kernel<1>).  One CTA per (point, slice of
 * experiments): the CTA forms the point's prior term once, then every warp takes experiments
 * e = slice start + warp, + ENS_WARPS, ...; lanes stride the bins, fixed shuffle tree => reproducible. */
constexpr int ENS_WARPS = FIN_THREADS / 32;

__global__ void __launch_bounds__(FIN_THREADS) ensemble_kernel(const __grid_constant__ FinalizeArgs a, int E,
                                                               int e_per_cta)
{
    const int p = blockIdx.x, lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const double *theta = a.params + (size_t)p * a.n_params;
    const double *mu = a.hist + (size_t)p * a.total_bins;
    __shared__ double wsum[ENS_WARPS];
    double part = prior_part(a, theta);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) part += __shfl_xor_sync(0xffffffffu, part, o);
    if (lane == 0) wsum[warp] = part;
    __syncthreads();
    double prior = 0.0;
#pragma unroll
    for (int i = 0; i < ENS_WARPS; ++i) prior += wsum[i];
    const int e0 = blockIdx.y * e_per_cta, e1 = min(E, e0 + e_per_cta);
    for (int e = e0 + warp; e < e1; e += ENS_WARPS) {
        const double *n = a.data + (size_t)e * a.total_bins;
        double dev = 0.0;
        for (int g = lane; g < a.total_bins; g += 32) dev += half_deviance(n[g], mu[g]);
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) dev += __shfl_xor_sync(0xffffffffu, dev, o);
        if (lane == 0) a.nll[(size_t)p * E + e] = dev + prior;
    }
}

} // namespace

cudaError_t launch_ensemble(const FinalizeArgs &a, int E, int sm_count, cudaStream_t st)
{
    if (a.P <= 0 || E <= 0) return cudaSuccess;
    /* enough CTAs to fill the chip a few times over, at least 4 experiments per warp */
    int slices = (int)std::min<long long>((E + 4 * ENS_WARPS - 1) / (4 * ENS_WARPS), std::max(1, 4 * sm_count * 8 / a.P));
    slices = std::max(1, std::min(slices, 65535));
    const int e_per_cta = (E + slices - 1) / slices;
    ensemble_kernel<<<dim3(a.P, (E + e_per_cta - 1) / e_per_cta), FIN_THREADS, 0, st>>>(a, E, e_per_cta);
    return cudaGetLastError();
}

cudaError_t launch_finalize(const FinalizeArgs &a, int mode, cudaStream_t st, bool pdl)
{
    if (a.P <= 0) return cudaSuccess;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(a.P);
    cfg.blockDim = dim3(FIN_THREADS);
    cfg.dynamicSmemBytes = a.staged ? (size_t)3 * a.total_bins * sizeof(double) : 0;
    cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = pdl ? 1 : 0;
    if (mode == 3) return cudaLaunchKernelEx(&cfg, finalize_kernel<3>, a);
    if (mode == 2) return cudaLaunchKernelEx(&cfg, finalize_kernel<2>, a);
    if (mode == 1) return cudaLaunchKernelEx(&cfg, finalize_kernel<1>, a);
    return cudaLaunchKernelEx(&cfg, finalize_kernel<0>, a);
}

} // namespace phylino
