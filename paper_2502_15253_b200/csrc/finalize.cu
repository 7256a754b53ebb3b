/*
 * finalize.cu -- SURVEY.md 8(a) rows a5-a7: fixed-point accumulators -> fp64 spectra, expectation
 * assembly, and the Poisson half-deviance + Gaussian-prior reduction.
 *
 *   mu[p,d,b] = eps_d norm_d f_db H[p,d,b] + sum_k r_dk s_dkb T_dkb
 *   nll[p]    = sum_{d,b} dev(n, mu) + 1/2 sum_j ((theta_j - mean_j)/sigma_j)^2
 *   dev(n,mu) = mu - n + n ln(n/mu)   (Eq. 3 over the saturated model of :96 Eq. 8; R9, R10)
 *
 * One CTA per parameter point.  Every thread sums a fixed strided subset of the bins and of the
 * priors, the warps combine by a fixed shuffle tree and warp 0 adds the warp totals in index
 * order: the result is bitwise reproducible.  The kernel re-zeroes the accumulators it reads so
 * the next call needs no memset launch.
 *
 * Component mode (cross-point caching): the spectra kernel summed, per
 * energy-scale class and distinct mass splitting, W[b] = sum_e w_e and C[b] = sum_e w_e g(h x_e);
 * here H[p,b] = P0(p) W[b] + sum_k A_k(p) C_k[b] -- the histogram is affine in the amplitudes
 * (Eq. 1; the paper's own "caching").  Cells are shared between points, so
 * the caller clears them after this kernel.
 */
#include <algorithm>

#include "devmath.cuh"

namespace phylino {

namespace {

constexpr int FIN_THREADS = 128;

__device__ __forceinline__ double half_deviance(double n, double mu)
{
    if (n != n || mu != mu) return __longlong_as_double(0x7ff8000000000000ll);
    if (mu < 0.0) return __longlong_as_double(0x7ff0000000000000ll);
    if (n > 0.0) {
        if (mu == 0.0) return __longlong_as_double(0x7ff0000000000000ll);
        return mu - n + n * log(n / mu);
    }
    if (n == 0.0) return mu;
    return __longlong_as_double(0x7ff8000000000000ll);     /* negative counts are not data */
}

/* this thread's share of the prior terms of one point: a fixed strided subset of the parameters and
 * of the rows of every correlated block */
__device__ __forceinline__ double prior_part(const FinalizeArgs &a, const double *theta)
{
    double part = 0.0;
    if (a.prior_mean && a.prior_sigma) {
        /* uncorrelated Gaussian priors (Eq. 6), constants dropped (R9) */
        for (int j = threadIdx.x; j < a.n_params; j += FIN_THREADS) {
            double sg = a.prior_sigma[j];
            if (!(sg > 0.0) || sg > 1.79769313486231570e308) continue;
            double z = (theta[j] - a.prior_mean[j]) / sg;
            part += 0.5 * z * z;
        }
    }

    /* correlated blocks: thread i takes rows i, i + FIN_THREADS, ... of every block */
    for (int k = 0; k < a.n_blocks; ++k) {
        const int o = a.blk_off[k], n = a.blk_off[k + 1] - o;
        const double *M = a.blk_inv + a.blk_moff[k];
        for (int i = threadIdx.x; i < n; i += FIN_THREADS) {
            const double di = theta[a.blk_idx[o + i]] - a.blk_mean[o + i];
            double row = 0.0;
            for (int j = 0; j < n; ++j)
                row = fma(M[(size_t)i * n + j], theta[a.blk_idx[o + j]] - a.blk_mean[o + j], row);
            part += 0.5 * di * row;
        }
    }

    return part;
}

template <int MODE>   /* 0 = spectra H, 1 = expectation mu, 2 = NLL */
__global__ void __launch_bounds__(FIN_THREADS) finalize_kernel(const __grid_constant__ FinalizeArgs a)
{
    /* launched as a programmatic dependent of the spectra kernel: wait for its accumulators */
    asm volatile("griddepcontrol.wait;" ::: "memory");
    const int p = blockIdx.x;
    const double *theta = a.params + (size_t)p * a.n_params;
    const size_t row = (size_t)p * a.total_bins;
    double part = 0.0;
    double A[MAX_TERMS] = {0.0, 0.0, 0.0}, P0 = 1.0;
    bool bad = false;
    if (a.comp) {
        double dm2[MAX_TERMS], asum = 0.0, half = 0.0;
        osc_terms(a.osc, theta, A, dm2);
        for (int k = 0; k < a.n_terms; ++k) { asum += fabs(A[k]); half += A[k]; }
        P0 = 1.0 - 0.5 * half;
        bad = !(asum <= 3.0);                               /* as the setup kernel's per-point check */
    }

    for (int g = threadIdx.x; g < a.total_bins; g += FIN_THREADS) {
        const int d = a.bin_ds[g];
        double H;
        unsigned fl = 0;
        if (a.comp) {
            const int32_t *rows = a.pt_comp + (size_t)p * (a.n_terms + 1);
            const size_t c0 = (size_t)rows[0] * a.total_bins + g;
            fl = a.flags[c0];
            H = P0 * ((double)a.acc[c0] * a.inv_scale[d]);
            for (int k = 0; k < a.n_terms; ++k) {
                const size_t ck = (size_t)rows[k + 1] * a.total_bins + g;
                fl |= a.flags[ck];
                H = fma(A[k], (double)a.acc[ck] * a.inv_scale[d], H);
            }
            if (fl || bad) fl = FLAG_NAN;
        } else {
            long long q = a.acc[row + g];
            fl = a.flags[row + g];
            if (q) a.acc[row + g] = 0;
            if (fl) a.flags[row + g] = 0;
            H = (double)q * a.inv_scale[d];                 /* 2^-e: exact scaling */
        }
        if (fl) {
            if ((fl & FLAG_NAN) || ((fl & FLAG_PINF) && (fl & FLAG_NINF)))
                H = __longlong_as_double(0x7ff8000000000000ll);
            else
                H = __longlong_as_double((fl & FLAG_PINF) ? 0x7ff0000000000000ll : 0xfff0000000000000ll);
        }
        if (MODE == 0) {
            a.hist[row + g] = H;
        } else {
            double eps = a.idx_signorm[d] >= 0 ? theta[a.idx_signorm[d]] : 1.0;
            double f = a.idx_flux[g] >= 0 ? theta[a.idx_flux[g]] : 1.0;
            double mu = eps * a.norm[d] * f * H;
            const int nb = a.n_bkg[d];
            for (int k = 0; k < nb; ++k) {
                int ir = a.idx_rate[d * a.max_bkg + k];
                int is = a.idx_shape[(size_t)k * a.total_bins + g];
                double r = ir >= 0 ? theta[ir] : 1.0;
                double s = is >= 0 ? theta[is] : 1.0;
                mu += r * s * a.tmpl[(size_t)k * a.total_bins + g];
            }
            if (MODE == 1) a.hist[row + g] = mu;
            else part += half_deviance(a.data[g], mu);
        }
    }
    if (MODE != 2) return;

    part += prior_part(a, theta);

    __shared__ double wsum[FIN_THREADS / 32];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) part += __shfl_xor_sync(0xffffffffu, part, o);
    if ((threadIdx.x & 31) == 0) wsum[threadIdx.x >> 5] = part;
    __syncthreads();
    if (threadIdx.x == 0) {
        double s = 0.0;
#pragma unroll
        for (int i = 0; i < FIN_THREADS / 32; ++i) s += wsum[i];
        a.nll[p] = s;
    }
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

cudaError_t launch_ensemble(const FinalizeArgs &a, int E, cudaStream_t st)
{
    if (a.P <= 0 || E <= 0) return cudaSuccess;
    /* enough CTAs to fill the chip a few times over, at least 4 experiments per warp */
    int slices = (int)std::min<long long>((E + 4 * ENS_WARPS - 1) / (4 * ENS_WARPS), std::max(1, 4 * 148 * 8 / a.P));
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
    cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = pdl ? 1 : 0;
    if (mode == 2) return cudaLaunchKernelEx(&cfg, finalize_kernel<2>, a);
    if (mode == 1) return cudaLaunchKernelEx(&cfg, finalize_kernel<1>, a);
    return cudaLaunchKernelEx(&cfg, finalize_kernel<0>, a);
}

} // namespace phylino
