/*
 * finalize.cuh -- the likelihood stage of one parameter point as a device function of one 128-thread CTA
 * (SURVEY.md 8(a) rows a5-a7), shared by finalize_kernel (finalize.cu) and by the last CTA of the
 * single-launch kernel for small batches (spectra.cu).
 *
 *   mu[p,d,b] = eps_d norm_d f_db H[p,d,b] + sum_k r_dk s_dkb T_dkb
 *   nll[p]    = sum_{d,b} dev(n, mu) + 1/2 sum_j ((theta_j - mean_j)/sigma_j)^2
 *   dev(n,mu) = mu - n + n ln(n/mu)   (Eq. 3 over the saturated model of :96 Eq. 8; R9, R10)
 */
#ifndef PHYLINO_FINALIZE_CUH
#define PHYLINO_FINALIZE_CUH

#include "devmath.cuh"

namespace phylino {

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

/* One CTA of FIN_THREADS threads, one parameter point p, in two phases around the wait for the spectra grid
 * (the kernel is its programmatic dependent, so its CTAs are resident while the events are still being walked):
 *
 *   finalize_pre  -- everything that does not need the histograms: the per-bin signal multiplier
 *                    m = eps_d norm_d f_db, the background sum sum_k r_dk s_dkb T_dkb, the observed count, the
 *                    amplitudes of component mode, this thread's share of the prior terms.  Per-bin values go
 *                    to shared memory (`stage`: 3 x total_bins doubles; NULL when the model has more than
 *                    FIN_STAGE_MAX_BINS bins: then finalize_post looks everything up itself).
 *   finalize_post -- H from the fixed-point accumulators, mu = m H + background, the half-deviance, the sum.
 *
 * Every thread sums a fixed strided subset of the bins and of the priors, the warps combine by a fixed shuffle
 * tree and thread 0 adds the warp totals in index order: bitwise reproducible.  The accumulators are read past
 * L1 (ld.cg) and re-zeroed (dense mode), so the next call needs no memset.
 * MODE 0 = spectra H, 1 = expectation mu, 2 = NLL, 3 = only clear the accumulators. */
struct FinPre {
    double A[MAX_TERMS], P0;    /* component mode */
    double prior;               /* MODE 2: this thread's share */
    bool bad;
};

/* signal multiplier and background sum of global bin g of dataset d at theta */
__device__ __forceinline__ void bin_model(const FinalizeArgs &a, const double *theta, int g, int d, double &m,
                                          double &bsum)
{
    const double eps = a.idx_signorm[d] >= 0 ? theta[a.idx_signorm[d]] : 1.0;
    const double f = a.idx_flux[g] >= 0 ? theta[a.idx_flux[g]] : 1.0;
    m = eps * a.norm[d] * f;
    bsum = 0.0;
    const int nb = a.n_bkg[d];
    for (int k = 0; k < nb; ++k) {
        const int ir = a.idx_rate[d * a.max_bkg + k];
        const int is = a.idx_shape[(size_t)k * a.total_bins + g];
        const double r = ir >= 0 ? theta[ir] : 1.0;
        const double sh = is >= 0 ? theta[is] : 1.0;
        bsum += r * sh * a.tmpl[(size_t)k * a.total_bins + g];
    }
}

template <int MODE>
__device__ __forceinline__ void finalize_pre(const FinalizeArgs &a, int p, double *stage, FinPre &pre)
{
    const double *theta = a.params + (size_t)p * a.n_params;
    pre.A[0] = pre.A[1] = pre.A[2] = 0.0;
    pre.P0 = 1.0;
    pre.prior = 0.0;
    pre.bad = false;
    if (MODE == 3) return;
    if (a.comp) {
        double dm2[MAX_TERMS], asum = 0.0, half = 0.0;
        osc_terms(a.osc, theta, pre.A, dm2);
        for (int k = 0; k < a.n_terms; ++k) { asum += fabs(pre.A[k]); half += pre.A[k]; }
        pre.P0 = 1.0 - 0.5 * half;
        pre.bad = !(asum <= 3.0);                           /* as the per-point check of the spectra stage */
    }
    if (MODE >= 1 && stage) {
        for (int g = threadIdx.x; g < a.total_bins; g += FIN_THREADS) {
            double m, bsum;
            bin_model(a, theta, g, a.bin_ds[g], m, bsum);
            stage[g] = m;
            stage[a.total_bins + g] = bsum;
            if (MODE == 2) stage[2 * a.total_bins + g] = a.data[g];
        }
    }
    if (MODE == 2) pre.prior = prior_part(a, theta);
}

template <int MODE>
__device__ __forceinline__ void finalize_post(const FinalizeArgs &a, int p, const double *stage, const FinPre &pre,
                                              double *wsum)
{
    const double *theta = a.params + (size_t)p * a.n_params;
    const size_t row = (size_t)p * a.total_bins;
    double part = 0.0;
    for (int g = threadIdx.x; g < a.total_bins; g += FIN_THREADS) {
        const int d = a.bin_ds[g];
        double H;
        unsigned fl = 0;
        if (a.comp) {
            const int32_t *rows = a.pt_comp + (size_t)p * (a.n_terms + 1);
            const size_t c0 = (size_t)rows[0] * a.total_bins + g;
            fl = __ldcg(a.flags + c0);
            H = pre.P0 * ((double)__ldcg(a.acc + c0) * a.inv_scale[d]);
            for (int k = 0; k < a.n_terms; ++k) {
                const size_t ck = (size_t)rows[k + 1] * a.total_bins + g;
                fl |= __ldcg(a.flags + ck);
                H = fma(pre.A[k], (double)__ldcg(a.acc + ck) * a.inv_scale[d], H);
            }
            if (fl || pre.bad) fl = FLAG_NAN;
        } else {
            long long q = __ldcg(a.acc + row + g);
            fl = __ldcg(a.flags + row + g);
            if (q) a.acc[row + g] = 0;
            if (fl) a.flags[row + g] = 0;
            H = (double)q * a.inv_scale[d];                 /* 2^-e: exact scaling */
        }
        if (MODE == 3) continue;
        if (fl) {
            if ((fl & FLAG_NAN) || ((fl & FLAG_PINF) && (fl & FLAG_NINF)))
                H = __longlong_as_double(0x7ff8000000000000ll);
            else
                H = __longlong_as_double((fl & FLAG_PINF) ? 0x7ff0000000000000ll : 0xfff0000000000000ll);
        }
        if (MODE == 0) {
            a.hist[row + g] = H;
        } else {
            double m, bsum, n = 0.0;
            if (stage) {
                m = stage[g];
                bsum = stage[a.total_bins + g];
                if (MODE == 2) n = stage[2 * a.total_bins + g];
            } else {
                bin_model(a, theta, g, d, m, bsum);
                if (MODE == 2) n = a.data[g];
            }
            const double mu = m * H + bsum;
            if (MODE == 1) a.hist[row + g] = mu;
            else part += half_deviance(n, mu);
        }
    }
    if (MODE != 2) return;

    part += pre.prior;

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

} // namespace phylino
#endif
