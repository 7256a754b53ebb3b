/*
 * finalize.cuh -- the likelihood stage of one parameter point as device functions of one 128-thread CTA
 * (SURVEY.md 8(a) rows a5-a7), called by finalize_kernel and ensemble_kernel (finalize.cu).
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

/* entry idx of a prior block: a parameter, or a constrained FUNCTION of the parameters (R29):
 * offset + the terms in order, a term = coef x its factors in order, a factor = theta^|power| by repeated
 * multiplication, multiplied in or divided out -- the sequence phylino.h states, in plain (unfused) arithmetic */
__device__ __forceinline__ double constrained_value(const FinalizeArgs &a, const double *theta, int idx)
{
    if (idx < a.n_params) return theta[idx];
    const int f = idx - a.n_params;
    PHYLINO_ASSERT(f >= 0 && f < a.n_functions);
    double v = a.fn_offset[f];
    for (int m = a.fn_term_off[f]; m < a.fn_term_off[f + 1]; ++m) {
        double term = a.term_coef[m];
        for (int i = a.term_fac_off[m]; i < a.term_fac_off[m + 1]; ++i) {
            const double x = theta[a.fac_idx[i]];
            const int pw = a.fac_pow[i], n = pw < 0 ? -pw : pw;
            if (n == 0) continue;
            double q = x;
            for (int r = 1; r < n; ++r) q *= x;
            if (pw > 0) term *= q; else term /= q;
        }
        v += term;
    }
    return v;
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
            const double di = constrained_value(a, theta, a.blk_idx[o + i]) - a.blk_mean[o + i];
            double row = 0.0;
            for (int j = 0; j < n; ++j)
                row = fma(M[(size_t)i * n + j], constrained_value(a, theta, a.blk_idx[o + j]) - a.blk_mean[o + j], row);
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
 *   finalize_post -- H from the fixed-point accumulators, mu = m H + background, the half-deviance, the sum; with
 *                    the bin-level energy correction (ec_mode) the corrected bins C_a(f . H) in between.
 *
 * Every thread sums a fixed strided subset of the bins and of the priors, the warps combine by a fixed shuffle
 * tree and thread 0 adds the warp totals in index order: bitwise reproducible.  The accumulators are read past
 * L1 (ld.cg) and re-zeroed (dense mode), so the next call needs no memset.
 * MODE 0 = spectra H, 1 = expectation mu, 2 = NLL, 3 = only clear the accumulators. */
/* ---- PAPER.md:177 steps 2-3 on the binned spectrum, PAPER.md:129 flux model (R27, R28) ----------------
 * Smoothing: inside source bin b the density is the parabola whose integrals over three consecutive bins (b-1, b,
 * b+1; the first / last three at the ends) equal their contents -- the derivative of the cubic through the four
 * cumulative points of the triple (two bins: a straight line; one: a constant).  Content arriving in a target
 * interval of the corrected energy is the integral of that density over the interval's pre-image. */
__device__ __forceinline__ double escale_inverse(double a0, double a1, double a2, double t)
{
    const double c = t - a0;
    if (a2 == 0.0) return c / a1;
    return (2.0 * c) / (a1 + sqrt(a1 * a1 + 4.0 * a2 * c));
}

/* cumulative integral, from the first edge of the triple, of the density that belongs to source bin b */
__device__ __forceinline__ double cumulative_quadratic(int n, const double *e, const double *h, int b, double E)
{
    if (n == 1) return h[0] / (e[1] - e[0]) * (E - e[0]);
    if (n == 2) {
        const double d1 = h[0] / (e[1] - e[0]), d1b = h[1] / (e[2] - e[1]);
        const double d2 = (d1b - d1) / (e[2] - e[0]);
        return d1 * (E - e[0]) + d2 * (E - e[0]) * (E - e[1]);
    }
    const int t0 = min(max(b - 1, 0), n - 3);
    const double *x = e + t0, *y = h + t0;
    const double f01 = y[0] / (x[1] - x[0]), f12 = y[1] / (x[2] - x[1]), f23 = y[2] / (x[3] - x[2]);
    const double f012 = (f12 - f01) / (x[2] - x[0]), f123 = (f23 - f12) / (x[3] - x[1]);
    const double f0123 = (f123 - f012) / (x[3] - x[0]);
    return f01 * (E - x[0]) + f012 * (E - x[0]) * (E - x[1]) + f0123 * (E - x[0]) * (E - x[1]) * (E - x[2]);
}

/* integral over [lo, hi) of the smoothed density of the n source bins (e, h): the bins the interval overlaps */
__device__ __forceinline__ double rebin_quadratic(int n, const double *e, const double *h, double lo, double hi)
{
    if (lo != lo || hi != hi) return __longlong_as_double(0x7ff8000000000000ll);
    /* first source bin that ends above lo */
    int b = 0, top = n;
    while (top - b > 0) {
        const int mid = (b + top) >> 1;
        if (e[mid + 1] > lo) top = mid; else b = mid + 1;
    }
    double s = 0.0;
    PHYLINO_ASSERT(b >= 0 && b <= n);
    for (; b < n && e[b] < hi; ++b) {
        const double a = fmax(lo, e[b]), z = fmin(hi, e[b + 1]);
        if (a < z) s += cumulative_quadratic(n, e, h, b, z) - cumulative_quadratic(n, e, h, b, a);
    }
    return s;
}

/* the uniform fine grid of a flux model as the `e` of the functions above would need too much memory for what it
 * is: the same formulas with e[j] = lo + j w written out */
__device__ __forceinline__ double flux_scale_of_bin(const FinalizeArgs &a, const double *theta, int d, double x_lo,
                                                    double x_hi)
{
    const int o = a.fm_off[d], n = a.fm_off[d + 1] - o;
    const double g0 = a.fm_grid[2 * d], w = a.fm_grid[2 * d + 1];
    if (x_lo != x_lo || x_hi != x_hi) return __longlong_as_double(0x7ff8000000000000ll);
    const double top = g0 + w * (double)n;
    const double lo = fmax(x_lo, g0), hi = fmin(x_hi, top);
    double s = 0.0;
    if (lo < hi) {
        int j = (int)floor((lo - g0) / w);
        j = min(max(j, 0), n - 1);
        while (j > 0 && g0 + w * (double)j > lo) --j;                   /* guard the rounding of the guess */
        while (j < n - 1 && g0 + w * (double)(j + 1) <= lo) ++j;
        for (; j < n && g0 + w * (double)j < hi; ++j) {
            const double ej = g0 + w * (double)j, ej1 = g0 + w * (double)(j + 1);
            const double lo_j = fmax(lo, ej), hi_j = fmin(hi, ej1);
            if (!(lo_j < hi_j)) continue;
            /* the triple of fine bins around j, contents theta * w, edges on the grid */
            const int t0 = n >= 3 ? min(max(j - 1, 0), n - 3) : 0;
            double e4[4], h3[3];
            const int m = min(n, 3);
            PHYLINO_ASSERT(t0 >= 0 && t0 + m <= n && j - t0 >= 0 && j - t0 < m);
            for (int i = 0; i <= m; ++i) e4[i] = g0 + w * (double)(t0 + i);
            for (int i = 0; i < m; ++i) h3[i] = theta[a.fm_idx[o + t0 + i]] * w;
            s += cumulative_quadratic(m, e4, h3, j - t0, hi_j) - cumulative_quadratic(m, e4, h3, j - t0, lo_j);
        }
    }
    const double inside = lo < hi ? hi - lo : 0.0;
    return (s + ((x_hi - x_lo) - inside)) / (x_hi - x_lo);              /* the nominal 1 outside the grid */
}

/* pre-image of edge i (0 ... n_bins) of dataset d under the dataset's energy scale at theta */
__device__ __forceinline__ double edge_preimage(const FinalizeArgs &a, const double *theta, int d, int i)
{
    const int32_t *ia = a.ds_idx_a + 3 * d;
    const double a0 = ia[0] >= 0 ? theta[ia[0]] : 0.0, a1 = ia[1] >= 0 ? theta[ia[1]] : 1.0;
    const double a2 = ia[2] >= 0 ? theta[ia[2]] : 0.0;
    return escale_inverse(a0, a1, a2, a.edges_all[a.ds_bin_off[d] + d + i]);
}

struct FinPre {
    double A[MAX_TERMS], P0;    /* component mode */
    double prior;               /* MODE 2: this thread's share */
    bool bad;
};

/* signal multiplier and background sum of global bin g of dataset d at theta.  The flux scale f is theta[idx_flux]
 * or, with a flux model on the dataset, the model's average over the bin's pre-image (R28).  ec_mode = 1: m is the
 * flux scale alone (step 2 of PAPER.md:177; the normalisation follows the bin-level correction, step 3). */
__device__ __forceinline__ void bin_model(const FinalizeArgs &a, const double *theta, int g, int d, double &m,
                                          double &bsum)
{
    const double eps = a.idx_signorm[d] >= 0 ? theta[a.idx_signorm[d]] : 1.0;
    double f = a.idx_flux[g] >= 0 ? theta[a.idx_flux[g]] : 1.0;
    if (a.have_fm && a.fm_off[d + 1] > a.fm_off[d]) {
        const int b = g - a.ds_bin_off[d];
        f = flux_scale_of_bin(a, theta, d, edge_preimage(a, theta, d, b), edge_preimage(a, theta, d, b + 1));
    }
    m = a.ec_mode ? f : eps * a.norm[d] * f;
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
            const int d = a.bin_ds[g];
            bin_model(a, theta, g, d, m, bsum);
            /* NLL of the plain (dense, per-event energy scale) path: the fixed-point scale 2^-e of the dataset goes
             * into the multiplier here -- an exact scaling, so m 2^-e q is the same double as m (q 2^-e) -- and the
             * second half of the kernel reads nothing but the accumulators (no dataset look-up behind the wait) */
            if (MODE == 2 && !a.comp && !a.ec_mode) m *= a.inv_scale[d];
            stage[g] = m;
            stage[a.total_bins + g] = bsum;
            if (MODE == 2) stage[2 * a.total_bins + g] = a.data[g];
        }
    }
    if (MODE == 2) pre.prior = prior_part(a, theta);
}

/* H of global bin g of point p from the accumulators (re-zeroed in dense mode); fl: its domain flags resolved */
__device__ __forceinline__ double load_H(const FinalizeArgs &a, int p, int g, int d, const FinPre &pre)
{
    const size_t row = (size_t)p * a.total_bins;
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
    if (fl) {
        if ((fl & FLAG_NAN) || ((fl & FLAG_PINF) && (fl & FLAG_NINF)))
            H = __longlong_as_double(0x7ff8000000000000ll);
        else
            H = __longlong_as_double((fl & FLAG_PINF) ? 0x7ff0000000000000ll : 0xfff0000000000000ll);
    }
    return H;
}

template <int MODE>
__device__ __forceinline__ void finalize_post(const FinalizeArgs &a, int p, double *stage, const FinPre &pre,
                                              double *wsum)
{
    const double *theta = a.params + (size_t)p * a.n_params;
    const size_t row = (size_t)p * a.total_bins;
    double part = 0.0;
    if (a.ec_mode && MODE != 3) {
        /* bin-level energy correction (needs the staged layout): step 2, G = f H into stage[0]; step 3, every
         * target bin integrates the smoothed G over its pre-image; then normalisation, backgrounds, deviance */
        for (int g = threadIdx.x; g < a.total_bins; g += FIN_THREADS) {
            const double H = load_H(a, p, g, a.bin_ds[g], pre);
            stage[g] = MODE == 0 ? H : stage[g] * H;
        }
        __syncthreads();
        for (int g = threadIdx.x; g < a.total_bins; g += FIN_THREADS) {
            const int d = a.bin_ds[g], off = a.ds_bin_off[d], B = a.ds_bin_off[d + 1] - off, b = g - off;
            const double Gc = rebin_quadratic(B, a.edges_all + off + d, stage + off, edge_preimage(a, theta, d, b),
                                              edge_preimage(a, theta, d, b + 1));
            if (MODE == 0) {
                a.hist[row + g] = Gc;
            } else {
                const double eps = a.idx_signorm[d] >= 0 ? theta[a.idx_signorm[d]] : 1.0;
                const double mu = eps * a.norm[d] * Gc + stage[a.total_bins + g];
                if (MODE == 1) a.hist[row + g] = mu;
                else part += half_deviance(stage[2 * a.total_bins + g], mu);
            }
        }
    } else {
        for (int g = threadIdx.x; g < a.total_bins; g += FIN_THREADS) {
            if (MODE == 2 && stage && !a.comp) {
                /* the staged multiplier carries the fixed-point scale (finalize_pre) */
                long long q = __ldcg(a.acc + row + g);
                const unsigned fl = __ldcg(a.flags + row + g);
                if (q) a.acc[row + g] = 0;
                if (fl) a.flags[row + g] = 0;
                double Hq = (double)q;
                if (fl) {
                    if ((fl & FLAG_NAN) || ((fl & FLAG_PINF) && (fl & FLAG_NINF)))
                        Hq = __longlong_as_double(0x7ff8000000000000ll);
                    else
                        Hq = __longlong_as_double((fl & FLAG_PINF) ? 0x7ff0000000000000ll : 0xfff0000000000000ll);
                }
                part += half_deviance(stage[2 * a.total_bins + g], stage[g] * Hq + stage[a.total_bins + g]);
                continue;
            }
            const int d = a.bin_ds[g];
            const double H = load_H(a, p, g, d, pre);
            if (MODE == 3) continue;
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
