/*
 * consumers.cu -- on-device consumers and producers of batches: Poisson pseudo-data for
 * ensembles of pseudo-experiments, the scan of one parameter under both mass orderings
 * (Fig. 4), the central-difference gradient of the NLL.
 *
 * Pseudo-data (R26; the paper names no generator).  data[e, i] is a function of (seed, e, i, mu_i) alone:
 *   uniform  Philox4x32-10, counter (i, e, 0, 0), key = seed; u = (x0 2^21 + (x1 >> 11)) 2^-53;
 *   count    exact inversion of the Poisson distribution from its mode m = floor(mu) outwards with the pmf
 *            ratios w_{k+1} = w_k (mu / (k+1)), w_{k-1} = w_k (k / mu): Z = sum of the weights (each tail summed
 *            until a term no longer changes it), [0, Z) cut into pieces w_k in the order m, m+1, m-1, m+2, ...;
 *            the count is the piece that holds u Z.  Only +, *, / -- every operation correctly rounded and none
 *            contracted (-fmad=false), so the integers are those of any other IEEE implementation of the same
 *            sequence: the parity bar for this stage is bit-exact.
 * One thread per bin forms Z (O(sqrt mu) steps), then one thread per (experiment, bin) draws (O(sqrt mu) steps).
 */
#include "internal.h"

namespace phylino {

namespace {

__device__ __forceinline__ void philox_round(unsigned &c0, unsigned &c1, unsigned &c2, unsigned &c3, unsigned k0,
                                             unsigned k1)
{
    const unsigned hi0 = __umulhi(0xD2511F53u, c0), lo0 = 0xD2511F53u * c0;
    const unsigned hi1 = __umulhi(0xCD9E8D57u, c2), lo1 = 0xCD9E8D57u * c2;
    const unsigned n0 = hi1 ^ c1 ^ k0, n2 = hi0 ^ c3 ^ k1;
    c0 = n0; c1 = lo1; c2 = n2; c3 = lo0;
}

/* u in [0, 1) of (seed, bin, experiment) */
__device__ __forceinline__ double uniform53(unsigned long long seed, unsigned bin, unsigned experiment)
{
    unsigned c0 = bin, c1 = experiment, c2 = 0u, c3 = 0u;
    unsigned k0 = (unsigned)seed, k1 = (unsigned)(seed >> 32);
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        philox_round(c0, c1, c2, c3, k0, k1);
        k0 += 0x9E3779B9u;
        k1 += 0xBB67AE85u;
    }
    return (double)(((unsigned long long)c0 << 21) | (unsigned long long)(c1 >> 11)) * 0x1p-53;
}

/* Domain of the sampler (R26): 0 < mu <= POISSON_MAX_MU.  The walk from the mode costs O(sqrt mu) steps --
 * about 3e5 per side at the limit -- and above 2^53 the step k -> k + 1 no longer moves, so a finite value in a
 * device buffer could otherwise keep a thread busy for good.  Beyond the limit the count is NaN.  POISSON_MAX_STEPS
 * bounds every loop as well; inside the domain it is never reached (it is ten times the longest walk). */
constexpr double POISSON_MAX_MU = 1e9;
constexpr int POISSON_MAX_STEPS = 1 << 22;

__device__ double poisson_norm(double mu)
{
    if (!(mu > 0.0) || mu > POISSON_MAX_MU) return 1.0;
    const double m = floor(mu);
    double L = 0.0, R = 0.0, t = 1.0;
    int steps = 0;
    for (double k = m; k >= 1.0 && steps < POISSON_MAX_STEPS; k -= 1.0, ++steps) {
        t = t * (k / mu);
        if (L + t == L) break;
        L += t;
    }
    t = 1.0;
    steps = 0;
    for (double k = m + 1.0; steps < POISSON_MAX_STEPS; k += 1.0, ++steps) {
        t = t * (mu / k);
        if (R + t == R) break;
        R += t;
    }
    return (L + 1.0) + R;
}

__device__ double poisson_inv(double mu, double Z, double u)
{
    if (mu > POISSON_MAX_MU && mu <= 1.79769313486231570e308) return __longlong_as_double(0x7ff8000000000000ll);
    if (!(mu > 0.0) || mu > 1.79769313486231570e308) return 0.0;
    const double m = floor(mu), target = u * Z;
    double acc = 1.0, tr = 1.0, tl = 1.0, kr = m, kl = m;
    if (target < acc) return m;
    for (int steps = 0;; ++steps) {
        if (steps >= POISSON_MAX_STEPS) return kr;
        kr += 1.0;
        tr = tr * (mu / kr);
        acc += tr;
        if (target < acc) return kr;
        bool left_done = true;
        if (kl >= 1.0) {
            tl = tl * (kl / mu);
            kl -= 1.0;
            const double before = acc;
            acc += tl;
            if (target < acc) return kl;
            left_done = acc == before;
        }
        if (acc + tr == acc && left_done) return kr;    /* u Z within rounding of Z: the last piece */
    }
}

__global__ void __launch_bounds__(128) poisson_norm_kernel(const double *mu, int n, double *Z)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) Z[i] = poisson_norm(mu[i]);
}

__global__ void __launch_bounds__(128) poisson_draw_kernel(const double *mu, const double *Z, int n, int E,
                                                           unsigned long long seed, double *data)
{
    const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= (long long)n * E) return;
    const int i = (int)(t % n), e = (int)(t / n);
    data[t] = poisson_inv(mu[i], Z[i], uniform53(seed, (unsigned)i, (unsigned)e));
}

/* batch[g] = theta with theta[col] = grid[g] */
__global__ void __launch_bounds__(128) scan_batch_kernel(const double *theta, int width, int col, const double *grid,
                                                         int n_grid, double *batch)
{
    const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= (long long)n_grid * width) return;
    const int j = (int)(t % width), g = (int)(t / width);
    batch[t] = j == col ? grid[g] : theta[j];
}

/* central-difference batch (R18): row 0 = theta, rows 1 + 2j / 2 + 2j = theta +- h_j e_j */
__global__ void __launch_bounds__(128) gradient_batch_kernel(const double *theta, const double *h, int width,
                                                             double *batch)
{
    const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= (long long)(2 * width + 1) * width) return;
    const int j = (int)(t % width), row = (int)(t / width);
    double v = theta[j];
    if (row > 0 && (row - 1) / 2 == j) v = (row & 1) ? v + h[j] : v - h[j];
    batch[t] = v;
}

/* g_j = (nll(theta + h_j e_j) - nll(theta - h_j e_j)) / ((theta_j + h_j) - (theta_j - h_j)): the divisor is the
 * step actually taken in floating point */
__global__ void __launch_bounds__(128) gradient_kernel(const double *theta, const double *h, const double *nll,
                                                       int width, double *nll0, double *grad)
{
    const int j = blockIdx.x * blockDim.x + threadIdx.x;
    if (j == 0 && nll0) *nll0 = nll[0];
    if (j >= width) return;
    const double up = theta[j] + h[j], dn = theta[j] - h[j];
    grad[j] = (nll[1 + 2 * j] - nll[2 + 2 * j]) / (up - dn);
}

/* ---- one variable-metric step of the minimiser's loop (R30) ---------------------------------
 * Every sum runs over j in index order in plain (unfused) double arithmetic -- one thread per row, one thread for the
 * scalars -- so the result is a function of the inputs alone, the same bits as any other IEEE evaluation of that
 * sequence; N is a few hundred, the work is nothing beside one gradient. */
__global__ void __launch_bounds__(128) vm_matvec_kernel(const double *V, const double *x, int N, double *out)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    double s = 0.0;
    for (int j = 0; j < N; ++j) s += V[(size_t)i * N + j] * x[j];
    out[i] = s;
}

/* ab[0] = dx.dg, ab[1] = dg.vg */
__global__ void vm_scalars_kernel(const double *dx, const double *dg, const double *vg, int N, double *ab)
{
    double a = 0.0, b = 0.0;
    for (int i = 0; i < N; ++i) a += dx[i] * dg[i];
    for (int i = 0; i < N; ++i) b += dg[i] * vg[i];
    ab[0] = a;
    ab[1] = b;
}

/* V += dx dx^T / a - vg vg^T / b (+ b u u^T, u = dx / a - vg / b, where a > b); nothing unless a > 0 and b > 0 */
__global__ void __launch_bounds__(128) vm_update_kernel(double *V, const double *dx, const double *vg, const double *ab,
                                                        int N)
{
    const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= (long long)N * N) return;
    const double a = ab[0], b = ab[1];
    if (!(a > 0.0 && b > 0.0)) return;
    const int i = (int)(t / N), j = (int)(t % N);
    double v = V[t];
    v += dx[i] * dx[j] / a;
    v -= vg[i] * vg[j] / b;
    if (a > b) {
        const double ui = dx[i] / a - vg[i] / b, uj = dx[j] / a - vg[j] / b;
        v += b * ui * uj;
    }
    V[t] = v;
}

/* direction = -V grad (s = V grad), out[0] = 1/2 grad.s, out[1] = 1 if the update was skipped */
__global__ void __launch_bounds__(128) vm_finish_kernel(const double *grad, const double *s, const double *ab, int N,
                                                        double *direction, double *out)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < N) direction[i] = -s[i];
    if (i == 0) {
        double e = 0.0;
        for (int k = 0; k < N; ++k) e += grad[k] * s[k];
        out[0] = 0.5 * e;
        out[1] = (ab && !(ab[0] > 0.0 && ab[1] > 0.0)) ? 1.0 : 0.0;
    }
}

} // namespace

/* work: DEVICE [2 N + 2] scratch (vg | s | a, b) */
cudaError_t launch_variable_metric_step(int N, double *V, const double *dx, const double *dg, const double *grad,
                                        double *direction, double *out, double *work, cudaStream_t st)
{
    if (N <= 0) return cudaSuccess;
    double *vg = work, *s = work + N, *ab = work + 2 * (size_t)N;
    const int blocks = (N + 127) / 128;
    if (dx && dg) {
        vm_matvec_kernel<<<blocks, 128, 0, st>>>(V, dg, N, vg);
        vm_scalars_kernel<<<1, 1, 0, st>>>(dx, dg, vg, N, ab);
        vm_update_kernel<<<(unsigned)(((long long)N * N + 127) / 128), 128, 0, st>>>(V, dx, vg, ab, N);
    }
    vm_matvec_kernel<<<blocks, 128, 0, st>>>(V, grad, N, s);
    vm_finish_kernel<<<blocks, 128, 0, st>>>(grad, s, (dx && dg) ? ab : nullptr, N, direction, out);
    return cudaGetLastError();
}

cudaError_t launch_pseudo_data(const double *mu, double *Z, int n, int E, unsigned long long seed, double *data,
                               cudaStream_t st)
{
    if (n <= 0 || E <= 0) return cudaSuccess;
    poisson_norm_kernel<<<(n + 127) / 128, 128, 0, st>>>(mu, n, Z);
    const long long total = (long long)n * E;
    poisson_draw_kernel<<<(unsigned)((total + 127) / 128), 128, 0, st>>>(mu, Z, n, E, seed, data);
    return cudaGetLastError();
}

cudaError_t launch_scan_batch(const double *theta, int width, int col, const double *grid, int n_grid, double *batch,
                              cudaStream_t st)
{
    const long long total = (long long)n_grid * width;
    if (total <= 0) return cudaSuccess;
    scan_batch_kernel<<<(unsigned)((total + 127) / 128), 128, 0, st>>>(theta, width, col, grid, n_grid, batch);
    return cudaGetLastError();
}

cudaError_t launch_gradient_batch(const double *theta, const double *h, int width, double *batch, cudaStream_t st)
{
    const long long total = (long long)(2 * width + 1) * width;
    if (width <= 0) return cudaSuccess;
    gradient_batch_kernel<<<(unsigned)((total + 127) / 128), 128, 0, st>>>(theta, h, width, batch);
    return cudaGetLastError();
}

cudaError_t launch_gradient(const double *theta, const double *h, const double *nll, int width, double *nll0,
                            double *grad, cudaStream_t st)
{
    if (width <= 0) return cudaSuccess;
    gradient_kernel<<<(width + 127) / 128, 128, 0, st>>>(theta, h, nll, width, nll0, grad);
    return cudaGetLastError();
}

} // namespace phylino
