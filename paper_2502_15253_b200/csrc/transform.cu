/*
 * transform.cu -- the transformation layer between the minimiser's parameters u and the model parameters
 * theta ("A transformation layer applies the covariance of any changed model parameter within the
 * calculation of the likelihood"; "the 9 polynomial coefficients can be expressed by 7 independent
 * parameters"):
 *
 *   theta_j = u[copy_src[j]]   (copy_const[j] where copy_src[j] < 0),  then for every block, in order,
 *   theta[idx_out[i]] = offset[i] + sum_j matrix[i][j] (u[idx_in[j]] - centre[j])
 *
 * One CTA per parameter point.  The sum runs over j in index order with fma -- the same correctly rounded
 * sequence as host_transform() in api.cu, so the host entry points (which transform on the host, where the
 * caching plan needs theta) and the device ones produce identical bits.
 */
#include "internal.h"

namespace phylino {

namespace {

constexpr int TF_THREADS = 128;

__global__ void __launch_bounds__(TF_THREADS) transform_kernel(const __grid_constant__ TransformArgs a)
{
    const int p = blockIdx.x;
    const double *u = a.u + (size_t)p * a.n_u;
    double *theta = a.theta + (size_t)p * a.n_params;
    for (int j = threadIdx.x; j < a.n_params; j += TF_THREADS) {
        const int s = a.copy_src[j];
        theta[j] = s >= 0 ? u[s] : a.copy_const[j];
    }
    for (int k = 0; k < a.n_blocks; ++k) {
        __syncthreads();                                    /* later blocks overwrite earlier ones */
        const int ro = a.row_off[k], n_out = a.row_off[k + 1] - ro;
        const int co = a.col_off[k], n_in = a.col_off[k + 1] - co;
        const double *M = a.matrix + a.mat_off[k];
        for (int i = threadIdx.x; i < n_out; i += TF_THREADS) {
            double acc = a.offset[ro + i];
            for (int j = 0; j < n_in; ++j)
                acc = fma(M[(size_t)i * n_in + j], u[a.idx_in[co + j]] - a.centre[co + j], acc);
            theta[a.idx_out[ro + i]] = acc;
        }
    }
}

} // namespace

cudaError_t launch_transform(const TransformArgs &a, cudaStream_t st)
{
    if (a.P <= 0) return cudaSuccess;
    transform_kernel<<<a.P, TF_THREADS, 0, st>>>(a);
    return cudaGetLastError();
}

} // namespace phylino
