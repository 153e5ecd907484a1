// mp_encode_score.cu -- the steps either side of the MP path, on the device:
//   encode  y = Psi x for a K-sparse x given as (index, value) pairs      Eq. 2, P:21-25 (the paper builds x that way, A2 P:328-332)
//   score   E = ||x~ - x||^2 / ||x||^2 * 100 %                             Eq. 14
// so that encode -> mp_recover -> score runs without host data.  Both are tiny next to the solve (4NK bytes against
// 4NM per iteration); they are written for exactness, not for a roofline: float64 sums in a fixed order.
#include "mp_common.cuh"
#include "mp_internal.h"

namespace mp {

// One thread per component n; the K atoms are walked in ascending k (the order of the definition), float64 accumulate,
// one rounding to fp32.  double(float) * double(float) is exact in float64, so the sum matches a plain CPU loop bit for bit.
// Rows are contiguous in the atom-major layout: consecutive threads read consecutive floats of each atom.
__global__ void __launch_bounds__(128)
encode_sparse_kernel(const float* __restrict__ psi_t, int N, int M, int64_t ld,
                     const int* __restrict__ idx, const float* __restrict__ val, int K, float* __restrict__ y)
{
    __shared__ int s_idx[512];
    __shared__ double s_val[512];
    const int n = blockIdx.x * blockDim.x + threadIdx.x;
    double s = 0.0;
    for (int k0 = 0; k0 < K; k0 += 512) {
        const int kc = min(512, K - k0);
        __syncthreads();
        for (int k = threadIdx.x; k < kc; k += blockDim.x) {
            const int m = idx[k0 + k];
            s_idx[k] = (m >= 0 && m < M) ? m : -1;                              // an index outside [0, M) contributes nothing
            s_val[k] = (double)val[k0 + k];
        }
        __syncthreads();
        if (n < N) {
            for (int k = 0; k < kc; k++) {
                const int m = s_idx[k];
                if (m >= 0) s = __dadd_rn(s, __dmul_rn(s_val[k], (double)__ldg(psi_t + (int64_t)m * ld + n)));
            }
        }
    }
    if (n < N) y[n] = (float)s;
}

// Single CTA, fixed-order float64 block reductions of ||x~ - x||^2 and ||x||^2 (the difference is formed in float64).
__global__ void __launch_bounds__(1024)
reconstruction_error_kernel(const float* __restrict__ x_hat, const float* __restrict__ x, int M, double* __restrict__ out)
{
    __shared__ double s_num[32], s_den[32];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    double num = 0.0, den = 0.0;
    for (int m = tid; m < M; m += blockDim.x) {
        const double a = (double)x_hat[m], b = (double)x[m];
        num += (a - b) * (a - b);
        den += b * b;
    }
    num = warp_sum(num);
    den = warp_sum(den);
    if (lane == 0) { s_num[warp] = num; s_den[warp] = den; }
    __syncthreads();
    if (tid == 0) {
        double a = 0.0, b = 0.0;
        for (int w = 0; w < (int)(blockDim.x >> 5); w++) { a += s_num[w]; b += s_den[w]; }
        out[0] = 100.0 * a / b;                                                // x = 0: NaN (0/0) or +inf, as Eq. 14 gives
    }
}

mp_status launch_encode_sparse(const float* psi_t, int N, int M, int64_t ld, const int* idx, const float* val, int K,
                               float* y, cudaStream_t stream)
{
    encode_sparse_kernel<<<(N + 127) / 128, 128, 0, stream>>>(psi_t, N, M, ld, idx, val, K, y);
    MP_CUDA(cudaGetLastError());
    count_launch();
    return MP_OK;
}

mp_status launch_reconstruction_error(const float* x_hat, const float* x, int M, double* out, cudaStream_t stream)
{
    reconstruction_error_kernel<<<1, 1024, 0, stream>>>(x_hat, x, M, out);
    MP_CUDA(cudaGetLastError());
    count_launch();
    return MP_OK;
}

}  // namespace mp
