// mp_normalize.cu -- column normalisation, Eq. 4: psi_m <- psi_m / ||psi_m||_2.
// HBM-bound: 4NM bytes read + 4NM bytes written.  One warp per atom (atoms are contiguous rows of the
// atom-major layout); the second pass re-reads the row from L1/L2, not from HBM.
#include "mp_common.cuh"
#include "mp_internal.h"

namespace mp {

constexpr int kNormWarps = 8;

__global__ void __launch_bounds__(kNormWarps * 32)
normalize_columns_kernel(float* __restrict__ psi_t, int N, int M, int64_t ld, float* __restrict__ norms_out)
{
    const int lane = threadIdx.x & 31;
    const int warp = threadIdx.x >> 5;
    const int n4 = N >> 2;
    for (int m = blockIdx.x * kNormWarps + warp; m < M; m += gridDim.x * kNormWarps) {
        float* row = psi_t + (int64_t)m * ld;
        float4* row4 = reinterpret_cast<float4*>(row);
        // pass 1: sum of squares in float64 (fp32 x fp32 products are exact in float64)
        double s0 = 0.0, s1 = 0.0;
        int j = lane;
        for (; j + 32 < n4; j += 64) {
            const float4 a = row4[j], b = row4[j + 32];
            s0 += (double)a.x * a.x; s0 += (double)a.y * a.y; s0 += (double)a.z * a.z; s0 += (double)a.w * a.w;
            s1 += (double)b.x * b.x; s1 += (double)b.y * b.y; s1 += (double)b.z * b.z; s1 += (double)b.w * b.w;
        }
        for (; j < n4; j += 32) {
            const float4 a = row4[j];
            s0 += (double)a.x * a.x; s0 += (double)a.y * a.y; s0 += (double)a.z * a.z; s0 += (double)a.w * a.w;
        }
        for (int n = (n4 << 2) + lane; n < N; n += 32) s1 += (double)row[n] * row[n];
        const double nrm = sqrt(warp_sum(s0 + s1));
        if (lane == 0 && norms_out) norms_out[m] = (float)nrm;
        if (!(nrm > 0.0)) continue;   // zero atom stays zero (reading R7)
        // pass 2: exact float64 quotient, rounded to fp32 once
        for (j = lane; j < n4; j += 32) {
            float4 a = row4[j];
            a.x = (float)((double)a.x / nrm); a.y = (float)((double)a.y / nrm);
            a.z = (float)((double)a.z / nrm); a.w = (float)((double)a.w / nrm);
            row4[j] = a;
        }
        for (int n = (n4 << 2) + lane; n < N; n += 32) row[n] = (float)((double)row[n] / nrm);
    }
}

mp_status launch_normalize(float* psi_t, int N, int M, int64_t ld, float* norms_out, cudaStream_t stream)
{
    DeviceInfo di;
    mp_status st = device_info(&di);
    if (st != MP_OK) return st;
    int blocks = (M + kNormWarps - 1) / kNormWarps;
    const int cap = di.sm_count * 8;
    if (blocks > cap) blocks = cap;
    normalize_columns_kernel<<<blocks, kNormWarps * 32, 0, stream>>>(psi_t, N, M, ld, norms_out);
    count_launch();
    MP_CUDA(cudaGetLastError());
    return MP_OK;
}

}  // namespace mp
