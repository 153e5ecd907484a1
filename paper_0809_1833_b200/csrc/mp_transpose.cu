// mp_transpose.cu -- ingestion of the paper's dictionary layout: the listings hold Psi row-major,
// psi[n*M + m] (A2 P:360), which makes every atom a stride-M gather; this library wants atom-major rows
// psi_t[m*ld + n].  A one-off out-of-place transpose, HBM-bound: 4NM bytes read + 4NM bytes written.
// 64 x 64 tiles through padded shared memory, both global sides coalesced, any N, M, ldr, ld; 128-bit accesses when the source
// is aligned, 4-byte accesses otherwise (no alignment demands on the source); persistent grid over the tiles.
#include "mp_common.cuh"
#include "mp_internal.h"

namespace mp {

constexpr int kTrTile = 64;

__global__ void __launch_bounds__(256)
transpose_rowmajor_kernel(const float* __restrict__ psi, int N, int M, int64_t ldr, float* __restrict__ psi_t, int64_t ld,
                          int tiles_n, int tiles_m)
{
    __shared__ float tile[kTrTile][kTrTile + 1];
    const int c = threadIdx.x & 63, r0 = threadIdx.x >> 6;
    for (int64_t tl = blockIdx.x; tl < (int64_t)tiles_n * tiles_m; tl += gridDim.x) {
        const int n0 = (int)(tl / tiles_m) * kTrTile, m0 = (int)(tl % tiles_m) * kTrTile;
#pragma unroll 4
        for (int k = 0; k < kTrTile / 4; k++) {                                 // rows of Psi (n), contiguous along m
            const int n = n0 + r0 + 4 * k, m = m0 + c;
            tile[r0 + 4 * k][c] = (n < N && m < M) ? __ldg(psi + (int64_t)n * ldr + m) : 0.f;
        }
        __syncthreads();
#pragma unroll 4
        for (int k = 0; k < kTrTile / 4; k++) {                                 // rows of Psi^T (atoms m), contiguous along n
            const int m = m0 + r0 + 4 * k, n = n0 + c;
            if (m < M && n < N) psi_t[(int64_t)m * ld + n] = tile[c][r0 + 4 * k];
        }
        __syncthreads();
    }
}

// Aligned case (psi 16-byte aligned, ldr % 4 == 0; psi_t always is): 128-bit accesses on both global sides.  A thread reads a
// float4 along m, scatters it into the padded tile, and after the barrier gathers a float4 along n (tile column, stride 65:
// conflict-free) for one 16-byte store.  Edge tiles fall back to scalars inside the same loop.
__global__ void __launch_bounds__(256)
transpose_rowmajor_vec_kernel(const float* __restrict__ psi, int N, int M, int64_t ldr, float* __restrict__ psi_t, int64_t ld,
                              int tiles_n, int tiles_m)
{
    __shared__ float tile[kTrTile][kTrTile + 1];
    const int c4 = (threadIdx.x & 15) * 4, r0 = threadIdx.x >> 4;             // 16 threads x float4 = 64 columns, 16 rows per pass
    for (int64_t tl = blockIdx.x; tl < (int64_t)tiles_n * tiles_m; tl += gridDim.x) {
        const int n0 = (int)(tl / tiles_m) * kTrTile, m0 = (int)(tl % tiles_m) * kTrTile;
#pragma unroll
        for (int k = 0; k < kTrTile / 16; k++) {
            const int n = n0 + r0 + 16 * k, m = m0 + c4;
            float4 v = make_float4(0.f, 0.f, 0.f, 0.f);
            if (n < N) {
                const float* src = psi + (int64_t)n * ldr + m;
                if (m + 3 < M) v = __ldg(reinterpret_cast<const float4*>(src));
                else {
                    if (m < M) v.x = __ldg(src);
                    if (m + 1 < M) v.y = __ldg(src + 1);
                    if (m + 2 < M) v.z = __ldg(src + 2);
                }
            }
            float* t = &tile[r0 + 16 * k][c4];
            t[0] = v.x; t[1] = v.y; t[2] = v.z; t[3] = v.w;
        }
        __syncthreads();
#pragma unroll
        for (int k = 0; k < kTrTile / 16; k++) {
            const int m = m0 + r0 + 16 * k, n = n0 + c4;
            if (m < M && n < N) {
                const float4 v = make_float4(tile[c4][r0 + 16 * k], tile[c4 + 1][r0 + 16 * k], tile[c4 + 2][r0 + 16 * k], tile[c4 + 3][r0 + 16 * k]);
                float* dst = psi_t + (int64_t)m * ld + n;
                if (n + 3 < N) *reinterpret_cast<float4*>(dst) = v;
                else {
                    dst[0] = v.x;
                    if (n + 1 < N) dst[1] = v.y;
                    if (n + 2 < N) dst[2] = v.z;
                }
            }
        }
        __syncthreads();
    }
}

mp_status launch_transpose_rowmajor(const float* psi, int N, int M, int64_t ldr, float* psi_t, int64_t ld, cudaStream_t stream)
{
    DeviceInfo di;
    mp_status st = device_info(&di);
    if (st != MP_OK) return st;
    const int tiles_n = (N + kTrTile - 1) / kTrTile, tiles_m = (M + kTrTile - 1) / kTrTile;
    int64_t blocks = (int64_t)tiles_n * tiles_m;
    const int64_t cap = (int64_t)di.sm_count * 8;
    if (blocks > cap) blocks = cap;
    if ((reinterpret_cast<uintptr_t>(psi) & 15u) == 0 && (ldr & 3) == 0)
        transpose_rowmajor_vec_kernel<<<(int)blocks, 256, 0, stream>>>(psi, N, M, ldr, psi_t, ld, tiles_n, tiles_m);
    else
        transpose_rowmajor_kernel<<<(int)blocks, 256, 0, stream>>>(psi, N, M, ldr, psi_t, ld, tiles_n, tiles_m);
    count_launch();
    MP_CUDA(cudaGetLastError());
    return MP_OK;
}

}  // namespace mp
