// mp_transpose.cu -- ingestion of the paper's dictionary layout: the listings hold Psi row-major,
// psi[n*M + m] (A2 P:360), which makes every atom a stride-M gather; this library wants atom-major rows
// psi_t[m*ld + n].  A one-off out-of-place transpose, HBM-bound: 4NM bytes read + 4NM bytes written.
// 64 x 64 tiles through padded shared memory, both global sides coalesced, any N, M, ldr, ld (4-byte accesses, so no
// alignment demands on the source); persistent grid over the tiles.
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

mp_status launch_transpose_rowmajor(const float* psi, int N, int M, int64_t ldr, float* psi_t, int64_t ld, cudaStream_t stream)
{
    DeviceInfo di;
    mp_status st = device_info(&di);
    if (st != MP_OK) return st;
    const int tiles_n = (N + kTrTile - 1) / kTrTile, tiles_m = (M + kTrTile - 1) / kTrTile;
    int64_t blocks = (int64_t)tiles_n * tiles_m;
    const int64_t cap = (int64_t)di.sm_count * 8;
    if (blocks > cap) blocks = cap;
    transpose_rowmajor_kernel<<<(int)blocks, 256, 0, stream>>>(psi, N, M, ldr, psi_t, ld, tiles_n, tiles_m);
    count_launch();
    MP_CUDA(cudaGetLastError());
    return MP_OK;
}

}  // namespace mp
