// mp_streamloop.cu -- "algo 2": the MP loop as a stream of small kernels (general fallback, any N).
// Two kernels per iteration (fused correlate+argmax; fused update+norm+stop test); the stop flag stays
// on the device and turns the remaining enqueued iterations into no-ops; the host polls it once per chunk.
// Same arithmetic contract as the persistent kernel (fp32 dots of an fp32 rounding of a float64 r).
#include "mp_common.cuh"
#include "mp_internal.h"

namespace mp {


constexpr int kSLThreads = 1024;

__device__ __forceinline__ double block_sum_1024(double v, double* scratch /* 32 doubles */)
{
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    v = warp_sum(v);
    __syncthreads();
    if (lane == 0) scratch[warp] = v;
    __syncthreads();
    double t = (lane < (int)(blockDim.x >> 5)) ? scratch[lane] : 0.0;
    return warp_sum(t);   // identical in every warp
}

__global__ void __launch_bounds__(kSLThreads)
sl_init_kernel(const float* __restrict__ y, int N, int M, int Nr, float eps, int max_iter,
               double* x64, double* r64, float* r32, unsigned long long* ctrl)
{
    __shared__ double scratch[32];
    for (int m = threadIdx.x; m < M; m += blockDim.x) x64[m] = 0.0;               // Eq. 8: x~ <- 0
    double ss = 0.0;
    for (int n = threadIdx.x; n < Nr; n += blockDim.x) {
        const float v = n < N ? y[n] : 0.f;                                        // Eq. 8: r <- y
        r64[n] = (double)v;
        r32[n] = v;
        ss += (double)v * (double)v;
    }
    const double yy = block_sum_1024(ss, scratch);
    if (threadIdx.x == 0) {
        ctrl[kCtrKey] = 0ull;
        ctrl[kCtrT] = 0ull;
        ctrl[kCtrYY] = (unsigned long long)__double_as_longlong(yy);
        ctrl[kCtrRR] = (unsigned long long)__double_as_longlong(yy);
        const bool go = (sqrt(yy) > (double)eps * sqrt(yy)) && (0 < max_iter);     // P:70 at t = 0
        ctrl[kCtrDone] = go ? 0ull : 1ull;
    }
}

// Eq. 9 + Eq. 16 fused: one warp per atom, float4 loads, shuffle reduce, packed-key max.
__global__ void __launch_bounds__(256)
sl_correlate_argmax_kernel(const float* __restrict__ psi_t, int N, int M, int64_t ld,
                           const float* __restrict__ r32, unsigned long long* ctrl)
{
    if (ctrl[kCtrDone]) return;
    __shared__ unsigned long long wkey[8];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int n4 = N >> 2;
    const float4* r4 = reinterpret_cast<const float4*>(r32);
    unsigned long long best = 0ull;
    for (int m = blockIdx.x * 8 + warp; m < M; m += gridDim.x * 8) {
        const float* row = psi_t + (int64_t)m * ld;
        const float4* row4 = reinterpret_cast<const float4*>(row);
        float a0 = 0.f, a1 = 0.f;
        int j = lane;
        for (; j + 224 < n4; j += 256) {                                     // 8 independent 16-byte loads in flight per lane
            float4 p[8];
#pragma unroll
            for (int u = 0; u < 8; u++) p[u] = __ldg(row4 + j + 32 * u);
#pragma unroll
            for (int u = 0; u < 8; u += 2) {
                const float4 u0 = r4[j + 32 * u], u1 = r4[j + 32 * u + 32];
                a0 = fmaf(p[u].x, u0.x, a0); a0 = fmaf(p[u].y, u0.y, a0); a0 = fmaf(p[u].z, u0.z, a0); a0 = fmaf(p[u].w, u0.w, a0);
                a1 = fmaf(p[u + 1].x, u1.x, a1); a1 = fmaf(p[u + 1].y, u1.y, a1); a1 = fmaf(p[u + 1].z, u1.z, a1); a1 = fmaf(p[u + 1].w, u1.w, a1);
            }
        }
        for (; j + 32 < n4; j += 64) {
            const float4 p = __ldg(row4 + j), q = __ldg(row4 + j + 32);
            const float4 u = r4[j], v = r4[j + 32];
            a0 = fmaf(p.x, u.x, a0); a0 = fmaf(p.y, u.y, a0); a0 = fmaf(p.z, u.z, a0); a0 = fmaf(p.w, u.w, a0);
            a1 = fmaf(q.x, v.x, a1); a1 = fmaf(q.y, v.y, a1); a1 = fmaf(q.z, v.z, a1); a1 = fmaf(q.w, v.w, a1);
        }
        for (; j < n4; j += 32) {
            const float4 p = __ldg(row4 + j);
            const float4 u = r4[j];
            a0 = fmaf(p.x, u.x, a0); a0 = fmaf(p.y, u.y, a0); a0 = fmaf(p.z, u.z, a0); a0 = fmaf(p.w, u.w, a0);
        }
        for (int n = (n4 << 2) + lane; n < N; n += 32) a1 = fmaf(__ldg(row + n), r32[n], a1);
        const float c = warp_sum(a0 + a1);
        const unsigned long long key = pack_key(c, m);
        best = key > best ? key : best;
    }
    if (lane == 0) wkey[warp] = best;
    __syncthreads();
    if (threadIdx.x == 0) {
        unsigned long long b = wkey[0];
#pragma unroll
        for (int w = 1; w < 8; w++) b = wkey[w] > b ? wkey[w] : b;
        if (b) red_max_u64(ctrl + kCtrKey, b);
    }
}

// Eq. 10-12 + nrm2 + stop test fused, one CTA.
__global__ void __launch_bounds__(kSLThreads)
sl_update_kernel(const float* __restrict__ psi_t, int N, int Nr, int64_t ld, float eps, int max_iter,
                 double* x64, double* r64, float* r32, unsigned long long* ctrl,
                 int* idx_trace, float* c_trace)
{
    if (ctrl[kCtrDone]) return;
    __shared__ double scratch[32];
    const unsigned long long key = ctrl[kCtrKey];
    const int i = key_index(key);
    const float c = key_value(key);
    const double cd = (double)c;
    const float* psi_i = psi_t + (int64_t)i * ld;
    double ss = 0.0;
    for (int n = threadIdx.x; n < N; n += blockDim.x) {
        const double v = r64[n] - cd * (double)__ldg(psi_i + n);                   // Eq. 11
        r64[n] = v;
        r32[n] = (float)v;
        ss += v * v;                                                               // Eq. 18, direct sum
    }
    const double rr = block_sum_1024(ss, scratch);
    if (threadIdx.x == 0) {
        const int t = (int)ctrl[kCtrT];
        x64[i] += cd;                                                              // Eq. 10
        if (idx_trace) idx_trace[t] = i;
        if (c_trace) c_trace[t] = c;
        const double yy = __longlong_as_double((long long)ctrl[kCtrYY]);
        ctrl[kCtrT] = (unsigned long long)(t + 1);                                 // Eq. 12
        ctrl[kCtrRR] = (unsigned long long)__double_as_longlong(rr);
        ctrl[kCtrKey] = 0ull;
        const bool go = (sqrt(rr) > (double)eps * sqrt(yy)) && (t + 1 < max_iter);
        if (!go) ctrl[kCtrDone] = 1ull;
    }
}

__global__ void __launch_bounds__(kSLThreads)
sl_finish_kernel(int N, int M, const double* x64, const double* r64, const unsigned long long* ctrl,
                 float* x, float* r, int* n_iter)
{
    for (int m = blockIdx.x * blockDim.x + threadIdx.x; m < M; m += gridDim.x * blockDim.x) x[m] = (float)x64[m];
    for (int n = blockIdx.x * blockDim.x + threadIdx.x; n < N; n += gridDim.x * blockDim.x) r[n] = (float)r64[n];
    if (blockIdx.x == 0 && threadIdx.x == 0) *n_iter = (int)ctrl[kCtrT];
}

mp_status launch_sl_correlate_argmax(const float* psi_t, int N, int M, int64_t ld, const float* r32, unsigned long long* ctrl,
                                     int blocks, cudaStream_t stream)
{
    sl_correlate_argmax_kernel<<<blocks, 256, 0, stream>>>(psi_t, N, M, ld, r32, ctrl);
    MP_CUDA(cudaGetLastError());
    count_launch();
    return MP_OK;
}

mp_status launch_recover_streamloop(const RecoverArgs& a, const Workspace& ws, cudaStream_t stream)
{
    DeviceInfo di;
    mp_status st = device_info(&di);
    if (st != MP_OK) return st;
    const int Nr = round_up(a.N, 128);
    sl_init_kernel<<<1, kSLThreads, 0, stream>>>(a.y, a.N, a.M, Nr, a.eps, a.max_iter, ws.x64, ws.r64, ws.r32, ws.ctrl);
    count_launch();
    MP_CUDA(cudaGetLastError());
    int blocks = (a.M + 7) / 8;
    if (blocks > di.sm_count * 8) blocks = di.sm_count * 8;
    const int64_t chunk_knob = options().chunk;
    const int64_t chunk = chunk_knob > 0 ? chunk_knob : 64;
    int done_iters = 0;
    while (done_iters < a.max_iter) {
        const int n = (int)((a.max_iter - done_iters) < chunk ? (a.max_iter - done_iters) : chunk);
        for (int k = 0; k < n; k++) {
            sl_correlate_argmax_kernel<<<blocks, 256, 0, stream>>>(a.psi_t, a.N, a.M, a.ld, ws.r32, ws.ctrl);
            sl_update_kernel<<<1, kSLThreads, 0, stream>>>(a.psi_t, a.N, Nr, a.ld, a.eps, a.max_iter,
                                                           ws.x64, ws.r64, ws.r32, ws.ctrl, a.idx_trace, a.c_trace);
        }
        count_launch(2 * n);
        MP_CUDA(cudaGetLastError());
        done_iters += n;
        if (done_iters < a.max_iter) {
            unsigned long long done = 0;   // the one host synchronisation of this fallback: poll the stop flag
            MP_CUDA(cudaMemcpyAsync(&done, ws.ctrl + kCtrDone, sizeof(done), cudaMemcpyDeviceToHost, stream));
            MP_CUDA(cudaStreamSynchronize(stream));
            if (done) break;
        }
    }
    int fb = (a.M + kSLThreads - 1) / kSLThreads;
    if (fb > di.sm_count) fb = di.sm_count;
    sl_finish_kernel<<<fb, kSLThreads, 0, stream>>>(a.N, a.M, ws.x64, ws.r64, ws.ctrl, a.x, a.r, a.n_iter);
    count_launch();
    MP_CUDA(cudaGetLastError());
    return MP_OK;
}

}  // namespace mp
