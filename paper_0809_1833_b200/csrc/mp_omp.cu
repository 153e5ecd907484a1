// mp_omp.cu -- Orthogonal Matching Pursuit (the paper's declared next target).
// MP's selection (Eq. 9 / Eq. 16, the same fused correlate+argmax kernel) followed by a least-squares refit on the
// selected atoms.  The refit is carried as a QR factorisation grown by one column per iteration (float64):
//     w   <- psi_i - Q Q^T psi_i          (classical Gram-Schmidt, applied twice: "twice is enough")
//     R[0:t, t] <- Q^T psi_i,  R[t, t] <- ||w||,  q_t <- w / ||w||
//     z_t <- <q_t, r>,  r <- r - z_t q_t  (so r = y - Psi_S x_S with x_S the least-squares solution, never formed
//                                          until the end:  R x_S = z by back substitution)
// A stream loop of small kernels (as algo 2 of the MP path): the stop flag lives on the device and turns the remaining
// enqueued iterations into no-ops, the host polls it once per chunk.  The correlation pass is what costs (4NM bytes
// per iteration); the refit reads the t x N basis twice per iteration (16 t N bytes, L2-resident at these sizes).
#include "mp_common.cuh"
#include "mp_internal.h"
#include "mp_omp.h"

namespace mp {

constexpr int kOmpThreads = 1024;

size_t omp_layout(int N, int T, void* base, OmpWs* ws)
{
    const size_t Nr = (size_t)round_up(N, 128), Tr = (size_t)round_up(T > 0 ? T : 1, 32);
    size_t off = 0;
    char* b = static_cast<char*>(base);
    auto take = [&](size_t bytes) { size_t o = off; off = (off + bytes + 255) / 256 * 256; return o; };
    const size_t o_ctrl = take(256), o_r64 = take(8 * Nr), o_r32 = take(4 * Nr), o_w = take(8 * Nr), o_h = take(8 * Tr),
                 o_z = take(8 * Tr), o_R = take(8 * Tr * Tr), o_sel = take(4 * Tr), o_Q = take(8 * Tr * Nr),
                 o_hp = take(8 * Tr * kOmpMaxCtas), o_sc = take(8 * 4 * kOmpMaxCtas);
    if (ws) {
        ws->ctrl = reinterpret_cast<unsigned long long*>(b + o_ctrl);
        ws->r64 = reinterpret_cast<double*>(b + o_r64); ws->r32 = reinterpret_cast<float*>(b + o_r32);
        ws->w = reinterpret_cast<double*>(b + o_w); ws->h = reinterpret_cast<double*>(b + o_h);
        ws->z = reinterpret_cast<double*>(b + o_z); ws->Rm = reinterpret_cast<double*>(b + o_R);
        ws->sel = reinterpret_cast<int*>(b + o_sel); ws->Q = reinterpret_cast<double*>(b + o_Q);
        ws->hpart = reinterpret_cast<double*>(b + o_hp); ws->scal = reinterpret_cast<double*>(b + o_sc);
        ws->bytes = off;
    }
    return off;
}

__device__ __forceinline__ double omp_block_sum(double v, double* scratch /* 32 doubles */)
{
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    v = warp_sum(v);
    __syncthreads();
    if (lane == 0) scratch[warp] = v;
    __syncthreads();
    double t = (lane < (int)(blockDim.x >> 5)) ? scratch[lane] : 0.0;
    return warp_sum(t);   // identical in every warp
}

__global__ void __launch_bounds__(kOmpThreads)
omp_init_kernel(const float* __restrict__ y, int N, int Nr, float eps, int T, OmpWs ws)
{
    __shared__ double scratch[32];
    double ss = 0.0;
    for (int n = threadIdx.x; n < Nr; n += blockDim.x) {
        const float v = n < N ? y[n] : 0.f;
        ws.r64[n] = (double)v;
        ws.r32[n] = v;
        ss += (double)v * (double)v;
    }
    const double yy = omp_block_sum(ss, scratch);
    if (threadIdx.x == 0) {
        ws.ctrl[kCtrKey] = 0ull;
        ws.ctrl[kCtrT] = 0ull;
        ws.ctrl[kCtrYY] = (unsigned long long)__double_as_longlong(yy);
        ws.ctrl[kCtrRR] = (unsigned long long)__double_as_longlong(yy);
        const bool go = (sqrt(yy) > (double)eps * sqrt(yy)) && (0 < T);
        ws.ctrl[kCtrDone] = go ? 0ull : 1ull;
    }
}

// h_j = <q_j, w> for j < t, one CTA of 8 warps per basis vector (fixed-order block sum).
// pass 0: w = psi_i (the atom just selected); pass 1: w = ws.w.
__global__ void __launch_bounds__(256)
omp_hdots_kernel(const float* __restrict__ psi_t, int N, int Nr, int64_t ld, int pass, OmpWs ws)
{
    if (ws.ctrl[kCtrDone]) return;
    const int t = (int)ws.ctrl[kCtrT];
    const int j = blockIdx.x;
    if (j >= t) return;
    __shared__ double part[8];
    const double* q = ws.Q + (size_t)j * Nr;
    double s0 = 0.0, s1 = 0.0;
    if (pass == 0) {
        const float* psi_i = psi_t + (int64_t)key_index(ws.ctrl[kCtrKey]) * ld;
        int n = threadIdx.x;
        for (; n + 256 < N; n += 512) { s0 += q[n] * (double)__ldg(psi_i + n); s1 += q[n + 256] * (double)__ldg(psi_i + n + 256); }
        if (n < N) s0 += q[n] * (double)__ldg(psi_i + n);
    } else {
        int n = threadIdx.x;
        for (; n + 256 < N; n += 512) { s0 += q[n] * ws.w[n]; s1 += q[n + 256] * ws.w[n + 256]; }
        if (n < N) s0 += q[n] * ws.w[n];
    }
    const double s = warp_sum(s0 + s1);
    if ((threadIdx.x & 31) == 0) part[threadIdx.x >> 5] = s;
    __syncthreads();
    if (threadIdx.x == 0) ws.h[j] = ((part[0] + part[1]) + (part[2] + part[3])) + ((part[4] + part[5]) + (part[6] + part[7]));
}

// w <- w - sum_{j<t} h_j q_j.  A CTA owns 32 components; its 8 warps take the basis vectors j = warp, warp + 8, ... and
// their partial sums are added in warp order (fixed order).  R[j][t] collects h_j of both passes.
__global__ void __launch_bounds__(256)
omp_waxpy_kernel(const float* __restrict__ psi_t, int N, int Nr, int64_t ld, int T, int pass, OmpWs ws)
{
    if (ws.ctrl[kCtrDone]) return;
    const int t = (int)ws.ctrl[kCtrT];
    __shared__ double part[8][32];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int n = blockIdx.x * 32 + lane;
    double a0 = 0.0, a1 = 0.0;
    if (n < N) {
        int j = warp;
        for (; j + 8 < t; j += 16) {
            a0 += ws.h[j] * ws.Q[(size_t)j * Nr + n];
            a1 += ws.h[j + 8] * ws.Q[(size_t)(j + 8) * Nr + n];
        }
        if (j < t) a0 += ws.h[j] * ws.Q[(size_t)j * Nr + n];
    }
    part[warp][lane] = a0 + a1;
    __syncthreads();
    if (warp == 0 && n < N) {
        double sum = 0.0;
#pragma unroll
        for (int w8 = 0; w8 < 8; w8++) sum += part[w8][lane];
        const double v0 = pass == 0 ? (double)__ldg(psi_t + (int64_t)key_index(ws.ctrl[kCtrKey]) * ld + n) : ws.w[n];
        ws.w[n] = v0 - sum;
    }
    if (blockIdx.x == 0)
        for (int j = threadIdx.x; j < t; j += blockDim.x) {
            if (pass == 0) ws.Rm[(size_t)j * T + t] = ws.h[j]; else ws.Rm[(size_t)j * T + t] += ws.h[j];
        }
}

// q_t <- w/||w||, z_t <- <q_t, r>, r <- r - z_t q_t, ||r||^2 (direct sum), bookkeeping and the stop test.  One CTA.
__global__ void __launch_bounds__(kOmpThreads)
omp_finalize_kernel(int N, int Nr, float eps, int T, int Tld, int* idx_trace, OmpWs ws)
{
    if (ws.ctrl[kCtrDone]) return;
    __shared__ double scratch[32];
    const int t = (int)ws.ctrl[kCtrT];
    const unsigned long long key = ws.ctrl[kCtrKey];
    double ss = 0.0;
    for (int n = threadIdx.x; n < N; n += blockDim.x) ss += ws.w[n] * ws.w[n];
    const double nrm = sqrt(omp_block_sum(ss, scratch));
    if (!(nrm > 1e-10)) {                        // the atom lies in the span of the selected ones (unit atoms): nothing to add
        if (threadIdx.x == 0) ws.ctrl[kCtrDone] = 1ull;
        return;
    }
    double* q = ws.Q + (size_t)t * Nr;
    double zs = 0.0;
    for (int n = threadIdx.x; n < N; n += blockDim.x) {
        const double qn = ws.w[n] / nrm;
        q[n] = qn;
        zs += qn * ws.r64[n];
    }
    const double zt = omp_block_sum(zs, scratch);
    double rs = 0.0;
    for (int n = threadIdx.x; n < N; n += blockDim.x) {
        const double v = ws.r64[n] - zt * q[n];
        ws.r64[n] = v;
        ws.r32[n] = (float)v;
        rs += v * v;
    }
    const double rr = omp_block_sum(rs, scratch);
    if (threadIdx.x == 0) {
        ws.Rm[(size_t)t * Tld + t] = nrm;
        ws.z[t] = zt;
        ws.sel[t] = key_index(key);
        if (idx_trace) idx_trace[t] = key_index(key);
        const double yy = __longlong_as_double((long long)ws.ctrl[kCtrYY]);
        ws.ctrl[kCtrT] = (unsigned long long)(t + 1);
        ws.ctrl[kCtrRR] = (unsigned long long)__double_as_longlong(rr);
        ws.ctrl[kCtrKey] = 0ull;
        const bool go = (sqrt(rr) > (double)eps * sqrt(yy)) && (t + 1 < T);
        if (!go) ws.ctrl[kCtrDone] = 1ull;
    }
}

// R x_S = z by column-oriented back substitution (one CTA), x~ <- x_S on S, r and n_iter out.
__global__ void __launch_bounds__(kOmpThreads)
omp_finish_kernel(int N, int M, int T, float* __restrict__ x, float* __restrict__ r, int* n_iter, OmpWs ws)
{
    __shared__ double xk_s;
    const int t = (int)ws.ctrl[kCtrT];
    for (int m = threadIdx.x; m < M; m += blockDim.x) x[m] = 0.f;
    for (int n = threadIdx.x; n < N; n += blockDim.x) r[n] = (float)ws.r64[n];
    __syncthreads();
    for (int k = t - 1; k >= 0; k--) {
        if (threadIdx.x == 0) {
            xk_s = ws.z[k] / ws.Rm[(size_t)k * T + k];
            x[ws.sel[k]] = (float)xk_s;
        }
        __syncthreads();
        const double xk = xk_s;
        for (int j = threadIdx.x; j < k; j += blockDim.x) ws.z[j] -= ws.Rm[(size_t)j * T + k] * xk;
        __syncthreads();
    }
    if (threadIdx.x == 0) *n_iter = t;
}

}  // namespace mp

using namespace mp;

extern "C" {

MP_API size_t mp_workspace_bytes_omp(int N, int M, int max_iter)
{
    if (N < 1 || M < 1 || max_iter < 0) return 0;
    return omp_layout(N, max_iter < N ? max_iter : N, nullptr, nullptr);
}

MP_API mp_status mp_recover_omp(const float* psi_t, int N, int M, int64_t ld,
                                const float* y, float eps, int max_iter,
                                float* x, float* r, int* n_iter, int* idx_trace,
                                void* workspace, size_t workspace_bytes, void* stream)
{
    if (!psi_t || !y || !x || !r || !n_iter) return fail(MP_ERR_INVALID_ARG, "psi_t, y, x, r and n_iter must be non-null");
    if (N < 1 || M < 1) return fail(MP_ERR_INVALID_ARG, "need N >= 1 and M >= 1 (got N=%d, M=%d)", N, M);
    if (ld < N || (ld & 3)) return fail(MP_ERR_INVALID_ARG, "need ld >= N and ld %% 4 == 0 (got ld=%lld, N=%d)", (long long)ld, N);
    if ((reinterpret_cast<uintptr_t>(psi_t) | reinterpret_cast<uintptr_t>(y)) & 15u)
        return fail(MP_ERR_INVALID_ARG, "psi_t and y must be 16-byte aligned");
    if (max_iter < 0) return fail(MP_ERR_INVALID_ARG, "max_iter must be >= 0 (got %d)", max_iter);
    if (!(eps >= 0.0f)) return fail(MP_ERR_INVALID_ARG, "eps must be >= 0 and not NaN");
    const int T = max_iter < N ? max_iter : N;          // more than N atoms cannot be linearly independent
    const size_t need = omp_layout(N, T, nullptr, nullptr);
    if (!workspace || (reinterpret_cast<uintptr_t>(workspace) & 255u) || workspace_bytes < need)
        return fail(MP_ERR_WORKSPACE, "workspace must be non-null, 256-byte aligned and >= %zu bytes (got %zu)", need, workspace_bytes);
    DeviceInfo di;
    mp_status st = device_info(&di);
    if (st != MP_OK) return st;
    OmpWs ws;
    omp_layout(N, T, workspace, &ws);
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    const int Nr = round_up(N, 128), Tld = round_up(T > 0 ? T : 1, 32);

    // omp_algo 0 = auto (the persistent kernel when the basis slices fit in shared memory), 1 = persistent or error,
    // 2 = the stream loop below
    const int64_t oalgo = options().omp_algo;
    if (T > 0 && oalgo != 2 && (oalgo == 1 || omp_persistent_supported(N, M, T))) {
        OmpArgs oa{psi_t, N, M, ld, y, eps, T, idx_trace};
        st = launch_omp_persistent(oa, ws, s);
        if (st != MP_OK) return st;
        omp_finish_kernel<<<1, kOmpThreads, 0, s>>>(N, M, Tld, x, r, n_iter, ws);
        MP_CUDA(cudaGetLastError());
        count_launch();
        options().info_omp_algo = 1;
        return MP_OK;
    }
    options().info_omp_algo = 2;
    omp_init_kernel<<<1, kOmpThreads, 0, s>>>(y, N, Nr, eps, T, ws);
    MP_CUDA(cudaGetLastError());
    count_launch();
    int blocks = (M + 7) / 8;
    if (blocks > di.sm_count * 8) blocks = di.sm_count * 8;
    const int64_t chunk_knob = options().chunk;
    const int64_t chunk = chunk_knob > 0 ? chunk_knob : 64;
    int done_iters = 0;
    while (done_iters < T) {
        const int n = (int)((T - done_iters) < chunk ? (T - done_iters) : chunk);
        for (int k = 0; k < n; k++) {
            st = launch_sl_correlate_argmax(psi_t, N, M, ld, ws.r32, ws.ctrl, blocks, s);
            if (st != MP_OK) return st;
            const int hb = done_iters + k;              // at most done_iters + k basis vectors exist at this iteration
            for (int pass = 0; pass < 2; pass++) {
                if (hb > 0) omp_hdots_kernel<<<hb, 256, 0, s>>>(psi_t, N, Nr, ld, pass, ws);
                omp_waxpy_kernel<<<(N + 31) / 32, 256, 0, s>>>(psi_t, N, Nr, ld, Tld, pass, ws);
            }
            omp_finalize_kernel<<<1, kOmpThreads, 0, s>>>(N, Nr, eps, T, Tld, idx_trace, ws);
            count_launch(hb > 0 ? 5 : 3);
        }
        MP_CUDA(cudaGetLastError());
        done_iters += n;
        if (done_iters < T) {
            unsigned long long done = 0;                 // the one host synchronisation of this loop: poll the stop flag
            MP_CUDA(cudaMemcpyAsync(&done, ws.ctrl + kCtrDone, sizeof(done), cudaMemcpyDeviceToHost, s));
            MP_CUDA(cudaStreamSynchronize(s));
            if (done) break;
        }
    }
    omp_finish_kernel<<<1, kOmpThreads, 0, s>>>(N, M, Tld, x, r, n_iter, ws);
    MP_CUDA(cudaGetLastError());
    count_launch();
    return MP_OK;
}

}  // extern "C"
