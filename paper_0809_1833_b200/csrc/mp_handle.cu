// mp_handle.cu -- the dictionary handle (include/mp_b200.h, "dictionary handle"): "the host to device dictionary
// transfer only takes place once, since all signals are encoded/decoded with the same dictionary".
//
// mp_dictionary_create puts the dictionary on the device once (chunked H2D on a copy stream, each chunk normalised by
// normalize_columns_kernel on a second stream as soon as it has landed) and keeps, for the HOST-buffer solves that follow,
// an internal stream, the workspace and the small per-call device buffers, so that a steady-state call moves only y up and
// x~, r, n_iter down.  The solves themselves are mp_recover / mp_recover_batched, unchanged: handle and non-handle paths give
// the same bits.
#include <new>

#include "mp_internal.h"

struct mp_dictionary {
    int N = 0, M = 0, device = -1;
    int64_t ld = 0;
    float* psi = nullptr;        // device, atom-major
    bool owns_psi = false;
    cudaStream_t stream = nullptr, copy_stream = nullptr;
    // buffers of the host-buffer solves, grown on demand (capacity in bytes)
    void* ws = nullptr; size_t ws_cap = 0;
    void* io = nullptr; size_t io_cap = 0;      // [Y | X | R | n_iter | idx_trace | c_trace]
};

namespace mp {

static mp_status grow(void** p, size_t* cap, size_t need)
{
    if (need <= *cap) return MP_OK;
    if (*p) MP_CUDA(cudaFree(*p));
    *p = nullptr; *cap = 0;
    MP_CUDA(cudaMalloc(p, need));
    *cap = need;
    return MP_OK;
}

static size_t up256(size_t v) { return (v + 255) / 256 * 256; }

struct DeviceGuard {
    int prev = -1;
    // dev < 0: a handle whose set-up failed before it learnt its device -- nothing to switch to
    explicit DeviceGuard(int dev) { if (dev < 0 || cudaGetDevice(&prev) != cudaSuccess || prev == dev) prev = -1; else cudaSetDevice(dev); }
    ~DeviceGuard() { if (prev >= 0) cudaSetDevice(prev); }
};

// Once a copy from or to the caller's HOST buffers has been enqueued, no return path may leave it in flight: the caller is
// entitled to free or reuse those buffers as soon as the call is back, error or not.  Armed until the call's own final
// synchronise has succeeded.
struct SyncOnExit {
    cudaStream_t s;
    bool armed = true;
    explicit SyncOnExit(cudaStream_t stream) : s(stream) {}
    ~SyncOnExit() { if (armed) (void)cudaStreamSynchronize(s); }
};

}  // namespace mp

using namespace mp;

extern "C" {

mp_status mp_dictionary_create(const float* psi_t, int psi_on_host, int N, int M, int64_t ld, int normalize, mp_dictionary** out)
{
    if (!out) return fail(MP_ERR_INVALID_ARG, "out is null");
    *out = nullptr;
    if (!psi_t) return fail(MP_ERR_INVALID_ARG, "psi_t is null");
    if (N < 1 || M < 1) return fail(MP_ERR_INVALID_ARG, "need N >= 1 and M >= 1 (got N=%d, M=%d)", N, M);
    if (ld < N) return fail(MP_ERR_INVALID_ARG, "need ld >= N (got ld=%lld, N=%d)", (long long)ld, N);
    if (!psi_on_host && (ld & 3)) return fail(MP_ERR_INVALID_ARG, "a device dictionary needs ld %% 4 == 0 (got ld=%lld)", (long long)ld);
    if (!psi_on_host && (reinterpret_cast<uintptr_t>(psi_t) & 15u)) return fail(MP_ERR_INVALID_ARG, "psi_t must be 16-byte aligned");
    mp_dictionary* h = new (std::nothrow) mp_dictionary;
    if (!h) return fail(MP_ERR_CUDA, "out of host memory");
    h->N = N; h->M = M; h->ld = ld;
    mp_status st = MP_OK;
    auto bail = [&](mp_status s) { mp_dictionary_destroy(h); return s; };
    {
        cudaError_t e = cudaGetDevice(&h->device);
        if (e == cudaSuccess) e = cudaStreamCreateWithFlags(&h->stream, cudaStreamNonBlocking);
        if (e == cudaSuccess) e = cudaStreamCreateWithFlags(&h->copy_stream, cudaStreamNonBlocking);
        if (e != cudaSuccess) return bail(cuda_fail(e, "mp_dictionary_create: stream setup"));
    }
    if (!psi_on_host) {
        h->psi = const_cast<float*>(psi_t);                 // borrowed: the caller keeps it alive; normalised in place if asked
        if (normalize) {
            st = launch_normalize(h->psi, N, M, ld, nullptr, h->stream);
            if (st != MP_OK) return bail(st);
            cudaError_t e = cudaStreamSynchronize(h->stream);
            if (e != cudaSuccess) return bail(cuda_fail(e, "mp_dictionary_create: normalise"));
        }
        *out = h;
        return MP_OK;
    }
    const int64_t ld_h = ld;                                 // host row stride: any value >= N; the device copy is re-pitched
    ld = h->ld = round_up(N, 4);
    {
        cudaError_t e = cudaMalloc(reinterpret_cast<void**>(&h->psi), sizeof(float) * (size_t)M * ld);
        if (e == cudaSuccess && ld != N) e = cudaMemsetAsync(h->psi, 0, sizeof(float) * (size_t)M * ld, h->copy_stream);   // defined pad columns
        if (e != cudaSuccess) return bail(cuda_fail(e, "mp_dictionary_create: cudaMalloc of the dictionary"));
        h->owns_psi = true;
    }
    // chunks of whole atoms (>= 8 MiB each, at most 16): chunk k is normalised while chunk k+1 is still on the bus
    int chunks = (int)((sizeof(float) * (size_t)M * ld) >> 23);
    chunks = chunks < 1 ? 1 : chunks > 16 ? 16 : chunks;
    if (chunks > M) chunks = M;
    cudaEvent_t ev[16];
    int n_ev = 0;
    cudaError_t e = cudaSuccess;
    for (int k = 0; k < chunks && e == cudaSuccess && st == MP_OK; k++) {
        const int m0 = (int)((int64_t)M * k / chunks), m1 = (int)((int64_t)M * (k + 1) / chunks);
        e = cudaMemcpy2DAsync(h->psi + (int64_t)m0 * ld, sizeof(float) * (size_t)ld, psi_t + (int64_t)m0 * ld_h, sizeof(float) * (size_t)ld_h,
                              sizeof(float) * (size_t)N, (size_t)(m1 - m0), cudaMemcpyHostToDevice, h->copy_stream);
        if (e != cudaSuccess || !normalize) continue;
        e = cudaEventCreateWithFlags(&ev[n_ev], cudaEventDisableTiming);
        if (e != cudaSuccess) break;
        n_ev++;
        e = cudaEventRecord(ev[n_ev - 1], h->copy_stream);
        if (e == cudaSuccess) e = cudaStreamWaitEvent(h->stream, ev[n_ev - 1], 0);
        if (e == cudaSuccess) st = launch_normalize(h->psi + (int64_t)m0 * ld, N, m1 - m0, ld, nullptr, h->stream);
    }
    if (e == cudaSuccess) e = cudaStreamSynchronize(h->copy_stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(h->stream);
    for (int k = 0; k < n_ev; k++) cudaEventDestroy(ev[k]);
    if (e != cudaSuccess) return bail(cuda_fail(e, "mp_dictionary_create: upload"));
    if (st != MP_OK) return bail(st);
    *out = h;
    return MP_OK;
}

mp_status mp_dictionary_destroy(mp_dictionary* h)
{
    if (!h) return MP_OK;
    DeviceGuard g(h->device);
    if (h->stream) cudaStreamSynchronize(h->stream);
    if (h->ws) cudaFree(h->ws);
    if (h->io) cudaFree(h->io);
    if (h->owns_psi && h->psi) cudaFree(h->psi);
    if (h->stream) cudaStreamDestroy(h->stream);
    if (h->copy_stream) cudaStreamDestroy(h->copy_stream);
    delete h;
    return MP_OK;
}

mp_status mp_dictionary_info(const mp_dictionary* h, int* N, int* M, int64_t* ld, const float** psi_t_device)
{
    if (!h) return fail(MP_ERR_INVALID_ARG, "handle is null");
    if (N) *N = h->N;
    if (M) *M = h->M;
    if (ld) *ld = h->ld;
    if (psi_t_device) *psi_t_device = h->psi;
    return MP_OK;
}

mp_status mp_recover_batched_host_h(mp_dictionary* h, const float* Y, int64_t ldy, int B, float eps, int max_iter,
                                    float* X, float* R, int* n_iter, int* idx_trace, float* c_trace, int64_t ldt)
{
    if (!h) return fail(MP_ERR_INVALID_ARG, "handle is null");
    if (!Y || !X || !R || !n_iter) return fail(MP_ERR_INVALID_ARG, "null host pointer");
    if (B < 1 || ldy < h->N || max_iter < 0 || !(eps >= 0.0f)) return fail(MP_ERR_INVALID_ARG, "invalid sizes");
    const bool traced = idx_trace || c_trace;
    if (traced && ldt < max_iter) return fail(MP_ERR_INVALID_ARG, "need ldt >= max_iter");
    DeviceGuard g(h->device);
    const int N = h->N, M = h->M;
    const int64_t ldy_d = round_up(N, 4);                               // device rows: 16-byte aligned whatever the host stride is
    const size_t wsb = mp_workspace_bytes(N, M, B);
    mp_status st = grow(&h->ws, &h->ws_cap, wsb);
    if (st != MP_OK) return st;
    const size_t o_Y = 0, o_X = o_Y + up256(sizeof(float) * (size_t)B * ldy_d), o_R = o_X + up256(sizeof(float) * (size_t)B * M),
                 o_n = o_R + up256(sizeof(float) * (size_t)B * N), o_it = o_n + up256(sizeof(int) * (size_t)B),
                 o_ct = o_it + (traced ? up256(sizeof(int) * (size_t)B * max_iter) : 0),
                 total = o_ct + (traced ? up256(sizeof(float) * (size_t)B * max_iter) : 0);
    st = grow(&h->io, &h->io_cap, total);
    if (st != MP_OK) return st;
    char* io = static_cast<char*>(h->io);
    float* dY = reinterpret_cast<float*>(io + o_Y);
    float* dX = reinterpret_cast<float*>(io + o_X);
    float* dR = reinterpret_cast<float*>(io + o_R);
    int* dn = reinterpret_cast<int*>(io + o_n);
    int* dit = traced ? reinterpret_cast<int*>(io + o_it) : nullptr;
    float* dct = traced ? reinterpret_cast<float*>(io + o_ct) : nullptr;
    cudaStream_t s = h->stream;
    SyncOnExit drain(s);
    MP_CUDA(cudaMemcpy2DAsync(dY, sizeof(float) * (size_t)ldy_d, Y, sizeof(float) * (size_t)ldy, sizeof(float) * (size_t)N, (size_t)B,
                              cudaMemcpyHostToDevice, s));
    if (B == 1)
        st = mp_recover(h->psi, N, M, h->ld, dY, eps, max_iter, dX, dR, dn, dit, dct, h->ws, h->ws_cap, s);
    else
        st = mp_recover_batched_traced(h->psi, N, M, h->ld, dY, ldy_d, B, eps, max_iter, dX, dR, dn, dit, dct, max_iter, h->ws, h->ws_cap, s);
    if (st != MP_OK) return st;
    MP_CUDA(cudaMemcpyAsync(X, dX, sizeof(float) * (size_t)B * M, cudaMemcpyDeviceToHost, s));
    MP_CUDA(cudaMemcpyAsync(R, dR, sizeof(float) * (size_t)B * N, cudaMemcpyDeviceToHost, s));
    MP_CUDA(cudaMemcpyAsync(n_iter, dn, sizeof(int) * (size_t)B, cudaMemcpyDeviceToHost, s));
    if (traced && max_iter > 0) {                                      // whole trace rows: entries t >= n_iter[b] are unspecified
        if (idx_trace) MP_CUDA(cudaMemcpy2DAsync(idx_trace, sizeof(int) * (size_t)ldt, dit, sizeof(int) * (size_t)max_iter,
                                                 sizeof(int) * (size_t)max_iter, (size_t)B, cudaMemcpyDeviceToHost, s));
        if (c_trace) MP_CUDA(cudaMemcpy2DAsync(c_trace, sizeof(float) * (size_t)ldt, dct, sizeof(float) * (size_t)max_iter,
                                               sizeof(float) * (size_t)max_iter, (size_t)B, cudaMemcpyDeviceToHost, s));
    }
    MP_CUDA(cudaStreamSynchronize(s));
    drain.armed = false;
    return MP_OK;
}

mp_status mp_recover_host_h(mp_dictionary* h, const float* y, float eps, int max_iter,
                            float* x, float* r, int* n_iter, int* idx_trace, float* c_trace)
{
    if (!h) return fail(MP_ERR_INVALID_ARG, "handle is null");
    return mp_recover_batched_host_h(h, y, h->N, 1, eps, max_iter, x, r, n_iter, idx_trace, c_trace, max_iter);
}

}  // extern "C"
