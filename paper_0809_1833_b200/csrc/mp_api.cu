// mp_api.cu -- the C ABI of libmp_b200.so (include/mp_b200.h): argument validation, workspace layout,
// algorithm dispatch, knobs, and the host-buffer convenience entry points.
#include <atomic>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstring>

#include "mp_internal.h"

namespace mp {

static thread_local char g_err[512] = "";

mp_status fail(mp_status code, const char* fmt, ...)
{
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof(g_err), fmt, ap);
    va_end(ap);
    return code;
}

mp_status cuda_fail(cudaError_t e, const char* what)
{
    return fail(MP_ERR_CUDA, "%s: %s (%s)", what, cudaGetErrorName(e), cudaGetErrorString(e));
}

Options& options()
{
    static Options o;
    return o;
}

static std::atomic<int64_t> g_launches{0};
void count_launch(int n) { g_launches.fetch_add(n, std::memory_order_relaxed); }

mp_status device_info(DeviceInfo* out)
{
    static thread_local DeviceInfo cache;
    int dev = -1;
    MP_CUDA(cudaGetDevice(&dev));
    if (cache.device != dev) {
        DeviceInfo d;
        d.device = dev;
        MP_CUDA(cudaDeviceGetAttribute(&d.sm_count, cudaDevAttrMultiProcessorCount, dev));
        MP_CUDA(cudaDeviceGetAttribute(&d.smem_optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev));
        MP_CUDA(cudaDeviceGetAttribute(&d.coop, cudaDevAttrCooperativeLaunch, dev));
        MP_CUDA(cudaDeviceGetAttribute(&d.l2_bytes, cudaDevAttrL2CacheSize, dev));
        cache = d;
    }
    *out = cache;
    return MP_OK;
}

double l2_scale()
{
    double bytes = (double)options().l2_bytes;
    if (!(bytes > 0.0)) {
        DeviceInfo di;
        bytes = (device_info(&di) == MP_OK && di.l2_bytes > 0) ? (double)di.l2_bytes : kL2TunedBytes;
    }
    options().info_l2_bytes = (int64_t)bytes;
    return bytes / kL2TunedBytes;
}

static size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

size_t workspace_layout(int N, int M, int B, void* base, Workspace* ws)
{
    const size_t Nr = (size_t)round_up(N, 128);
    size_t off = 0;
    char* b = static_cast<char*>(base);
    auto take = [&](size_t bytes) { size_t o = off; off = align_up(off + bytes, 256); return o; };
    const size_t o_ctrl = take(256);
    const size_t o_x64 = take(sizeof(double) * (size_t)B * M);     // must directly follow ctrl (one memset covers both)
    const size_t o_r64 = take(sizeof(double) * (size_t)B * Nr);
    const size_t o_r32 = take(sizeof(float) * (size_t)B * Nr);
    // the lock-step tensor-core kernel always works on 64 key slots and 128 operand rows, whatever B >= 1 is
    const size_t o_keys = take(sizeof(unsigned long long) * 3 * (size_t)(B < 64 ? 64 : B));
    const size_t o_state = take(sizeof(int) * 4 * (size_t)B);
    const size_t o_rs = take(sizeof(float) * 128 * Nr);
    if (ws) {
        ws->ctrl = reinterpret_cast<unsigned long long*>(b + o_ctrl);
        ws->x64 = reinterpret_cast<double*>(b + o_x64);
        ws->r64 = reinterpret_cast<double*>(b + o_r64);
        ws->r32 = reinterpret_cast<float*>(b + o_r32);
        ws->keys = reinterpret_cast<unsigned long long*>(b + o_keys);
        ws->state = reinterpret_cast<int*>(b + o_state);
        ws->rs = reinterpret_cast<float*>(b + o_rs);
        ws->bytes = off;
    }
    return off;
}

static bool aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }
static bool aligned4(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 3u) == 0; }

static mp_status check_dictionary(const float* psi_t, int N, int M, int64_t ld)
{
    if (!psi_t) return fail(MP_ERR_INVALID_ARG, "psi_t is null");
    if (N < 1 || M < 1) return fail(MP_ERR_INVALID_ARG, "need N >= 1 and M >= 1 (got N=%d, M=%d)", N, M);
    if (ld < N || (ld & 3)) return fail(MP_ERR_INVALID_ARG, "need ld >= N and ld %% 4 == 0 (got ld=%lld, N=%d)", (long long)ld, N);
    if (!aligned16(psi_t)) return fail(MP_ERR_INVALID_ARG, "psi_t must be 16-byte aligned");
    return MP_OK;
}

}  // namespace mp

namespace {
// Device buffers of the host-buffer entry points: stream-ordered allocations from the device's default memory pool, whose
// release threshold is raised once so that repeated calls reuse the memory instead of going back to the driver
// (cudaMalloc + cudaFree of 256 MiB per call cost ~2 ms of a 46 ms end-to-end solve).
struct DevBuf {
    void* p = nullptr;
    cudaStream_t s = nullptr;
    ~DevBuf() { if (p) cudaFreeAsync(p, s); }
    cudaError_t alloc(size_t bytes, cudaStream_t stream)
    {
        static thread_local int pool_dev = -1;
        int dev = -1;
        if (cudaGetDevice(&dev) == cudaSuccess && dev != pool_dev) {
            cudaMemPool_t pool;
            if (cudaDeviceGetDefaultMemPool(&pool, dev) == cudaSuccess) {
                unsigned long long keep = ~0ull;
                (void)cudaMemPoolSetAttribute(pool, cudaMemPoolAttrReleaseThreshold, &keep);
            }
            pool_dev = dev;
        }
        s = stream;
        return cudaMallocAsync(&p, bytes ? bytes : 16, stream);
    }
    template <class T> T* as() { return static_cast<T*>(p); }
};
struct Stream {
    cudaStream_t s = nullptr;
    // Synchronise first: an error return must not leave a copy from or to the caller's host buffers in flight (the caller may
    // free them as soon as the call is back); after a successful call the stream is idle and this costs nothing.
    ~Stream() { if (s) { (void)cudaStreamSynchronize(s); cudaStreamDestroy(s); } }
};
}  // namespace

using namespace mp;

extern "C" {

size_t mp_workspace_bytes(int N, int M, int B)
{
    if (N < 1 || M < 1 || B < 1) return 0;
    return workspace_layout(N, M, B, nullptr, nullptr);
}

const char* mp_last_error(void) { return g_err; }

int64_t mp_launch_count(void) { return g_launches.load(std::memory_order_relaxed); }

static std::atomic<int64_t>* option_slot(const char* name)
{
    Options& o = options();
    if (!name) return nullptr;
    if (!strcmp(name, "algo")) return &o.algo;
    if (!strcmp(name, "warps")) return &o.warps;
    if (!strcmp(name, "slot_bytes")) return &o.slot_bytes;
    if (!strcmp(name, "depth")) return &o.depth;
    if (!strcmp(name, "grid")) return &o.grid;
    if (!strcmp(name, "chunk")) return &o.chunk;
    if (!strcmp(name, "batched_algo")) return &o.batched_algo;
    if (!strcmp(name, "batched_coop")) return &o.batched_coop;
    if (!strcmp(name, "info_algo")) return &o.info_algo;
    if (!strcmp(name, "info_batched_algo")) return &o.info_batched_algo;
    if (!strcmp(name, "info_l2_pingpong")) return &o.info_l2_pingpong;
    if (!strcmp(name, "info_l2_resident_mb")) return &o.info_l2_resident_mb;
    if (!strcmp(name, "info_l2_dynamic")) return &o.info_l2_dynamic;
    if (!strcmp(name, "omp_algo")) return &o.omp_algo;
    if (!strcmp(name, "info_omp_algo")) return &o.info_omp_algo;
    if (!strcmp(name, "l2_resident_mb")) return &o.l2_resident_mb;
    if (!strcmp(name, "l2_demote")) return &o.l2_demote;
    if (!strcmp(name, "l2_bytes")) return &o.l2_bytes;
    if (!strcmp(name, "info_l2_bytes")) return &o.info_l2_bytes;
    if (!strcmp(name, "balance")) return &o.balance;
    if (!strcmp(name, "pingpong")) return &o.pingpong;
    if (!strcmp(name, "pin_margin_pct")) return &o.pin_margin_pct;
    if (!strcmp(name, "many_cluster")) return &o.many_cluster;
    if (!strcmp(name, "many_threads")) return &o.many_threads;
    if (!strcmp(name, "many_stat")) return &o.many_stat;
    if (!strcmp(name, "many_l2_mb")) return &o.many_l2_mb;
    if (!strcmp(name, "info_many_cluster")) return &o.info_many_cluster;
    if (!strcmp(name, "info_many_stat")) return &o.info_many_stat;
    if (!strcmp(name, "info_many_clusters")) return &o.info_many_clusters;
    if (!strcmp(name, "info_many_threads")) return &o.info_many_threads;
    if (!strcmp(name, "info_tc_clusters")) return &o.info_tc_clusters;
    if (!strcmp(name, "info_tc_at")) return &o.info_tc_at;
    if (!strcmp(name, "info_tc_stages")) return &o.info_tc_stages;
    return nullptr;
}

mp_status mp_set_int(const char* name, int64_t value)
{
    std::atomic<int64_t>* s = option_slot(name);
    if (!s) return fail(MP_ERR_INVALID_ARG, "unknown option '%s'", name ? name : "(null)");
    if (value < 0) return fail(MP_ERR_INVALID_ARG, "option '%s' must be >= 0", name);
    *s = value;
    return MP_OK;
}

mp_status mp_get_int(const char* name, int64_t* value)
{
    std::atomic<int64_t>* s = option_slot(name);
    if (!s || !value) return fail(MP_ERR_INVALID_ARG, "unknown option or null output");
    *value = *s;
    return MP_OK;
}

mp_status mp_normalize_columns(float* psi_t, int N, int M, int64_t ld, float* norms_out, void* stream)
{
    mp_status st = check_dictionary(psi_t, N, M, ld);
    if (st != MP_OK) return st;
    return launch_normalize(psi_t, N, M, ld, norms_out, static_cast<cudaStream_t>(stream));
}

mp_status mp_transpose_rowmajor(const float* psi, int N, int M, int64_t ldr, float* psi_t, int64_t ld, void* stream)
{
    if (!psi) return fail(MP_ERR_INVALID_ARG, "psi is null");
    if (ldr < M) return fail(MP_ERR_INVALID_ARG, "need ldr >= M (got ldr=%lld, M=%d)", (long long)ldr, M);
    mp_status st = check_dictionary(psi_t, N, M, ld);
    if (st != MP_OK) return st;
    const char* a = reinterpret_cast<const char*>(psi);
    const char* b = reinterpret_cast<const char*>(psi_t);
    if (a < b + sizeof(float) * (size_t)M * ld && b < a + sizeof(float) * (size_t)N * ldr)
        return fail(MP_ERR_INVALID_ARG, "psi and psi_t overlap: the transpose is out of place");
    return launch_transpose_rowmajor(psi, N, M, ldr, psi_t, ld, static_cast<cudaStream_t>(stream));
}

mp_status mp_encode_sparse(const float* psi_t, int N, int M, int64_t ld, const int* idx, const float* val, int K,
                           float* y, void* stream)
{
    mp_status st = check_dictionary(psi_t, N, M, ld);
    if (st != MP_OK) return st;
    if (K < 0) return fail(MP_ERR_INVALID_ARG, "need K >= 0 (got %d)", K);
    if (!y || (K > 0 && (!idx || !val))) return fail(MP_ERR_INVALID_ARG, "y (and idx, val when K > 0) must be non-null");
    return launch_encode_sparse(psi_t, N, M, ld, idx, val, K, y, static_cast<cudaStream_t>(stream));
}

mp_status mp_reconstruction_error(const float* x_hat, const float* x, int M, double* err_pct, void* stream)
{
    if (!x_hat || !x || !err_pct) return fail(MP_ERR_INVALID_ARG, "x_hat, x and err_pct must be non-null");
    if (M < 1) return fail(MP_ERR_INVALID_ARG, "need M >= 1 (got %d)", M);
    if (reinterpret_cast<uintptr_t>(err_pct) & 7u) return fail(MP_ERR_INVALID_ARG, "err_pct must be 8-byte aligned");
    return launch_reconstruction_error(x_hat, x, M, err_pct, static_cast<cudaStream_t>(stream));
}

mp_status mp_recover(const float* psi_t, int N, int M, int64_t ld,
                     const float* y, float eps, int max_iter,
                     float* x, float* r, int* n_iter,
                     int* idx_trace, float* c_trace,
                     void* workspace, size_t workspace_bytes, void* stream)
{
    mp_status st = check_dictionary(psi_t, N, M, ld);
    if (st != MP_OK) return st;
    if (!y || !x || !r || !n_iter) return fail(MP_ERR_INVALID_ARG, "y, x, r and n_iter must be non-null");
    if (!aligned4(y) || !aligned4(x) || !aligned4(r)) return fail(MP_ERR_INVALID_ARG, "y, x, r must be 4-byte aligned");
    if (max_iter < 0) return fail(MP_ERR_INVALID_ARG, "max_iter must be >= 0 (got %d)", max_iter);
    if (!(eps >= 0.0f)) return fail(MP_ERR_INVALID_ARG, "eps must be >= 0 and not NaN");
    const size_t need = mp_workspace_bytes(N, M, 1);
    if (!workspace || (reinterpret_cast<uintptr_t>(workspace) & 255u) || workspace_bytes < need)
        return fail(MP_ERR_WORKSPACE, "workspace must be non-null, 256-byte aligned and >= %zu bytes (got %zu)", need, workspace_bytes);

    Workspace ws;
    workspace_layout(N, M, 1, workspace, &ws);
    RecoverArgs a{psi_t, N, M, ld, y, eps, max_iter, x, r, n_iter, idx_trace, c_trace};
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    const int64_t algo = options().algo;
    int64_t use = algo;
    if (use < 1 || use > 4)
        use = many_single_stationary(N, M) ? 4 : persistent_ldg_supported(N, M) ? 3 : persistent_supported(N, M) ? 1 : 2;
    options().info_algo = use;
    if (use == 4) {                                                 // one thread-block cluster, dictionary stationary in shared memory
        if (!many_supported(N, M)) return fail(MP_ERR_UNSUPPORTED, "algo 4 (cluster kernel) needs N <= 2048 (got %d)", N);
        ManyArgs m{psi_t, N, M, ld, 0, y, N, 1, eps, max_iter, x, r, n_iter, idx_trace, c_trace, max_iter};
        return launch_recover_many(m, reinterpret_cast<unsigned int*>(ws.ctrl), s);
    }
    if (use == 3) return launch_recover_persistent_ldg(a, ws, s);
    if (use == 1) return launch_recover_persistent(a, ws, s);
    return launch_recover_streamloop(a, ws, s);
}

mp_status mp_recover_batched_traced(const float* psi_t, int N, int M, int64_t ld,
                                    const float* Y, int64_t ldy, int B,
                                    float eps, int max_iter,
                                    float* X, float* R, int* n_iter,
                                    int* idx_trace, float* c_trace, int64_t ldt,
                                    void* workspace, size_t workspace_bytes, void* stream)
{
    mp_status st = check_dictionary(psi_t, N, M, ld);
    if (st != MP_OK) return st;
    if (B < 1) return fail(MP_ERR_INVALID_ARG, "need B >= 1 (got %d)", B);
    if (!Y || !X || !R || !n_iter) return fail(MP_ERR_INVALID_ARG, "Y, X, R and n_iter must be non-null");
    if (!aligned16(Y) || !aligned16(X) || !aligned16(R)) return fail(MP_ERR_INVALID_ARG, "Y, X, R must be 16-byte aligned");
    if (ldy < N || (ldy & 3)) return fail(MP_ERR_INVALID_ARG, "need ldy >= N and ldy %% 4 == 0");
    if (max_iter < 0) return fail(MP_ERR_INVALID_ARG, "max_iter must be >= 0 (got %d)", max_iter);
    if (!(eps >= 0.0f)) return fail(MP_ERR_INVALID_ARG, "eps must be >= 0 and not NaN");
    if ((idx_trace || c_trace) && ldt < max_iter) return fail(MP_ERR_INVALID_ARG, "need ldt >= max_iter");
    const size_t need = mp_workspace_bytes(N, M, B);
    if (!workspace || (reinterpret_cast<uintptr_t>(workspace) & 255u) || workspace_bytes < need)
        return fail(MP_ERR_WORKSPACE, "workspace must be non-null, 256-byte aligned and >= %zu bytes (got %zu)", need, workspace_bytes);
    Workspace ws;
    workspace_layout(N, M, B, workspace, &ws);
    BatchedArgs a{psi_t, N, M, ld, Y, ldy, B, eps, max_iter, X, R, n_iter, idx_trace, c_trace, ldt};
    return launch_recover_batched(a, ws, static_cast<cudaStream_t>(stream));
}

mp_status mp_recover_batched(const float* psi_t, int N, int M, int64_t ld,
                             const float* Y, int64_t ldy, int B,
                             float eps, int max_iter,
                             float* X, float* R, int* n_iter,
                             void* workspace, size_t workspace_bytes, void* stream)
{
    return mp_recover_batched_traced(psi_t, N, M, ld, Y, ldy, B, eps, max_iter, X, R, n_iter, nullptr, nullptr, 0,
                                     workspace, workspace_bytes, stream);
}

mp_status mp_correlate_batched(const float* psi_t, int N, int M, int64_t ld,
                               const float* Y, int64_t ldy, int B, float* C,
                               void* workspace, size_t workspace_bytes, void* stream)
{
    mp_status st = check_dictionary(psi_t, N, M, ld);
    if (st != MP_OK) return st;
    if (B < 1 || B > 64) return fail(MP_ERR_INVALID_ARG, "need 1 <= B <= 64 (got %d)", B);
    if (!Y || !C) return fail(MP_ERR_INVALID_ARG, "Y and C must be non-null");
    if (!aligned16(Y) || !aligned16(C)) return fail(MP_ERR_INVALID_ARG, "Y and C must be 16-byte aligned");
    if (ldy < N || (ldy & 3)) return fail(MP_ERR_INVALID_ARG, "need ldy >= N and ldy %% 4 == 0");
    const int Bw = B < 2 ? 2 : B;                                   // the batched workspace layout (B > 1)
    const size_t scratch_off = (mp_workspace_bytes(N, M, Bw) + 255) / 256 * 256;
    const size_t need = scratch_off + sizeof(float) * ((size_t)Bw * M + (size_t)Bw * N) + sizeof(int) * (size_t)Bw + 512;
    if (!workspace || (reinterpret_cast<uintptr_t>(workspace) & 255u) || workspace_bytes < need)
        return fail(MP_ERR_WORKSPACE, "workspace must be non-null, 256-byte aligned and >= %zu bytes (got %zu)", need, workspace_bytes);
    Workspace ws;
    workspace_layout(N, M, Bw, workspace, &ws);
    // scratch X, R, n_iter of the one iteration that is run
    char* sc = static_cast<char*>(workspace) + scratch_off;
    float* X = reinterpret_cast<float*>(sc);
    float* R = X + (size_t)Bw * M;
    int* n_iter = reinterpret_cast<int*>(R + (size_t)Bw * N);
    BatchedArgs a{psi_t, N, M, ld, Y, ldy, B, 0.0f, 1, X, R, n_iter, nullptr, nullptr, 0};
    return launch_recover_batched_tc(a, ws, C, static_cast<cudaStream_t>(stream));
}

size_t mp_correlate_batched_workspace_bytes(int N, int M, int B)
{
    if (N < 1 || M < 1 || B < 1 || B > 64) return 0;
    const int Bw = B < 2 ? 2 : B;
    const size_t scratch_off = (mp_workspace_bytes(N, M, Bw) + 255) / 256 * 256;
    return scratch_off + sizeof(float) * ((size_t)Bw * M + (size_t)Bw * N) + sizeof(int) * (size_t)Bw + 512;
}

size_t mp_workspace_bytes_many(int N, int M, int P)
{
    if (N < 1 || M < 1 || P < 1) return 0;
    return 256 + mp_workspace_bytes(N, M, 1);
}

mp_status mp_recover_many(const float* psi_t, int N, int M, int64_t ld, int64_t problem_stride,
                          const float* Y, int64_t ldy, int P, float eps, int max_iter,
                          float* X, float* R, int* n_iter,
                          int* idx_trace, float* c_trace, int64_t ldt,
                          void* workspace, size_t workspace_bytes, void* stream)
{
    mp_status st = check_dictionary(psi_t, N, M, ld);
    if (st != MP_OK) return st;
    if (P < 1) return fail(MP_ERR_INVALID_ARG, "need P >= 1 (got %d)", P);
    if (problem_stride != 0 && (problem_stride < (int64_t)M * ld || (problem_stride & 3)))
        return fail(MP_ERR_INVALID_ARG, "problem_stride must be 0 (one shared dictionary) or >= M*ld and a multiple of 4 floats");
    if (!Y || !X || !R || !n_iter) return fail(MP_ERR_INVALID_ARG, "Y, X, R and n_iter must be non-null");
    if (ldy < N) return fail(MP_ERR_INVALID_ARG, "need ldy >= N");
    if (max_iter < 0) return fail(MP_ERR_INVALID_ARG, "max_iter must be >= 0 (got %d)", max_iter);
    if (!(eps >= 0.0f)) return fail(MP_ERR_INVALID_ARG, "eps must be >= 0 and not NaN");
    if ((idx_trace || c_trace) && ldt < max_iter) return fail(MP_ERR_INVALID_ARG, "need ldt >= max_iter");
    const size_t need = mp_workspace_bytes_many(N, M, P);
    if (!workspace || (reinterpret_cast<uintptr_t>(workspace) & 255u) || workspace_bytes < need)
        return fail(MP_ERR_WORKSPACE, "workspace must be non-null, 256-byte aligned and >= %zu bytes (got %zu)", need, workspace_bytes);
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    if (many_supported(N, M)) {
        ManyArgs a{psi_t, N, M, ld, problem_stride, Y, ldy, P, eps, max_iter, X, R, n_iter, idx_trace, c_trace, ldt};
        return launch_recover_many(a, static_cast<unsigned int*>(workspace), s);
    }
    // long residuals (N > 2048): these are not "small" problems -- one grid-wide single-signal solve after another
    char* ws1 = static_cast<char*>(workspace) + 256;
    for (int q = 0; q < P; q++) {
        st = mp_recover(psi_t + (int64_t)q * problem_stride, N, M, ld, Y + (int64_t)q * ldy, eps, max_iter,
                        X + (int64_t)q * M, R + (int64_t)q * N, n_iter + q,
                        idx_trace ? idx_trace + (int64_t)q * ldt : nullptr, c_trace ? c_trace + (int64_t)q * ldt : nullptr,
                        ws1, workspace_bytes - 256, s);
        if (st != MP_OK) return st;
    }
    options().info_many_cluster = 0;
    return MP_OK;
}

// ---------------------------------------------------------------------------------------------------------
// host-buffer entry points
// ---------------------------------------------------------------------------------------------------------

mp_status mp_recover_batched_host(const float* psi_t, int N, int M, int64_t ld, int normalize,
                                  const float* Y, int64_t ldy, int B, float eps, int max_iter,
                                  float* X, float* R, int* n_iter)
{
    if (!psi_t || !Y || !X || !R || !n_iter) return fail(MP_ERR_INVALID_ARG, "null host pointer");
    if (N < 1 || M < 1 || B < 1 || ld < N || (ld & 3) || ldy < N || (ldy & 3) || max_iter < 0 || !(eps >= 0.0f))
        return fail(MP_ERR_INVALID_ARG, "invalid sizes");
    Stream st;
    MP_CUDA(cudaStreamCreateWithFlags(&st.s, cudaStreamNonBlocking));
    DevBuf d_psi, d_Y, d_X, d_R, d_n, d_ws;
    const size_t wsb = mp_workspace_bytes(N, M, B);
    MP_CUDA(d_psi.alloc(sizeof(float) * (size_t)M * ld, st.s));
    MP_CUDA(d_Y.alloc(sizeof(float) * (size_t)B * ldy, st.s));
    MP_CUDA(d_X.alloc(sizeof(float) * (size_t)B * M, st.s));
    MP_CUDA(d_R.alloc(sizeof(float) * (size_t)B * N, st.s));
    MP_CUDA(d_n.alloc(sizeof(int) * (size_t)B, st.s));
    MP_CUDA(d_ws.alloc(wsb, st.s));
    MP_CUDA(cudaMemcpyAsync(d_psi.p, psi_t, sizeof(float) * (size_t)M * ld, cudaMemcpyHostToDevice, st.s));
    MP_CUDA(cudaMemcpyAsync(d_Y.p, Y, sizeof(float) * (size_t)B * ldy, cudaMemcpyHostToDevice, st.s));
    mp_status rc;
    if (normalize) {
        rc = mp_normalize_columns(d_psi.as<float>(), N, M, ld, nullptr, st.s);
        if (rc != MP_OK) return rc;
    }
    rc = mp_recover_batched(d_psi.as<float>(), N, M, ld, d_Y.as<float>(), ldy, B, eps, max_iter,
                            d_X.as<float>(), d_R.as<float>(), d_n.as<int>(), d_ws.p, wsb, st.s);
    if (rc != MP_OK) return rc;
    MP_CUDA(cudaMemcpyAsync(X, d_X.p, sizeof(float) * (size_t)B * M, cudaMemcpyDeviceToHost, st.s));
    MP_CUDA(cudaMemcpyAsync(R, d_R.p, sizeof(float) * (size_t)B * N, cudaMemcpyDeviceToHost, st.s));
    MP_CUDA(cudaMemcpyAsync(n_iter, d_n.p, sizeof(int) * (size_t)B, cudaMemcpyDeviceToHost, st.s));
    MP_CUDA(cudaStreamSynchronize(st.s));
    return MP_OK;
}

mp_status mp_recover_host(const float* psi_t, int N, int M, int64_t ld, int normalize,
                          const float* y, float eps, int max_iter,
                          float* x, float* r, int* n_iter, int* idx_trace, float* c_trace)
{
    if (!psi_t || !y || !x || !r || !n_iter) return fail(MP_ERR_INVALID_ARG, "null host pointer");
    if (N < 1 || M < 1 || ld < N || (ld & 3) || max_iter < 0 || !(eps >= 0.0f))
        return fail(MP_ERR_INVALID_ARG, "invalid sizes");
    Stream st;
    MP_CUDA(cudaStreamCreateWithFlags(&st.s, cudaStreamNonBlocking));
    DevBuf d_psi, d_y, d_x, d_r, d_n, d_ws, d_it, d_ct;
    const size_t wsb = mp_workspace_bytes(N, M, 1);
    MP_CUDA(d_psi.alloc(sizeof(float) * (size_t)M * ld, st.s));
    MP_CUDA(d_y.alloc(sizeof(float) * (size_t)N, st.s));
    MP_CUDA(d_x.alloc(sizeof(float) * (size_t)M, st.s));
    MP_CUDA(d_r.alloc(sizeof(float) * (size_t)N, st.s));
    MP_CUDA(d_n.alloc(sizeof(int), st.s));
    MP_CUDA(d_ws.alloc(wsb, st.s));
    if (idx_trace) MP_CUDA(d_it.alloc(sizeof(int) * (size_t)max_iter, st.s));
    if (c_trace) MP_CUDA(d_ct.alloc(sizeof(float) * (size_t)max_iter, st.s));
    MP_CUDA(cudaMemcpyAsync(d_psi.p, psi_t, sizeof(float) * (size_t)M * ld, cudaMemcpyHostToDevice, st.s));
    MP_CUDA(cudaMemcpyAsync(d_y.p, y, sizeof(float) * (size_t)N, cudaMemcpyHostToDevice, st.s));
    mp_status rc;
    if (normalize) {
        rc = mp_normalize_columns(d_psi.as<float>(), N, M, ld, nullptr, st.s);
        if (rc != MP_OK) return rc;
    }
    rc = mp_recover(d_psi.as<float>(), N, M, ld, d_y.as<float>(), eps, max_iter, d_x.as<float>(), d_r.as<float>(),
                    d_n.as<int>(), idx_trace ? d_it.as<int>() : nullptr, c_trace ? d_ct.as<float>() : nullptr,
                    d_ws.p, wsb, st.s);
    if (rc != MP_OK) return rc;
    MP_CUDA(cudaMemcpyAsync(x, d_x.p, sizeof(float) * (size_t)M, cudaMemcpyDeviceToHost, st.s));
    MP_CUDA(cudaMemcpyAsync(r, d_r.p, sizeof(float) * (size_t)N, cudaMemcpyDeviceToHost, st.s));
    MP_CUDA(cudaMemcpyAsync(n_iter, d_n.p, sizeof(int), cudaMemcpyDeviceToHost, st.s));
    MP_CUDA(cudaStreamSynchronize(st.s));
    if (idx_trace || c_trace) {
        const int t = *n_iter;
        if (idx_trace && t > 0) MP_CUDA(cudaMemcpyAsync(idx_trace, d_it.p, sizeof(int) * (size_t)t, cudaMemcpyDeviceToHost, st.s));
        if (c_trace && t > 0) MP_CUDA(cudaMemcpyAsync(c_trace, d_ct.p, sizeof(float) * (size_t)t, cudaMemcpyDeviceToHost, st.s));
        MP_CUDA(cudaStreamSynchronize(st.s));
    }
    return MP_OK;
}

}  // extern "C"
