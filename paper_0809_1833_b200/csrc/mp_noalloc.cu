// mp_noalloc.cu -- mp_recover_noalloc: the single-signal MP loop (Eq. 8-12) for callers that have no device
// memory to hand over as a workspace and no way of getting any.
//
// Who that is: code that runs inside somebody else's process and memory budget.  A plug-in of an inference server or of a
// numerical framework whose own pool has already claimed the whole device finds cudaMalloc failing, or forbidden by the host's
// rules; a service loop with a latency bound cannot afford cudaMalloc either, because it may stall the whole device while the
// driver maps memory.  Every other solver of this library asks such a caller for a `workspace`, which it cannot produce.
//
// What is done instead: the register-streaming persistent kernel (mp_persistent_ldg.cu, "algo 3", the kernel the headline
// configuration runs) needs only a small scratch area next to its inputs and outputs -- one 256-byte control block (grid
// barrier counter, three rotating argmax key slots) and the float64 accumulator of x~ (M doubles).  Here that area is a
// file-scope __device__ array, part of the library image: every GPU on which this library's code gets loaded holds its
// kNoAllocScratchBytes (about 512 KiB) from then until the process exits, whether this entry point is ever called or not.
//
// Host code cannot use the array's name as a pointer: on the host side the name is only a handle by which the runtime finds the
// symbol.  The device address comes from cudaGetSymbolAddress, asked once per device with that device current (the first call
// on a device does it, under a lock), and it is that address the kernel receives as its `ctrl` / `x64` arguments.
#include <mutex>

#include "mp_internal.h"

namespace mp {

constexpr int kNoAllocMaxM = MP_NOALLOC_MAX_M;                                        // atoms (include/mp_b200.h)
constexpr size_t kNoAllocScratchBytes = 256 + sizeof(double) * (size_t)kNoAllocMaxM;   // control block + float64 x~
static __device__ __align__(256) unsigned char g_noalloc_scratch[kNoAllocScratchBytes];

constexpr int kNoAllocMaxDevices = 64;
static std::mutex g_noalloc_mutex;
static void* g_noalloc_ptr[kNoAllocMaxDevices];                                        // device address of the array, per device ordinal

// The device address of g_noalloc_scratch on the CURRENT device.  Looked up once per device; later calls only read the table.
static mp_status noalloc_scratch_address(void** out)
{
    int dev = -1;
    MP_CUDA(cudaGetDevice(&dev));
    if (dev < 0 || dev >= kNoAllocMaxDevices)
        return fail(MP_ERR_UNSUPPORTED, "mp_recover_noalloc: device ordinal %d is outside the %d it keeps an address for", dev, kNoAllocMaxDevices);
    std::lock_guard<std::mutex> lock(g_noalloc_mutex);
    if (!g_noalloc_ptr[dev]) {
        void* ptr = nullptr;
        MP_CUDA(cudaGetSymbolAddress((void**)&ptr, g_noalloc_scratch));
        if (!ptr) return fail(MP_ERR_CUDA, "mp_recover_noalloc: cudaGetSymbolAddress returned a null address");
        g_noalloc_ptr[dev] = ptr;
    }
    *out = g_noalloc_ptr[dev];
    return MP_OK;
}

}  // namespace mp

using namespace mp;

extern "C" mp_status mp_recover_noalloc(const float* psi_t, int N, int M, int64_t ld,
                                        const float* y, float eps, int max_iter,
                                        float* x, float* r, int* n_iter,
                                        int* idx_trace, float* c_trace, void* stream)
{
    // the argument rules of mp_recover, checked before anything touches the device
    if (!psi_t) return fail(MP_ERR_INVALID_ARG, "psi_t is null");
    if (N < 1 || M < 1) return fail(MP_ERR_INVALID_ARG, "need N >= 1 and M >= 1 (got N=%d, M=%d)", N, M);
    if (ld < N || (ld & 3)) return fail(MP_ERR_INVALID_ARG, "need ld >= N and ld %% 4 == 0 (got ld=%lld, N=%d)", (long long)ld, N);
    if (reinterpret_cast<uintptr_t>(psi_t) & 15u) return fail(MP_ERR_INVALID_ARG, "psi_t must be 16-byte aligned");
    if (!y || !x || !r || !n_iter) return fail(MP_ERR_INVALID_ARG, "y, x, r and n_iter must be non-null");
    if ((reinterpret_cast<uintptr_t>(y) | reinterpret_cast<uintptr_t>(x) | reinterpret_cast<uintptr_t>(r)) & 3u)
        return fail(MP_ERR_INVALID_ARG, "y, x, r must be 4-byte aligned");
    if (max_iter < 0) return fail(MP_ERR_INVALID_ARG, "max_iter must be >= 0 (got %d)", max_iter);
    if (!(eps >= 0.0f)) return fail(MP_ERR_INVALID_ARG, "eps must be >= 0 and not NaN");
    if (M > kNoAllocMaxM)
        return fail(MP_ERR_UNSUPPORTED, "mp_recover_noalloc: M=%d is beyond the %d atoms its built-in scratch area holds; "
                    "use mp_recover with a caller-provided workspace", M, kNoAllocMaxM);

    void* scratch = nullptr;
    mp_status st = noalloc_scratch_address(&scratch);
    if (st != MP_OK) return st;

    // The two workspace fields the register-streaming kernel reads; the launcher clears both (256 + 8M bytes, one memset on
    // `stream`) before the kernel, so nothing of the previous call -- barrier count, key slots, x~ -- is carried over.
    Workspace ws = {};
    ws.ctrl = static_cast<unsigned long long*>(scratch);
    ws.x64 = reinterpret_cast<double*>(static_cast<unsigned char*>(scratch) + 256);
    ws.bytes = kNoAllocScratchBytes;
    RecoverArgs a{psi_t, N, M, ld, y, eps, max_iter, x, r, n_iter, idx_trace, c_trace};
    return launch_recover_persistent_ldg(a, ws, static_cast<cudaStream_t>(stream));
}
