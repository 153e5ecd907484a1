// mp_batched.cu -- B signals sharing one dictionary.
// Dispatch of the batched path, and batched_algo 2: one single-signal solve after another on the stream
// (the FP32-CUDA-core baseline of the tensor-core kernel in mp_batched_tc.cu).
#include "mp_common.cuh"
#include "mp_internal.h"

namespace mp {

static mp_status launch_batched_sequential(const BatchedArgs& a, const Workspace& ws, cudaStream_t stream)
{
    Workspace one;
    // the single-signal layout is a prefix-compatible carve-up of the same buffer
    workspace_layout(a.N, a.M, 1, ws.ctrl, &one);
    for (int b = 0; b < a.B; b++) {
        RecoverArgs s{a.psi_t, a.N, a.M, a.ld, a.Y + (int64_t)b * a.ldy, a.eps, a.max_iter,
                      a.X + (int64_t)b * a.M, a.R + (int64_t)b * a.N, a.n_iter + b,
                      a.idx_trace ? a.idx_trace + (int64_t)b * a.ldt : nullptr,
                      a.c_trace ? a.c_trace + (int64_t)b * a.ldt : nullptr};
        const int64_t algo = options().algo;
        mp_status st = (algo != 2 && algo != 1 && persistent_ldg_supported(a.N, a.M)) ? launch_recover_persistent_ldg(s, one, stream)
                       : (algo != 2 && persistent_supported(a.N, a.M))                 ? launch_recover_persistent(s, one, stream)
                                                                                       : launch_recover_streamloop(s, one, stream);
        if (st != MP_OK) return st;
    }
    return MP_OK;
}

// batched_algo 3: one thread-block cluster per signal, all clusters reading the one dictionary (mp_many.cu with problem stride 0).
static mp_status launch_batched_clusters(const BatchedArgs& a, const Workspace& ws, cudaStream_t stream)
{
    ManyArgs m{a.psi_t, a.N, a.M, a.ld, 0, a.Y, a.ldy, a.B, a.eps, a.max_iter, a.X, a.R, a.n_iter, a.idx_trace, a.c_trace, a.ldt};
    return launch_recover_many(m, reinterpret_cast<unsigned int*>(ws.ctrl), stream);
}

// batched_algo 0 = auto: the lock-step tensor-core kernel (mp_batched_tc.cu) in groups of at most 64 signals when the
// shape fits it and the dictionary is larger than 1.5 MB, else one cluster per signal (N <= 2048), else the sequential baseline.  1 = tensor-core kernel or error.
// 2 = sequential.  3 = one cluster per signal or error.
mp_status launch_recover_batched(const BatchedArgs& a, const Workspace& ws, cudaStream_t stream)
{
    const int64_t algo = options().batched_algo;
    // "info_batched_algo": which of the three ran (1 tensor-core lock-step, 2 sequential, 3 clusters) -- the only way to see that
    // auto dispatch left the tensor-core kernel, e.g. after a refused cooperative launch (a 20x slower solve that still succeeds)
    auto ran = [](int64_t which, mp_status st) { if (st == MP_OK) options().info_batched_algo = which; return st; };
    if (algo == 2) return ran(2, launch_batched_sequential(a, ws, stream));
    if (algo == 3) return ran(3, launch_batched_clusters(a, ws, stream));
    const int group = a.B < 64 ? a.B : 64;
    // one signal is not a batch: the single-signal kernels stream the dictionary at the HBM / L2 rate, the lock-step kernel would
    // run a 128-row contraction for one useful row
    if (algo == 0 && a.B == 1) return ran(2, launch_batched_sequential(a, ws, stream));
    // measured (B = 64): 1 MiB dictionary 0.50 ms with clusters against 0.75 ms lock-step; 4 MiB 2.7 against 1.8 ms; 16 MiB 18 against 4.7
    if (algo == 0 && many_supported(a.N, a.M) && 4.0 * a.N * a.M <= 1.5e6) return ran(3, launch_batched_clusters(a, ws, stream));
    if (algo == 0 && !batched_tc_supported(a.N, a.M, group))
        return many_supported(a.N, a.M) ? ran(3, launch_batched_clusters(a, ws, stream)) : ran(2, launch_batched_sequential(a, ws, stream));
    for (int b0 = 0; b0 < a.B; b0 += 64) {
        BatchedArgs g = a;
        g.B = a.B - b0 < 64 ? a.B - b0 : 64;
        g.Y = a.Y + (int64_t)b0 * a.ldy;
        g.X = a.X + (int64_t)b0 * a.M;
        g.R = a.R + (int64_t)b0 * a.N;
        g.n_iter = a.n_iter + b0;
        g.idx_trace = a.idx_trace ? a.idx_trace + (int64_t)b0 * a.ldt : nullptr;
        g.c_trace = a.c_trace ? a.c_trace + (int64_t)b0 * a.ldt : nullptr;
        mp_status st = launch_recover_batched_tc(g, ws, nullptr, stream);   // groups reuse the workspace in stream order
        if (st == MP_ERR_UNSUPPORTED && algo == 0 && b0 == 0)              // e.g. the cooperative cluster launch was refused: nothing ran yet.
            // The solve still succeeds on a much slower kernel; mp_last_error() keeps the refusal's text and info_batched_algo says 2 or 3.
            return many_supported(a.N, a.M) ? ran(3, launch_batched_clusters(a, ws, stream)) : ran(2, launch_batched_sequential(a, ws, stream));
        if (st != MP_OK) return st;
    }
    return ran(1, MP_OK);
}

}  // namespace mp
