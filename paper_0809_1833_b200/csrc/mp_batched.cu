// mp_batched.cu -- B signals sharing one dictionary.
// batched_algo 2: one single-signal solve after another on the stream (baseline for the fused path).
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
        mp_status st = (options().algo != 2 && persistent_supported(a.N, a.M))
                           ? launch_recover_persistent(s, one, stream)
                           : launch_recover_streamloop(s, one, stream);
        if (st != MP_OK) return st;
    }
    return MP_OK;
}

mp_status launch_recover_batched(const BatchedArgs& a, const Workspace& ws, cudaStream_t stream)
{
    return launch_batched_sequential(a, ws, stream);
}

}  // namespace mp
