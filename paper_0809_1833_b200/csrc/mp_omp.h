// mp_omp.h -- workspace of the Orthogonal MP paths (mp_omp.cu: stream loop; mp_omp_persistent.cu: one persistent kernel).
#pragma once
#include "mp_internal.h"

namespace mp {

constexpr int kOmpMaxCtas = 256;     // >= CTAs of the persistent OMP grid

struct OmpWs {
    unsigned long long* ctrl;   // control block: stream loop kCtr* slots; persistent kernel [0] barrier, [1..3] keys, [kCtrT] t
    double* r64;                // Nr
    float* r32;                 // Nr
    double* w;                  // Nr   the new direction being orthogonalised (persistent kernel: gathered slices)
    double* h;                  // T    Q^T w of the current pass (reduced)
    double* z;                  // T    Q^T y
    double* Rm;                 // T x T upper triangular, row-major
    int* sel;                   // T    selected atoms in order
    double* Q;                  // T x Nr orthonormal basis of span(Psi_S), row-major (stream loop only)
    double* hpart;              // kOmpMaxCtas x T per-CTA partial dots (persistent kernel)
    double* scal;               // kOmpMaxCtas x 4 per-CTA partial ||w||^2, <w, r>, ||psi_i||^2 (persistent kernel)
    size_t bytes;
};

size_t omp_layout(int N, int T, void* base, OmpWs* ws);

struct OmpArgs {
    const float* psi_t; int N, M; int64_t ld;
    const float* y; float eps; int T;      // T = min(max_iter, N)
    int* idx_trace;
};
bool omp_persistent_supported(int N, int M, int T);
mp_status launch_omp_persistent(const OmpArgs& a, const OmpWs& ws, cudaStream_t stream);

}  // namespace mp
