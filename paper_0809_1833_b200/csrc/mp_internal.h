// mp_internal.h -- host-side plumbing shared by the translation units of libmp_b200.so.
#pragma once
#include <cuda_runtime.h>
#include <atomic>
#include <stddef.h>
#include <stdint.h>

#include "../../include/mp_b200.h"

namespace mp {

// ---- error reporting (thread-local message behind mp_last_error) --------------------------------------
mp_status fail(mp_status code, const char* fmt, ...);
mp_status cuda_fail(cudaError_t e, const char* what);
#define MP_CUDA(call)                                                   \
    do {                                                                \
        cudaError_t e__ = (call);                                       \
        if (e__ != cudaSuccess) return ::mp::cuda_fail(e__, #call);     \
    } while (0)

// ---- process-wide knobs (mp_set_int) ---------------------------------------------------------------------
// Atomics: the header lets several host threads issue solves at once, and every launch records its plan in the info_* fields
// (and reads the knobs); plain int64_t fields would make that a data race.  The VALUES are still process-wide: with solves
// running on several threads an info_* read returns the plan of whichever launch wrote last.
struct Options {
    std::atomic<int64_t> algo{0}, warps{0}, slot_bytes{0}, depth{0}, grid{0}, chunk{64};
    std::atomic<int64_t> batched_algo{0}, batched_coop{1};
    std::atomic<int64_t> info_batched_algo{0};     // batched path the last mp_recover_batched call took: 1 tensor-core lock-step, 2 sequential, 3 clusters
    std::atomic<int64_t> omp_algo{0}, info_omp_algo{0};   // Orthogonal MP: 0 auto, 1 persistent kernel, 2 stream loop; and the one last used
    std::atomic<int64_t> pin_margin_pct{0};        // with pingpong: percent of a CTA's groups at either end that are never pinned (0 = auto = 10, 100 = none)
    std::atomic<int64_t> pingpong{0};              // register-streaming kernel: reversed item order on odd iterations; 0 = auto (with the residency hints), 1 = off, 2 = on
    std::atomic<int64_t> balance{0};               // register-streaming kernel: 0 = warps draw their items from a counter when the shares are long, 1 = plain round-robin
    std::atomic<int64_t> l2_demote{0};             // 0 = pinned rows are demoted to evict_normal when a solve ends, 1 = left pinned (measurements)
    std::atomic<int64_t> l2_resident_mb{0};        // register-streaming kernel: MB of dictionary kept in L2 with evict_last (0 = auto, 1 = off)
    std::atomic<int64_t> many_cluster{0}, many_threads{0}, many_stat{0}, many_l2_mb{0};   // cluster-per-problem kernel: CTAs per problem (0 auto), threads per CTA (0 auto), 2 = never stationary
    std::atomic<int64_t> info_many_cluster{0}, info_many_stat{0}, info_many_clusters{0}, info_many_threads{0};   // plan of its last launch
    std::atomic<int64_t> info_l2_pingpong{0}, info_l2_resident_mb{0}, info_l2_dynamic{0};   // L2 plan of the last register-streaming launch (read-only use)
    std::atomic<int64_t> l2_bytes{0};              // L2 size the plan is made for: 0 = the device's cudaDevAttrL2CacheSize, other = pretend it is this many bytes (tests)
    std::atomic<int64_t> info_l2_bytes{0};         // the L2 size the last plan was made for
    std::atomic<int64_t> info_algo{0};             // kernel the last mp_recover call used (1, 2 or 3)
    std::atomic<int64_t> info_tc_clusters{0}, info_tc_at{0}, info_tc_stages{0};   // plan of the last batched tensor-core launch (read-only use)
};
Options& options();
void count_launch(int n = 1);

// ---- device info (cached per device) ---------------------------------------------------------------------
struct DeviceInfo {
    int device = -1, sm_count = 0, smem_optin = 0, coop = 0, l2_bytes = 0;
};
mp_status device_info(DeviceInfo* out);
// The megabyte figures of the L2 plan below were measured on a B200 whose cudaDevAttrL2CacheSize is 132 644 864 bytes (126.5 MiB);
// on a device (or MIG slice, or carve-out) with another L2 size they are scaled by l2_scale() = that size / 132 644 864, i.e. they
// are fractions of the L2: reversed order above 0.68 L2, 0.51 L2 pinned above 0.83 L2 (same-order stream), 0.66 L2 pinned above
// 1.06 L2 (reversed order).  Knob "l2_bytes" overrides the attribute (tests); "info_l2_bytes" reports the size used.
constexpr double kL2TunedBytes = 132644864.0;
double l2_scale();

// ---- workspace layout --------------------------------------------------------------------------------------
// [ctrl: 256 B][x64: B*M doubles][r64: B*Nr doubles][r32: B*Nr floats][keys: B u64, padded][flags ...]
struct Workspace {
    unsigned long long* ctrl;   // [0] grid-barrier counter, [1..3] rotating key slots (single), [4] done flag, [8..] misc
    double* x64;                // B*M
    double* r64;                // B*Nr   (Nr = N rounded up to 128)
    float* r32;                 // B*Nr
    unsigned long long* keys;   // 3*B  rotating per-signal key slots (batched)
    int* state;                 // 4*B ints: per-signal stop state of the batched kernel
    float* rs;                  // 128*Nr  (B > 1 only) hi / lo split of the fp32 residuals, the tensor-core A operand
    size_t bytes;
};
size_t workspace_layout(int N, int M, int B, void* base, Workspace* ws);
static inline int round_up(int v, int m) { return (v + m - 1) / m * m; }
// L2 residency (mp_common.cuh): groups of rows per CTA to load with evict_last.  Auto (knob "l2_resident_mb" = 0): 68 MB, the
// measured optimum on B200, for dictionaries above 110 MB -- up to ~100 MB the plain LRU behaviour of the L2 already serves a
// cyclic stream (84 MB: 9.3 us per iteration without hints, 10.5 us with) and above it the stream thrashes (134 MB: 22.2 us
// without, 15.2 us with).  1 = off; any other value = that many MB, for every dictionary larger than it.
// auto_mb: 68 for a kernel that streams in the same order every iteration, 88 with the reversed order on odd iterations (K1's "ping-pong":
// the pinned rows then share the L2 with a recency-served part of the stream, and the measured optimum moves up).
// With it the recency-served part alone carries dictionaries up to ~140 MB (134 MB: 11.6 us per iteration without pinned rows, 12.8 with,
// 15.3 for the same-order stream with 68 MB pinned), so the hints then start at auto_min_mb = 140.
static inline int l2_resident_groups(double dict_bytes, int grid, double group_bytes, double auto_mb = 68.0, double auto_min_mb = 110.0)
{
    const int64_t knob = options().l2_resident_mb;
    const double sc = l2_scale();
    const double target = knob == 0 ? 1e6 * auto_mb * sc : knob == 1 ? 0.0 : 1e6 * (double)knob;
    if (!(target > 0.0) || grid < 1 || !(dict_bytes > (knob == 0 ? 1e6 * auto_min_mb * sc : target))) return 0;
    return (int)(target / grid / group_bytes);
}

// The L2 plan of a register-streaming persistent kernel (K1, float64, Orthogonal MP) for one launch.
//   pingpong         odd iterations visit a CTA's work items in reverse order (knob "pingpong": 0 = auto for dictionaries above 90 MB --
//                    below that the L2 serves the same-order stream by itself --, 1 = off, 2 = on); only kernels that can do it ask for it
//   resident_groups  groups of rows per CTA loaded evict_last: with the reversed order 88 MB for dictionaries above 140 MB (the
//                    recency-served part alone carries smaller ones), without it 68 MB above 110 MB
//   pin_margin       with the reversed order: groups at either end of a CTA's share that are never pinned (knob "pin_margin_pct", auto 10 %)
// Measured per size in profiles/k1_boundary_r02.md.
struct L2Plan { int pingpong, resident_groups, pin_margin; };
static inline L2Plan l2_plan(double dict_bytes, int grid, double group_bytes, int groups_per_cta, bool can_pingpong)
{
    L2Plan l;
    l.pingpong = can_pingpong && (options().pingpong == 2 || (options().pingpong == 0 && dict_bytes > 90e6 * l2_scale()));
    l.resident_groups = l.pingpong ? l2_resident_groups(dict_bytes, grid, group_bytes, 88.0, 140.0) : l2_resident_groups(dict_bytes, grid, group_bytes);
    const int64_t knob_pct = options().pin_margin_pct;
    const int64_t pct = knob_pct == 0 ? 10 : knob_pct >= 100 ? 0 : knob_pct;
    int e = l.pingpong ? (int)(pct * groups_per_cta / 100) : 0;
    if (groups_per_cta - 2 * e < l.resident_groups + 1) e = (groups_per_cta - l.resident_groups - 1) / 2;
    l.pin_margin = e > 0 ? e : 0;
    return l;
}

// ---- launchers (each enqueues on `stream`, returns MP_OK or an error) ---------------------------------------
mp_status launch_normalize(float* psi_t, int N, int M, int64_t ld, float* norms_out, cudaStream_t stream);

mp_status launch_transpose_rowmajor(const float* psi, int N, int M, int64_t ldr, float* psi_t, int64_t ld, cudaStream_t stream);

mp_status launch_encode_sparse(const float* psi_t, int N, int M, int64_t ld, const int* idx, const float* val, int K,
                               float* y, cudaStream_t stream);
mp_status launch_reconstruction_error(const float* x_hat, const float* x, int M, double* out, cudaStream_t stream);

struct RecoverArgs {
    const float* psi_t; int N, M; int64_t ld;
    const float* y; float eps; int max_iter;
    float* x; float* r; int* n_iter; int* idx_trace; float* c_trace;
};
mp_status launch_recover_persistent(const RecoverArgs& a, const Workspace& ws, cudaStream_t stream);
bool persistent_supported(int N, int M);
mp_status launch_recover_persistent_ldg(const RecoverArgs& a, const Workspace& ws, cudaStream_t stream);
bool persistent_ldg_supported(int N, int M);
mp_status launch_recover_streamloop(const RecoverArgs& a, const Workspace& ws, cudaStream_t stream);
// control-block slots of the stream-loop kernels (unsigned long long each) and its fused correlate+argmax launch,
// shared with the Orthogonal MP loop (mp_omp.cu)
enum { kCtrKey = 1, kCtrDone = 4, kCtrT = 5, kCtrYY = 6, kCtrRR = 7 };
mp_status launch_sl_correlate_argmax(const float* psi_t, int N, int M, int64_t ld, const float* r32, unsigned long long* ctrl,
                                     int blocks, cudaStream_t stream);

struct BatchedArgs {
    const float* psi_t; int N, M; int64_t ld;
    const float* Y; int64_t ldy; int B; float eps; int max_iter;
    float* X; float* R; int* n_iter;
    int* idx_trace; float* c_trace; int64_t ldt;
};
mp_status launch_recover_batched(const BatchedArgs& a, const Workspace& ws, cudaStream_t stream);
// tensor-core lock-step kernel (B <= 64 per launch); dbg_C (nullable, B x M) receives the correlations of iteration 0
mp_status launch_recover_batched_tc(const BatchedArgs& a, const Workspace& ws, float* dbg_C, cudaStream_t stream);
bool batched_tc_supported(int N, int M, int B);

// P independent problems of one shape, one thread-block cluster per problem (mp_many.cu)
struct ManyArgs {
    const float* psi_t; int N, M; int64_t ld, pstride;
    const float* Y; int64_t ldy; int P; float eps; int max_iter;
    float* X; float* R; int* n_iter; int* idx_trace; float* c_trace; int64_t ldt;
};
bool many_supported(int N, int M);
bool many_single_stationary(int N, int M);
mp_status launch_recover_many(const ManyArgs& a, unsigned int* counter, cudaStream_t stream);

}  // namespace mp
