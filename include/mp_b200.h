/* mp_b200.h -- C ABI of the B200-native Matching Pursuit library (libmp_b200.so).
 *
 * The method is the Matching Pursuit (MP) iteration of arxiv 0809.1833 (M. Andrecut), cited below as
 * "P:n" = line n of PAPER.md:
 *
 *     t <- 0, x~ <- 0, r <- y                                        Eq. 8,
 *     while ||r||_2 > eps ||y||_2 and t < T:
 *         i  <- argmax_m |<r, psi_m>|   (smallest index on ties)      Eq. 9,  P:73;  Eq. 16
 *         x~_i <- x~_i + <r, psi_i>                                   Eq. 10
 *         r  <- r - <r, psi_i> psi_i                                  Eq. 11
 *         t  <- t + 1                                                 Eq. 12
 *     return x~ (and r, t)
 *
 * over a dictionary Psi (N x M) whose columns psi_m have unit l2 norm (Eq. 4).
 *
 * CONVENTIONS (all entry points unless stated otherwise)
 *   - Every data pointer is a DEVICE pointer on the current CUDA device, caller-owned, fp32 (int32
 *     for indices / counters).  The dictionary and the batched Y, X, R must be 16-byte aligned;
 *     the vectors y, x, r of mp_recover need only their natural 4-byte alignment.  The *_host
 *     entry points at the end take HOST pointers instead and say so.
 *   - The dictionary is ATOM-MAJOR: psi_t[m*ld + n] = Psi[n][m], m = 0..M-1 (atom / column of Psi),
 *     n = 0..N-1, ld >= N and ld % 4 == 0.  (= Psi^T row-major = Psi column-major; each atom is
 *     contiguous so the reduction over n is coalesced.)  Elements psi_t[m*ld + n], N <= n < ld, may
 *     be read by the library but never influence a result.  The paper's own layout (Psi row-major,
 *     A2 P:360) is NOT accepted by the solvers; mp_transpose_rowmajor converts it once.
 *   - `stream` is a cudaStream_t passed as void* (NULL = the legacy default stream).  Calls are
 *     asynchronous on `stream`: they validate arguments on the host, enqueue work and return; they
 *     never synchronise the host (exception: the stream-loop fallback algorithm, see mp_set_int).
 *     All outputs, n_iter included, are device memory and valid once the stream has reached the
 *     end of the call.
 *   - The library allocates nothing on the hot path and keeps no per-problem state between calls
 *     (the optional dictionary handle at the end is the one exception, and says what it keeps);
 *     the caller provides `workspace` (>= mp_workspace_bytes(N, M, B) bytes, 256-byte aligned).
 *   - Errors: a status code is returned, nothing is printed, nothing throws.  Argument errors are
 *     detected before anything is enqueued and leave every output untouched.  mp_last_error()
 *     describes the most recent failure on the calling thread.
 *   - Indices are 0-based.  Non-finite inputs: results unspecified, but the call
 *     terminates within max_iter iterations and a NaN correlation never wins the argmax.
 */
#ifndef MP_B200_H
#define MP_B200_H

#include <stddef.h>
#include <stdint.h>

#if defined(__GNUC__)
#define MP_API __attribute__((visibility("default")))
#else
#define MP_API
#endif

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
    MP_OK = 0,
    MP_ERR_INVALID_ARG = 1, /* null / misaligned pointer, N<1, M<1, B<1, max_iter<0, eps<0 or NaN, ld<N, ld%4 */
    MP_ERR_CUDA = 2,        /* a CUDA runtime call or launch failed; see mp_last_error() */
    MP_ERR_UNSUPPORTED = 3, /* shape outside what the selected algorithm supports */
    MP_ERR_WORKSPACE = 4    /* workspace null, misaligned or smaller than mp_workspace_bytes() */
} mp_status;

/* Bytes of device workspace mp_recover (B = 1) / mp_recover_batched (B signals) need.  0 on invalid sizes. */
MP_API size_t mp_workspace_bytes(int N, int M, int B);

/* Column normalisation, Eq. 4: psi_m <- psi_m / ||psi_m||_2 for every atom, in place.
 * The sum of squares is accumulated in float64 and each element is divided in float64 and rounded to
 * fp32 once.  A zero atom is left zero.  norms_out (M floats, nullable) receives the norms BEFORE
 * scaling.  The paper assumes Eq. 4 and never executes it (its Bernoulli atoms are unit by
 * construction, Eq. 13). */
MP_API mp_status mp_normalize_columns(float* psi_t, int N, int M, int64_t ld, float* norms_out, void* stream);

/* Ingestion of the paper's own layout.  The listings hold Psi ROW-MAJOR, psi[n*ldr + m] (A2 P:360,
 * P:424; ldr >= M, any alignment), which makes every atom a stride-M gather (the axpy column of A2 P:470); this copies it once
 * into the atom-major psi_t[m*ld + n] every other entry point takes (ld >= N, ld % 4 == 0, 16-byte aligned).  Out of place
 * (overlapping buffers are refused), bit-exact, HBM-bound (8NM bytes; 128-bit accesses when psi is 16-byte aligned and ldr % 4 == 0); elements psi_t[m*ld + n], n >= N, are not written. */
MP_API mp_status mp_transpose_rowmajor(const float* psi, int N, int M, int64_t ldr, float* psi_t, int64_t ld, void* stream);

/* The MP loop above for one signal.
 *   psi_t      in   dictionary, ASSUMED column-normalised (not checked; the update uses <r,psi_i> as is)
 *   y          in   N measurements, y = Psi x (Eq. 2)
 *   eps        in   stop once ||r||_2 <= eps*||y||_2 (tested at the top of the loop)
 *   max_iter   in   T of Eq. 8 / P:88;  max_iter = 0 or y = 0 returns x~ = 0, r = y, n_iter = 0
 *   x          out  M floats, x~ (zeroed by the call, then accumulated in float64, rounded once at the end)
 *   r          out  N floats, the final residual (held in float64 inside the call, rounded once)
 *   n_iter     out  1 int, number of completed updates t
 *   idx_trace  out  nullable, max_iter ints:   atom chosen at iteration t, for t < n_iter
 *   c_trace    out  nullable, max_iter floats: the signed <r,psi_i> added at iteration t
 * Arithmetic: correlations are fp32 dot products of an fp32 rounding of r; r itself, ||r||^2 (a direct sum of
 * squares every iteration, as nrm2 at A2 P:471) and the stop test are float64. */
MP_API mp_status mp_recover(const float* psi_t, int N, int M, int64_t ld,
                     const float* y, float eps, int max_iter,
                     float* x, float* r, int* n_iter,
                     int* idx_trace, float* c_trace,
                     void* workspace, size_t workspace_bytes, void* stream);

/* mp_recover for callers that cannot provide a workspace because they cannot allocate device memory at all: a plug-in
 * running inside a server or framework whose own pool already owns the whole GPU (cudaMalloc fails there, or the host's
 * rules forbid it), or a latency-bound loop that must not risk the device-wide stall an allocation can cause.  Same loop
 * (Eq. 8-12), same arguments minus the workspace, same arithmetic contract and -- for the same inputs -- the same
 * bits as mp_recover run with knob "algo" = 3: it is that kernel (the persistent register-streaming one), with its scratch
 * area (a 256-byte control block and the float64 accumulator of x~) placed in a fixed array inside the library image.
 *   - No cudaMalloc / cudaFree / pool allocation, and no library routine that allocates, is called on any path of this
 *     entry point.  The caller still owns and passes every input and output (device pointers, as for mp_recover).
 *   - Limit: M <= MP_NOALLOC_MAX_M atoms; a larger M returns MP_ERR_UNSUPPORTED with a message and touches nothing.
 *     Shapes the register-streaming kernel itself cannot take (N above roughly 18 000: the residual no longer fits in shared
 *     memory) are refused the same way; there is no fallback to another algorithm.
 *   - Cost: the array is 256 + 8 * MP_NOALLOC_MAX_M bytes (512.25 KiB).  Every GPU on which the library is loaded keeps
 *     that much memory until the process exits, used or not.
 *   - The first call on each device looks the array's device address up (cudaGetSymbolAddress, with that device current,
 *     under a lock) and remembers it.  Make that first call ahead of time, outside any stream capture.
 *   - All calls on a device share the one array.  Each call clears the part it needs to start from zero (one memset on
 *     `stream` ahead of the kernel), so calls issued one after another on one stream, or otherwise ordered on the GPU, are
 *     independent of each other.  Two calls that can run on the GPU at the same time (different streams without an event
 *     between them, different host threads) race on the array and return garbage or hang: serialise them. */
#define MP_NOALLOC_MAX_M 65536
MP_API mp_status mp_recover_noalloc(const float* psi_t, int N, int M, int64_t ld,
                             const float* y, float eps, int max_iter,
                             float* x, float* r, int* n_iter,
                             int* idx_trace, float* c_trace, void* stream);

/* B signals sharing one dictionary ("all signals are encoded/decoded with the same dictionary").
 * Signal b's result equals mp_recover on (psi_t, Y[b]); signals are independent and a signal that has
 * stopped is frozen (x_b, r_b, n_iter_b no longer change) while the others continue.
 *   Y  in  B x N row-major, row stride ldy >= N (ldy % 4 == 0);   X out B x M;   R out B x N;   n_iter out B ints.
 * The correlation step is the dense contraction Psi^T R. */
MP_API mp_status mp_recover_batched(const float* psi_t, int N, int M, int64_t ld,
                             const float* Y, int64_t ldy, int B,
                             float eps, int max_iter,
                             float* X, float* R, int* n_iter,
                             void* workspace, size_t workspace_bytes, void* stream);

/* mp_recover_batched plus per-signal traces (both nullable): idx_trace[b*ldt + t], c_trace[b*ldt + t] for
 * t < n_iter[b], ldt >= max_iter.  Same results bit for bit; the traces make every iteration of every signal
 * gradable after a legal near-tie flip. */
MP_API mp_status mp_recover_batched_traced(const float* psi_t, int N, int M, int64_t ld,
                                    const float* Y, int64_t ldy, int B,
                                    float eps, int max_iter,
                                    float* X, float* R, int* n_iter,
                                    int* idx_trace, float* c_trace, int64_t ldt,
                                    void* workspace, size_t workspace_bytes, void* stream);

/* The correlation step of the batched path alone (Eq. 9 / Eq. 15 for B signals at once, NS subsystem 5):
 *   C[b*M + m] = <Y[b], psi_m>,   b < B <= 64,   C out B x M row-major (device).
 * Runs the same split-TF32 tensor-core contraction (tcgen05, TMEM accumulators, split-K over a 4-CTA cluster)
 * that mp_recover_batched runs every iteration, so the contraction can be checked element by element.
 * Needs mp_correlate_batched_workspace_bytes(N, M, B) bytes of 256-byte aligned workspace.
 * MP_ERR_UNSUPPORTED if the shape does not fit the tensor-core kernel (N <= 96). */
MP_API size_t mp_correlate_batched_workspace_bytes(int N, int M, int B);
MP_API mp_status mp_correlate_batched(const float* psi_t, int N, int M, int64_t ld,
                               const float* Y, int64_t ldy, int B, float* C,
                               void* workspace, size_t workspace_bytes, void* stream);

/* ---- the steps either side of the path: encode and score on the device ------------------
 * mp_encode_sparse, Eq. 2: y = Psi x for a K-sparse x given as K (index, value) pairs, the way the paper
 * builds x (A2 P:328-332):   y[n] = sum_{k<K} val[k] * psi_t[idx[k]*ld + n],   ascending k, float64 accumulation,
 * one rounding to fp32.  Reads 4NK bytes instead of the 4NM of a dense product.  idx (K ints, device) is 0-based;
 * repeated indices accumulate; an index outside [0, M) contributes nothing.  K = 0 gives y = 0.
 * mp_reconstruction_error, Eq. 14: err_pct[0] = 100 * ||x_hat - x||_2^2 / ||x||_2^2 (one double, device,
 * 8-byte aligned), float64 sums in a fixed order.  x = 0 gives NaN or +inf as the formula does. */
MP_API mp_status mp_encode_sparse(const float* psi_t, int N, int M, int64_t ld, const int* idx, const float* val, int K,
                           float* y, void* stream);
MP_API mp_status mp_reconstruction_error(const float* x_hat, const float* x, int M, double* err_pct, void* stream);

/* ---- double-precision path (the paper reports both precisions) -------------
 * The same loop on a float64 dictionary: psi_t[m*ld + n], ld >= N, ld % 2 == 0, 16-byte aligned; y, x, r, c_trace and
 * eps are double.  All arithmetic is float64 (dots, residual, norms, coefficients); ties go to the lowest index.
 * Workspace: mp_workspace_bytes_f64(N, M) bytes, 256-byte aligned.  One persistent cooperative kernel per solve;
 * MP_ERR_UNSUPPORTED if the residual does not fit in shared memory (N > ~28 000).  HBM roofline: 8NM bytes per iteration. */
MP_API size_t mp_workspace_bytes_f64(int N, int M);
MP_API mp_status mp_normalize_columns_f64(double* psi_t, int N, int M, int64_t ld, double* norms_out, void* stream);
MP_API mp_status mp_recover_f64(const double* psi_t, int N, int M, int64_t ld,
                         const double* y, double eps, int max_iter,
                         double* x, double* r, int* n_iter,
                         int* idx_trace, double* c_trace,
                         void* workspace, size_t workspace_bytes, void* stream);

/* ---- Orthogonal Matching Pursuit (the paper's declared next target) -------------
 * MP's selection (Eq. 9, Eq. 16: fp32 dots of the fp32 rounding of r, lowest index on ties) followed by a least-squares
 * refit on the selected atoms, so that r = y - Psi_S x_S with x_S = argmin ||y - Psi_S z||_2 after every step.  The refit is
 * a float64 QR factorisation grown by one column per iteration (Gram-Schmidt, a second pass whenever the first removed more than half of the atom); x~ is obtained once, at the
 * end, by back substitution.  Stop rule as MP; at most min(max_iter, N) atoms are taken; an atom that lies in the
 * span of the selected ones ends the run.  Same layouts as mp_recover; idx_trace (nullable) receives the atoms in order.
 * Runs as one persistent cooperative kernel when the orthonormal basis, sliced by components over the CTAs, fits in shared
 * memory (knob "omp_algo": 0 = auto, 1 = that kernel or MP_ERR_UNSUPPORTED, 2 = stream loop), else as a stream of small
 * kernels (the stop flag stays on the device; the host polls it every "chunk" iterations).
 * Workspace: mp_workspace_bytes_omp(N, M, max_iter) bytes (dominated by the 8 * min(max_iter, N) * N byte basis). */
MP_API size_t mp_workspace_bytes_omp(int N, int M, int max_iter);
MP_API mp_status mp_recover_omp(const float* psi_t, int N, int M, int64_t ld,
                         const float* y, float eps, int max_iter,
                         float* x, float* r, int* n_iter, int* idx_trace,
                         void* workspace, size_t workspace_bytes, void* stream);

/* ---- sign-packed Bernoulli dictionary (Eq. 13: psi_nm = +-1/sqrt(N)) ------------------
 * mp_pack_signs: bits[m*ldw + w] bit k = 1 iff psi_t[m*ld + 32w + k] < 0 (ldw >= ceil(N/32) uint32 words per atom, pad
 * bits 0); scale_out[0] = |psi_t[0]|; n_bad[0] = number of entries whose magnitude is not bit-identical to it (device int:
 * a dictionary with n_bad != 0 is not a +-scale one and must not be used packed).
 * mp_recover_signs: the MP loop of mp_recover on the packed dictionary (same outputs, traces, stop rule and arithmetic
 * contract; c_m = scale * (sum_n r_n - 2 sum_{bit=1} r_n)).  The packed dictionary is 32x smaller than fp32 and is held in
 * shared memory for the whole solve (N*M/8 bytes over all SMs), so an iteration is bound by the ALUs, not by memory.
 * Workspace: mp_workspace_bytes(N, M, 1).  MP_ERR_UNSUPPORTED if a CTA's share of the bits does not fit in shared memory. */
MP_API mp_status mp_pack_signs(const float* psi_t, int N, int M, int64_t ld, uint32_t* bits, int64_t ldw,
                        float* scale_out, int* n_bad, void* stream);
MP_API mp_status mp_recover_signs(const uint32_t* bits, int N, int M, int64_t ldw, float scale,
                           const float* y, float eps, int max_iter,
                           float* x, float* r, int* n_iter, int* idx_trace, float* c_trace,
                           void* workspace, size_t workspace_bytes, void* stream);

/* mp_recover_signs_many: P independent problems, each with its OWN sign-packed Bernoulli dictionary -- the paper's Fig. 1
 * experiment in the paper's own representation.  bits: problem q's words start at bits + q*problem_stride (uint32
 * words; [M][ldw] as mp_pack_signs writes them -- packing the P dictionaries stacked as one [P*M, N] dictionary gives exactly
 * this with problem_stride = M*ldw; 0 = one shared dictionary).  Y P x N (row stride ldy >= N), X P x M, R P x N, n_iter P ints,
 * traces nullable [q*ldt + t], ldt >= max_iter.  One CTA owns a problem: its N*M/8 bytes of bits stay in that SM's shared memory
 * for the whole solve, and the correlations come from a per-iteration table of the 16 signed sums of every four residual values
 * (one lookup per four entries).  Contract as mp_recover_signs (fp32 sums of the fp32 rounding of a float64 residual, lowest
 * index on ties).  MP_ERR_UNSUPPORTED if bits + table do not fit in one SM's shared memory (N*M/8 + 28 N + 8 M > ~227 KB).
 * Workspace: mp_workspace_bytes_signs_many(N, M, P) (256 bytes). */
MP_API size_t mp_workspace_bytes_signs_many(int N, int M, int P);
MP_API mp_status mp_recover_signs_many(const uint32_t* bits, int N, int M, int64_t ldw, int64_t problem_stride, float scale,
                                const float* Y, int64_t ldy, int P, float eps, int max_iter,
                                float* X, float* R, int* n_iter, int* idx_trace, float* c_trace, int64_t ldt,
                                void* workspace, size_t workspace_bytes, void* stream);

/* ---- many independent small problems (the paper's Fig. 1 experiment) -----------------
 * P problems of one shape (N, M), each with its OWN dictionary and measurement vector -- the (sigma, rho) phase diagram is
 * 100 trials per cell at M = 1000 with a fresh Bernoulli dictionary per trial -- solved by one launch:
 *   psi_t   in   problem q's dictionary starts at psi_t + q*problem_stride (floats; atom-major, row stride ld as above);
 *                problem_stride = 0 means all P problems share ONE dictionary (then this equals mp_recover_batched)
 *   Y       in   P x N, row stride ldy >= N (any; only 4-byte alignment is needed for Y, X, R here);   X out P x M;
 *                R out P x N;   n_iter out P ints
 *   idx_trace / c_trace   nullable, [q*ldt + t] for t < n_iter[q], ldt >= max_iter
 * Problem q's result equals mp_recover on (dictionary q, Y[q]) under the same arithmetic contract.  One thread-block
 * cluster (1-16 CTAs) owns a problem at a time: its dictionary is held in the cluster's shared memory for the whole solve
 * when it fits (<= ~3.5 MB), else streamed from L2; the argmax is exchanged without any barrier instruction: every warp's packed
 * key is stored into every CTA of the cluster with st.async, which also counts on the destination's mbarrier, and a CTA waits on
 * its own mbarrier until all keys have landed; clusters draw problems from a device counter.  N > 2048 falls back to one
 * single-signal solve after another.  Knobs: "many_cluster" (CTAs per problem, 0 = auto), "many_threads", "many_stat"
 * (2 = never stationary), "many_l2_mb" (MB of dictionaries the plan keeps in flight, 0 = auto = 64).  Workspace: mp_workspace_bytes_many(N, M, P). */
MP_API size_t mp_workspace_bytes_many(int N, int M, int P);
MP_API mp_status mp_recover_many(const float* psi_t, int N, int M, int64_t ld, int64_t problem_stride,
                          const float* Y, int64_t ldy, int P, float eps, int max_iter,
                          float* X, float* R, int* n_iter,
                          int* idx_trace, float* c_trace, int64_t ldt,
                          void* workspace, size_t workspace_bytes, void* stream);

/* Description of the last error on this thread ("" if none).  Static storage, never NULL. */
MP_API const char* mp_last_error(void);

/* Tuning / diagnostic knobs (process-wide, not part of the method).  Unknown name -> MP_ERR_INVALID_ARG.
 * The knobs and the info_* read-outs are process-wide atomics: setting or reading one never races with a solve on another host
 * thread, and with the knobs left alone solves may be issued from several host threads at once (each call keeps its state in its
 * own arguments and workspace; mp_recover_noalloc is the exception, see there).  What stays process-wide is their MEANING: a knob
 * changed while another thread is inside a library call may or may not apply to that call, and an info_* value is the plan of
 * whichever launch recorded it last.  Set knobs before the solves they are meant for.
 *   "algo"          0 = auto (default: 4 if one cluster can hold the dictionary in shared memory -- 4NM <= ~3.4 MB, N <= 2048 --
 *                   else 3 if it fits, else 1, else 2), 4 = the cluster kernel of mp_recover_many with P = 1 (N <= 2048),
 *                   1 = persistent cooperative kernel fed by TMA bulk
 *                   copies through shared memory, 2 = stream loop of small kernels (general fallback; synchronises the
 *                   host every "chunk" iterations to read the stop flag), 3 = persistent cooperative kernel that streams
 *                   the dictionary into registers with 128-bit loads
 *   "l2_resident_mb" algo 3 (and the float64 / Orthogonal MP kernels): MB of dictionary rows loaded L2::evict_last so that they
 *                   stay in L2 across iterations (the rest is loaded evict_first); 0 = auto (68 MB for dictionaries above
 *                   110 MB), 1 = off, other = that many MB for every dictionary larger than it
 *   "pingpong"      algo 3: odd iterations visit a CTA's work items in reverse order, so that the rows read last are read first again
 *                   and the part of the L2 not held by pinned rows serves the start of every pass (results do not depend on it);
 *                   0 = auto (dictionaries above 90 MB), 1 = off, 2 = on.  With it on, "l2_resident_mb" auto = 88 MB for
 *                   dictionaries above 140 MB (none below), and "pin_margin_pct" (0 = auto = 10, 100 = none) percent of a CTA's
 *                   rows at either end of its share are never pinned: the reversed order re-reads them soonest
 *   "info_l2_pingpong", "info_l2_resident_mb", "info_l2_dynamic"  (read with mp_get_int) the L2 plan the last algo-3 launch used
 *   "l2_bytes"      the L2 size the automatic plan is made for: 0 (default) = the device's cudaDevAttrL2CacheSize; the megabyte figures
 *                   above are those of a 126.5 MiB L2 and scale with it (they are fractions of the L2); another value = plan as if the
 *                   L2 had that many bytes (tests; a co-tenant that owns part of the L2).  "info_l2_bytes": the size the last plan used
 *   "balance"       algo 3, shares of >= 8 work items per warp (dictionaries that stream from HBM): 0 (default) = the warps of a CTA
 *                   draw their work items from a counter, so a CTA finishes when its share is done and not when its slowest warp
 *                   is (results do not depend on it), 1 = plain round-robin
 *   "l2_demote"     0 (default) = when a solve ends the pinned rows are handed back (applypriority L2::evict_normal), so later
 *                   kernels find a normal L2; 1 = left as they are (measurements)
 *   "warps"         consumer warps per CTA of the persistent kernel (0 = auto)
 *   "slot_bytes"    bytes of one shared-memory stage (0 = auto);   "depth"  stages per warp (0 = auto)
 *   "grid"          CTAs of the persistent kernel (0 = auto = one per SM)
 *   "chunk"         iterations enqueued between stop-flag polls of algo 2 (default 64)
 *   "batched_algo"  0 = auto (default): lock-step tensor-core kernel in groups of <= 64 signals when the shape fits and the
 *                   dictionary is larger than 1.5 MB, else one thread-block cluster per signal (N <= 2048), else sequential;
 *                   1 = tensor-core kernel or MP_ERR_UNSUPPORTED, 2 = one single-signal solve after another,
 *                   3 = one cluster per signal (the mp_recover_many kernel on the shared dictionary) or MP_ERR_UNSUPPORTED
 *   "info_batched_algo"  (read with mp_get_int) which of 1, 2, 3 the last successful mp_recover_batched call ran.  Auto dispatch falls
 *                   back from the tensor-core kernel when its cooperative launch is refused; the call still returns MP_OK (the
 *                   results are the same) but is many times slower, mp_last_error() keeps the refusal and this reads 2 or 3
 *   "batched_coop"  1 (default) = launch the batched kernel with the cooperative attribute (co-residency checked by
 *                   the driver), 0 = plain cluster launch of a grid sized from cudaOccupancyMaxActiveClusters: only on a device
 *                   where nothing else runs (profilers that cannot launch cooperative cluster kernels); the library never drops
 *                   the attribute on its own */
MP_API mp_status mp_set_int(const char* name, int64_t value);
MP_API mp_status mp_get_int(const char* name, int64_t* value);

/* Read-only streaming diagnostic (not part of the method): the ceiling the correlation pass (Eq. 9) is measured against.
 * Reads the first k * 8 KiB * (number of SMs) bytes of buf (k = the largest integer that fits in `bytes`) `passes` times with the
 * access pattern of the single-signal kernel -- one CTA per SM on a contiguous share, 16 independent 128-bit loads per lane in flight,
 * four FMAs per load -- and nothing else (no shared memory, no barrier, no argmax).  A buffer that fits in L2 read for many passes
 * gives the L2 read rate, the roofline of the cache-resident configurations; a buffer much larger than L2 gives the HBM read rate.
 *   buf         in   device, 16-byte aligned, `bytes` long (contents irrelevant but finite values keep the FMAs cheap)
 *   sink        out  device, 1 float: receives a sum that only exists to keep the loads alive (accumulated with atomicAdd)
 *   bytes_read  out  HOST pointer, nullable: bytes the launch reads in total (all passes), for the caller's GB/s
 * Asynchronous on `stream`; the caller times it (CUDA events).  MP_ERR_INVALID_ARG if the buffer is smaller than 8 KiB per SM. */
MP_API mp_status mp_probe_read(const void* buf, size_t bytes, int passes, float* sink, unsigned long long* bytes_read, void* stream);

/* Number of kernels the library has launched on behalf of this process so far (for bench.py's gpu_launches). */
MP_API int64_t mp_launch_count(void);

/* ---- HOST-buffer entry points (end-to-end convenience; every pointer below is a HOST pointer) ----------
 * mp_recover_host allocates device buffers (stream-ordered, from the device's default memory pool, whose release threshold it
 * raises so that the next call reuses them), copies psi_t (M*ld floats) and y to the device on an internal
 * stream, optionally normalises the columns on the device (normalize != 0; the host copy of psi_t is not
 * modified), runs mp_recover, copies x, r, n_iter (and the traces if non-null) back, synchronises and frees.
 * Pinned host memory makes the copies faster but is not required.  mp_recover_batched_host likewise. */
MP_API mp_status mp_recover_host(const float* psi_t, int N, int M, int64_t ld, int normalize,
                          const float* y, float eps, int max_iter,
                          float* x, float* r, int* n_iter, int* idx_trace, float* c_trace);
MP_API mp_status mp_recover_batched_host(const float* psi_t, int N, int M, int64_t ld, int normalize,
                                  const float* Y, int64_t ldy, int B, float eps, int max_iter,
                                  float* X, float* R, int* n_iter);

/* ---- dictionary handle ("the host to device dictionary transfer only takes place once, since all signals are
 * encoded/decoded with the same dictionary"; SURVEY 8(b) allows an optional opaque handle) -------------------------------
 * mp_dictionary_create puts ONE dictionary on the current device and keeps it there:
 *   psi_on_host != 0   psi_t is a HOST pointer (M rows of N floats, row stride ld >= N, any alignment; pinned memory makes the
 *                      copy faster).  The library allocates the device copy (row stride N rounded up to 4), uploads it in chunks and, if normalize != 0, normalises each chunk on the device (Eq. 4)
 *                      while the next one is still in flight.  The host buffer is not modified and may be freed on return.
 *   psi_on_host == 0   psi_t is a DEVICE pointer (16-byte aligned, ld % 4 == 0) that the handle BORROWS: the caller keeps it alive until
 *                      mp_dictionary_destroy; with normalize != 0 it is normalised in place.
 * The call synchronises (a one-off per dictionary).  The handle also owns an internal stream, the solver workspace and the
 * small per-call device buffers of the *_host_h entry points, so a steady-state call moves only y up and x~, r, n_iter down.
 * A handle is used by one host thread at a time.  mp_dictionary_info returns the shape and the DEVICE pointer of the
 * dictionary (for the device-pointer entry points above); any output may be NULL.
 * mp_recover_host_h / mp_recover_batched_host_h: as mp_recover_host / mp_recover_batched_host (HOST pointers, synchronous,
 * same arithmetic, same bits) without the dictionary argument; Y rows need only ldy >= N.  Traces (nullable) as in
 * mp_recover_batched_traced: [b*ldt + t], ldt >= max_iter; entries t >= n_iter[b] are unspecified. */
typedef struct mp_dictionary mp_dictionary;
MP_API mp_status mp_dictionary_create(const float* psi_t, int psi_on_host, int N, int M, int64_t ld, int normalize,
                               mp_dictionary** out);
MP_API mp_status mp_dictionary_destroy(mp_dictionary* handle);   /* NULL is allowed */
MP_API mp_status mp_dictionary_info(const mp_dictionary* handle, int* N, int* M, int64_t* ld, const float** psi_t_device);
MP_API mp_status mp_recover_host_h(mp_dictionary* handle, const float* y, float eps, int max_iter,
                            float* x, float* r, int* n_iter, int* idx_trace, float* c_trace);
MP_API mp_status mp_recover_batched_host_h(mp_dictionary* handle, const float* Y, int64_t ldy, int B, float eps, int max_iter,
                                    float* X, float* R, int* n_iter, int* idx_trace, float* c_trace, int64_t ldt);

#ifdef __cplusplus
}
#endif
#endif /* MP_B200_H */
