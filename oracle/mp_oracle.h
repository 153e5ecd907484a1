/* mp_oracle.h -- CPU ORACLE for Matching Pursuit.  TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain C99, float64 arithmetic, straightforward loops in the paper's order and notation.
 * Written from /root/reference/PAPER.md (arxiv 0809.1833, M. Andrecut); "P:n" = PAPER.md line n.
 * It shares no code with the CUDA path (paper_0809_1833_b200/csrc) and neither includes the
 * other.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
 * legs may load it.
 *
 * Layout.  The dictionary is passed ATOM-MAJOR: psi_t[m*ld + n] = Psi[n][m] (n = 0..N-1 row of
 * Psi, m = 0..M-1 column/atom; ld >= N).  That is Psi^T row-major = Psi column-major; it is only
 * an addressing convention, all sums below run exactly as the paper states them.
 * Two instantiations of every routine that reads Psi: *_f64 takes double Psi; *_f32 takes float
 * Psi and promotes each element to double on the fly (exact), so the oracle can be fed the very
 * bits the GPU sees.
 *
 * Readings of the paper where it is silent/ambiguous (DESIGN.md section "Readings"):
 *   R1 stop test at loop top, continue while ||r||_2 > eps*||y||_2 and t < T (text P:70, P:88;
 *      NOT the listings' sqrt(eps*||y||), A1 P:272 / A2 P:459);
 *   R2 argmax = smallest index of the maximum magnitude; NaN never wins;
 *   R3 indices 0-based;   R4 the signed <r,psi_i> is added (Eq. 10);
 *   R5 ||r|| is a direct sum of squares every iteration (nrm2, A1 P:283 / A2 P:471);
 *   R6 update is r - c*psi_i with no division by ||psi_i||^2 (Eq. 11).
 *
 * Pins (tests/test_oracle_pins.py): orthonormal Psi recovers K-sparse x in K steps; two-atom
 * closed form ||r_{t+1}|| = |mu| ||r_t||; M=1 projection; brute-force argmax / tie-breaks;
 * energy identity, monotone ||r||, consistency y - Psi x = r; numpy gemv+argmax for one step;
 * scaling / permutation / negation symmetries; edge cases.  Parity NOT pinned by anything but
 * agreement with these properties: the free-running n_iter on random inputs ("parity unpinned"
 * for that one number).
 */
#ifndef MP_ORACLE_H
#define MP_ORACLE_H
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

/* Eq. 4: psi_m <- psi_m / ||psi_m||_2 for every atom m, in place, float64.
 * A zero column is left zero.  norms_out (M, nullable) receives the norms BEFORE scaling. */
void oracle_normalize_columns_f64(double* psi_t, int N, int M, int64_t ld, double* norms_out);

/* Eq. 9 (cost P:90): c[m] = sum_{n=0}^{N-1} r[n]*Psi[n][m], ascending n, for all m.
 * nthreads > 1 splits the loop over m across OpenMP threads (each c[m] is still one serial sum). */
void oracle_correlate_f64(const double* psi_t, int N, int M, int64_t ld, const double* r, double* c, int nthreads);
void oracle_correlate_f32(const float*  psi_t, int N, int M, int64_t ld, const double* r, double* c, int nthreads);

/* Eq. 16: smallest index of the maximum magnitude element. M >= 1. */
int oracle_argmax_abs(const double* c, int M);

/* Eq. 18: Euclidean norm, direct sum of squares, ascending index. */
double oracle_nrm2(const double* v, int n);

/* The MP loop, Eq. 8-12.  Outputs: x[M], r[N], *n_iter.
 * Optional per-iteration traces (each nullable):
 *   idx_trace[t], c_trace[t]   the atom chosen at iteration t and the signed <r,psi_i> added;
 *   gap_trace[t]               (a1 - a2)/a1, a1 = max|c|, a2 = largest |c_m| over m != i (0 if a1 == 0);
 *   rnorm_trace[t]             ||r||_2 at the top of iteration t; entry [n_iter] is the final norm
 *                              (so it needs T+1 slots).
 * Returns 0, or 1 on invalid arguments. */
int oracle_mp_f64(const double* psi_t, int N, int M, int64_t ld, const double* y, double eps, int T,
                  double* x, double* r, int* n_iter,
                  int* idx_trace, double* c_trace, double* gap_trace, double* rnorm_trace, int nthreads);
int oracle_mp_f32(const float* psi_t, int N, int M, int64_t ld, const double* y, double eps, int T,
                  double* x, double* r, int* n_iter,
                  int* idx_trace, double* c_trace, double* gap_trace, double* rnorm_trace, int nthreads);

/* Teacher-forced replay: the same state update, but at step t
 * the atom is idx_run[t] and the step is c_run[t] if c_run != NULL, else the oracle's own
 * <r,psi_idx>.  Before advancing it records, from the oracle's own r:
 *   argmax_ref[t], cmax_ref[t] = |c| at that argmax, c_at_idx[t] = signed c at idx_run[t],
 *   gap[t] as above (w.r.t. the oracle's argmax), rnorm[t] (t = 0..t_run, t_run+1 slots).
 * Outputs x[M], r[N] are the state after t_run forced steps. */
int oracle_mp_replay_f64(const double* psi_t, int N, int M, int64_t ld, const double* y,
                         const int* idx_run, const double* c_run, int t_run,
                         double* x, double* r,
                         int* argmax_ref, double* cmax_ref, double* c_at_idx, double* gap, double* rnorm,
                         int nthreads);
int oracle_mp_replay_f32(const float* psi_t, int N, int M, int64_t ld, const double* y,
                         const int* idx_run, const double* c_run, int t_run,
                         double* x, double* r,
                         int* argmax_ref, double* cmax_ref, double* c_at_idx, double* gap, double* rnorm,
                         int nthreads);

/* B signals sharing one dictionary: signal b is exactly oracle_mp on (Psi, Y[b]).
 * Y is B x N (row stride ldy), X is B x M, R is B x N, n_iter has B entries. */
int oracle_mp_batched_f32(const float* psi_t, int N, int M, int64_t ld, const double* Y, int64_t ldy, int B,
                          double eps, int T, double* X, double* R, int* n_iter, int nthreads);

/* Orthogonal MP (textbook definition, see mp_oracle.c): MP's selection followed by a least-squares
 * refit on the selected atoms (normal equations, Cholesky from scratch every iteration).  idx_force != NULL: the
 * teacher-forced replay over t_force imposed atoms.  Returns 0, 1 (invalid arguments) or 2 (an atom selected twice or
 * a singular Gram matrix ended the run). */
int oracle_omp_f32(const float* psi_t, int N, int M, int64_t ld, const double* y, double eps, int T,
                   const int* idx_force, int t_force,
                   double* x, double* r, int* n_iter,
                   int* idx_trace, double* gap_trace, double* rnorm_trace,
                   int* argmax_ref, double* cmax_ref, double* c_at_idx, int nthreads);

/* Eq. 2: y = Psi x for a K-sparse x given as (index, value) pairs (the paper builds x that way, A2 P:328-332):
 *   y[n] = sum_{k=0}^{K-1} val[k] * Psi[n][idx[k]],  ascending k, float64.  Repeated indices accumulate (the paper's
 * rand()%M support can repeat).  Returns 0, or 1 on invalid arguments (an index outside [0, M)). */
int oracle_encode_sparse_f32(const float* psi_t, int N, int M, int64_t ld, const int* idx, const double* val, int K, double* y);

/* Eq. 14: E = ||x_hat - x||_2^2 / ||x||_2^2 * 100 (percent). */
double oracle_reconstruction_error_pct(const double* x_hat, const double* x, int M);

#ifdef __cplusplus
}
#endif
#endif
