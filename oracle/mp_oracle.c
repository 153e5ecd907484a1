/* mp_oracle.c -- CPU ORACLE for Matching Pursuit.  TEST INFRASTRUCTURE, NOT THE PRODUCT.
 * Plain float64 C loops written from PAPER.md (arxiv 0809.1833); see mp_oracle.h for the
 * contract, the readings and the pins.  Build: oracle/build.py (gcc -O2 -fopenmp, no fast-math). */
#include "mp_oracle.h"
#include <math.h>
#include <stdlib.h>

/* Eq. 18: ||v||_2 = sqrt(sum v_n^2), direct sum, ascending n. */
double oracle_nrm2(const double* v, int n)
{
    double s = 0.0;
    for (int k = 0; k < n; k++) s += v[k] * v[k];
    return sqrt(s);
}

/* Eq. 16: "the smallest index of the maximum magnitude element".
 * Strict '>' scan from m = 0, so the first maximiser wins; a NaN never compares greater. */
int oracle_argmax_abs(const double* c, int M)
{
    int best = 0;
    double best_abs = -1.0;
    for (int m = 0; m < M; m++) {
        const double a = fabs(c[m]);
        if (a > best_abs) { best_abs = a; best = m; }
    }
    return best;
}

/* (a1 - a2)/a1 with a1 = |c[i]| the maximum and a2 the largest magnitude among m != i. */
static double top_two_gap(const double* c, int M, int i)
{
    const double a1 = fabs(c[i]);
    double a2 = 0.0;
    for (int m = 0; m < M; m++)
        if (m != i && fabs(c[m]) > a2) a2 = fabs(c[m]);
    return a1 > 0.0 ? (a1 - a2) / a1 : 0.0;
}

/* Eq. 4: ||psi_m||_2 = 1 for all m. */
void oracle_normalize_columns_f64(double* psi_t, int N, int M, int64_t ld, double* norms_out)
{
    for (int m = 0; m < M; m++) {
        double* psi_m = psi_t + (int64_t)m * ld;
        const double s = oracle_nrm2(psi_m, N);
        if (norms_out) norms_out[m] = s;
        if (s > 0.0)
            for (int n = 0; n < N; n++) psi_m[n] /= s;
    }
}

#define PSI_T double
#define FN(name) name##_f64
#include "mp_oracle_body.inc"
#undef PSI_T
#undef FN

#define PSI_T float
#define FN(name) name##_f32
#include "mp_oracle_body.inc"
#undef PSI_T
#undef FN

/* P:165 "all signals are encoded/decoded with the same dictionary": B independent MP runs. */
int oracle_mp_batched_f32(const float* psi_t, int N, int M, int64_t ld, const double* Y, int64_t ldy, int B,
                          double eps, int T, double* X, double* R, int* n_iter, int nthreads)
{
    if (B < 1 || !Y || !X || !R || !n_iter || ldy < N) return 1;
    for (int b = 0; b < B; b++) {
        int rc = oracle_mp_f32(psi_t, N, M, ld, Y + (int64_t)b * ldy, eps, T,
                               X + (int64_t)b * M, R + (int64_t)b * N, n_iter + b,
                               NULL, NULL, NULL, NULL, nthreads);
        if (rc) return rc;
    }
    return 0;
}

/* Orthogonal Matching Pursuit -- the paper's declared next target ("orthogonal MP"; it gives no
 * listing, so this is the textbook definition of its refs [5], [12]):
 *     S <- {}, r <- y, t <- 0
 *     while ||r||_2 > eps ||y||_2 and t < T:                            (the stop rule of MP)
 *         i <- argmax_m |<r, psi_m>|   (smallest index on ties)          (Eq. 9 / Eq. 16, the selection of MP)
 *         S <- S + {i}
 *         x_S <- argmin_z || y - Psi_S z ||_2                            (least squares on the selected atoms)
 *         r <- y - Psi_S x_S ;  t <- t + 1
 *     x~ <- x_S on S, 0 elsewhere
 * The least-squares problem is solved by its normal equations (Psi_S^T Psi_S) z = Psi_S^T y with a Cholesky
 * factorisation recomputed FROM SCRATCH every iteration (the Gram matrix itself gets one new row per iteration).
 * If idx_force != NULL the atom taken at step t is idx_force[t] (teacher-forced replay, t_force steps, no stop
 * test); the oracle's own argmax, |c| at it, the signed c at the imposed atom and the top-two gap are recorded
 * from the oracle's own r before the step.  An atom already in S, or a Gram matrix that is not positive definite,
 * ends the run (return 2: the state of the last completed step is kept).
 * Outputs x[M], r[N], *n_iter; traces nullable: idx[t], gap[t], rnorm[t] (t+1 entries), and for replay
 * argmax_ref[t], cmax_ref[t], c_at_idx[t]. */
int oracle_omp_f32(const float* psi_t, int N, int M, int64_t ld, const double* y, double eps, int T,
                   const int* idx_force, int t_force,
                   double* x, double* r, int* n_iter,
                   int* idx_trace, double* gap_trace, double* rnorm_trace,
                   int* argmax_ref, double* cmax_ref, double* c_at_idx, int nthreads)
{
    if (!psi_t || !y || !x || !r || !n_iter || N < 1 || M < 1 || ld < N || T < 0 || !(eps >= 0.0)) return 1;
    const int Tmax = idx_force ? t_force : (T < N ? T : N);                /* more than N atoms cannot be independent */
    const int cap = Tmax > 0 ? Tmax : 1;
    double* c = (double*)malloc((size_t)M * sizeof(double));
    double* G = (double*)malloc((size_t)cap * cap * sizeof(double));       /* Gram matrix Psi_S^T Psi_S, row-major */
    double* L = (double*)malloc((size_t)cap * cap * sizeof(double));       /* its Cholesky factor */
    double* b = (double*)malloc((size_t)cap * sizeof(double));             /* Psi_S^T y */
    double* z = (double*)malloc((size_t)cap * sizeof(double));
    int* S = (int*)malloc((size_t)cap * sizeof(int));
    if (!c || !G || !L || !b || !z || !S) { free(c); free(G); free(L); free(b); free(z); free(S); return 1; }
    int rc = 0, t = 0;
    for (int m = 0; m < M; m++) x[m] = 0.0;
    for (int n = 0; n < N; n++) r[n] = y[n];
    const double norm_y = oracle_nrm2(y, N);
    for (;;) {
        const double norm_r = oracle_nrm2(r, N);
        if (rnorm_trace) rnorm_trace[t] = norm_r;
        if (idx_force) { if (t >= t_force) break; }
        else if (!(norm_r > eps * norm_y) || !(t < Tmax)) break;

        oracle_correlate_f32(psi_t, N, M, ld, r, c, nthreads);
        const int i_ref = oracle_argmax_abs(c, M);
        const int i = idx_force ? idx_force[t] : i_ref;
        if (i < 0 || i >= M) { rc = 1; break; }
        if (gap_trace) gap_trace[t] = top_two_gap(c, M, i_ref);
        if (argmax_ref) argmax_ref[t] = i_ref;
        if (cmax_ref) cmax_ref[t] = fabs(c[i_ref]);
        if (c_at_idx) c_at_idx[t] = c[i];
        int dup = 0;
        for (int k = 0; k < t; k++) dup |= (S[k] == i);
        if (dup) { rc = 2; break; }

        /* S <- S + {i}: one new row/column of the Gram matrix and one new entry of Psi_S^T y */
        const float* psi_i = psi_t + (int64_t)i * ld;
        S[t] = i;
        for (int k = 0; k <= t; k++) {
            const float* psi_k = psi_t + (int64_t)S[k] * ld;
            double g = 0.0;
            for (int n = 0; n < N; n++) g += (double)psi_k[n] * (double)psi_i[n];
            G[(size_t)t * cap + k] = g;
            G[(size_t)k * cap + t] = g;
        }
        { double s = 0.0; for (int n = 0; n < N; n++) s += (double)psi_i[n] * y[n]; b[t] = s; }
        const int ts = t + 1;

        /* Cholesky G = L L^T from scratch, then L w = b, L^T z = w */
        int ok = 1;
        for (int p = 0; p < ts && ok; p++) {
            for (int q = 0; q <= p; q++) {
                double s = G[(size_t)p * cap + q];
                for (int k = 0; k < q; k++) s -= L[(size_t)p * cap + k] * L[(size_t)q * cap + k];
                if (p == q) { if (!(s > 0.0)) { ok = 0; break; } L[(size_t)p * cap + p] = sqrt(s); }
                else L[(size_t)p * cap + q] = s / L[(size_t)q * cap + q];
            }
        }
        if (!ok) { rc = 2; break; }
        for (int p = 0; p < ts; p++) {
            double s = b[p];
            for (int k = 0; k < p; k++) s -= L[(size_t)p * cap + k] * z[k];
            z[p] = s / L[(size_t)p * cap + p];
        }
        for (int p = ts - 1; p >= 0; p--) {
            double s = z[p];
            for (int k = p + 1; k < ts; k++) s -= L[(size_t)k * cap + p] * z[k];
            z[p] = s / L[(size_t)p * cap + p];
        }
        /* x_S <- z, r <- y - Psi_S x_S */
        for (int k = 0; k < ts; k++) x[S[k]] = z[k];
        for (int n = 0; n < N; n++) {
            double s = y[n];
            for (int k = 0; k < ts; k++) s -= z[k] * (double)psi_t[(int64_t)S[k] * ld + n];
            r[n] = s;
        }
        if (idx_trace) idx_trace[t] = i;
        t += 1;
    }
    *n_iter = t;
    free(c); free(G); free(L); free(b); free(z); free(S);
    return rc;
}

/* Eq. 2: y = Psi x, x K-sparse as (idx, val) pairs; one serial ascending-k sum per component. */
int oracle_encode_sparse_f32(const float* psi_t, int N, int M, int64_t ld, const int* idx, const double* val, int K, double* y)
{
    if (!psi_t || !y || N < 1 || M < 1 || K < 0 || ld < N || (K > 0 && (!idx || !val))) return 1;
    for (int k = 0; k < K; k++)
        if (idx[k] < 0 || idx[k] >= M) return 1;
    for (int n = 0; n < N; n++) {
        double s = 0.0;
        for (int k = 0; k < K; k++) s += val[k] * (double)psi_t[(int64_t)idx[k] * ld + n];
        y[n] = s;
    }
    return 0;
}

/* Eq. 14: E = ||x~ - x||^2 ||x||^-2 x 100%. */
double oracle_reconstruction_error_pct(const double* x_hat, const double* x, int M)
{
    double num = 0.0, den = 0.0;
    for (int m = 0; m < M; m++) {
        num += (x_hat[m] - x[m]) * (x_hat[m] - x[m]);
        den += x[m] * x[m];
    }
    return 100.0 * num / den;
}
