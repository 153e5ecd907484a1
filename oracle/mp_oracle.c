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
