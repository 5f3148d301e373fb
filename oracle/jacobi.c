/*
 * oracle/jacobi.c -- TEST INFRASTRUCTURE ONLY (CPU oracle of the Triad-ATRG hot path).
 *
 * Plain, LAPACK-free dense decompositions used by oracle/tatrg_oracle.py:
 *   orc_jacobi_svd   one-sided (Hestenes) Jacobi SVD of a tall matrix
 *   orc_jacobi_eigh  two-sided (classical) Jacobi eigen-decomposition of a symmetric matrix
 *
 * PAPER.md is silent on how its SVDs are computed (":213 tensor contraction and SVD"); the paper's
 * truncated SVDs (Eq. 2.4 :76, Eq. 2.5 :90, Eq. 2.9 :135, Eq. A.8 :376) are *defined* by the SVD itself,
 * so the oracle uses the textbook Jacobi iterations, which converge to the exact decomposition.
 * Both use the round-robin ("chess tournament") ordering so that the n/2 rotations of one round are
 * independent; OpenMP runs them in parallel.  No code here is shared with the CUDA path.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may load this.
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>

/* round-robin pairing: n even "players" (pad with a bye if n odd), round r in [0, np-1) gives np/2 pairs */
static void rr_pairs(int np, int r, int *p, int *q)
{
    /* player np-1 is fixed, others rotate */
    int half = np / 2;
    for (int k = 0; k < half; ++k) {
        int a, b;
        if (k == 0) { a = np - 1; b = r % (np - 1); }
        else { a = (r + k) % (np - 1); b = (r - k + (np - 1)) % (np - 1); }
        if (a < b) { p[k] = a; q[k] = b; } else { p[k] = b; q[k] = a; }
    }
}

/*
 * One-sided Jacobi SVD.  At is n x m row-major: row j of At is COLUMN j of the m x n matrix A (m >= 1).
 * On exit: row j of At = sigma_j * u_j (NOT normalised), Vt is n x n row-major with row j = right singular
 * vector v_j (so A v_j = sigma_j u_j), sigma[j] = ||A v_j||.  Nothing is sorted (the caller sorts).
 * Rotation rule (Hestenes): for columns p<q with alpha=|a_p|^2, beta=|a_q|^2, gamma=a_p.a_q, rotate when
 * |gamma| > tol*sqrt(m)*sqrt(alpha*beta) (sqrt(m): the rounding floor of an m-term dot product, as in the
 * textbook criterion).  Returns the number of sweeps used, or -1 if max_sweeps was hit.
 */
int orc_jacobi_svd(int m, int n, double *At, double *sigma, double *Vt, double tol, int max_sweeps)
{
    tol *= sqrt((double)m);
    double amax = 0; /* largest squared column norm: columns 1e-40 times shorter are exactly null for FP64 */
    for (int j = 0; j < n; ++j) { double a2 = 0; for (int i = 0; i < m; ++i) a2 += At[(size_t)j * m + i] * At[(size_t)j * m + i]; if (a2 > amax) amax = a2; }
    const double null2 = 1e-80 * amax;
    memset(Vt, 0, sizeof(double) * (size_t)n * n);
    for (int j = 0; j < n; ++j) Vt[(size_t)j * n + j] = 1.0;
    int np = n + (n & 1);
    int half = np / 2;
    int *P = (int *)malloc(sizeof(int) * (half > 0 ? half : 1));
    int *Q = (int *)malloc(sizeof(int) * (half > 0 ? half : 1));
    int sweeps = 0, converged = (n < 2);
    while (!converged && sweeps < max_sweeps) {
        int rotated = 0;
        for (int r = 0; r < np - 1; ++r) {
            rr_pairs(np, r, P, Q);
#pragma omp parallel for schedule(static) reduction(+ : rotated)
            for (int k = 0; k < half; ++k) {
                int p = P[k], q = Q[k];
                if (q >= n) continue; /* bye */
                double *ap = At + (size_t)p * m, *aq = At + (size_t)q * m;
                double alpha = 0, beta = 0, gamma = 0;
                for (int i = 0; i < m; ++i) { alpha += ap[i] * ap[i]; beta += aq[i] * aq[i]; gamma += ap[i] * aq[i]; }
                if (alpha <= null2 || beta <= null2) continue;
                if (fabs(gamma) <= tol * sqrt(alpha) * sqrt(beta)) continue;
                double zeta = (beta - alpha) / (2.0 * gamma);
                double t = (zeta >= 0 ? 1.0 : -1.0) / (fabs(zeta) + sqrt(1.0 + zeta * zeta));
                double c = 1.0 / sqrt(1.0 + t * t), s = c * t;
                for (int i = 0; i < m; ++i) { double x = ap[i], y = aq[i]; ap[i] = c * x - s * y; aq[i] = s * x + c * y; }
                double *vp = Vt + (size_t)p * n, *vq = Vt + (size_t)q * n;
                for (int i = 0; i < n; ++i) { double x = vp[i], y = vq[i]; vp[i] = c * x - s * y; vq[i] = s * x + c * y; }
                rotated += 1;
            }
        }
        ++sweeps;
        if (!rotated) converged = 1;
    }
    for (int j = 0; j < n; ++j) {
        double *a = At + (size_t)j * m, s2 = 0;
        for (int i = 0; i < m; ++i) s2 += a[i] * a[i];
        sigma[j] = sqrt(s2);
    }
    free(P); free(Q);
    return converged ? sweeps : -1;
}

/*
 * Two-sided Jacobi eigen-decomposition of a symmetric n x n matrix S (row-major, overwritten; its diagonal
 * holds the eigenvalues on exit).  Vt is n x n row-major with row j = eigenvector j.  Each round computes the
 * n/2 independent rotations from (s_pp, s_qq, s_pq), applies them to the columns, then to the rows
 * (J^T S J with J a direct sum of plane rotations), and accumulates V.  Returns sweeps used or -1.
 */
int orc_jacobi_eigh(int n, double *S, double *lambda, double *Vt, double tol, int max_sweeps)
{
    memset(Vt, 0, sizeof(double) * (size_t)n * n);
    for (int j = 0; j < n; ++j) Vt[(size_t)j * n + j] = 1.0;
    int np = n + (n & 1);
    int half = np / 2;
    int *P = (int *)malloc(sizeof(int) * (half > 0 ? half : 1));
    int *Q = (int *)malloc(sizeof(int) * (half > 0 ? half : 1));
    double *Cs = (double *)malloc(sizeof(double) * (half > 0 ? half : 1));
    double *Sn = (double *)malloc(sizeof(double) * (half > 0 ? half : 1));
    int sweeps = 0, converged = (n < 2);
    double normF = 0;
    for (size_t i = 0; i < (size_t)n * n; ++i) normF += S[i] * S[i];
    normF = sqrt(normF);
    const double floor_abs = 1e-22 * normF; /* entries this far below ||S||_F are rounding noise */
    while (!converged && sweeps < max_sweeps) {
        int rotated = 0;
        for (int r = 0; r < np - 1; ++r) {
            rr_pairs(np, r, P, Q);
            for (int k = 0; k < half; ++k) {
                int p = P[k], q = Q[k];
                Cs[k] = 1.0; Sn[k] = 0.0;
                if (q >= n) continue;
                double app = S[(size_t)p * n + p], aqq = S[(size_t)q * n + q], apq = S[(size_t)p * n + q];
                if (fabs(apq) <= floor_abs) continue;
                if (fabs(apq) <= tol * sqrt(fabs(app * aqq))) continue;
                double zeta = (aqq - app) / (2.0 * apq);
                double t = (zeta >= 0 ? 1.0 : -1.0) / (fabs(zeta) + sqrt(1.0 + zeta * zeta));
                Cs[k] = 1.0 / sqrt(1.0 + t * t); Sn[k] = Cs[k] * t;
                rotated += 1;
            }
            /* columns: S <- S J  (row-wise loop so that memory access is contiguous) */
#pragma omp parallel for schedule(static)
            for (int i = 0; i < n; ++i) {
                double *row = S + (size_t)i * n;
                for (int k = 0; k < half; ++k) {
                    if (Sn[k] == 0.0) continue;
                    int p = P[k], q = Q[k];
                    double x = row[p], y = row[q];
                    row[p] = Cs[k] * x - Sn[k] * y; row[q] = Sn[k] * x + Cs[k] * y;
                }
            }
            /* rows: S <- J^T S, and V rows likewise */
#pragma omp parallel for schedule(static)
            for (int k = 0; k < half; ++k) {
                if (Sn[k] == 0.0) continue;
                int p = P[k], q = Q[k];
                double c = Cs[k], s = Sn[k];
                double *rp = S + (size_t)p * n, *rq = S + (size_t)q * n;
                for (int i = 0; i < n; ++i) { double x = rp[i], y = rq[i]; rp[i] = c * x - s * y; rq[i] = s * x + c * y; }
                double *vp = Vt + (size_t)p * n, *vq = Vt + (size_t)q * n;
                for (int i = 0; i < n; ++i) { double x = vp[i], y = vq[i]; vp[i] = c * x - s * y; vq[i] = s * x + c * y; }
                rp[q] = 0.0; rq[p] = 0.0; /* the rotation annihilates s_pq exactly; what is left is rounding */
            }
        }
        ++sweeps;
        if (!rotated) converged = 1;
    }
    for (int j = 0; j < n; ++j) lambda[j] = S[(size_t)j * n + j];
    free(P); free(Q); free(Cs); free(Sn);
    return converged ? sweeps : -1;
}
