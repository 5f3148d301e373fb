// cholesky.cu -- blocked Cholesky factorisation and the triangular solve X L^-T, the orthonormalisation step of
//   * the subspace iterations that replace full eigen-decompositions where only a leading invariant subspace is needed
//     (triad isometries, Eq. 2.9 :135 -- top-K eigenvectors of a D^2 x D^2 Gram matrix; squeezers :171 -- top-D
//     eigenvectors of Theta_b Theta_f), and
//   * the QR pre-reduction of the bond swap (Eq. A.2-A.3 :345-348) as a Cholesky QR when the operand has full
//     numerical rank.
//
//   A (n x n, symmetric positive semi-definite, lower triangle read and destroyed) = L L^T,  L lower triangular.
//   Right-looking over 64-wide panels: the diagonal block is factored and inverted by ONE CTA in shared memory
//   (potrf_block_kernel), the panel below it and the trailing update are DGEMMs on the FP64 tensor cores.
//   Q = X L^-T by forward substitution over the same panels: two DGEMMs per panel.
//
// Cholesky's rounding error is invariant under diagonal scaling (|dA_ij| <= c eps sqrt(a_ii a_jj)), so graded Gram
// matrices (columns of very different norm, the normal state of a converging subspace iteration) need no explicit
// equilibration; the optional shift multiplies the diagonal by (1 + shift), which bounds the condition of the
// *scaled* matrix, and a pivot is never taken below guard_rel x its original diagonal entry.
#include "internal.h"

namespace tatrg {
namespace {
constexpr int PB = 64;        // panel width
constexpr int PP = PB + 1;    // shared-memory pitch
constexpr int kPotrfSmem = (2 * PB * PP + 2 * PB) * 8;

__global__ void symmetrize_kernel(int n, double* __restrict__ A) {
    const int64_t total = (int64_t)n * n;
    for (int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; e < total; e += (int64_t)gridDim.x * blockDim.x) {
        const int i = (int)(e / n), j = (int)(e - (int64_t)i * n);
        if (i < j) {
            const double v = 0.5 * (A[e] + A[(int64_t)j * n + i]);
            A[e] = v; A[(int64_t)j * n + i] = v;
        }
    }
}

__global__ void diag_shift_kernel(int n, double* __restrict__ A, int64_t lda, double shift, double* __restrict__ d0) {
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) {
        const double v = A[(int64_t)i * lda + i];
        d0[i] = v;
        A[(int64_t)i * lda + i] = v * (1.0 + shift);
    }
}

// Diagonal block [j0, j0+nb) of A -> L block (upper part of the block zeroed) and its inverse Linv (PB x PB, zero padded).
// info[0] |= 1 when a pivot had to be raised to the guard, |= 2 when a pivot was not finite.
__global__ void __launch_bounds__(256, 1) potrf_block_kernel(int nb, int j0, const double* __restrict__ A, int64_t lda, double* __restrict__ L,
                                                             int64_t ldl, double* __restrict__ Linv, const double* __restrict__ d0,
                                                             double guard_rel, int* __restrict__ info) {
    extern __shared__ double sh_potrf[];
    double* S = sh_potrf; double* X = S + PB * PP; double* dg = X + PB * PP; double* rdg = dg + PB;
    const int tid = threadIdx.x;
    for (int e = tid; e < PB * PB; e += 256) {
        const int i = e >> 6, j = e & 63;
        S[i * PP + j] = (i < nb && j <= i) ? A[(int64_t)(j0 + i) * lda + j0 + j] : 0.0;
        X[i * PP + j] = 0.0;
    }
    __syncthreads();
    int flag = 0;
    for (int j = 0; j < nb; ++j) {
        // left-looking: s_i = a_ij - sum_{k<j} l_ik l_jk   (thread i, i >= j)
        if (tid >= j && tid < nb) {
            double s0 = S[tid * PP + j], s1 = 0, s2 = 0, s3 = 0;
            int k = 0;
            for (; k + 3 < j; k += 4) {
                s0 -= S[tid * PP + k] * S[j * PP + k];
                s1 -= S[tid * PP + k + 1] * S[j * PP + k + 1];
                s2 -= S[tid * PP + k + 2] * S[j * PP + k + 2];
                s3 -= S[tid * PP + k + 3] * S[j * PP + k + 3];
            }
            for (; k < j; ++k) s0 -= S[tid * PP + k] * S[j * PP + k];
            S[tid * PP + j] = (s0 + s1) + (s2 + s3);
        }
        __syncthreads();
        if (tid >= j && tid < nb) {
            double p = S[j * PP + j];
            const double floor_p = fmax(guard_rel * fabs(d0[j0 + j]), 1e-290);
            if (!(p == p) || fabs(p) > 1e300) { flag |= 2; p = floor_p; }
            if (p < floor_p) { flag |= 1; p = floor_p; }
            const double r = 1.0 / sqrt(p);
            if (tid == j) { dg[j] = p * r; rdg[j] = r; }
            else S[tid * PP + j] *= r;
        }
        __syncthreads();
    }
    if (tid < nb) S[tid * PP + tid] = dg[tid];
    if (flag) atomicOr(info, flag);
    __syncthreads();
    // inverse of the lower-triangular block, one column per thread: x_c = 1/l_cc, x_i = -(sum_{k<i} l_ik x_k) / l_ii
    if (tid < nb) {
        const int c = tid;
        for (int i = 0; i < nb; ++i) {
            double a0 = 0, a1 = 0;
            int k = 0;
            for (; k + 1 < i; k += 2) { a0 += S[i * PP + k] * X[k * PP + c]; a1 += S[i * PP + k + 1] * X[(k + 1) * PP + c]; }
            for (; k < i; ++k) a0 += S[i * PP + k] * X[k * PP + c];
            const double rhs = (i == c) ? 1.0 : 0.0;
            X[i * PP + c] = (i < c) ? 0.0 : (rhs - (a0 + a1)) * rdg[i];
        }
    }
    __syncthreads();
    for (int e = tid; e < PB * PB; e += 256) {
        const int i = e >> 6, j = e & 63;
        Linv[e] = (i < nb && j < nb) ? X[i * PP + j] : 0.0;
        if (i < nb && j < nb) L[(int64_t)(j0 + i) * ldl + j0 + j] = (j <= i) ? S[i * PP + j] : 0.0;
    }
}

__global__ void extract_diag_ld_kernel(int n, const double* __restrict__ A, int64_t lda, double* __restrict__ d) {
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) d[i] = A[(int64_t)i * lda + i];
}
}  // namespace

cudaError_t symmetrize(cudaStream_t st, int n, double* A) {
    int64_t blocks = ((int64_t)n * n + 255) / 256; if (blocks > 148 * 8) blocks = 148 * 8;
    symmetrize_kernel<<<(unsigned)blocks, 256, 0, st>>>(n, A); count_launch();
    return cudaGetLastError();
}

size_t cholesky_work_doubles(int n) { return (size_t)((n + PB - 1) / PB) * PB * PB + (size_t)n + 64; }

// A [n x n, lda] (lower triangle read, destroyed) -> L [n x n, ldl] lower triangular (strict upper part of the diagonal
// blocks zeroed; blocks above the diagonal are not touched).  work: cholesky_work_doubles(n) doubles [dev]:
// [Linv of every panel | d0 | info].  Asynchronous.
cudaError_t cholesky(cudaStream_t st, int n, double* A, int64_t lda, double* L, int64_t ldl, double shift, double guard_rel, double* work) {
    const int np = (n + PB - 1) / PB;
    double* Linv = work; double* d0 = work + (size_t)np * PB * PB; int* info = (int*)(d0 + n);
    static bool cfg = false;
    if (!cfg) {
        cudaError_t ea = cudaFuncSetAttribute(potrf_block_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, kPotrfSmem);
        if (ea != cudaSuccess) return ea;
        cfg = true;
    }
    cudaError_t e = cudaMemsetAsync(info, 0, sizeof(int), st);
    if (e != cudaSuccess) return e;
    diag_shift_kernel<<<(n + 255) / 256, 256, 0, st>>>(n, A, lda, shift, d0); count_launch();
    for (int p = 0; p < np; ++p) {
        const int j0 = p * PB, nb = n - j0 < PB ? n - j0 : PB, m = n - j0 - nb;
        potrf_block_kernel<<<1, 256, kPotrfSmem, st>>>(nb, j0, A, lda, L, ldl, Linv + (size_t)p * PB * PB, d0, guard_rel, info); count_launch();
        if (m <= 0) break;
        // panel below: L[i, j0:j0+nb] = A[i, j0:j0+nb] Linv^T
        e = dgemm(st, false, true, m, nb, nb, 1.0, A + (int64_t)(j0 + nb) * lda + j0, lda, Linv + (size_t)p * PB * PB, PB, 0.0,
                  L + (int64_t)(j0 + nb) * ldl + j0, ldl);
        if (e != cudaSuccess) return e;
        // trailing update: A[i, k] -= sum_j L[i, j] L[k, j]
        e = dgemm(st, false, true, m, m, nb, -1.0, L + (int64_t)(j0 + nb) * ldl + j0, ldl, L + (int64_t)(j0 + nb) * ldl + j0, ldl, 1.0,
                  A + (int64_t)(j0 + nb) * lda + j0 + nb, lda);
        if (e != cudaSuccess) return e;
    }
    return cudaGetLastError();
}
const double* cholesky_d0(const double* work, int n) { return work + (size_t)((n + PB - 1) / PB) * PB * PB; }
const int* cholesky_info(const double* work, int n) { return (const int*)(work + (size_t)((n + PB - 1) / PB) * PB * PB + n); }

// Q [m x n, ldq] = X [m x n, ldx] L^-T with L, Linv from cholesky().  X is overwritten (it holds the partially reduced
// right-hand side afterwards).  Asynchronous.
cudaError_t trsm_right_lt(cudaStream_t st, int64_t m, int n, double* X, int64_t ldx, double* Q, int64_t ldq, const double* L, int64_t ldl,
                          const double* work) {
    const int np = (n + PB - 1) / PB;
    const double* Linv = work;
    for (int p = 0; p < np; ++p) {
        const int j0 = p * PB, nb = n - j0 < PB ? n - j0 : PB;
        cudaError_t e;
        if (j0 > 0) {   // X_j -= Q[:, 0:j0] L[j0:j0+nb, 0:j0]^T
            e = dgemm(st, false, true, m, nb, j0, -1.0, Q, ldq, L + (int64_t)j0 * ldl, ldl, 1.0, X + j0, ldx);
            if (e != cudaSuccess) return e;
        }
        e = dgemm(st, false, true, m, nb, nb, 1.0, X + j0, ldx, Linv + (size_t)p * PB * PB, PB, 0.0, Q + j0, ldq);
        if (e != cudaSuccess) return e;
    }
    return cudaSuccess;
}

// X [n x n, ldx] = L^-1 (lower triangular; X must be zero-filled on entry) from the factor and the inverted diagonal blocks
// that cholesky() left in work.  T: scratch of 64 x n doubles.  Row panel i: X[i, <i] = -Linv_ii (L[i, <i] X[<i, <i]).
cudaError_t tri_inverse(cudaStream_t st, int n, const double* L, int64_t ldl, const double* work, double* X, int64_t ldx, double* T) {
    const int np = (n + PB - 1) / PB;
    const double* Linv = work;
    for (int p = 0; p < np; ++p) {
        const int i0 = p * PB, nb = n - i0 < PB ? n - i0 : PB;
        cudaError_t e = cudaMemcpy2DAsync(X + (int64_t)i0 * ldx + i0, ldx * 8, Linv + (size_t)p * PB * PB, PB * 8, (size_t)nb * 8, nb,
                                          cudaMemcpyDeviceToDevice, st);
        count_launch();
        if (e != cudaSuccess) return e;
        if (i0 == 0) continue;
        e = dgemm(st, false, false, nb, i0, i0, 1.0, L + (int64_t)i0 * ldl, ldl, X, ldx, 0.0, T, i0);
        if (e != cudaSuccess) return e;
        e = dgemm(st, false, false, nb, i0, nb, -1.0, Linv + (size_t)p * PB * PB, PB, T, i0, 0.0, X + (int64_t)i0 * ldx, ldx);
        if (e != cudaSuccess) return e;
    }
    return cudaSuccess;
}

cudaError_t extract_diag(cudaStream_t st, int n, const double* A, int64_t lda, double* d) {
    extract_diag_ld_kernel<<<(n + 255) / 256, 256, 0, st>>>(n, A, lda, d); count_launch();
    return cudaGetLastError();
}

}  // namespace tatrg
