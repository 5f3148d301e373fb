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
#ifndef TATRG_POTRF_CW
#define TATRG_POTRF_CW 16
#endif
constexpr int kPotrfCW = TATRG_POTRF_CW;
constexpr int kPotrfSmem = (2 * PB * PP + 32 * 33 + 4 * PB) * 8;

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

__global__ void mirror_lower_kernel(int n, double* __restrict__ A) {      // 32 x 32 tiles through shared memory
    __shared__ double t[32][33];
    const int bi = blockIdx.y, bj = blockIdx.x;
    if (bj < bi) return;                                                   // (bi, bj) upper tile <- transpose of lower tile (bj, bi)
    for (int r = threadIdx.y; r < 32; r += 8) {
        const int i = bj * 32 + r, j = bi * 32 + threadIdx.x;
        t[r][threadIdx.x] = (i < n && j < n) ? A[(int64_t)i * n + j] : 0.0;
    }
    __syncthreads();
    for (int r = threadIdx.y; r < 32; r += 8) {
        const int i = bi * 32 + r, j = bj * 32 + threadIdx.x;
        if (i < n && j < n && i < j) A[(int64_t)i * n + j] = t[threadIdx.x][r];
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
// 256 threads: thread (i = tid & 63, g = tid >> 6) keeps the 16 entries [i][16 g .. 16 g + 15] of its row in registers.
// Factorisation, right-looking: step j publishes column j through shared memory (double-buffered: one barrier per step),
// every thread scales it by 1/sqrt(pivot) and updates its 16 entries.  Inverse, also right-looking: once row k of
// X = L^-1 is final, every row i > k accumulates l_ik x_k; row k+1 is finished by its own four threads.
template <int CW>      // columns per thread: 64 / CW column groups, 64 * (64 / CW) threads
__global__ void __launch_bounds__(64 * (PB / CW), 1) potrf_block_kernel(int nb, int j0, const double* __restrict__ A, int64_t lda, double* __restrict__ L,
                                                             int64_t ldl, double* __restrict__ Linv, const double* __restrict__ d0,
                                                             double guard_rel, int* __restrict__ info) {
    extern __shared__ double sh_potrf[];
    double* Ls = sh_potrf;                               // the factor, for the inverse
    double* Xs = Ls + PB * PP;                           // the inverse
    double* Ts = Xs + PB * PP;                           // 32 x 33 scratch of the doubling levels
    double (*col)[PB] = reinterpret_cast<double (*)[PB]>(Ts + 32 * 33);     // published column, double-buffered
    double* floor_s = &col[2][0];                        // pivot floors (global loads kept out of the column loop)
    double* rdiag_s = floor_s + PB;                      // 1 / l_jj
    const int tid = threadIdx.x, i = tid & 63, g = tid >> 6, c0 = g * CW;
    if (tid < PB) floor_s[tid] = fmax(guard_rel * (tid < nb ? fabs(d0[j0 + tid]) : 1.0), 1e-290);
    double a[CW];
#pragma unroll
    for (int cc = 0; cc < CW; ++cc) {
        const int c = c0 + cc;
        a[cc] = (i < nb && c <= i) ? A[(int64_t)(j0 + i) * lda + j0 + c] : ((i == c) ? 1.0 : 0.0);   // identity padding beyond nb
    }
    int flag = 0;
    // Column j = gj CW + jj: the inner loop is unrolled so that the owners publish a[jj] with a static register index (a
    // run-time index costs a chain of CW dependent selects per column, ~20 % of the whole step).
#pragma unroll 1
    for (int gj = 0; gj < PB / CW; ++gj) {
#pragma unroll
        for (int jj = 0; jj < CW; ++jj) {
            const int j = gj * CW + jj, buf = jj & 1;
            if (g == gj) col[buf][i] = a[jj];
            __syncthreads();
            double p = col[buf][j];
            const double floor_p = floor_s[j];
            if (!(p >= floor_p && p <= 1e300)) {        // rare: the reciprocal square root below does not wait for this test
                flag |= (p < floor_p) ? 1 : 2;
                p = floor_p;
            }
            // warps whose rows all lie above the pivot row, or whose columns all lie left of it, have nothing to update
            // (both conditions are warp-uniform)
            if ((i | 31) < j || c0 + CW - 1 < j) continue;
            // l_i l_c = (a_ij / p) a_cj: one DMUL per thread and one DFMA per entry instead of a DMUL + DFMA per entry
            const double r = rsqrt(p);
            if (i == j && g == gj) rdiag_s[j] = r;       // 1 / l_jj = 1 / sqrt(p)
            const double ci = (i >= j) ? col[buf][i] : 0.0;
            const double lip = ci * (r * r);
            const double li = (i == j) ? p * r : ci * r;
#pragma unroll
            for (int cc = 0; cc < CW; ++cc) {
                const int c = c0 + cc;
                if (c > j) a[cc] -= lip * col[buf][c];
                else if (c == j) a[cc] = li;
            }
        }
    }
    if (flag && tid == 0) atomicOr(info, flag);
    // factor to shared memory and to L
#pragma unroll
    for (int cc = 0; cc < CW; ++cc) {
        const int c = c0 + cc;
        const double v = (c <= i) ? a[cc] : 0.0;
        Ls[i * PP + c] = v;
        if (i < nb && c < nb) L[(int64_t)(j0 + i) * ldl + j0 + c] = v;
    }
    __syncthreads();
    // X = L^-1 without a serial pass over the 64 rows: the four 16 x 16 diagonal blocks are inverted side by side (one
    // column per thread, right-looking substitution in registers, no barrier), then two doubling levels
    // [[X11, 0], [-X22 (L21 X11), X22]] (block size 16, then 32) with all threads: five barriers in total.
    constexpr int NT = 64 * (PB / CW);
    for (int e = tid; e < PB * PB; e += NT) Xs[(e >> 6) * PP + (e & 63)] = 0.0;
    __syncthreads();
    if (tid < PB) {
        const int o = tid & ~15, c = tid & 15;         // block origin, column inside the block
        double x[16];
#pragma unroll
        for (int r = 0; r < 16; ++r) x[r] = (r == c) ? 1.0 : 0.0;
#pragma unroll
        for (int r = 0; r < 16; ++r) {
            const double xr = (r < c) ? 0.0 : x[r] * rdiag_s[o + r];
            x[r] = xr;
#pragma unroll
            for (int r2 = r + 1; r2 < 16; ++r2) x[r2] -= Ls[(o + r2) * PP + o + r] * xr;
        }
#pragma unroll
        for (int r = 0; r < 16; ++r) Xs[(o + r) * PP + o + c] = x[r];
    }
    __syncthreads();
#pragma unroll 1
    for (int sz = 16; sz < PB; sz *= 2) {
        const int total = (PB / 2) * sz;               // (64 / 2 sz) pairs of sz x sz outputs
        for (int e = tid; e < total; e += NT) {        // T = L21 X11
            const int q = e / (sz * sz), r = e - q * sz * sz, ii = r / sz, c = r - ii * sz, o = 2 * sz * q;
            double acc = 0.0;
            for (int k = c; k < sz; ++k) acc += Ls[(o + sz + ii) * PP + o + k] * Xs[(o + k) * PP + o + c];     // X11 is lower triangular
            Ts[(q * sz + ii) * 33 + c] = acc;
        }
        __syncthreads();
        for (int e = tid; e < total; e += NT) {        // X21 = -X22 T
            const int q = e / (sz * sz), r = e - q * sz * sz, ii = r / sz, c = r - ii * sz, o = 2 * sz * q;
            double acc = 0.0;
            for (int k = 0; k <= ii; ++k) acc += Xs[(o + sz + ii) * PP + o + sz + k] * Ts[(q * sz + k) * 33 + c];   // X22 too
            Xs[(o + sz + ii) * PP + o + c] = -acc;
        }
        __syncthreads();
    }
    for (int e = tid; e < PB * PB; e += NT) {
        const int r = e >> 6, c = e & 63;
        Linv[e] = (r < nb && c < nb) ? Xs[r * PP + c] : 0.0;
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

cudaError_t mirror_lower(cudaStream_t st, int n, double* A) {
    const int nt = (n + 31) / 32;
    mirror_lower_kernel<<<dim3(nt, nt), dim3(32, 8), 0, st>>>(n, A); count_launch();
    return cudaGetLastError();
}

size_t cholesky_work_doubles(int n) { return (size_t)((n + PB - 1) / PB) * PB * PB + (size_t)n + 64; }

// A [n x n, lda] (lower triangle read, destroyed) -> L [n x n, ldl] lower triangular (strict upper part of the diagonal
// blocks zeroed; blocks above the diagonal are not touched).  work: cholesky_work_doubles(n) doubles [dev]:
// [Linv of every panel | d0 | info].  Asynchronous.
cudaError_t cholesky(cudaStream_t st, int n, double* A, int64_t lda, double* L, int64_t ldl, double shift, double guard_rel, double* work,
                     bool reset_info) {
    const int np = (n + PB - 1) / PB;
    double* Linv = work; double* d0 = work + (size_t)np * PB * PB; int* info = (int*)(d0 + n);
    static unsigned long long cfg = 0;
    if (first_use_on_device(cfg)) {
        cudaError_t ea = cudaFuncSetAttribute(potrf_block_kernel<kPotrfCW>, cudaFuncAttributeMaxDynamicSharedMemorySize, kPotrfSmem);
        if (ea != cudaSuccess) return ea;
    }
    cudaError_t e = cudaSuccess;
    if (reset_info) { e = cudaMemsetAsync(info, 0, sizeof(int), st); count_launch(); }
    if (e != cudaSuccess) return e;
    diag_shift_kernel<<<(n + 255) / 256, 256, 0, st>>>(n, A, lda, shift, d0); count_launch();
    for (int p = 0; p < np; ++p) {
        const int j0 = p * PB, nb = n - j0 < PB ? n - j0 : PB, m = n - j0 - nb;
        potrf_block_kernel<kPotrfCW><<<1, 64 * (PB / kPotrfCW), kPotrfSmem, st>>>(nb, j0, A, lda, L, ldl, Linv + (size_t)p * PB * PB, d0, guard_rel, info); count_launch();
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
// that cholesky() left in work.  T: scratch of tri_inverse_scratch_doubles(n).
//   n = 64 * 2^k: recursive doubling, [[X11, 0], [-X22 L21 X11, X22]] for all pairs of a level in two batched DGEMMs
//   (2 log2(n/64) launches, square products);  otherwise row panels: X[i, <i] = -Linv_ii (L[i, <i] X[<i, <i]).
size_t tri_inverse_scratch_doubles(int n) { const size_t a = (size_t)n * n / 4, b = (size_t)PB * n; return a > b ? a : b; }
cudaError_t tri_inverse(cudaStream_t st, int n, const double* L, int64_t ldl, const double* work, double* X, int64_t ldx, double* T) {
    const int np = (n + PB - 1) / PB;
    const double* Linv = work;
    const bool pow2 = (n % PB == 0) && ((np & (np - 1)) == 0);
    for (int p = 0; p < np; ++p) {
        const int i0 = p * PB, nb = n - i0 < PB ? n - i0 : PB;
        cudaError_t e = cudaMemcpy2DAsync(X + (int64_t)i0 * ldx + i0, ldx * 8, Linv + (size_t)p * PB * PB, PB * 8, (size_t)nb * 8, nb,
                                          cudaMemcpyDeviceToDevice, st);
        count_launch();
        if (e != cudaSuccess) return e;
        if (pow2 || i0 == 0) continue;
        e = dgemm(st, false, false, nb, i0, i0, 1.0, L + (int64_t)i0 * ldl, ldl, X, ldx, 0.0, T, i0);
        if (e != cudaSuccess) return e;
        e = dgemm(st, false, false, nb, i0, nb, -1.0, Linv + (size_t)p * PB * PB, PB, T, i0, 0.0, X + (int64_t)i0 * ldx, ldx);
        if (e != cudaSuccess) return e;
    }
    if (pow2)
        for (int64_t s = PB; s < n; s *= 2) {
            const int pairs = (int)(n / (2 * s));
            cudaError_t e = dgemm(st, false, false, s, s, s, 1.0, L + s * ldl, ldl, X, ldx, 0.0, T, s, pairs, 2 * s * (ldl + 1), 2 * s * (ldx + 1), s * s);
            if (e != cudaSuccess) return e;
            e = dgemm(st, false, false, s, s, s, -1.0, X + s * ldx + s, ldx, T, s, 0.0, X + s * ldx, ldx, pairs, 2 * s * (ldx + 1), s * s, 2 * s * (ldx + 1));
            if (e != cudaSuccess) return e;
        }
    return cudaSuccess;
}

cudaError_t extract_diag(cudaStream_t st, int n, const double* A, int64_t lda, double* d) {
    extract_diag_ld_kernel<<<(n + 255) / 256, 256, 0, st>>>(n, A, lda, d); count_launch();
    return cudaGetLastError();
}

}  // namespace tatrg
