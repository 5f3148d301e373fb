// internal.h -- declarations shared by the CUDA sources of libtatrg (product path; shares nothing with oracle/).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <stddef.h>
#include <string>
#include <vector>
#include <map>
#include "../../include/tatrg.h"

namespace tatrg {

// ---- numerical readings: stated here independently of the oracle ----------------------
constexpr double kTauDefault = 1e-6;      // R7 multiplet gap
constexpr double kEpsOrthLambda = 1e-12;  // R14: Gram eigenvalue floor in orth() = (1e-6)^2 on singular values
constexpr double kEpsSV = 1e-12;          // R14: small accurate cores
constexpr double kEpsLambda = 1e-12;      // R14: Gram eigenvalues
constexpr double kEpsSqueezer = 1e-6;     // R14: squeezer singular values
constexpr int kRhoCols = 64;              // R10: reference vectors rho[:, j], j < 64

struct LaunchCounter { long long n = 0; };
extern thread_local LaunchCounter* g_counter;  // counts kernel launches of the current step
inline void count_launch(int k = 1) { if (g_counter) g_counter->n += k; }

// ---- kernels (each file exposes host launchers only) --------------------------------------------------------
// dgemm.cu : C[M,N] = alpha*op(A)*op(B) + beta*C on FP64 tensor cores (DMMA m8n8k4)
cudaError_t dgemm(cudaStream_t st, bool transa, bool transb, int64_t M, int64_t N, int64_t K, double alpha, const double* A,
                  int64_t lda, const double* B, int64_t ldb, double beta, double* C, int64_t ldc, int batch = 1,
                  int64_t sA = 0, int64_t sB = 0, int64_t sC = 0);

// permute.cu
cudaError_t permute(cudaStream_t st, int nd, const int64_t* dims, const int* perm, const double* in, double* out);

// elementwise.cu
cudaError_t scale_last(cudaStream_t st, double* out, const double* in, const double* vec, int64_t rows, int64_t cols,
                       int mode);  // out[r,c] = in[r,c] * f(vec[c]); mode 0: v, 1: 1/v, 2: 1/sqrt(v), 3: sqrt(v), 4: 1/sqrt(sqrt(v))...
cudaError_t scale_rows(cudaStream_t st, double* out, const double* in, const double* vec, int64_t rows, int64_t cols, int mode);
cudaError_t gather_cols(cudaStream_t st, double* out, const double* in, int64_t rows, int64_t ld_in, int64_t c0, int64_t ncols);
cudaError_t gather_rows_scaled(cudaStream_t st, double* out, const double* in, const int* idx, const double* scale, int64_t nrows,
                               int64_t cols);  // out[r,:] = scale[r]*in[idx[r],:]
cudaError_t dot(cudaStream_t st, int64_t n, const double* x, const double* y, double* result);
cudaError_t init_ising(cudaStream_t st, double beta, double h, double* phi, double* psi);
cudaError_t fill_zero(cudaStream_t st, double* p, int64_t n);

// philox.cu
cudaError_t philox_raw(cudaStream_t st, uint64_t seed, uint32_t call, uint32_t stream, uint64_t start, int64_t count, uint32_t* raw);
cudaError_t philox_gauss(cudaStream_t st, uint64_t seed, uint32_t call, uint32_t stream, uint64_t start, int64_t count, double* z);
cudaError_t philox_rho(cudaStream_t st, uint64_t seed, uint32_t call, uint32_t stream, int64_t rows, int ncols, double* out);

// jacobi.cu : rows-are-vectors storage.  eigh: G n x n symmetric (destroyed) -> lam (desc), V (columns = eigvecs)
size_t eigh_work_bytes(int n);
int eigh(cudaStream_t st, int n, double* G, double* lam, double* V, void* work, std::string* err);
size_t svd_work_bytes(int m, int n);
int svd(cudaStream_t st, int m, int n, const double* A, double* U, double* s, double* V, void* work, std::string* err);

// ---- tensors and the workspace stack ------------------------------------------------------------------------
struct Tens {
    double* p = nullptr;
    int nd = 0;
    int64_t d[8] = {0};
    int64_t size() const { int64_t s = 1; for (int i = 0; i < nd; ++i) s *= d[i]; return s; }
};

struct Arena {
    char* base = nullptr; size_t cap = 0, top = 0, peak = 0;
    double* alloc(int64_t n_doubles) {
        size_t bytes = ((size_t)(n_doubles > 0 ? n_doubles : 1) * 8 + 255) & ~(size_t)255;
        if (top + bytes > cap) return nullptr;
        double* p = (double*)(base + top); top += bytes; if (top > peak) peak = top; return p;
    }
    size_t mark() const { return top; }
    void release(size_t m) { top = m; }
};

// contract.cu : einsum-style pairwise contraction = permutes + one DGEMM.  Output allocated by the caller.
struct ContractStats { double flops = 0; int64_t permuted_bytes = 0; };
int contract(cudaStream_t st, const char* spec, const Tens& A, const Tens& B, Tens& C, Arena& scratch, ContractStats* stats,
             std::string* err);
// shape of the result of `spec` applied to A and B (no computation)
int contract_shape(const char* spec, const Tens& A, const Tens& B, Tens& C, std::string* err);

}  // namespace tatrg
