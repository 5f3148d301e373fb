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

// per-thread launch/GEMM accounting of the step being enqueued
struct Counters {
    long long launches = 0;
    double gemm_flops = 0;          // 2*M*N*K of every DGEMM launched
    long long gemm_calls = 0;
    long long permuted_bytes = 0;   // read + write bytes of every leg permutation
    long long permute_calls = 0;
    long long host_syncs = 0;       // host <-> device synchronisations inside the step (read-backs of spectra / flags)
    // optional device timing of the two kernel families (TATRG_OPT_STAGE_TIMING = 2): events bracket each launch
    bool time_kernels = false;
    std::vector<std::pair<cudaEvent_t, cudaEvent_t>> gemm_ev, perm_ev;
    std::vector<long long> perm_ev_bytes;   // algorithmic bytes of the permute timed by perm_ev[i]
    struct GemmShape { int64_t M, N, K; int batch; bool ta, tb; double frac = 1.0; };   // frac < 1: lower-triangular tiles only
    std::vector<GemmShape> gemm_shapes;   // parallel to gemm_ev (time_kernels only)
    std::vector<cudaEvent_t> ev_pool;
    size_t ev_used = 0;
    cudaEvent_t next_event();
};
extern thread_local Counters* g_counter;
inline void count_launch(int k = 1) { if (g_counter) g_counter->launches += k; }
inline void count_sync() { if (g_counter) g_counter->host_syncs += 1; }
// TATRG_OPT_VERBOSE of the handle whose step is being enqueued (debugging aid): bit 0 solver chains, bit 1 eigh, bit 2 per-DGEMM rates
extern thread_local int g_verbose;

// cudaFuncSetAttribute (the > 48 KB shared-memory opt-in) is per device: true the first time a launcher runs on the current device
inline bool first_use_on_device(unsigned long long& seen) {
    int dev = 0; cudaGetDevice(&dev);
    const unsigned long long bit = 1ull << (dev & 63);
    if (seen & bit) return false;
    seen |= bit; return true;
}

// ---- kernels (each file exposes host launchers only) --------------------------------------------------------
// dgemm.cu : C[M,N] = alpha*op(A)*op(B) + beta*C on FP64 tensor cores (DMMA m8n8k4)
cudaError_t dgemm(cudaStream_t st, bool transa, bool transb, int64_t M, int64_t N, int64_t K, double alpha, const double* A,
                  int64_t lda, const double* B, int64_t ldb, double beta, double* C, int64_t ldc, int batch = 1,
                  int64_t sA = 0, int64_t sB = 0, int64_t sC = 0);
// split-K variant for skinny outputs (Gram matrices of tall operands): partial products of K-chunks go to `part`
// (>= dgemm_splitk_doubles(M,N,K) doubles, [dev]) and are summed by a second kernel.  Falls back to dgemm when
// the output already fills the machine.  part may be null when dgemm_splitk_doubles() == 0.
int64_t dgemm_splitk_doubles(int64_t M, int64_t N, int64_t K, bool lower_only = false);
cudaError_t dgemm_splitk(cudaStream_t st, bool transa, bool transb, int64_t M, int64_t N, int64_t K, double alpha, const double* A,
                         int64_t lda, const double* B, int64_t ldb, double* C, int64_t ldc, double* part, bool lower_only = false);

// dgemm_tma.cu : the 128 x 128 x 16 tile fed by TMA (tensor maps, mbarrier ring, producer warp).  a_kc: A stored [M][K]; b_kc: B stored
// [N][K].  cudaErrorNotSupported when the operands do not meet the tensor-map alignment rules (dgemm_tma_applicable).
bool dgemm_tma_applicable(int64_t M, int64_t N, int64_t K, const double* A, int64_t lda, const double* B, int64_t ldb, int batch, int64_t sA, int64_t sB);
cudaError_t dgemm_tma(cudaStream_t st, bool a_kc, bool b_kc, int64_t M, int64_t N, int64_t K, double alpha, const double* A, int64_t lda, const double* B,
                      int64_t ldb, double beta, double* C, int64_t ldc, int batch, int64_t sA, int64_t sB, int64_t sC, bool lower_only);
extern thread_local int g_dgemm_tma;      // TATRG_OPT_DGEMM_TMA of the handle whose step is being enqueued (dgemm.cu)

// permute.cu
cudaError_t permute(cudaStream_t st, int nd, const int64_t* dims, const int* perm, const double* in, double* out);

// elementwise.cu
cudaError_t scale_last(cudaStream_t st, double* out, const double* in, const double* vec, int64_t rows, int64_t cols,
                       int mode);  // out[r,c] = in[r,c] * f(vec[c]); mode 0: v, 1: 1/v, 2: 1/sqrt(v), 3: sqrt(v), 4: v^-3/2
cudaError_t scale_rows(cudaStream_t st, double* out, const double* in, const double* vec, int64_t rows, int64_t cols, int mode);
cudaError_t lincomb3(cudaStream_t st, double* out, double a, const double* x, double b, const double* y, double c, const double* z, int64_t n);   // out = a x + b y + c z (z may be null)
cudaError_t gather_rows_scaled(cudaStream_t st, double* out, const double* in, const int* idx, const double* scale, int64_t nrows,
                               int64_t cols, int64_t ld_in);  // out[r,:] = scale[r]*in[idx[r], 0:cols]
cudaError_t gather_vec(cudaStream_t st, double* out, const double* in, const int* idx, int64_t n, int64_t stride_in, double mul);
cudaError_t dot(cudaStream_t st, int64_t n, const double* x, const double* y, double* result);
cudaError_t init_ising(cudaStream_t st, double beta, double h, double* phi, double* psi);
cudaError_t traces(cudaStream_t st, const double* A, int n, double* out);   // out[0] = Tr A, out[1] = Tr A^2
cudaError_t fill_zero(cudaStream_t st, double* p, int64_t n);
// G (k x k, row-major) = block-diagonal orthogonal gauge rotation: for every group [a,b) the block is the Q factor
// (modified Gram-Schmidt, positive diagonal of R) of C[a:b, 0:b-a], C = cfull (k x ldc).  groups: 2*ngroups ints [dev].
cudaError_t gauge_blocks(cudaStream_t st, const double* cfull, int ldc, const int* groups, int ngroups, int k, double* G);

// philox.cu
cudaError_t philox_raw(cudaStream_t st, uint64_t seed, uint32_t call, uint32_t stream, uint64_t start, int64_t count, uint32_t* raw);
cudaError_t philox_gauss(cudaStream_t st, uint64_t seed, uint32_t call, uint32_t stream, uint64_t start, int64_t count, double* z);
// element (a, b, c) of the tensor [na][nb][nc] drawn with counter (a nb + b) nc + c and stored at [b][a][c]
cudaError_t philox_gauss_swap01(cudaStream_t st, uint64_t seed, uint32_t call, uint32_t stream, int64_t na, int64_t nb, int64_t nc, double* z);
cudaError_t philox_rho(cudaStream_t st, uint64_t seed, uint32_t call, uint32_t stream, int64_t rows, int ncols, double* out);

// jacobi.cu.  All decompositions return vectors as ROWS.
//   eigh : G n x n symmetric [dev] (destroyed) -> lam[n] descending, Vt[n x n], row j = eigenvector j.  Synchronises.
//   svd_rows : X [nv x len] [dev] (nv <= 96, len <= 96 ... see jacobi.cu) -> X = Vacc^T diag(s) Ut,  Ut rows orthonormal,
//   sorted descending; s[nv], Ut[nv x len], Vacc[nv x nv] (row j = left vector j in the basis of the input rows).
size_t eigh_work_bytes(int n);
int eigh(cudaStream_t st, int n, double* G, double* lam, double* Vt, void* work, std::vector<double>* lam_host, std::string* err);
struct EighItem { int n; double* G; double* lam; double* Vt; std::vector<double>* lam_host; };
size_t eigh_batched_work_bytes(int nmax, int count);
int eigh_batched(cudaStream_t st, int count, const EighItem* items, void* work, std::string* err);
size_t svd_rows_work_bytes(int nv, int len);
int svd_rows(cudaStream_t st, int nv, int len, const double* X, double* s, double* Ut, double* Vacc, void* work,
             std::vector<double>* s_host, std::string* err);

// cholesky.cu : blocked Cholesky (64-wide panels: one-CTA diagonal factor + inverse, DGEMM panel / trailing updates) and
// the triangular solve Q = X L^-T.  All asynchronous on st.
cudaError_t symmetrize(cudaStream_t st, int n, double* A);                      // A = (A + A^T) / 2 in place
cudaError_t mirror_lower(cudaStream_t st, int n, double* A);                    // A[i][j] = A[j][i] for i < j
size_t cholesky_work_doubles(int n);
// reset_info = false accumulates the flags of several factorisations that share `work` (the caller clears them once)
cudaError_t cholesky(cudaStream_t st, int n, double* A, int64_t lda, double* L, int64_t ldl, double shift, double guard_rel, double* work,
                     bool reset_info = true);
const int* cholesky_info(const double* work, int n);                            // [dev] bit 0: a pivot was raised to the guard, bit 1: non-finite
cudaError_t trsm_right_lt(cudaStream_t st, int64_t m, int n, double* X, int64_t ldx, double* Q, int64_t ldq, const double* L, int64_t ldl,
                          const double* work);
size_t tri_inverse_scratch_doubles(int n);
cudaError_t tri_inverse(cudaStream_t st, int n, const double* L, int64_t ldl, const double* work, double* X, int64_t ldx, double* T);
const double* cholesky_d0(const double* work, int n);                           // [dev] the n original diagonal entries
cudaError_t extract_diag(cudaStream_t st, int n, const double* A, int64_t lda, double* d);

// pchol.cu : truncated Cholesky with diagonal pivoting, G = L L^T + S with tr S <= tol_rel tr G (one cooperative kernel)
size_t pchol_work_doubles(int n);
cudaError_t pchol(cudaStream_t st, int n, const double* G, double* L, int64_t ldl, double tol_rel, double* work);
const double* pchol_info(const double* work);                                   // [dev] rank, residual trace, tr G, first pivot

// ---- tensors and the workspace pool -------------------------------------------------------------------------
struct Tens {
    double* p = nullptr;
    int nd = 0;
    int64_t d[8] = {0};
    int64_t size() const { int64_t s = 1; for (int i = 0; i < nd; ++i) s *= d[i]; return s; }
};

// First-fit free-list allocator over the caller's workspace.  Host bookkeeping only: all work is enqueued on one
// stream, so a block may be reused as soon as the kernels that read it have been *enqueued*.
class Pool {
public:
    void reset(void* base, size_t bytes);
    double* alloc(int64_t n_doubles);  // nullptr when full
    void free(const void* p);
    size_t peak() const { return peak_; }
    size_t in_use() const { return used_; }
    size_t capacity() const { return cap_; }
private:
    char* base_ = nullptr; size_t cap_ = 0, used_ = 0, peak_ = 0, high_ = 0;
    std::map<size_t, size_t> free_;   // offset -> size
    std::map<size_t, size_t> live_;   // offset -> size
};

// contract.cu : einsum-style pairwise contraction = (permutes only where the layout forces them) + one DGEMM.
// Single-letter legs; an UPPERCASE letter is a batch leg (may be missing from one operand: broadcast).
// C.p must point to room for the result; C.nd / C.d are filled in.
int contract(cudaStream_t st, const char* spec, const Tens& A, const Tens& B, Tens& C, Pool& pool, std::string* err);
int contract_shape(const char* spec, const Tens& A, const Tens& B, Tens& C, std::string* err);

}  // namespace tatrg
