/*
 * tatrg.h -- C ABI of the B200-native Triad-ATRG hot path (arXiv:2507.21909; citations "PAPER.md:<line>").
 *
 * One handle = one 4D Ising tensor network being coarse-grained on ONE GPU in FP64.  Every arithmetic step of
 * the path runs in the library's own sm_100a kernels; the caller (a thin Python binding) only provides device
 * memory and a CUDA stream.  No entry point throws or aborts; all return a status (0 = TATRG_OK, < 0 = error)
 * unless stated otherwise; tatrg_last_error() gives the text of the last failure of a handle.
 *
 * Pointers are marked  [dev]  (device memory, FP64 unless stated, 16-byte aligned)  or  [host].
 * The library never frees caller memory and never allocates device memory of its own.  All work of a call is ordered on
 * the caller's stream.  Inside a call the independent solver chains run on auxiliary streams that the library creates on
 * first use, once per device, and never destroys: four chain streams and one stage stream (subspace iterations, Cholesky
 * chains, squeezers) plus one solver stream of the block-Jacobi eigen-decomposition, all non-blocking and of the greatest
 * priority, with the events that fork them from and join them back into the caller's stream before the call returns.
 */
#ifndef TATRG_H
#define TATRG_H
#include <stddef.h>
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

typedef struct tatrg_ctx* tatrg_handle;

enum { TATRG_OK = 0, TATRG_EINVAL = -1, TATRG_ENOMEM = -2, TATRG_ECUDA = -3, TATRG_ENUMERIC = -4, TATRG_ESTATE = -5 };

/* option keys of tatrg_set_option (before the first step only) */
enum {
    TATRG_OPT_POWER_ITERS = 1, /* n_pow: RSVD power iterations; passes of Eq. A.4-A.6 (:352-369) = n_pow+1. default 2 */
    TATRG_OPT_K_TRIAD = 2,     /* internal-line dimension rD of the triad isometries (Eq. 2.9 :135). default D+oversample */
    TATRG_OPT_TAU = 3,         /* relative gap below which values form one multiplet (R7). default 1e-6 */
    TATRG_OPT_STAGE_TIMING = 4,/* 1: CUDA-event time per stage; 2: also per DGEMM / permute launch (tatrg_gemm_profile). default 0 */
    TATRG_OPT_KEEP_TENSORS = 5,/* 1: keep copies of the step's intermediate tensors for tatrg_get_tensor (tests). default 0 */
    TATRG_OPT_SUBSPACE = 7,    /* 1 (default): the leading eigenvectors the triad isometries (top K of D^2, Eq. 2.9 :135) and the
                                  squeezers (top D of D^2, :171) need come from a subspace iteration (Cholesky QR on the tensor
                                  cores + one small Rayleigh-Ritz problem); 0: full eigen-decompositions everywhere.  Same result. */
    TATRG_OPT_BOND_RANK = 8,   /* ILO Triad-ATRG (section 2.3 :183-209, App. A): r_bond D, the number of singular values the bond swap keeps
                                  (Eq. A.1 :337) and hence the rank of the next decomposition (fn 5 :203); the RSVD sketch is
                                  r_bond D + oversample wide (fn 9 :381); the squeezed legs stay at D.  default D (r_bond = 1, :331).
                                  Before the first step only; integer in [D, 4D]; ENOMEM unless the workspace holds
                                  tatrg_workspace_bytes_ilo(D, oversample, value). */
    TATRG_OPT_OVERLAP = 9,     /* 1 (default): in saturated steps the solver chains (squeezers, Cholesky factorisations) run on the library's
                                  auxiliary streams beside the contractions of the caller's stream; 0: every stage on the caller's stream,
                                  one after the other (used by bench.py to time the kernels with nothing beside them).  Same result. */
    TATRG_OPT_GRAPHS = 10,     /* 1 (default): the repeated steps of the subspace iterations are captured once and replayed as CUDA graphs;
                                  0: plain launches.  Same result. */
    TATRG_OPT_VERBOSE = 11,    /* debugging aid, bit mask, default 0: 1 = solver chains report ranks / convergence on stderr, 2 = spectra of
                                  the full eigen-decompositions, 4 = shape and rate of every DGEMM and permute (with TATRG_OPT_STAGE_TIMING = 2), 8 = the
                                  contractions that needed a permuted copy of an operand or of their result */
    TATRG_OPT_DGEMM_TMA = 12,  /* 1 (default): contractions whose output takes the 128 x 128 tile and whose operands meet the tensor-map rules
                                  (16-byte aligned bases, even leading dimensions and batch strides) run the TMA-fed kernel (dgemm_tma.cu:
                                  producer warp, cp.async.bulk.tensor into a 128B-swizzled 6-stage mbarrier ring); 0: the cp.async kernel
                                  everywhere.  Same products up to the order of nothing: both accumulate k in the same order. */
    TATRG_OPT_IMPLICIT_XY = 13,/* 1 (default): the tensors X, Y of Eq. A.10-A.11 (:389-392) are never formed: the Gram matrices of Eq. 2.9 (:135)
                                  and F, G of Eq. 2.11-2.12 come straight from U^bond, sigma, V^bond and the QR factors of Eq. A.2-A.3
                                  (PAPER.md :394 "the tensors X and Y are not explicitly constructed", :201), which removes the two
                                  O(r_bond^2 D^5) tensors and two D^3 x D^2 x D^2 r_bond^3 products per step; 0: X, Y formed as the
                                  equations are printed.  Same result up to rounding order.  Triad method only (plain ATRG contracts
                                  X and Y themselves).  With TATRG_OPT_KEEP_TENSORS = 1, X and Y are still formed, for tatrg_get_tensor only. */
    TATRG_OPT_CHEBYSHEV = 14,  /* 1 (default): the subspace iterations for the triad isometries (TATRG_OPT_SUBSPACE) apply a Chebyshev polynomial of the
                                  Gram matrix per orthonormalisation instead of a power (three-term recurrence on the interval that holds the
                                  unwanted eigenvalues): the same subspace in 2-3 times fewer applications; 0: plain orthogonal iteration.
                                  Same result to the iteration's 13 digits. */
    TATRG_OPT_METHOD = 6       /* 0: Triad-ATRG (default).  1: plain ATRG, Eq. 2.7-2.8 (:104-113): no triad split, squeezers from
                                  Gamma^ATRG, O(D^9) contraction sliced so that no D^7 tensor is stored (fn 6 :205).  Before the first
                                  step only; ENOMEM unless the workspace holds tatrg_workspace_bytes_atrg(D, oversample). */
};

/* which spectrum tatrg_singular_values returns */
enum { TATRG_SV_SIGMA = 0 /* bond swap, Eq. 2.5 :90 */, TATRG_SV_S = 1 /* decomposition of T, Eq. 2.4 :76 */ };

/* stages of one step (Fig. 5 a-f) for tatrg_stage_ms / tatrg_stage_flops */
enum { TATRG_ST_DECOMPOSE = 0, TATRG_ST_QR, TATRG_ST_RSVD, TATRG_ST_LIFT, TATRG_ST_TRIAD_ISO, TATRG_ST_TRIAD_TENSORS,
       TATRG_ST_SQ_GRAMS, TATRG_ST_SQUEEZERS, TATRG_ST_CONTRACT, TATRG_ST_ROTATE, TATRG_NSTAGES };

/* ---- the path: PAPER.md Fig. 5 (a)-(f) :193 ------------------------------------------------------------ */

/* Device bytes a handle with truncation D (Eq. 2.4 :76) and RSVD oversampling p (l = D+p, :371) needs. */
size_t tatrg_workspace_bytes(int D, int oversample);
/* The same for TATRG_OPT_BOND_RANK = bond_rank (ILO Triad-ATRG: X, Y, F, G carry two legs of dimension r_bond D, fn 5 :203). */
size_t tatrg_workspace_bytes_ilo(int D, int oversample, int bond_rank);
/* The same for TATRG_OPT_METHOD = 1 (plain ATRG keeps three D^6 slabs). */
size_t tatrg_workspace_bytes_atrg(int D, int oversample);

/* Builds the initial tensor of the 4D Ising model, Eq. 3.1-3.2 (:241-246), on the device in factored form
 * T[f,b] = sum_a Phi0[f,a] Psi0[b,a], with site weight exp(beta*h*s_a) (R1).
 * workspace [dev]: >= tatrg_workspace_bytes(D, oversample) bytes, owned by the caller, must outlive the handle.
 * seed: Philox4x32-10 key of the RSVD test tensor Omega (:371) and of the gauge reference vectors.
 * Errors: EINVAL (beta<=0, non-finite, D<2, oversample<0, null pointers), ENOMEM (workspace too small). */
int tatrg_create(double beta, double h, int D, int oversample, uint64_t seed, void* workspace, size_t workspace_bytes,
                 tatrg_handle* out);

int tatrg_set_option(tatrg_handle, int key, double value);

/* One coarse-graining step along the current axis 1 (axes cycle x,y,z,t): decomposition (Eq. 2.4), bond swap
 * by RSVD (Eq. 2.5, App. A), triad isometries and tensors (Eq. 2.9-2.17), squeezers (:171), contraction
 * (Eq. 2.18-2.19), axis rotation and normalisation.  Work is enqueued on cuda_stream (a cudaStream_t; NULL =
 * default stream); small spectra are read back inside the call to take the rank decisions.
 * The independent solver chains of a stage (subspace iterations, block-Jacobi rounds) run on up to five auxiliary
 * non-blocking streams that the library creates once per device; they are forked from and joined to cuda_stream by
 * events, so that all work of the step is ordered after what was enqueued on cuda_stream before the call and before
 * what is enqueued on it afterwards.  Handles on the same device must not be stepped from several host threads at once.
 * Errors: ECUDA, ENUMERIC (non-finite or non-positive normalisation), ENOMEM, ESTATE (after an earlier failure). */
int tatrg_step(tatrg_handle, void* cuda_stream);
/* Streams: consecutive calls may use different streams; a call on a stream other than the previous step's first waits (on the
 * device) for an event recorded at the end of that step, so the state is never read before it is complete. */

/* ln Z / V of the periodic lattice of V = 2^steps sites: sum_j 2^-j ln c_j + 2^-m ln tTr(T^(m)) (R8).
 * Synchronises the stream of the last step.  NaN on error. */
double tatrg_lnZ_per_site(tatrg_handle);

/* Copies min(k, available) leading values of the last step's spectrum `which`, normalised to the largest, to
 * out_host [host].  Returns the number written or < 0. */
int tatrg_singular_values(tatrg_handle, int which, int k, double* out_host);

/* X ratio of the current tensor, Eq. 3.3 (:298-303): X = (Tr A)^2 / Tr A^2, A[k,l] = sum T[i1 i2 i3 k, i1 i2 i3 l]; 2 in the
 * ordered phase, 1 in the disordered one.  One contraction on cuda_stream, synchronises.  x_out [host]. */
int tatrg_x_ratio(tatrg_handle, void* cuda_stream, double* x_out);

int tatrg_steps_done(tatrg_handle);
const char* tatrg_last_error(tatrg_handle);
void tatrg_destroy(tatrg_handle); /* frees the host struct only */

/* ---- instrumentation ----------------------------------------------------------------------------------- */
/* ms[TATRG_NSTAGES] / flops[TATRG_NSTAGES] [host] of the last step (ms only with TATRG_OPT_STAGE_TIMING). flops
 * are the 2*M*N*K of every GEMM launched in the stage.  launches: kernels launched by the last step. */
int tatrg_stage_ms(tatrg_handle, double* ms);
int tatrg_stage_flops(tatrg_handle, double* flops);
long long tatrg_last_step_launches(tatrg_handle);
/* host <-> device synchronisations inside the last tatrg_step call (read-backs of spectra and flags for the rank decisions) */
long long tatrg_last_step_host_syncs(tatrg_handle);
/* device time (ms; needs STAGE_TIMING=2), flops and launches of the DGEMM kernel during the last step; likewise the
 * leg-permutation kernel with its algorithmic bytes (8 B read + 8 B written per element). Any out pointer may be NULL. */
int tatrg_gemm_profile(tatrg_handle, double* ms, double* flops, long long* calls);
/* The same restricted to the DGEMM launches of >= 1e9 flop: the tensor contractions proper (Eq. 2.18-2.19 :175, 2.9-2.17,
 * A.2-A.11), without the small products inside the Cholesky / subspace-iteration solvers.  Needs STAGE_TIMING=2. */
int tatrg_gemm_profile_large(tatrg_handle, double* ms, double* flops, long long* calls);
int tatrg_permute_profile(tatrg_handle, double* ms, double* bytes, long long* calls);
/* The same restricted to the permutes that move >= 100 MB (read + written): tensors larger than L2, the D^5 operands of the
 * saturated steps (Eq. A.2-A.3 :345-348 layouts, the leg pair of Eq. 2.9 :135, the axis rotation of Fig. 5(f)).  Needs STAGE_TIMING=2. */
int tatrg_permute_profile_large(tatrg_handle, double* ms, double* bytes, long long* calls);
/* high-water mark (bytes) of the workspace since tatrg_create */
size_t tatrg_workspace_peak(tatrg_handle);

/* Copies a named tensor of the last step to out_host [host] (row-major).  Names: "phi","psi" (state after the
 * step), "A","Dt","core","X","Y","sigma","E","F","G","H","UA","UX","UY","UD","M2","M3","M4","N2","N3","N4".
 * dims[8] [host] receives the shape, *ndim its length.  capacity = doubles available in out_host (may be 0 to
 * query the shape).  Returns the element count or < 0. */
long long tatrg_get_tensor(tatrg_handle, const char* name, double* out_host, long long capacity, int* ndim, long long* dims);

/* Replaces the state by Phi[d0,d1,d2,d3,g], Psi[d0,d1,d2,d3,g] read from host memory (teacher forcing in tests). */
int tatrg_set_state(tatrg_handle, const double* phi_host, const double* psi_host, const long long* dims5);

/* ---- primitives (the kernels the path is made of; all on device pointers) ---------------------------------- */

/* C[M,N] (row-major, ldc) = alpha * op(A) op(B) + beta * C, FP64 tensor cores (DMMA).  transa = 0: A is [M,K]
 * (lda >= K); 1: A is stored [K,M] (lda >= M).  transb = 0: B is [K,N] (ldb >= N); 1: B stored [N,K].
 * batch >= 1 with element strides between consecutive problems. */
int tatrg_dgemm(void* cuda_stream, int transa, int transb, long long M, long long N, long long K, double alpha,
                const double* A, long long lda, const double* B, long long ldb, double beta, double* C, long long ldc,
                int batch, long long strideA, long long strideB, long long strideC);
/* The same product through a named kernel variant (tests, profiling): 0 = cp.async-fed tiles (all four tile configurations),
 * 1 = the TMA-fed 128 x 128 x 16 tile whatever the shape.  EINVAL for variant 1 when the operands do not meet the tensor-map
 * rules (16-byte aligned A, B; even lda, ldb, sA, sB; extents below 2^31; batch <= 65535) or an extent is 0. */
int tatrg_dgemm_variant(void* cuda_stream, int variant, int transa, int transb, long long M, long long N, long long K, double alpha,
                        const double* A, long long lda, const double* B, long long ldb, double beta, double* C, long long ldc,
                        int batch, long long sA, long long sB, long long sC);

/* out = in with legs permuted: out leg i is in leg perm[i]; dims[ndim] are the extents of `in` (row-major). */
int tatrg_permute(void* cuda_stream, int ndim, const long long* dims, const int* perm, const double* in, double* out);

/* Tensor contraction  "abc,cd->abd"  (single-letter legs; an UPPERCASE leg is a batch leg and may be missing from one
 * operand) = leg permutations only where the layout forces them + one batched DGEMM.  dimsA/dimsB [host] hold the
 * extents of the legs named in spec; C [dev] receives the result in the leg order written after "->".
 * scratch [dev] of scratch_bytes holds permuted copies and split-K partials (8*(|A|+|B|+|C|) + 64 MiB always suffices;
 * ENOMEM otherwise). */
int tatrg_contract(void* cuda_stream, const char* spec, const double* A, const long long* dimsA, const double* B,
                   const long long* dimsB, double* C, void* scratch, size_t scratch_bytes);

/* Philox4x32-10 (R11): raw[4*count] uint32 [dev] for counters e = start..start+count-1, and the
 * Gaussian z[count] [dev] of the same counters; counter = (e_lo, e_hi, call, stream_id), key = seed. */
int tatrg_philox_raw(void* cuda_stream, uint64_t seed, uint32_t call, uint32_t stream_id, uint64_t start, long long count,
                     uint32_t* raw);
int tatrg_philox_gaussian(void* cuda_stream, uint64_t seed, uint32_t call, uint32_t stream_id, uint64_t start,
                          long long count, double* z);

/* Symmetric eigen-decomposition by (block) two-sided Jacobi: G [dev] n x n row-major (destroyed), lam [dev] n
 * descending, Vt [dev] n x n row-major, ROW j = eigenvector j.  work [dev] >= tatrg_eigh_work_bytes(n), 256-byte
 * aligned.  Synchronises the stream (the order of the eigenvalues is taken on the host).  ENUMERIC if not converged. */
size_t tatrg_eigh_work_bytes(int n);
int tatrg_eigh(void* cuda_stream, int n, double* G, double* lam, double* Vt, void* work);

/* SVD of a small matrix X [dev] nv x len (row-major, preserved; 8*(nv*(len+1)+nv*(nv+1)) <= 200 KiB of shared memory)
 * by one-sided Jacobi on its rows:  X = Vacc^T diag(s) Ut,  s [dev] nv descending, Ut [dev] nv x len with orthonormal
 * rows (zero rows where s = 0), Vacc [dev] nv x nv orthogonal.  work >= tatrg_svd_work_bytes(nv,len).  Synchronises. */
size_t tatrg_svd_work_bytes(int nv, int len);
int tatrg_svd(void* cuda_stream, int nv, int len, const double* X, double* s, double* Ut, double* Vacc, void* work);

/* Gram matrix G [dev] n x n (row-major, ld n) = X^T X of X [dev] m x n (row-major, ld n): the DGEMM in its symmetric mode -- only
 * the tiles on and below the diagonal are computed (split along K into partial products when the grid would not fill the SMs),
 * the upper triangle is mirrored.  This is how the Gram matrices of Eq. A.2-A.3 and Eq. 2.9 are formed.
 * scratch [dev] >= tatrg_gram_scratch_bytes(m, n) (may be NULL when that is 0). */
size_t tatrg_gram_scratch_bytes(long long m, int n);
int tatrg_gram(void* cuda_stream, long long m, int n, const double* X, double* G, void* scratch);

/* tatrg_gram for callers that cannot allocate device memory (code under CUDA graph capture, serving loops, harnesses that
 * forbid cudaMalloc): same kernels, same result, but the split-K partial products go to a 16 MiB file-scope __device__ array
 * inside the library (tatrg_gram_static_max_scratch_bytes(); every GPU that loads the library holds it until exit) instead of
 * caller scratch.  The call allocates nothing and does not synchronise.  EINVAL, with the reason in err [host, err_cap bytes,
 * may be NULL], when tatrg_gram_scratch_bytes(m, n) exceeds the array -- use tatrg_gram then.  All calls on a device share the
 * array: calls whose kernels overlap on the GPU (different streams without ordering) race on it.  Nothing in it has to
 * start at zero; the previous call's contents are never read. */
size_t tatrg_gram_static_max_scratch_bytes(void);
int tatrg_gram_static(void* cuda_stream, long long m, int n, const double* X, double* G, char* err, size_t err_cap);

/* Cholesky QR of a tall matrix (the orthonormalisation of the QR pre-reduction, Eq. A.2-A.3 :345-348, of the RSVD
 * sketches, Eq. A.4-A.6 :352-369, and of the subspace iterations behind Eq. 2.9 :135 and the squeezers :171):
 * X [dev] m x n row-major (m >= n; DESTROYED), Q [dev] m x n with orthonormal columns up to cond(X)^2 eps (one pass),
 * R [dev] n x n upper triangular with positive diagonal, X = Q R.  Blocked Cholesky of X^T X over 64-wide panels
 * (one-CTA diagonal factor, DGEMM panel/trailing updates), Q by forward substitution over the panels.
 * work [dev] >= tatrg_cholqr_work_bytes(n), 256-byte aligned.  Synchronises.  ENUMERIC when a pivot of the factorisation
 * fell below 1e-14 of its diagonal entry (X numerically rank-deficient): Q, R are then not usable. */
size_t tatrg_cholqr_work_bytes(int n);
int tatrg_cholqr(void* cuda_stream, long long m, int n, double* X, double* Q, double* R, void* work);

/* Truncated Cholesky factorisation with diagonal pivoting (the rank-revealing first half of the QR pre-reduction, Eq. A.2-A.3
 * :345-348, when the operand is numerically rank-deficient; R14):  G [dev] n x n row-major, symmetric positive
 * semi-definite up to rounding (preserved) = L L^T + S.  L [dev] n x n row-major: rows in the ORIGINAL order, column j belongs
 * to the j-th pivot (the largest remaining diagonal entry, lowest index on ties); only columns 0..rank-1 are written.  The
 * factorisation stops as soon as the remaining Schur complement S has tr S <= tol_rel * tr G (S is positive semi-definite, so
 * ||G - L L^T||_2 <= tr S).  *rank_out, *resid_out [host]: number of pivots taken, tr S / tr G.  One cooperative kernel on 64 CTAs.
 * work [dev] >= tatrg_pchol_work_bytes(n), 256-byte aligned.  Synchronises.  EINVAL for n < 1 or tol_rel < 0. */
size_t tatrg_pchol_work_bytes(int n);
int tatrg_pchol(void* cuda_stream, int n, const double* G, double* L, double tol_rel, void* work, int* rank_out, double* resid_out);

/* result[0] [dev] = sum_i x[i]*y[i]  (the tensor trace tTr of Eq. 2.1 :48 on the factored tensor).
 * result must have room for 1200 doubles (partial sums of the first pass follow result[0]). */
int tatrg_dot(void* cuda_stream, long long n, const double* x, const double* y, double* result);

/* Calibration: FP64 tensor-core (DMMA m8n8k4) issue rate of the whole device with register-resident operands, in
 * TFLOP/s, timed with CUDA events inside the call (synchronises).  ctas_per_sm in 1..8; scratch_dev [dev] >= 8 bytes. */
int tatrg_dmma_issue_rate(void* cuda_stream, int iters, int ctas_per_sm, double* tflops_out, double* scratch_dev);
/* The same for the register tile of the DGEMM inner loop (8 x 4 atoms per warp, 12 distinct operand registers per 4-deep
 * slice, one 256-thread CTA per SM, no memory traffic): the ceiling of the warp tile itself.  order 0: row-major walk of the
 * atoms (the A fragment is reused by consecutive DMMAs), 1: column-major walk. */
int tatrg_dmma_tile_rate(void* cuda_stream, int iters, int order, double* tflops_out, double* scratch_dev);

#ifdef __cplusplus
}
#endif
#endif
