// pchol.cu -- Cholesky factorisation with complete (diagonal) pivoting, truncated: the rank-revealing first half of the
// QR pre-reduction (Eq. A.2-A.3 :345-348) when the operand is numerically rank-deficient (R14 of DESIGN.md section 3: the
// unsaturated first steps and every step after the flow has left criticality).
//
//   G (n x n, symmetric positive semi-definite up to rounding)  =  L L^T + S,   L n x r in the ORIGINAL row order (column j
//   belongs to the j-th pivot), S the positive semi-definite Schur complement that is dropped, ||S||_2 <= tr S <= tol_rel tr G.
//
// Why: the numerical rank decision of R14 needs the eigenvalues of G above 1e-12 lam_max.  The two-sided Jacobi iteration
// on G itself takes 24-32 sweeps at n = 1024 when G is strongly graded; on the r x r matrix L^T L -- one step of the pivoted
// LR iteration, same non-zero eigenvalues, already diagonally dominant, r well below n -- it takes about 8
// (Veselic / Hari preconditioning), and the eigenvectors of G follow as L V lam^-1/2.
//
// One cooperative kernel per matrix.  The Schur complement lives in the shared memory of the grid, a band of rows per CTA
// (16 rows x 1024 doubles = 128 KB per CTA on 64 CTAs for n = 1024), and stays exactly symmetric because entry (i,c) and
// entry (c,i) receive the same products.  One grid barrier per pivot: after its update every CTA publishes its best
// remaining diagonal entry TOGETHER WITH that whole row; after the barrier every CTA picks the same winner (largest value,
// lowest row index on ties), reads the winner's row -- by symmetry the pivot column -- and updates its band.  Bands that do
// not fit in shared memory (n > ~1400) live in global memory (L2) instead; same code.
#include "internal.h"
#include <cooperative_groups.h>
#include <algorithm>

namespace cg = cooperative_groups;

namespace tatrg {
namespace {

constexpr int kThreads = 512;

struct PcholArgs {
    const double* G;      // n x n row-major
    double* L;            // n x ldl, columns 0..rank-1 written
    int64_t ldl;
    double* band_glob;    // n x n scratch when the bands do not fit in shared memory, else null
    double* cand;         // [2][nctas][n + 2]: value, row index, then the row; [2][nctas][n + 2] more whose first entries hold the traces
    double* info;         // [4]: rank, residual trace, initial trace, largest pivot
    int n, rows_per_cta;
    double tol_rel;
};

__global__ void __launch_bounds__(kThreads, 1) pchol_kernel(PcholArgs a) {
    extern __shared__ double sm[];
    cg::grid_group grid = cg::this_grid();
    const int n = a.n, tid = threadIdx.x, nctas = gridDim.x, cta = blockIdx.x;
    const int r0 = cta * a.rows_per_cta, rows = max(0, min(a.rows_per_cta, n - r0));
    double* lrow = sm;                                  // n: the scaled pivot column l_c
    double* diag = lrow + n;                            // rows_per_cta (+ pad): remaining diagonal of the band, -1 for rows that were pivots
    double* red = diag + ((a.rows_per_cta + 1) & ~1);   // 2 * 32 scratch for the reductions
    unsigned char* celim = (unsigned char*)(red + 64);  // n flags: column already a pivot
    double* band = a.band_glob ? a.band_glob + (int64_t)r0 * n : (double*)(celim + ((n + 7) & ~7));
    const int64_t cstride = (int64_t)n + 2;

    for (int64_t e = tid; e < (int64_t)rows * n; e += kThreads) band[e] = a.G[(int64_t)r0 * n + e];
    for (int c = tid; c < n; c += kThreads) celim[c] = 0;
    __syncthreads();
    for (int i = tid; i < rows; i += kThreads) diag[i] = band[(int64_t)i * n + r0 + i];
    __syncthreads();

    double trace0 = 0.0;
    int rank = 0;
    for (int j = 0; j <= n; ++j) {
        // ---- publish the band's best remaining diagonal entry, its row, and the band's remaining trace ----
        double* mine = a.cand + ((int64_t)(j & 1) * nctas + cta) * cstride;
        if (tid < 32) {
            double best = -1.0, tr = 0.0; int bi = -1;
            for (int i = tid; i < rows; i += 32) {
                const double d = diag[i];
                if (d > 0.0) tr += d;
                if (d > best) { best = d; bi = i; }
            }
            for (int o = 16; o > 0; o >>= 1) {
                const double ob = __shfl_down_sync(0xffffffffu, best, o); const int oi = __shfl_down_sync(0xffffffffu, bi, o);
                tr += __shfl_down_sync(0xffffffffu, tr, o);
                if (ob > best || (ob == best && oi >= 0 && (bi < 0 || oi < bi))) { best = ob; bi = oi; }
            }
            if (tid == 0) { red[0] = best; red[1] = (double)bi; red[2] = tr; }
        }
        __syncthreads();
        const int bi = (int)red[1];
        if (tid == 0) { mine[0] = bi >= 0 ? red[0] : -1.0; mine[1] = (double)(bi >= 0 ? r0 + bi : -1); }
        if (bi >= 0) for (int c = tid; c < n; c += kThreads) mine[2 + c] = band[(int64_t)bi * n + c];
        if (tid == 1) a.cand[((int64_t)(2 + (j & 1)) * nctas + cta) * cstride] = red[2];      // traces live behind the two row buffers
        grid.sync();
        // ---- every CTA takes the same decision ----
        if (tid < 32) {
            double best = -1.0, tr = 0.0; int bc = -1, brow = -1;
            for (int c = tid; c < nctas; c += 32) {
                const double* o = a.cand + ((int64_t)(j & 1) * nctas + c) * cstride;
                const double v = __ldcg(o); const int row = (int)__ldcg(o + 1);
                tr += __ldcg(a.cand + ((int64_t)(2 + (j & 1)) * nctas + c) * cstride);
                if (row >= 0 && (v > best || (v == best && row < brow))) { best = v; bc = c; brow = row; }
            }
            // fixed-order tree: every CTA adds the same numbers in the same order, hence takes the same decision
            for (int o = 16; o > 0; o >>= 1) {
                const double ob = __shfl_down_sync(0xffffffffu, best, o); const int oc = __shfl_down_sync(0xffffffffu, bc, o);
                const int orow = __shfl_down_sync(0xffffffffu, brow, o);
                tr += __shfl_down_sync(0xffffffffu, tr, o);
                if (orow >= 0 && (ob > best || (ob == best && (brow < 0 || orow < brow)))) { best = ob; bc = oc; brow = orow; }
            }
            if (tid == 0) { red[0] = best; red[1] = (double)bc; red[2] = (double)brow; red[3] = tr; }
        }
        __syncthreads();
        const double piv = red[0], trem = red[3];
        const int wc = (int)red[1], k = (int)red[2];
        if (j == 0) trace0 = trem;
        if (j == n || wc < 0 || !(piv > 0.0) || !(trem > a.tol_rel * trace0)) {
            if (cta == 0 && tid == 0) { a.info[0] = (double)rank; a.info[1] = trem; a.info[2] = trace0; }
            break;
        }
        const double* win = a.cand + ((int64_t)(j & 1) * nctas + wc) * cstride + 2;
        const double scale = rsqrt(piv);
        __syncthreads();                                 // red[] is rewritten at the top of the next round
        for (int c = tid; c < n; c += kThreads) lrow[c] = celim[c] ? 0.0 : __ldcg(win + c) * scale;
        __syncthreads();
        // column j of L for the band's rows, then the rank-1 update of the band (rows that were pivots are left alone)
        for (int i = tid; i < rows; i += kThreads) a.L[(int64_t)(r0 + i) * a.ldl + j] = lrow[r0 + i];
        for (int c = tid; c < n; c += kThreads) {
            const double lc = lrow[c];
            for (int i = 0; i < rows; ++i)
                if (!celim[r0 + i]) band[(int64_t)i * n + c] = fma(-lrow[r0 + i], lc, band[(int64_t)i * n + c]);
        }
        __syncthreads();
        if (tid == 0) { celim[k] = 1; if (cta == 0 && j == 0) a.info[3] = piv; }
        __syncthreads();
        for (int i = tid; i < rows; i += kThreads) diag[i] = celim[r0 + i] ? -1.0 : band[(int64_t)i * n + r0 + i];
        __syncthreads();
        ++rank;
    }
}

int g_sms[64] = {0};
int sm_count() {
    int dev = 0; cudaGetDevice(&dev);
    int& s = g_sms[dev & 63];
    if (!s) cudaDeviceGetAttribute(&s, cudaDevAttrMultiProcessorCount, dev);
    return s;
}
// CTAs per matrix: two factorisations run side by side (B and C of Eq. A.2-A.3), each on at most 64 SMs
void geometry(int n, int& nctas, int& rows, size_t& smem, bool& in_smem) {
    nctas = std::min(64, std::max(1, (sm_count() - 4) / 2));
    nctas = std::min(nctas, (n + 3) / 4);
    rows = (n + nctas - 1) / nctas;
    nctas = (n + rows - 1) / rows;
    const size_t fixed = 8 * ((size_t)n + ((rows + 1) & ~1) + 64) + ((n + 7) & ~7);
    in_smem = fixed + 8 * (size_t)rows * n <= 220 * 1024;
    smem = fixed + (in_smem ? 8 * (size_t)rows * n : 0);
}
}  // namespace

size_t pchol_work_doubles(int n) {
    int nctas, rows; size_t smem; bool in_smem;
    geometry(n, nctas, rows, smem, in_smem);
    return 4 * (size_t)nctas * (n + 2) + 8 + (in_smem ? 0 : (size_t)n * n);
}

// G [dev] n x n (preserved) -> L [dev] n x ldl (columns 0..rank-1), info [dev, 4 doubles inside work]: rank, residual trace,
// trace of G, first pivot.  Asynchronous on st; pchol_info(work) points at the four doubles.
cudaError_t pchol(cudaStream_t st, int n, const double* G, double* L, int64_t ldl, double tol_rel, double* work) {
    static unsigned long long configured = 0;
    int nctas, rows; size_t smem; bool in_smem;
    geometry(n, nctas, rows, smem, in_smem);
    if (first_use_on_device(configured)) {
        cudaError_t e = cudaFuncSetAttribute(pchol_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 220 * 1024);
        if (e != cudaSuccess) return e;
    }
    PcholArgs a;
    a.G = G; a.L = L; a.ldl = ldl; a.n = n; a.rows_per_cta = rows; a.tol_rel = tol_rel;
    a.info = work; a.cand = work + 8;
    a.band_glob = in_smem ? nullptr : work + 8 + 4 * (size_t)nctas * (n + 2);
    void* params[] = {&a};
    count_launch();
    return cudaLaunchCooperativeKernel((const void*)pchol_kernel, dim3(nctas), dim3(kThreads), params, smem, st);
}
const double* pchol_info(const double* work) { return work; }

}  // namespace tatrg
