// capi.cu -- the C ABI of include/tatrg.h.  No exception leaves this file; every entry point validates its arguments.
#include "step.h"
#include <cstring>
#include <new>

using namespace tatrg;

namespace {
constexpr int kTraceDoubles = 1 + 148 * 8 + 7;
int64_t workspace_doubles(int D, int p) {
    const double d = D, k = D + p;
    double w = 16 * std::pow(d, 5) + 2 * d * d * d * k * k + 6 * d * d * d * d * k + 4 * k * k * k * k + 16 * d * d * d * d + 64 * k * k + (1 << 20);
    return (int64_t)w;
}
bool finite_pos(double x) { return std::isfinite(x) && x > 0; }
}  // namespace

extern "C" {

size_t tatrg_workspace_bytes(int D, int oversample) {
    if (D < 2 || oversample < 0 || D > 64 || D + oversample > 96) return 0;
    return (size_t)workspace_doubles(D, oversample) * 8;
}

size_t tatrg_workspace_bytes_ilo(int D, int oversample, int bond_rank) {
    const size_t base = tatrg_workspace_bytes(D, oversample);
    if (base == 0 || bond_rank < D || bond_rank > 4 * D || bond_rank + oversample > 112) return 0;
    // every tensor carries at most two overspanned legs (X, Y, F, G of fn 5 :203): the plain bound times (r_bond)^2
    const double r = (double)bond_rank / D;
    return (size_t)((double)base * r * r);
}

size_t tatrg_workspace_bytes_atrg(int D, int oversample) {
    const size_t base = tatrg_workspace_bytes(D, oversample);
    if (base == 0) return 0;
    const double d = D;
    return base + (size_t)(8.0 * (4.0 * std::pow(d, 6) + 8.0 * std::pow(d, 5)));
}

int tatrg_create(double beta, double h, int D, int oversample, uint64_t seed, void* workspace, size_t workspace_bytes, tatrg_handle* out) {
    if (!out) return TATRG_EINVAL;
    *out = nullptr;
    if (!finite_pos(beta) || !std::isfinite(h) || D < 2 || D > 64 || oversample < 0 || D + oversample > 96 || !workspace) return TATRG_EINVAL;
    if (((uintptr_t)workspace & 255) != 0) return TATRG_EINVAL;
    if (workspace_bytes < tatrg_workspace_bytes(D, oversample)) return TATRG_ENOMEM;
    tatrg_ctx* c = new (std::nothrow) tatrg_ctx();
    if (!c) return TATRG_ENOMEM;
    c->beta = beta; c->h = h; c->D = D; c->p = oversample; c->seed = seed; c->Ktri = D + oversample; c->Dbond = D;
    c->pool.reset(workspace, workspace_bytes);
    c->trace_dev = c->pool.alloc(kTraceDoubles);
    c->phi.nd = c->psi.nd = 5;
    for (int i = 0; i < 4; ++i) c->phi.d[i] = c->psi.d[i] = 2;
    c->phi.d[4] = c->psi.d[4] = 2;
    c->phi.p = c->pool.alloc(32); c->psi.p = c->pool.alloc(32);
    cudaError_t e = init_ising(nullptr, beta, h, c->phi.p, c->psi.p);          // Eq. 3.1-3.2 :241-246
    if (e == cudaSuccess) e = dot(nullptr, 32, c->phi.p, c->psi.p, c->trace_dev);
    if (e == cudaSuccess) e = cudaStreamSynchronize(nullptr);
    if (e != cudaSuccess) { delete c; return TATRG_ECUDA; }
    *out = c;
    return TATRG_OK;
}

int tatrg_set_option(tatrg_handle c, int key, double value) {
    if (!c) return TATRG_EINVAL;
    switch (key) {
        case TATRG_OPT_POWER_ITERS: if (c->m > 0) return TATRG_ESTATE; if (value < 0 || value > 64) return TATRG_EINVAL; c->n_pow = (int)value; return TATRG_OK;
        case TATRG_OPT_K_TRIAD: if (c->m > 0) return TATRG_ESTATE; if (value < 1 || value > c->D + c->p) return TATRG_EINVAL; c->Ktri = (int)value; return TATRG_OK;
        case TATRG_OPT_TAU: if (c->m > 0) return TATRG_ESTATE; if (!(value >= 0) || value > 0.1) return TATRG_EINVAL; c->tau = value; return TATRG_OK;
        case TATRG_OPT_STAGE_TIMING: c->timing = (int)value; return TATRG_OK;
        case TATRG_OPT_KEEP_TENSORS: c->keep_tensors = value != 0; return TATRG_OK;
        case TATRG_OPT_SUBSPACE: c->use_subspace = value != 0; return TATRG_OK;
        case TATRG_OPT_OVERLAP: c->use_overlap = value != 0; return TATRG_OK;
        case TATRG_OPT_GRAPHS: c->use_graphs = value != 0; return TATRG_OK;
        case TATRG_OPT_VERBOSE: if (value < 0 || value > 15) return TATRG_EINVAL; c->verbose = (int)value; return TATRG_OK;
        case TATRG_OPT_DGEMM_TMA: c->dgemm_tma = value != 0; return TATRG_OK;
        case TATRG_OPT_IMPLICIT_XY: c->implicit_xy = value != 0; return TATRG_OK;
        case TATRG_OPT_CHEBYSHEV: c->use_cheb = value != 0; return TATRG_OK;
        case TATRG_OPT_BOND_RANK: {
            if (c->m > 0) return TATRG_ESTATE;
            if (value != std::floor(value) || value < c->D) return TATRG_EINVAL;
            const size_t need = tatrg_workspace_bytes_ilo(c->D, c->p, (int)value);
            if (need == 0) return TATRG_EINVAL;
            if (c->pool.capacity() < (need & ~(size_t)255)) return TATRG_ENOMEM;
            c->Dbond = (int)value; return TATRG_OK;
        }
        case TATRG_OPT_METHOD:
            if (c->m > 0) return TATRG_ESTATE;
            if (value != 0 && value != 1) return TATRG_EINVAL;
            if (value == 1 && c->pool.capacity() < (tatrg_workspace_bytes_atrg(c->D, c->p) & ~(size_t)255)) return TATRG_ENOMEM;
            c->method = (int)value; return TATRG_OK;
        default: return TATRG_EINVAL;
    }
}

int tatrg_step(tatrg_handle c, void* cuda_stream) {
    if (!c) return TATRG_EINVAL;
    if (c->failed) return TATRG_ESTATE;
    return run_step(c, (cudaStream_t)cuda_stream);
}

double tatrg_lnZ_per_site(tatrg_handle c) {
    if (!c || c->failed) return NAN;
    double tr = 0;
    if (cudaMemcpyAsync(&tr, c->trace_dev, 8, cudaMemcpyDeviceToHost, c->last_stream) != cudaSuccess) return NAN;
    if (cudaStreamSynchronize(c->last_stream) != cudaSuccess) return NAN;
    if (!(tr > 0) || !std::isfinite(tr)) { c->err = "non-positive tensor trace"; return NAN; }
    double v = 0, w = 1;
    for (double l : c->lnc) { v += w * l; w *= 0.5; }          // R8: sum_j 2^-j ln c_j + 2^-m ln tTr
    return v + w * std::log(tr);
}

int tatrg_x_ratio(tatrg_handle c, void* cuda_stream, double* x_out) {
    if (!c || !x_out) return TATRG_EINVAL;
    if (c->failed) return TATRG_ESTATE;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    if (c->done_ev && st != c->last_stream && cudaStreamWaitEvent(st, c->done_ev, 0) != cudaSuccess) return TATRG_ECUDA;
    const int n = (int)c->phi.d[3];
    Tens a; a.p = c->pool.alloc((int64_t)n * n + 2);
    if (!a.p) return TATRG_ENOMEM;
    std::string err;
    int rc = contract(st, "ijkag,ijkbg->ab", c->phi, c->psi, a, c->pool, &err);      // A[k,l] = sum T[i1 i2 i3 k, i1 i2 i3 l]
    double tr[2] = {0, 0};
    if (rc == TATRG_OK && traces(st, a.p, n, a.p + (int64_t)n * n) != cudaSuccess) rc = TATRG_ECUDA;
    if (rc == TATRG_OK && cudaMemcpyAsync(tr, a.p + (int64_t)n * n, 16, cudaMemcpyDeviceToHost, st) != cudaSuccess) rc = TATRG_ECUDA;
    if (rc == TATRG_OK && cudaStreamSynchronize(st) != cudaSuccess) rc = TATRG_ECUDA;
    c->pool.free(a.p);
    if (rc != TATRG_OK) { c->err = err; return rc; }
    if (!(tr[1] > 0)) { c->err = "x_ratio: non-positive Tr A^2"; return TATRG_ENUMERIC; }
    *x_out = tr[0] * tr[0] / tr[1];
    return TATRG_OK;
}

int tatrg_singular_values(tatrg_handle c, int which, int k, double* out_host) {
    if (!c || !out_host || k < 0) return TATRG_EINVAL;
    if (c->m == 0) return TATRG_ESTATE;
    const std::vector<double>& v = which == TATRG_SV_S ? c->sv_s : c->sv_sigma;
    if (which != TATRG_SV_S && which != TATRG_SV_SIGMA) return TATRG_EINVAL;
    int n = std::min<int>(k, (int)v.size());
    for (int i = 0; i < n; ++i) out_host[i] = v[i];
    return n;
}

int tatrg_steps_done(tatrg_handle c) { return c ? c->m : TATRG_EINVAL; }
const char* tatrg_last_error(tatrg_handle c) { return c ? c->err.c_str() : "null handle"; }
size_t tatrg_workspace_peak(tatrg_handle c) { return c ? c->pool.peak() : 0; }

void tatrg_destroy(tatrg_handle c) {
    if (!c) return;
    for (auto e : c->stage_ev) cudaEventDestroy(e);
    for (auto e : c->cnt.ev_pool) cudaEventDestroy(e);
    if (c->done_ev) cudaEventDestroy(c->done_ev);
    if (!c->graveyard.empty()) { cudaStreamSynchronize(c->last_stream); for (auto g : c->graveyard) cudaGraphExecDestroy(g); }
    delete c;
}

int tatrg_stage_ms(tatrg_handle c, double* ms) {
    if (!c || !ms) return TATRG_EINVAL;
    for (int i = 0; i < TATRG_NSTAGES; ++i) ms[i] = c->stage_ms[i];
    return TATRG_OK;
}
int tatrg_stage_flops(tatrg_handle c, double* fl) {
    if (!c || !fl) return TATRG_EINVAL;
    for (int i = 0; i < TATRG_NSTAGES; ++i) fl[i] = c->stage_flops[i];
    return TATRG_OK;
}
long long tatrg_last_step_launches(tatrg_handle c) { return c ? c->last_launches : TATRG_EINVAL; }
long long tatrg_last_step_host_syncs(tatrg_handle c) { return c ? c->last_host_syncs : TATRG_EINVAL; }
int tatrg_gemm_profile(tatrg_handle c, double* ms, double* flops, long long* calls) {
    if (!c) return TATRG_EINVAL;
    if (ms) *ms = c->gemm_ms; if (flops) *flops = c->gemm_flops; if (calls) *calls = c->gemm_calls;
    return TATRG_OK;
}
int tatrg_gemm_profile_large(tatrg_handle c, double* ms, double* flops, long long* calls) {
    if (!c) return TATRG_EINVAL;
    if (ms) *ms = c->gemm_large_ms; if (flops) *flops = c->gemm_large_flops; if (calls) *calls = c->gemm_large_calls;
    return TATRG_OK;
}
int tatrg_permute_profile(tatrg_handle c, double* ms, double* bytes, long long* calls) {
    if (!c) return TATRG_EINVAL;
    if (ms) *ms = c->perm_ms; if (bytes) *bytes = (double)c->perm_bytes; if (calls) *calls = c->perm_calls;
    return TATRG_OK;
}
int tatrg_permute_profile_large(tatrg_handle c, double* ms, double* bytes, long long* calls) {
    if (!c) return TATRG_EINVAL;
    if (ms) *ms = c->perm_large_ms; if (bytes) *bytes = (double)c->perm_large_bytes; if (calls) *calls = c->perm_large_calls;
    return TATRG_OK;
}

long long tatrg_get_tensor(tatrg_handle c, const char* name, double* out_host, long long capacity, int* ndim, long long* dims) {
    if (!c || !name) return TATRG_EINVAL;
    Tens t;
    if (!strcmp(name, "phi")) t = c->phi;
    else if (!strcmp(name, "psi")) t = c->psi;
    else { auto it = c->kept.find(name); if (it == c->kept.end()) return TATRG_ESTATE; t = it->second; }
    if (ndim) *ndim = t.nd;
    if (dims) for (int i = 0; i < t.nd; ++i) dims[i] = t.d[i];
    const long long n = t.size();
    if (!out_host || capacity < n) return n;
    if (cudaMemcpyAsync(out_host, t.p, 8 * n, cudaMemcpyDeviceToHost, c->last_stream) != cudaSuccess) return TATRG_ECUDA;
    if (cudaStreamSynchronize(c->last_stream) != cudaSuccess) return TATRG_ECUDA;
    return n;
}

int tatrg_set_state(tatrg_handle c, const double* phi_host, const double* psi_host, const long long* dims5) {
    if (!c || !phi_host || !psi_host || !dims5) return TATRG_EINVAL;
    Tens t; t.nd = 5;
    for (int i = 0; i < 5; ++i) { if (dims5[i] < 1 || dims5[i] > 64) return TATRG_EINVAL; t.d[i] = dims5[i]; }
    double* a = c->pool.alloc(t.size()); double* b = c->pool.alloc(t.size());
    if (!a || !b) { c->pool.free(a); c->pool.free(b); return TATRG_ENOMEM; }
    cudaStream_t st = c->last_stream;
    cudaError_t e = cudaMemcpyAsync(a, phi_host, 8 * t.size(), cudaMemcpyHostToDevice, st);
    if (e == cudaSuccess) e = cudaMemcpyAsync(b, psi_host, 8 * t.size(), cudaMemcpyHostToDevice, st);
    if (e == cudaSuccess) e = dot(st, t.size(), a, b, c->trace_dev);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    if (e != cudaSuccess) { c->pool.free(a); c->pool.free(b); return TATRG_ECUDA; }
    c->pool.free(c->phi.p); c->pool.free(c->psi.p);
    c->phi = t; c->phi.p = a; c->psi = t; c->psi.p = b;
    c->failed = false;
    return TATRG_OK;
}

// ---- primitives ----------------------------------------------------------------------------------------------
int tatrg_dgemm(void* st, int transa, int transb, long long M, long long N, long long K, double alpha, const double* A, long long lda,
                const double* B, long long ldb, double beta, double* C, long long ldc, int batch, long long sA, long long sB, long long sC) {
    if (M < 0 || N < 0 || K < 0 || batch < 1 || (!A && M * K > 0) || (!B && N * K > 0) || !C) return TATRG_EINVAL;
    cudaError_t e = dgemm((cudaStream_t)st, transa != 0, transb != 0, M, N, K, alpha, A, lda, B, ldb, beta, C, ldc, batch, sA, sB, sC);
    return e == cudaSuccess ? TATRG_OK : TATRG_ECUDA;
}

int tatrg_dgemm_variant(void* st, int variant, int transa, int transb, long long M, long long N, long long K, double alpha, const double* A, long long lda,
                        const double* B, long long ldb, double beta, double* C, long long ldc, int batch, long long sA, long long sB, long long sC) {
    if (M < 1 || N < 1 || K < 1 || batch < 1 || !A || !B || !C || (variant != 0 && variant != 1)) return TATRG_EINVAL;
    if (variant == 1) {
        cudaError_t e = dgemm_tma((cudaStream_t)st, transa == 0, transb != 0, M, N, K, alpha, A, lda, B, ldb, beta, C, ldc, batch, sA, sB, sC, false);
        return e == cudaSuccess ? TATRG_OK : (e == cudaErrorNotSupported ? TATRG_EINVAL : TATRG_ECUDA);
    }
    const int saved = g_dgemm_tma;
    g_dgemm_tma = 0;
    cudaError_t e = dgemm((cudaStream_t)st, transa != 0, transb != 0, M, N, K, alpha, A, lda, B, ldb, beta, C, ldc, batch, sA, sB, sC);
    g_dgemm_tma = saved;
    return e == cudaSuccess ? TATRG_OK : TATRG_ECUDA;
}

int tatrg_permute(void* st, int ndim, const long long* dims, const int* perm, const double* in, double* out) {
    if (ndim < 1 || ndim > 8 || !dims || !perm || !in || !out) return TATRG_EINVAL;
    int64_t d[8]; bool seen[8] = {false};
    for (int i = 0; i < ndim; ++i) { d[i] = dims[i]; if (dims[i] < 0 || perm[i] < 0 || perm[i] >= ndim || seen[perm[i]]) return TATRG_EINVAL; seen[perm[i]] = true; }
    cudaError_t e = permute((cudaStream_t)st, ndim, d, perm, in, out);
    return e == cudaSuccess ? TATRG_OK : TATRG_ECUDA;
}

int tatrg_contract(void* st, const char* spec, const double* A, const long long* dimsA, const double* B, const long long* dimsB, double* C,
                   void* scratch, size_t scratch_bytes) {
    if (!spec || !A || !B || !C || !dimsA || !dimsB) return TATRG_EINVAL;
    const char* comma = strchr(spec, ','); const char* arrow = strstr(spec, "->");
    if (!comma || !arrow || comma > arrow) return TATRG_EINVAL;
    Tens a, b, c;
    a.nd = (int)(comma - spec); b.nd = (int)(arrow - comma - 1);
    if (a.nd > 8 || b.nd > 8 || a.nd < 1 || b.nd < 1) return TATRG_EINVAL;
    for (int i = 0; i < a.nd; ++i) a.d[i] = dimsA[i];
    for (int i = 0; i < b.nd; ++i) b.d[i] = dimsB[i];
    a.p = const_cast<double*>(A); b.p = const_cast<double*>(B); c.p = C;
    Pool pool;
    uintptr_t base = ((uintptr_t)scratch + 255) & ~(uintptr_t)255;
    size_t lost = base - (uintptr_t)scratch;
    pool.reset((void*)base, scratch && scratch_bytes > lost ? scratch_bytes - lost : 0);
    std::string err;
    try { return contract((cudaStream_t)st, spec, a, b, c, pool, &err); } catch (...) { return TATRG_ECUDA; }
}

int tatrg_philox_raw(void* st, uint64_t seed, uint32_t call, uint32_t stream_id, uint64_t start, long long count, uint32_t* raw) {
    if (count < 0 || (!raw && count > 0)) return TATRG_EINVAL;
    return philox_raw((cudaStream_t)st, seed, call, stream_id, start, count, raw) == cudaSuccess ? TATRG_OK : TATRG_ECUDA;
}
int tatrg_philox_gaussian(void* st, uint64_t seed, uint32_t call, uint32_t stream_id, uint64_t start, long long count, double* z) {
    if (count < 0 || (!z && count > 0)) return TATRG_EINVAL;
    return philox_gauss((cudaStream_t)st, seed, call, stream_id, start, count, z) == cudaSuccess ? TATRG_OK : TATRG_ECUDA;
}

size_t tatrg_eigh_work_bytes(int n) { return n > 0 ? eigh_work_bytes(n) : 0; }
int tatrg_eigh(void* st, int n, double* G, double* lam, double* Vt, void* work) {
    if (n < 1 || !G || !lam || !Vt || !work) return TATRG_EINVAL;
    std::string err;
    try { return eigh((cudaStream_t)st, n, G, lam, Vt, work, nullptr, &err); } catch (...) { return TATRG_ECUDA; }
}
size_t tatrg_svd_work_bytes(int nv, int len) { return (nv > 0 && len > 0) ? svd_rows_work_bytes(nv, len) : 0; }
int tatrg_svd(void* st, int nv, int len, const double* X, double* s, double* Ut, double* Vacc, void* work) {
    if (nv < 1 || len < 1 || !X || !s || !Ut || !Vacc || !work) return TATRG_EINVAL;
    std::string err;
    try { return svd_rows((cudaStream_t)st, nv, len, X, s, Ut, Vacc, work, nullptr, &err); } catch (...) { return TATRG_ECUDA; }
}
size_t tatrg_gram_scratch_bytes(long long m, int n) { return (m > 0 && n > 0) ? 8 * (size_t)dgemm_splitk_doubles(n, n, m, n >= 256) : 0; }
int tatrg_gram(void* stp, long long m, int n, const double* X, double* G, void* scratch) {
    if (m < 1 || n < 1 || !X || !G) return TATRG_EINVAL;
    cudaStream_t st = (cudaStream_t)stp;
    const bool lower = n >= 256;
    cudaError_t e = dgemm_splitk(st, true, false, n, n, m, 1.0, X, n, X, n, G, n, (double*)scratch, lower);
    if (e == cudaSuccess && lower) e = mirror_lower(st, n, G);
    return e == cudaSuccess ? TATRG_OK : TATRG_ECUDA;
}
size_t tatrg_cholqr_work_bytes(int n) { return n > 0 ? 8 * (2 * (size_t)n * n + cholesky_work_doubles(n)) + 4096 : 0; }
int tatrg_cholqr(void* stp, long long m, int n, double* X, double* Q, double* R, void* work) {
    if (m < n || n < 1 || !X || !Q || !R || !work) return TATRG_EINVAL;
    cudaStream_t st = (cudaStream_t)stp;
    double* G = (double*)work; double* L = G + (size_t)n * n; double* cw = L + (size_t)n * n;
    cudaError_t e = dgemm(st, true, false, n, n, m, 1.0, X, n, X, n, 0.0, G, n);
    if (e == cudaSuccess) e = fill_zero(st, L, (int64_t)n * n);
    if (e == cudaSuccess) e = cholesky(st, n, G, n, L, n, 0.0, 1e-14, cw);
    if (e == cudaSuccess) e = trsm_right_lt(st, m, n, X, n, Q, n, L, n, cw);
    const int64_t dims[2] = {n, n}; const int perm[2] = {1, 0};
    if (e == cudaSuccess) e = permute(st, 2, dims, perm, L, R);
    int info = 0;
    if (e == cudaSuccess) e = cudaMemcpyAsync(&info, cholesky_info(cw, n), sizeof(int), cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    if (e != cudaSuccess) return TATRG_ECUDA;
    return info == 0 ? TATRG_OK : TATRG_ENUMERIC;
}
size_t tatrg_pchol_work_bytes(int n) { return n > 0 ? 8 * pchol_work_doubles(n) + 4096 : 0; }
int tatrg_pchol(void* stp, int n, const double* G, double* L, double tol_rel, void* work, int* rank_out, double* resid_out) {
    if (n < 1 || !(tol_rel >= 0) || !G || !L || !work || !rank_out || !resid_out) return TATRG_EINVAL;
    cudaStream_t st = (cudaStream_t)stp;
    double info[4] = {0, 0, 0, 0};
    cudaError_t e = pchol(st, n, G, L, n, tol_rel, (double*)work);
    if (e == cudaSuccess) e = cudaMemcpyAsync(info, pchol_info((const double*)work), sizeof info, cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    if (e != cudaSuccess) return TATRG_ECUDA;
    *rank_out = (int)info[0]; *resid_out = info[2] > 0 ? info[1] / info[2] : 0.0;
    return TATRG_OK;
}
int tatrg_dot(void* st, long long n, const double* x, const double* y, double* result) {
    if (n < 0 || !x || !y || !result) return TATRG_EINVAL;
    return dot((cudaStream_t)st, n, x, y, result) == cudaSuccess ? TATRG_OK : TATRG_ECUDA;
}

}  // extern "C"
