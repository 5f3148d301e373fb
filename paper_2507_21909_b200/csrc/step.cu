// step.cu -- one Triad-ATRG coarse-graining step, Fig. 5 (a)-(f) of PAPER.md (:193), enqueued on one CUDA stream.
//
//   (a) decomposition of T = Phi Psi^T            Eq. 2.4 :76            decompose()
//   (b) bond swap by RSVD                         Eq. 2.5 :90, App. A    bond_swap()
//   (c) triad isometries / triad tensors          Eq. 2.9-2.17 :135-167  triad()
//   (d) squeezers                                 :113, :171             half_grams(), squeezer()
//   (e) coarse-graining contraction               Eq. 2.18-2.19 :175     contract_upper/lower()
//   (f) axis rotation, trace                      Fig. 5(f)              run()
//
// All arithmetic is in the kernels of dgemm.cu / permute.cu / elementwise.cu / philox.cu / jacobi.cu; the host code
// here only takes the rank decisions (from read-back spectra) and sizes / sequences the launches.
// Readings R1..R14 are those of DESIGN.md section 3.
#include "step.h"
#include <algorithm>
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <functional>
#include <mutex>
#include <chrono>

namespace tatrg {
namespace {

[[noreturn]] void fail(int code, const char* fmt, ...) {
    char buf[512];
    va_list ap; va_start(ap, fmt); vsnprintf(buf, sizeof buf, fmt, ap); va_end(ap);
    throw Fail{code, buf};
}
void ck(cudaError_t e, const char* what) { if (e != cudaSuccess) fail(TATRG_ECUDA, "%s: %s", what, cudaGetErrorString(e)); }

// R7: number of leading values to keep: at most kmax, only values > eps*v[0], never cutting through a multiplet
int select_rank(const std::vector<double>& v, int kmax, double eps, double tau) {
    if (v.empty() || !(v[0] > 0)) return 0;
    int npos = 0;
    for (double x : v) if (x > eps * v[0]) ++npos;
    if (npos <= kmax) return npos;
    int k = kmax;
    while (k > 0 && (v[k - 1] - v[k]) <= tau * v[k - 1]) --k;
    return k > 0 ? k : kmax;
}
// runs of consecutive values with relative gap <= tau among the first k
std::vector<int> multiplets(const std::vector<double>& v, int k, double tau) {
    std::vector<int> g; int start = 0;
    for (int i = 1; i <= k; ++i)
        if (i == k || (v[i - 1] - v[i]) > tau * v[i - 1]) { g.push_back(start); g.push_back(i); start = i; }
    return g;
}

struct Stepper {
    tatrg_ctx& c;
    cudaStream_t st;
    std::vector<std::vector<double*>> scopes;
    int call;

    std::function<void()> submark;   // closes a timing sub-stage from inside a stage function (set by run())

    Stepper(tatrg_ctx& ctx, cudaStream_t s) : c(ctx), st(s), call(ctx.m + 1) { scopes.emplace_back(); }
    ~Stepper() { while (!scopes.empty()) pop(); }

    // ---- memory ----------------------------------------------------------------------------------------------
    void push() { scopes.emplace_back(); }
    void pop() { for (double* p : scopes.back()) c.pool.free(p); scopes.pop_back(); }
    struct Scope { Stepper& s; Scope(Stepper& s_) : s(s_) { s.push(); } ~Scope() { s.pop(); } };
    double* raw(int64_t n) {
        double* p = c.pool.alloc(n);
        if (!p) fail(TATRG_ENOMEM, "workspace exhausted: need %lld more doubles (in use %zu of %zu bytes)", (long long)n, c.pool.in_use(), c.pool.capacity());
        scopes.back().push_back(p);
        return p;
    }
    // optional scratch (split-K partials, the overlap arena): null when the workspace has no room; registered in the current scope so
    // that an exception between here and release() cannot leave the block live in the caller's workspace
    double* scratch(int64_t n) {
        double* p = n > 0 ? c.pool.alloc(n) : nullptr;
        if (p) scopes.back().push_back(p);
        return p;
    }
    void release(double* p) { if (p) { Tens t; t.p = p; drop(t); } }
    Tens make(std::initializer_list<int64_t> dims) {
        Tens t; t.nd = 0; for (int64_t d : dims) t.d[t.nd++] = d;
        t.p = raw(t.size());
        return t;
    }
    static Tens view(const Tens& t, std::initializer_list<int64_t> dims) {
        Tens v; v.p = t.p; v.nd = 0; for (int64_t d : dims) v.d[v.nd++] = d;
        if (v.size() != t.size()) fail(TATRG_EINVAL, "internal: bad view");
        return v;
    }
    // move ownership of t one scope up (so that it survives the current scope)
    void keep(const Tens& t) {
        auto& cur = scopes.back();
        auto it = std::find(cur.begin(), cur.end(), t.p);
        if (it == cur.end()) return;
        cur.erase(it);
        scopes[scopes.size() - 2].push_back(t.p);
    }
    void drop(Tens& t) {
        for (auto sc = scopes.rbegin(); sc != scopes.rend(); ++sc) {
            auto it = std::find(sc->begin(), sc->end(), t.p);
            if (it != sc->end()) { sc->erase(it); c.pool.free(t.p); t.p = nullptr; return; }
        }
    }
    // hand a tensor over to the context (state, or kept for inspection): leaves every scope
    void detach(const Tens& t) {
        for (auto& sc : scopes) { auto it = std::find(sc.begin(), sc.end(), t.p); if (it != sc.end()) { sc.erase(it); return; } }
    }
    void save(const char* name, const Tens& t) {   // copy for tatrg_get_tensor (tests); only with keep_tensors
        if (!c.keep_tensors) return;
        Tens k = t; k.p = c.pool.alloc(t.size());
        if (!k.p) fail(TATRG_ENOMEM, "workspace exhausted keeping tensor %s", name);
        ck(cudaMemcpyAsync(k.p, t.p, 8 * t.size(), cudaMemcpyDeviceToDevice, st), "save"); count_launch();
        auto it = c.kept.find(name);
        if (it != c.kept.end()) c.pool.free(it->second.p);
        c.kept[name] = k;
    }

    // ---- thin wrappers ---------------------------------------------------------------------------------------
    Tens ein(const char* spec, const Tens& A, const Tens& B) {
        Tens C; std::string e;
        int rc = contract_shape(spec, A, B, C, &e);
        if (rc != TATRG_OK) fail(rc, "%s", e.c_str());
        C.p = raw(C.size());
        rc = contract(st, spec, A, B, C, c.pool, &e);
        if (rc != TATRG_OK) fail(rc, "%s [%s]", e.c_str(), spec);
        return C;
    }
    Tens perm(const Tens& t, std::initializer_list<int> p) {
        Tens o; o.nd = t.nd; int pr[8]; int i = 0;
        for (int x : p) { pr[i] = x; o.d[i] = t.d[x]; ++i; }
        o.p = raw(o.size());
        ck(permute(st, t.nd, t.d, pr, t.p, o.p), "permute");
        return o;
    }
    // C[M,N] = op(A) op(B), plain 2-D, with split-K when the output is small
    // sym: the result is symmetric (a Gram matrix): only the tiles on and below the diagonal are computed, then mirrored
    Tens mm(bool ta, bool tb, int64_t M, int64_t N, int64_t K, const double* A, int64_t lda, const double* B, int64_t ldb, bool sym = false) {
        Tens C = make({M, N});
        const bool lower = sym && M == N && M >= 256;
        int64_t need = dgemm_splitk_doubles(M, N, K, lower);
        double* part = scratch(need);
        ck(dgemm_splitk(st, ta, tb, M, N, K, 1.0, A, lda, B, ldb, C.p, N, part, lower), "dgemm");
        release(part);
        if (lower) ck(mirror_lower(st, (int)M, C.p), "mirror");
        return C;
    }
    // the same into caller-provided storage (leading dimension ldc)
    // While several problems are in flight on their own streams (sub_iterate) the split-K partials must not come from the
    // pool's enqueue-order reuse: part_fixed then points to the problem's own scratch of part_cap doubles.
    double* part_fixed = nullptr; int64_t part_cap = 0;
    void mm_into(double* C, int64_t ldc, bool ta, bool tb, int64_t M, int64_t N, int64_t K, const double* A, int64_t lda, const double* B, int64_t ldb) {
        int64_t need = dgemm_splitk_doubles(M, N, K);
        if (part_fixed) {
            ck(dgemm_splitk(st, ta, tb, M, N, K, 1.0, A, lda, B, ldb, C, ldc, need <= part_cap ? part_fixed : nullptr), "dgemm");
            return;
        }
        double* part = scratch(need);
        ck(dgemm_splitk(st, ta, tb, M, N, K, 1.0, A, lda, B, ldb, C, ldc, part), "dgemm");
        release(part);
    }
    std::vector<double> to_host(const double* d, int64_t n) {
        std::vector<double> h(n);
        ck(cudaMemcpyAsync(h.data(), d, 8 * n, cudaMemcpyDeviceToHost, st), "readback");
        ck(cudaStreamSynchronize(st), "sync"); count_sync();
        return h;
    }
    double* to_dev(const std::vector<double>& h) {
        double* d = raw((int64_t)h.size());
        ck(cudaMemcpyAsync(d, h.data(), 8 * h.size(), cudaMemcpyHostToDevice, st), "upload");
        return d;
    }
    int* to_dev_int(const std::vector<int>& h) {
        int* d = (int*)raw((int64_t)(h.size() + 1) / 2 + 1);
        ck(cudaMemcpyAsync(d, h.data(), 4 * h.size(), cudaMemcpyHostToDevice, st), "upload");
        return d;
    }

    // ---- decompositions --------------------------------------------------------------------------------------
    // eigen-decomposition of the symmetric n x n matrix G (destroyed): lam [dev], Vt rows [dev], lam on the host
    void eig(Tens& G, int n, double*& lam, Tens& Vt, std::vector<double>& lam_h) {
        lam = raw(n);
        Vt = make({n, n});
        size_t wb = eigh_work_bytes(n);
        double* work = c.pool.alloc((int64_t)(wb / 8 + 1));
        if (!work) fail(TATRG_ENOMEM, "workspace exhausted (eigh work, n=%d)", n);
        std::string e;
        int rc = eigh(st, n, G.p, lam, Vt.p, work, &lam_h, &e);
        c.pool.free(work);
        if (rc != TATRG_OK) fail(rc, "%s", e.c_str());
    }

    // the same for several independent matrices in the same launches (jacobi.cu: eigh_batched)
    struct EigOut { double* lam; Tens Vt; std::vector<double> lh; };
    void eig_batch(const std::vector<Tens*>& G, const std::vector<int>& n, std::vector<EigOut>& out) {
        const int cnt = (int)G.size();
        out.resize(cnt);
        int nmax = 0;
        std::vector<EighItem> items(cnt);
        for (int i = 0; i < cnt; ++i) {
            out[i].lam = raw(n[i]);
            out[i].Vt = make({n[i], n[i]});
            items[i] = EighItem{n[i], G[i]->p, out[i].lam, out[i].Vt.p, &out[i].lh};
            nmax = std::max(nmax, n[i]);
        }
        size_t wb = eigh_batched_work_bytes(nmax, cnt);
        double* work = c.pool.alloc((int64_t)(wb / 8 + 1));
        if (!work) fail(TATRG_ENOMEM, "workspace exhausted (batched eigh work, n=%d x %d)", nmax, cnt);
        std::string e;
        int rc = eigh_batched(st, cnt, items.data(), work, &e);
        c.pool.free(work);
        if (rc != TATRG_OK) fail(rc, "%s", e.c_str());
    }

    // Orthonormal basis of the numerical column space of mat [m x n]:  mat = Q R, Q [m x r], R [r x n]   (R14).
    // Gram matrix -> eigen-decomposition -> Q = mat V lam^-1/2 (directions with lam <= 1e-12 lam_max dropped), and a
    // second identical pass on Q for narrow matrices (n <= 128), where it is cheap, to restore orthogonality to eps.
    // span_only: the caller uses Q only as a basis of the column space that is multiplied by the operator and orthonormalised
    // again (the intermediate passes of Eq. A.4-A.6): one Cholesky pass (Q^T Q = 1 to cond^2 eps) is enough there.
    void orth(const Tens& mat, Tens& Q, Tens& R, bool span_only = false) {
        if (c.use_subspace && mat.d[1] >= 8 && mat.d[1] <= 128 && mat.d[0] >= 4 * mat.d[1] && orth_chol(mat, Q, R, span_only ? 1 : 2)) return;
        Scope sc(*this);
        const int64_t m = mat.d[0], n = mat.d[1];
        Tens G = mm(true, false, n, n, m, mat.p, n, mat.p, n);
        double* lam; Tens Vt; std::vector<double> lh;
        eig(G, (int)n, lam, Vt, lh);
        if (!(lh[0] > 0)) fail(TATRG_ENUMERIC, "orth: zero matrix");
        int r = 0;
        for (double x : lh) if (x > kEpsOrthLambda * lh[0]) ++r;
        Tens Q1 = mm(false, true, m, r, n, mat.p, n, Vt.p, n);
        ck(scale_last(st, Q1.p, Q1.p, lam, m, r, 2), "scale");
        Tens R1 = make({r, n});
        ck(scale_rows(st, R1.p, Vt.p, lam, r, n, 3), "scale");
        if (n > 128) { Q = Q1; R = R1; keep(Q); keep(R); return; }
        Tens G2 = mm(true, false, r, r, m, Q1.p, r, Q1.p, r);
        double* lam2; Tens V2; std::vector<double> l2;
        eig(G2, r, lam2, V2, l2);
        if (!(l2[r - 1] > 0)) fail(TATRG_ENUMERIC, "orth: second pass lost rank");
        Q = mm(false, true, m, r, r, Q1.p, r, V2.p, r);
        ck(scale_last(st, Q.p, Q.p, lam2, m, r, 2), "scale");
        Tens SV = make({r, r});
        ck(scale_rows(st, SV.p, V2.p, lam2, r, r, 3), "scale");
        R = mm(false, false, r, n, r, SV.p, r, R1.p, n);
        keep(Q); keep(R);
    }

    // Cholesky QR of a tall matrix of full numerical rank (Eq. A.2-A.3 :345-348): G = mat^T mat = L L^T, R = L^T,
    // Q = mat R^-1 (one GEMM with the explicit triangular inverse).  Same span and same product Q R as orth(); accepted
    // only when the factor PROVES that orth() would drop nothing (R14): lam_min(G) = sigma_min(L)^2 >= 1 / ||L^-1||_F^2
    // and lam_max(G) <= tr G, so 1 / (||L^-1||_F^2 tr G) > 1e-12 implies lam_min > 1e-12 lam_max.  Returns false otherwise.
    bool orth_chol(const Tens& mat, Tens& Q, Tens& R, int passes = 1) {
        Scope sc(*this);
        const int64_t m = mat.d[0], n = mat.d[1];
        Tens G = mm(true, false, n, n, m, mat.p, n, mat.p, n, true);
        Tens L = make({n, n}), X = make({n, n}), T = make({(int64_t)tri_inverse_scratch_doubles((int)n)});
        double* cw = raw((int64_t)cholesky_work_doubles((int)n));
        double* res = raw(1 + 148 * 8 + 7);
        ck(fill_zero(st, L.p, n * n), "zero"); ck(fill_zero(st, X.p, n * n), "zero");
        ck(cholesky(st, (int)n, G.p, n, L.p, n, 0.0, 1e-14, cw), "cholesky");
        ck(tri_inverse(st, (int)n, L.p, n, cw, X.p, n, T.p), "tri_inverse");
        ck(dot(st, n * n, X.p, X.p, res), "dot");
        int info = 0;
        std::vector<double> d0(n), xn(1);              // three read-backs, one synchronisation
        ck(cudaMemcpyAsync(&info, cholesky_info(cw, (int)n), sizeof(int), cudaMemcpyDeviceToHost, st), "readback");
        ck(cudaMemcpyAsync(d0.data(), cholesky_d0(cw, (int)n), 8 * n, cudaMemcpyDeviceToHost, st), "readback");
        ck(cudaMemcpyAsync(xn.data(), res, 8, cudaMemcpyDeviceToHost, st), "readback");
        ck(cudaStreamSynchronize(st), "sync"); count_sync();
        double tr = 0; for (double v : d0) tr += v;
        if (g_verbose & 1) fprintf(stderr, "[tatrg cholesky qr %lld x %lld] info %d, proven lam_min/lam_max >= %.3e\n", (long long)m, (long long)n, info, 1.0 / (xn[0] * tr));
        if (info != 0 || !std::isfinite(xn[0]) || !(xn[0] > 0) || !(tr > 0)) return false;
        if (!(1.0 / (xn[0] * tr) > kEpsOrthLambda)) return false;
        Q = mm(false, true, m, n, n, mat.p, n, X.p, n);
        if (passes < 2) {
            R = perm(view(L, {n, n}), {1, 0});
        } else {
            // second pass on the almost orthonormal Q (CholeskyQR2): Q^T Q = L2 L2^T, Q <- Q L2^-T, R = (L L2)^T
            Tens G2 = mm(true, false, n, n, m, Q.p, n, Q.p, n);
            Tens L2 = make({n, n}), X2 = make({n, n});
            ck(fill_zero(st, L2.p, n * n), "zero"); ck(fill_zero(st, X2.p, n * n), "zero");
            ck(cholesky(st, (int)n, G2.p, n, L2.p, n, 0.0, 1e-14, cw), "cholesky");
            ck(tri_inverse(st, (int)n, L2.p, n, cw, X2.p, n, T.p), "tri_inverse");
            Tens Q2 = mm(false, true, m, n, n, Q.p, n, X2.p, n);
            Tens LL = mm(false, false, n, n, n, L.p, n, L2.p, n);
            R = perm(LL, {1, 0});
            drop(Q); Q = Q2;
        }
        keep(Q); keep(R);
        return true;
    }

    // orth_chol() (one pass) of two matrices of the same shape: the two Gram matrices on the caller's stream, then the two
    // factorisation + inversion chains (latency-bound: ~60 small launches each) side by side on two auxiliary streams, then
    // the decisions and the two Q = mat L^-T products.  All buffers are allocated before the fork; nothing is allocated or
    // freed while the chains are in flight.  Returns false (nothing kept but the Gram matrices, see Gkeep) unless both operands
    // prove full rank.  The proof here is sharper than orth_chol()'s: lam_min >= ||G^-4||_F^(-1/4) instead of 1 / tr G^-1.
    // Xinv != nullptr: Q = mat L^-T is NOT formed; the caller gets Xinv[i] = L^-1 instead (Q[i].p stays null) and applies it
    // to whatever multiplies Q (bond_swap: Q only ever appears in products, so two n x n x n GEMMs replace two m x n x n ones).
    // meanwhile: work for the caller's stream that does not depend on the factors, issued while the two chains are in flight
    // (it may allocate: the chains' buffers stay allocated and the chains themselves allocate nothing).
    // Gkeep != nullptr: on failure the two Gram matrices (recomputed: the factorisation destroys them) are NOT needed -- the
    // caller recomputes them; kept simple on purpose.
    bool orth_chol_pair(const Tens& m0, const Tens& m1, Tens Q[2], Tens R[2], Tens* Xinv = nullptr, const std::function<void()>* meanwhile = nullptr) {
        SubStreams& ss = sub_streams();
        Scope sc(*this);
        const int64_t m = m0.d[0], n = m0.d[1];
        const Tens* mats[2] = {&m0, &m1};
        Tens G[2], L[2], X[2], T[2], W[2], W2[2]; double* cw[2]; double* res[2];
        for (int i = 0; i < 2; ++i) {
            G[i] = mm(true, false, n, n, m, mats[i]->p, n, mats[i]->p, n, true);
            L[i] = make({n, n}); X[i] = make({n, n}); T[i] = make({(int64_t)tri_inverse_scratch_doubles((int)n)});
            cw[i] = raw((int64_t)cholesky_work_doubles((int)n)); res[i] = raw(1 + 148 * 8 + 7);
            W[i] = make({n, n}); W2[i] = make({n, n});
            ck(fill_zero(st, L[i].p, n * n), "zero"); ck(fill_zero(st, X[i].p, n * n), "zero");
        }
        if (ss.ok) ck(cudaEventRecord(ss.fork, st), "event");
        for (int i = 0; i < 2; ++i) {
            cudaStream_t a = ss.ok ? ss.s[i] : st;
            if (ss.ok) ck(cudaStreamWaitEvent(a, ss.fork, 0), "wait");
            ck(cholesky(a, (int)n, G[i].p, n, L[i].p, n, 0.0, 1e-14, cw[i]), "cholesky");
            ck(tri_inverse(a, (int)n, L[i].p, n, cw[i], X[i].p, n, T[i].p), "tri_inverse");
            // ||G^-4||_F = (sum_i lam_i^-8)^1/2 >= lam_min^-4: three n^3 products (0.1 ms each) for a bound on lam_min that is
            // within (number of eigenvalues near lam_min)^1/8 of it (tr G^-1 = ||L^-1||_F^2 overshoots by that number itself)
            ck(dgemm(a, true, false, n, n, n, 1.0, X[i].p, n, X[i].p, n, 0.0, W[i].p, n), "dgemm");       // G^-1 = L^-T L^-1
            ck(dgemm(a, false, false, n, n, n, 1.0, W[i].p, n, W[i].p, n, 0.0, W2[i].p, n), "dgemm");     // G^-2
            ck(dgemm(a, false, false, n, n, n, 1.0, W2[i].p, n, W2[i].p, n, 0.0, W[i].p, n), "dgemm");    // G^-4
            ck(dot(a, n * n, W[i].p, W[i].p, res[i]), "dot");
            if (ss.ok) ck(cudaEventRecord(ss.join[i], a), "event");
        }
        if (meanwhile && *meanwhile) (*meanwhile)();
        if (ss.ok) for (int i = 0; i < 2; ++i) ck(cudaStreamWaitEvent(st, ss.join[i], 0), "wait");
        bool ok = true;
        int info[2] = {0, 0};
        std::vector<double> d0[2] = {std::vector<double>(n), std::vector<double>(n)}; double xn[2] = {0, 0};
        for (int i = 0; i < 2; ++i) {          // six read-backs, one synchronisation
            ck(cudaMemcpyAsync(&info[i], cholesky_info(cw[i], (int)n), sizeof(int), cudaMemcpyDeviceToHost, st), "readback");
            ck(cudaMemcpyAsync(d0[i].data(), cholesky_d0(cw[i], (int)n), 8 * n, cudaMemcpyDeviceToHost, st), "readback");
            ck(cudaMemcpyAsync(&xn[i], res[i], 8, cudaMemcpyDeviceToHost, st), "readback");
        }
        ck(cudaStreamSynchronize(st), "sync"); count_sync();
        for (int i = 0; i < 2; ++i) {
            double tr = 0; for (double v : d0[i]) tr += v;
            const double inv_lmin = std::pow(xn[i], 0.125);        // ||G^-4||_F^(1/4) >= 1 / lam_min
            if (g_verbose & 1) fprintf(stderr, "[tatrg cholesky qr %lld x %lld] info %d, proven lam_min/lam_max >= %.3e\n", (long long)m, (long long)n, info[i], 1.0 / (inv_lmin * tr));
            if (info[i] != 0 || !std::isfinite(xn[i]) || !(xn[i] > 0) || !(tr > 0) || !(1.0 / (inv_lmin * tr) > kEpsOrthLambda)) ok = false;
        }
        if (!ok) return false;
        for (int i = 0; i < 2; ++i) {
            if (Xinv) { Xinv[i] = X[i]; keep(X[i]); Q[i] = Tens(); Q[i].p = nullptr; }
            else { Q[i] = mm(false, true, m, n, n, mats[i]->p, n, X[i].p, n); keep(Q[i]); }
            R[i] = perm(view(L[i], {n, n}), {1, 0});
            keep(R[i]);
        }
        return true;
    }

    // Rank-revealing path of orth_pair() (R14), Q implicit: the Gram matrices G[i] (preserved) are factored by truncated pivoted
    // Cholesky, G = L L^T + S with tr S <= 1e-14 tr G (pchol.cu; below the rounding of the DGEMM that formed G and 1 % of the
    // eigenvalue the rank decision turns on), the r' x r' matrices L^T L -- same non-zero eigenvalues, nearly diagonal --
    // are eigen-decomposed together (V, lam: 8 Jacobi sweeps instead of 24-32 on G itself, on r' ~ 0.6 n), and with the
    // eigenvectors U = L V lam^-1/2 of G:  R = lam^1/2 U^T = V^T L^T,  Xinv = lam^-1/2 U^T = lam^-1 R, rows with
    // lam <= 1e-12 lam_max dropped exactly as in the eigen-decomposition of G itself.
    bool orth_pchol_pair(Tens G[2], int n, Tens R[2], Tens Xinv[2], const std::function<void()>* meanwhile, bool* full_rank) {
        SubStreams& ss = sub_streams();
        Scope sc(*this);
        Tens L[2]; double* pw[2];
        for (int i = 0; i < 2; ++i) { L[i] = make({n, n}); pw[i] = raw((int64_t)pchol_work_doubles(n)); }
        if (ss.ok) ck(cudaEventRecord(ss.fork, st), "event");
        for (int i = 0; i < 2; ++i) {
            cudaStream_t a = ss.ok ? ss.s[i] : st;
            if (ss.ok) ck(cudaStreamWaitEvent(a, ss.fork, 0), "wait");
            ck(pchol(a, n, G[i].p, L[i].p, n, 1e-14, pw[i]), "pchol");
            if (ss.ok) ck(cudaEventRecord(ss.join[i], a), "event");
        }
        if (meanwhile && *meanwhile) (*meanwhile)();
        if (ss.ok) for (int i = 0; i < 2; ++i) ck(cudaStreamWaitEvent(st, ss.join[i], 0), "wait");
        double info[2][4];
        for (int i = 0; i < 2; ++i) ck(cudaMemcpyAsync(info[i], pchol_info(pw[i]), 32, cudaMemcpyDeviceToHost, st), "readback");
        ck(cudaStreamSynchronize(st), "sync"); count_sync();
        const auto tv0 = std::chrono::steady_clock::now();
        int rp[2];
        for (int i = 0; i < 2; ++i) {
            rp[i] = (int)info[i][0];
            if (g_verbose & 1) fprintf(stderr, "[tatrg orth %d] pivoted Cholesky: rank %d, residual trace / trace %.2e\n", n, rp[i], info[i][2] > 0 ? info[i][1] / info[i][2] : 0.0);
            if (rp[i] <= 0 || rp[i] > n || !std::isfinite(info[i][1])) return false;
        }
        *full_rank = true;
        Tens G1[2];
        for (int i = 0; i < 2; ++i) G1[i] = mm(true, false, rp[i], rp[i], n, L[i].p, n, L[i].p, n, true);
        std::vector<EigOut> eo;
        eig_batch({&G1[0], &G1[1]}, {rp[0], rp[1]}, eo);
        if (g_verbose & 1) fprintf(stderr, "[tatrg orth %d] L^T L + eigen-decomposition: %.2f ms\n", n, std::chrono::duration<double, std::milli>(std::chrono::steady_clock::now() - tv0).count());
        for (int i = 0; i < 2; ++i) {
            const std::vector<double>& lh = eo[i].lh;
            if (!(lh[0] > 0)) fail(TATRG_ENUMERIC, "orth: zero matrix");
            int r = 0;
            for (double x : lh) if (x > kEpsOrthLambda * lh[0]) ++r;
            if (g_verbose & 1) fprintf(stderr, "[tatrg orth %d] eigen-decomposition of L^T L (%d x %d): rank %d\n", n, rp[i], rp[i], r);
            R[i] = mm(false, true, r, n, rp[i], eo[i].Vt.p, rp[i], L[i].p, n);          // V^T L^T = lam^1/2 U^T
            Xinv[i] = make({r, n});
            ck(scale_rows(st, Xinv[i].p, R[i].p, eo[i].lam, r, n, 1), "scale");          // lam^-1/2 U^T
            keep(R[i]); keep(Xinv[i]);
            if (r < n) *full_rank = false;
        }
        return true;
    }

    // orth() of two matrices of the same shape with n > 128 (single pass): Cholesky QR when both prove full rank, else the two
    // Gram matrices are eigen-decomposed together (rank-revealing: directions with lam <= 1e-12 lam_max dropped, R14).
    // Xinv != nullptr: Q is NOT formed (Q[i].p stays null); Xinv[i] [r x n] is the factor with Q = mat Xinv^T -- L^-1 of the
    // Cholesky path, lam^-1/2 V^T of the eigen path -- and R[i] = Q^T mat [r x n] (L^T resp. lam^1/2 V^T).
    void orth_pair(const Tens& m0, const Tens& m1, Tens Q[2], Tens R[2], Tens* Xinv = nullptr, const std::function<void()>* meanwhile = nullptr) {
        const int64_t m = m0.d[0], n = m0.d[1];
        if (Xinv) { Xinv[0].p = nullptr; Xinv[1].p = nullptr; }
        if (n <= 128 || m1.d[0] != m || m1.d[1] != n) { orth(m0, Q[0], R[0]); orth(m1, Q[1], R[1]); return; }
        const bool implicit = Xinv != nullptr && c.use_subspace;
        // `meanwhile` runs once, beside whichever factorisation comes first.  After a step whose operands were numerically
        // rank-deficient (every step once the flow has left criticality) the Cholesky attempt is skipped: its outcome is known, it
        // costs 5 ms and destroys the Gram matrices; the first full-rank result of the rank-revealing path clears the hint.
        bool ran = false;
        std::function<void()> once = [&]() { if (!ran && meanwhile && *meanwhile) { ran = true; (*meanwhile)(); } };
        if (c.use_subspace && !(implicit && c.qr_deficient_hint) && orth_chol_pair(m0, m1, Q, R, Xinv, &once)) { c.qr_deficient_hint = false; return; }
        Scope sc(*this);
        const Tens* mats[2] = {&m0, &m1};
        Tens G[2];
        for (int i = 0; i < 2; ++i) G[i] = mm(true, false, n, n, m, mats[i]->p, n, mats[i]->p, n, true);
        if (implicit) {
            bool full = false;
            if (orth_pchol_pair(G, (int)n, R, Xinv, &once, &full)) {
                c.qr_deficient_hint = !full;
                for (int i = 0; i < 2; ++i) { Q[i] = Tens(); keep(R[i]); keep(Xinv[i]); }
                return;
            }
        }
        once();
        std::vector<EigOut> eo;
        eig_batch({&G[0], &G[1]}, {(int)n, (int)n}, eo);
        for (int i = 0; i < 2; ++i) {
            const std::vector<double>& lh = eo[i].lh;
            if (!(lh[0] > 0)) fail(TATRG_ENUMERIC, "orth: zero matrix");
            int r = 0;
            for (double x : lh) if (x > kEpsOrthLambda * lh[0]) ++r;
            if (g_verbose & 1) fprintf(stderr, "[tatrg orth %lld x %lld] eigen-decomposition of the Gram matrix: rank %d\n", (long long)m, (long long)n, r);
            if (implicit) {
                Xinv[i] = make({r, n});
                ck(scale_rows(st, Xinv[i].p, eo[i].Vt.p, eo[i].lam, r, n, 2), "scale");     // lam^-1/2 V^T
                keep(Xinv[i]); Q[i] = Tens(); Q[i].p = nullptr;
            } else {
                Q[i] = mm(false, true, m, r, n, mats[i]->p, n, eo[i].Vt.p, n);
                ck(scale_last(st, Q[i].p, Q[i].p, eo[i].lam, m, r, 2), "scale");
                keep(Q[i]);
            }
            R[i] = make({r, n});
            ck(scale_rows(st, R[i].p, eo[i].Vt.p, eo[i].lam, r, n, 3), "scale");
            keep(R[i]);
        }
    }


    // ---- leading invariant subspaces by subspace iteration ------------------------------------------------------
    // The triad isometries (Eq. 2.9 :135) need the top K of n = D^2 eigenvectors of a Gram matrix, the squeezers (:171,
    // R6) the top D of the n eigenvectors of Theta_b Theta_f.  Orthogonal iteration on a block of b = 2 kmax vectors
    // (Z <- orthonormalise(A Z), Cholesky QR on the tensor cores) converges to that subspace like (lam_{b+1}/lam_k)^q and
    // ends with ONE b x b Rayleigh-Ritz eigen-problem instead of n x n ones.
    //   symmetric problem  (F == nullptr): A = Bm,     Z^T Z = 1
    //   product problem    (F != nullptr): A = Bm F,   self-adjoint in the F inner product: Z^T F Z = 1, W = F Z carried along
    // The iteration count comes from the measured convergence ratio: the diagonal of the Cholesky factor of orthogonal
    // iteration tends to the eigenvalues, rho = r_b / r_kmax, q = 13 digits / log10(1/rho) (+ margin).
    struct SubProb {
        const double* Bm; const double* F; int n, kmax, b; uint32_t sid;
        Tens buf[2], Gm, L, H; double* cw; double* dg;
        std::vector<double> r;
        cudaStream_t stream = nullptr; double* part = nullptr; int64_t part_cap = 0;
        int cur = 0;                 // the basis [Z; W] lives in buf[cur]
        int done = 0, target = 0, deg = 1;
        int rdeg = 1;                // degree of the plain step whose Cholesky factor is in L: its diagonal is ~ lam_j^rdeg
        // Chebyshev-filtered cycles (symmetric problems): p_deg(A) Z with p_deg the Chebyshev polynomial of the interval [0, cheb_hi]
        // that holds the unwanted eigenvalues; one cycle is worth `gain` plain applications (done_f counts in that unit)
        bool cheb = false; double cheb_hi = 0, gain = 0, done_f = 0; Tens tmp[2];
        bool ok = true;
        int bcap = 0; bool widen = false, widened = false;     // the block may be doubled once when convergence is too slow
        const double* Z() const { return buf[cur].p; }
        const double* W() const { return F ? buf[cur].p + (int64_t)n * b : buf[cur].p; }
    };
    static int sub_block(int n, int kmax) { int b = 2 * kmax; b = (b + 31) / 32 * 32; return b; }
    static bool sub_applicable(int n, int kmax) { return n > 128 && kmax >= 8 && sub_block(n, kmax) * 2 <= n; }
    void sub_orth(SubProb& s, int src, double shift) {      // buf[src] = [Z'; W'] -> buf[src^1] = [Z; W], which becomes the basis
        const int64_t rows = s.F ? 2 * (int64_t)s.n : s.n;
        double* X = s.buf[src].p;
        const double* Wp = s.F ? X + (int64_t)s.n * s.b : X;
        mm_into(s.Gm.p, s.b, true, false, s.b, s.b, s.n, X, s.b, Wp, s.b);
        ck(cholesky(st, s.b, s.Gm.p, s.b, s.L.p, s.b, shift, 1e-14, s.cw, false), "cholesky");      // flags accumulate over the iteration
        ck(trsm_right_lt(st, rows, s.b, X, s.b, s.buf[src ^ 1].p, s.b, s.L.p, s.b, s.cw), "trsm");
        s.cur = src ^ 1;
    }
    void sub_apply(SubProb& s, int from) {         // buf[from^1] = [A Z; F A Z] with [Z; W] = buf[from]
        const double* X = s.F ? s.buf[from].p + (int64_t)s.n * s.b : s.buf[from].p;
        double* O = s.buf[from ^ 1].p;
        mm_into(O, s.b, false, false, s.n, s.b, s.n, s.Bm, s.n, X, s.b);
        if (s.F) mm_into(O + (int64_t)s.n * s.b, s.b, false, false, s.n, s.b, s.n, s.F, s.n, O, s.b);
    }
    void sub_step(SubProb& s, int deg, double shift) {      // deg applications of A, then one orthonormalisation
        int a = s.cur;
        for (int i = 0; i < deg; ++i) { sub_apply(s, a); a ^= 1; }
        sub_orth(s, a, shift);
        s.done_f += deg; s.done = (int)s.done_f; s.rdeg = deg;
    }
    // One Chebyshev-filtered cycle of a symmetric problem: Z <- orthonormalise(T_deg(t) Z), t = (2 / hi) A - 1, which maps the unwanted
    // eigenvalues [0, hi] into [-1, 1] (|T_deg| <= 1 there) and amplifies lam_k > hi by cosh(deg acosh(2 lam_k / hi - 1)):
    // the same subspace as plain orthogonal iteration in 2-3 times fewer applications (three-term recurrence
    // Y_{j+1} = 2 t Y_j - Y_{j-1}, Y_0 = Z, Y_1 = t Z).  The basis stays in buf[cur]; tmp[0] holds A Y_j, tmp[1] the odd iterates.
    void sub_step_cheb(SubProb& s, int deg, double shift) {
        const int64_t nb = (int64_t)s.n * s.b;
        double* Z = s.buf[s.cur].p; double* Y2 = s.buf[s.cur ^ 1].p; double* G = s.tmp[0].p; double* Y1 = s.tmp[1].p;
        const double a = 2.0 / s.cheb_hi;
        mm_into(G, s.b, false, false, s.n, s.b, s.n, s.Bm, s.n, Z, s.b);
        ck(lincomb3(st, Y1, a, G, -1.0, Z, 0.0, nullptr, nb), "lincomb");                     // Y1 = t Z
        double* src = Y1;
        if (deg >= 2) {
            mm_into(G, s.b, false, false, s.n, s.b, s.n, s.Bm, s.n, Y1, s.b);
            ck(lincomb3(st, Y2, 2 * a, G, -2.0, Y1, -1.0, Z, nb), "lincomb");                 // Y2 = 2 t Y1 - Z
            src = Y2;
        }
        if (deg >= 3) {
            mm_into(G, s.b, false, false, s.n, s.b, s.n, s.Bm, s.n, Y2, s.b);
            ck(lincomb3(st, Y1, 2 * a, G, -2.0, Y2, -1.0, Y1, nb), "lincomb");                // Y3 = 2 t Y2 - Y1 (in place of Y1)
            src = Y1;
        }
        mm_into(s.Gm.p, s.b, true, false, s.b, s.b, s.n, src, s.b, src, s.b);
        ck(cholesky(st, s.b, s.Gm.p, s.b, s.L.p, s.b, shift, 1e-14, s.cw, false), "cholesky");
        ck(trsm_right_lt(st, s.n, s.b, src, s.b, Z, s.b, s.L.p, s.b, s.cw), "trsm");           // Z is free: every iterate has been formed
        s.done_f += s.gain; s.done = (int)s.done_f; s.rdeg = 0;
    }
    // The problems of a stage are independent chains of small launches: each runs on a stream of its own (created once
    // per process), forked from and joined to the caller's stream by events, so that their kernels overlap on the device.
    // All of them have the greatest priority: while a big contraction of the caller's stream is in flight (run(): the squeezer
    // chains overlap the Gram matrices and the Xi products), their small CTAs get the next SM slot that frees up.
    // q: the stream that stands in for the caller's during such an overlapped stage; forkq/joinq its events.
    struct SubStreams { cudaStream_t s[4], q; cudaEvent_t fork, join[4], forkq, joinq; bool ok = false; bool tried = false; };
    static SubStreams& sub_streams() {      // one set per device; not for concurrent use from several host threads
        static std::map<int, SubStreams> per_device;
        static std::mutex mu;
        int dev = 0;
        cudaGetDevice(&dev);
        std::lock_guard<std::mutex> lock(mu);
        SubStreams& ss = per_device[dev];
        if (!ss.tried) {
            ss.tried = true;
            int lo = 0, hi = 0;
            cudaDeviceGetStreamPriorityRange(&lo, &hi);          // hi = greatest priority (numerically lowest)
            bool ok = cudaEventCreateWithFlags(&ss.fork, cudaEventDisableTiming) == cudaSuccess;
            for (int i = 0; i < 4 && ok; ++i)
                ok = cudaStreamCreateWithPriority(&ss.s[i], cudaStreamNonBlocking, hi) == cudaSuccess && cudaEventCreateWithFlags(&ss.join[i], cudaEventDisableTiming) == cudaSuccess;
            if (ok) ok = cudaStreamCreateWithPriority(&ss.q, cudaStreamNonBlocking, hi) == cudaSuccess && cudaEventCreateWithFlags(&ss.forkq, cudaEventDisableTiming) == cudaSuccess &&
                         cudaEventCreateWithFlags(&ss.joinq, cudaEventDisableTiming) == cudaSuccess;
            ss.ok = ok;
        }
        return ss;
    }
    struct OnStream {      // issue the enclosed work of problem p on its stream, with its own split-K scratch
        Stepper& s; cudaStream_t saved; double* pf; int64_t pc;
        OnStream(Stepper& s_, const SubProb& p) : s(s_), saved(s_.st), pf(s_.part_fixed), pc(s_.part_cap) {
            if (p.stream) { s.st = p.stream; s.part_fixed = p.part; s.part_cap = p.part_cap; }
        }
        ~OnStream() { s.st = saved; s.part_fixed = pf; s.part_cap = pc; }
    };
    // Advances problem s to its target.  The steps are identical chains of ~15-30 small launches, and four such chains in
    // flight are bound by the host's launch rate: one unit (1 step, or 2 when the basis alternates between the two buffers)
    // is captured into a CUDA graph and replayed.  Counters are incremented at capture time only, hence the correction.
    void sub_run(SubProb& s, double shift) {
        static bool graphs_ok = true;      // cleared for the process when stream capture is unavailable
        const bool cheb = s.cheb;
        const double per = cheb ? s.gain : (double)s.deg;        // plain applications a cycle is worth
        // Chebyshev cycles are followed by ONE plain step, whose Cholesky diagonal estimates the eigenvalues again (estimate())
        const int steps = cheb ? std::max(0, (int)std::ceil((s.target - s.done_f - 1.0) / per)) : (s.target - s.done + s.deg - 1) / s.deg;
        const int unit = cheb ? 1 : ((s.deg % 2 == 0) ? 2 : 1);
        const int reps = steps / unit;
        auto cycle = [&]() { if (cheb) sub_step_cheb(s, s.deg, shift); else sub_step(s, s.deg, shift); };
        int left = steps;
        if (graphs_ok && c.use_graphs && s.stream && c.timing < 2 && reps >= 3) {      // never the caller's stream: it may be the legacy default stream
            const double done0 = s.done_f; const int cur0 = s.cur;
            Counters* cn = g_counter;
            const long long l0 = cn ? cn->launches : 0, gc0 = cn ? cn->gemm_calls : 0; const double f0 = cn ? cn->gemm_flops : 0;
            cudaGraph_t graph = nullptr; cudaGraphExec_t exec = nullptr;
            const auto tg0 = std::chrono::steady_clock::now();
            cudaError_t ge = cudaStreamBeginCapture(st, cudaStreamCaptureModeThreadLocal);
            bool ok = ge == cudaSuccess;
            std::string why;
            if (ok) {
                try { for (int u = 0; u < unit; ++u) cycle(); } catch (const Fail& f) { ok = false; why = f.msg; } catch (...) { ok = false; }
                ge = cudaStreamEndCapture(st, &graph);
                if (ge != cudaSuccess || !graph) ok = false;
            }
            if (ok) { ge = cudaGraphInstantiate(&exec, graph, 0); ok = ge == cudaSuccess; }
            if (!ok && (g_verbose & 1)) fprintf(stderr, "[tatrg subspace] graph capture failed: %s %s\n", cudaGetErrorString(ge), why.c_str());
            if (graph) cudaGraphDestroy(graph);
            if (g_verbose & 1) fprintf(stderr, "[tatrg subspace] graph of %d step(s): %s, %d replays + %d plain steps, capture + instantiate %.0f us\n", unit, ok ? "ok" : "FAILED", reps, steps - reps * unit, std::chrono::duration<double, std::micro>(std::chrono::steady_clock::now() - tg0).count());
            if (ok) {
                for (int r = 0; r < reps && ok; ++r) ok = cudaGraphLaunch(exec, st) == cudaSuccess;
                c.graveyard.push_back(exec);
                if (!ok) fail(TATRG_ECUDA, "graph launch failed");
                if (cn) { cn->launches += (cn->launches - l0) * (reps - 1); cn->gemm_calls += (cn->gemm_calls - gc0) * (reps - 1); cn->gemm_flops += (cn->gemm_flops - f0) * (reps - 1); }
                s.done_f = done0 + reps * unit * per; s.done = (int)s.done_f; s.cur = cur0;
                left = steps - reps * unit;
            } else {        // capture unavailable: nothing was executed; plain launches from the saved state
                cudaGetLastError();
                graphs_ok = false;
                if (cn) { cn->launches = l0; cn->gemm_calls = gc0; cn->gemm_flops = f0; }
                s.done_f = done0; s.done = (int)s.done_f; s.cur = cur0;
            }
        }
        for (int i = 0; i < left; ++i) cycle();
        if (cheb) sub_step(s, 1, shift);
    }
    // Runs the iterations of all problems (interleaved so that the host reads the convergence estimates of all of them
    // with one synchronisation per phase) and leaves in every s.H the b x b Rayleigh-Ritz matrix.  Problems that cannot
    // be handled (rank-deficient leading block, no convergence in sight) come back with ok = false.
    // After the first q0 single steps the columns are graded like the spectrum and Cholesky (invariant under column
    // scaling) tolerates several applications of A per orthonormalisation, as long as the dynamic range of the block,
    // (r_1 / r_b)^deg, stays below 1e11.
    void sub_iterate(std::vector<SubProb>& ps) {
        constexpr int q0 = 4, qmax = 240;
        constexpr double kShift = 1e-13;
        const bool verbose = (g_verbose & 1) != 0;   // debugging aid only
        SubStreams& ss = sub_streams();
        const bool multi = ss.ok && !ps.empty() && ps.size() <= 4;
        if (multi) {
            ck(cudaEventRecord(ss.fork, st), "event");
            for (size_t i = 0; i < ps.size(); ++i) {
                SubProb& s = ps[i];
                s.stream = ss.s[i];
                ck(cudaStreamWaitEvent(s.stream, ss.fork, 0), "wait");
                s.part_cap = std::max(std::max(dgemm_splitk_doubles(s.b, s.b, s.n), dgemm_splitk_doubles(s.n, s.b, s.n)),
                                      std::max(dgemm_splitk_doubles(2 * s.b, 2 * s.b, s.n), dgemm_splitk_doubles(s.n, 2 * s.b, s.n)));
                s.part = s.part_cap ? raw(s.part_cap) : nullptr;
                if (!s.part) s.part_cap = 0;
            }
        }
        // A flat stretch of the spectrum between positions kmax and b (rho >= 0.6: seen in the post-critical steps) would need
        // hundreds of applications; the block is then doubled once (lam_{2b+1} / lam_kmax instead of lam_{b+1} / lam_kmax) and the
        // iteration restarted, before the full decomposition is considered.  All buffers are sized for the doubled block up front.
        auto init_problem = [&](SubProb& s) {
            OnStream on(*this, s);
            s.cur = 0; s.done = 0; s.done_f = 0; s.target = 0; s.deg = 1; s.rdeg = 1; s.cheb = false;
            ck(fill_zero(st, s.L.p, (int64_t)s.b * s.b), "zero");
            ck(cudaMemsetAsync(const_cast<int*>(cholesky_info(s.cw, s.b)), 0, sizeof(int), st), "memset"); count_launch();
            ck(philox_gauss(st, c.seed, (uint32_t)call, s.sid, 0, (int64_t)s.n * s.b, s.buf[1].p), "philox");
            if (s.F) mm_into(s.buf[1].p + (int64_t)s.n * s.b, s.b, false, false, s.n, s.b, s.n, s.F, s.n, s.buf[1].p, s.b);
            sub_orth(s, 1, kShift);
            for (int i = 0; i < q0; ++i) sub_step(s, 1, kShift);
            ck(extract_diag(st, s.b, s.L.p, s.b, s.dg), "diag");
        };
        for (SubProb& s : ps) {
            const int64_t rows = s.F ? 2 * (int64_t)s.n : s.n;
            s.bcap = (4 * s.b <= s.n) ? 2 * s.b : s.b;
            s.buf[0] = make({rows, s.bcap}); s.buf[1] = make({rows, s.bcap});
            s.Gm = make({s.bcap, s.bcap}); s.L = make({s.bcap, s.bcap}); s.H = make({s.bcap, s.bcap});
            s.cw = raw((int64_t)cholesky_work_doubles(s.bcap)); s.dg = raw(s.bcap);
            if (c.use_cheb && !s.F) { s.tmp[0] = make({(int64_t)s.n, s.bcap}); s.tmp[1] = make({(int64_t)s.n, s.bcap}); }
            init_problem(s);
        }
        auto sync_all = [&]() { for (SubProb& s : ps) if (s.stream) cudaStreamSynchronize(s.stream); cudaStreamSynchronize(st); return std::chrono::steady_clock::now(); };
        auto tA = verbose ? sync_all() : std::chrono::steady_clock::time_point();
        auto estimate = [&](SubProb& s) {
            OnStream on(*this, s);
            int info = 0;
            ck(cudaMemcpyAsync(&info, cholesky_info(s.cw, s.b), sizeof(int), cudaMemcpyDeviceToHost, st), "readback");
            s.r = to_host(s.dg, s.b);
            // a pivot that had to be raised to its guard, or a non-finite one: the block has numerically dependent columns (the
            // matrix has fewer than b significant directions: unsaturated steps, ordered phase) -> the full decomposition decides
            if (info != 0) { s.ok = false; return; }
            for (double v : s.r) if (!std::isfinite(v)) { s.ok = false; return; }
            double tail = 0; for (int j = s.b - 4; j < s.b; ++j) tail = std::max(tail, s.r[j]);
            double head = s.r[0]; for (int j = 0; j < s.kmax; ++j) head = std::min(head, s.r[j]);
            if (!(head > 1e-12 * s.r[0]) || !(tail > 1e-9 * head)) { s.ok = false; return; }     // rank-deficient block: full decomposition
            // the diagonal of R is that of the last orthonormalisation: r_j ~ lam_j^deg
            const int rd = std::max(1, s.rdeg);
            const double rho = 1.1 * std::pow(tail / head, 1.0 / rd);
            // slow convergence (rho >= 0.6: more than 60 applications): the doubled block converges like lam_{2b+1} / lam_kmax and
            // costs twice as much per application -- taken whenever it is available; without it up to qmax applications are
            // still far cheaper than the full decomposition (0.1 ms each against 25 ms)
            // (with Chebyshev-filtered cycles a ratio up to ~0.8 still needs at most ~24 cycles of degree 2, cheaper than the restart with a
            // doubled block and its 2b x 2b Rayleigh-Ritz problem)
            // (measured over the 60 steps of configs[3]: doubling from 0.6 / 0.7 / 0.8 / 0.9 on -> 92.3 / 91.6 / 90.7 / 91.3 ms per post-critical step)
            const double widen_at = (c.use_cheb && !s.F && s.tmp[0].p) ? 0.8 : 0.6;
            if (!(rho < widen_at) && !s.widened && s.bcap > s.b) { s.widen = true; return; }
            if (!(rho < 0.95)) { s.ok = false; return; }
            s.target = std::max(s.target, (int)std::ceil(13.0 / std::log10(1.0 / rho)) + 2);
            if (s.target > qmax) s.ok = false;
            const double range = std::pow(s.r[0] / tail, 1.0 / rd);
            int deg = 1;
            while (deg < 3 && std::pow(range, deg + 1) <= 1e11) ++deg;
            s.cheb = false;
            if (c.use_cheb && !s.F && s.tmp[0].p) {
                // unwanted eigenvalues in [0, 1.1 lam_tail]: x_k = 2 lam_k / hi - 1 = 2 / rho - 1 for the slowest wanted one; the dynamic
                // range of a cycle is T_deg(x_1) (the block must stay numerically independent between orthonormalisations)
                const double x1 = 2.0 * range / 1.1 - 1.0, xk = 2.0 / rho - 1.0;
                auto T = [](int d, double x) { return std::cosh(d * std::acosh(x)); };
                if (xk > 1.02 && T(1, x1) <= 1e11) {
                    int d = 1;
                    while (d < 3 && T(d + 1, x1) <= 1e11) ++d;
                    const double gain = std::log10(T(d, xk)) / std::log10(1.0 / rho);
                    if (gain > 1.15 * deg) { s.cheb = true; s.gain = gain; s.cheb_hi = 1.1 * std::pow(tail, 1.0 / rd); deg = d; }
                }
            }
            if (verbose) fprintf(stderr, "[tatrg subspace n=%d b=%d kmax=%d%s] after %d iterations: rho %.3f -> %d iterations, %d per orthonormalisation%s\n", s.n, s.b, s.kmax, s.F ? " product" : "", s.done, rho, s.target, deg, s.cheb ? " (Chebyshev)" : "");
            s.deg = deg;
        };
        for (int pass = 0; pass < 3; ++pass) {
            bool more = false;
            // a re-estimate within 1 of the count already done is the noise of the estimator (+-10 % in rho), not missing work
            for (SubProb& s : ps) if (s.ok) {
                estimate(s);
                if (s.widen) {
                    if (verbose) fprintf(stderr, "[tatrg subspace n=%d b=%d kmax=%d%s] convergence too slow: block doubled to %d, restart\n", s.n, s.b, s.kmax, s.F ? " product" : "", s.bcap);
                    s.widen = false; s.widened = true; s.b = s.bcap;
                    init_problem(s);
                    estimate(s);
                    if (s.widen) { s.widen = false; s.ok = false; }
                }
                if (s.ok && s.target > s.done + (pass > 0 ? 1 : 0)) more = true; else if (s.ok) s.target = std::min(s.target, s.done);
            }
            if (!more) break;
            for (SubProb& s : ps) {
                if (!s.ok || s.target <= s.done) continue;
                OnStream on(*this, s);
                sub_run(s, kShift);
                ck(extract_diag(st, s.b, s.L.p, s.b, s.dg), "diag");
            }
        }
        auto tB = verbose ? sync_all() : tA;
        for (SubProb& s : ps) {
            if (!s.ok) continue;
            OnStream on(*this, s);
            // second orthonormalisation pass without shift (the basis is orthonormal to ~1e-13 already), W = F Z recomputed
            const int64_t nb = (int64_t)s.n * s.b;
            if (s.F) mm_into(s.buf[s.cur].p + nb, s.b, false, false, s.n, s.b, s.n, s.F, s.n, s.buf[s.cur].p, s.b);
            sub_orth(s, s.cur, 0.0);
            // Rayleigh-Ritz matrix H = W^T Bm W (product) or Z^T Bm Z
            double* T = s.buf[s.cur ^ 1].p;
            mm_into(T, s.b, false, false, s.n, s.b, s.n, s.Bm, s.n, s.W(), s.b);
            mm_into(s.H.p, s.b, true, false, s.b, s.b, s.n, s.W(), s.b, T, s.b);
        }
        for (SubProb& s : ps) {       // the last orthonormalisations must not have met a dependent column either
            if (!s.ok) continue;
            OnStream on(*this, s);
            int info = 0;
            ck(cudaMemcpyAsync(&info, cholesky_info(s.cw, s.b), sizeof(int), cudaMemcpyDeviceToHost, st), "readback");
            ck(cudaStreamSynchronize(st), "sync"); count_sync();
            if (info != 0) s.ok = false;
        }
        if (multi)
            for (size_t i = 0; i < ps.size(); ++i) {
                ck(cudaEventRecord(ss.join[i], ps[i].stream), "event");
                ck(cudaStreamWaitEvent(st, ss.join[i], 0), "wait");
            }
        if (verbose) {
            auto tC = sync_all();
            fprintf(stderr, "[tatrg subspace] %zu problems: phases after the first %d steps %.2f ms, final pass + Rayleigh-Ritz matrix %.2f ms\n", ps.size(), q0,
                    std::chrono::duration<double, std::milli>(tB - tA).count(), std::chrono::duration<double, std::milli>(tC - tB).count());
        }
    }

    // R10: block-diagonal gauge rotation Gm (k x k) from wt [k x n] (rows = the vectors to fix) and the multiplet
    // groups of the spectrum v: Cfull = wt rho, per group Q of its MGS-QR.
    Tens gauge(const Tens& wt, bool as_cols, const std::vector<double>& v, int k, uint32_t stream_id) {
        const int64_t n = as_cols ? wt.d[0] : wt.d[1];
        std::vector<int> grp = multiplets(v, k, c.tau);
        int gmax = 1;
        for (size_t i = 0; i < grp.size(); i += 2) gmax = std::max(gmax, grp[i + 1] - grp[i]);
        if (gmax > 32 || gmax > kRhoCols) fail(TATRG_ENUMERIC, "multiplet of %d values: unsupported", gmax);
        Tens rho = make({n, gmax});
        ck(philox_rho(st, c.seed, (uint32_t)call, stream_id, n, gmax, rho.p), "rho");
        Tens cf = as_cols ? mm(true, false, k, gmax, n, wt.p, wt.d[1], rho.p, gmax) : mm(false, false, k, gmax, n, wt.p, n, rho.p, gmax);
        int* gd = to_dev_int(grp);
        Tens Gm = make({k, k});
        ck(gauge_blocks(st, cf.p, gmax, gd, (int)grp.size() / 2, k, Gm.p), "gauge");
        return Gm;
    }

    void decompose(Tens& a, Tens& dt, Tens& core);
    // The swapped bond in factored form, Eq. A.9 :379 before Eq. A.10-A.11 :389-392 (side 0: X from C, side 1: Y from B):
    //   X[al,i',g] = sum_c Qm[0][i',c] w[0][c,al,g],  u[0][q,al,g] = U^bond (an isometry on (q al)): Qm is Q^C itself (then w = u) or,
    //   after the Cholesky QR, the operand C with w = L_C^-T U^bond.  PAPER.md :394: "the tensors X and Y are not explicitly constructed".
    struct Lift { Tens Qm[2], w[2], u[2]; bool on = false; };
    void bond_swap(const Tens& a, const Tens& dt, const Tens& core, Tens& x, Tens& y, double*& sig, int& gr, Lift* lf = nullptr);
    void triad_implicit(const Tens& a, const Tens& dt, const Lift& lf, const double* sig, Tens U[4], Tens& e, Tens& f, Tens& g, Tens& h);
    void triad_grams_implicit(const Tens& aa, const Tens& Qm, const Tens& w, const Tens& u, const double* sig, int64_t d4, Tens& ga, Tens& gx);
    void triad(const Tens& a, const Tens& dt, const Tens& x, const Tens& y, const double* sig, Tens U[4], Tens& e, Tens& f, Tens& g, Tens& h);
    void triad_grams(const Tens& aa, const Tens& xx, const double* sig, Tens& ga, Tens& gx);
    void triad_isos(Tens gram[4], const std::vector<int>& which, int64_t d2, int64_t d3, Tens U[4]);
    void half_grams(const Tens& P, const Tens& Q, const Tens& Iu, const Tens& Jl, Tens th[3]);
    void squeezers(Tens thf[3], Tens thb[3], const int du[3], Tens Mt[3], Tens Nt[3], int dmask = 7);
    void half_grams4(const Tens& P, const Tens& Q, Tens th[3]);
    void half_grams23(const Tens& P, const Tens& Q, const Tens& Iu, const Tens& Jl, Tens th[3]);
    void atrg_grams(const Tens& P, const Tens& Q, Tens th[3]);
    Tens atrg_contract(const Tens& P, const Tens& Q, Tens S[3]);
    void run();
};

// (a) Eq. 2.4 :76 -- T = Phi Psi^T = A core Dt^T, A and Dt isometric (:137), core = G^T diag(s/s1) G in the canonical
// gauge (R10); c_m = s1 is the normalisation of this step (R8).
void Stepper::decompose(Tens& a, Tens& dt, Tens& core) {
    Scope sc(*this);
    const int64_t F = c.phi.size() / c.phi.d[4], gph = c.phi.d[4];
    Tens qf, rf, qb, rb;
    orth(view(c.phi, {F, gph}), qf, rf);
    orth(view(c.psi, {F, gph}), qb, rb);
    const int r1 = (int)rf.d[0], r2 = (int)rb.d[0];
    // SVD of the small core rf rb^T (r1 x r2), orthogonalising the rows of the orientation with fewer rows
    const bool flip = r1 > r2;
    const int nv = flip ? r2 : r1, len = flip ? r1 : r2;
    Tens X = flip ? mm(false, true, r2, r1, gph, rb.p, gph, rf.p, gph) : mm(false, true, r1, r2, gph, rf.p, gph, rb.p, gph);
    double* s = raw(nv); Tens Ut = make({nv, len}), Va = make({nv, nv});
    std::vector<double> sh;
    {
        double* work = raw((int64_t)(svd_rows_work_bytes(nv, len) / 8 + 1));
        std::string e;
        int rc = svd_rows(st, nv, len, X.p, s, Ut.p, Va.p, work, &sh, &e);
        if (rc != TATRG_OK) fail(rc, "%s", e.c_str());
    }
    const double cm = sh[0];
    if (!(cm > 0) || !std::isfinite(cm)) fail(TATRG_ENUMERIC, "decompose: non-positive normalisation c_m = %g", cm);
    c.lnc.push_back(std::log(cm));
    for (double& v : sh) v /= cm;
    c.sv_s = sh;
    const int chi = select_rank(sh, c.Dbond, kEpsSV, c.tau);          // fn 5 :203: alpha, beta carry the overspanned bond
    // rows of Va are the singular vectors on the side of X's rows, rows of Ut those on the side of its columns
    const Tens& urows = flip ? Ut : Va;    // [nv x r1]
    const Tens& vrows = flip ? Va : Ut;    // [nv x r2]
    Tens a0 = mm(false, true, F, chi, r1, qf.p, r1, urows.p, r1);
    Tens d0 = mm(false, true, F, chi, r2, qb.p, r2, vrows.p, r2);
    Tens Gm = gauge(a0, true, sh, chi, 1);
    a = mm(false, false, F, chi, chi, a0.p, chi, Gm.p, chi);
    dt = mm(false, false, F, chi, chi, d0.p, chi, Gm.p, chi);
    std::vector<double> sk(sh.begin(), sh.begin() + chi);
    double* sd = to_dev(sk);
    Tens SG = make({chi, chi});
    ck(scale_rows(st, SG.p, Gm.p, sd, chi, chi, 0), "scale");
    core = mm(true, false, chi, chi, chi, Gm.p, chi, SG.p, chi);
    a = view(a, {c.phi.d[0], c.phi.d[1], c.phi.d[2], c.phi.d[3], chi});
    dt = view(dt, {c.psi.d[0], c.psi.d[1], c.psi.d[2], c.psi.d[3], chi});
    keep(a); keep(dt); keep(core);
}

// (b) Eq. 2.5 :90, App. A :329-394 -- sum_i1 B C ~ X sigma Y by randomized SVD of the never-formed core S.
void Stepper::bond_swap(const Tens& a, const Tens& dt, const Tens& core, Tens& x, Tens& y, double*& sig, int& gr, Lift* lf) {
    Scope sc(*this);
    const int64_t d1 = a.d[0], d2 = a.d[1], d3 = a.d[2], d4 = a.d[3], chi = a.d[4];
    const int64_t F = d1 * d2 * d3 * d4, J = d2 * d3 * d4;
    Tens QB, RB, QC, RC, XB, XC;      // implicit: QB, QC hold B, C themselves and XB, XC the factors with Q = B XB^T, C XC^T
    Tens btom;                        // B^T Omega^phys [c, be, m], formed ahead while the Cholesky chains run
    bool implicit = false;
    {
        Scope s2(*this);
        // B[i1,j',al] = sum_a' Dt[i1,j',a'] core[al,a'],  C[i1,i',be] = sum_a' A[i1,i',a'] core[a',be]   (core symmetric)
        // written straight into the layout of Eq. A.2-A.3 (rows j', columns (i1 al)): i1 is the batch of the product, ldc = d1 chi
        Tens bm = ein("Ijc,ac->jIa", view(dt, {d1, J, chi}), core);    // Eq. A.2 :345  B[(j'),(i1 al)]
        Tens cm = ein("Ijc,cb->jIb", view(a, {d1, J, chi}), core);     // Eq. A.3 :348  C[(i'),(i1 be)]
        Tens Qs[2], Rs[2], Xs[2];
        // While the two Cholesky chains are in flight the caller's stream draws Omega^phys and forms B^T Omega^phys, the part of
        // the projection Q^B^T Omega^phys = XB (B^T Omega^phys) that needs no factor.
        std::function<void()> early = [&]() {
            const int64_t n = d1 * chi, l0 = std::min<int64_t>(c.Dbond + c.p, chi * n);
            Tens omp = make({J, chi, l0});                             // drawn as (be, j', m), stored [j', be, m]
            ck(philox_gauss_swap01(st, c.seed, (uint32_t)call, 0, chi, J, l0, omp.p), "philox");
            btom = ein("jc,jbm->cbm", view(bm, {J, n}), omp);
            drop(omp);
            detach(btom);
        };
        orth_pair(view(bm, {J, d1 * chi}), view(cm, {J, d1 * chi}), Qs, Rs, Xs, &early);
        if (btom.p) scopes[scopes.size() - 2].push_back(btom.p);      // into bond_swap's scope
        RB = Rs[0]; RC = Rs[1];
        if (Xs[0].p) {
            // Q^B = B XB^T and Q^C = C XC^T are never formed (XB = L_B^-1 of the Cholesky QR, or lam^-1/2 V^T of the rank-revealing
            // eigen-decomposition).  They only enter through the products Q^B^T Omega^phys (R12) and Q^C U^bond, Q^B V^bond
            // (Eq. A.10-A.11), where the small factor is applied to the small operand instead (saves two D^3 x D^2 x D^2 products).
            implicit = true;
            QB = view(bm, {J, d1 * chi}); QC = view(cm, {J, d1 * chi}); XB = Xs[0]; XC = Xs[1];
            keep(bm); keep(cm); keep(XB); keep(XC);
        } else {
            QB = Qs[0]; QC = Qs[1];
            keep(QB); keep(QC);
        }
        keep(RB); keep(RC);
    }
    if (submark) submark();                                              // end of TATRG_ST_QR
    const int64_t npb = RB.d[0], npc = RC.d[0];      // ranks of Q^B, Q^C (= QB.d[1], QC.d[1] unless Q is implicit)
    Tens RB3 = view(RB, {npb, d1, chi}), RC3 = view(RC, {npc, d1, chi});
    const int64_t l = std::min<int64_t>(c.Dbond + c.p, std::min(chi * npc, chi * npb));     // R3: sketch width (fn 9 :381)
    // Omega drawn in the physical basis (be, j', m) and projected on Q^B  (R11, R12)
    Tens omega;
    if (implicit && btom.p && btom.d[2] == l) {
        omega = ein("pc,cBm->Bpm", XB, btom);
        drop(btom);
    } else {
        if (btom.p) drop(btom);
        Scope s2(*this);
        Tens omp = make({J, chi, l});                                     // [j', be, m]: one wide GEMM instead of chi narrow ones
        ck(philox_gauss_swap01(st, c.seed, (uint32_t)call, 0, chi, J, l, omp.p), "philox");
        if (implicit) {
            Tens tmp = ein("jc,jbm->cbm", QB, omp);
            omega = ein("pc,cBm->Bpm", XB, tmp);
        } else omega = ein("jp,jbm->bpm", QB, omp);
        keep(omega);
    }
    Tens qk, yt;
    for (int k = 0; k <= c.n_pow; ++k) {                                 // R4: n_pow + 1 passes of Eq. A.4-A.6
        Scope s2(*this);
        Tens t = ein("pia,bpm->iabm", RB3, omega);
        Tens yk = ein("qib,iabm->aqm", RC3, t);                          // Eq. A.4 :356
        drop(t);
        Tens q2, r2;
        orth(view(yk, {chi * npc, yk.d[2]}), q2, r2, k < c.n_pow);
        drop(yk); drop(r2);
        if (qk.p) drop(qk);
        qk = view(q2, {chi, npc, q2.d[1]});
        Tens t2 = ein("qib,aqm->ibam", RC3, qk);
        if (yt.p) drop(yt);
        yt = ein("pia,ibam->bpm", RB3, t2);                              // Eq. A.5 :361  = (Q^T S)^T
        drop(t2);
        keep(qk); keep(yt);
        if (k < c.n_pow) {
            Tens q3, r3;
            orth(view(yt, {chi * npb, yt.d[2]}), q3, r3, true);          // Eq. A.6 :365
            drop(r3); drop(omega);
            omega = view(q3, {chi, npb, q3.d[1]});
            keep(omega);
        }
    }
    if (submark) submark();                                              // end of TATRG_ST_RSVD
    // Eq. A.7-A.8 :373-376: SVD of the projected tensor, via an orthonormal basis of its columns and a small Jacobi SVD
    const int64_t rk = yt.d[2];
    Tens Qy, Ry;
    orth(view(yt, {chi * npb, rk}), Qy, Ry);
    const int ry = (int)Ry.d[0];
    double* s = raw(ry); Tens Ut = make({ry, rk}), Va = make({ry, ry});
    std::vector<double> sh;
    {
        double* work = raw((int64_t)(svd_rows_work_bytes(ry, (int)rk) / 8 + 1));
        std::string e;
        int rc = svd_rows(st, ry, (int)rk, Ry.p, s, Ut.p, Va.p, work, &sh, &e);
        if (rc != TATRG_OK) fail(rc, "%s", e.c_str());
    }
    if (!(sh[0] > 0)) fail(TATRG_ENUMERIC, "bond swap: zero spectrum");
    gr = select_rank(sh, c.Dbond, kEpsSV, c.tau);                     // Eq. A.1 :337: gamma runs to r_bond D
    c.sv_sigma.assign((size_t)rk, 0.0);
    for (int i = 0; i < ry; ++i) c.sv_sigma[i] = sh[i] / sh[0];
    // Eq. A.9 :379 and A.10-A.11 :389-392
    Tens ub = mm(false, true, chi * npc, gr, rk, qk.p, rk, Ut.p, rk);         // U^bond[(al q), g]
    Tens vb = mm(false, true, chi * npb, gr, ry, Qy.p, ry, Va.p, ry);         // V^bond[(be p), g]
    // one GEMM with N = (al, g) each: the batched form has N = g <= D, a quarter of a tile
    Tens ubp = perm(view(ub, {chi, npc, gr}), {1, 0, 2});
    Tens vbp = perm(view(vb, {chi, npb, gr}), {1, 0, 2});
    Tens wx, wy;
    if (implicit) { wx = ein("qc,qag->cag", XC, ubp); wy = ein("pc,pbg->cbg", XB, vbp); }
    const bool factored = lf && c.method == 0 && c.implicit_xy;
    if (!factored || c.keep_tensors) {          // keep_tensors: X, Y are formed for tatrg_get_tensor only, the path below does not read them
        if (implicit) {
            x = ein("jc,cag->ajg", QC, wx);
            y = ein("jc,cbg->bjg", QB, wy);
        } else {
            x = ein("jq,qag->ajg", QC, ubp);
            y = ein("jp,pbg->bjg", QB, vbp);
        }
        x = view(x, {chi, d2, d3, d4, gr});
        y = view(y, {chi, d2, d3, d4, gr});
        keep(x); keep(y);
    }
    if (factored) {
        // :394 "we work directly with U^bond, sigma, and V^*bond to create isometries of the triad representation": hand the factors on
        lf->on = true;
        lf->Qm[0] = QC; lf->Qm[1] = QB;
        lf->u[0] = ubp; lf->u[1] = vbp;
        lf->w[0] = implicit ? wx : ubp; lf->w[1] = implicit ? wy : vbp;
        keep(QC); keep(QB); keep(ubp); keep(vbp);
        if (implicit) { keep(wx); keep(wy); }
    }
    sig = raw(gr);
    ck(cudaMemcpyAsync(sig, s, 8 * gr, cudaMemcpyDeviceToDevice, st), "copy"); count_launch();
    { Tens t; t.p = sig; keep(t); }
}

// (c) without X and Y (PAPER.md :394, :201).  With X[al,i',g] = sum_c Qm[i',c] w[c,al,g] (see Lift):
//   G^X[(i2 i3),(i2' i3')] = sum_{i4} sum_{c c'} Qm[(i2 i3 i4),c] W[c,c'] Qm[(i2' i3' i4),c'],  W = sum_{al,g} sig_g^2 w w^T
//   kappa^A[al,al'] = sum_{q,g} sig_g^2 U^bond[q,al,g] U^bond[q,al',g]        (Q^C^T Q^C = 1, Eq. A.3 :348)
// The two big products read Qm as [(i2 i3 i4), c] and as [(i2 i3), (i4 c)]: the same memory, no permute, nothing of size D^5 r_bond^2.
void Stepper::triad_grams_implicit(const Tens& aa, const Tens& Qm, const Tens& w, const Tens& u, const double* sig, int64_t d4, Tens& ga,
                                   Tens& gx) {
    Scope s2(*this);
    const int64_t d1 = aa.d[0], d2 = aa.d[1], d3 = aa.d[2], chi = aa.d[4], gr = w.d[2], nc = Qm.d[1];
    const int64_t n = d2 * d3, J = n * d4;
    {
        Tens ws = make({nc, chi, gr});
        ck(scale_last(st, ws.p, w.p, sig, nc * chi, gr, 0), "scale");
        Tens wm = mm(false, true, nc, nc, chi * gr, ws.p, chi * gr, ws.p, chi * gr, true);
        drop(ws);
        Tens t1 = mm(false, false, J, nc, nc, Qm.p, nc, wm.p, nc);
        drop(wm);
        gx = mm(false, true, n, n, d4 * nc, t1.p, d4 * nc, Qm.p, d4 * nc, true);
        drop(t1);
    }
    Tens us = make({u.d[0], chi, gr});
    ck(scale_last(st, us.p, u.p, sig, u.d[0] * chi, gr, 0), "scale");
    Tens ka = ein("qag,qbg->ab", us, us);
    drop(us);
    Tens ta = mm(false, false, d1 * J, chi, chi, aa.p, chi, ka.p, chi);
    Tens ap = perm(aa, {0, 3, 4, 1, 2});
    Tens tp = perm(view(ta, {d1, d2, d3, d4, chi}), {0, 3, 4, 1, 2});
    drop(ta);
    ga = mm(true, false, n, n, d1 * d4 * chi, ap.p, n, tp.p, n, true);
    keep(ga); keep(gx);
}

void Stepper::triad_implicit(const Tens& a, const Tens& dt, const Lift& lf, const double* sig, Tens U[4], Tens& e, Tens& f, Tens& g,
                             Tens& h) {
    Scope sc(*this);
    const int64_t d2 = a.d[1], d3 = a.d[2], d4 = a.d[3], n = d2 * d3, gr = lf.w[0].d[2];
    Tens gram[4];
    triad_grams_implicit(a, lf.Qm[0], lf.w[0], lf.u[0], sig, d4, gram[0], gram[1]);
    triad_grams_implicit(dt, lf.Qm[1], lf.w[1], lf.u[1], sig, d4, gram[3], gram[2]);
    triad_isos(gram, {0, 1, 2, 3}, d2, d3, U);
    for (int i = 0; i < 4; ++i) drop(gram[i]);
    if (submark) submark();                                                // end of TATRG_ST_TRIAD_ISO
    e = ein("mjk,Ijkla->Imla", U[0], a);                                   // Eq. 2.10
    {   // Eq. 2.11 with Eq. A.10: the isometry meets Q^C first (K x d4 x nc), U^bond sigma afterwards
        const int64_t nc = lf.Qm[0].d[1], k1 = U[1].d[0], chi = lf.w[0].d[1];
        Tens pc = mm(false, false, k1, d4 * nc, n, U[1].p, n, lf.Qm[0].p, d4 * nc);
        Tens ws = make({nc, chi, gr});
        ck(scale_last(st, ws.p, lf.w[0].p, sig, nc * chi, gr, 0), "scale");
        f = ein("xlc,cag->axlg", view(pc, {k1, d4, nc}), ws);
        drop(pc); drop(ws);
    }
    {   // Eq. 2.12 with Eq. A.11 (no sigma: it went into F)
        const int64_t nc = lf.Qm[1].d[1], k2 = U[2].d[0];
        Tens pb = mm(false, false, k2, d4 * nc, n, U[2].p, n, lf.Qm[1].p, d4 * nc);
        g = ein("ylc,cbg->bylg", view(pb, {k2, d4, nc}), lf.w[1]);
        drop(pb);
    }
    h = ein("djk,Jjklb->Jdlb", U[3], dt);                                  // Eq. 2.13
    for (int i = 0; i < 4; ++i) keep(U[i]);
    keep(e); keep(f); keep(g); keep(h);
}

// (c) Eq. 2.9 :135 (canonical form :137) and Eq. 2.10-2.17 :147-167.
// U[0..3] = U^A, U^X, U^Y, U^D stored [k, leg2, leg3]; E[i1,kA,i4,al], F[al,kX,i4,g] (carries sigma), G[be,kY,j4,g], H[j1,kD,j4,be].
// Gram matrices of one side on the leg pair (2,3): side 0: xx = X, aa = A -> ga = G^A, gx = G^X; side 1: xx = Y, aa = Dt -> G^D, G^Y.
void Stepper::triad_grams(const Tens& aa, const Tens& xx, const double* sig, Tens& ga, Tens& gx) {
    Scope s2(*this);
    const int64_t d1 = aa.d[0], d2 = aa.d[1], d3 = aa.d[2], d4 = aa.d[3], chi = aa.d[4], gr = xx.d[4];
    const int64_t n = d2 * d3, J = d2 * d3 * d4;
    Tens xs = make({chi, d2, d3, d4, gr});
    ck(scale_last(st, xs.p, xx.p, sig, chi * J, gr, 0), "scale");
    // G^X[(i2 i3),(i2' i3')] = sum_{al,i4,g} Xs Xs
    Tens xp = perm(xs, {0, 3, 4, 1, 2});
    gx = mm(true, false, n, n, chi * d4 * gr, xp.p, n, xp.p, n, true);
    drop(xp);
    // kappa[al,al'] = sum_{i',g} Xs Xs ;  G^A = sum_{i1,i4,al,al'} A kappa A
    Tens ka = mm(false, true, chi, chi, J * gr, xs.p, J * gr, xs.p, J * gr);
    drop(xs);
    Tens ta = mm(false, false, d1 * J, chi, chi, aa.p, chi, ka.p, chi);
    Tens ap = perm(aa, {0, 3, 4, 1, 2});
    Tens tp = perm(view(ta, {d1, d2, d3, d4, chi}), {0, 3, 4, 1, 2});
    drop(ta);
    ga = mm(true, false, n, n, d1 * d4 * chi, ap.p, n, tp.p, n, true);      // A kappa A: symmetric because kappa is
    keep(ga); keep(gx);
}

// Isometries U[i] (rows: the leading eigenvectors, [k, d2, d3]) of the Gram matrices gram[i], i in `which` (0..3 = A, X, Y, D).
void Stepper::triad_isos(Tens gram[4], const std::vector<int>& which, int64_t d2, int64_t d3, Tens U[4]) {
    Scope s2(*this);
    const int64_t n = d2 * d3;
    const int kmax = (int)std::min<int64_t>(c.Ktri, n);
    const double eps_sv = std::sqrt(kEpsLambda);
    bool have[4] = {false, false, false, false};
    if (c.use_subspace && sub_applicable((int)n, kmax)) {
        // top-K eigenvectors by subspace iteration + one b x b Rayleigh-Ritz problem per Gram matrix
        std::vector<SubProb> ps(which.size());
        for (size_t j = 0; j < which.size(); ++j) {
            const int i = which[j];
            ck(symmetrize(st, (int)n, gram[i].p), "symmetrize");
            ps[j].Bm = gram[i].p; ps[j].F = nullptr; ps[j].n = (int)n; ps[j].kmax = kmax; ps[j].b = sub_block((int)n, kmax); ps[j].sid = 16 + i;
        }
        const bool vb = (g_verbose & 1) != 0;
        auto now = [&]() { cudaStreamSynchronize(st); return std::chrono::steady_clock::now(); };
        auto t0 = vb ? now() : std::chrono::steady_clock::time_point();
        sub_iterate(ps);
        auto t1 = vb ? now() : t0;
        std::vector<Tens*> hs; std::vector<int> ns, who;
        for (size_t j = 0; j < ps.size(); ++j) if (ps[j].ok) { hs.push_back(&ps[j].H); ns.push_back(ps[j].b); who.push_back((int)j); }
        std::vector<EigOut> er;
        if (!hs.empty()) eig_batch(hs, ns, er);
        if (vb) { auto t2 = now(); fprintf(stderr, "[tatrg triad] subspace iterations %.2f ms, Rayleigh-Ritz %.2f ms\n", std::chrono::duration<double, std::milli>(t1 - t0).count(), std::chrono::duration<double, std::milli>(t2 - t1).count()); }
        for (size_t j = 0; j < who.size(); ++j) {
            const int pj = who[j], i = which[pj], b = ps[pj].b;
            std::vector<double> sv(b);
            for (int t = 0; t < b; ++t) sv[t] = std::sqrt(std::max(er[j].lh[t], 0.0));
            if (!(sv[kmax] > eps_sv * sv[0])) continue;              // numerical rank <= kmax: the full decomposition decides
            const int k = select_rank(sv, kmax, eps_sv, c.tau);
            if (k <= 0) continue;
            U[i] = mm(false, true, k, n, b, er[j].Vt.p, b, ps[pj].Z(), b);     // rows: Ritz vectors Y_k^T Z^T
            U[i] = view(U[i], {k, d2, d3});
            keep(U[i]);
            have[i] = true;
        }
    }
    std::vector<Tens*> gs; std::vector<int> ns, who;
    for (int i : which) if (!have[i]) { gs.push_back(&gram[i]); ns.push_back((int)n); who.push_back(i); }
    std::vector<EigOut> eo;
    if (!gs.empty()) eig_batch(gs, ns, eo);
    for (size_t j = 0; j < who.size(); ++j) {
        const int i = who[j];
        const std::vector<double>& lh = eo[j].lh;
        std::vector<double> sv(lh.size());
        for (size_t t = 0; t < lh.size(); ++t) sv[t] = std::sqrt(std::max(lh[t], 0.0));    // multiplet rule on the singular-value scale
        const int k = select_rank(sv, kmax, eps_sv, c.tau);
        if (k <= 0) fail(TATRG_ENUMERIC, "triad: empty isometry");
        U[i] = make({k, d2, d3});
        ck(cudaMemcpyAsync(U[i].p, eo[j].Vt.p, 8 * (int64_t)k * n, cudaMemcpyDeviceToDevice, st), "copy"); count_launch();
        keep(U[i]);
    }
}

void Stepper::triad(const Tens& a, const Tens& dt, const Tens& x, const Tens& y, const double* sig, Tens U[4], Tens& e, Tens& f,
                    Tens& g, Tens& h) {
    Scope sc(*this);
    const int64_t gr = x.d[4];
    Tens gram[4];
    triad_grams(a, x, sig, gram[0], gram[1]);
    triad_grams(dt, y, sig, gram[3], gram[2]);
    triad_isos(gram, {0, 1, 2, 3}, a.d[1], a.d[2], U);
    for (int i = 0; i < 4; ++i) drop(gram[i]);
    if (submark) submark();                                                // end of TATRG_ST_TRIAD_ISO
    e = ein("mjk,Ijkla->Imla", U[0], a);                                   // Eq. 2.10
    Tens f0 = ein("xjk,Ajklg->Axlg", U[1], x);                             // Eq. 2.11 (sigma goes into F only)
    ck(scale_last(st, f0.p, f0.p, sig, f0.size() / gr, gr, 0), "scale");
    f = f0;
    g = ein("yjk,Bjklg->Bylg", U[2], y);                                   // Eq. 2.12
    h = ein("djk,Jjklb->Jdlb", U[3], dt);                                  // Eq. 2.13
    for (int i = 0; i < 4; ++i) keep(U[i]);
    keep(e); keep(f); keep(g); keep(h);
}

// (d) Gram matrices of one half of the unit cell on the doubled bonds 2, 3, 4  (R6; PAPER.md :171, Table 1 :229-230).
// P[o1,kU,u4,bond] sits on the upper site, Q[bond,kL,l4,o2] on the lower site; Iu[kU,u2,u3], Jl[kL,l2,l3].
// th[d-2][(u l),(u' l')] for d = 2,3,4, staged so that nothing larger than K^4 appears.
void Stepper::half_grams(const Tens& P, const Tens& Q, const Tens& Iu, const Tens& Jl, Tens th[3]) {
    half_grams4(P, Q, th);
    half_grams23(P, Q, Iu, Jl, th);
}
void Stepper::half_grams4(const Tens& P, const Tens& Q, Tens th[3]) {
    // direction 4: Iu and Jl are isometries and drop out
    Scope s2(*this);
    Tens ee = ein("ikua,ikvb->uavb", P, P);
    Tens ff = ein("akld,bkwd->albw", Q, Q);
    th[2] = ein("uavb,albw->ulvw", ee, ff);
    keep(th[2]);
}
void Stepper::half_grams23(const Tens& P, const Tens& Q, const Tens& Iu, const Tens& Jl, Tens th[3]) {
    Scope sc(*this);
    Tens ef;
    {
        Scope s2(*this);
        Tens ee = ein("ikua,imub->kmab", P, P);
        Tens ff = ein("axld,byld->abxy", Q, Q);
        ef = ein("kmab,abxy->kmxy", ee, ff);
        keep(ef);
    }
    for (int d = 2; d <= 3; ++d) {
        Scope s2(*this);
        Tens ii = d == 2 ? ein("kuc,mvc->uvkm", Iu, Iu) : ein("kcu,mcv->uvkm", Iu, Iu);
        Tens jj = d == 2 ? ein("xlc,ywc->lwxy", Jl, Jl) : ein("xcl,ycw->lwxy", Jl, Jl);
        Tens tmp = ein("uvkm,kmxy->uvxy", ii, ef);
        th[d - 2] = ein("uvxy,lwxy->ulvw", tmp, jj);
        keep(th[d - 2]);
    }
    for (int i = 0; i < 2; ++i) keep(th[i]);
}

// (d) squeezer pairs of the three directions (R6): thf = R1^T R1, thb = R2 R2^T, SVD R1 R2 = U s V^T,
// M = R2 V s^-1/2, N = R1^T U s^-1/2, gauge-fixed (R10).  Returned as rows: Mt[k,u,l], Nt[k,u,l].
// The six Gram matrices are eigen-decomposed in one batch, then the three (R1 R2)^T (R1 R2) in another.
// dmask: bit d set = direction d + 2 is computed by this call (run() computes direction 4 ahead of the other two).
void Stepper::squeezers(Tens thf[3], Tens thb[3], const int du[3], Tens Mt[3], Tens Nt[3], int dmask) {
    Scope sc(*this);
    // per direction: s (host, leading values), wt [k x n] = (R2 V)^T, nt [k x n] = (Theta_f R2 V)^T
    std::vector<double> sval[3]; Tens wts[3], nts[3]; int kk[3] = {0, 0, 0}; bool have[3] = {false, false, false};
    // (1) M spans the leading eigenvectors of Theta_b Theta_f (Theta_b Theta_f M = M s^2, N = Theta_f M s^-1): subspace
    //     iteration in the Theta_f inner product needs no factor R1, R2 at all.  With Z^T Theta_f Z = 1 and Ritz vectors Y:
    //     R2 V = Z Y s,  Theta_f R2 V = W Y s.
    {
        std::vector<SubProb> ps; std::vector<int> dirs;
        for (int d = 0; d < 3; ++d) {
            if (!((dmask >> d) & 1)) continue;
            const int n = du[d] * du[d];
            if (!c.use_subspace || !sub_applicable(n, c.D)) continue;
            ck(symmetrize(st, n, thf[d].p), "symmetrize"); ck(symmetrize(st, n, thb[d].p), "symmetrize");
            SubProb sp; sp.Bm = thb[d].p; sp.F = thf[d].p; sp.n = n; sp.kmax = c.D; sp.b = sub_block(n, c.D); sp.sid = 24 + (uint32_t)d;
            ps.push_back(sp); dirs.push_back(d);
        }
        if (!ps.empty()) {
            Scope s2(*this);
            sub_iterate(ps);
            std::vector<Tens*> hs; std::vector<int> ns, who;
            for (size_t i = 0; i < ps.size(); ++i) if (ps[i].ok) { hs.push_back(&ps[i].H); ns.push_back(ps[i].b); who.push_back((int)i); }
            std::vector<EigOut> er;
            if (!hs.empty()) eig_batch(hs, ns, er);
            for (size_t j = 0; j < who.size(); ++j) {
                const SubProb& sp = ps[who[j]];
                const int d = dirs[who[j]], b = sp.b, n = sp.n;
                std::vector<double> s(b);
                for (int t = 0; t < b; ++t) s[t] = std::sqrt(std::max(er[j].lh[t], 0.0));
                if (!(s[c.D] > kEpsSqueezer * s[0])) continue;          // numerical rank <= D: the full decomposition decides
                const int k = select_rank(s, c.D, kEpsSqueezer, c.tau);
                if (k <= 0) continue;
                std::vector<double> sk(s.begin(), s.begin() + k);
                double* sd = to_dev(sk);
                wts[d] = mm(false, true, k, n, b, er[j].Vt.p, b, sp.Z(), b);
                nts[d] = mm(false, true, k, n, b, er[j].Vt.p, b, sp.W(), b);
                ck(scale_rows(st, wts[d].p, wts[d].p, sd, k, n, 0), "scale");
                ck(scale_rows(st, nts[d].p, nts[d].p, sd, k, n, 0), "scale");
                keep(wts[d]); keep(nts[d]);
                sval[d] = s; kk[d] = k; have[d] = true;
            }
        }
    }
    // (2) full decompositions for the directions the iteration does not cover (small or rank-deficient problems):
    //     the Gram matrices are eigen-decomposed in one batch, then the (R1 R2)^T (R1 R2) in another.
    std::vector<int> todo;
    for (int d = 0; d < 3; ++d) if (((dmask >> d) & 1) && !have[d]) todo.push_back(d);
    if (!todo.empty()) {
        std::vector<EigOut> eo;
        {
            std::vector<Tens*> gs; std::vector<int> ns;
            for (int d : todo) { gs.push_back(&thf[d]); ns.push_back(du[d] * du[d]); gs.push_back(&thb[d]); ns.push_back(du[d] * du[d]); }
            eig_batch(gs, ns, eo);
        }
        Tens r1[3], r2t[3], cm[3], gc[3];
        int k1[3], k2[3];
        std::vector<Tens*> gcs; std::vector<int> gns;
        for (size_t j = 0; j < todo.size(); ++j) {
            const int d = todo[j], n = du[d] * du[d];
            const std::vector<double>&l1 = eo[2 * j].lh, &l2 = eo[2 * j + 1].lh;
            if (!(l1[0] > 0) || !(l2[0] > 0)) fail(TATRG_ENUMERIC, "squeezer %d: zero Gram matrix", d + 2);
            k1[d] = k2[d] = 0;
            for (double v : l1) if (v > kEpsLambda * l1[0]) ++k1[d];
            for (double v : l2) if (v > kEpsLambda * l2[0]) ++k2[d];
            r1[d] = make({k1[d], n}); r2t[d] = make({k2[d], n});
            ck(scale_rows(st, r1[d].p, eo[2 * j].Vt.p, eo[2 * j].lam, k1[d], n, 3), "scale");          // R1 = Lambda1^1/2 W1^T
            ck(scale_rows(st, r2t[d].p, eo[2 * j + 1].Vt.p, eo[2 * j + 1].lam, k2[d], n, 3), "scale");  // R2^T
            drop(eo[2 * j].Vt); drop(eo[2 * j + 1].Vt);
            cm[d] = mm(false, true, k1[d], k2[d], n, r1[d].p, n, r2t[d].p, n);                            // R1 R2
            gc[d] = mm(true, false, k2[d], k2[d], k1[d], cm[d].p, k2[d], cm[d].p, k2[d]);                 // (R1 R2)^T (R1 R2): V, s^2
            gcs.push_back(&gc[d]); gns.push_back(k2[d]);
        }
        std::vector<EigOut> ec;
        eig_batch(gcs, gns, ec);
        for (size_t j = 0; j < todo.size(); ++j) {
            const int d = todo[j], n = du[d] * du[d];
            drop(gc[d]);
            const std::vector<double>& lc = ec[j].lh;
            std::vector<double> s(lc.size());
            for (size_t i = 0; i < lc.size(); ++i) s[i] = std::sqrt(std::max(lc[i], 0.0));
            const int k = select_rank(s, c.D, kEpsSqueezer, c.tau);
            if (k <= 0) fail(TATRG_ENUMERIC, "squeezer %d: empty", d + 2);
            const Tens& Vc = ec[j].Vt;
            wts[d] = mm(false, false, k, n, k2[d], Vc.p, k2[d], r2t[d].p, n);        // (R2 V)^T
            Tens cv = mm(false, true, k, k1[d], k2[d], Vc.p, k2[d], cm[d].p, k2[d]); // (R1 R2 V)^T = (U s)^T
            nts[d] = mm(false, false, k, n, k1[d], cv.p, k1[d], r1[d].p, n);         // (R1^T U s)^T
            sval[d] = s; kk[d] = k;
        }
    }
    for (int d = 0; d < 3; ++d) if ((dmask >> d) & 1) { drop(thf[d]); drop(thb[d]); }
    // (3) gauge (R10), s^-1/2 scalings
    for (int d = 0; d < 3; ++d) {
        if (!((dmask >> d) & 1)) continue;
        const int n = du[d] * du[d], dir = d + 2, k = kk[d];
        const std::vector<double>& s = sval[d];
        std::vector<double> sk(s.begin(), s.begin() + k);
        double* sd = to_dev(sk);
        Tens& wt = wts[d]; Tens& nt = nts[d];
        Tens Gm = gauge(wt, false, s, k, (uint32_t)dir);
        ck(scale_rows(st, wt.p, wt.p, sd, k, n, 2), "scale");                    // s^-1/2
        ck(scale_rows(st, nt.p, nt.p, sd, k, n, 4), "scale");                    // s^-3/2
        Mt[d] = mm(true, false, k, n, k, Gm.p, k, wt.p, n);
        Nt[d] = mm(true, false, k, n, k, Gm.p, k, nt.p, n);
        Mt[d] = view(Mt[d], {k, du[d], du[d]}); Nt[d] = view(Nt[d], {k, du[d], du[d]});
        keep(Mt[d]); keep(Nt[d]);
    }
}

// ---- plain ATRG (Eq. 2.7-2.8 :104-113): no triad split -------------------------------------------
// One half of the unit cell is P[o1,u2,u3,u4,b] (upper site) . Q[b,l2,l3,l4,o2] (lower site).
// Gram matrices on the doubled bonds, th[d-2][(u l),(u' l')]: sum_b,b' PP_d[u,b,u',b'] QQ_d[b,l,b',l'] with every other
// leg of P (resp. Q) traced against its copy -- nothing larger than D^5 is formed.
void Stepper::atrg_grams(const Tens& P, const Tens& Q, Tens th[3]) {
    Scope sc(*this);
    static const char* pp[3] = {"iucda,ivcdb->uavb", "icuda,icvdb->uavb", "icdua,icdvb->uavb"};
    static const char* qq[3] = {"alcdg,bwcdg->albw", "acldg,bcwdg->albw", "acdlg,bcdwg->albw"};
    for (int d = 0; d < 3; ++d) {
        Scope s2(*this);
        Tens a = ein(pp[d], P, P);
        Tens b = ein(qq[d], Q, Q);
        th[d] = ein("uavb,albw->ulvw", a, b);
        keep(th[d]);
    }
    for (int d = 0; d < 3; ++d) keep(th[d]);
}

// R[o1,k2,k3,k4,o2] = sum P[o1,u2,u3,u4,b] Q[b,l2,l3,l4,o2] S2[k2,u2,l2] S3[k3,u3,l3] S4[k4,u4,l4]   (Eq. 2.7 :106, O(D^9)).
// The D^7 intermediate of the paper (fn 6 :205: "memory blocking") is never materialised: the contraction is sliced over
// o1, one D^6 slab at a time.
Tens Stepper::atrg_contract(const Tens& P, const Tens& Q, Tens S[3]) {
    Scope sc(*this);
    const int64_t o1 = P.d[0], o2 = Q.d[4], k2 = S[0].d[0], k3 = S[1].d[0], k4 = S[2].d[0];
    Tens R = make({o1, k2, k3, k4, o2});
    Tens pm = ein("iuvda,zdl->iuvalz", P, S[2]);                    // [o1,u2,u3,b,l4,k4]
    const int64_t slab = pm.size() / o1;
    for (int64_t i = 0; i < o1; ++i) {
        Scope s2(*this);
        Tens pi; pi.p = pm.p + i * slab; pi.nd = 5; for (int d = 0; d < 5; ++d) pi.d[d] = pm.d[d + 1];
        Tens big = ein("uvalz,amnlg->uvzmng", pi, Q);               // [u2,u3,k4,l2,l3,o2]: 2 D^8 flop per slab
        Tens t2 = ein("uvzmng,pum->vzngp", big, S[0]);
        drop(big);
        Tens ri; ri.p = R.p + i * (k2 * k3 * k4 * o2);
        std::string e;
        int rc = contract(st, "vzngp,qvn->pqzg", t2, S[1], ri, c.pool, &e);
        if (rc != TATRG_OK) fail(rc, "%s", e.c_str());
    }
    keep(R);
    return R;
}

void Stepper::run() {
    Counters& cn = c.cnt;
    const bool timed = c.timing >= 1;
    if (timed && c.stage_ev.empty()) { c.stage_ev.resize(TATRG_NSTAGES + 1); for (auto& e : c.stage_ev) ck(cudaEventCreate(&e), "event"); }
    double flops_mark = cn.gemm_flops;
    int stage = 0;
    auto mark = [&]() {   // closes stage `stage`
        c.stage_flops[stage] = cn.gemm_flops - flops_mark; flops_mark = cn.gemm_flops;
        ++stage;
        if (timed) ck(cudaEventRecord(c.stage_ev[stage], st), "event");
    };
    if (timed) ck(cudaEventRecord(c.stage_ev[0], st), "event");
    if (c.phi.nd != 5 || c.psi.nd != 5) fail(TATRG_ESTATE, "no state");
    for (int i = 0; i < 5; ++i) if (c.phi.d[i] != c.psi.d[i]) fail(TATRG_ESTATE, "Phi and Psi shapes differ");

    Tens a, dt, core;
    decompose(a, dt, core);                                         // (a)
    save("A", a); save("Dt", dt); save("core", core);
    mark();
    // (b) the QR / RSVD / lift stages are timed together under TATRG_ST_QR..LIFT: QR and RSVD flops are attributed by bond_swap
    Tens x, y; double* sig; int gr;
    Lift lf;
    submark = mark;
    bond_swap(a, dt, core, x, y, sig, gr, &lf);
    submark = nullptr;
    if (x.p) { save("X", x); save("Y", y); }
    { Tens s; s.p = sig; s.nd = 1; s.d[0] = gr; save("sigma", s); }
    if (lf.on && x.p) { drop(x); drop(y); }                  // formed for inspection only (TATRG_OPT_KEEP_TENSORS)
    mark();
    Tens phin, psin;
    if (c.method == 1) {
        // ---- plain ATRG: squeezers from Gamma^ATRG = A (X sigma) | (sigma Y) Dt, contraction by Eq. 2.7-2.8 ----
        const int64_t gq = x.d[4];
        Tens xs = make({x.d[0], x.d[1], x.d[2], x.d[3], gq}), ys = make({y.d[0], y.d[1], y.d[2], y.d[3], gq});
        ck(scale_last(st, xs.p, x.p, sig, x.size() / gq, gq, 0), "scale");
        ck(scale_last(st, ys.p, y.p, sig, y.size() / gq, gq, 0), "scale");
        Tens yp = perm(y, {4, 1, 2, 3, 0});          // [g, u2,u3,u4, be]   (upper site of the lower half)
        Tens ysp = perm(ys, {4, 1, 2, 3, 0});
        Tens dp = perm(dt, {4, 1, 2, 3, 0});         // [be, l2,l3,l4, j1]  (lower site of the lower half)
        drop(ys); drop(y); drop(x); drop(core);
        mark(); mark();
        Tens thf[3], thb[3];
        atrg_grams(a, xs, thf);
        atrg_grams(ysp, dp, thb);
        drop(ysp);
        mark();
        Tens Mt[3], Nt[3];
        {
            const int du[3] = {(int)c.phi.d[1], (int)c.phi.d[2], (int)c.phi.d[3]};
            squeezers(thf, thb, du, Mt, Nt);
        }
        save("M2", Mt[0]); save("M3", Mt[1]); save("M4", Mt[2]); save("N2", Nt[0]); save("N3", Nt[1]); save("N4", Nt[2]);
        mark();
        {
            Scope s2(*this);
            Tens ph = atrg_contract(a, xs, Mt);                       // Phi'[i1,k2,k3,k4,g]
            phin = perm(ph, {1, 2, 3, 0, 4});
            keep(phin);
        }
        drop(a); drop(xs);
        {
            Scope s2(*this);
            Tens ps = atrg_contract(yp, dp, Nt);                      // [g,k2,k3,k4,j1]
            psin = perm(ps, {1, 2, 3, 4, 0});                         // -> Psi[k2,k3,k4,j1,g]
            keep(psin);
        }
        drop(dt);
        mark();
    } else {
        const int du[3] = {(int)c.phi.d[1], (int)c.phi.d[2], (int)c.phi.d[3]};
        Tens U[4], e, f, g, h, thf[3], thb[3], Mt[3], Nt[3];
        // Overlapped schedule (saturated steps): the squeezers are chains of small launches with host decisions in between
        // (subspace iteration, Rayleigh-Ritz) that leave the SMs almost idle.  Direction 4 is the only one the Xi products of
        // Eq. 2.18-2.19 need, so: Gram matrices of direction 4 | squeezer 4 on the auxiliary stream q while the caller's stream
        // computes the Gram matrices of directions 2, 3 | squeezers 2, 3 on q while the caller's stream computes Xi and Xi' |
        // Lambda, Phi', Psi'.  Everything the q stage allocates comes from an arena of its own (a block of the workspace taken
        // before the fork), because the pool's reuse rule is enqueue order on ONE stream.
        SubStreams& ss = sub_streams();
        bool overlap = c.use_subspace && ss.ok && c.use_overlap;
        for (int d = 0; d < 3; ++d) overlap = overlap && sub_applicable(du[d] * du[d], c.D);
        double* arena = nullptr; size_t arena_bytes = 0;
        if (overlap) {
            const size_t n = (size_t)std::max(du[0], std::max(du[1], du[2])); const size_t n2 = n * n;
            arena_bytes = 8 * (64 * n2 * n2 + (2u << 20));
            // both Xi tensors are alive at once in this schedule; leave the arena's size again as headroom
            const size_t kt = (size_t)std::min<int64_t>(c.Ktri, a.d[1] * a.d[2]);
            const size_t xi_bytes = 8 * (size_t)a.d[0] * kt * kt * (size_t)gr * (size_t)c.D;
            if (c.pool.in_use() + 2 * arena_bytes + 3 * xi_bytes <= c.pool.capacity())
                arena = scratch((int64_t)(arena_bytes / 8));        // released at the end of the step, after the joins (or by the unwinding scope)
            if (!arena) overlap = false;
        }
        Pool arena_pool;
        if (arena) arena_pool.reset(arena, arena_bytes);
        struct ArenaGuard {        // c.pool stands for the arena while the q stage issues work; restored on every exit path
            tatrg_ctx& c; Pool& other;
            ArenaGuard(tatrg_ctx& c_, Pool& o) : c(c_), other(o) { std::swap(other, c.pool); }
            ~ArenaGuard() { std::swap(other, c.pool); }
        };
        auto on_q = [&](cudaEvent_t after, int dmask) {      // squeezers of the directions in dmask on stream q after event `after`; ends with joinq
            ArenaGuard guard(c, arena_pool);
            Stepper sq(c, ss.q);
            ck(cudaStreamWaitEvent(ss.q, after, 0), "wait");
            sq.squeezers(thf, thb, du, Mt, Nt, dmask);
            for (int d = 0; d < 3; ++d) if ((dmask >> d) & 1) { sq.detach(Mt[d]); sq.detach(Nt[d]); }
            ck(cudaEventRecord(ss.joinq, ss.q), "event");
        };
        // (The triad stage itself is not overlapped: splitting its four subspace iterations into two pairs, the second one hidden
        // behind E, F and the Gram matrices of the upper half, was measured slower -- a pair of chains takes as long as all four.)
        submark = mark;
        if (lf.on) {
            triad_implicit(a, dt, lf, sig, U, e, f, g, h);              // (c) straight from U^bond, sigma, V^bond (:394)
            for (int i = 0; i < 2; ++i) { if (lf.w[i].p != lf.u[i].p) drop(lf.w[i]); drop(lf.u[i]); drop(lf.Qm[i]); }
        } else triad(a, dt, x, y, sig, U, e, f, g, h);                  // (c)
        submark = nullptr;
        mark();
        save("E", e); save("F", f); save("G", g); save("H", h);
        save("UA", U[0]); save("UX", U[1]); save("UY", U[2]); save("UD", U[3]);
        drop(a); drop(dt); drop(core);
        if (x.p) { drop(x); drop(y); }
        // (d) squeezer Gram matrices of the upper half (E F I J) and of the sigma-weighted lower half (G sigma, H, K, L)
        Tens P, Q;
        {
            Tens gs = make({g.d[0], g.d[1], g.d[2], g.d[3]});
            ck(scale_last(st, gs.p, g.p, sig, g.size() / gr, gr, 0), "scale");
            P = perm(gs, {3, 1, 2, 0});          // [g, kY, j4u, be]
            Q = perm(h, {3, 1, 2, 0});           // [be, kD, j4l, j1]
            drop(gs);
        }
        half_grams4(e, f, thf);
        half_grams4(P, Q, thb);
        if (overlap) ck(cudaEventRecord(ss.forkq, st), "event");
        half_grams23(e, f, U[0], U[1], thf);
        half_grams23(P, Q, U[2], U[3], thb);
        drop(P); drop(Q);
        mark();
        if (overlap) {
            on_q(ss.forkq, 4);                                          // direction 4 (bit 2)
            ck(cudaStreamWaitEvent(st, ss.joinq, 0), "wait");
            ck(cudaEventRecord(ss.forkq, st), "event");                 // after the Gram matrices of directions 2, 3
        } else {
            squeezers(thf, thb, du, Mt, Nt);
        }
        mark();
        // (e) Eq. 2.18-2.19 :175  Xi[i1,kA,kX,k4,g], Xi'[j1,kD,kY,k4,g]
        Tens xi, xip;
        {
            Tens fm = ein("zul,axld->uaxzd", Mt[2], f);
            xi = ein("ikua,uaxzd->ikxzd", e, fm);
            drop(fm);
            Tens gn = ein("zul,byug->lbyzg", Nt[2], g);
            xip = ein("jdlb,lbyzg->jdyzg", h, gn);
            drop(gn);
        }
        if (overlap) {
            on_q(ss.forkq, 3);                                          // directions 2, 3 while Xi, Xi' are computed
            ck(cudaStreamWaitEvent(st, ss.joinq, 0), "wait");
            for (int d = 0; d < 3; ++d) { drop(thf[d]); drop(thb[d]); }
        }
        save("M2", Mt[0]); save("M3", Mt[1]); save("M4", Mt[2]); save("N2", Nt[0]); save("N3", Nt[1]); save("N4", Nt[2]);
        {   // Phi'[i1,k2,k3,k4,g]
            Scope s2(*this);
            // Lambda[kA,kX,k2,k3] = sum_{u,c,l,w} I[kA,u,c] M2[k2,u,l] M3[k3,c,w] J[kX,l,w]: each isometry meets one squeezer first
            // (two K D^3 tensors), then one K^2 D^2 x D^2 product -- no K D^4 intermediate
            Tens im = ein("kuc,zul->kzcl", U[0], Mt[0]);                // sum over the upper leg 2
            Tens jm = ein("xlw,ycw->xycl", U[1], Mt[1]);                // sum over the lower leg 3
            Tens lam = ein("kzcl,xycl->kxzy", im, jm);
            drop(im); drop(jm);
            Tens ph = ein("Ikxzd,kxpq->Ipqzd", xi, lam);
            drop(xi);
            phin = perm(ph, {1, 2, 3, 0, 4});                           // (f) rotate: axis 1 becomes axis 4  (R5)
            keep(phin);
        }
        {   // Psi'[j1,k2,k3,k4,g]
            Scope s2(*this);
            Tens kn = ein("yuc,zul->yzcl", U[2], Nt[0]);
            Tens ln = ein("dlw,vcw->dvcl", U[3], Nt[1]);
            Tens lam = ein("yzcl,dvcl->dyzv", kn, ln);                  // Lambda'[kD,kY,k2,k3]
            drop(kn); drop(ln);
            Tens ps = ein("Jdyzg,dypq->Jpqzg", xip, lam);
            drop(xip);
            psin = perm(ps, {1, 2, 3, 0, 4});
            keep(psin);
        }
        release(arena);
        mark();
    }
    c.pool.free(c.phi.p); c.pool.free(c.psi.p);
    detach(phin); detach(psin);
    c.phi = phin; c.psi = psin;
    ck(dot(st, c.phi.size(), c.phi.p, c.psi.p, c.trace_dev), "dot");
    mark();
    c.m += 1;
}
}  // namespace

int run_step(tatrg_ctx* c, cudaStream_t st) {
    Counters& cn = c->cnt;
    cn.launches = 0; cn.gemm_flops = 0; cn.gemm_calls = 0; cn.permuted_bytes = 0; cn.permute_calls = 0; cn.host_syncs = 0;
    cn.time_kernels = c->timing >= 2; cn.gemm_ev.clear(); cn.perm_ev.clear(); cn.perm_ev_bytes.clear(); cn.gemm_shapes.clear(); cn.ev_used = 0;
    g_counter = &cn;
    g_verbose = c->verbose;
    const int tma_saved = g_dgemm_tma;
    g_dgemm_tma = c->dgemm_tma;
    for (cudaGraphExec_t g : c->graveyard) cudaGraphExecDestroy(g);    // their launches completed before the previous step's last read-back
    c->graveyard.clear();
    int rc = TATRG_OK;
    const size_t lnc0 = c->lnc.size();
    // the state (Phi, Psi, trace) and the workspace were last written on last_stream: order a different stream behind it
    if (c->done_ev && st != c->last_stream && cudaStreamWaitEvent(st, c->done_ev, 0) != cudaSuccess) { c->err = "cannot order the new stream behind the previous step"; return TATRG_ECUDA; }
    try {
        Stepper s(*c, st);
        s.run();
    } catch (const Fail& f) {
        rc = f.code; c->err = f.msg;
    } catch (const std::exception& e) {
        rc = TATRG_ECUDA; c->err = e.what();
    }
    g_counter = nullptr;
    g_verbose = 0;
    g_dgemm_tma = tma_saved;
    c->last_stream = st;
    if (rc == TATRG_OK) {
        if (!c->done_ev && cudaEventCreateWithFlags(&c->done_ev, cudaEventDisableTiming) != cudaSuccess) c->done_ev = nullptr;
        if (c->done_ev) cudaEventRecord(c->done_ev, st);
    }
    c->last_launches = cn.launches;
    c->last_host_syncs = cn.host_syncs;
    if (rc != TATRG_OK) { cudaDeviceSynchronize(); c->failed = true; c->lnc.resize(lnc0); return rc; }   // auxiliary streams may still be running
    c->gemm_flops = cn.gemm_flops; c->gemm_calls = cn.gemm_calls; c->perm_calls = cn.permute_calls; c->perm_bytes = cn.permuted_bytes;
    if (c->timing >= 1) {
        cudaError_t e = cudaStreamSynchronize(st);
        if (e != cudaSuccess) { c->failed = true; c->err = cudaGetErrorString(e); return TATRG_ECUDA; }
        for (int i = 0; i < TATRG_NSTAGES; ++i) { float ms = 0; cudaEventElapsedTime(&ms, c->stage_ev[i], c->stage_ev[i + 1]); c->stage_ms[i] = ms; }
        c->gemm_ms = 0; c->perm_ms = 0;
        const bool verbose = (c->verbose & 4) != 0;   // debugging aid: per-launch shapes and rates
        c->gemm_large_ms = 0; c->gemm_large_flops = 0; c->gemm_large_calls = 0;
        for (size_t i = 0; i < cn.gemm_ev.size(); ++i) {
            float ms = 0; cudaEventElapsedTime(&ms, cn.gemm_ev[i].first, cn.gemm_ev[i].second); c->gemm_ms += ms;
            if (i < cn.gemm_shapes.size()) {
                const auto& g = cn.gemm_shapes[i];
                const double fl = 2.0 * g.frac * g.M * g.N * g.K * g.batch;
                if (fl >= kLargeGemmFlops) { c->gemm_large_ms += ms; c->gemm_large_flops += fl; c->gemm_large_calls += 1; }
            }
            if (verbose && i < cn.gemm_shapes.size()) {
                const auto& g = cn.gemm_shapes[i];
                fprintf(stderr, "[tatrg gemm] M=%lld N=%lld K=%lld batch=%d ta=%d tb=%d  %.3f ms  %.2f TF/s\n", (long long)g.M, (long long)g.N,
                        (long long)g.K, g.batch, (int)g.ta, (int)g.tb, ms, 2.0 * g.frac * g.M * g.N * g.K * g.batch / (ms * 1e-3) / 1e12);
            }
        }
        c->perm_large_ms = 0; c->perm_large_bytes = 0; c->perm_large_calls = 0;
        for (size_t i = 0; i < cn.perm_ev.size(); ++i) {
            float ms = 0; cudaEventElapsedTime(&ms, cn.perm_ev[i].first, cn.perm_ev[i].second); c->perm_ms += ms;
            if (i < cn.perm_ev_bytes.size() && cn.perm_ev_bytes[i] >= kLargePermuteBytes) { c->perm_large_ms += ms; c->perm_large_bytes += cn.perm_ev_bytes[i]; c->perm_large_calls += 1; }
            if (verbose && i < cn.perm_ev_bytes.size())
                fprintf(stderr, "[tatrg perm] %lld bytes  %.4f ms  %.0f GB/s\n", cn.perm_ev_bytes[i], ms, cn.perm_ev_bytes[i] / (ms * 1e-3) / 1e9);
        }
    }
    return TATRG_OK;
}

}  // namespace tatrg
