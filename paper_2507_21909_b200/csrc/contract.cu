// contract.cu -- pairwise tensor contraction "abc,cd->abd" = leg permutations (only where a layout forces one) + one
// batched DGEMM, and the workspace pool.  Every contraction of the Triad-ATRG step (Eq. 2.9-2.19 :135-175,
// A.4-A.11 :356-392) goes through here.
//
// Leg classes: batch (in A, B and C, or written UPPERCASE = batch even if missing from one operand), M (A and C),
// N (B and C), K (A and B).  An operand needs no copy when its legs form contiguous class blocks in an order the GEMM
// can address with (leading dimension, batch stride): [batch][M][K], [M][batch][K], [batch][K][M], [K][batch][M].
// The leg order inside the M, N and K blocks is a free choice; all eight combinations (take it from C or from the
// operand) are costed in permuted elements and the cheapest is used.
#include "internal.h"
#include <algorithm>
#include <cstring>
#include <cstdio>

namespace tatrg {

// ---------------------------------------------------------------------------------------------------------------
// Pool
// ---------------------------------------------------------------------------------------------------------------
void Pool::reset(void* base, size_t bytes) {
    base_ = (char*)base; cap_ = bytes & ~(size_t)255; used_ = 0; peak_ = 0; high_ = 0;
    free_.clear(); live_.clear();
    if (cap_) free_[0] = cap_;
}
double* Pool::alloc(int64_t n_doubles) {
    size_t bytes = ((size_t)(n_doubles > 0 ? n_doubles : 1) * 8 + 255) & ~(size_t)255;
    for (auto it = free_.begin(); it != free_.end(); ++it) {
        if (it->second >= bytes) {
            size_t off = it->first, sz = it->second;
            free_.erase(it);
            if (sz > bytes) free_[off + bytes] = sz - bytes;
            live_[off] = bytes;
            used_ += bytes;
            if (off + bytes > high_) high_ = off + bytes;
            if (high_ > peak_) peak_ = high_;
            return (double*)(base_ + off);
        }
    }
    return nullptr;
}
void Pool::free(const void* p) {
    if (!p) return;
    size_t off = (size_t)((const char*)p - base_);
    auto it = live_.find(off);
    if (it == live_.end()) return;
    size_t sz = it->second;
    live_.erase(it);
    used_ -= sz;
    auto nx = free_.lower_bound(off);
    if (nx != free_.end() && off + sz == nx->first) { sz += nx->second; nx = free_.erase(nx); }
    if (nx != free_.begin()) {
        auto pv = std::prev(nx);
        if (pv->first + pv->second == off) { pv->second += sz; return; }
    }
    free_[off] = sz;
}

// ---------------------------------------------------------------------------------------------------------------
// spec parsing
// ---------------------------------------------------------------------------------------------------------------
namespace {
struct Spec {
    std::string a, b, c;             // leg letters of the operands
    std::map<char, int64_t> ext;     // extent of every leg
    std::string batch, m, n, k;      // class members (unordered here)
};

bool parse(const char* spec, const Tens& A, const Tens& B, Spec& s, std::string* err) {
    std::string t(spec);
    size_t c1 = t.find(','), ar = t.find("->");
    if (c1 == std::string::npos || ar == std::string::npos || c1 > ar) { if (err) *err = "contract: bad spec " + t; return false; }
    s.a = t.substr(0, c1); s.b = t.substr(c1 + 1, ar - c1 - 1); s.c = t.substr(ar + 2);
    if ((int)s.a.size() != A.nd || (int)s.b.size() != B.nd) { if (err) *err = "contract: rank mismatch in " + t; return false; }
    for (int i = 0; i < A.nd; ++i) s.ext[s.a[i]] = A.d[i];
    for (int i = 0; i < B.nd; ++i) {
        auto it = s.ext.find(s.b[i]);
        if (it != s.ext.end() && it->second != B.d[i]) { if (err) *err = "contract: extent mismatch on leg " + std::string(1, s.b[i]) + " in " + t; return false; }
        s.ext[s.b[i]] = B.d[i];
    }
    for (auto& kv : s.ext) {
        char ch = kv.first;
        bool ia = s.a.find(ch) != std::string::npos, ib = s.b.find(ch) != std::string::npos, ic = s.c.find(ch) != std::string::npos;
        bool forced = (ch >= 'A' && ch <= 'Z');
        if (ic && (forced || (ia && ib))) s.batch += ch;
        else if (ia && ic) s.m += ch;
        else if (ib && ic) s.n += ch;
        else if (ia && ib) s.k += ch;
        else { if (err) *err = "contract: leg " + std::string(1, ch) + " appears once in " + t; return false; }
    }
    for (char ch : s.c) if (!s.ext.count(ch)) { if (err) *err = "contract: unknown output leg in " + t; return false; }
    return true;
}

std::string order_as(const std::string& members, const std::string& ref) {   // members in the order they appear in ref
    std::string o;
    for (char ch : ref) if (members.find(ch) != std::string::npos) o += ch;
    return o;
}
int64_t extent(const Spec& s, const std::string& legs) { int64_t e = 1; for (char ch : legs) e *= s.ext.at(ch); return e; }

// Addressing of one operand as (rows, cols, batch) blocks.  ok == false: needs a permuted copy.
struct Layout { bool ok = false; bool cols_inner = true; int64_t ld = 0, sb = 0; };

Layout analyse(const Spec& s, const std::string& legs, const std::string& bat, const std::string& rows, const std::string& cols) {
    Layout L;
    // legs of extent 1 never matter for addressing: drop them
    auto strip = [&](const std::string& x) { std::string o; for (char ch : x) if (s.ext.at(ch) != 1) o += ch; return o; };
    const std::string lg = strip(legs), bb = strip(bat), rr = strip(rows), cc = strip(cols);
    std::string bp;   // batch legs present in this operand, in the global batch order
    for (char ch : bb) if (legs.find(ch) != std::string::npos) bp += ch;
    if (!bp.empty() && bp.size() != bb.size()) return L;   // partially broadcast batch: not addressable with one stride
    const std::string* blk[3] = {&bp, &rr, &cc};
    const int64_t ext3[3] = {extent(s, bp), extent(s, rr), extent(s, cc)};
    static const int perm3[6][3] = {{0, 1, 2}, {0, 2, 1}, {1, 0, 2}, {1, 2, 0}, {2, 0, 1}, {2, 1, 0}};
    for (auto& p : perm3) {
        if (*blk[p[0]] + *blk[p[1]] + *blk[p[2]] != lg) continue;
        int64_t stride[3], acc = 1;
        for (int i = 2; i >= 0; --i) { stride[p[i]] = acc; acc *= ext3[p[i]]; }
        if (!bp.empty() && stride[0] == 1 && (!rr.empty() || !cc.empty())) continue;   // batch innermost: no
        if (!cc.empty() && stride[2] == 1) { L.cols_inner = true; L.ld = rr.empty() ? ext3[2] : stride[1]; }
        else if (cc.empty()) { L.cols_inner = true; L.ld = rr.empty() ? 1 : stride[1]; }
        else if (!rr.empty() && stride[1] == 1) { L.cols_inner = false; L.ld = stride[2]; }
        else if (rr.empty()) { L.cols_inner = true; L.ld = ext3[2]; if (stride[2] != 1) continue; }
        else continue;
        L.sb = bp.empty() ? 0 : stride[0];
        L.ok = true;
        return L;
    }
    return L;
}

// permuted copy of T (legs `from`) into leg order `to` (same letters)
cudaError_t permute_to(cudaStream_t st, const Spec& s, const std::string& from, const std::string& to, const double* in, double* out) {
    int64_t dims[8]; int perm[8];
    for (size_t i = 0; i < from.size(); ++i) dims[i] = s.ext.at(from[i]);
    for (size_t i = 0; i < to.size(); ++i) perm[i] = (int)from.find(to[i]);
    return permute(st, (int)from.size(), dims, perm, in, out);
}
}  // namespace

int contract_shape(const char* spec, const Tens& A, const Tens& B, Tens& C, std::string* err) {
    Spec s;
    if (!parse(spec, A, B, s, err)) return TATRG_EINVAL;
    C.nd = (int)s.c.size();
    for (int i = 0; i < C.nd; ++i) C.d[i] = s.ext.at(s.c[i]);
    return TATRG_OK;
}

int contract(cudaStream_t st, const char* spec, const Tens& A0, const Tens& B0, Tens& C, Pool& pool, std::string* err) {
    Spec s;
    if (!parse(spec, A0, B0, s, err)) return TATRG_EINVAL;
    C.nd = (int)s.c.size();
    for (int i = 0; i < C.nd; ++i) C.d[i] = s.ext.at(s.c[i]);
    if (C.size() == 0) return TATRG_OK;
    // make N the class of C's innermost leg: C^T = B^T A^T swaps the operands
    const double* Ap = A0.p; const double* Bp = B0.p;
    {
        char last = 0;
        for (int i = C.nd - 1; i >= 0; --i) if (s.ext.at(s.c[i]) != 1) { last = s.c[i]; break; }
        if (last && s.m.find(last) != std::string::npos) { std::swap(s.a, s.b); std::swap(s.m, s.n); std::swap(Ap, Bp); }
    }
    const std::string batch = order_as(s.batch, s.c);
    const int64_t eM = extent(s, s.m), eN = extent(s, s.n), eK = extent(s, s.k), eB = extent(s, batch);
    const int64_t szA = extent(s, s.a), szB = extent(s, s.b), szC = extent(s, s.c);
    // cost every choice of intra-block orders
    struct Choice { std::string m, n, k; Layout la, lb, lc; int64_t cost; };
    Choice best; best.cost = -1;
    const std::string mo[2] = {order_as(s.m, s.c), order_as(s.m, s.a)};
    const std::string no[2] = {order_as(s.n, s.c), order_as(s.n, s.b)};
    const std::string ko[2] = {order_as(s.k, s.a), order_as(s.k, s.b)};
    for (int im = 0; im < 2; ++im) for (int in = 0; in < 2; ++in) for (int ik = 0; ik < 2; ++ik) {
        Choice c; c.m = mo[im]; c.n = no[in]; c.k = ko[ik];
        c.la = analyse(s, s.a, batch, c.m, c.k);
        c.lb = analyse(s, s.b, batch, c.k, c.n);
        c.lc = analyse(s, s.c, batch, c.m, c.n);
        if (c.lc.ok && !c.lc.cols_inner && eM != 1) c.lc.ok = false;   // C must have N innermost
        c.cost = (c.la.ok ? 0 : szA) + (c.lb.ok ? 0 : szB) + (c.lc.ok ? 0 : szC);
        if (best.cost < 0 || c.cost < best.cost) best = c;
    }
    if ((g_verbose & 8) && best.cost > 0)      // debugging aid: contractions that need a permuted copy of an operand or of the result
        fprintf(stderr, "[tatrg contract] %s copies:%s%s%s  A %lld B %lld C %lld doubles\n", spec, best.la.ok ? "" : " A", best.lb.ok ? "" : " B",
                best.lc.ok ? "" : " C", (long long)szA, (long long)szB, (long long)szC);
    std::vector<double*> temps;
    auto fail = [&](int code, const std::string& msg) { for (double* t : temps) pool.free(t); if (err) *err = msg; return code; };
    // operands
    bool ta = false, tb = false; int64_t lda, ldb, sA, sB;
    const double* a_use = Ap; const double* b_use = Bp;
    if (best.la.ok) { ta = !best.la.cols_inner; lda = best.la.ld; sA = best.la.sb; }
    else {
        double* t = pool.alloc(szA); if (!t) return fail(TATRG_ENOMEM, "contract: workspace exhausted (A copy)");
        temps.push_back(t);
        std::string to = order_as(batch, s.a) + best.m + best.k;   // [batch][M][K]
        bool all_batch = order_as(batch, s.a).size() == batch.size();
        if (!all_batch && !order_as(batch, s.a).empty()) return fail(TATRG_EINVAL, std::string("contract: partial batch legs in ") + spec);
        cudaError_t e = permute_to(st, s, s.a, to, Ap, t);
        if (e != cudaSuccess) return fail(TATRG_ECUDA, cudaGetErrorString(e));
        a_use = t; ta = false; lda = std::max<int64_t>(eK, 1); sA = all_batch ? eM * eK : 0;
    }
    if (best.lb.ok) { tb = best.lb.cols_inner ? false : true; ldb = best.lb.ld; sB = best.lb.sb; }
    else {
        double* t = pool.alloc(szB); if (!t) return fail(TATRG_ENOMEM, "contract: workspace exhausted (B copy)");
        temps.push_back(t);
        std::string to = order_as(batch, s.b) + best.k + best.n;   // [batch][K][N]
        bool all_batch = order_as(batch, s.b).size() == batch.size();
        if (!all_batch && !order_as(batch, s.b).empty()) return fail(TATRG_EINVAL, std::string("contract: partial batch legs in ") + spec);
        cudaError_t e = permute_to(st, s, s.b, to, Bp, t);
        if (e != cudaSuccess) return fail(TATRG_ECUDA, cudaGetErrorString(e));
        b_use = t; tb = false; ldb = std::max<int64_t>(eN, 1); sB = all_batch ? eK * eN : 0;
    }
    double* c_use = C.p; int64_t ldc, sC;
    if (best.lc.ok) { ldc = best.lc.ld; sC = best.lc.sb; }
    else {
        double* t = pool.alloc(szC); if (!t) return fail(TATRG_ENOMEM, "contract: workspace exhausted (C copy)");
        temps.push_back(t);
        c_use = t; ldc = std::max<int64_t>(eN, 1); sC = eM * eN;
    }
    // For B, rows = K and cols = N: cols_inner means stored [K][N] (transb = false).
    cudaError_t e;
    int64_t need = (eB == 1) ? dgemm_splitk_doubles(eM, eN, eK) : 0;
    if (need > 0 && ldc >= eN) {
        double* part = pool.alloc(need);
        if (part) {
            temps.push_back(part);
            e = dgemm_splitk(st, ta, tb, eM, eN, eK, 1.0, a_use, lda, b_use, ldb, c_use, ldc, part);
        } else e = dgemm(st, ta, tb, eM, eN, eK, 1.0, a_use, lda, b_use, ldb, 0.0, c_use, ldc);
    } else {
        e = dgemm(st, ta, tb, eM, eN, eK, 1.0, a_use, lda, b_use, ldb, 0.0, c_use, ldc, (int)eB, sA, sB, sC);
    }
    if (e != cudaSuccess) return fail(TATRG_ECUDA, cudaGetErrorString(e));
    if (!best.lc.ok) {
        std::string from = batch + best.m + best.n;
        e = permute_to(st, s, from, s.c, c_use, C.p);
        if (e != cudaSuccess) return fail(TATRG_ECUDA, cudaGetErrorString(e));
    }
    for (double* t : temps) pool.free(t);
    return TATRG_OK;
}

}  // namespace tatrg
