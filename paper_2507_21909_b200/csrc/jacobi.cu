// jacobi.cu -- dense decompositions of the Triad-ATRG step on the device (PAPER.md: truncated SVD of Eq. 2.4 :76 and
// Eq. 2.5 :90 / A.8 :376, HOSVD of Eq. 2.9 :135, squeezers :171; "SVD ... based on matrix multiplication" :213).
//
//   eigh      symmetric eigen-decomposition, two-sided Jacobi.
//             n <= 64: one CTA, matrix and eigenvectors in shared memory, round-robin parallel ordering.
//             n  > 64: block Jacobi with 32-wide column blocks.  One round = nb/2 disjoint block pairs; each pair's
//             64 x 64 diagonal sub-problem is solved to convergence by one CTA in shared memory (the n <= 64 code),
//             its accumulated 64 x 64 rotation is then applied to the block columns, block rows and to V^T as tile
//             GEMMs.  nb - 1 rounds = one sweep; sweeps repeat until no CTA rotated anything.
//   svd_rows  one-sided (Hestenes) Jacobi of a small matrix held in shared memory: one warp per row pair.
//
// Vectors are returned as ROWS, sorted by descending value (the order is taken on the host from the read-back
// spectrum, which the caller needs anyway for its rank decisions).
#include "internal.h"
#include <algorithm>
#include <cmath>
#include <numeric>
#include <map>
#include <mutex>
#include <cstdio>
#include <cstdlib>

namespace tatrg {
namespace {
constexpr int SB = 64;          // side of the shared-memory sub-problem
constexpr int SP = SB + 1;      // pitch
constexpr int BW = 32;          // block width of the block-Jacobi
constexpr double kTolRel = 1e-15;
constexpr int kMaxSweeps = 40;        // sweeps of the in-CTA solvers
constexpr int kMaxBlockSweeps = 120;  // sweeps of the block method (n = 2304 Gram matrices with wide noise-level clusters take ~40)
// off-diagonal entries below kFloorRel * max|diag| are not rotated: one order below the rounding of the GEMM that
// produced the matrix
constexpr double kFloorRel = 1e-17;

// round-robin tournament on np (even) players: round r in [0, np-1), table k in [0, np/2)
__device__ __host__ __forceinline__ void rr_pair(int np, int r, int k, int& p, int& q) {
    const int m = np - 1;
    int a, b;
    if (k == 0) { a = m; b = r; }
    else { a = (r + k) % m; b = (r + m - k) % m; }
    p = a < b ? a : b; q = a < b ? b : a;
}

// plane rotation that annihilates a_pq of [[app, apq], [apq, aqq]] with J = [[c, s], [-s, c]]  (J^T A J diagonal):
// t = tan(theta) is the smaller root of t^2 + 2 zeta t - 1 = 0, zeta = (aqq - app) / (2 apq), evaluated without
// division or sqrt (FP64 div / sqrt are long software sequences and sit on the critical path of a round).
__device__ __forceinline__ void sym_rot(double app, double aqq, double apq, double& c, double& s) {
    // With d = aqq - app, r = sqrt(d^2 + 4 apq^2), w = r (r + |d|) / 2:  c = (r + |d|) / (2 sqrt(w)),  s = +-apq / sqrt(w)
    // (tan = s / c = +-2 apq / (|d| + r), the smaller root, and c^2 + s^2 = 1 identically).  Two rsqrt, no division.
    const double d = aqq - app, ad = fabs(d);
    const double q2 = fma(d, d, 4.0 * apq * apq);
    const double r = q2 * rsqrt(q2);
    const double h = 0.5 * (r + ad);
    const double inv = rsqrt(r * h);
    c = h * inv;
    s = (d >= 0 ? apq : -apq) * inv;
}
// rotate only above the relative threshold (no sqrt: compare squares) and above the absolute floor
__device__ __forceinline__ bool needs_rot(double app, double aqq, double apq, double floor_abs) {
    return fabs(apq) > floor_abs && apq * apq > (kTolRel * kTolRel) * fabs(app * aqq);
}
// A rotation counts against convergence of the block method only above 10 x that threshold: the 64-term tile products
// that apply the rotations leave rounding of a few ulp of sqrt(a_pp a_qq) in a_pq, which inside a cluster of nearly equal
// eigenvalues keeps triggering (harmless, 45-degree) rotations at 1e-15 for ever (seen at n = 2304).
__device__ __forceinline__ bool significant_rot(double app, double aqq, double apq, double floor_abs) {
    return fabs(apq) > floor_abs && apq * apq > (100.0 * kTolRel * kTolRel) * fabs(app * aqq);
}

// Two-sided Jacobi on the n x n symmetric S (shared, pitch SP), accumulating J (S_out = J^T S_in J, columns of J).
// All threads of the CTA call it.  Returns the number of rotations applied.
__device__ int jacobi_smem(double* S, double* J, int n, double abs_floor, double* cs, double* sn, int* pp, int* qq, int* cnt) {
    const int tid = threadIdx.x, nt = blockDim.x;
    const int np = n + (n & 1), half = np >> 1;
    int total = 0;
    for (int sweep = 0; sweep < kMaxSweeps; ++sweep) {
        if (tid == 0) *cnt = 0;
        __syncthreads();
        for (int r = 0; r < np - 1; ++r) {
            if (tid < half) {
                int p, q; rr_pair(np, r, tid, p, q);
                double c = 1.0, s = 0.0;
                if (q < n) {
                    double app = S[p * SP + p], aqq = S[q * SP + q], apq = S[p * SP + q];
                    if (needs_rot(app, aqq, apq, abs_floor)) { sym_rot(app, aqq, apq, c, s); atomicAdd(cnt, 1); }
                }
                cs[tid] = c; sn[tid] = s; pp[tid] = p; qq[tid] = q;
            }
            __syncthreads();
            // columns of S and of J
            for (int e = tid; e < n * half; e += nt) {
                int k = e / n, i = e - k * n;
                double s = sn[k];
                if (s == 0.0) continue;
                double c = cs[k]; int p = pp[k], q = qq[k];
                double x = S[i * SP + p], y = S[i * SP + q];
                S[i * SP + p] = c * x - s * y; S[i * SP + q] = s * x + c * y;
                x = J[i * SP + p]; y = J[i * SP + q];
                J[i * SP + p] = c * x - s * y; J[i * SP + q] = s * x + c * y;
            }
            __syncthreads();
            // rows of S
            for (int e = tid; e < n * half; e += nt) {
                int k = e / n, j = e - k * n;
                double s = sn[k];
                if (s == 0.0) continue;
                double c = cs[k]; int p = pp[k], q = qq[k];
                double x = S[p * SP + j], y = S[q * SP + j];
                double xn = c * x - s * y, yn = s * x + c * y;
                if (j == q) xn = 0.0;      // the rotation annihilates s_pq exactly
                if (j == p) yn = 0.0;
                S[p * SP + j] = xn; S[q * SP + j] = yn;
            }
            __syncthreads();
        }
        int c = *cnt;
        __syncthreads();
        total += c;
        if (c == 0) break;
    }
    return total;
}

__device__ __forceinline__ double block_max(double v, double* red) {
    for (int o = 16; o > 0; o >>= 1) v = fmax(v, __shfl_xor_sync(0xffffffffu, v, o));
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = v;
    __syncthreads();
    double m = 0;
    for (int w = 0; w < (int)(blockDim.x >> 5); ++w) m = fmax(m, red[w]);
    __syncthreads();
    return m;
}

// ---- n <= 64 ---------------------------------------------------------------------------------------------------
struct SmallBatch { int n[8]; const double* G[8]; double* lam[8]; double* Vt[8]; };
// one CTA per matrix of the batch (independent problems of a stage share one launch)
__global__ void __launch_bounds__(512, 1) eigh_small_kernel(SmallBatch sb) {
    extern __shared__ double sh[];
    const int n = sb.n[blockIdx.x];
    const double* __restrict__ G = sb.G[blockIdx.x];
    double* __restrict__ lam = sb.lam[blockIdx.x];
    double* __restrict__ Vt = sb.Vt[blockIdx.x];
    double* S = sh; double* J = S + SB * SP;
    double* cs = J + SB * SP; double* sn = cs + 32; double* red = sn + 32;
    int* pp = (int*)(red + 32); int* qq = pp + 32; int* cnt = qq + 32;
    const int tid = threadIdx.x, nt = blockDim.x;
    double dmax = 0;
    for (int e = tid; e < n * n; e += nt) {
        int i = e / n, j = e - i * n;
        S[i * SP + j] = 0.5 * (G[i * n + j] + G[j * n + i]);
        J[i * SP + j] = (i == j) ? 1.0 : 0.0;
        if (i == j) dmax = fmax(dmax, fabs(G[e]));
    }
    __syncthreads();
    dmax = block_max(dmax, red);
    jacobi_smem(S, J, n, kFloorRel * dmax, cs, sn, pp, qq, cnt);
    for (int e = tid; e < n * n; e += nt) { int i = e / n, j = e - i * n; Vt[i * n + j] = J[j * SP + i]; }   // row i = eigenvector i
    for (int i = tid; i < n; i += nt) lam[i] = S[i * SP + i];
}

// ---- n > 64: block Jacobi ----------------------------------------------------------------------------------------
constexpr int kMaxBatch = 8;
struct BatchIn { int n[kMaxBatch]; const double* G[kMaxBatch]; };
// blockIdx.y = matrix of the batch; every per-matrix array sits at (base + blockIdx.y * wstride)
__global__ void pad_sym_kernel(BatchIn bin, int N, double* __restrict__ Gp, double* __restrict__ Vt, int64_t wstride) {
    const int n = bin.n[blockIdx.y];
    const double* __restrict__ G = bin.G[blockIdx.y];
    Gp += blockIdx.y * wstride; Vt += blockIdx.y * wstride;
    int64_t total = (int64_t)N * N;
    for (int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; e < total; e += (int64_t)gridDim.x * blockDim.x) {
        int i = (int)(e / N), j = (int)(e - (int64_t)i * N);
        Gp[e] = (i < n && j < n) ? 0.5 * (G[(int64_t)i * n + j] + G[(int64_t)j * n + i]) : 0.0;
        Vt[e] = (i == j) ? 1.0 : 0.0;
    }
}
__global__ void diag_max_kernel(int N, const double* __restrict__ Gp, double* out, double floor_rel, int64_t wstride) {   // one block per matrix
    __shared__ double red[32];
    Gp += blockIdx.x * wstride; out += blockIdx.x * wstride;
    double m = 0;
    for (int i = threadIdx.x; i < N; i += blockDim.x) m = fmax(m, fabs(Gp[(int64_t)i * N + i]));
    m = block_max(m, red);
    if (threadIdx.x == 0) { out[0] = m; out[1] = floor_rel * m; }
}

__device__ __forceinline__ int gidx(int P, int Q, int li) { return li < BW ? P * BW + li : Q * BW + li - BW; }

// ---- block pair solver, v2: 1024 threads, two barriers per round --------------------------------------------------
// Pair schedule of the 64 local indices.  mode 0 (FULL): round-robin over all 64 (63 rounds): every pair once.
// mode 1 (CROSS): p = k, q = 32 + (k + r) mod 32 (32 rounds): only pairs across the two 32-blocks, whose diagonal
// blocks were diagonalised earlier in the sweep.
__device__ __forceinline__ void sched(int mode, int r, int k, int& p, int& q) {
    if (mode == 0) rr_pair(SB, r, k, p, q);
    else { p = k; q = BW + ((k + r) & (BW - 1)); }
}
struct Rot { double c, s; int p, q; };

// entry (a, b) of R^T S R for the round's direct sum of plane rotations R, from the un-rotated S (read-only here)
__device__ __forceinline__ double rotated_entry(const double* S, const Rot* cur, const int* pair_of, int a, int b) {
    const Rot ra = cur[pair_of[a]], rb = cur[pair_of[b]];
    if (ra.s != 0.0 && ra.p == rb.p && a != b) return 0.0;            // the annihilated pair entry
    const double wap = (a == ra.p) ? ra.c : ra.s, waq = (a == ra.p) ? -ra.s : ra.c;
    const double wbp = (b == rb.p) ? rb.c : rb.s, wbq = (b == rb.p) ? -rb.s : rb.c;
    const double top = wbp * S[ra.p * SP + rb.p] + wbq * S[ra.p * SP + rb.q];
    const double bot = wbp * S[ra.q * SP + rb.p] + wbq * S[ra.q * SP + rb.q];
    return wap * top + waq * bot;
}

// One CTA (1024 threads) per block pair.  A round costs ONE barrier:
//   warps 1..31 write R_k1^T S_block R_k2 for the 32 x 32 blocks of 2 x 2 entries (row pair k1, column pair k2) into the
//   second buffer (both sides of the two-sided update in one pass over S) and then rotate the columns of the
//   accumulated J in place, while warp 0 derives the next round's rotations from the OLD buffer (rotated_entry).
//   None of the three touches data another one writes.
__global__ void __launch_bounds__(1024, 1) blk_solve2_kernel(int N, int nb, int round, int prev_round, int mode, const double* __restrict__ Gp,
                                                             const double* __restrict__ misc, const double* __restrict__ Jprev,
                                                             const double* __restrict__ Dprev, double* __restrict__ Jb,
                                                             double* __restrict__ Dg, int* __restrict__ active, int* __restrict__ counter,
                                                             int64_t wstride) {
    Gp += blockIdx.y * wstride; misc += blockIdx.y * wstride; Jb += blockIdx.y * wstride; Dg += blockIdx.y * wstride;
    Jprev += blockIdx.y * wstride; Dprev += blockIdx.y * wstride;
    active += blockIdx.y * wstride * 2;      // wstride counts doubles
    extern __shared__ double sh[];
    double* Sa = sh; double* Sb = Sa + SB * SP; double* J = Sb + SB * SP;
    Rot* rots = reinterpret_cast<Rot*>(J + SB * SP);          // 2 x 32
    double* red = reinterpret_cast<double*>(rots + 64);       // 32
    int* pair_of = reinterpret_cast<int*>(red + 32);          // 2 x 64
    int* cnt = pair_of + 128;
    const int tid = threadIdx.x, k = blockIdx.x, warp = tid >> 5, lane = tid & 31;
    int P, Q; rr_pair(nb, round, k, P, Q);
    if (prev_round < 0) {
        // the matrix in Gp is up to date: take the diagonal sub-problem from it
        for (int e = tid; e < SB * SB; e += 1024) {
            int i = e >> 6, j = e & 63;
            Sa[i * SP + j] = Gp[(int64_t)gidx(P, Q, i) * N + gidx(P, Q, j)];
        }
    } else {
        // Gp is the matrix BEFORE the previous round's rotations were applied (that apply runs concurrently on another
        // stream and writes a different buffer).  The sub-problem of this pair is assembled from the previous round's
        // solver outputs: diagonal 32-blocks from the solved sub-problems (Dprev), the cross block as the needed
        // 32 x 32 corner of J_a^T G[PQ_a, PQ_b] J_b.
        int* loc = cnt + 4;                                   // a, hP, b, hQ, Pa, Qa, Pb, Qb
        if (tid == 0) {
            for (int kk = 0; kk < (nb >> 1); ++kk) {
                int A, B; rr_pair(nb, prev_round, kk, A, B);
                if (A == P) { loc[0] = kk; loc[1] = 0; loc[4] = A; loc[5] = B; }
                if (B == P) { loc[0] = kk; loc[1] = 1; loc[4] = A; loc[5] = B; }
                if (A == Q) { loc[2] = kk; loc[3] = 0; loc[6] = A; loc[7] = B; }
                if (B == Q) { loc[2] = kk; loc[3] = 1; loc[6] = A; loc[7] = B; }
            }
        }
        __syncthreads();
        const int a = loc[0], hP = loc[1], b = loc[2], hQ = loc[3], Pa = loc[4], Qa = loc[5], Pb = loc[6], Qb = loc[7];
        const double* Ja = Jprev + (int64_t)a * SB * SB; const double* Jbb = Jprev + (int64_t)b * SB * SB;
        for (int e = tid; e < SB * SB; e += 1024) {
            int i = e >> 6, j = e & 63;
            Sb[i * SP + j] = Gp[(int64_t)gidx(Pa, Qa, i) * N + gidx(Pb, Qb, j)];                    // X = G[PQ_a, PQ_b]
            J[i * SP + j] = (j < BW) ? Ja[i * SB + hP * BW + j] : Jbb[i * SB + hQ * BW + j - BW];   // [J_a half | J_b half]
        }
        __syncthreads();
        for (int e = tid; e < BW * SB; e += 1024) {           // T1 = (J_a half)^T X   (32 x 64), parked in rows 32..63 of Sa
            int r = e >> 6, j = e & 63;
            double acc = 0;
#pragma unroll 8
            for (int i = 0; i < SB; ++i) acc += J[i * SP + r] * Sb[i * SP + j];
            Sa[(BW + r) * SP + j] = acc;
        }
        __syncthreads();
        double pq;
        {
            const int r = tid >> 5, c = tid & 31;                 // cross block = T1 (J_b half)   (32 x 32)
            double acc = 0;
#pragma unroll 8
            for (int j = 0; j < SB; ++j) acc += Sa[(BW + r) * SP + j] * J[j * SP + BW + c];
            pq = acc;
        }
        __syncthreads();
        {
            const int r = tid >> 5, c = tid & 31;
            Sa[r * SP + BW + c] = pq; Sa[(BW + c) * SP + r] = pq;
            Sa[r * SP + c] = Dprev[(int64_t)a * SB * SB + (hP * BW + r) * SB + hP * BW + c];
            Sa[(BW + r) * SP + BW + c] = Dprev[(int64_t)b * SB * SB + (hQ * BW + r) * SB + hQ * BW + c];
        }
    }
    __syncthreads();
    for (int e = tid; e < SB * SB; e += 1024) { int i = e >> 6, j = e & 63; J[i * SP + j] = (i == j) ? 1.0 : 0.0; }
    if (tid == 0) { cnt[0] = 0; cnt[1] = 0; }
    __syncthreads();
    const double floor_abs = misc[1];
    // quick test: anything to rotate among the pairs this mode visits?
    double worst = 0;
    for (int e = tid; e < SB * SB; e += 1024) {
        int i = e >> 6, j = e & 63;
        if (i < j && (mode == 0 || (i < BW && j >= BW))) {
            double a = fabs(Sa[i * SP + j]);
            if (needs_rot(Sa[i * SP + i], Sa[j * SP + j], a, floor_abs)) worst = 1.0;
        }
    }
    worst = block_max(worst, red);
    if (worst == 0.0) {     // nothing to rotate: publish the block as it is and an identity rotation (the next round reads them)
        if (tid == 0) active[k] = 0;
        for (int e = tid; e < SB * SB; e += 1024) {
            int i = e >> 6, j = e & 63;
            Jb[(int64_t)k * SB * SB + e] = (i == j) ? 1.0 : 0.0;
            Dg[(int64_t)k * SB * SB + e] = Sa[i * SP + j];
        }
        return;
    }
    const int nrounds = mode == 0 ? SB - 1 : BW;
    const int max_sweeps = mode == 0 ? 2 : 1;
    double* S = Sa; double* T = Sb;
    int total = 0, total_sig = 0;
    for (int sweep = 0; sweep < max_sweeps; ++sweep) {
        // rotations of round 0 from the current S
        if (tid < 32) {
            int p, q; sched(mode, 0, tid, p, q);
            Rot rt; rt.c = 1.0; rt.s = 0.0; rt.p = p; rt.q = q;
            double app = S[p * SP + p], aqq = S[q * SP + q], apq = S[p * SP + q];
            const bool need = needs_rot(app, aqq, apq, floor_abs);
            if (need) sym_rot(app, aqq, apq, rt.c, rt.s);
            const int nrot = __popc(__ballot_sync(0xffffffffu, need));
            const int nsig = __popc(__ballot_sync(0xffffffffu, need && significant_rot(app, aqq, apq, floor_abs)));
            if (tid == 0) { cnt[0] += nrot; cnt[1] += nsig; }
            rots[tid] = rt; pair_of[p] = tid; pair_of[q] = tid;
        }
        __syncthreads();
        for (int r = 0; r < nrounds; ++r) {
            const Rot* cur = rots + (r & 1) * 32; Rot* nxt = rots + ((r + 1) & 1) * 32;
            const int* pof = pair_of + (r & 1) * 64; int* pof_n = pair_of + ((r + 1) & 1) * 64;
            // two-sided update of the 2x2 blocks (row pair k1, column pair k2): S -> T.  Warp 0 is kept free for the
            // rotation arithmetic (the longest dependent chain of a round); its 32 blocks go to the first 32 other threads.
            if (warp != 0) {
                for (int bidx = tid - 32; bidx < 32 * 32; bidx += 1024 - 32) {
                    const int k1 = bidx >> 5, k2 = bidx & 31;
                    const Rot r1 = cur[k1], r2 = cur[k2];
                    const double a = S[r1.p * SP + r2.p], b = S[r1.p * SP + r2.q], c_ = S[r1.q * SP + r2.p], d = S[r1.q * SP + r2.q];
                    const double a1 = r2.c * a - r2.s * b, b1 = r2.s * a + r2.c * b, c1 = r2.c * c_ - r2.s * d, d1 = r2.s * c_ + r2.c * d;
                    double A = r1.c * a1 - r1.s * c1, C = r1.s * a1 + r1.c * c1, B = r1.c * b1 - r1.s * d1, D = r1.s * b1 + r1.c * d1;
                    if (k1 == k2 && r1.s != 0.0) { B = 0.0; C = 0.0; }      // the rotation annihilates s_pq exactly
                    T[r1.p * SP + r2.p] = A; T[r1.p * SP + r2.q] = B; T[r1.q * SP + r2.p] = C; T[r1.q * SP + r2.q] = D;
                }
            }
            if (warp == 0) {
                if (r + 1 < nrounds) {      // next round's rotations, from the old buffer
                    int p, q; sched(mode, r + 1, lane, p, q);
                    Rot rt; rt.c = 1.0; rt.s = 0.0; rt.p = p; rt.q = q;
                    const double app = rotated_entry(S, cur, pof, p, p), aqq = rotated_entry(S, cur, pof, q, q), apq = rotated_entry(S, cur, pof, p, q);
                    const bool need = needs_rot(app, aqq, apq, floor_abs);
                    if (need) sym_rot(app, aqq, apq, rt.c, rt.s);
                    const int nrot = __popc(__ballot_sync(0xffffffffu, need));
                    const int nsig = __popc(__ballot_sync(0xffffffffu, need && significant_rot(app, aqq, apq, floor_abs)));
                    if (lane == 0) { cnt[0] += nrot; cnt[1] += nsig; }
                    nxt[lane] = rt; pof_n[p] = lane; pof_n[q] = lane;
                }
            } else {                        // columns of J, in place
                for (int e = tid - 32; e < SB * 32; e += 1024 - 32) {
                    const int kk = e >> 6, i = e & 63;
                    const Rot rt = cur[kk];
                    if (rt.s != 0.0) {
                        const double x = J[i * SP + rt.p], y = J[i * SP + rt.q];
                        J[i * SP + rt.p] = rt.c * x - rt.s * y; J[i * SP + rt.q] = rt.s * x + rt.c * y;
                    }
                }
            }
            __syncthreads();
            double* tmp = S; S = T; T = tmp;
        }
        const int c = cnt[0], cs = cnt[1];
        __syncthreads();
        if (tid == 0) { cnt[0] = 0; cnt[1] = 0; }
        total += c; total_sig += cs;
        if (c == 0) break;
        __syncthreads();
    }
    if (tid == 0) { active[k] = total > 0; if (total_sig > 0) atomicAdd(counter, total_sig); }
    for (int e = tid; e < SB * SB; e += 1024) { int i = e >> 6, j = e & 63; Jb[(int64_t)k * SB * SB + e] = J[i * SP + j]; }
    for (int e = tid; e < SB * SB; e += 1024) { int i = e >> 6, j = e & 63; Dg[(int64_t)k * SB * SB + e] = S[i * SP + j]; }
}

// 64x64x64 tile products on FP64 tensor cores (mma.sync.m8n8k4).  256 threads = 8 warps as 4 (M) x 2 (N); a warp owns
// a 16 x 32 block = 2 x 4 atoms.  Shared tiles have pitch AP = 68 doubles (= 4 mod 16): the 8-byte fragment loads of a
// half-warp then hit 16 distinct banks whether the fragment index runs along a row or down a column.
constexpr int AP = 68;
__device__ __forceinline__ void dmma884(double& d0, double& d1, double a, double b) {
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n" : "+d"(d0), "+d"(d1) : "d"(a), "d"(b));
}
// acc = A^T B (TRANS_A) or A B, for the warp's block at (m0, n0)
template <bool TRANS_A>
__device__ __forceinline__ void tile_mma(const double* __restrict__ A, const double* __restrict__ B, double acc[2][4][2], int m0, int n0, int g, int t) {
#pragma unroll 4
    for (int k0 = 0; k0 < SB; k0 += 4) {
        double a[2], b[4];
#pragma unroll
        for (int i = 0; i < 2; ++i) a[i] = TRANS_A ? A[(k0 + t) * AP + m0 + 8 * i + g] : A[(m0 + 8 * i + g) * AP + k0 + t];
#pragma unroll
        for (int j = 0; j < 4; ++j) b[j] = B[(k0 + t) * AP + n0 + 8 * j + g];
#pragma unroll
        for (int i = 0; i < 2; ++i)
#pragma unroll
            for (int j = 0; j < 4; ++j) dmma884(acc[i][j][0], acc[i][j][1], a[i], b[j]);
    }
}

// One launch applies the round's rotations to G (both sides, tile by tile, using the symmetry) and to V^T:
//   blockIdx.y <  npair : tile (k = blockIdx.y, l = blockIdx.x), k <= l:  G[PQ_k,PQ_l] <- J_k^T G[PQ_k,PQ_l] J_l  (+ mirror)
//   blockIdx.y >= npair : V^T[PQ_k, 64-column tile blockIdx.x] <- J_k^T V^T[...]
__global__ void __launch_bounds__(256, 2) blk_apply2_kernel(int N, int nb, int round, const double* __restrict__ Gin, double* __restrict__ Gout,
                                                            double* __restrict__ Vt, const double* __restrict__ Jb, const double* __restrict__ Dg,
                                                            const int* __restrict__ active, int64_t wstride) {
    Gin += blockIdx.z * wstride; Gout += blockIdx.z * wstride; Vt += blockIdx.z * wstride; Jb += blockIdx.z * wstride; Dg += blockIdx.z * wstride;
    active += blockIdx.z * wstride * 2;
    extern __shared__ double sh2[];
    double* Xs = sh2; double* Ja = sh2 + SB * AP; double* Jc = sh2 + 2 * SB * AP;
    const int npair = nb >> 1, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int g = lane >> 2, t = lane & 3, m0 = (warp >> 1) * 16, n0 = (warp & 1) * 32;
    double acc[2][4][2];
#pragma unroll
    for (int i = 0; i < 2; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) acc[i][j][0] = acc[i][j][1] = 0.0;
    if ((int)blockIdx.y >= npair) {      // V^T rows of pair k, in place
        const int k = blockIdx.y - npair;
        if (!active[k]) return;
        int P, Q; rr_pair(nb, round, k, P, Q);
        const int c0 = blockIdx.x * SB;
        for (int e = tid; e < SB * SB / 2; e += 256) {
            int i = e >> 5, j = (e & 31) * 2;
            *reinterpret_cast<double2*>(Xs + i * AP + j) = *reinterpret_cast<const double2*>(Vt + (int64_t)gidx(P, Q, i) * N + c0 + j);
            *reinterpret_cast<double2*>(Ja + i * AP + j) = *reinterpret_cast<const double2*>(Jb + (int64_t)k * SB * SB + i * SB + j);
        }
        __syncthreads();
        tile_mma<true>(Ja, Xs, acc, m0, n0, g, t);
#pragma unroll
        for (int i = 0; i < 2; ++i)
#pragma unroll
            for (int j = 0; j < 4; ++j)
                *reinterpret_cast<double2*>(Vt + (int64_t)gidx(P, Q, m0 + 8 * i + g) * N + c0 + n0 + 8 * j + 2 * t) = make_double2(acc[i][j][0], acc[i][j][1]);
        return;
    }
    // G: out of place (Gin -> Gout), every tile k <= l is written (copied when neither pair rotated)
    const int k = blockIdx.y, l = blockIdx.x;
    if (l >= npair || k > l) return;
    const bool ak = active[k] != 0, al = active[l] != 0;
    int P, Q, R, S2; rr_pair(nb, round, k, P, Q); rr_pair(nb, round, l, R, S2);
    if (k == l) {   // the solved diagonal block: exactly what the solver left (annihilated entries are exact zeros)
        for (int e = tid; e < SB * SB; e += 256) {
            int i = e >> 6, j = e & 63;
            Gout[(int64_t)gidx(P, Q, i) * N + gidx(P, Q, j)] = Dg[(int64_t)k * SB * SB + e];
        }
        return;
    }
    if (!ak && !al) {
        for (int e = tid; e < SB * SB / 2; e += 256) {
            int i = e >> 5, j = (e & 31) * 2;
            *reinterpret_cast<double2*>(Gout + (int64_t)gidx(P, Q, i) * N + gidx(R, S2, j)) = *reinterpret_cast<const double2*>(Gin + (int64_t)gidx(P, Q, i) * N + gidx(R, S2, j));
            *reinterpret_cast<double2*>(Gout + (int64_t)gidx(R, S2, i) * N + gidx(P, Q, j)) = *reinterpret_cast<const double2*>(Gin + (int64_t)gidx(R, S2, i) * N + gidx(P, Q, j));
        }
        return;
    }
    for (int e = tid; e < SB * SB / 2; e += 256) {
        int i = e >> 5, j = (e & 31) * 2;      // j, j+1 lie in the same 32-wide block
        *reinterpret_cast<double2*>(Xs + i * AP + j) = *reinterpret_cast<const double2*>(Gin + (int64_t)gidx(P, Q, i) * N + gidx(R, S2, j));
        *reinterpret_cast<double2*>(Ja + i * AP + j) = *reinterpret_cast<const double2*>(Jb + (int64_t)k * SB * SB + i * SB + j);
        *reinterpret_cast<double2*>(Jc + i * AP + j) = *reinterpret_cast<const double2*>(Jb + (int64_t)l * SB * SB + i * SB + j);
    }
    __syncthreads();
    tile_mma<true>(Ja, Xs, acc, m0, n0, g, t);        // J_k^T X
    __syncthreads();
#pragma unroll
    for (int i = 0; i < 2; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            *reinterpret_cast<double2*>(Xs + (m0 + 8 * i + g) * AP + n0 + 8 * j + 2 * t) = make_double2(acc[i][j][0], acc[i][j][1]);
            acc[i][j][0] = acc[i][j][1] = 0.0;
        }
    __syncthreads();
    tile_mma<false>(Xs, Jc, acc, m0, n0, g, t);       // (J_k^T X) J_l
    // write the tile, then its mirror through shared memory so that both stores are row-contiguous
#pragma unroll
    for (int i = 0; i < 2; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j)
            *reinterpret_cast<double2*>(Gout + (int64_t)gidx(P, Q, m0 + 8 * i + g) * N + gidx(R, S2, n0 + 8 * j + 2 * t)) = make_double2(acc[i][j][0], acc[i][j][1]);
    __syncthreads();
#pragma unroll
    for (int i = 0; i < 2; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            Ja[(n0 + 8 * j + 2 * t) * AP + m0 + 8 * i + g] = acc[i][j][0];         // transposed
            Ja[(n0 + 8 * j + 2 * t + 1) * AP + m0 + 8 * i + g] = acc[i][j][1];
        }
    __syncthreads();
    for (int e = tid; e < SB * SB / 2; e += 256) {
        int i = e >> 5, j = (e & 31) * 2;
        *reinterpret_cast<double2*>(Gout + (int64_t)gidx(R, S2, i) * N + gidx(P, Q, j)) = *reinterpret_cast<const double2*>(Ja + i * AP + j);
    }
}
__global__ void extract_diag_kernel(int N, const double* __restrict__ Gp, double* __restrict__ d) {
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < N; i += gridDim.x * blockDim.x) d[i] = Gp[(int64_t)i * N + i];
}

// ---- one-sided Jacobi of a small matrix ---------------------------------------------------------------------------
// W [nv x len] rows in shared memory (pitch len+1), Va [nv x nv] (pitch nv+1).  One warp per pair and round.
__global__ void __launch_bounds__(1024, 1) svd_rows_kernel(int nv, int len, const double* __restrict__ X, double* __restrict__ s_out,
                                                           double* __restrict__ Ut, double* __restrict__ Vacc) {
    extern __shared__ double sh[];
    const int pw = len + 1, pv = nv + 1;
    double* W = sh; double* Va = W + nv * pw;
    __shared__ int cnt;
    const int tid = threadIdx.x, nt = blockDim.x, lane = tid & 31, warp = tid >> 5, nw = nt >> 5;
    for (int e = tid; e < nv * len; e += nt) { int i = e / len, j = e - i * len; W[i * pw + j] = X[e]; }
    for (int e = tid; e < nv * nv; e += nt) { int i = e / nv, j = e - i * nv; Va[i * pv + j] = (i == j) ? 1.0 : 0.0; }
    __syncthreads();
    const int np = nv + (nv & 1), half = np >> 1;
    const double tol = kTolRel * sqrt((double)len);
    for (int sweep = 0; sweep < kMaxSweeps; ++sweep) {
        if (tid == 0) cnt = 0;
        __syncthreads();
        for (int r = 0; r < np - 1; ++r) {
            for (int k = warp; k < half; k += nw) {
                int p, q; rr_pair(np, r, k, p, q);
                if (q >= nv) continue;
                double* wp = W + p * pw; double* wq = W + q * pw;
                double al = 0, be = 0, ga = 0;
                for (int i = lane; i < len; i += 32) { double x = wp[i], y = wq[i]; al += x * x; be += y * y; ga += x * y; }
                for (int o = 16; o > 0; o >>= 1) {
                    al += __shfl_xor_sync(0xffffffffu, al, o); be += __shfl_xor_sync(0xffffffffu, be, o); ga += __shfl_xor_sync(0xffffffffu, ga, o);
                }
                if (al * be == 0.0 || ga * ga <= (tol * tol) * al * be) continue;
                double c, s; sym_rot(al, be, ga, c, s);
                for (int i = lane; i < len; i += 32) { double x = wp[i], y = wq[i]; wp[i] = c * x - s * y; wq[i] = s * x + c * y; }
                double* vp = Va + p * pv; double* vq = Va + q * pv;
                for (int i = lane; i < nv; i += 32) { double x = vp[i], y = vq[i]; vp[i] = c * x - s * y; vq[i] = s * x + c * y; }
                if (lane == 0) atomicAdd(&cnt, 1);
            }
            __syncthreads();
        }
        int c = cnt;
        __syncthreads();
        if (c == 0) break;
    }
    for (int k = warp; k < nv; k += nw) {
        double* w = W + k * pw; double n2 = 0;
        for (int i = lane; i < len; i += 32) n2 += w[i] * w[i];
        for (int o = 16; o > 0; o >>= 1) n2 += __shfl_xor_sync(0xffffffffu, n2, o);
        double sv = sqrt(n2), inv = sv > 0 ? 1.0 / sv : 0.0;
        for (int i = lane; i < len; i += 32) Ut[k * len + i] = w[i] * inv;
        for (int i = lane; i < nv; i += 32) Vacc[k * nv + i] = Va[k * pv + i];
        if (lane == 0) s_out[k] = sv;
    }
}

bool check(cudaError_t e, std::string* err, const char* what) {
    if (e == cudaSuccess) return true;
    if (err) *err = std::string(what) + ": " + cudaGetErrorString(e);
    return false;
}
constexpr int kSmallSmem = (2 * SB * SP + 96) * 8 + 3 * 32 * 4 + 64;
constexpr int kApplySmem = 3 * SB * 68 * 8;
constexpr int kSolve2Smem = 3 * SB * SP * 8 + 64 * 24 + 32 * 8 + 128 * 4 + 128;
}  // namespace

static int padded_n(int n) { if (n <= SB) return n; int nb = (n + BW - 1) / BW; if (nb & 1) ++nb; return nb * BW; }

// per-matrix work layout (doubles): [lam_u N][idx N][misc 64][Vt_unsorted N*N][G0 N*N][G1 N*N][Jb 2 x npair*4096][Dg 2 x npair*4096][active 2 x npair]
static size_t work_doubles(int N) {
    size_t nb2 = (size_t)N / BW / 2 + 1;
    size_t d = 2 * (size_t)N + 64 + 3 * (size_t)N * N + 4 * nb2 * SB * SB + 2 * nb2;
    return (d + 63) & ~(size_t)63;
}
size_t eigh_work_bytes(int n) { return 8 * work_doubles(padded_n(n)) + 4096; }
size_t eigh_batched_work_bytes(int nmax, int count) { return 8 * work_doubles(padded_n(nmax)) * (size_t)(count > 0 ? count : 1) + 4096; }

// sorts the spectra of a batch on the host and gathers the eigenvectors: one synchronisation for all read-backs, one for
// all uploads / gathers (the index vectors must outlive the copies)
struct FinishItem { int n; double* lam_u; int* idx; double* Vu; double* lam; double* Vt; std::vector<double>* lam_host; };
static int finish_batch(cudaStream_t st, int N, const std::vector<FinishItem>& items, std::string* err) {
    const size_t cnt = items.size();
    std::vector<std::vector<double>> lh(cnt);
    for (size_t z = 0; z < cnt; ++z) {
        lh[z].resize(items[z].n);
        if (!check(cudaMemcpyAsync(lh[z].data(), items[z].lam_u, sizeof(double) * items[z].n, cudaMemcpyDeviceToHost, st), err, "eigh readback")) return TATRG_ECUDA;
    }
    count_sync(); if (!check(cudaStreamSynchronize(st), err, "eigh sync")) return TATRG_ECUDA;
    std::vector<std::vector<int>> order(cnt);
    for (size_t z = 0; z < cnt; ++z) {
        const FinishItem& it = items[z];
        const int n = it.n;
        for (int i = 0; i < n; ++i) if (!std::isfinite(lh[z][i])) { if (err) *err = "eigh: non-finite eigenvalue"; return TATRG_ENUMERIC; }
        order[z].resize(n);
        std::iota(order[z].begin(), order[z].end(), 0);
        std::stable_sort(order[z].begin(), order[z].end(), [&](int a, int b) { return lh[z][a] > lh[z][b]; });
        if (!check(cudaMemcpyAsync(it.idx, order[z].data(), sizeof(int) * n, cudaMemcpyHostToDevice, st), err, "eigh upload")) return TATRG_ECUDA;
        if (!check(gather_rows_scaled(st, it.Vt, it.Vu, it.idx, nullptr, n, n, N > 0 ? N : n), err, "eigh gather")) return TATRG_ECUDA;
        if (!check(gather_vec(st, it.lam, it.lam_u, it.idx, n, 1, 1.0), err, "eigh gather")) return TATRG_ECUDA;
        if (it.lam_host) { it.lam_host->resize(n); for (int i = 0; i < n; ++i) (*it.lam_host)[i] = lh[z][order[z][i]]; }
        if (g_verbose & 2) {
            int c[5] = {0, 0, 0, 0, 0}; const double l0 = lh[z][order[z][0]]; const double th[5] = {1e-4, 1e-8, 1e-12, 1e-14, 1e-16};
            for (int i = 0; i < n; ++i) for (int j = 0; j < 5; ++j) if (lh[z][i] > th[j] * l0) ++c[j];
            fprintf(stderr, "[tatrg eigh n=%d] spectrum: >1e-4:%d >1e-8:%d >1e-12:%d >1e-14:%d >1e-16:%d\n", n, c[0], c[1], c[2], c[3], c[4]);
        }
    }
    count_sync(); if (!check(cudaStreamSynchronize(st), err, "eigh sync")) return TATRG_ECUDA;   // `order` leaves scope
    return TATRG_OK;
}

// auxiliary stream + events of the two-stream round pipeline (created once per process, never destroyed)
struct Aux { cudaStream_t st = nullptr; cudaEvent_t evS[2], evA[2], ev0; bool ok = false; bool tried = false; };
// one set per device (streams belong to the device that was current when they were created); calls on the same device
// from several host threads at once are not supported
static Aux& aux() {
    static std::map<int, Aux> per_device;
    static std::mutex mu;
    int dev = 0;
    cudaGetDevice(&dev);
    std::lock_guard<std::mutex> lock(mu);
    Aux& a = per_device[dev];
    if (!a.tried) {
        a.tried = true;
        int lo = 0, hi = 0;
        cudaDeviceGetStreamPriorityRange(&lo, &hi);          // hi = greatest priority (numerically lowest)
        bool ok = cudaStreamCreateWithPriority(&a.st, cudaStreamNonBlocking, hi) == cudaSuccess;
        for (int i = 0; i < 2 && ok; ++i) ok = cudaEventCreateWithFlags(&a.evS[i], cudaEventDisableTiming) == cudaSuccess && cudaEventCreateWithFlags(&a.evA[i], cudaEventDisableTiming) == cudaSuccess;
        if (ok) ok = cudaEventCreateWithFlags(&a.ev0, cudaEventDisableTiming) == cudaSuccess;
        a.ok = ok;
    }
    return a;
}

// Eigen-decompositions of up to kMaxBatch independent symmetric matrices in the same launches: the pair solver runs
// on n/64 CTAs per matrix only, so a batch fills the SMs that a single decomposition leaves idle, and the barrier /
// launch latency of a round is paid once for the whole batch.  All matrices are padded to the largest one.
int eigh_batched(cudaStream_t st, int count, const EighItem* items, void* work, std::string* err) {
    if (count <= 0) return TATRG_OK;
    static unsigned long long cfg = 0;
    if (first_use_on_device(cfg)) {
        if (!check(cudaFuncSetAttribute(eigh_small_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, kSmallSmem), err, "eigh attr")) return TATRG_ECUDA;
        if (!check(cudaFuncSetAttribute(blk_solve2_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, kSolve2Smem), err, "eigh attr")) return TATRG_ECUDA;
        if (!check(cudaFuncSetAttribute(blk_apply2_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, kApplySmem), err, "eigh attr")) return TATRG_ECUDA;
    }
    int nmax = 0;
    for (int i = 0; i < count; ++i) { if (items[i].n <= 0) { if (err) *err = "eigh: empty matrix"; return TATRG_EINVAL; } nmax = std::max(nmax, items[i].n); }
    const int N = padded_n(nmax);
    const int64_t ws = (int64_t)work_doubles(N);
    double* base = (double*)work;
    auto lam_u = [&](int z) { return base + z * ws; };
    auto idx = [&](int z) { return (int*)(base + z * ws + N); };
    auto misc = [&](int z) { return base + z * ws + 2 * (int64_t)N; };
    auto Vu = [&](int z) { return base + z * ws + 2 * (int64_t)N + 64; };
    if (nmax <= SB) {
        for (int z0 = 0; z0 < count; z0 += 8) {
            const int bc = std::min(8, count - z0);
            SmallBatch sb;
            for (int z = 0; z < bc; ++z) { sb.n[z] = items[z0 + z].n; sb.G[z] = items[z0 + z].G; sb.lam[z] = lam_u(z0 + z); sb.Vt[z] = Vu(z0 + z); }
            eigh_small_kernel<<<bc, 512, kSmallSmem, st>>>(sb); count_launch();
        }
        // every matrix keeps its own leading dimension n here: one finish per distinct stride
        for (int z = 0; z < count; ++z) {
            std::vector<FinishItem> fi{FinishItem{items[z].n, lam_u(z), idx(z), Vu(z), items[z].lam, items[z].Vt, items[z].lam_host}};
            int z2 = z + 1;
            for (; z2 < count && items[z2].n == items[z].n; ++z2)
                fi.push_back(FinishItem{items[z2].n, lam_u(z2), idx(z2), Vu(z2), items[z2].lam, items[z2].Vt, items[z2].lam_host});
            int rc = finish_batch(st, items[z].n, fi, err);
            if (rc != TATRG_OK) return rc;
            z = z2 - 1;
        }
        return TATRG_OK;
    }
    const bool verbose = (g_verbose & 2) != 0;   // debugging aid only
    const int nb = N / BW, npair = nb / 2;
    for (int z0 = 0; z0 < count; z0 += kMaxBatch) {
        const int bc = std::min(kMaxBatch, count - z0);
        BatchIn bin;
        for (int z = 0; z < bc; ++z) { bin.n[z] = items[z0 + z].n; bin.G[z] = items[z0 + z].G; }
        double* Vu0 = Vu(z0);
        double* Gbuf[2] = {Vu0 + (int64_t)N * N, Vu0 + 2 * (int64_t)N * N};
        double* Jbuf[2]; double* Dbuf[2]; int* abuf[2];
        Jbuf[0] = Gbuf[1] + (int64_t)N * N; Jbuf[1] = Jbuf[0] + (int64_t)npair * SB * SB;
        Dbuf[0] = Jbuf[1] + (int64_t)npair * SB * SB; Dbuf[1] = Dbuf[0] + (int64_t)npair * SB * SB;
        abuf[0] = (int*)(Dbuf[1] + (int64_t)npair * SB * SB); abuf[1] = abuf[0] + 2 * ((npair + 1) / 2);
        double* misc0 = misc(z0);
        int* counter = (int*)misc0 + 8;
        pad_sym_kernel<<<dim3(148 * 2, bc), 256, 0, st>>>(bin, N, Gbuf[0], Vu0, ws);
        diag_max_kernel<<<bc, 256, 0, st>>>(N, Gbuf[0], misc0, kFloorRel, ws);
        count_launch(2);
        // Two streams: the pair solver of round t+1 assembles its sub-problems from the previous round's solver outputs and the
        // matrix BEFORE that round's rotations (G[t % 2]), so it does not wait for apply(t), which writes G[(t+1) % 2].  The
        // solvers run on a high-priority auxiliary stream (their few large CTAs must get an SM as soon as one apply CTA
        // retires), the applies on the caller's stream.  A round then costs max(solver, apply) instead of their sum.
        Aux& ax = aux();
        if (!ax.ok) { if (err) *err = "eigh: cannot create the auxiliary stream"; return TATRG_ECUDA; }
        cudaStream_t ss = ax.st;                       // solver stream
        cudaEventRecord(ax.ev0, st);
        cudaStreamWaitEvent(ss, ax.ev0, 0);
        int t = 0, sweep = 0;
        for (; sweep < kMaxBlockSweeps; ++sweep) {
            cudaMemsetAsync(counter, 0, sizeof(int), ss);
            for (int r = 0; r < nb - 1; ++r, ++t) {
                const int cur = t & 1, prv = cur ^ 1;
                // solve(t): needs solve(t-1) (stream order) and apply(t-2): it wrote G[prv], the buffer read here, and was the last
                // reader of the J/D/active buffers of parity `cur`
                if (t >= 2) cudaStreamWaitEvent(ss, ax.evA[prv], 0);
                const int prev_round = (t == 0) ? -1 : (r == 0 ? nb - 2 : r - 1);
                blk_solve2_kernel<<<dim3(npair, bc), 1024, kSolve2Smem, ss>>>(N, nb, r, prev_round, r == 0 ? 0 : 1, t == 0 ? Gbuf[0] : Gbuf[prv], misc0,
                                                                              Jbuf[prv], Dbuf[prv], Jbuf[cur], Dbuf[cur], abuf[cur], counter, ws);
                cudaEventRecord(ax.evS[cur], ss);
                // apply(t): G[cur] -> G[prv] with the rotations of solve(t); apply(t-1) precedes it in stream order
                cudaStreamWaitEvent(st, ax.evS[cur], 0);
                blk_apply2_kernel<<<dim3(N / SB, 2 * npair, bc), 256, kApplySmem, st>>>(N, nb, r, Gbuf[cur], Gbuf[prv], Vu0, Jbuf[cur], Dbuf[cur], abuf[cur], ws);
                cudaEventRecord(ax.evA[prv], st);         // evA[p]: "the apply that wrote G[p] is done"
                count_launch(2);
            }
            int rot = 0;
            if (!check(cudaMemcpyAsync(&rot, counter, sizeof(int), cudaMemcpyDeviceToHost, ss), err, "eigh readback")) return TATRG_ECUDA;
            count_sync(); if (!check(cudaStreamSynchronize(ss), err, "eigh sync")) return TATRG_ECUDA;
            if (verbose) fprintf(stderr, "[tatrg eigh batch=%d N=%d] sweep %d rotations %d\n", bc, N, sweep, rot);
            if (rot == 0) break;
        }
        if (sweep == kMaxBlockSweeps) { if (err) *err = "eigh: block Jacobi did not converge"; return TATRG_ENUMERIC; }
        double* Gfin = Gbuf[t & 1];
        for (int z = 0; z < bc; ++z) { extract_diag_kernel<<<(N + 255) / 256, 256, 0, st>>>(N, Gfin + z * ws, lam_u(z0 + z)); count_launch(); }
        {
            std::vector<FinishItem> fi;
            for (int z = 0; z < bc; ++z) {
                const EighItem& it = items[z0 + z];
                fi.push_back(FinishItem{it.n, lam_u(z0 + z), idx(z0 + z), Vu(z0 + z), it.lam, it.Vt, it.lam_host});
            }
            int rc = finish_batch(st, N, fi, err);
            if (rc != TATRG_OK) return rc;
        }
    }
    return TATRG_OK;
}

int eigh(cudaStream_t st, int n, double* G, double* lam, double* Vt, void* work, std::vector<double>* lam_host, std::string* err) {
    if (n <= 0) return TATRG_OK;
    EighItem it{n, G, lam, Vt, lam_host};
    return eigh_batched(st, 1, &it, work, err);
}

size_t svd_rows_work_bytes(int nv, int len) { return 8 * ((size_t)nv * (len + nv + 2)) + 4096; }

int svd_rows(cudaStream_t st, int nv, int len, const double* X, double* s, double* Ut, double* Vacc, void* work,
             std::vector<double>* s_host, std::string* err) {
    if (nv <= 0 || len <= 0) return TATRG_OK;
    size_t smem = 8 * ((size_t)nv * (len + 1) + (size_t)nv * (nv + 1));
    if (smem > 200 * 1024) { if (err) *err = "svd_rows: matrix too large for shared memory"; return TATRG_EINVAL; }
    static size_t cfg_dev[64] = {0};
    int dev = 0; cudaGetDevice(&dev);
    size_t& cfg = cfg_dev[dev & 63];
    if (smem > cfg) {
        if (!check(cudaFuncSetAttribute(svd_rows_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem), err, "svd attr")) return TATRG_ECUDA;
        cfg = smem;
    }
    double* w = (double*)work;
    double* su = w; w += nv;
    int* idx = (int*)w; w += nv;
    double* Uu = w; w += (size_t)nv * len;
    double* Vu = w;
    svd_rows_kernel<<<1, 1024, smem, st>>>(nv, len, X, su, Uu, Vu); count_launch();
    std::vector<double> sh(nv);
    if (!check(cudaMemcpyAsync(sh.data(), su, sizeof(double) * nv, cudaMemcpyDeviceToHost, st), err, "svd readback")) return TATRG_ECUDA;
    count_sync(); if (!check(cudaStreamSynchronize(st), err, "svd sync")) return TATRG_ECUDA;
    for (int i = 0; i < nv; ++i) if (!std::isfinite(sh[i])) { if (err) *err = "svd_rows: non-finite singular value"; return TATRG_ENUMERIC; }
    std::vector<int> order(nv);
    std::iota(order.begin(), order.end(), 0);
    std::stable_sort(order.begin(), order.end(), [&](int a, int b) { return sh[a] > sh[b]; });
    if (!check(cudaMemcpyAsync(idx, order.data(), sizeof(int) * nv, cudaMemcpyHostToDevice, st), err, "svd upload")) return TATRG_ECUDA;
    if (!check(gather_rows_scaled(st, Ut, Uu, idx, nullptr, nv, len, len), err, "svd gather")) return TATRG_ECUDA;
    if (!check(gather_rows_scaled(st, Vacc, Vu, idx, nullptr, nv, nv, nv), err, "svd gather")) return TATRG_ECUDA;
    if (!check(gather_vec(st, s, su, idx, nv, 1, 1.0), err, "svd gather")) return TATRG_ECUDA;
    count_sync(); if (!check(cudaStreamSynchronize(st), err, "svd sync")) return TATRG_ECUDA;
    if (s_host) { s_host->resize(nv); for (int i = 0; i < nv; ++i) (*s_host)[i] = sh[order[i]]; }
    return TATRG_OK;
}

}  // namespace tatrg
