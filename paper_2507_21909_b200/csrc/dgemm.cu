// dgemm.cu -- FP64 tensor-core GEMM for the Triad-ATRG contractions (Eq. 2.18-2.19 :175, A.4-A.5 :356-361,
// 2.9-2.13 :135-157 are all permute + GEMM).  sm_100a has no tcgen05 kind for f64; the FP64 tensor path is
// mma.sync.m8n8k4.f64 (SASS DMMA), fed here by a 4-stage cp.async pipeline of padded shared-memory tiles.
//
//   C[M,N] (row-major) = alpha * A(m,k) * B(k,n) + beta * C
//   A is stored [M][K] (A_KC: k contiguous) or [K][M];  B is stored [K][N] or [N][K] (B_KC: k contiguous).
//
// Two tile configurations:
//   L: CTA tile 128x128x16, 8 warps as 2(M) x 4(N), warp tile 64x32 = 8x4 DMMA atoms (64 accumulator doubles/thread)
//   S: CTA tile  64x 64x16, 4 warps as 2 x 2,        warp tile 32x32 = 4x4 atoms; for outputs with min(M,N) <= 64
//      (Gram matrices of D^4 x D operands, A.G with G = D x D), where L would spend >= 3/4 of its DMMAs on padding.
// Shared-memory row pitches are = 4 (mod 16) doubles, which makes the 8-byte fragment loads of a half-warp hit
// 16 distinct bank pairs for both storage orders.
// Batched launches take a K of their own for the last batch entry (klast): split-K passes its ragged tail that way.
#include "internal.h"
#include <algorithm>

namespace tatrg {
thread_local Counters* g_counter = nullptr;
thread_local int g_verbose = 0;
thread_local int g_dgemm_tma = 1;
cudaEvent_t Counters::next_event() {
    if (ev_used == ev_pool.size()) { cudaEvent_t e; cudaEventCreate(&e); ev_pool.push_back(e); }
    return ev_pool[ev_used++];
}

namespace {
constexpr int kChunkAlign = 32;    // split-K chunks are multiples of every configuration's BK

template <int BM_, int BN_, int WM_, int WN_, int BK_, int STAGES_>
struct Cfg {
    static constexpr int BM = BM_, BN = BN_, WM = WM_, WN = WN_, BK = BK_, STAGES = STAGES_;
    static constexpr int PITCH_KC = BK + 4;   // operand stored [row][k]: = 4 (mod 16) doubles
    static constexpr int NT = 32 * WM * WN;
    static constexpr int MI = BM / WM / 8, NI = BN / WN / 8;          // atoms per warp
    // an operand tile holds ROWS x BK doubles in either storage order
    static constexpr int tile_doubles(int rows) { return rows * PITCH_KC > BK * (rows + 4) ? rows * PITCH_KC : BK * (rows + 4); }
    static constexpr int TILE_A = tile_doubles(BM), TILE_B = tile_doubles(BN);
    static constexpr int SMEM = STAGES * (TILE_A + TILE_B) * 8;
};
using CfgL = Cfg<128, 128, 2, 4, 16, 4>;     // BK = 32 with 3 stages (221 KB) measured no faster
using CfgS = Cfg<64, 64, 2, 2, 16, 4>;
using CfgT = Cfg<128, 32, 4, 1, 16, 4>;      // tall and skinny: C = A G with G = D x D (M = D^4): HBM-bound, no padded DMMAs along N
using CfgT2 = Cfg<128, 32, 4, 1, 16, 2>;     // the same for K <= 32 (two k-steps: two stages are all it can use): 51 KB, four CTAs per SM
using CfgS2 = Cfg<64, 64, 2, 2, 16, 2>;      // wide outputs with K <= 32 (M4 F, N4 G of Eq. 2.18-2.19): written once, HBM-bound; many small CTAs in flight
using CfgU = Cfg<32, 32, 2, 2, 16, 4>;       // 32 x 32 outputs (Gram matrices of D^4 x D operands, batched over K-chunks)
enum { CFG_AUTO = -1, CFG_L = 0, CFG_S = 1, CFG_T = 2, CFG_U = 3 };

__device__ __forceinline__ void cp16(double* dst, const double* src, bool ok) {
    unsigned d = (unsigned)__cvta_generic_to_shared(dst);
    int n = ok ? 16 : 0;
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;\n" ::"r"(d), "l"(src), "r"(n));
}
__device__ __forceinline__ void cp16u(double* dst, const double* src) {      // unpredicated
    unsigned d = (unsigned)__cvta_generic_to_shared(dst);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" ::"r"(d), "l"(src));
}
__device__ __forceinline__ void cp8(double* dst, const double* src, bool ok) {
    unsigned d = (unsigned)__cvta_generic_to_shared(dst);
    int n = ok ? 8 : 0;
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8, %2;\n" ::"r"(d), "l"(src), "r"(n));
}
__device__ __forceinline__ void cp_commit() { asm volatile("cp.async.commit_group;\n" ::); }
template <int N> __device__ __forceinline__ void cp_wait() { asm volatile("cp.async.wait_group %0;\n" ::"n"(N)); }

__device__ __forceinline__ void dmma(double& d0, double& d1, double a, double b) {
    asm("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
                 : "+d"(d0), "+d"(d1) : "d"(a), "d"(b));
}

// Load one ROWS x 16 operand tile.  KC: global element (r, k) at g[r*ld + k]; else at g[k*ld + r].
// rows = extent of the non-contracted dimension, K = extent of k; r0/k0 tile origin.
template <bool KC, bool V16, int ROWS, int NT, int BK>
__device__ __forceinline__ void load_tile(double* s, const double* __restrict__ g, int64_t ld, int64_t r0, int64_t k0,
                                          int64_t rows, int64_t K, int tid) {
    constexpr int PITCH_MC = ROWS + 4, PITCH_KC = BK + 4, CPR = BK / 2;
    if (KC) {
        if (V16) {
#pragma unroll
            for (int c = tid; c < ROWS * BK / 2; c += NT) {
                int r = c / CPR, kc = (c % CPR) * 2;
                bool ok = (r0 + r < rows) && (k0 + kc < K);
                const double* src = ok ? g + (r0 + r) * ld + k0 + kc : g;
                cp16(s + r * PITCH_KC + kc, src, ok);
            }
        } else {
#pragma unroll
            for (int c = tid; c < ROWS * BK; c += NT) {
                int r = c / BK, kc = c % BK;
                bool ok = (r0 + r < rows) && (k0 + kc < K);
                const double* src = ok ? g + (r0 + r) * ld + k0 + kc : g;
                cp8(s + r * PITCH_KC + kc, src, ok);
            }
        }
    } else {
        if (V16) {
#pragma unroll
            for (int c = tid; c < ROWS * BK / 2; c += NT) {
                int k = c / (ROWS / 2), rc = (c % (ROWS / 2)) * 2;
                bool ok = (k0 + k < K) && (r0 + rc < rows);
                const double* src = ok ? g + (k0 + k) * ld + r0 + rc : g;
                cp16(s + k * PITCH_MC + rc, src, ok);
            }
        } else {
#pragma unroll
            for (int c = tid; c < ROWS * BK; c += NT) {
                int k = c / ROWS, rc = c % ROWS;
                bool ok = (k0 + k < K) && (r0 + rc < rows);
                const double* src = ok ? g + (k0 + k) * ld + r0 + rc : g;
                cp8(s + k * PITCH_MC + rc, src, ok);
            }
        }
    }
}

// The same for the 16-byte path with everything loop-invariant hoisted: the k-loop then spends one pointer add, one
// compare and one cp.async per 16-byte chunk (the generic index arithmetic of load_tile costs ~140 integer instructions
// per k-step, during which neither warp of a scheduler issues DMMAs).  Chunk `it` of a thread sits at a fixed stride
// from its chunk 0 in global and in shared memory:
//   KC: r = tid/(BK/2) + it*NT/(BK/2), kc = 2*(tid%(BK/2))     MC: k = tid/(ROWS/2) + it*NT/(ROWS/2), rc = 2*(tid%(ROWS/2))
template <bool KC, int ROWS, int NT, int BK>
struct TileLoader {
    static constexpr int ITERS = ROWS * BK / 2 / NT;
    static constexpr int HALF = ROWS / 2, CPR = BK / 2;
    static constexpr int PITCH_MC = ROWS + 4, PITCH_KC = BK + 4;
    const double* pk; const double* safe;
    int64_t step_it, step_k;
    unsigned mask; bool full;
    int kofs0, kofs_it, soff0, soff_it;
    __device__ __forceinline__ void init(const double* __restrict__ g, int64_t ld, int64_t r0, int64_t rows, int tid) {
        safe = g;
        if (KC) {
            const int r = tid / CPR, kc = (tid % CPR) * 2;
            pk = g + (r0 + r) * ld + kc; step_it = (int64_t)(NT / CPR) * ld; step_k = BK;
            mask = 0;
#pragma unroll
            for (int it = 0; it < ITERS; ++it) if (r0 + r + it * (NT / CPR) < rows) mask |= 1u << it;
            kofs0 = kc; kofs_it = 0; soff0 = r * PITCH_KC + kc; soff_it = (NT / CPR) * PITCH_KC;
        } else {
            const int k = tid / HALF, rc = (tid % HALF) * 2;
            pk = g + (int64_t)k * ld + r0 + rc; step_it = (int64_t)(NT / HALF) * ld; step_k = (int64_t)BK * ld;
            mask = (r0 + rc < rows) ? 0xffffffffu : 0u;
            kofs0 = k; kofs_it = NT / HALF; soff0 = k * PITCH_MC + rc; soff_it = (NT / HALF) * PITCH_MC;
        }
        full = r0 + ROWS <= rows;       // CTA-uniform
    }
    // tile kt (k origin kt*BK) -> stage buffer s.  Tiles are issued in order kt = 0, 1, 2, ...: `pk` runs along.
    // A tile that lies inside the matrix in both directions takes the unpredicated path: per chunk one 64-bit add and one cp.async.
    __device__ __forceinline__ void issue(double* s, int kt, int64_t K) {
        const double* p = pk;
        pk += step_k;
        if (full && (int64_t)(kt + 1) * BK <= K) {
#pragma unroll
            for (int it = 0; it < ITERS; ++it) { cp16u(s + soff0 + it * soff_it, p); p += step_it; }
            return;
        }
        const int64_t krem = K - (int64_t)kt * BK - kofs0;      // chunk it is inside K iff it*kofs_it < krem
#pragma unroll
        for (int it = 0; it < ITERS; ++it) {
            const bool ok = ((mask >> it) & 1u) && (int64_t)(it * kofs_it) < krem;
            cp16(s + soff0 + it * soff_it, ok ? p + it * step_it : safe, ok);
        }
    }
};

template <class C_, bool A_KC, bool B_KC, bool AV16, bool BV16>
__global__ void __launch_bounds__(C_::NT, C_::NT == 256 ? 1 : (C_::STAGES == 2 ? 4 : 2))
dgemm_kernel(int64_t M, int64_t N, int64_t Kall, int64_t Klast, double alpha, const double* __restrict__ A, int64_t lda,
             const double* __restrict__ B, int64_t ldb, double beta, double* __restrict__ C, int64_t ldc, int64_t sA,
             int64_t sB, int64_t sC, int tiles_m, int lower_only) {
    constexpr int BM = C_::BM, BN = C_::BN, NT = C_::NT, MI = C_::MI, NI = C_::NI, TILE_A = C_::TILE_A, TILE_S = C_::TILE_A + C_::TILE_B;
    constexpr int BK = C_::BK, STAGES = C_::STAGES, PITCH_KC = C_::PITCH_KC;
    constexpr int PA = BM + 4, PB = BN + 4;
    extern __shared__ __align__(16) double smem[];
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int g = lane >> 2, t = lane & 3;
    const int wm = warp / C_::WN, wn = warp % C_::WN;
    // tile order: consecutive CTAs walk down M for a fixed N-panel so that the B panel stays in L2
    const int64_t tile = blockIdx.x;
    const int64_t m0 = (tile % tiles_m) * BM, n0 = (tile / tiles_m) * BN;
    if (lower_only && n0 >= m0 + BM) return;          // symmetric result: tiles strictly above the diagonal are mirrored later
    const int64_t K = (Klast > 0 && blockIdx.z == gridDim.z - 1) ? Klast : Kall;
    A += (int64_t)blockIdx.z * sA; B += (int64_t)blockIdx.z * sB; C += (int64_t)blockIdx.z * sC;

    double acc[MI][NI][2];
#pragma unroll
    for (int i = 0; i < MI; ++i)
#pragma unroll
        for (int j = 0; j < NI; ++j) acc[i][j][0] = acc[i][j][1] = 0.0;

    const int nk = (int)((K + BK - 1) / BK);
    TileLoader<A_KC, BM, NT, BK> ldA; TileLoader<B_KC, BN, NT, BK> ldB;
    if (AV16) ldA.init(A, lda, m0, M, tid);
    if (BV16) ldB.init(B, ldb, n0, N, tid);
    auto load_stage = [&](int kt) {
        double* sa = smem + (kt % STAGES) * TILE_S;
        if (AV16) ldA.issue(sa, kt, K); else load_tile<A_KC, false, BM, NT, BK>(sa, A, lda, m0, (int64_t)kt * BK, M, K, tid);
        if (BV16) ldB.issue(sa + TILE_A, kt, K); else load_tile<B_KC, false, BN, NT, BK>(sa + TILE_A, B, ldb, n0, (int64_t)kt * BK, N, K, tid);
    };
#pragma unroll
    for (int s = 0; s < STAGES - 1; ++s) {
        if (s < nk) load_stage(s);
        cp_commit();
    }
    for (int kt = 0; kt < nk; ++kt) {
        cp_wait<STAGES - 2>();
        __syncthreads();
        {
            int nxt = kt + STAGES - 1;
            if (nxt < nk) load_stage(nxt);
            cp_commit();
        }
        const double* As = smem + (kt % STAGES) * TILE_S;
        const double* Bs = As + TILE_A;
        // fragments of the next 4-deep slice are loaded while the DMMAs of the current one issue (register double buffer)
        double a[2][MI], b[2][NI];
        auto load_frag = [&](int ks, double (&af)[MI], double (&bf)[NI]) {
            const int k = ks * 4 + t;
#pragma unroll
            for (int i = 0; i < MI; ++i) {
                int m = wm * (MI * 8) + i * 8 + g;
                af[i] = A_KC ? As[m * PITCH_KC + k] : As[k * PA + m];
            }
#pragma unroll
            for (int j = 0; j < NI; ++j) {
                int n = wn * (NI * 8) + j * 8 + g;
                bf[j] = B_KC ? Bs[n * PITCH_KC + k] : Bs[k * PB + n];
            }
        };
        load_frag(0, a[0], b[0]);
#pragma unroll
        for (int ks = 0; ks < BK / 4; ++ks) {
            if (ks + 1 < BK / 4) load_frag(ks + 1, a[(ks + 1) & 1], b[(ks + 1) & 1]);
#pragma unroll
            for (int i = 0; i < MI; ++i)
#pragma unroll
                for (int j = 0; j < NI; ++j) dmma(acc[i][j][0], acc[i][j][1], a[ks & 1][i], b[ks & 1][j]);
        }
    }
    cp_wait<0>();
    const bool vec = ((ldc & 1) == 0) && ((((uintptr_t)C) & 15) == 0);
#pragma unroll
    for (int i = 0; i < MI; ++i) {
        int64_t m = m0 + wm * (MI * 8) + i * 8 + g;
        if (m >= M) continue;
#pragma unroll
        for (int j = 0; j < NI; ++j) {
            int64_t n = n0 + wn * (NI * 8) + j * 8 + 2 * t;
            if (n >= N) continue;
            double* c = C + m * ldc + n;
            double v0 = alpha * acc[i][j][0], v1 = alpha * acc[i][j][1];
            if (n + 1 < N) {
                if (beta != 0.0) { v0 += beta * c[0]; v1 += beta * c[1]; }
                if (vec) *reinterpret_cast<double2*>(c) = make_double2(v0, v1);
                else { c[0] = v0; c[1] = v1; }
            } else {
                if (beta != 0.0) v0 += beta * c[0];
                c[0] = v0;
            }
        }
    }
}

struct Args {
    cudaStream_t st; int64_t M, N, K, Klast; double alpha; const double* A; int64_t lda; const double* B; int64_t ldb; double beta;
    double* C; int64_t ldc; int batch; int64_t sA, sB, sC; int force_cfg = CFG_AUTO; bool lower_only = false;
};

template <class C_, bool A_KC, bool B_KC, bool AV, bool BV>
cudaError_t launch(const Args& a) {
    auto kern = dgemm_kernel<C_, A_KC, B_KC, AV, BV>;
    static unsigned long long configured = 0;
    if (first_use_on_device(configured)) {
        cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, C_::SMEM);
        if (e != cudaSuccess) return e;
    }
    int64_t tm = (a.M + C_::BM - 1) / C_::BM, tn = (a.N + C_::BN - 1) / C_::BN;
    dim3 grid((unsigned)(tm * tn), 1, (unsigned)a.batch);
    kern<<<grid, C_::NT, C_::SMEM, a.st>>>(a.M, a.N, a.K, a.Klast, a.alpha, a.A, a.lda, a.B, a.ldb, a.beta, a.C, a.ldc, a.sA, a.sB, a.sC, (int)tm, a.lower_only ? 1 : 0);
    count_launch();
    return cudaGetLastError();
}
template <class C_, bool A_KC, bool B_KC>
cudaError_t pick_vec(bool av, bool bv, const Args& a) {
    if (av && bv) return launch<C_, A_KC, B_KC, true, true>(a);
    if (av) return launch<C_, A_KC, B_KC, true, false>(a);
    if (bv) return launch<C_, A_KC, B_KC, false, true>(a);
    return launch<C_, A_KC, B_KC, false, false>(a);
}
template <class C_>
cudaError_t pick_order(bool a_kc, bool b_kc, bool av, bool bv, const Args& a) {
    if (a_kc && b_kc) return pick_vec<C_, true, true>(av, bv, a);
    if (a_kc && !b_kc) return pick_vec<C_, true, false>(av, bv, a);
    if (!a_kc && b_kc) return pick_vec<C_, false, true>(av, bv, a);
    return pick_vec<C_, false, false>(av, bv, a);
}
// U for outputs of at most 32 x 32, T for N <= 32 below a tall M, S for the other skinny outputs and for launches whose L tiles
// would cover at most a quarter of the 148 SMs (the small products of the subspace iterations: there the number of CTAs in
// flight matters more than the reuse inside one tile), L otherwise.
inline int pick_cfg(int64_t M, int64_t N, int64_t batch = 1) {
    if (M <= 32 && N <= 32) return CFG_U;
    if (N <= 32 && M >= 128) return CFG_T;
    if ((M < N ? M : N) <= 64) return CFG_S;
    const int64_t tl = ((M + CfgL::BM - 1) / CfgL::BM) * ((N + CfgL::BN - 1) / CfgL::BN);
    return tl * batch <= 37 ? CFG_S : CFG_L;
}
inline void cfg_dims(int cfg, int& bm, int& bn, int& per_sm) {
    switch (cfg) {
        case CFG_L: bm = CfgL::BM; bn = CfgL::BN; per_sm = 1; break;
        case CFG_S: bm = CfgS::BM; bn = CfgS::BN; per_sm = 2; break;
        case CFG_T: bm = CfgT::BM; bn = CfgT::BN; per_sm = 2; break;
        default: bm = CfgU::BM; bn = CfgU::BN; per_sm = 4; break;
    }
}

cudaError_t dgemm_raw(bool transa, bool transb, const Args& a) {
    if (a.M <= 0 || a.N <= 0 || a.batch <= 0) return cudaSuccess;
    // transa == false: A stored [M][K] -> k contiguous.  transb == false: B stored [K][N] -> n contiguous.
    const bool a_kc = !transa, b_kc = transb;
    // 16-byte cp.async needs: even leading dimension, 16B-aligned base and batch stride, even contiguous extent
    auto v16 = [](const double* p, int64_t ld, int64_t contig_extent, int64_t bs) {
        return ((uintptr_t)p % 16 == 0) && (ld % 2 == 0) && (contig_extent % 2 == 0) && (bs % 2 == 0);
    };
    const bool kodd = (a.K % 2 != 0) || (a.Klast % 2 != 0);
    const bool av = v16(a.A, a.lda, a_kc ? (kodd ? 1 : 2) : a.M, a.sA), bv = v16(a.B, a.ldb, b_kc ? (kodd ? 1 : 2) : a.N, a.sB);
    const int cfg = a.force_cfg != CFG_AUTO ? a.force_cfg : pick_cfg(a.M, a.N, a.batch);
    if ((cfg == CFG_L || cfg == CFG_S) && a.K <= 2 * CfgS2::BK && a.Klast == 0 && a.force_cfg == CFG_AUTO && !a.lower_only && a.M * a.N >= (1 << 22))
        return pick_order<CfgS2>(a_kc, b_kc, av, bv, a);
    // the 128 x 128 tile fed by TMA (dgemm_tma.cu) whenever the operands meet the tensor-map alignment rules
    if (cfg == CFG_L && g_dgemm_tma && a.Klast == 0) {
        cudaError_t e = dgemm_tma(a.st, a_kc, b_kc, a.M, a.N, a.K, a.alpha, a.A, a.lda, a.B, a.ldb, a.beta, a.C, a.ldc, a.batch, a.sA, a.sB, a.sC, a.lower_only);
        if (e != cudaErrorNotSupported) return e;
    }
    switch (cfg) {
        case CFG_L: return pick_order<CfgL>(a_kc, b_kc, av, bv, a);
        case CFG_S: return pick_order<CfgS>(a_kc, b_kc, av, bv, a);
        case CFG_T: return (a.K <= 2 * CfgT2::BK && a.Klast == 0) ? pick_order<CfgT2>(a_kc, b_kc, av, bv, a) : pick_order<CfgT>(a_kc, b_kc, av, bv, a);
        default: return pick_order<CfgU>(a_kc, b_kc, av, bv, a);
    }
}
}  // namespace

static cudaError_t dgemm_klast(cudaStream_t st, bool transa, bool transb, int64_t M, int64_t N, int64_t K, int64_t Klast, double alpha,
                               const double* A, int64_t lda, const double* B, int64_t ldb, double beta, double* C, int64_t ldc, int batch,
                               int64_t sA, int64_t sB, int64_t sC, int force_cfg = CFG_AUTO, bool lower_only = false) {
    if (M <= 0 || N <= 0 || batch <= 0) return cudaSuccess;
    Counters* c = g_counter;
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    const double kk = Klast > 0 ? (double)K * (batch - 1) + (double)Klast : (double)K * batch;
    // lower_only: only the tiles on and below the diagonal are computed (counted as such)
    double mn = (double)M * (double)N;
    if (lower_only) {
        int bm_, bn_, psm_;
        cfg_dims(force_cfg != CFG_AUTO ? force_cfg : pick_cfg(M, N, batch), bm_, bn_, psm_);
        const int64_t bm = bm_, bn = bn_;
        mn = 0;
        for (int64_t m0 = 0; m0 < M; m0 += bm)
            for (int64_t n0 = 0; n0 < N && n0 < m0 + bm; n0 += bn) mn += (double)std::min(bm, M - m0) * (double)std::min(bn, N - n0);
    }
    if (c) { c->gemm_flops += 2.0 * mn * kk; c->gemm_calls += 1; }
    if (c && c->time_kernels) { e0 = c->next_event(); e1 = c->next_event(); cudaEventRecord(e0, st); }
    cudaError_t e = cudaSuccess;
    // grid.z carries the batch: split very large batches
    for (int b0 = 0; b0 < batch && e == cudaSuccess; b0 += 32768) {
        int nb = batch - b0 < 32768 ? batch - b0 : 32768;
        Args a{st, M, N, K, (b0 + nb == batch) ? Klast : 0, alpha, A + (int64_t)b0 * sA, lda, B + (int64_t)b0 * sB, ldb, beta,
               C + (int64_t)b0 * sC, ldc, nb, sA, sB, sC, force_cfg, lower_only};
        e = dgemm_raw(transa, transb, a);
    }
    if (e0) { cudaEventRecord(e1, st); c->gemm_ev.push_back({e0, e1}); c->gemm_shapes.push_back({M, N, (int64_t)(kk / batch), batch, transa, transb, mn / ((double)M * (double)N)}); }
    return e;
}

cudaError_t dgemm(cudaStream_t st, bool transa, bool transb, int64_t M, int64_t N, int64_t K, double alpha, const double* A,
                  int64_t lda, const double* B, int64_t ldb, double beta, double* C, int64_t ldc, int batch, int64_t sA,
                  int64_t sB, int64_t sC) {
    return dgemm_klast(st, transa, transb, M, N, K, 0, alpha, A, lda, B, ldb, beta, C, ldc, batch, sA, sB, sC);
}

// ---- split-K ---------------------------------------------------------------------------------------------------
namespace {
// Number of K-chunks for a non-batched GEMM: the smallest split whose CTA count fills whole waves of the 148 SMs
// (>= 93 % of the last wave used), chunks of >= 256, partials capped at 64 M doubles.  1 = no split.
int splitk_count(int64_t M, int64_t N, int64_t K, bool lower_only = false) {
    int bm, bn, per_sm;
    cfg_dims(pick_cfg(M, N), bm, bn, per_sm);
    int64_t tiles = ((M + bm - 1) / bm) * ((N + bn - 1) / bn);
    if (lower_only) {      // only the tiles on and below the diagonal do work
        tiles = 0;
        for (int64_t m0 = 0; m0 < M; m0 += bm) for (int64_t n0 = 0; n0 < N && n0 < m0 + bm; n0 += bn) ++tiles;
    }
    const int64_t slots = 148 * per_sm;
    auto eff = [&](int64_t ctas) { int64_t waves = (ctas + slots - 1) / slots; return (double)ctas / (double)(waves * slots); };
    if (K < 256 || eff(tiles) >= 0.93) return 1;
    // chunks of >= 256 for outputs that already give every SM a tile; down to 64 for the small products (a few tiles only)
    const int64_t min_chunk = tiles >= slots ? 256 : (tiles * 4 >= slots ? 128 : 64);
    int64_t maxs = K / min_chunk;
    if (maxs > 1024) maxs = 1024;
    const int64_t cap = (64LL << 20) / (M * N > 0 ? M * N : 1);
    if (maxs > cap) maxs = cap;
    int best = 1; double best_eff = eff(tiles);
    for (int64_t sp = 2; sp <= maxs; ++sp) {
        const double e = eff(tiles * sp);
        if (e >= 0.93) return (int)sp;
        if (e > best_eff * 1.1) { best_eff = e; best = (int)sp; }
    }
    return best;
}
__global__ void splitk_reduce_kernel(const double* __restrict__ part, int nsplit, int64_t MN, int64_t N, double alpha,
                                     double* __restrict__ C, int64_t ldc) {
    for (int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; e < MN; e += (int64_t)gridDim.x * blockDim.x) {
        double s = 0;
        for (int k = 0; k < nsplit; ++k) s += part[(int64_t)k * MN + e];
        int64_t r = e / N, c = e - r * N;
        C[r * ldc + c] = alpha * s;
    }
}
// Many partials of a small output (Gram matrices of very tall operands: 64 x 64 from 256 chunks): the sum over the
// partials is itself spread over 8 threads per element (4 independent accumulators each), combined in shared memory.
__global__ void __launch_bounds__(256) splitk_reduce_wide_kernel(const double* __restrict__ part, int nsplit, int64_t MN, int64_t N, double alpha,
                                                                 double* __restrict__ C, int64_t ldc) {
    __shared__ double red[8][33];
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    const int64_t e = (int64_t)blockIdx.x * 32 + lane;
    double s0 = 0, s1 = 0, s2 = 0, s3 = 0;
    if (e < MN) {
        int k = w;
        for (; k + 24 < nsplit; k += 32) {
            s0 += part[(int64_t)k * MN + e]; s1 += part[(int64_t)(k + 8) * MN + e];
            s2 += part[(int64_t)(k + 16) * MN + e]; s3 += part[(int64_t)(k + 24) * MN + e];
        }
        for (; k < nsplit; k += 8) s0 += part[(int64_t)k * MN + e];
    }
    red[w][lane] = (s0 + s1) + (s2 + s3);
    __syncthreads();
    if (w == 0 && e < MN) {
        double s = 0;
#pragma unroll
        for (int j = 0; j < 8; ++j) s += red[j][lane];
        const int64_t r = e / N, c = e - r * N;
        C[r * ldc + c] = alpha * s;
    }
}
}  // namespace

int64_t dgemm_splitk_doubles(int64_t M, int64_t N, int64_t K, bool lower_only) {
    int s = splitk_count(M, N, K, lower_only);
    return s > 1 ? (int64_t)s * M * N : 0;
}

cudaError_t dgemm_splitk(cudaStream_t st, bool transa, bool transb, int64_t M, int64_t N, int64_t K, double alpha, const double* A,
                         int64_t lda, const double* B, int64_t ldb, double* C, int64_t ldc, double* part, bool lower_only) {
    int ns = splitk_count(M, N, K, lower_only);
    if (ns <= 1 || part == nullptr) return dgemm_klast(st, transa, transb, M, N, K, 0, alpha, A, lda, B, ldb, 0.0, C, ldc, 1, 0, 0, 0, CFG_AUTO, lower_only);
    // chunk: multiple of BK; the last batch entry takes the ragged tail (klast)
    int64_t chunk = ((K + ns - 1) / ns + kChunkAlign - 1) / kChunkAlign * kChunkAlign;
    int nchunks = (int)((K + chunk - 1) / chunk);
    int64_t tail = K - (int64_t)(nchunks - 1) * chunk;
    const int64_t stepA = transa ? chunk * lda : chunk, stepB = transb ? chunk : chunk * ldb;
    cudaError_t e = dgemm_klast(st, transa, transb, M, N, chunk, tail == chunk ? 0 : tail, 1.0, A, lda, B, ldb, 0.0, part, N, nchunks,
                                stepA, stepB, M * N, pick_cfg(M, N), lower_only);
    if (e != cudaSuccess) return e;
    int64_t MN = M * N;
    if (nchunks >= 16 && MN <= (1 << 18)) {
        splitk_reduce_wide_kernel<<<(unsigned)((MN + 31) / 32), 256, 0, st>>>(part, nchunks, MN, N, alpha, C, ldc);
    } else {
        int64_t blocks = (MN + 255) / 256; if (blocks > 148 * 8) blocks = 148 * 8;
        splitk_reduce_kernel<<<(unsigned)blocks, 256, 0, st>>>(part, nchunks, MN, N, alpha, C, ldc);
    }
    count_launch();
    return cudaGetLastError();
}

}  // namespace tatrg
