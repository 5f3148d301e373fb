// dgemm_tma.cu -- the 128 x 128 x 16 DMMA tile of dgemm.cu fed by TMA instead of cp.async (north_star: "contraction GEMMs on
// FP64 tensor cores (DMMA) with TMA-fed shared-memory tiles"; the contractions are PAPER.md Eq. 2.18-2.19 :175, 2.9-2.17, A.2-A.11).
//
//   * one producer warp: an elected lane issues cp.async.bulk.tensor (3-D tensor maps: contiguous leg, strided leg, batch) into a
//     6-stage ring of dense 128-byte-swizzled tiles (CU_TENSOR_MAP_SWIZZLE_128B), completion through mbarrier transaction counts;
//   * eight consumer warps (2 x 4, warp tile 64 x 32 = 8 x 4 DMMA atoms, as in dgemm.cu): mbarrier wait on `full`, fragment loads +
//     DMMA, one mbarrier arrive per warp on `empty`.  No CTA-wide barrier and no address arithmetic for global memory in the k-loop;
//   * ragged M, N, K need no predicates: the tensor maps zero-fill what lies outside the operand.
//
// Shared-memory layout.  An operand tile is 128 rows x 16 k.  Stored k-contiguous ([row][k], "KC") it is ONE box of 128 rows of 128
// bytes; stored row-contiguous ([k][row], "MC") it is EIGHT boxes of 16 k-rows x 16 rows (the swizzle span limits the contiguous
// extent of a box to 128 bytes).  The swizzle XORs the 16-byte chunk index of a 128-byte line with (line index mod 8).
// A DMMA fragment load reads element (row g, k t) for lane 4 g + t, a half-warp (g = 0..3) per wavefront; the rows an atom works on
// are permuted so that those 16 lanes hit 16 distinct 8-byte bank pairs:
//   KC: atom row g -> tile row 8 i + P[g], P = 0,2,4,6,1,3,5,7     MC: atoms 2 j, 2 j + 1 share box j: rows 0,1,8,9,2,3,10,11 | +4
// The C rows follow the A permutation for free; for B only the MC order keeps a lane's two C columns adjacent, so B in KC order is
// read with the natural mapping (2-way conflict on 4 of the 12 loads of a slice; none of the large contractions has that order).
#include "internal.h"
#include <cuda.h>
#include <mutex>

namespace tatrg {
namespace {

constexpr int BM = 128, BN = 128, BK = 16, STAGES = 6;
constexpr int TILE_BYTES = 128 * BK * 8;                 // 16 KB per operand tile
constexpr int STAGE_BYTES = 2 * TILE_BYTES;
constexpr int SMEM_BYTES = STAGES * STAGE_BYTES + 1024;  // + slack for the 1024-byte alignment the swizzle needs
constexpr int NCONS = 256, NT = NCONS + 32;
constexpr int WN = 4, MI = 8, NI = 4;

__device__ __forceinline__ unsigned smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(unsigned bar, unsigned count) { asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;\n" ::"r"(bar), "r"(count)); }
__device__ __forceinline__ void mbar_expect_tx(unsigned bar, unsigned bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;\n" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(unsigned bar) { asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];\n" ::"r"(bar) : "memory"); }
__device__ __forceinline__ void mbar_wait(unsigned bar, unsigned parity) {
    asm volatile(
        "{\n .reg .pred p;\n WAIT_%=:\n mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n @p bra DONE_%=;\n bra WAIT_%=;\n DONE_%=:\n}\n" ::"r"(bar),
        "r"(parity)
        : "memory");
}
__device__ __forceinline__ void tma_load_3d(unsigned dst, const CUtensorMap* map, unsigned bar, int c0, int c1, int c2) {
    asm volatile("cp.async.bulk.tensor.3d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5}], [%2];\n" ::"r"(dst),
                 "l"((unsigned long long)map), "r"(bar), "r"(c0), "r"(c1), "r"(c2)
                 : "memory");
}
__device__ __forceinline__ void dmma(double& d0, double& d1, double a, double b) {
    asm("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n" : "+d"(d0), "+d"(d1) : "d"(a), "d"(b));
}

// byte offset, inside a swizzled operand tile, of the fragment element of this lane for atom i and 4-deep slice ks
template <bool KC>
struct Frag {
    int base, c0, c1;      // KC: c0 only.  MC: c0 / c1 for even / odd atoms
    // wrow: first tile row of the warp; perm: permuted atom rows (always for MC)
    __device__ __forceinline__ void init(int wrow, int g, int t, bool perm) {
        if (KC) {
            const int r = perm ? (((g & 3) << 1) | (g >> 2)) : g;
            base = (wrow + r) * 128 + ((t & 1) << 3);
            c0 = (t >> 1) ^ r; c1 = 0;
        } else {
            base = (wrow >> 4) * 2048 + t * 128 + ((g & 1) << 3);
            const int h = (((g >> 1) & 1) << 2) | ((g >> 2) & 1);      // (row in box) >> 1 for an even atom; odd atoms add 2
            c0 = h ^ t; c1 = (h | 2) ^ t;
        }
    }
    __device__ __forceinline__ int off(int i, int ks) const {
        if (KC) return base + i * 1024 + (((2 * ks) ^ c0) << 4);
        return base + (i >> 1) * 2048 + ks * 512 + ((((i & 1) ? c1 : c0) ^ ((ks & 1) << 2)) << 4);
    }
};
// tile row an atom row stands for (the C row / column of the accumulators): q = g for A, q = 2 t for B
template <bool KC> __device__ __forceinline__ int tile_row(int i, int q, bool perm) {
    if (KC) return i * 8 + (perm ? (((q & 3) << 1) | (q >> 2)) : q);
    return (i >> 1) * 16 + ((q & 1) | (((q >> 1) & 1) << 3) | (((q >> 2) & 1) << 1) | ((i & 1) << 2));
}

template <bool A_KC, bool B_KC>
__global__ void __launch_bounds__(NT, 1)
dgemm_tma_kernel(const __grid_constant__ CUtensorMap mapA, const __grid_constant__ CUtensorMap mapB, int64_t M, int64_t N, int64_t K,
                 double alpha, double beta, double* __restrict__ C, int64_t ldc, int64_t sC, int tiles_m, int lower_only, int zA, int zB) {
    extern __shared__ unsigned char smem_raw[];
    __shared__ __align__(8) unsigned long long bars[2 * STAGES];      // full[0..STAGES), empty[STAGES..2 STAGES)
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int64_t tile = blockIdx.x;
    const int64_t m0 = (tile % tiles_m) * BM, n0 = (tile / tiles_m) * BN;
    if (lower_only && n0 >= m0 + BM) return;
    const unsigned sbase = (smem_u32(smem_raw) + 1023u) & ~1023u;
    unsigned char* tiles = smem_raw + (sbase - smem_u32(smem_raw));
    const unsigned bar0 = smem_u32(bars);
    if (tid == 0) {
        for (int s = 0; s < STAGES; ++s) { mbar_init(bar0 + 8 * s, 1); mbar_init(bar0 + 8 * (STAGES + s), NCONS / 32); }
        asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
        asm volatile("fence.proxy.async.shared::cta;\n" ::: "memory");
    }
    __syncthreads();
    const int nk = (int)((K + BK - 1) / BK);

    if (warp == NCONS / 32) {
        // ---- producer ----
        if (lane == 0) {
            const int z = blockIdx.z;
            for (int kt = 0; kt < nk; ++kt) {
                const int s = kt % STAGES;
                mbar_wait(bar0 + 8 * (STAGES + s), ((kt / STAGES) & 1) ^ 1);
                const unsigned full = bar0 + 8 * s, dst = sbase + s * STAGE_BYTES;
                mbar_expect_tx(full, STAGE_BYTES);
                const int k0 = kt * BK;
                if (A_KC) tma_load_3d(dst, &mapA, full, k0, (int)m0, z * zA);
                else
#pragma unroll
                    for (int j = 0; j < 8; ++j) tma_load_3d(dst + j * 2048, &mapA, full, (int)m0 + 16 * j, k0, z * zA);
                if (B_KC) tma_load_3d(dst + TILE_BYTES, &mapB, full, k0, (int)n0, z * zB);
                else
#pragma unroll
                    for (int j = 0; j < 8; ++j) tma_load_3d(dst + TILE_BYTES + j * 2048, &mapB, full, (int)n0 + 16 * j, k0, z * zB);
            }
        }
        return;
    }
    // ---- consumers ----
    const int g = lane >> 2, t = lane & 3;
    const int wm = warp / WN, wn = warp % WN;
    Frag<A_KC> fa; Frag<B_KC> fb;
    fa.init(wm * 64, g, t, true);
    fb.init(wn * 32, g, t, !B_KC);
    double acc[MI][NI][2];
#pragma unroll
    for (int i = 0; i < MI; ++i)
#pragma unroll
        for (int j = 0; j < NI; ++j) acc[i][j][0] = acc[i][j][1] = 0.0;

    for (int kt = 0; kt < nk; ++kt) {
        const int s = kt % STAGES;
        mbar_wait(bar0 + 8 * s, (kt / STAGES) & 1);
        const unsigned char* As = tiles + s * STAGE_BYTES;
        const unsigned char* Bs = As + TILE_BYTES;
        double a[2][MI], b[2][NI];
        auto load_frag = [&](int ks, double (&af)[MI], double (&bf)[NI]) {
#pragma unroll
            for (int i = 0; i < MI; ++i) af[i] = *reinterpret_cast<const double*>(As + fa.off(i, ks));
#pragma unroll
            for (int j = 0; j < NI; ++j) bf[j] = *reinterpret_cast<const double*>(Bs + fb.off(j, ks));
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
        __syncwarp();
        if (lane == 0) mbar_arrive(bar0 + 8 * (STAGES + s));
    }
    C += (int64_t)blockIdx.z * sC;
    const bool vec = ((ldc & 1) == 0) && ((((uintptr_t)C) & 15) == 0);
#pragma unroll
    for (int i = 0; i < MI; ++i) {
        const int64_t m = m0 + wm * 64 + tile_row<A_KC>(i, g, true);
        if (m >= M) continue;
#pragma unroll
        for (int j = 0; j < NI; ++j) {
            const int64_t n = n0 + wn * 32 + tile_row<B_KC>(j, 2 * t, !B_KC);
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

typedef CUresult (*EncodeTiled)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*, const cuuint32_t*,
                                const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
EncodeTiled encoder() {      // the driver entry point through the runtime (the library links cudart only)
    static EncodeTiled fn = nullptr;
    static std::once_flag once;
    std::call_once(once, []() {
        void* p = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) == cudaSuccess && q == cudaDriverEntryPointSuccess) fn = (EncodeTiled)p;
    });
    return fn;
}
// 3-D map of one operand: kc: element (row, k) at p[row * ld + k], else at p[k * ld + row]; third leg = batch (extent 1 when broadcast)
bool make_map(CUtensorMap* map, const double* p, bool kc, int64_t rows, int64_t K, int64_t ld, int batch, int64_t bstride) {
    EncodeTiled enc = encoder();
    if (!enc) return false;
    const cuuint64_t inner = kc ? K : rows, outer = kc ? rows : K;
    const cuuint64_t dims[3] = {inner, outer, (cuuint64_t)batch};
    const cuuint64_t strides[2] = {(cuuint64_t)ld * 8, batch > 1 ? (cuuint64_t)bstride * 8 : (cuuint64_t)ld * 8 * outer};
    const cuuint32_t box[3] = {16, kc ? 128u : 16u, 1};
    const cuuint32_t estr[3] = {1, 1, 1};
    return enc(map, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 3, (void*)p, dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B,
               CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

template <bool A_KC, bool B_KC>
cudaError_t launch(cudaStream_t st, const CUtensorMap& ma, const CUtensorMap& mb, int64_t M, int64_t N, int64_t K, double alpha, double beta, double* C,
                   int64_t ldc, int batch, int64_t sC, bool lower_only, int zA, int zB) {
    auto kern = dgemm_tma_kernel<A_KC, B_KC>;
    static unsigned long long configured = 0;
    if (first_use_on_device(configured)) {
        cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM_BYTES);
        if (e != cudaSuccess) return e;
    }
    const int64_t tm = (M + BM - 1) / BM, tn = (N + BN - 1) / BN;
    kern<<<dim3((unsigned)(tm * tn), 1, (unsigned)batch), NT, SMEM_BYTES, st>>>(ma, mb, M, N, K, alpha, beta, C, ldc, sC, (int)tm, lower_only ? 1 : 0, zA, zB);
    count_launch();
    return cudaGetLastError();
}
}  // namespace

// What the tensor maps need: 16-byte aligned bases, leading dimensions and batch strides that are multiples of 16 bytes, extents
// below 2^31.  A batch stride of 0 (broadcast operand) becomes a map without batch leg.
bool dgemm_tma_applicable(int64_t M, int64_t N, int64_t K, const double* A, int64_t lda, const double* B, int64_t ldb, int batch, int64_t sA, int64_t sB) {
    if (M < 1 || N < 1 || K < 1 || batch < 1 || batch > 65535) return false;
    if (M >= (1LL << 31) || N >= (1LL << 31) || K >= (1LL << 31)) return false;
    if (((uintptr_t)A & 15) || ((uintptr_t)B & 15) || (lda & 1) || (ldb & 1) || (sA & 1) || (sB & 1)) return false;
    if (lda * 8 >= (1LL << 40) || ldb * 8 >= (1LL << 40) || sA * 8 >= (1LL << 40) || sB * 8 >= (1LL << 40)) return false;
    return encoder() != nullptr;
}

cudaError_t dgemm_tma(cudaStream_t st, bool a_kc, bool b_kc, int64_t M, int64_t N, int64_t K, double alpha, const double* A, int64_t lda, const double* B,
                      int64_t ldb, double beta, double* C, int64_t ldc, int batch, int64_t sA, int64_t sB, int64_t sC, bool lower_only) {
    if (!dgemm_tma_applicable(M, N, K, A, lda, B, ldb, batch, sA, sB)) return cudaErrorNotSupported;
    CUtensorMap ma, mb;
    const int zA = (batch > 1 && sA != 0) ? 1 : 0, zB = (batch > 1 && sB != 0) ? 1 : 0;
    if (!make_map(&ma, A, a_kc, M, K, lda, zA ? batch : 1, sA) || !make_map(&mb, B, b_kc, N, K, ldb, zB ? batch : 1, sB)) return cudaErrorNotSupported;
    if (a_kc && b_kc) return launch<true, true>(st, ma, mb, M, N, K, alpha, beta, C, ldc, batch, sC, lower_only, zA, zB);
    if (a_kc) return launch<true, false>(st, ma, mb, M, N, K, alpha, beta, C, ldc, batch, sC, lower_only, zA, zB);
    if (b_kc) return launch<false, true>(st, ma, mb, M, N, K, alpha, beta, C, ldc, batch, sC, lower_only, zA, zB);
    return launch<false, false>(st, ma, mb, M, N, K, alpha, beta, C, ldc, batch, sC, lower_only, zA, zB);
}

}  // namespace tatrg
