// permute.cu -- leg permutation of a dense row-major FP64 tensor (the reshapes between the contractions of
// PAPER.md Eq. 2.18-2.19 :175, A.2-A.5 :345-361, and the axis rotation of Fig. 5(f) :193).  HBM-bound:
// out leg i = in leg perm[i].  Adjacent legs that stay adjacent are merged on the host; if the innermost leg
// is preserved the copy is coalesced on both sides directly, otherwise a 32x32 (or 64x64) tile goes through
// padded shared memory so that reads run along the input's innermost leg and writes along the output's.
#include "internal.h"
#include <cstdlib>

namespace tatrg {
namespace {
struct PermArgs {
    int nd;             // number of "outer" legs (all but the tile legs for the tiled kernel)
    int64_t ext[8];     // extents of the outer legs (in OUTPUT order)
    int64_t sin[8];     // their strides in the input
    int64_t sout[8];    // their strides in the output
};

// innermost leg preserved: element-wise with both sides coalesced along the innermost leg
__global__ void permute_rows_kernel(PermArgs a, int64_t inner, int64_t n_rows, const double* __restrict__ in, double* __restrict__ out) {
    // one block row = one (outer index) row of `inner` contiguous elements, several rows per block if inner small
    int64_t total = n_rows * inner;
    for (int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; e < total; e += (int64_t)gridDim.x * blockDim.x) {
        int64_t row = e / inner, c = e - row * inner;
        int64_t off_in = 0, r = row;
#pragma unroll 1
        for (int d = a.nd - 1; d >= 0; --d) { int64_t q = r / a.ext[d]; int64_t i = r - q * a.ext[d]; r = q; off_in += i * a.sin[d]; }
        out[e] = in[off_in + c];
    }
}

// general case: tile over (A = input-innermost leg, B = output-innermost leg)
template <int T>
__global__ void permute_tiled_kernel(PermArgs a, int64_t extA, int64_t extB, int64_t sinB, int64_t soutA, int64_t tilesA,
                                     int64_t tilesB, const double* __restrict__ in, double* __restrict__ out) {
    __shared__ double tile[T][T + 1];
    int64_t blk = blockIdx.x;
    int64_t ta = blk % tilesA; blk /= tilesA;
    int64_t tb = blk % tilesB; blk /= tilesB;
    int64_t off_in = 0, off_out = 0, r = blk;
#pragma unroll 1
    for (int d = a.nd - 1; d >= 0; --d) { int64_t q = r / a.ext[d]; int64_t i = r - q * a.ext[d]; r = q; off_in += i * a.sin[d]; off_out += i * a.sout[d]; }
    const int tx = threadIdx.x, ty = threadIdx.y;  // blockDim = (T, 8)
    const int64_t a0 = ta * T, b0 = tb * T;
#pragma unroll
    for (int j = ty; j < T; j += 8) {
        int64_t ia = a0 + tx, ib = b0 + j;
        if (ia < extA && ib < extB) tile[j][tx] = in[off_in + ib * sinB + ia];
    }
    __syncthreads();
#pragma unroll
    for (int j = ty; j < T; j += 8) {
        int64_t ia = a0 + j, ib = b0 + tx;
        if (ia < extA && ib < extB) out[off_out + ia * soutA + ib] = tile[tx][j];
    }
}

// innermost leg preserved, vectorised: one warp per "run" = all rows that share every outer index but the last one.
// A run is ext_last rows of `inner` contiguous doubles, contiguous in the output and strided (sin_last) in the input;
// the outer index is decoded once per run, lanes then walk the run in 16-byte units.
__global__ void __launch_bounds__(256) permute_runs_kernel(PermArgs a, int64_t ext_last, int64_t sin_last, int64_t inner, int64_t nruns,
                                                           int64_t chunk_rows, int64_t chunks, const double* __restrict__ in, double* __restrict__ out) {
    const int lane = threadIdx.x & 31;
    const int64_t warps = (int64_t)gridDim.x * (blockDim.x >> 5);
    const int h = (int)(inner >> 1);                      // 16-byte units per row
    const int64_t rstride = sin_last >> 1;
    const int drow = 32 / h, dcol = 32 - drow * h;
    for (int64_t w = (int64_t)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5); w < nruns * chunks; w += warps) {
        const int64_t run = w / chunks, ch = w - run * chunks;
        int64_t off_in = 0, r = run;
#pragma unroll 1
        for (int d = a.nd - 1; d >= 0; --d) { int64_t q = r / a.ext[d]; int64_t i = r - q * a.ext[d]; r = q; off_in += i * a.sin[d]; }
        const int64_t row0 = ch * chunk_rows;
        const int64_t nrows = (ext_last - row0 < chunk_rows) ? ext_last - row0 : chunk_rows;
        const double2* src = reinterpret_cast<const double2*>(in + off_in + row0 * sin_last);
        double2* dst = reinterpret_cast<double2*>(out + (run * ext_last + row0) * inner);
        const int64_t units = nrows * h;
        int row = lane / h, col = lane - row * h;         // position of unit `lane`
#pragma unroll 4
        for (int64_t u = lane; u < units; u += 32) {
            dst[u] = src[(int64_t)row * rstride + col];
            row += drow; col += dcol;
            if (col >= h) { col -= h; ++row; }
        }
    }
}

// general case, vectorised: 64 x 64 tile over (A = input-innermost leg, B = output-innermost leg), 16-byte global
// accesses on both sides, 8-byte shared-memory accesses with pitch 65.
__global__ void __launch_bounds__(256) permute_tiled64_kernel(PermArgs a, int64_t extA, int64_t extB, int64_t sinB, int64_t soutA, int64_t tilesA,
                                                              int64_t tilesB, const double* __restrict__ in, double* __restrict__ out) {
    __shared__ double tile[64][65];                       // tile[b][a]
    int64_t blk = blockIdx.x;
    int64_t ta = blk % tilesA; blk /= tilesA;
    int64_t tb = blk % tilesB; blk /= tilesB;
    int64_t off_in = 0, off_out = 0, r = blk;
#pragma unroll 1
    for (int d = a.nd - 1; d >= 0; --d) { int64_t q = r / a.ext[d]; int64_t i = r - q * a.ext[d]; r = q; off_in += i * a.sin[d]; off_out += i * a.sout[d]; }
    const int tid = threadIdx.x, c2 = (tid & 31) * 2, r0 = tid >> 5;       // 32 lanes x 16 B = one 64-double row; 8 rows per pass
    const int64_t a0 = ta * 64, b0 = tb * 64;
#pragma unroll
    for (int j = r0; j < 64; j += 8) {
        const int64_t ia = a0 + c2, ib = b0 + j;
        if (ia < extA && ib < extB) {                     // extA even: ia + 1 < extA too
            const double2 v = *reinterpret_cast<const double2*>(in + off_in + ib * sinB + ia);
            tile[j][c2] = v.x; tile[j][c2 + 1] = v.y;
        }
    }
    __syncthreads();
#pragma unroll
    for (int j = r0; j < 64; j += 8) {
        const int64_t ia = a0 + j, ib = b0 + c2;
        if (ia < extA && ib < extB)
            *reinterpret_cast<double2*>(out + off_out + ia * soutA + ib) = make_double2(tile[c2][j], tile[c2 + 1][j]);
    }
}
}  // namespace

static cudaError_t permute_raw(cudaStream_t st, int nd, const int64_t* dims, const int* perm, const double* in, double* out);
cudaError_t permute(cudaStream_t st, int nd, const int64_t* dims, const int* perm, const double* in, double* out) {
    Counters* c = g_counter;
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    if (c) { int64_t t = 1; for (int i = 0; i < nd; ++i) t *= dims[i]; c->permuted_bytes += 16 * t; c->permute_calls += 1; }
    if (c && c->time_kernels) { e0 = c->next_event(); e1 = c->next_event(); cudaEventRecord(e0, st); }
    cudaError_t e = permute_raw(st, nd, dims, perm, in, out);
    if (e0) { cudaEventRecord(e1, st); c->perm_ev.push_back({e0, e1}); int64_t t = 1; for (int i = 0; i < nd; ++i) t *= dims[i]; c->perm_ev_bytes.push_back(16 * t); }
    return e;
}
static cudaError_t permute_raw(cudaStream_t st, int nd, const int64_t* dims, const int* perm, const double* in, double* out) {
    if (nd < 1 || nd > 8) return cudaErrorInvalidValue;
    // drop unit legs, then merge input legs that remain adjacent and in order in the output
    int64_t d[8]; int p[8]; int n = 0;
    {
        int map[8]; int m = 0;
        for (int i = 0; i < nd; ++i) { map[i] = (dims[i] != 1) ? m : -1; if (dims[i] != 1) d[m++] = dims[i]; }
        for (int i = 0; i < nd; ++i) if (map[perm[i]] >= 0) p[n++] = map[perm[i]];
        if (n == 0) { cudaError_t e = cudaMemcpyAsync(out, in, 8, cudaMemcpyDeviceToDevice, st); count_launch(); return e; }
    }
    int64_t total = 1; for (int i = 0; i < n; ++i) total *= d[i];
    if (total == 0) return cudaSuccess;
    // merge: output legs p[i], p[i+1] with p[i+1] == p[i]+1 form one leg
    int64_t od[8]; int64_t sin_o[8];  // output-ordered extents and their input strides
    int64_t sin[8]; { int64_t s = 1; for (int i = n - 1; i >= 0; --i) { sin[i] = s; s *= d[i]; } }
    int m = 0;
    for (int i = 0; i < n;) {
        int j = i; int64_t ext = d[p[i]];
        while (j + 1 < n && p[j + 1] == p[j] + 1) { ++j; ext *= d[p[j]]; }
        od[m] = ext; sin_o[m] = sin[p[j]]; ++m; i = j + 1;
    }
    int64_t sout_o[8]; { int64_t s = 1; for (int i = m - 1; i >= 0; --i) { sout_o[i] = s; s *= od[i]; } }
    if (m == 1) { cudaError_t e = cudaMemcpyAsync(out, in, total * 8, cudaMemcpyDeviceToDevice, st); count_launch(); return e; }
    PermArgs a;
    if (sin_o[m - 1] == 1) {  // innermost preserved
        a.nd = m - 1;
        for (int i = 0; i < m - 1; ++i) { a.ext[i] = od[i]; a.sin[i] = sin_o[i]; a.sout[i] = sout_o[i]; }
        int64_t inner = od[m - 1], rows = total / inner;
        const bool al16 = (((uintptr_t)in | (uintptr_t)out) & 15) == 0;
        if (al16 && inner % 2 == 0 && inner / 2 <= 32 * 1024 && m >= 2) {
            // vectorised: runs over the last outer leg (all input strides are multiples of `inner`, hence even)
            PermArgs b; b.nd = m - 2;
            for (int i = 0; i < m - 2; ++i) { b.ext[i] = od[i]; b.sin[i] = sin_o[i]; b.sout[i] = sout_o[i]; }
            const int64_t ext_last = od[m - 2], nruns = rows / ext_last;
            int64_t chunk_rows = 1024 / (inner / 2); if (chunk_rows < 1) chunk_rows = 1;      // ~16 KB per warp visit
            // small (L2-resident) tensors: shorter visits until every SM has 16 warps to hide the latency with (a 8 MB tensor at 16 KB
            // per visit is 512 visits = 64 CTAs: 10 us, latency-bound)
            while (chunk_rows > 1 && nruns * ((ext_last + chunk_rows - 1) / chunk_rows) < 148 * 16) chunk_rows = (chunk_rows + 1) / 2;
            const int64_t chunks = (ext_last + chunk_rows - 1) / chunk_rows;
            int64_t nb = (nruns * chunks + 7) / 8; if (nb > 148 * 64) nb = 148 * 64;
            permute_runs_kernel<<<(unsigned)nb, 256, 0, st>>>(b, ext_last, sin_o[m - 2], inner, nruns, chunk_rows, chunks, in, out);
            count_launch();
            return cudaGetLastError();
        }
        int64_t blocks = (total + 255) / 256; if (blocks > 148 * 32) blocks = 148 * 32;
        permute_rows_kernel<<<(unsigned)blocks, 256, 0, st>>>(a, inner, rows, in, out);
        count_launch();
        return cudaGetLastError();
    }
    // find the output leg that is the input's innermost (stride 1)
    int ia = -1; for (int i = 0; i < m; ++i) if (sin_o[i] == 1) ia = i;
    if (ia < 0) return cudaErrorInvalidValue;
    const int ib = m - 1;
    a.nd = 0;
    for (int i = 0; i < m; ++i) if (i != ia && i != ib) { a.ext[a.nd] = od[i]; a.sin[a.nd] = sin_o[i]; a.sout[a.nd] = sout_o[i]; ++a.nd; }
    int64_t extA = od[ia], extB = od[ib];
    int64_t outer = total / (extA * extB);
    {
        bool even = (extA % 2 == 0) && (extB % 2 == 0) && (sin_o[ib] % 2 == 0) && (sout_o[ia] % 2 == 0) && ((((uintptr_t)in | (uintptr_t)out) & 15) == 0);
        for (int i = 0; i < a.nd; ++i) even = even && (a.sin[i] % 2 == 0) && (a.sout[i] % 2 == 0);
        if (even && extA >= 64 && extB >= 64) {
            int64_t tA = (extA + 63) / 64, tB = (extB + 63) / 64, nb = tA * tB * outer;
            if (nb > 0x7fffffffLL) return cudaErrorInvalidValue;
            permute_tiled64_kernel<<<(unsigned)nb, 256, 0, st>>>(a, extA, extB, sin_o[ib], sout_o[ia], tA, tB, in, out);
            count_launch();
            return cudaGetLastError();
        }
    }
    const int T = 32;
    int64_t tilesA = (extA + T - 1) / T, tilesB = (extB + T - 1) / T;
    int64_t blocks = tilesA * tilesB * outer;
    if (blocks > 0x7fffffffLL) return cudaErrorInvalidValue;
    permute_tiled_kernel<T><<<(unsigned)blocks, dim3(T, 8), 0, st>>>(a, extA, extB, sin_o[ib], sout_o[ia], tilesA, tilesB, in, out);
    count_launch();
    return cudaGetLastError();
}

}  // namespace tatrg
