// philox.cu -- Philox4x32-10 (Salmon et al., SC'11) and the Gaussian streams of the RSVD test tensor Omega
// (App. A :352,:371 "Omega is a random tensor") and of the gauge reference vectors (R10, R11).
//   key = (seed_lo, seed_hi), counter = (e_lo, e_hi, call, stream), one Gaussian per counter:
//   u1 = ((x0>>6)*2^27 + (x1>>5) + 0.5)*2^-53, u2 likewise from (x2,x3), z = sqrt(-2 ln u1) cos(2 pi u2).
// Written from the published round function; shares no code with oracle/philox.py.
#include "internal.h"

namespace tatrg {
namespace {
struct U4 { uint32_t x, y, z, w; };

__device__ __forceinline__ U4 philox4x32_10(U4 c, uint32_t k0, uint32_t k1) {
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        uint32_t hi0 = __umulhi(0xD2511F53u, c.x), lo0 = 0xD2511F53u * c.x;
        uint32_t hi1 = __umulhi(0xCD9E8D57u, c.z), lo1 = 0xCD9E8D57u * c.z;
        U4 n;
        n.x = hi1 ^ c.y ^ k0; n.y = lo1; n.z = hi0 ^ c.w ^ k1; n.w = lo0;
        c = n;
        k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
    }
    return c;
}
__device__ __forceinline__ double u53(uint32_t a, uint32_t b) {
    return ((double)(a >> 6) * 134217728.0 + (double)(b >> 5) + 0.5) * (1.0 / 9007199254740992.0);
}
__device__ __forceinline__ double gauss_of(uint64_t e, uint32_t call, uint32_t stream, uint32_t k0, uint32_t k1) {
    U4 c; c.x = (uint32_t)e; c.y = (uint32_t)(e >> 32); c.z = call; c.w = stream;
    U4 x = philox4x32_10(c, k0, k1);
    double u1 = u53(x.x, x.y), u2 = u53(x.z, x.w);
    return sqrt(-2.0 * log(u1)) * cospi(2.0 * u2);
}
__global__ void raw_kernel(uint32_t k0, uint32_t k1, uint32_t call, uint32_t stream, uint64_t start, int64_t count, uint32_t* raw) {
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < count; i += (int64_t)gridDim.x * blockDim.x) {
        uint64_t e = start + (uint64_t)i;
        U4 c; c.x = (uint32_t)e; c.y = (uint32_t)(e >> 32); c.z = call; c.w = stream;
        U4 x = philox4x32_10(c, k0, k1);
        raw[4 * i] = x.x; raw[4 * i + 1] = x.y; raw[4 * i + 2] = x.z; raw[4 * i + 3] = x.w;
    }
}
__global__ void gauss_kernel(uint32_t k0, uint32_t k1, uint32_t call, uint32_t stream, uint64_t start, int64_t count, double* z) {
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < count; i += (int64_t)gridDim.x * blockDim.x)
        z[i] = gauss_of(start + (uint64_t)i, call, stream, k0, k1);
}
// the same Gaussians, element e = (a, b, c) of a tensor [na][nb][nc] written at [b][a][c]: Omega^phys is drawn in the order (be, j', m)
// (R11/R12) and consumed as [j'][be][m]; writing it there saves a 16-byte-per-element permute of the largest tensor of the bond swap
__global__ void gauss_swap01_kernel(uint32_t k0, uint32_t k1, uint32_t call, uint32_t stream, int64_t na, int64_t nb, int64_t nc, double* z) {
    // one block per b (grid-stride): the (a, c) plane of the output is contiguous, (a, c) advance without a division
    const int64_t per = na * nc;
    const int64_t da = blockDim.x / nc, dc = blockDim.x % nc;
    for (int64_t b = blockIdx.x; b < nb; b += gridDim.x) {
        int64_t a = threadIdx.x / nc, c = threadIdx.x % nc;
        double* out = z + b * per;
        for (int64_t t = threadIdx.x; t < per; t += blockDim.x) {
            out[t] = gauss_of((uint64_t)((a * nb + b) * nc + c), call, stream, k0, k1);
            a += da; c += dc;
            if (c >= nc) { c -= nc; a += 1; }
        }
    }
}
// rho[r, j] = Gaussian(counter e = r*kRhoCols + j), j < ncols, stored densely as rows x ncols
__global__ void rho_kernel(uint32_t k0, uint32_t k1, uint32_t call, uint32_t stream, int64_t rows, int ncols, double* out) {
    int64_t total = rows * ncols;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < total; i += (int64_t)gridDim.x * blockDim.x) {
        int64_t r = i / ncols; int j = (int)(i - r * ncols);
        out[i] = gauss_of((uint64_t)r * kRhoCols + j, call, stream, k0, k1);
    }
}
inline unsigned nb(int64_t n) { int64_t b = (n + 255) / 256; if (b > 148 * 16) b = 148 * 16; if (b < 1) b = 1; return (unsigned)b; }
}  // namespace

cudaError_t philox_raw(cudaStream_t st, uint64_t seed, uint32_t call, uint32_t stream, uint64_t start, int64_t count, uint32_t* raw) {
    if (count <= 0) return cudaSuccess;
    raw_kernel<<<nb(count), 256, 0, st>>>((uint32_t)seed, (uint32_t)(seed >> 32), call, stream, start, count, raw); count_launch();
    return cudaGetLastError();
}
cudaError_t philox_gauss(cudaStream_t st, uint64_t seed, uint32_t call, uint32_t stream, uint64_t start, int64_t count, double* z) {
    if (count <= 0) return cudaSuccess;
    gauss_kernel<<<nb(count), 256, 0, st>>>((uint32_t)seed, (uint32_t)(seed >> 32), call, stream, start, count, z); count_launch();
    return cudaGetLastError();
}
cudaError_t philox_gauss_swap01(cudaStream_t st, uint64_t seed, uint32_t call, uint32_t stream, int64_t na, int64_t nb_, int64_t nc, double* z) {
    if (na * nb_ * nc <= 0) return cudaSuccess;
    const int64_t blocks = nb_ < (1 << 20) ? nb_ : (1 << 20);
    gauss_swap01_kernel<<<(unsigned)blocks, 256, 0, st>>>((uint32_t)seed, (uint32_t)(seed >> 32), call, stream, na, nb_, nc, z); count_launch();
    return cudaGetLastError();
}
cudaError_t philox_rho(cudaStream_t st, uint64_t seed, uint32_t call, uint32_t stream, int64_t rows, int ncols, double* out) {
    if (rows <= 0 || ncols <= 0) return cudaSuccess;
    rho_kernel<<<nb(rows * ncols), 256, 0, st>>>((uint32_t)seed, (uint32_t)(seed >> 32), call, stream, rows, ncols, out); count_launch();
    return cudaGetLastError();
}

}  // namespace tatrg
