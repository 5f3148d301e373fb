// elementwise.cu -- the small HBM-bound kernels of the path: initial tensor (Eq. 3.1-3.2 :241-246),
// diagonal scalings by singular values (Eq. 2.11 :150 "sigma goes into F"), column/row gathers after a
// truncation, and the tensor trace tTr (Eq. 2.1 :48) as a two-level warp-shuffle reduction.
#include "internal.h"

namespace tatrg {
namespace {
__device__ __forceinline__ double fmode(double v, int mode) {
    switch (mode) {
        case 0: return v;
        case 1: return 1.0 / v;
        case 2: return 1.0 / sqrt(v);
        case 3: return sqrt(v);
        case 4: return 1.0 / (v * sqrt(v));
        default: return v;
    }
}
__global__ void scale_last_kernel(double* out, const double* in, const double* vec, int64_t total, int64_t cols, int mode) {
    for (int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; e < total; e += (int64_t)gridDim.x * blockDim.x)
        out[e] = in[e] * fmode(vec[e % cols], mode);
}
// out = a x + b y + c z (z may be null; out may alias any input): the three-term recurrence of the Chebyshev-filtered subspace iteration
__global__ void lincomb3_kernel(double* out, double a, const double* x, double b, const double* y, double c, const double* z, int64_t total) {
    for (int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; e < total; e += (int64_t)gridDim.x * blockDim.x) {
        double v = a * x[e] + b * y[e];
        if (z) v += c * z[e];
        out[e] = v;
    }
}
__global__ void scale_rows_kernel(double* out, const double* in, const double* vec, int64_t total, int64_t cols, int mode) {
    for (int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; e < total; e += (int64_t)gridDim.x * blockDim.x)
        out[e] = in[e] * fmode(vec[e / cols], mode);
}
__global__ void gather_rows_kernel(double* out, const double* in, const int* idx, const double* scale, int64_t nrows, int64_t cols,
                                   int64_t ld) {
    int64_t total = nrows * cols;
    for (int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; e < total; e += (int64_t)gridDim.x * blockDim.x) {
        int64_t r = e / cols, c = e - r * cols;
        out[e] = in[(int64_t)idx[r] * ld + c] * (scale ? scale[r] : 1.0);
    }
}
__global__ void gather_vec_kernel(double* out, const double* in, const int* idx, int64_t n, int64_t stride, double mul) {
    for (int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; e < n; e += (int64_t)gridDim.x * blockDim.x)
        out[e] = in[(int64_t)idx[e] * stride] * mul;
}
// One warp per multiplet: modified Gram-Schmidt of the g x g block C[a:b, 0:g] (columns), diag(R) > 0, written as the
// diagonal block of G.  g == 1 reduces to the sign of C[a,0].  Lane i holds row i of the block (g <= 32).
__global__ void gauge_blocks_kernel(const double* __restrict__ cfull, int ldc, const int* __restrict__ groups, int ngroups, int k,
                                    double* __restrict__ G) {
    int grp = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    if (grp >= ngroups) return;
    const int lane = threadIdx.x & 31;
    const int a = groups[2 * grp], b = groups[2 * grp + 1], g = b - a;
    double q[32];   // row `lane` of Q, columns 0..g-1 (fully unrolled access would be needed for registers; g is tiny)
    for (int j = 0; j < g; ++j) {
        double col = (lane < g) ? cfull[(int64_t)(a + lane) * ldc + j] : 0.0;
        for (int i = 0; i < j; ++i) {
            double d = q[i] * col;
            for (int o = 16; o > 0; o >>= 1) d += __shfl_xor_sync(0xffffffffu, d, o);
            col -= d * q[i];
        }
        double n2 = col * col;
        for (int o = 16; o > 0; o >>= 1) n2 += __shfl_xor_sync(0xffffffffu, n2, o);
        q[j] = col / sqrt(n2);
    }
    if (lane < g)
        for (int j = 0; j < g; ++j) G[(int64_t)(a + lane) * k + a + j] = q[j];
}
__global__ void zero_kernel(double* p, int64_t n) {
    for (int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; e < n; e += (int64_t)gridDim.x * blockDim.x) p[e] = 0.0;
}

// tTr: sum_i x_i y_i.  Pass 1: grid-stride partial sums, warp shuffle + shared; pass 2: one block reduces the partials.
__global__ void dot_partial_kernel(const double* __restrict__ x, const double* __restrict__ y, int64_t n, double* partial) {
    double s = 0;
    for (int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; e < n; e += (int64_t)gridDim.x * blockDim.x) s += x[e] * y[e];
    __shared__ double sh[32];
    for (int o = 16; o > 0; o >>= 1) s += __shfl_down_sync(0xffffffffu, s, o);
    if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5] = s;
    __syncthreads();
    if (threadIdx.x < 32) {
        s = (threadIdx.x < (blockDim.x >> 5)) ? sh[threadIdx.x] : 0.0;
        for (int o = 16; o > 0; o >>= 1) s += __shfl_down_sync(0xffffffffu, s, o);
        if (threadIdx.x == 0) partial[blockIdx.x] = s;
    }
}
__global__ void dot_final_kernel(const double* partial, int np, double* result) {
    double s = 0;
    for (int i = threadIdx.x; i < np; i += blockDim.x) s += partial[i];
    __shared__ double sh[32];
    for (int o = 16; o > 0; o >>= 1) s += __shfl_down_sync(0xffffffffu, s, o);
    if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5] = s;
    __syncthreads();
    if (threadIdx.x < 32) {
        s = (threadIdx.x < (blockDim.x >> 5)) ? sh[threadIdx.x] : 0.0;
        for (int o = 16; o > 0; o >>= 1) s += __shfl_down_sync(0xffffffffu, s, o);
        if (threadIdx.x == 0) result[0] = s;
    }
}

// Eq. 3.1-3.2: Phi0[i1,i2,i3,i4,a] = e^{beta h s_a} prod_mu W[a,i_mu], Psi0 = prod_mu W[a,j_mu]
__global__ void init_ising_kernel(double beta, double h, double* phi, double* psi) {
    int e = threadIdx.x;  // 32 elements: (i1,i2,i3,i4,a)
    if (e >= 32) return;
    int a = e & 1, bits = e >> 1;
    double c = sqrt(cosh(beta)), s = sqrt(sinh(beta));
    double sgn = a ? -1.0 : 1.0;
    double v = 1.0;
    for (int mu = 0; mu < 4; ++mu) v *= ((bits >> mu) & 1) ? sgn * s : c;
    psi[e] = v;
    phi[e] = v * exp(beta * h * sgn);
}
// out[0] = Tr A, out[1] = Tr A^2 of a small n x n matrix (one block): the two reductions of the X ratio, Eq. 3.3 :301
__global__ void traces_kernel(const double* __restrict__ A, int n, double* out) {
    double t1 = 0, t2 = 0;
    for (int e = threadIdx.x; e < n * n; e += blockDim.x) { int i = e / n, j = e - i * n; if (i == j) t1 += A[e]; t2 += A[e] * A[j * n + i]; }
    __shared__ double sh[2][32];
    for (int o = 16; o > 0; o >>= 1) { t1 += __shfl_down_sync(0xffffffffu, t1, o); t2 += __shfl_down_sync(0xffffffffu, t2, o); }
    if ((threadIdx.x & 31) == 0) { sh[0][threadIdx.x >> 5] = t1; sh[1][threadIdx.x >> 5] = t2; }
    __syncthreads();
    if (threadIdx.x < 32) {
        t1 = (threadIdx.x < (blockDim.x >> 5)) ? sh[0][threadIdx.x] : 0.0; t2 = (threadIdx.x < (blockDim.x >> 5)) ? sh[1][threadIdx.x] : 0.0;
        for (int o = 16; o > 0; o >>= 1) { t1 += __shfl_down_sync(0xffffffffu, t1, o); t2 += __shfl_down_sync(0xffffffffu, t2, o); }
        if (threadIdx.x == 0) { out[0] = t1; out[1] = t2; }
    }
}
inline unsigned nblocks(int64_t total) { int64_t b = (total + 255) / 256; if (b > 148 * 16) b = 148 * 16; if (b < 1) b = 1; return (unsigned)b; }
}  // namespace

cudaError_t scale_last(cudaStream_t st, double* out, const double* in, const double* vec, int64_t rows, int64_t cols, int mode) {
    if (rows * cols == 0) return cudaSuccess;
    scale_last_kernel<<<nblocks(rows * cols), 256, 0, st>>>(out, in, vec, rows * cols, cols, mode); count_launch();
    return cudaGetLastError();
}
cudaError_t lincomb3(cudaStream_t st, double* out, double a, const double* x, double b, const double* y, double c, const double* z, int64_t n) {
    if (n == 0) return cudaSuccess;
    lincomb3_kernel<<<nblocks(n), 256, 0, st>>>(out, a, x, b, y, c, z, n); count_launch();
    return cudaGetLastError();
}
cudaError_t scale_rows(cudaStream_t st, double* out, const double* in, const double* vec, int64_t rows, int64_t cols, int mode) {
    if (rows * cols == 0) return cudaSuccess;
    scale_rows_kernel<<<nblocks(rows * cols), 256, 0, st>>>(out, in, vec, rows * cols, cols, mode); count_launch();
    return cudaGetLastError();
}
cudaError_t gather_rows_scaled(cudaStream_t st, double* out, const double* in, const int* idx, const double* scale, int64_t nrows,
                               int64_t cols, int64_t ld_in) {
    if (nrows * cols == 0) return cudaSuccess;
    gather_rows_kernel<<<nblocks(nrows * cols), 256, 0, st>>>(out, in, idx, scale, nrows, cols, ld_in); count_launch();
    return cudaGetLastError();
}
cudaError_t gather_vec(cudaStream_t st, double* out, const double* in, const int* idx, int64_t n, int64_t stride_in, double mul) {
    if (n == 0) return cudaSuccess;
    gather_vec_kernel<<<nblocks(n), 256, 0, st>>>(out, in, idx, n, stride_in, mul); count_launch();
    return cudaGetLastError();
}
cudaError_t gauge_blocks(cudaStream_t st, const double* cfull, int ldc, const int* groups, int ngroups, int k, double* G) {
    if (k <= 0 || ngroups <= 0) return cudaSuccess;
    cudaError_t e = fill_zero(st, G, (int64_t)k * k);
    if (e != cudaSuccess) return e;
    gauge_blocks_kernel<<<(ngroups + 3) / 4, 128, 0, st>>>(cfull, ldc, groups, ngroups, k, G); count_launch();
    return cudaGetLastError();
}
cudaError_t fill_zero(cudaStream_t st, double* p, int64_t n) {
    if (n == 0) return cudaSuccess;
    zero_kernel<<<nblocks(n), 256, 0, st>>>(p, n); count_launch();
    return cudaGetLastError();
}
cudaError_t dot(cudaStream_t st, int64_t n, const double* x, const double* y, double* result) {
    // result[1..] is used as scratch for the partials: callers give result room for 1 + 148*8 doubles
    int np = (int)nblocks(n); if (np > 148 * 8) np = 148 * 8;
    dot_partial_kernel<<<np, 256, 0, st>>>(x, y, n, result + 1);
    dot_final_kernel<<<1, 256, 0, st>>>(result + 1, np, result); count_launch(2);
    return cudaGetLastError();
}
cudaError_t traces(cudaStream_t st, const double* A, int n, double* out) {
    traces_kernel<<<1, 256, 0, st>>>(A, n, out); count_launch();
    return cudaGetLastError();
}
cudaError_t init_ising(cudaStream_t st, double beta, double h, double* phi, double* psi) {
    init_ising_kernel<<<1, 32, 0, st>>>(beta, h, phi, psi); count_launch();
    return cudaGetLastError();
}

}  // namespace tatrg
