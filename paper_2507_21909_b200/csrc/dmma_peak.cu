// dmma_peak.cu -- calibration: register-resident DMMA (mma.sync.m8n8k4.f64) issue rate of the whole GPU.
// The FP64 tensor peak is absent from MEASURED_PEAKS.json; bench.py reports this figure next to the derived roofline
// denominator.  No memory traffic: 8 independent accumulator chains per warp, 8 warps per CTA.
#include "internal.h"

namespace tatrg {
namespace {
__global__ void __launch_bounds__(256) dmma_rate_kernel(int iters, double* sink) {
    double acc[8][2];
#pragma unroll
    for (int i = 0; i < 8; ++i) { acc[i][0] = threadIdx.x * 1e-9; acc[i][1] = i; }
    double a = 1.0 + threadIdx.x * 1e-12, b = 1.0 - threadIdx.x * 1e-12;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int i = 0; i < 8; ++i)
            asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
                         : "+d"(acc[i][0]), "+d"(acc[i][1]) : "d"(a), "d"(b));
    }
    double s = 0;
#pragma unroll
    for (int i = 0; i < 8; ++i) s += acc[i][0] + acc[i][1];
    if (s == 123.456) sink[0] = s;   // never true: keeps the chain alive
}
// The register tile of the DGEMM inner loop (8 x 4 atoms = 64 accumulators per thread, 8 + 4 distinct operand registers
// per 4-deep slice) without any memory traffic: what the warp tile can reach when operands are free.
template <int ORDER>
__global__ void __launch_bounds__(256, 1) dmma_tile_kernel(int iters, double* sink) {
    double acc[8][4][2], a[8], b[4];
#pragma unroll
    for (int i = 0; i < 8; ++i) { a[i] = 1.0 + (threadIdx.x + i) * 1e-12;
#pragma unroll
        for (int j = 0; j < 4; ++j) { acc[i][j][0] = threadIdx.x * 1e-9; acc[i][j][1] = i + j; } }
#pragma unroll
    for (int j = 0; j < 4; ++j) b[j] = 1.0 - (threadIdx.x + j) * 1e-12;
    for (int it = 0; it < iters; ++it) {
        if (ORDER == 0) {
#pragma unroll
            for (int i = 0; i < 8; ++i)
#pragma unroll
                for (int j = 0; j < 4; ++j)
                    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
                                 : "+d"(acc[i][j][0]), "+d"(acc[i][j][1]) : "d"(a[i]), "d"(b[j]));
        } else {
#pragma unroll
            for (int j = 0; j < 4; ++j)
#pragma unroll
                for (int i = 0; i < 8; ++i)
                    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
                                 : "+d"(acc[i][j][0]), "+d"(acc[i][j][1]) : "d"(a[i]), "d"(b[j]));
        }
#pragma unroll
        for (int i = 0; i < 8; ++i) a[i] += 1e-13;       // operands change every slice, as in the GEMM
#pragma unroll
        for (int j = 0; j < 4; ++j) b[j] -= 1e-13;
    }
    double s = 0;
#pragma unroll
    for (int i = 0; i < 8; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) s += acc[i][j][0] + acc[i][j][1];
    if (s == 123.456) sink[0] = s;
}
}  // namespace
}  // namespace tatrg

extern "C" int tatrg_dmma_tile_rate(void* cuda_stream, int iters, int order, double* tflops_out, double* scratch_dev) {
    using namespace tatrg;
    if (iters < 1 || !tflops_out || !scratch_dev) return TATRG_EINVAL;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) return TATRG_ECUDA;
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    auto run = [&](int n) { if (order == 0) dmma_tile_kernel<0><<<sms, 256, 0, st>>>(n, scratch_dev); else dmma_tile_kernel<1><<<sms, 256, 0, st>>>(n, scratch_dev); };
    run(iters / 10 + 1);
    cudaEventRecord(e0, st);
    run(iters);
    cudaEventRecord(e1, st);
    cudaError_t e = cudaEventSynchronize(e1);
    float ms = 0;
    if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, e0, e1);
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    if (e != cudaSuccess || ms <= 0) return TATRG_ECUDA;
    *tflops_out = 2.0 * 8 * 8 * 4 * 32.0 * iters * 8.0 * sms / (ms * 1e-3) / 1e12;
    return TATRG_OK;
}

extern "C" int tatrg_dmma_issue_rate(void* cuda_stream, int iters, int ctas_per_sm, double* tflops_out, double* scratch_dev) {
    using namespace tatrg;
    if (iters < 1 || ctas_per_sm < 1 || ctas_per_sm > 8 || !tflops_out || !scratch_dev) return TATRG_EINVAL;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) return TATRG_ECUDA;
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    const int grid = sms * ctas_per_sm;
    dmma_rate_kernel<<<grid, 256, 0, st>>>(iters / 10 + 1, scratch_dev);       // warm-up
    cudaEventRecord(e0, st);
    dmma_rate_kernel<<<grid, 256, 0, st>>>(iters, scratch_dev);
    cudaEventRecord(e1, st);
    cudaError_t e = cudaEventSynchronize(e1);
    float ms = 0;
    if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, e0, e1);
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    if (e != cudaSuccess || ms <= 0) return TATRG_ECUDA;
    const double flops = 2.0 * 8 * 8 * 4 * 8.0 * iters * 8.0 * grid;   // per mma 2*8*8*4, 8 chains, 8 warps
    *tflops_out = flops / (ms * 1e-3) / 1e12;
    return TATRG_OK;
}
