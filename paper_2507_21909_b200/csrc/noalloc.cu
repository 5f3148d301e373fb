// noalloc.cu -- tatrg_gram_static: the Gram matrix X^T X (the first half of every Cholesky QR of the path: Eq. A.2-A.6
// :345-369, Eq. 2.4 :76) for callers that cannot allocate device memory -- code under CUDA graph capture, tight serving
// loops, harnesses that forbid cudaMalloc.  Same kernels and same split along K as tatrg_gram; the split-K partial products
// go to a file-scope __device__ array instead of caller scratch.
//
// The array is 16 MiB (kStaticScratchBytes); every GPU that loads the library holds it until the process exits.  All calls on
// a device share it: two calls whose kernels overlap on the GPU (different streams, no ordering between them) RACE on it --
// keep them on one stream or order them with events.  Nothing has to start at zero: every partial product the reduction
// kernel reads was written earlier in the same call (beta = 0), so the previous call's contents are never observed.
//
// In host code `g_static_scratch` is a host-side stand-in, not a device address; the address a kernel can use comes from
// cudaGetSymbolAddress, taken once per device with that device current (static_scratch()).
#include "internal.h"
#include <cstdio>
#include <mutex>

namespace tatrg {
namespace {

constexpr size_t kStaticScratchBytes = (size_t)16 << 20;
static __device__ __align__(256) unsigned char g_static_scratch[kStaticScratchBytes];

struct PerDevice { double* ptr = nullptr; bool tried = false; cudaError_t err = cudaSuccess; };

// device address of the array on the CURRENT device (resolved once per device)
cudaError_t static_scratch(double** out) {
    static std::map<int, PerDevice> per_device;
    static std::mutex mu;
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    std::lock_guard<std::mutex> lock(mu);
    PerDevice& p = per_device[dev];
    if (!p.tried) {
        p.tried = true;
        void* addr = nullptr;
        p.err = cudaGetSymbolAddress(&addr, g_static_scratch);
        p.ptr = p.err == cudaSuccess ? (double*)addr : nullptr;
    }
    *out = p.ptr;
    return p.err;
}

void say(char* err, size_t cap, const char* fmt, long long a = 0, long long b = 0, long long c = 0, long long d = 0) {
    if (err && cap) snprintf(err, cap, fmt, a, b, c, d);
}

}  // namespace
}  // namespace tatrg

using namespace tatrg;

extern "C" {

size_t tatrg_gram_static_max_scratch_bytes(void) { return kStaticScratchBytes; }

int tatrg_gram_static(void* stp, long long m, int n, const double* X, double* G, char* err, size_t err_cap) {
    if (err && err_cap) err[0] = 0;
    if (m < 1 || n < 1 || !X || !G) { say(err, err_cap, "tatrg_gram_static: bad argument (m = %lld, n = %lld, null pointer?)", m, n); return TATRG_EINVAL; }
    const bool lower = n >= 256;
    const size_t need = 8 * (size_t)dgemm_splitk_doubles(n, n, m, lower);
    if (need > kStaticScratchBytes) {
        say(err, err_cap, "tatrg_gram_static: m = %lld, n = %lld needs %lld bytes of split-K scratch, the static array holds %lld; use tatrg_gram with caller scratch",
            m, n, (long long)need, (long long)kStaticScratchBytes);
        return TATRG_EINVAL;
    }
    double* scratch = nullptr;
    cudaError_t e = static_scratch(&scratch);
    if (e != cudaSuccess || !scratch) { say(err, err_cap, "tatrg_gram_static: cudaGetSymbolAddress failed (CUDA error %lld)", (long long)e); return TATRG_ECUDA; }
    cudaStream_t st = (cudaStream_t)stp;
    e = dgemm_splitk(st, true, false, n, n, m, 1.0, X, n, X, n, G, n, need ? scratch : nullptr, lower);
    if (e == cudaSuccess && lower) e = mirror_lower(st, n, G);
    if (e != cudaSuccess) { say(err, err_cap, "tatrg_gram_static: launch failed (CUDA error %lld)", (long long)e); return TATRG_ECUDA; }
    return TATRG_OK;
}

}  // extern "C"
