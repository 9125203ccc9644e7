// ts_noalloc.cu -- ts_norm_static: the squared norm sum |psi|^2 for callers that
// cannot call cudaMalloc (code under CUDA graph capture, tight serving loops, harnesses that forbid
// it).  A variant of the two-kernel reduction of ts_norm (ts_generic.cu: norm_partial_kernel +
// norm_final_kernel) whose partial sums live in a file-scope __device__ array instead of a
// plan-owned allocation.  This file calls no cudaMalloc / cudaFree / allocating library routine,
// creates no stream or event, and never synchronises.
//
// The scratch: kStaticPartials doubles = 256 KB, held by every GPU that loads libts until the
// process exits.  One partial sum per chunk of kChunkSites consecutive sites, so the maximum is
// kStaticPartials * kChunkSites = 2^29 sites (C4's 16384^2 is 2^28); larger inputs are rejected.
// All calls on a device share the array and it keeps the last call's contents.  Nothing in it
// has to start at zero: the final kernel reads exactly the partials [0, n_chunks) that the first
// kernel of the SAME call has just written (same stream, in order), never an older one.  Two
// calls that overlap on the GPU (different streams, no dependency between them) race on it.
//
// In host code the array's name is a host-side stand-in, not a device address; the address a
// kernel can use comes from cudaGetSymbolAddress, looked up once per device with that device
// current (static_scratch below).  The kernels take it as a parameter.
#include <atomic>
#include <string>

#include "ts_internal.h"

namespace ts {
namespace {

constexpr int kStaticPartials = 32768;        // doubles of scratch: 256 KB
constexpr int kChunkSites = 16384;            // sites per partial sum
constexpr int64_t kStaticMaxSites = (int64_t)kStaticPartials * kChunkSites;   // 2^29
constexpr int kThreads = 256;
constexpr int kMaxBlocks = 148 * 8;
constexpr int kDevices = 64;                  // devices whose scratch address is remembered

static __device__ __align__(256) double g_norm_scratch[kStaticPartials];

// partial[c] = sum over chunk c of re^2 + im^2, in double, in a fixed order (the result does not
// depend on the grid size)
template <typename T>
__global__ void __launch_bounds__(kThreads)
static_partial_kernel(const T* __restrict__ re, const T* __restrict__ im, int64_t n, int n_chunks,
                      double* __restrict__ partial) {
    __shared__ double sh[kThreads / 32];
    for (int c = blockIdx.x; c < n_chunks; c += gridDim.x) {
        const int64_t base = (int64_t)c * kChunkSites;
        const int64_t rem = n - base;
        const int len = rem < kChunkSites ? (int)rem : kChunkSites;
        double acc = 0.0;
#pragma unroll 4
        for (int t = threadIdx.x; t < len; t += kThreads) {
            const double r = (double)re[base + t], m = (double)im[base + t];
            acc = fma(r, r, fma(m, m, acc));
        }
        for (int o = 16; o > 0; o >>= 1) acc += __shfl_down_sync(0xffffffffu, acc, o);
        if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5] = acc;
        __syncthreads();
        if (threadIdx.x < 32) {
            double v = threadIdx.x < kThreads / 32 ? sh[threadIdx.x] : 0.0;
            for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
            if (threadIdx.x == 0) partial[c] = v;
        }
        __syncthreads();     // sh is reused by the next chunk
    }
}

__global__ void __launch_bounds__(1024)
static_final_kernel(const double* __restrict__ partial, int n_chunks, double* __restrict__ out) {
    __shared__ double sh[32];
    double acc = 0.0;
    for (int t = threadIdx.x; t < n_chunks; t += blockDim.x) acc += partial[t];
    for (int o = 16; o > 0; o >>= 1) acc += __shfl_down_sync(0xffffffffu, acc, o);
    if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5] = acc;
    __syncthreads();
    if (threadIdx.x < 32) {
        double v = sh[threadIdx.x];
        for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
        if (threadIdx.x == 0) *out = v;
    }
}

// device address of g_norm_scratch on the CURRENT device (each device has its own copy of the
// array); looked up once per device and remembered
int static_scratch(double** out) {
    static std::atomic<double*> known[kDevices];
    int dev = -1;
    TS_CUDA_TRY(cudaGetDevice(&dev));
    if (dev >= 0 && dev < kDevices) {
        double* p = known[dev].load(std::memory_order_acquire);
        if (p) { *out = p; return TS_OK; }
    }
    double* p = nullptr;
    TS_CUDA_TRY(cudaGetSymbolAddress((void**)&p, g_norm_scratch));
    if (!p) { set_error("cudaGetSymbolAddress returned a null scratch address"); return TS_ECUDA; }
    if (dev >= 0 && dev < kDevices) known[dev].store(p, std::memory_order_release);
    *out = p;
    return TS_OK;
}

bool on_device(const void* p) {
    cudaPointerAttributes a;
    if (cudaPointerGetAttributes(&a, p) != cudaSuccess) {
        (void)cudaGetLastError();
        return false;
    }
    return a.type != cudaMemoryTypeUnregistered;
}

int reject(int code, const std::string& msg) {
    set_error(msg);
    return code;
}

}  // namespace
}  // namespace ts

extern "C" int ts_norm_static(int dtype, const void* psi_re, const void* psi_im, int64_t n_sites,
                              double* out_norm2_device, void* cuda_stream) {
    using namespace ts;
    if (dtype != TS_F32 && dtype != TS_F64) return reject(TS_EINVAL, "unknown dtype");
    if (!psi_re || !psi_im || !out_norm2_device) return reject(TS_EINVAL, "NULL argument");
    if (n_sites < 0) return reject(TS_EINVAL, "n_sites must be >= 0");
    if (n_sites > kStaticMaxSites)
        return reject(TS_EUNSUPPORTED,
                      "ts_norm_static: n_sites " + std::to_string(n_sites) +
                          " exceeds the static scratch maximum of " +
                          std::to_string(kStaticMaxSites) + " sites (use ts_norm)");
    if (!on_device(psi_re) || !on_device(psi_im) || !on_device(out_norm2_device))
        return reject(TS_EINVAL, "psi planes and out_norm2_device must be device memory");
    double* scratch = nullptr;
    int rc = static_scratch(&scratch);
    if (rc != TS_OK) return rc;
    cudaStream_t st = reinterpret_cast<cudaStream_t>(cuda_stream);
    const int n_chunks = (int)((n_sites + kChunkSites - 1) / kChunkSites);
    if (n_chunks > 0) {
        const int blocks = n_chunks < kMaxBlocks ? n_chunks : kMaxBlocks;
        if (dtype == TS_F32)
            static_partial_kernel<float><<<blocks, kThreads, 0, st>>>(
                (const float*)psi_re, (const float*)psi_im, n_sites, n_chunks, scratch);
        else
            static_partial_kernel<double><<<blocks, kThreads, 0, st>>>(
                (const double*)psi_re, (const double*)psi_im, n_sites, n_chunks, scratch);
        TS_CUDA_TRY(cudaGetLastError());
    }
    static_final_kernel<<<1, 1024, 0, st>>>(scratch, n_chunks, out_norm2_device);
    TS_CUDA_TRY(cudaGetLastError());
    return TS_OK;
}
