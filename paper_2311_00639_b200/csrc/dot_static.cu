// syk_dot_static: the complex inner product <a|b> = sum conj(a[k]) b[k] (the dot of the OTOC / Green pipelines, PAPER.md:230,
// 218, and of the Lanczos recurrence) for callers that cannot allocate: code under CUDA graph capture, tight
// serving loops, harnesses that forbid cudaMalloc.  A variant of cdot_kernel (vector_ops.cu), whose per-CTA partial sums live
// in a caller-supplied scratch buffer; here they live in ONE file-scope __device__ array of fixed size, so the call needs
// nothing but its inputs and a device slot for the result.  It calls no cudaMalloc / cudaFree / allocating library routine,
// does not synchronise and copies nothing to the host: every step is a kernel launch on `stream`.
//
// Fixed work per CTA (kSdUnitsPerCta 16-byte units, not a grid-stride loop over an SM-count-sized grid): the summation order
// depends on the vector length only, so the result is bitwise the same on every GPU.  The price is the size limit:
// kSdMaxCtas partials = 2^25 units = 2^25 complex128 / 2^26 complex64 amplitudes (N <= 50 / 52); beyond it SYK_ELIMIT.
//
// The array is shared by every call of the process on a device and keeps the last call's contents.  Nothing in it has to
// start at zero: the first kernel overwrites partials [0, n_ctas) and the second reads exactly those.  Two calls that overlap
// on the GPU (different streams, or graph branches without a dependency) race on it and give wrong results.
#include <mutex>

#include "device_utils.cuh"

namespace syk {
namespace {

constexpr int kSdThreads = 256;
constexpr int kSdUnitsPerCta = 8192;     // 16-byte units per CTA: 32 per thread
constexpr int kSdMaxCtas = 4096;         // 64 KiB of partial sums, resident on every GPU that loads the library
constexpr int kSdMaxDevices = 64;

static __device__ __align__(256) double2 g_dot_static_scratch[kSdMaxCtas];

// fixed-order sum over the block: lanes by shuffle tree, warps through shared memory, warp 0 adds them in lane order
__device__ __forceinline__ double sd_block_sum(double v, double* red) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    __syncthreads();   // red may still be read from a previous call
    if (lane == 0) red[warp] = v;
    __syncthreads();
    double s = 0.0;
    if (warp == 0) {
        s = lane < kSdThreads / 32 ? red[lane] : 0.0;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) s += __shfl_down_sync(0xffffffffu, s, o);
    }
    return s;   // valid in thread 0
}

// one unit = one complex128 amplitude (double2) or two adjacent complex64 amplitudes (float4); conj(a) * b in fp64
__device__ __forceinline__ void sd_accumulate(const double2 a, const double2 b, double& sr, double& si) {
    sr += a.x * b.x + a.y * b.y;
    si += a.x * b.y - a.y * b.x;
}
__device__ __forceinline__ void sd_accumulate(const float4 a, const float4 b, double& sr, double& si) {
    sr += (double)a.x * (double)b.x + (double)a.y * (double)b.y;
    si += (double)a.x * (double)b.y - (double)a.y * (double)b.x;
    sr += (double)a.z * (double)b.z + (double)a.w * (double)b.w;
    si += (double)a.z * (double)b.w - (double)a.w * (double)b.z;
}

template <typename V>
__global__ void __launch_bounds__(kSdThreads) dot_static_partial_kernel(const V* __restrict__ a, const V* __restrict__ b,
                                                                        uint64_t n_units, double2* scratch) {
    __shared__ double red[kSdThreads / 32];
    const uint64_t first = (uint64_t)blockIdx.x * kSdUnitsPerCta + threadIdx.x;
    double sr = 0.0, si = 0.0;
#pragma unroll 8
    for (int k = 0; k < kSdUnitsPerCta / kSdThreads; ++k) {
        const uint64_t i = first + (uint64_t)k * kSdThreads;
        if (i < n_units) sd_accumulate(a[i], b[i], sr, si);
    }
    sr = sd_block_sum(sr, red);
    si = sd_block_sum(si, red);
    if (threadIdx.x == 0) scratch[blockIdx.x] = make_double2(sr, si);
}

// result[0..1] = sum of partials [0, n) in a fixed order: thread t adds t, t + 256, ..., then the block tree
__global__ void __launch_bounds__(kSdThreads) dot_static_final_kernel(const double2* __restrict__ scratch, int n,
                                                                      double* result) {
    __shared__ double red[kSdThreads / 32];
    double sr = 0.0, si = 0.0;
    for (int i = threadIdx.x; i < n; i += kSdThreads) {
        sr += scratch[i].x;
        si += scratch[i].y;
    }
    sr = sd_block_sum(sr, red);
    si = sd_block_sum(si, red);
    if (threadIdx.x == 0) {
        result[0] = sr;
        result[1] = si;
    }
}

// Device address of the scratch array, resolved once per device with that device current.  In host code the name
// g_dot_static_scratch is only a handle of the symbol, not a device address: it must never be passed to a kernel.
std::mutex g_sd_mutex;
double2* g_sd_ptr[kSdMaxDevices] = {};

int dot_static_scratch(double2** out) {
    int dev = -1;
    SYK_CUDA(cudaGetDevice(&dev));
    if (dev < 0 || dev >= kSdMaxDevices) return SYK_EINVAL;
    std::lock_guard<std::mutex> lock(g_sd_mutex);
    if (!g_sd_ptr[dev]) {
        void* p = nullptr;
        SYK_CUDA(cudaGetSymbolAddress(&p, g_dot_static_scratch));
        if (!p) return SYK_ECUDA;
        g_sd_ptr[dev] = (double2*)p;
    }
    *out = g_sd_ptr[dev];
    return SYK_OK;
}

}  // namespace
}  // namespace syk

extern "C" {

int syk_dot_static_max_N(int dtype) {
    if (dtype != SYK_C64 && dtype != SYK_C128) return SYK_EINVAL;
    // kSdMaxCtas * kSdUnitsPerCta = 2^25 units; a complex64 unit holds two amplitudes
    return dtype == SYK_C128 ? 50 : 52;
}

int syk_dot_static_prepare(void) {
    double2* p = nullptr;
    return syk::dot_static_scratch(&p);
}

int syk_dot_static(int N, int dtype, const void* d_a, const void* d_b, double* d_result, void* stream) {
    using namespace syk;
    if (N < 4 || (N & 1) || (dtype != SYK_C64 && dtype != SYK_C128) || !d_a || !d_b || !d_result) return SYK_EINVAL;
    if (((uintptr_t)d_a & 15) || ((uintptr_t)d_b & 15) || ((uintptr_t)d_result & 7)) return SYK_EINVAL;
    if (N > syk_dot_static_max_N(dtype)) return SYK_ELIMIT;
    const uint64_t D = 1ull << (N / 2);
    const uint64_t n_units = dtype == SYK_C128 ? D : D / 2;
    const int n_ctas = (int)((n_units + kSdUnitsPerCta - 1) / kSdUnitsPerCta);
    if (n_ctas < 1 || n_ctas > kSdMaxCtas) return SYK_ELIMIT;
    double2* scratch = nullptr;
    SYK_TRY(dot_static_scratch(&scratch));
    cudaStream_t st = (cudaStream_t)stream;
    if (dtype == SYK_C128)
        dot_static_partial_kernel<double2><<<n_ctas, kSdThreads, 0, st>>>((const double2*)d_a, (const double2*)d_b, n_units, scratch);
    else
        dot_static_partial_kernel<float4><<<n_ctas, kSdThreads, 0, st>>>((const float4*)d_a, (const float4*)d_b, n_units, scratch);
    dot_static_final_kernel<<<1, kSdThreads, 0, st>>>(scratch, n_ctas, d_result);
    count_launch(2);
    SYK_CUDA(cudaGetLastError());
    return SYK_OK;
}

}  // extern "C"
