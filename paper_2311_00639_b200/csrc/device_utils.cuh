// Device helpers shared by the kernels: complex types, sign flips, fixed-order reductions, mbarrier / bulk-copy PTX.
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

#include "common.h"

namespace syk {

template <typename T> struct Cx;
template <> struct Cx<double> { using type = double2; };
template <> struct Cx<float> { using type = float2; };

// multiply by (-1)^s where sbit = s << 31
__device__ __forceinline__ double flip_sign(double v, uint32_t sbit) {
    return __hiloint2double(__double2hiint(v) ^ (int)sbit, __double2loint(v));
}
__device__ __forceinline__ float flip_sign(float v, uint32_t sbit) {
    return __uint_as_float(__float_as_uint(v) ^ sbit);
}

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
    return v;   // valid in lane 0
}

// Sum over the block in a fixed order (per-thread value -> warp shuffle tree -> warp 0 tree); every thread gets
// the result.  All threads of the block must call it.  `red` is shared scratch of >= 33 doubles.
__device__ __forceinline__ double block_sum(double v, double* red) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarp = (blockDim.x + 31) >> 5;
    v = warp_sum(v);
    if (lane == 0) red[warp] = v;
    __syncthreads();
    if (warp == 0) {
        double s = lane < nwarp ? red[lane] : 0.0;
        s = warp_sum(s);
        if (lane == 0) red[32] = s;
    }
    __syncthreads();
    double r = red[32];
    __syncthreads();
    return r;
}

// Sum of n per-CTA partials, same value in every CTA that uses the same block size.
__device__ __forceinline__ double reduce_partials(const double* p, int n, double* red) {
    double s = 0.0;
    for (int i = threadIdx.x; i < n; i += blockDim.x) s += p[i];
    return block_sum(s, red);
}

// Lock-step of persistent CTAs (register-tile and scatter-tile apply_H kernels).  The L2 reuse of those kernels is
// BETWEEN CTAs: source tile (T ^ d) ^ hi of a neighbouring output tile T ^ d is the source tile T ^ (hi ^ d) of tile
// T, and loads are sorted by hi, so a line fetched from DRAM for one CTA is wanted by another CTA one or two loads
// later -- provided both CTAs are at the same place of the load list.  Free-running CTAs drift apart by more loads
// than L2 holds (ncu, N = 64: 5 % hit rate), so the producers pace each other: loads are counted in epochs of
// `epoch_len`; a producer that starts epoch e first reports epoch e-1 as issued (one atomicAdd on a ring of
// kSyncRing counters) and then waits until all gridDim.x CTAs have reported epoch e-1-lag.  Timing only: no data
// depends on it, results stay bitwise equal.  All CTAs are co-resident (grid <= number of SMs, one CTA per SM) and the
// wait is bounded, so it cannot deadlock.
__device__ __forceinline__ void lockstep_gate(uint32_t* sync, uint32_t e, uint32_t lag) {
    if (e == 0) return;
    atomicAdd(sync + ((e - 1) % kSyncRing), 1u);
    if (e < 1 + lag) return;
    const uint32_t f = e - 1 - lag;
    const uint32_t target = gridDim.x * (f / kSyncRing + 1);
    const volatile uint32_t* c = sync + (f % kSyncRing);
    // bounded wait (~2 ms): pacing is an optimisation, never a dependency -- if the counters are disturbed (two launches
    // on one handle in flight on different streams) the CTA simply runs on unpaced
    for (int spins = 0; *c < target && spins < 32768; ++spins) __nanosleep(64);
}

// ---- mbarrier and bulk async copy (TMA unit, non-tensor form: SASS UBLKCP) -------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_fence_init() {
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint32_t bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ bool mbar_try_wait(uint32_t bar, uint32_t parity) {
    uint32_t ok;
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n"
        "selp.u32 %0, 1, 0, p;\n"
        "}\n"
        : "=r"(ok)
        : "r"(bar), "r"(parity)
        : "memory");
    return ok != 0;
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
    while (!mbar_try_wait(bar, parity)) {
    }
}
// global -> shared bulk copy of `bytes` (multiple of 16; both addresses 16-byte aligned), completion counted on
// the mbarrier `bar`
__device__ __forceinline__ void bulk_load(uint32_t dst_smem, const void* src, uint32_t bytes, uint32_t bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(dst_smem), "l"(src), "r"(bytes), "r"(bar)
                 : "memory");
}

}  // namespace syk
