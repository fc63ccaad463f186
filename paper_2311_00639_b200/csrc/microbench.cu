// On-chip peak measurements for the roofline of the apply_H kernels ("hard parts"; DESIGN.md
// section 6).  MEASURED_PEAKS.json has the HBM copy bandwidth only; what bounds the tile kernels of a-2 is on-chip:
//   * how fast 148 persistent CTAs can pull an L2-resident vector into shared memory with cp.async.bulk (the ring of
//     3 x 64 KiB chunks of apply_h_scatter.cu, no arithmetic)                         -> L2 -> SM bytes per clock,
//   * how fast 8 consumer warps can read a staged chunk with XOR-permuted LDS.128 + 2 FMA per element (the inner
//     loop of accumulate_chunk, no loads)                                             -> shared-memory bytes per clock,
//   * both at once with `terms_per_chunk` passes over every staged chunk             -> how the two overlap,
// and for the dense-table kernel (ALU bound): the issue rate of its per-term sequence (broadcast LDS of the entry, AND,
// POPC, shift, XOR into the sign bit, FP64 add into a bin register) and of plain FP64 adds.
// Nothing here touches the method's data; the kernels only exist to give `bench.py` measured denominators.
#include <algorithm>
#include <vector>

#include "device_utils.cuh"

namespace syk {
namespace {

constexpr int kMbConsumerWarps = 8;
constexpr int kMbConsumerThreads = kMbConsumerWarps * 32;
constexpr int kMbThreads = kMbConsumerThreads + 128;
constexpr uint32_t kMbSlice = kMbConsumerThreads * 16;      // 4 KiB: one 16-byte element per consumer thread
constexpr int kMbRC = 16;                                   // slices per chunk (64 KiB)
constexpr uint32_t kMbChunk = kMbRC * kMbSlice;
constexpr uint32_t kMbRun = 8 * kMbSlice;                   // 32 KiB per bulk copy
constexpr int kMbRing = 3;

struct MbParams {
    const unsigned char* buf;     // source region (device), size = 1 << buf_log2 bytes
    int buf_log2;
    int n_chunks;                 // chunks streamed per CTA
    int terms_per_chunk;          // LDS passes over every staged chunk
    int load;                     // 0: the producer only signals, nothing is copied
    int small_log2;               // > 0: odd CTAs walk only the first 2^small_log2 bytes (an L2-resident region) and stream
                                  // `small_mult` times as many chunks, even CTAs walk the whole buffer (kind 5)
    int small_mult;
    double2* sink;                // [grid * 256]
    unsigned long long* cycles;   // [grid]
};

__global__ void __launch_bounds__(kMbThreads, 1) mb_stream_kernel(const MbParams p) {
    extern __shared__ __align__(128) unsigned char smem[];
    uint64_t* bars = reinterpret_cast<uint64_t*>(smem + (size_t)kMbRing * kMbChunk);
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const uint32_t bar_full = smem_u32(bars), bar_empty = smem_u32(bars + kMbRing);
    if (tid == 0) {
        for (int s = 0; s < kMbRing; ++s) {
            mbar_init(bar_full + 8 * s, 1);
            mbar_init(bar_empty + 8 * s, kMbConsumerWarps);
        }
        mbar_fence_init();
    }
    for (uint32_t i = (uint32_t)tid; i < kMbRing * kMbChunk / 16u; i += kMbThreads)
        reinterpret_cast<uint4*>(smem)[i] = make_uint4(0u, 0u, 0u, 0u);   // defined values when nothing is copied
    __syncthreads();
    const bool small_grp = p.small_log2 > 0 && (blockIdx.x & 1);
    const uint64_t mask = ((uint64_t)1 << (small_grp ? p.small_log2 : p.buf_log2)) - 1;
    const int n_chunks = small_grp ? p.n_chunks * p.small_mult : p.n_chunks;
    if (warp >= kMbConsumerWarps) {
        if (warp != kMbConsumerWarps || lane != 0) return;
        int pos = 0;
        uint32_t phase = 0;
        const uint32_t stage0 = smem_u32(smem);
        // every CTA walks its own sequence of 64 KiB chunks through the buffer (odd multiplier: all chunks are visited)
        uint64_t at = ((uint64_t)blockIdx.x * 0x9E3779B1ull) * kMbChunk;
        for (int c = 0; c < n_chunks; ++c) {
            mbar_wait(bar_empty + 8 * pos, phase ^ 1u);
            if (p.load) {
                mbar_arrive_expect_tx(bar_full + 8 * pos, kMbChunk);
                const unsigned char* src = p.buf + (at & mask);
                bulk_load(stage0 + (uint32_t)pos * kMbChunk, src, kMbRun, bar_full + 8 * pos);
                bulk_load(stage0 + (uint32_t)pos * kMbChunk + kMbRun, src + kMbRun, kMbRun, bar_full + 8 * pos);
            } else {
                mbar_arrive(bar_full + 8 * pos);
            }
            at += (uint64_t)kMbChunk * 149ull;
            if (++pos == kMbRing) {
                pos = 0;
                phase ^= 1u;
            }
        }
    } else {
        int pos = 0;
        uint32_t phase = 0;
        double ar[kMbRC], ai[kMbRC];
#pragma unroll
        for (int r = 0; r < kMbRC; ++r) {
            ar[r] = 0.0;
            ai[r] = 0.0;
        }
        const unsigned long long t0 = clock64();
        for (int c = 0; c < n_chunks; ++c) {
            mbar_wait(bar_full + 8 * pos, phase);
            const unsigned char* cp = smem + (size_t)pos * kMbChunk;
            for (int t = 0; t < p.terms_per_chunk; ++t) {
                // the access pattern of accumulate_chunk: element tid ^ xt of slice rl ^ xr, coefficient with a sign
                const uint32_t xt = (uint32_t)(t * 37 + c) & 255u, xr = (uint32_t)(t + c) & (uint32_t)(kMbRC - 1);
                const double a = __hiloint2double(0x3FF00000 ^ (int)(((uint32_t)__popc((uint32_t)tid & xt) & 1u) << 31), 0);
                const unsigned char* pb = cp + (((uint32_t)tid ^ xt) * 16u);
#pragma unroll
                for (int rl = 0; rl < kMbRC; ++rl) {
                    const double2 v = *reinterpret_cast<const double2*>(pb + (((uint32_t)rl ^ xr) * kMbSlice));
                    ar[rl] = __fma_rn(a, v.x, ar[rl]);
                    ai[rl] = __fma_rn(a, v.y, ai[rl]);
                }
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(bar_empty + 8 * pos);
            if (++pos == kMbRing) {
                pos = 0;
                phase ^= 1u;
            }
        }
        const unsigned long long t1 = clock64();
        double sr = 0.0, si = 0.0;
#pragma unroll
        for (int r = 0; r < kMbRC; ++r) {
            sr += ar[r];
            si += ai[r];
        }
        p.sink[(size_t)blockIdx.x * kMbConsumerThreads + tid] = make_double2(sr, si);
        if (tid == 0) p.cycles[blockIdx.x] = t1 - t0;
    }
}

// mode 0: 8 independent FP64 add chains per thread; mode 1: the per-term sequence of the dense-table kernel
// (apply_h_dense.cu walk_bins): broadcast LDS of a 16-byte entry, AND + POPC + shift + XOR into the sign, FP64 add into one
// of 8 bin registers.  512 threads per SM (16 warps), as that kernel.
__global__ void __launch_bounds__(512, 1) mb_alu_kernel(int iters, int mode, double seed, double* sink,
                                                        unsigned long long* cycles) {
    __shared__ uint4 ent[512];
    const int tid = threadIdx.x;
    {
        const double a = seed * (1.0 + tid);
        ent[tid] = make_uint4(0x9E3779B1u * (uint32_t)(tid + 1), 0u, (uint32_t)__double2loint(a), (uint32_t)__double2hiint(a));
    }
    __syncthreads();
    double c[8];
#pragma unroll
    for (int k = 0; k < 8; ++k) c[k] = seed * k;
    const uint32_t bt = blockIdx.x * 512u + (uint32_t)tid;
    const unsigned long long t0 = clock64();
    if (mode == 0) {
        const double x = seed;
        for (int i = 0; i < iters; ++i) {
#pragma unroll
            for (int u = 0; u < 8; ++u) {
#pragma unroll
                for (int k = 0; k < 8; ++k) c[k] += x;
            }
        }
    } else {
        uint32_t t = 0;
        for (int i = 0; i < iters; ++i) {
#pragma unroll
            for (int u = 0; u < 8; ++u) {
#pragma unroll
                for (int k = 0; k < 8; ++k) {
                    const uint4 e = ent[t];
                    t = (t + 1) & 511u;
                    const uint32_t sgn = (uint32_t)__popc(bt & e.x) << 31;
                    c[k] += __hiloint2double((int)(e.w ^ sgn), (int)e.z);
                }
            }
        }
    }
    const unsigned long long t1 = clock64();
    double s = 0.0;
#pragma unroll
    for (int k = 0; k < 8; ++k) s += c[k];
    sink[(size_t)blockIdx.x * 512 + tid] = s;
    if (tid == 0) cycles[blockIdx.x] = t1 - t0;
}

// Do global loads share the shared-memory data path?  256 threads per SM; per iteration every thread issues 16 LDG.128
// (ld.global.cg: one 64 KiB stretch of an L2-resident buffer per CTA and iteration, coalesced) and `lds_passes` x 16
// LDS.128 over a 64 KiB staged chunk (the consumers' access pattern), each value used by one FP64 FMA pair.
__global__ void __launch_bounds__(256, 1) mb_ldg_kernel(const double2* __restrict__ g, uint32_t n_el_log2, int iters,
                                                        int lds_passes, int with_ldg, double2* sink,
                                                        unsigned long long* cycles) {
    extern __shared__ __align__(128) unsigned char mb_smem[];
    const int tid = threadIdx.x;
    for (int i = tid; i < 65536 / 16; i += 256) reinterpret_cast<double2*>(mb_smem)[i] = make_double2(1.0, 0.5);
    __syncthreads();
    const uint32_t sb = smem_u32(mb_smem) + (uint32_t)tid * 16u;
    double ar[16], ai[16];
#pragma unroll
    for (int r = 0; r < 16; ++r) {
        ar[r] = 0.0;
        ai[r] = 0.0;
    }
    const uint32_t mask = (1u << n_el_log2) - 1u;
    uint32_t pos = (blockIdx.x * 4096u * 37u) & mask;
    const unsigned long long t0 = clock64();
    for (int it = 0; it < iters; ++it) {
        double2 vg[16];
        if (with_ldg) {
#pragma unroll
            for (int r = 0; r < 16; ++r) {
                const double2* q = g + ((pos + (uint32_t)r * 256u + (uint32_t)tid) & mask);
                asm volatile("ld.global.cg.v2.f64 {%0, %1}, [%2];" : "=d"(vg[r].x), "=d"(vg[r].y) : "l"(q));
            }
            pos = (pos + 4096u * 149u) & mask;
        }
        for (int s = 0; s < lds_passes; ++s) {
            double2 vs[16];
#pragma unroll
            for (int r = 0; r < 16; ++r)
                asm volatile("ld.shared.v2.f64 {%0, %1}, [%2];"
                             : "=d"(vs[r].x), "=d"(vs[r].y)
                             : "r"(sb + (((uint32_t)r ^ ((uint32_t)(it + s) & 15u)) << 12)));
#pragma unroll
            for (int r = 0; r < 16; ++r) {
                ar[r] = __fma_rn(1.0000001, vs[r].x, ar[r]);
                ai[r] = __fma_rn(1.0000001, vs[r].y, ai[r]);
            }
        }
        if (with_ldg) {
#pragma unroll
            for (int r = 0; r < 16; ++r) {
                ar[r] = __fma_rn(1.0000001, vg[r].x, ar[r]);
                ai[r] = __fma_rn(1.0000001, vg[r].y, ai[r]);
            }
        }
    }
    const unsigned long long t1 = clock64();
    double sr = 0.0, si = 0.0;
#pragma unroll
    for (int r = 0; r < 16; ++r) {
        sr += ar[r];
        si += ai[r];
    }
    sink[(size_t)blockIdx.x * 256 + tid] = make_double2(sr, si);
    if (tid == 0) cycles[blockIdx.x] = t1 - t0;
}

// Distributed shared memory: clusters of two CTAs (two SMs); every thread reads 16-byte elements of a staged 64 KiB chunk with
// the consumers' access pattern through the shared::cluster window -- of its OWN CTA (remote = 0) or of the PEER CTA (remote =
// 1: SM-to-SM reads).  What a 2-CTA variant of the scatter-tile kernel (one 256 KiB tile pair per cluster) would pay for the
// half of its reads that land in the peer's shared memory.
__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(256, 1)
mb_dsmem_kernel(int iters, int remote, double2* sink, unsigned long long* cycles) {
    extern __shared__ __align__(128) unsigned char mb_smem[];
    const int tid = threadIdx.x;
    for (int i = tid; i < 65536 / 16; i += 256) reinterpret_cast<double2*>(mb_smem)[i] = make_double2(1.0, 0.5);
    uint32_t rank;
    asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(rank));
    asm volatile("barrier.cluster.arrive.release.aligned;\nbarrier.cluster.wait.acquire.aligned;" ::: "memory");
    const uint32_t local = smem_u32(mb_smem) + (uint32_t)tid * 16u;
    uint32_t base;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(base) : "r"(local), "r"(remote ? rank ^ 1u : rank));
    double ar[16], ai[16];
#pragma unroll
    for (int r = 0; r < 16; ++r) {
        ar[r] = 0.0;
        ai[r] = 0.0;
    }
    const unsigned long long t0 = clock64();
    for (int it = 0; it < iters; ++it) {
        double2 v[16];
#pragma unroll
        for (int r = 0; r < 16; ++r)
            asm volatile("ld.shared::cluster.v2.f64 {%0, %1}, [%2];"
                         : "=d"(v[r].x), "=d"(v[r].y)
                         : "r"(base + (((uint32_t)r ^ ((uint32_t)it & 15u)) << 12)));
#pragma unroll
        for (int r = 0; r < 16; ++r) {
            ar[r] = __fma_rn(1.0000001, v[r].x, ar[r]);
            ai[r] = __fma_rn(1.0000001, v[r].y, ai[r]);
        }
    }
    const unsigned long long t1 = clock64();
    // the peer may still be reading this CTA's shared memory
    asm volatile("barrier.cluster.arrive.release.aligned;\nbarrier.cluster.wait.acquire.aligned;" ::: "memory");
    double sr = 0.0, si = 0.0;
#pragma unroll
    for (int r = 0; r < 16; ++r) {
        sr += ar[r];
        si += ai[r];
    }
    sink[(size_t)blockIdx.x * 256 + tid] = make_double2(sr, si);
    if (tid == 0) cycles[blockIdx.x] = t1 - t0;
}

}  // namespace
}  // namespace syk

extern "C" {

size_t syk_microbench_workspace_bytes(void) { return (size_t)4 << 20; }

int syk_microbench(int kind, int arg0, int arg1, const void* d_buf, size_t buf_bytes, void* d_work, size_t work_bytes,
                   double* result, void* stream) {
    using namespace syk;
    if (!result || !d_work || work_bytes < syk_microbench_workspace_bytes()) return SYK_EINVAL;
    cudaStream_t st = (cudaStream_t)stream;
    const int sms = num_sms();
    if (sms <= 0) return SYK_ECUDA;
    unsigned long long* d_cycles = (unsigned long long*)d_work;
    void* d_sink = (char*)d_work + 4096;
    if ((size_t)sms * 512 * 16 + 4096 > work_bytes) return SYK_EINVAL;
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    SYK_CUDA(cudaEventCreate(&e0));
    SYK_CUDA(cudaEventCreate(&e1));
    double units = 0.0, units2 = 0.0;
    int rc = SYK_OK;
    double cyc_even = 0.0, cyc_odd = 0.0;
    if ((kind >= 0 && kind <= 2) || kind == 5) {
        // 0: loads only; 1: LDS + FMA only; 2: both.  arg0 = chunks per CTA, arg1 = terms per chunk
        // 5: loads only, two groups: even CTAs walk the whole buffer (DRAM), odd CTAs its first 32 MB (L2) with arg1 times
        //    as many chunks
        int buf_log2 = 0;
        while (((size_t)2 << buf_log2) <= buf_bytes) ++buf_log2;
        if (kind != 1 && (!d_buf || buf_log2 < 17 || ((uintptr_t)d_buf & 127))) rc = SYK_EINVAL;
        if (arg0 < 1 || arg1 < 0) rc = SYK_EINVAL;
        // kind 0: arg1 > 0 limits the launch to arg1 CTAs (per-SM rate when only some SMs pull from L2)
        const int grid = kind == 0 && arg1 > 0 && arg1 < sms ? arg1 : sms;
        if (rc == SYK_OK) {
            MbParams p;
            p.buf = (const unsigned char*)d_buf;
            p.buf_log2 = buf_log2;
            p.n_chunks = arg0;
            p.terms_per_chunk = (kind == 0 || kind == 5) ? 0 : arg1;
            p.load = kind != 1;
            p.small_log2 = kind == 5 ? 25 : 0;
            p.small_mult = kind == 5 ? (arg1 > 0 ? arg1 : 1) : 1;
            p.sink = (double2*)d_sink;
            p.cycles = d_cycles;
            const size_t smem = (size_t)kMbRing * kMbChunk + 2 * kMbRing * 8 + 64;
            cudaError_t e = cudaFuncSetAttribute(mb_stream_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
            if (e == cudaSuccess) {
                cudaEventRecord(e0, st);
                cudaMemsetAsync(d_cycles, 0, sizeof(unsigned long long) * (size_t)sms, st);
                mb_stream_kernel<<<grid, kMbThreads, smem, st>>>(p);
                cudaEventRecord(e1, st);
                e = cudaGetLastError();
            }
            if (e != cudaSuccess) {
                set_cuda_error(e, "mb_stream_kernel");
                rc = SYK_ECUDA;
            }
            units = p.load ? (double)grid * arg0 * (double)kMbChunk : 0.0;                      // bytes L2/DRAM -> smem
            units2 = (double)sms * arg0 * (double)p.terms_per_chunk * (double)kMbChunk;         // bytes read by LDS
            if (kind == 5) {   // bytes of the even (whole buffer) and of the odd (L2-resident region) group
                units = (double)((sms + 1) / 2) * arg0 * (double)kMbChunk;
                units2 = (double)(sms / 2) * arg0 * (double)p.small_mult * (double)kMbChunk;
            }
            count_launch();
        }
    } else if (kind == 3 || kind == 4) {
        if (arg0 < 1) rc = SYK_EINVAL;
        if (rc == SYK_OK) {
            cudaEventRecord(e0, st);
            mb_alu_kernel<<<sms, 512, 0, st>>>(arg0, kind == 3 ? 0 : 1, 1.0 + 1e-9 * arg1, (double*)d_sink, d_cycles);
            cudaEventRecord(e1, st);
            cudaError_t e = cudaGetLastError();
            if (e != cudaSuccess) {
                set_cuda_error(e, "mb_alu_kernel");
                rc = SYK_ECUDA;
            }
            units = (double)sms * 512.0 * 64.0 * arg0;   // thread-level adds
            count_launch();
        }
    } else if (kind == 6) {
        // arg0 = iterations, arg1 = LDS passes per iteration (0 = global loads only); d_buf = NULL: LDS only
        int buf_log2 = 0;
        while (d_buf && ((size_t)2 << buf_log2) <= buf_bytes) ++buf_log2;
        if (arg0 < 1 || arg1 < 0 || (!d_buf && arg1 < 1) || (d_buf && (buf_log2 < 17 || ((uintptr_t)d_buf & 127)))) rc = SYK_EINVAL;
        if (rc == SYK_OK) {
            cudaError_t e = cudaFuncSetAttribute(mb_ldg_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 65536);
            if (e == cudaSuccess) {
                cudaEventRecord(e0, st);
                mb_ldg_kernel<<<sms, 256, 65536, st>>>((const double2*)d_buf, d_buf ? (uint32_t)(buf_log2 - 4) : 0u, arg0, arg1,
                                                       d_buf ? 1 : 0, (double2*)d_sink, d_cycles);
                cudaEventRecord(e1, st);
                e = cudaGetLastError();
            }
            if (e != cudaSuccess) {
                set_cuda_error(e, "mb_ldg_kernel");
                rc = SYK_ECUDA;
            }
            units = d_buf ? (double)sms * arg0 * 65536.0 : 0.0;       // bytes by global loads
            units2 = (double)sms * arg0 * (double)arg1 * 65536.0;     // bytes by LDS
            count_launch();
        }
    } else if (kind == 7) {
        // arg0 = iterations, arg1 = 0: own shared memory through the cluster window, 1: the peer CTA's (DSMEM)
        if (arg0 < 1 || (arg1 != 0 && arg1 != 1)) rc = SYK_EINVAL;
        if (rc == SYK_OK) {
            const int grid = sms & ~1;   // whole clusters of two
            cudaError_t e = cudaFuncSetAttribute(mb_dsmem_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 65536);
            if (e == cudaSuccess) e = cudaMemsetAsync(d_cycles, 0, sizeof(unsigned long long) * (size_t)sms, st);
            if (e == cudaSuccess) {
                cudaEventRecord(e0, st);
                mb_dsmem_kernel<<<grid, 256, 65536, st>>>(arg0, arg1, (double2*)d_sink, d_cycles);
                cudaEventRecord(e1, st);
                e = cudaGetLastError();
            }
            if (e != cudaSuccess) {
                set_cuda_error(e, "mb_dsmem_kernel");
                rc = SYK_ECUDA;
            }
            units2 = (double)grid * arg0 * 65536.0;   // bytes read through the cluster window
            count_launch();
        }
    } else {
        rc = SYK_EINVAL;
    }
    if (rc == SYK_OK) {
        float ms = 0.f;
        std::vector<unsigned long long> cyc((size_t)sms);
        cudaError_t e = cudaEventSynchronize(e1);
        if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, e0, e1);
        if (e == cudaSuccess) e = cudaMemcpy(cyc.data(), d_cycles, sizeof(unsigned long long) * (size_t)sms, cudaMemcpyDeviceToHost);
        if (e != cudaSuccess) {
            set_cuda_error(e, "syk_microbench");
            rc = SYK_ECUDA;
        } else {
            const unsigned long long cmax = *std::max_element(cyc.begin(), cyc.end());
            for (int i = 0; i < sms; ++i) {
                double& dst = (i & 1) ? cyc_odd : cyc_even;
                dst = std::max(dst, (double)cyc[(size_t)i]);
            }
            result[0] = ms;
            result[1] = (double)cmax;
            result[2] = units;
            result[3] = units2;
            result[4] = cyc_even;
            result[5] = cyc_odd;
        }
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    return rc;
}

}  // extern "C"
