// a-2  apply_H: the gather form of the paper's Algorithm 1
//
//     out[b] = sum_g in[b ^ x_g] * sum_{t in g} c_t (-1)^popcount(b & z_t)
//
// Algorithm 1's three loops become: outer loop over m -> one thread per output amplitude (a few per thread);
// middle loop over tuples -> loop over X-mask groups and their terms (tables in shared memory); inner loop over
// set bits -> one XOR and one POPC.  It is a gather: no atomics, results bitwise reproducible.
//
// Two kernels:
//   * apply_h_tma_kernel  -- the sm_100a path.  Persistent CTAs (one per SM).  The vector is cut into aligned
//     tiles of 16 KiB; for an output tile B and a mask x the sources {b ^ x} are exactly the aligned tile
//     B ^ (x >> tile_log2), permuted by the low bits of x.  A producer warp streams those source tiles into a
//     shared-memory ring with cp.async.bulk (the TMA unit; SASS UBLKCP) signalling mbarriers; eight consumer
//     warps read the ring with the XOR-permuted index (conflict-free 8/16-byte LDS) and accumulate in registers.
//     Groups are sorted by x, so masks that share x >> tile_log2 reuse one staged tile, and all CTAs walk the
//     mask list in the same order on neighbouring tiles, so masks that share their high bits hit in L2.
//   * apply_h_generic_kernel -- plain per-thread gather with tables read through the read-only path; used when
//     the table does not fit in shared memory (dense H, N >= 20) or the vector is smaller than one tile.
//
// Fused epilogue for the Lanczos step (a-3): out = acc/|u_j| - (|u_j|/|u_{j-1}|) prev, partial sums of
// Re <in|out> per CTA (fp64), see common.h FusedArgs.
#include <vector>

#include "device_utils.cuh"

namespace syk {

namespace {

constexpr int kConsumerWarps = 8;
constexpr int kConsumerThreads = kConsumerWarps * 32;
constexpr int kTmaThreads = kConsumerThreads + 32;
constexpr int kMaxStages = 13;
constexpr int kTileBytes = 16384;
constexpr int kSmemLimit = 232448;   // 227 KiB opt-in maximum per CTA on sm_100

template <typename T>
struct Params {
    using C = typename Cx<T>::type;
    const C* in;
    C* out;
    const C* prev;            // fused only; may alias out
    LanczosScalars* sc;       // nullptr = plain
    int j;
    const uint32_t* gx;
    const uint32_t* goff;
    const uint32_t* tz;
    const C* tc;
    const uint32_t* load_hi;
    const uint32_t* load_g0;
    int n_groups, n_terms, n_loads;
    int L;
    int nstage;
};

// Scalars of the fused epilogue: finalises |u_j| from the partial sums left by the preceding vector kernel.
__device__ __forceinline__ void fused_prologue(LanczosScalars* sc, int j, double* red, double& s_in, double& s_prev) {
    double n2 = reduce_partials(sc->partial_nrm, sc->n_partial_nrm, red);
    double nj = sqrt(n2);
    if (blockIdx.x == 0 && threadIdx.x == 0) sc->nrm[j] = nj;
    s_in = nj > 0.0 ? 1.0 / nj : 0.0;
    s_prev = 0.0;
    if (j > 1) {
        double np = sc->nrm[j - 1];
        s_prev = np > 0.0 ? nj / np : 0.0;
    }
}

// ---------------------------------------------------------------------------------------------------------
// generic kernel
// ---------------------------------------------------------------------------------------------------------
template <typename T, bool FUSED>
__global__ void __launch_bounds__(256) apply_h_generic_kernel(Params<T> p) {
    using C = typename Cx<T>::type;
    __shared__ double red[40];
    double s_in = 1.0, s_prev = 0.0;
    if (FUSED) fused_prologue(p.sc, p.j, red, s_in, s_prev);
    const uint64_t D = 1ull << p.L;
    double dot = 0.0;
    for (uint64_t b = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; b < D; b += (uint64_t)gridDim.x * blockDim.x) {
        const uint32_t b32 = (uint32_t)b;
        T ar = 0, ai = 0;
        for (int g = 0; g < p.n_groups; ++g) {
            const uint32_t x = __ldg(p.gx + g);
            const uint32_t t0 = __ldg(p.goff + g), t1 = __ldg(p.goff + g + 1);
            T cr = 0, ci = 0;
            for (uint32_t t = t0; t < t1; ++t) {
                const uint32_t sbit = (__popc(b32 & __ldg(p.tz + t)) & 1u) << 31;
                const C c = __ldg(p.tc + t);
                cr += flip_sign(c.x, sbit);
                ci += flip_sign(c.y, sbit);
            }
            const C v = __ldg(p.in + (b ^ (uint64_t)x));
            ar += cr * v.x - ci * v.y;
            ai += cr * v.y + ci * v.x;
        }
        C o;
        if (FUSED) {
            const C mine = __ldg(p.in + b);
            double orr = (double)ar * s_in, oi = (double)ai * s_in;
            if (p.prev) {
                const C pv = p.prev[b];
                orr -= s_prev * (double)pv.x;
                oi -= s_prev * (double)pv.y;
            }
            o.x = (T)orr;
            o.y = (T)oi;
            dot += (double)mine.x * (double)o.x + (double)mine.y * (double)o.y;
        } else {
            o.x = ar;
            o.y = ai;
        }
        p.out[b] = o;
    }
    if (FUSED) {
        double s = block_sum(dot, red);
        if (threadIdx.x == 0) {
            p.sc->partial_dot[blockIdx.x] = s;
            if (blockIdx.x == 0) p.sc->n_partial_dot = gridDim.x;
        }
    }
}

// ---------------------------------------------------------------------------------------------------------
// generic kernel for tiny vectors with many X-masks (dense N <= 24: 256..4096 amplitudes, thousands of terms): one
// amplitude per LANE, the groups shared out over the 32 warps of the block (warp w takes groups w, w + 32, ...), partial
// sums added across warps in a fixed order.  The plain generic kernel walks all terms serially in every thread
// (75 us per product at N = 16 dense); this one is bounded by launch latency.
// ---------------------------------------------------------------------------------------------------------
template <typename T, bool FUSED>
__global__ void __launch_bounds__(1024) apply_h_small_kernel(Params<T> p) {
    using C = typename Cx<T>::type;
    __shared__ double red[40];
    __shared__ T part[32][32][2];
    double s_in = 1.0, s_prev = 0.0;
    if (FUSED) fused_prologue(p.sc, p.j, red, s_in, s_prev);
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const uint32_t b32 = blockIdx.x * 32u + (uint32_t)lane;
    T ar = 0, ai = 0;
    for (int g = warp; g < p.n_groups; g += 32) {
        const uint32_t x = __ldg(p.gx + g);
        const uint32_t t0 = __ldg(p.goff + g), t1 = __ldg(p.goff + g + 1);
        T cr = 0, ci = 0;
        for (uint32_t t = t0; t < t1; ++t) {
            const uint32_t sbit = (__popc(b32 & __ldg(p.tz + t)) & 1u) << 31;
            const C c = __ldg(p.tc + t);
            cr += flip_sign(c.x, sbit);
            ci += flip_sign(c.y, sbit);
        }
        const C v = __ldg(p.in + (b32 ^ x));
        ar += cr * v.x - ci * v.y;
        ai += cr * v.y + ci * v.x;
    }
    part[warp][lane][0] = ar;
    part[warp][lane][1] = ai;
    __syncthreads();
    double dot = 0.0;
    if (warp == 0) {
        T sr = 0, si = 0;
#pragma unroll
        for (int w = 0; w < 32; ++w) {
            sr += part[w][lane][0];
            si += part[w][lane][1];
        }
        C o;
        if (FUSED) {
            const C mine = __ldg(p.in + b32);
            double orr = (double)sr * s_in, oi = (double)si * s_in;
            if (p.prev) {
                const C pv = p.prev[b32];
                orr -= s_prev * (double)pv.x;
                oi -= s_prev * (double)pv.y;
            }
            o.x = (T)orr;
            o.y = (T)oi;
            dot = (double)mine.x * (double)o.x + (double)mine.y * (double)o.y;
        } else {
            o.x = sr;
            o.y = si;
        }
        p.out[b32] = o;
    }
    if (FUSED) {
        double s = block_sum(dot, red);
        if (threadIdx.x == 0) {
            p.sc->partial_dot[blockIdx.x] = s;
            if (blockIdx.x == 0) p.sc->n_partial_dot = gridDim.x;
        }
    }
}

// ---------------------------------------------------------------------------------------------------------
// TMA-pipelined tile kernel.  R = outputs per consumer thread; tile = R * 256 amplitudes = 16 KiB.
// ---------------------------------------------------------------------------------------------------------
template <typename T, int R, bool FUSED>
__device__ __forceinline__ void tma_body(const Params<T>& p) {
    using C = typename Cx<T>::type;
    constexpr int TILE = R * kConsumerThreads;
    static_assert(TILE * sizeof(C) == kTileBytes, "tile must be 16 KiB");
    constexpr int TILE_LOG2 = (sizeof(C) == 16) ? 10 : 11;
    static_assert((1 << TILE_LOG2) == TILE, "tile size");

    extern __shared__ __align__(128) unsigned char smem[];
    C* stages = reinterpret_cast<C*>(smem);
    unsigned char* q = smem + (size_t)p.nstage * kTileBytes;
    C* s_tc = reinterpret_cast<C*>(q);              q += (size_t)p.n_terms * sizeof(C);
    uint64_t* bars = reinterpret_cast<uint64_t*>(q); q += (size_t)2 * kMaxStages * 8;
    double* red = reinterpret_cast<double*>(q);      q += 40 * 8;
    uint32_t* s_gx = reinterpret_cast<uint32_t*>(q); q += (size_t)p.n_groups * 4;
    uint32_t* s_goff = reinterpret_cast<uint32_t*>(q); q += (size_t)(p.n_groups + 1) * 4;
    uint32_t* s_tz = reinterpret_cast<uint32_t*>(q); q += (size_t)p.n_terms * 4;
    uint32_t* s_hi = reinterpret_cast<uint32_t*>(q); q += (size_t)p.n_loads * 4;
    uint32_t* s_g0 = reinterpret_cast<uint32_t*>(q);

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;

    for (int i = tid; i < p.n_groups; i += kTmaThreads) s_gx[i] = p.gx[i] & (uint32_t)(TILE - 1);
    for (int i = tid; i <= p.n_groups; i += kTmaThreads) s_goff[i] = p.goff[i];
    for (int i = tid; i < p.n_terms; i += kTmaThreads) {
        s_tz[i] = p.tz[i];
        s_tc[i] = p.tc[i];
    }
    for (int i = tid; i < p.n_loads; i += kTmaThreads) s_hi[i] = p.load_hi[i];
    for (int i = tid; i <= p.n_loads; i += kTmaThreads) s_g0[i] = p.load_g0[i];
    const uint32_t bar_full = smem_u32(bars), bar_empty = smem_u32(bars + kMaxStages);
    if (tid == 0) {
        for (int s = 0; s < p.nstage; ++s) {
            mbar_init(bar_full + 8 * s, 1);
            mbar_init(bar_empty + 8 * s, kConsumerWarps);
        }
        mbar_fence_init();
    }
    __syncthreads();

    double s_in = 1.0, s_prev = 0.0;
    if (FUSED) fused_prologue(p.sc, p.j, red, s_in, s_prev);

    const uint32_t n_tiles = 1u << (p.L - TILE_LOG2);
    const int nstage = p.nstage, n_loads = p.n_loads;
    double dot = 0.0;

    if (warp == kConsumerWarps) {
        // ---------------- producer: one lane streams source tiles into the ring ----------------
        if (lane == 0) {
            int stage = 0;
            uint32_t phase = 0;
            const uint32_t stage0 = smem_u32(stages);
            for (uint32_t tile = blockIdx.x; tile < n_tiles; tile += gridDim.x) {
                for (int l = 0; l < n_loads; ++l) {
                    mbar_wait(bar_empty + 8 * stage, phase ^ 1u);
                    mbar_arrive_expect_tx(bar_full + 8 * stage, kTileBytes);
                    const C* src = p.in + ((uint64_t)(tile ^ s_hi[l]) << TILE_LOG2);
                    bulk_load(stage0 + (uint32_t)stage * kTileBytes, src, kTileBytes, bar_full + 8 * stage);
                    if (++stage == nstage) {
                        stage = 0;
                        phase ^= 1u;
                    }
                }
            }
        }
        __syncwarp();
    } else {
        // ---------------- consumers: R outputs per thread, accumulate over all masks ----------------
        int stage = 0;
        uint32_t phase = 0;
        for (uint32_t tile = blockIdx.x; tile < n_tiles; tile += gridDim.x) {
            const uint32_t base = tile << TILE_LOG2;
            T ar[R], ai[R];
            C mine[R];
#pragma unroll
            for (int r = 0; r < R; ++r) {
                ar[r] = 0;
                ai[r] = 0;
            }
            for (int l = 0; l < n_loads; ++l) {
                mbar_wait(bar_full + 8 * stage, phase);
                const C* st = stages + (size_t)stage * TILE;
                if (FUSED && l == 0) {
#pragma unroll
                    for (int r = 0; r < R; ++r) mine[r] = st[tid + r * kConsumerThreads];
                }
                const int g1 = s_g0[l + 1];
                for (int g = s_g0[l]; g < g1; ++g) {
                    const uint32_t xlo = s_gx[g];
                    const uint32_t t0 = s_goff[g], t1 = s_goff[g + 1];
                    if (t1 - t0 == 1) {
                        const uint32_t z = s_tz[t0];
                        const C c = s_tc[t0];
#pragma unroll
                        for (int r = 0; r < R; ++r) {
                            const uint32_t loc = tid + r * kConsumerThreads;
                            const uint32_t sbit = (__popc((base | loc) & z) & 1u) << 31;
                            const C v = st[loc ^ xlo];
                            const T cr = flip_sign(c.x, sbit), ci = flip_sign(c.y, sbit);
                            ar[r] += cr * v.x - ci * v.y;
                            ai[r] += cr * v.y + ci * v.x;
                        }
                    } else {
                        T cr[R], ci[R];
#pragma unroll
                        for (int r = 0; r < R; ++r) {
                            cr[r] = 0;
                            ci[r] = 0;
                        }
                        for (uint32_t t = t0; t < t1; ++t) {
                            const uint32_t z = s_tz[t];
                            const C c = s_tc[t];
#pragma unroll
                            for (int r = 0; r < R; ++r) {
                                const uint32_t loc = tid + r * kConsumerThreads;
                                const uint32_t sbit = (__popc((base | loc) & z) & 1u) << 31;
                                cr[r] += flip_sign(c.x, sbit);
                                ci[r] += flip_sign(c.y, sbit);
                            }
                        }
#pragma unroll
                        for (int r = 0; r < R; ++r) {
                            const uint32_t loc = tid + r * kConsumerThreads;
                            const C v = st[loc ^ xlo];
                            ar[r] += cr[r] * v.x - ci[r] * v.y;
                            ai[r] += cr[r] * v.y + ci[r] * v.x;
                        }
                    }
                }
                __syncwarp();
                if (lane == 0) mbar_arrive(bar_empty + 8 * stage);
                if (++stage == nstage) {
                    stage = 0;
                    phase ^= 1u;
                }
            }
            // epilogue: 32 lanes write 32 consecutive amplitudes
#pragma unroll
            for (int r = 0; r < R; ++r) {
                const uint64_t b = (uint64_t)base + tid + r * kConsumerThreads;
                C o;
                if (FUSED) {
                    double orr = (double)ar[r] * s_in, oi = (double)ai[r] * s_in;
                    if (p.prev) {
                        const C pv = p.prev[b];
                        orr -= s_prev * (double)pv.x;
                        oi -= s_prev * (double)pv.y;
                    }
                    o.x = (T)orr;
                    o.y = (T)oi;
                    dot += (double)mine[r].x * (double)o.x + (double)mine[r].y * (double)o.y;
                } else {
                    o.x = ar[r];
                    o.y = ai[r];
                }
                p.out[b] = o;
            }
        }
    }
    if (FUSED) {
        double s = block_sum(dot, red);
        if (tid == 0) {
            p.sc->partial_dot[blockIdx.x] = s;
            if (blockIdx.x == 0) p.sc->n_partial_dot = gridDim.x;
        }
    }
}

template <typename T, int R, bool FUSED>
__global__ void __launch_bounds__(kTmaThreads, 1) apply_h_tma_kernel(Params<T> p) {
    tma_body<T, R, FUSED>(p);
}

// Batched over disorder realizations (configs[1]): grid.y = realization.  Every realization has its own
// tables (tab[r]); the vectors and Lanczos scalars of realization r sit at base + r * stride bytes.  Small vectors:
// few stages, so that two CTAs share an SM.
template <typename T>
struct BatchedParams {
    const Params<T>* tab;
    const char* in;
    char* out;
    const char* prev;
    char* sc;
    size_t s_in, s_out, s_prev, s_sc;
    int j;
};

template <typename T, int R, bool FUSED>
__global__ void __launch_bounds__(kTmaThreads, 2) apply_h_tma_batched_kernel(BatchedParams<T> bp) {
    using C = typename Cx<T>::type;
    Params<T> p = bp.tab[blockIdx.y];
    const size_t r = blockIdx.y;
    p.in = reinterpret_cast<const C*>(bp.in + r * bp.s_in);
    p.out = reinterpret_cast<C*>(bp.out + r * bp.s_out);
    p.prev = bp.prev ? reinterpret_cast<const C*>(bp.prev + r * bp.s_prev) : nullptr;
    p.sc = bp.sc ? reinterpret_cast<LanczosScalars*>(bp.sc + r * bp.s_sc) : nullptr;
    p.j = bp.j;
    tma_body<T, R, FUSED>(p);
}

size_t tma_table_bytes(int n_groups, int n_terms, int n_loads, size_t csize) {
    size_t b = (size_t)n_terms * csize + 2 * kMaxStages * 8 + 40 * 8;
    b += (size_t)n_groups * 4 + (size_t)(n_groups + 1) * 4 + (size_t)n_terms * 4;
    b += (size_t)n_loads * 4 + (size_t)(n_loads + 1) * 4;
    return (b + 127) & ~(size_t)127;
}

int tma_stages(const syk_ham* h, int dtype) {
    const int k = dtype == SYK_C128 ? 1 : 0;
    if (h->L < kTileLog2[k]) return 0;
    // n_loads <= n_groups + 1 (known exactly only after the device tables exist; this bound is enough here)
    size_t tb = tma_table_bytes((int)h->n_groups(), (int)h->n_terms(), (int)h->n_groups() + 1, elem_bytes(dtype));
    if (tb + 3 * (size_t)kTileBytes > (size_t)kSmemLimit) return 0;
    int ns = (int)(((size_t)kSmemLimit - tb) / kTileBytes);
    return ns > kMaxStages ? kMaxStages : ns;
}

template <typename T, int R>
int launch_typed(const syk_ham* h, const void* d_in, void* d_out, const FusedArgs& fa, int kind, cudaStream_t stream) {
    using C = typename Cx<T>::type;
    const int k = sizeof(C) == 16 ? 1 : 0;
    const DeviceTables& d = h->dev;
    Params<T> p;
    p.in = (const C*)d_in;
    p.out = (C*)d_out;
    p.prev = (const C*)fa.prev;
    p.sc = fa.sc;
    p.j = fa.j;
    p.gx = d.gx;
    p.goff = d.goff;
    p.tz = d.tz;
    p.tc = k ? (const C*)d.tc128 : (const C*)d.tc64;
    p.load_hi = d.load_hi[k];
    p.load_g0 = d.load_g0[k];
    p.n_groups = (int)h->n_groups();
    p.n_terms = (int)h->n_terms();
    p.n_loads = d.n_loads[k];
    p.L = h->L;
    p.nstage = 0;
    const int sms = num_sms();
    if (sms <= 0) return SYK_ECUDA;
    const bool fused = fa.sc != nullptr;
    if (kind == 1) {
        p.nstage = tma_stages(h, k ? SYK_C128 : SYK_C64);
        const size_t smem = (size_t)p.nstage * kTileBytes +
                            tma_table_bytes(p.n_groups, p.n_terms, p.n_loads, sizeof(C));
        const uint64_t n_tiles = 1ull << (h->L - kTileLog2[k]);
        const int grid = (int)(n_tiles < (uint64_t)sms ? n_tiles : (uint64_t)sms);
        if (fused) {
            SYK_CUDA(cudaFuncSetAttribute(apply_h_tma_kernel<T, R, true>,
                                          cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
            apply_h_tma_kernel<T, R, true><<<grid, kTmaThreads, smem, stream>>>(p);
        } else {
            SYK_CUDA(cudaFuncSetAttribute(apply_h_tma_kernel<T, R, false>,
                                          cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
            apply_h_tma_kernel<T, R, false><<<grid, kTmaThreads, smem, stream>>>(p);
        }
    } else if (h->L >= 5 && h->L <= 12 && p.n_groups >= 64) {
        const int grid = (int)(1u << (h->L - 5));
        if (fused)
            apply_h_small_kernel<T, true><<<grid, 1024, 0, stream>>>(p);
        else
            apply_h_small_kernel<T, false><<<grid, 1024, 0, stream>>>(p);
    } else {
        const uint64_t D = 1ull << h->L;
        uint64_t blocks = (D + 255) / 256;
        const uint64_t cap = (uint64_t)sms * 8;   // 8 resident CTAs of 256 threads per SM: one full wave
        const int grid = (int)(blocks < cap ? blocks : cap);
        if (fused)
            apply_h_generic_kernel<T, true><<<grid, 256, 0, stream>>>(p);
        else
            apply_h_generic_kernel<T, false><<<grid, 256, 0, stream>>>(p);
    }
    count_launch();
    SYK_CUDA(cudaGetLastError());
    return SYK_OK;
}

constexpr int kBatchedStages = 5;

template <typename T, int R>
int launch_batched_typed(const syk_ham* const* hams, int nb, void* d_tab, const void* in, size_t s_in, void* out,
                         size_t s_out, const void* prev, size_t s_prev, void* sc, size_t s_sc, int j, bool upload,
                         cudaStream_t stream) {
    using C = typename Cx<T>::type;
    const int k = sizeof(C) == 16 ? 1 : 0;
    size_t table_max = 0;
    std::vector<Params<T>> host;
    if (upload) host.resize((size_t)nb);
    for (int r = 0; r < nb; ++r) {
        const syk_ham* h = hams[r];
        const DeviceTables& d = h->dev;
        const size_t tb = tma_table_bytes((int)h->n_groups(), (int)h->n_terms(), d.n_loads[k], sizeof(C));
        table_max = tb > table_max ? tb : table_max;
        if (!upload) continue;
        Params<T>& p = host[(size_t)r];
        p.in = nullptr;
        p.out = nullptr;
        p.prev = nullptr;
        p.sc = nullptr;
        p.j = 0;
        p.gx = d.gx;
        p.goff = d.goff;
        p.tz = d.tz;
        p.tc = k ? (const C*)d.tc128 : (const C*)d.tc64;
        p.load_hi = d.load_hi[k];
        p.load_g0 = d.load_g0[k];
        p.n_groups = (int)h->n_groups();
        p.n_terms = (int)h->n_terms();
        p.n_loads = d.n_loads[k];
        p.L = h->L;
        p.nstage = kBatchedStages;
    }
    if (upload) {
        SYK_CUDA(cudaMemcpyAsync(d_tab, host.data(), sizeof(Params<T>) * (size_t)nb, cudaMemcpyHostToDevice, stream));
        SYK_CUDA(cudaStreamSynchronize(stream));   // `host` goes out of scope
    }
    const size_t smem = (size_t)kBatchedStages * kTileBytes + table_max;
    if (smem > (size_t)kSmemLimit) return SYK_EINVAL;
    BatchedParams<T> bp;
    bp.tab = (const Params<T>*)d_tab;
    bp.in = (const char*)in;
    bp.out = (char*)out;
    bp.prev = (const char*)prev;
    bp.sc = (char*)sc;
    bp.s_in = s_in;
    bp.s_out = s_out;
    bp.s_prev = s_prev;
    bp.s_sc = s_sc;
    bp.j = j;
    const uint64_t n_tiles = 1ull << (hams[0]->L - kTileLog2[k]);
    const int sms = num_sms();
    if (sms <= 0) return SYK_ECUDA;
    const unsigned gx = (unsigned)(n_tiles < (uint64_t)sms ? n_tiles : (uint64_t)sms);
    const dim3 grid(gx, (unsigned)nb);
    if (sc) {
        SYK_CUDA(cudaFuncSetAttribute(apply_h_tma_batched_kernel<T, R, true>,
                                      cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        apply_h_tma_batched_kernel<T, R, true><<<grid, kTmaThreads, smem, stream>>>(bp);
    } else {
        SYK_CUDA(cudaFuncSetAttribute(apply_h_tma_batched_kernel<T, R, false>,
                                      cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        apply_h_tma_batched_kernel<T, R, false><<<grid, kTmaThreads, smem, stream>>>(bp);
    }
    count_launch();
    SYK_CUDA(cudaGetLastError());
    return SYK_OK;
}

}  // namespace

size_t batched_table_bytes(int nb) {
    const size_t a = sizeof(Params<double>) > sizeof(Params<float>) ? sizeof(Params<double>) : sizeof(Params<float>);
    return (a * (size_t)nb + 4095) & ~(size_t)4095;
}

// Can these realizations go through the batched tile kernel?  Same N, every table fits the shared-memory budget, the
// vector spans at least one 16 KiB tile.
bool batched_apply_ok(const syk_ham* const* hams, int nb, int dtype) {
    if (!hams || nb < 1 || !hams[0]) return false;
    const int k = dtype == SYK_C128 ? 1 : 0;
    for (int r = 0; r < nb; ++r) {
        const syk_ham* h = hams[r];
        if (!h || h->N != hams[0]->N || h->L < kTileLog2[k] || h->n_terms() == 0 || !h->hermitian) return false;
        // one gamma scaling, one kind of operator and one space for the whole batch (the pipelines take them from hams[0])
        if (h->gamma_norm != hams[0]->gamma_norm || h->generic != hams[0]->generic ||
            h->block_of_N != hams[0]->block_of_N || h->sector != hams[0]->sector || h->perm != hams[0]->perm)
            return false;
        const size_t tb = tma_table_bytes((int)h->n_groups(), (int)h->n_terms(), (int)h->n_groups() + 1, elem_bytes(dtype));
        if (tb + (size_t)kBatchedStages * kTileBytes > (size_t)kSmemLimit / 2 - 1024) return false;   // two CTAs per SM
    }
    return true;
}

int launch_apply_h_batched(const syk_ham* const* hams, int nb, int dtype, void* d_tab, bool upload, const void* in,
                           size_t s_in, void* out, size_t s_out, const void* prev, size_t s_prev, void* sc, size_t s_sc,
                           int j, cudaStream_t stream) {
    for (int r = 0; r < nb; ++r) SYK_TRY(ensure_device_tables(hams[r]));
    profile_begin(stream);
    const int rc = dtype == SYK_C128
                       ? launch_batched_typed<double, 4>(hams, nb, d_tab, in, s_in, out, s_out, prev, s_prev, sc, s_sc, j,
                                                         upload, stream)
                       : launch_batched_typed<float, 8>(hams, nb, d_tab, in, s_in, out, s_out, prev, s_prev, sc, s_sc, j,
                                                        upload, stream);
    profile_end(stream);
    return rc;
}

int apply_h_kernel_kind(const syk_ham* h, int dtype) {
    const int avail = tma_stages(h, dtype) >= 3 ? 1 : 0;
    if (h->forced_kernel == 0) return 0;
    if (h->forced_kernel == 1) return avail;
    if (h->forced_kernel == 4) return dense_kernel_ok(h, true) ? 4 : 0;
    if (h->forced_kernel < 0 && dense_kernel_ok(h, false)) return 4;
    if (h->forced_kernel != 2 && scatter_tile_log2(h, dtype, h->forced_kernel == 3) > 0) return 3;
    if (regtile_tile_log2(h, dtype, h->forced_kernel >= 2) > 0) return 2;
    return avail;
}

int launch_apply_h(const syk_ham* h, int dtype, const void* d_in, void* d_out, const FusedArgs& fa,
                   cudaStream_t stream) {
    if (h->L > 32) return SYK_EINVAL;   // N = 66: only the parity blocks (32 qubits) can be applied
    SYK_TRY(ensure_device_tables(h));
    const int kind = apply_h_kernel_kind(h, dtype);
    profile_begin(stream);
    const int rc = kind == 4   ? launch_apply_h_dense(h, dtype, d_in, d_out, fa, stream)
                   : kind == 3 ? launch_apply_h_scatter(h, dtype, d_in, d_out, fa, stream)
                   : kind == 2 ? launch_apply_h_regtile(h, dtype, d_in, d_out, fa, stream)
                   : dtype == SYK_C128 ? launch_typed<double, 4>(h, d_in, d_out, fa, kind, stream)
                                       : launch_typed<float, 8>(h, d_in, d_out, fa, kind, stream);
    profile_end(stream);
    return rc;
}

}  // namespace syk

extern "C" {

int syk_apply_H(const syk_ham* h, int dtype, const void* d_in, void* d_out, void* stream) {
    if (!h || !d_in || !d_out || (dtype != SYK_C64 && dtype != SYK_C128)) return SYK_EINVAL;
    if (((uintptr_t)d_in & 15) || ((uintptr_t)d_out & 15)) return SYK_EINVAL;
    const size_t bytes = ((size_t)1 << h->L) * syk::elem_bytes(dtype);
    const uintptr_t a = (uintptr_t)d_in, b = (uintptr_t)d_out;
    if (a < b + bytes && b < a + bytes) return SYK_EINVAL;   // overlap (includes in == out)
    syk::FusedArgs fa;
    return syk::launch_apply_h(h, dtype, d_in, d_out, fa, (cudaStream_t)stream);
}

int syk_apply_H_batched(const syk_ham* const* hams, int n_batch, int dtype, const void* d_in, void* d_out,
                        int64_t batch_stride, void* stream) {
    if (!hams || n_batch < 0 || (dtype != SYK_C64 && dtype != SYK_C128)) return SYK_EINVAL;
    const size_t eb = syk::elem_bytes(dtype);
    for (int r = 0; r < n_batch; ++r) {
        if (!hams[r] || hams[r]->N != hams[0]->N) return SYK_EINVAL;
        if (batch_stride < ((int64_t)1 << hams[r]->L)) return SYK_EINVAL;
    }
    for (int r = 0; r < n_batch; ++r) {
        const char* in = (const char*)d_in + (size_t)r * (size_t)batch_stride * eb;
        char* out = (char*)d_out + (size_t)r * (size_t)batch_stride * eb;
        SYK_TRY(syk_apply_H(hams[r], dtype, in, out, stream));
    }
    return SYK_OK;
}

int syk_apply_H_kernel_kind(const syk_ham* h, int dtype) {
    if (!h || (dtype != SYK_C64 && dtype != SYK_C128)) return SYK_EINVAL;
    return syk::apply_h_kernel_kind(h, dtype);
}

int syk_ham_prepare(const syk_ham* h, int dtype) {
    if (!h || (dtype != SYK_C64 && dtype != SYK_C128)) return SYK_EINVAL;
    if (h->L > 32) return SYK_EINVAL;
    SYK_TRY(syk::ensure_device_tables(h));
    const int kind = syk::apply_h_kernel_kind(h, dtype);   // builds the host tables of the tile kernels
    if (kind == 4) SYK_TRY(syk::prepare_dense_tables(h, dtype));
    return SYK_OK;
}

int syk_apply_H_dense_info(const syk_ham* h, int dtype, int* n_loads, int* n_chunks, int* split, int* n_local_groups) {
    if (!h || (dtype != SYK_C64 && dtype != SYK_C128) || !syk::dense_kernel_ok(h, true)) return SYK_EINVAL;
    return syk::dense_tables_info(h, dtype, n_loads, n_chunks, split, n_local_groups);
}

int syk_apply_H_layout(const syk_ham* h, int dtype, int* n_loads, int* n_passes, uint32_t* tile_mask,
                       uint32_t* window_mask) {
    if (!h || (dtype != SYK_C64 && dtype != SYK_C128)) return SYK_EINVAL;
    return syk::scatter_layout_info(h, dtype, n_loads, n_passes, tile_mask, window_mask);
}

int syk_apply_H_trace(const syk_ham* h, int dtype, const void* d_in, void* d_out, int cta, int round, int detail, uint64_t* clk,
                      int clk_capacity, int32_t* load_terms, uint32_t* load_xo, int load_capacity, int* n_loads, int* rot,
                      void* stream) {
    if (!h || !d_in || !d_out || !clk || !load_terms || !load_xo || !n_loads || !rot ||
        (dtype != SYK_C64 && dtype != SYK_C128))
        return SYK_EINVAL;
    if (((uintptr_t)d_in & 15) || ((uintptr_t)d_out & 15) || h->L > 32) return SYK_EINVAL;
    const size_t bytes = ((size_t)1 << h->L) * syk::elem_bytes(dtype);
    const uintptr_t a = (uintptr_t)d_in, b = (uintptr_t)d_out;
    if (a < b + bytes && b < a + bytes) return SYK_EINVAL;
    if (syk::apply_h_kernel_kind(h, dtype) != 3) return SYK_EINVAL;
    SYK_TRY(syk::ensure_device_tables(h));
    return syk::scatter_trace(h, dtype, d_in, d_out, cta, round, detail != 0, clk, clk_capacity, load_terms, load_xo, load_capacity,
                              n_loads, rot, (cudaStream_t)stream);
}

int syk_set_lockstep(int epoch_len, int lag) {
    if (epoch_len < 0 || lag < 0 || lag > syk::kSyncRing - 2) return SYK_EINVAL;
    syk::set_lockstep(epoch_len, lag);
    return SYK_OK;
}

int syk_set_apply_H_kernel(syk_ham* h, int kind) {
    if (!h || kind < -1 || kind > 4) return SYK_EINVAL;
    h->forced_kernel = kind;
    return SYK_OK;
}

}  // extern "C"
