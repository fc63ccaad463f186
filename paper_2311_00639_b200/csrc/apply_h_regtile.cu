// a-2  apply_H, register-tile kernel: the gather form of Algorithm 1 with LARGE output tiles.
//
//     out[b] = sum_t c_t (-1)^popcount(b & z_t) in[b ^ x_t]
//
// Persistent CTAs (one per SM), 8 consumer warps + 1 producer warp.  A CTA owns an aligned output tile of
// TILE = 256 R amplitudes (64 KiB: R = 16 complex128 / R = 32 complex64) whose accumulators live in registers
// (R per thread, amplitude loc = tid + 256 r).  For a term with mask x the sources of the tile are exactly the
// aligned tile  tile ^ (x >> tile_log2)  permuted by the low bits of x, so the producer streams whole source tiles
// into a ring of shared-memory slots with cp.async.bulk (TMA unit, SASS UBLKCP; completion on mbarriers) and the
// consumers read slot[(loc ^ xlo)].  Terms are sorted by x: terms with equal x >> tile_log2 share one staged tile
// ("load"), and the 148 CTAs walk the same load list on 148 neighbouring tiles, so terms that agree above
// log2(148 TILE) hit the same lines in L2 shortly after one another.  Larger tiles => fewer L2->SM loads and fewer
// DRAM passes; that is the whole point of keeping the accumulators in registers.
//
// Inner loop cost per (amplitude, term): one LDS, one LOP3 (sign), two FMAs.  Everything that does not depend on
// the thread comes from the __grid_constant__ table (constant bank => uniform registers):
//   * address: slot + ((tid ^ xlo_low8) + 256 (r ^ xlo_high)) * sizeof(amplitude); the second summand is uniform;
//   * sign: popcount((base | tid) & z) once per term and thread, then the r-dependent part (z bits 8..) is walked
//     in Gray-code order so consecutive r differ by one uniform XOR;
//   * the coefficient is exactly real or exactly imaginary (c = J s^4 x {1,-1,i,-i}), so a term costs 2 FMAs per
//     amplitude, not 4; the two cases are a uniform branch.
// No atomics, one write per output: results are bitwise reproducible.
//
// Fused Lanczos epilogue (a-3 part 1) as in apply_h.cu: out = acc/|u_j| - (|u_j|/|u_{j-1}|) prev, per-CTA fp64
// partial sums of Re<in|out>.  in[b] for that sum is read from the LAST load's slot (hi == 0: the tile itself).
#include <atomic>
#include <cstring>
#include <new>
#include <vector>

#include "device_utils.cuh"

namespace syk {

namespace {

constexpr int kConsumerWarps = 8;
constexpr int kConsumerThreads = kConsumerWarps * 32;
constexpr int kThreads = kConsumerThreads + 32;
constexpr int kMaxSlots = 12;
constexpr int kChunkBytes = 16384;                 // one cp.async.bulk
constexpr int kSmemLimit = 232448;                 // 227 KiB opt-in maximum per CTA on sm_100
constexpr int kMiscBytes = 2 * kMaxSlots * 8 + 40 * 8 + 128;

template <typename T>
struct RtParams {
    using C = typename Cx<T>::type;
    const C* in;
    C* out;
    const C* prev;
    LanczosScalars* sc;
    int j;
    int L;
    int nslot;
    // lock-step of the persistent CTAs (see lockstep_gate): nullptr = free running
    uint32_t* sync;
    int epoch_len;   // loads per epoch
    int lag;         // a CTA may start epoch e once every CTA has issued epoch e-1-lag
};

__host__ __device__ constexpr int ilog2(int v) { return v <= 1 ? 0 : 1 + ilog2(v >> 1); }

__device__ __forceinline__ void fused_scalars(LanczosScalars* sc, int j, double* red, double& s_in, double& s_prev) {
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

__device__ __forceinline__ double fma_rn(double a, double b, double c) { return __fma_rn(a, b, c); }
__device__ __forceinline__ float fma_rn(float a, float b, float c) { return __fmaf_rn(a, b, c); }

// One term applied to the R accumulators of a thread.  `w` = sign-carrying word of the coefficient (high word of
// the double / the float itself) already multiplied by the thread's own sign; the remaining sign depends on r only
// through z bits 8.. and is walked in Gray-code order (one uniform XOR per step).
template <typename T, int R, bool IMAG>
__device__ __forceinline__ void accumulate_term(const unsigned char* __restrict__ pb, uint32_t xr, uint32_t z, uint32_t a_lo, uint32_t w, T (&ar)[R],
                                                T (&ai)[R]) {
    using C = typename Cx<T>::type;
#pragma unroll
    for (int i = 0; i < R; ++i) {
        const int r = i ^ (i >> 1);
        if (i > 0) w ^= (z * (0x800000u / (uint32_t)(i & -i))) & 0x80000000u;   // z bit 8 + ctz(i) -> bit 31; a shift after unrolling
        T a;
        if constexpr (sizeof(T) == 8) a = __hiloint2double((int)w, (int)a_lo);
        else a = __uint_as_float(w);
        const C v = *reinterpret_cast<const C*>(pb + ((((uint32_t)r ^ xr) << 8) * (uint32_t)sizeof(C)));
        if constexpr (IMAG) {   // (i a)(vx + i vy) = -a vy + i a vx
            ar[r] = fma_rn(-a, v.y, ar[r]);
            ai[r] = fma_rn(a, v.x, ai[r]);
        } else {
            ar[r] = fma_rn(a, v.x, ar[r]);
            ai[r] = fma_rn(a, v.y, ai[r]);
        }
    }
}

template <typename T, int R, bool FUSED>
__global__ void __launch_bounds__(kThreads, 1)
apply_h_regtile_kernel(const __grid_constant__ RtTable tab, const RtParams<T> p) {
    using C = typename Cx<T>::type;
    constexpr int TILE = R * kConsumerThreads;
    constexpr int TILE_LOG2 = ilog2(TILE);
    constexpr uint32_t TILE_BYTES = TILE * sizeof(C);
    static_assert((1 << TILE_LOG2) == TILE && TILE_BYTES % kChunkBytes == 0, "tile size");

    extern __shared__ __align__(128) unsigned char smem[];
    C* stages = reinterpret_cast<C*>(smem);
    unsigned char* q = smem + (size_t)p.nslot * TILE_BYTES;
    uint64_t* bars = reinterpret_cast<uint64_t*>(q);
    q += 2 * kMaxSlots * 8;
    double* red = reinterpret_cast<double*>(q);

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const uint32_t bar_full = smem_u32(bars), bar_empty = smem_u32(bars + kMaxSlots);
    if (tid == 0) {
        for (int s = 0; s < p.nslot; ++s) {
            mbar_init(bar_full + 8 * s, 1);
            mbar_init(bar_empty + 8 * s, kConsumerWarps);
        }
        mbar_fence_init();
    }
    __syncthreads();

    double s_in = 1.0, s_prev = 0.0;
    if (FUSED) fused_scalars(p.sc, p.j, red, s_in, s_prev);

    const uint32_t n_tiles = 1u << (p.L - TILE_LOG2);
    const int nslot = p.nslot, n_loads = tab.n_loads;
    double dot = 0.0;

    if (warp == kConsumerWarps) {
        // ---------------- producer: one lane streams source tiles into the ring ----------------
        if (lane == 0) {
            int slot = 0;
            uint32_t phase = 0;
            const uint32_t stage0 = smem_u32(stages);
            uint32_t g = 0, until_epoch = 0;   // loads issued; loads left in the current epoch
            for (uint32_t tile = blockIdx.x; tile < n_tiles; tile += gridDim.x) {
                for (int l = 0; l < n_loads; ++l) {
                    if (p.sync) {
                        if (until_epoch == 0) {
                            lockstep_gate(p.sync, g / (uint32_t)p.epoch_len, (uint32_t)p.lag);
                            until_epoch = (uint32_t)p.epoch_len;
                        }
                        --until_epoch;
                        ++g;
                    }
                    mbar_wait(bar_empty + 8 * slot, phase ^ 1u);
                    mbar_arrive_expect_tx(bar_full + 8 * slot, TILE_BYTES);
                    const unsigned char* src =
                        reinterpret_cast<const unsigned char*>(p.in + ((uint64_t)(tile ^ tab.load_hi[l]) << TILE_LOG2));
                    const uint32_t dst = stage0 + (uint32_t)slot * TILE_BYTES;
#pragma unroll
                    for (uint32_t c = 0; c < TILE_BYTES; c += kChunkBytes)
                        bulk_load(dst + c, src + c, kChunkBytes, bar_full + 8 * slot);
                    if (++slot == nslot) {
                        slot = 0;
                        phase ^= 1u;
                    }
                }
            }
            if (p.sync) {
                // report every remaining epoch of the longest-running CTA, so that nobody waits for this one
                const uint32_t E = (uint32_t)p.epoch_len;
                const uint32_t max_loads = ((n_tiles + gridDim.x - 1) / gridDim.x) * (uint32_t)n_loads;
                const uint32_t n_epochs = (max_loads + E - 1) / E;
                for (uint32_t f = g == 0 ? 0 : (g - 1) / E; f < n_epochs; ++f) atomicAdd(p.sync + (f % kSyncRing), 1u);
            }
        }
        __syncwarp();
    } else {
        // ---------------- consumers ----------------
        int slot = 0;
        uint32_t phase = 0;
        for (uint32_t tile = blockIdx.x; tile < n_tiles; tile += gridDim.x) {
            const uint32_t base = tile << TILE_LOG2;
            const uint32_t bt = base | (uint32_t)tid;
            T ar[R], ai[R];
#pragma unroll
            for (int r = 0; r < R; ++r) {
                ar[r] = 0;
                ai[r] = 0;
            }
            for (int l = 0; l < n_loads; ++l) {
                mbar_wait(bar_full + 8 * slot, phase);
                const C* sp = stages + (size_t)slot * TILE;
                const int t1 = tab.load_t0[l + 1];
                for (int t = tab.load_t0[l]; t < t1; ++t) {
                    const uint4 e = tab.term[t];
                    const uint32_t xlo = e.x & 0x7fffffffu;
                    const unsigned char* pb =
                        reinterpret_cast<const unsigned char*>(sp + ((uint32_t)tid ^ (xlo & 255u)));
                    const uint32_t xr = xlo >> 8;
                    const uint32_t sgn = (uint32_t)__popc(bt & e.y) << 31;
                    const uint32_t w = (sizeof(T) == 8 ? e.w : e.z) ^ sgn;
                    if (e.x >> 31) accumulate_term<T, R, true>(pb, xr, e.y, e.z, w, ar, ai);
                    else accumulate_term<T, R, false>(pb, xr, e.y, e.z, w, ar, ai);
                }
                if (l == n_loads - 1) {
                    // epilogue; the last load is the tile itself (hi == 0), still staged in `sp`
#pragma unroll
                    for (int r = 0; r < R; ++r) {
                        const uint32_t loc = (uint32_t)tid + r * kConsumerThreads;
                        const uint64_t b = (uint64_t)base + loc;
                        C o;
                        if (FUSED) {
                            const C mine = sp[loc];
                            double orr = (double)ar[r] * s_in, oi = (double)ai[r] * s_in;
                            if (p.prev) {
                                const C pv = p.prev[b];
                                orr -= s_prev * (double)pv.x;
                                oi -= s_prev * (double)pv.y;
                            }
                            o.x = (T)orr;
                            o.y = (T)oi;
                            dot += (double)mine.x * (double)o.x + (double)mine.y * (double)o.y;
                        } else {
                            o.x = ar[r];
                            o.y = ai[r];
                        }
                        p.out[b] = o;
                    }
                }
                __syncwarp();
                if (lane == 0) mbar_arrive(bar_empty + 8 * slot);
                if (++slot == nslot) {
                    slot = 0;
                    phase ^= 1u;
                }
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

// R per dtype index (SYK_C64 = 0, SYK_C128 = 1): 64 KiB tiles
constexpr int kRt_R[2] = {32, 16};
constexpr int kRtTileLog2[2] = {13, 12};
constexpr uint32_t kRtTileBytes = 65536;

// Flattened term list in canonical order (groups by ascending x, terms by ascending z) cut into loads =
// runs of equal x >> tile_log2, rotated so that the hi == 0 load (always present, possibly empty) comes last.
bool build_rt_table(const syk_ham* h, int dtype, int tile_log2, RtTable& tab) {
    const size_t nt = h->z.size();
    if (nt > (size_t)kRtMaxTerms) return false;
    struct Item { uint32_t hi; uint4 e; };
    std::vector<Item> items;
    items.reserve(nt);
    const uint32_t lo_mask = (1u << tile_log2) - 1u;
    for (size_t g = 0; g < h->x.size(); ++g) {
        const uint32_t x = (uint32_t)h->x[g];
        for (uint32_t t = h->group_off[g]; t < h->group_off[g + 1]; ++t) {
            const std::complex<double> c = h->c[t];
            const bool imag = c.imag() != 0.0;
            if (imag && c.real() != 0.0) return false;   // never for SYK strings (c = J s^4 {1,-1,i,-i})
            const double a = imag ? c.imag() : c.real();
            Item it;
            it.hi = x >> tile_log2;
            it.e.x = (x & lo_mask) | (imag ? 0x80000000u : 0u);
            it.e.y = (uint32_t)h->z[t];
            if (dtype == SYK_C128) {
                uint64_t bits;
                std::memcpy(&bits, &a, 8);
                it.e.z = (uint32_t)bits;
                it.e.w = (uint32_t)(bits >> 32);
            } else {
                const float af = (float)a;   // R-C64: rounded once
                uint32_t bits;
                std::memcpy(&bits, &af, 4);
                it.e.z = bits;
                it.e.w = 0;
            }
            items.push_back(it);
        }
    }
    // items are sorted by x, hence by hi; loads with hi != 0 first, then the hi == 0 load
    size_t first_nonzero = 0;
    while (first_nonzero < items.size() && items[first_nonzero].hi == 0) ++first_nonzero;
    int n_loads = 0;
    size_t out = 0;
    for (size_t i = first_nonzero; i < items.size(); ++i) {
        if (i == first_nonzero || items[i].hi != items[i - 1].hi) {
            if (n_loads >= kRtMaxLoads - 1) return false;
            tab.load_hi[n_loads] = items[i].hi;
            tab.load_t0[n_loads] = (uint16_t)out;
            ++n_loads;
        }
        tab.term[out++] = items[i].e;
    }
    tab.load_hi[n_loads] = 0;
    tab.load_t0[n_loads] = (uint16_t)out;
    ++n_loads;
    for (size_t i = 0; i < first_nonzero; ++i) tab.term[out++] = items[i].e;
    tab.load_t0[n_loads] = (uint16_t)out;
    tab.n_loads = n_loads;
    tab.tile_log2 = tile_log2;
    return true;
}

const RtTable* get_rt_table(const syk_ham* h, int dtype) {
    const int k = dtype == SYK_C128 ? 1 : 0;
    const int key = k * 64 + kRtTileLog2[k];
    if (!h->rt[k]) h->rt[k] = new (std::nothrow) RtCache();
    if (!h->rt[k]) return nullptr;
    if (h->rt[k]->valid_for != key) {
        if (!build_rt_table(h, dtype, kRtTileLog2[k], h->rt[k]->tab)) return nullptr;
        h->rt[k]->valid_for = key;
    }
    return &h->rt[k]->tab;
}

// epoch length / lag of the lock-step (syk_set_lockstep; epoch_len 0 = free running).  Defaults from the sweeps
// in profiles/r1e_lockstep_sweep.md (this kernel: N = 64 complex64 505 -> 345..361 ms, N = 56 complex128 unchanged).
struct LockstepConfig { int epoch_len; int lag; };
std::atomic<int> g_ls_epoch{8}, g_ls_lag{1};
LockstepConfig lockstep_config() { return LockstepConfig{g_ls_epoch.load(), g_ls_lag.load()}; }

template <typename T, int R>
int launch_rt(const syk_ham* h, const RtTable& tab, const void* d_in, void* d_out, const FusedArgs& fa,
              cudaStream_t stream) {
    using C = typename Cx<T>::type;
    RtParams<T> p;
    p.in = (const C*)d_in;
    p.out = (C*)d_out;
    p.prev = (const C*)fa.prev;
    p.sc = fa.sc;
    p.j = fa.j;
    p.L = h->L;
    p.nslot = (int)((kSmemLimit - kMiscBytes) / kRtTileBytes);
    if (p.nslot > kMaxSlots) p.nslot = kMaxSlots;
    const size_t smem = (size_t)p.nslot * kRtTileBytes + kMiscBytes;
    const int sms = num_sms();
    if (sms <= 0) return SYK_ECUDA;
    const uint64_t n_tiles = 1ull << (h->L - tab.tile_log2);
    const int grid = (int)(n_tiles < (uint64_t)sms ? n_tiles : (uint64_t)sms);
    // lock-step only where it pays: the vector does not fit in L2 and there are several rounds of tiles
    const LockstepConfig ls = lockstep_config();
    p.sync = nullptr;
    p.epoch_len = ls.epoch_len;
    p.lag = ls.lag;
    if (ls.epoch_len > 0 && n_tiles * kRtTileBytes > ((uint64_t)64 << 20) && n_tiles >= 4 * (uint64_t)grid) {
        p.sync = h->dev.sync;
        SYK_CUDA(cudaMemsetAsync(p.sync, 0, kSyncRing * sizeof(uint32_t), stream));
    }
    if (fa.sc) {
        SYK_CUDA(cudaFuncSetAttribute(apply_h_regtile_kernel<T, R, true>,
                                      cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        apply_h_regtile_kernel<T, R, true><<<grid, kThreads, smem, stream>>>(tab, p);
    } else {
        SYK_CUDA(cudaFuncSetAttribute(apply_h_regtile_kernel<T, R, false>,
                                      cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        apply_h_regtile_kernel<T, R, false><<<grid, kThreads, smem, stream>>>(tab, p);
    }
    count_launch();
    SYK_CUDA(cudaGetLastError());
    return SYK_OK;
}

}  // namespace

int regtile_tile_log2(const syk_ham* h, int dtype, bool forced) {
    const int k = dtype == SYK_C128 ? 1 : 0;
    if (h->n_terms() > kRtMaxTerms || h->L < kRtTileLog2[k]) return 0;
    // automatic choice: needs enough 64 KiB tiles to fill the 148 SMs a few times over; smaller vectors use the
    // 16 KiB-tile kernel (more, smaller tiles)
    if (!forced && h->L < kRtTileLog2[k] + 10) return 0;
    return get_rt_table(h, dtype) ? kRtTileLog2[k] : 0;
}

int launch_apply_h_regtile(const syk_ham* h, int dtype, const void* d_in, void* d_out, const FusedArgs& fa,
                           cudaStream_t stream) {
    const RtTable* tab = get_rt_table(h, dtype);
    if (!tab) return SYK_EINVAL;
    if (dtype == SYK_C128) return launch_rt<double, kRt_R[1]>(h, *tab, d_in, d_out, fa, stream);
    return launch_rt<float, kRt_R[0]>(h, *tab, d_in, d_out, fa, stream);
}

void set_lockstep(int epoch_len, int lag) {
    g_ls_epoch.store(epoch_len);
    g_ls_lag.store(lag);
}

void get_lockstep(int* epoch_len, int* lag) {
    *epoch_len = g_ls_epoch.load();
    *lag = g_ls_lag.load();
}

void free_regtile_tables(const syk_ham* h) {
    for (int k = 0; k < 2; ++k) {
        delete h->rt[k];
        h->rt[k] = nullptr;
    }
}

}  // namespace syk
