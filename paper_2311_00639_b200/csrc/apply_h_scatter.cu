// a-2  apply_H, scatter-tile kernel: the gather form of Algorithm 1 with 128 KiB output tiles
// whose index bits are CHOSEN per Hamiltonian.
//
//     out[b] = sum_t c_t (-1)^popcount(b & z_t) in[b ^ x_t]
//
// What bounds this product on B200 is not arithmetic but how often the vector is moved: once from DRAM per
// distinct value of (x restricted to the bits above the L2 window), once from L2 into an SM per distinct value of
// (x restricted to the bits outside a tile).  Both counts depend on WHICH qubits are the tile / window bits, and
// the X-masks of a sparse SYK Hamiltonian are random 2- and 4-subsets of the qubits, so the host picks the bits
// (choose_layout: hill climbing on  #loads + 2 #passes; on top of it syk_ham_optimize_layout relabels the qubits so that
// all 13 / 14 tile bits and the 7 window bits are chosen, term_compiler.cpp):
//   * slice bits   : index bits 0..TB-1: a slice = 256 consecutive 16-byte ELEMENTS, one per consumer thread; an
//                    element is one complex128 amplitude (TB = 8) or a pair of adjacent complex64 amplitudes
//                    (TB = 9: both precisions move 16 bytes per LDS and per store);
//   * r bits       : NR = 5 further bit positions P[0..4]; a thread keeps the R = 32 elements
//                    base | deposit(r, P) | element  in registers (128 KiB of accumulators per SM).  P[0..2] = TB..TB+2
//                    (a "run" of 8 slices = 32 KiB contiguous = one cp.async.bulk: the TMA unit costs ~85 clk per
//                    copy, measured, so 2-4 KiB copies cannot feed an SM); the other 2 r bits sit ANYWHERE in the index;
//   * outer bits   : the rest, in an order O[0..]: the tile counter tau is deposited into them, O[0] fastest, so
//                    the 148 tiles in flight differ in O[0..7] only -- those are the L2-window bits.
// No data is permuted: a source tile is fetched run by run (cp.async.bulk, TMA unit, SASS UBLKCP; completion on
// mbarriers) into a ring of shared-memory chunks.  Persistent CTAs, one per SM: two consumer warpgroups (232
// registers per thread after setmaxnreg) and one producer warpgroup (40 registers, one working lane).
//
// Chunked ring: a 128 KiB tile does not fit twice in shared memory, so the ring holds 3 chunks of 64 KiB (half a
// tile).  The source slice of output slice r under mask x is r ^ xr (xr = the r bits of x), so source chunk c feeds
// output chunk oc = c ^ (xr >> LRC): the consumers take the chunks of a load in arrival order and branch
// (uniformly) to the code that owns the accumulator registers of chunk oc.
//
// Per (amplitude, term): one LDS.128 at [thread register + warp-uniform offset] and two FMAs (the coefficient is exactly
// real or exactly imaginary: c = J s^4 times 1, -1, i, -i).  The sign is popcount((base | element) & z) once per
// (term, chunk) and thread; over the 16 slices of a chunk it is a Walsh function of the slice number, walked in groups of
// four: one XOR per group, and inside a group the signs are compile-time FMA operand negations of a kernel variant chosen
// by a uniform branch on the two low slice bits of z (accumulate_chunk).  Per-term data comes from the __grid_constant__
// table (constant bank), the next entry fetched one term ahead.  No atomics on data, one write per output: bitwise
// reproducible.  ~100 warp instructions per (term, chunk of 16 slices) instead of ~150 with a per-slice sign walk; what
// the launch is bound by is the shared-memory data path (every term reads the staged tile once, every load fills it once:
// 134 B/clk/SM at N = 56; syk_apply_H_trace, profiles/r2_chunk_trace.md), plus waits for the loads that miss in L2 (a
// staggered start of the CTAs -- each walks the list rotated by a few places -- spreads the misses: -6 % at N = 64; L2
// prefetching by the TMA unit or by prefetch.global.L2, of every load or only of the loads that must miss, 1..12 loads
// ahead, made every configuration slower: DESIGN.md section 6).
//
// Fused Lanczos epilogue (a-3 part 1) as in apply_h.cu: out = acc/|u_j| - (|u_j|/|u_{j-1}|) prev, per-CTA fp64
// partial sums of Re<in|out>.  The tile of `in` and of `prev` are staged through the same ring after the last
// source tile (their DRAM latency would otherwise be exposed once per tile: measured 50 ms of 385 ms at N = 64).
//
// Measured peaks of this box (syk_microbench, profiles/r2_measured_onchip_peaks.md): L2 -> SM 88 B/clk/SM (25 TB/s),
// DRAM -> SM 7.2-7.5 TB/s, LDS 125 B/clk/SM; the headline launches run at 12-13 TB/s of L2 -> SM traffic.
#include <algorithm>
#include <atomic>
#include <cstring>
#include <new>
#include <type_traits>
#include <vector>

#include "device_utils.cuh"

namespace syk {

namespace {

constexpr int kConsumerWarps = 8;
constexpr int kConsumerThreads = kConsumerWarps * 32;
// Two consumer warpgroups + one producer warpgroup (only its first warp works).  The kernel is launched with
// 65536 / 384 = 168 registers per thread; the consumers then take 232 and the producer warpgroup drops to 40
// (setmaxnreg, per warpgroup): 2 x 232 + 40 <= 512 registers per lane on every SM sub-partition.
constexpr int kThreads = kConsumerThreads + 128;
constexpr int kConsumerRegs = 232, kProducerRegs = 40;
constexpr int kRun = 8;                            // consecutive slices per bulk copy (r bits 0..2 = index bits 8..10)
constexpr int kMaxRing = 16;
constexpr int kSmemLimit = 232448;                 // 227 KiB opt-in maximum per CTA on sm_100
constexpr int kMiscBytes = 2 * kMaxRing * 8 + 40 * 8 + 128;
constexpr uint32_t kRingAlign = 4096;              // alignment of the ring inside the shared window
constexpr int kWindowBits = 7;                     // ~log2(148 tiles in flight)
constexpr int kStagger = 8;                        // spread of the per-CTA rotation of the load list, in loads
constexpr int kFixedR = 3;                         // r bits 0..2 sit at index bits 8..10: a chunk is one contiguous run

template <typename T>
struct StParams {
    using C = typename Cx<T>::type;
    const C* in;
    C* out;
    const C* prev;
    LanczosScalars* sc;
    int j;
    int nring;
    uint32_t* sync;   // lock-step counters (device_utils.cuh lockstep_gate); nullptr = free running
    int epoch_len;
    int lag;
    int stagger;      // CTA i walks the load list of its tiles rotated by (37 i) mod stagger places (0 = all in phase)
    // diagnostic timeline (syk_apply_H_trace; nullptr otherwise): CTA trace_cta records, for its trace_round-th tile, seven
    // clock64 stamps per ring chunk v = list position * NC + chunk (n = n_loads * NC): [v] producer issue; thread 0 of the
    // consumers: [n + v] before the wait for the chunk, [2 n + v] after it, [3 n + v] first term decoded (its LDS stream is
    // next), [4 n + v] first term issued, [5 n + v] all terms issued, [6 n + v] arrived on the empty-barrier
    unsigned long long* trace;
    int trace_cta, trace_round;
};


__device__ __forceinline__ void st_fused_scalars(LanczosScalars* sc, int j, double* red, double& s_in, double& s_prev) {
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

__device__ __forceinline__ double st_fma(double a, double b, double c) { return __fma_rn(a, b, c); }
__device__ __forceinline__ float st_fma(float a, float b, float c) { return __fmaf_rn(a, b, c); }

// A consumer thread owns one 16-byte ELEMENT per slice: one complex128 amplitude, or a pair of adjacent complex64
// amplitudes (index bit 0) -- so both precisions move 16 bytes per LDS and a slice is 4 KiB.  PAIR amplitudes per
// element, TB index bits inside a slice.
template <typename T> struct El;
template <> struct El<double> { static constexpr int PAIR = 1, TB = 8; };
template <> struct El<float> { static constexpr int PAIR = 2, TB = 9; };
constexpr uint32_t kSliceBytes = kConsumerThreads * 16;

__device__ __forceinline__ double2 lds_el(uint32_t addr, double) {
    double2 v;
    asm volatile("ld.shared.v2.f64 {%0, %1}, [%2];" : "=d"(v.x), "=d"(v.y) : "r"(addr));
    return v;
}
__device__ __forceinline__ float4 lds_el(uint32_t addr, float) {
    float4 v;
    asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(addr));
    return v;
}

// One term applied to the RC slices of output chunk OC.  `pb` = shared-memory address of the thread's element in slice 0
// of the staged source chunk; `w` = sign-carrying word of the coefficient times the sign of (thread, tile, chunk, term).
// The slices are taken in groups of four, rl = 4 g + j: the sign of slice rl relative to `w` is
// (-1)^(popcount(g & zg) + popcount(j & ZJ)) with zg / ZJ the upper / lower two bits of the term's Z-mask on the slice
// bits of a chunk.  ZJ is a template parameter -- the caller branches on it (uniformly) -- so inside a group the four
// signs are compile-time negations of one coefficient register pair (FMA operand modifiers: no instruction), and only the
// group sign costs an XOR.  Source addresses are pb + a warp-uniform offset ((rl ^ xr_lo) slices).  complex64: `aux` =
// (z & 1) << 31, the relative sign of the second amplitude of the pair; SWAP = the mask flips index bit 0 (the pair arrives
// swapped).  Per slice: one LDS.128 and two FP64 (four FP32) FMAs.
template <typename T, int R, int RC, int OC, bool IMAG, bool SWAP, int ZJ>
__device__ __forceinline__ void accumulate_chunk(uint32_t pb, uint32_t xr_lo, uint32_t zg, uint32_t aux, uint32_t w,
                                                 T (&ar)[R * El<T>::PAIR], T (&ai)[R * El<T>::PAIR]) {
    static_assert(RC % 4 == 0, "slices of a chunk are walked in groups of four");
    constexpr int r0 = OC * RC;
#pragma unroll
    for (int g = 0; g < RC / 4; ++g) {
        // sign of the group: parity of (g & zg); g is a compile-time constant of the unrolled loop
        uint32_t wg = w;
        if (g & 1) wg ^= zg << 31;                  // bit 0 of zg -> bit 31
        if (g & 2) wg ^= (zg << 30) & 0x80000000u;  // bit 1 of zg -> bit 31
        if constexpr (sizeof(T) == 8) {
            const double a = __hiloint2double((int)wg, (int)aux);   // aux = low word of the coefficient
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                constexpr int dummy = 0;
                (void)dummy;
                const int rl = 4 * g + j;
                const bool neg = (__builtin_popcount(j & ZJ) & 1) != 0;
                const double2 v = lds_el(pb + (((uint32_t)rl ^ xr_lo) * kSliceBytes), double());
                const double aj = neg ? -a : a;
                if constexpr (IMAG) {   // (i a)(vx + i vy) = -a vy + i a vx
                    ar[r0 + rl] = st_fma(-aj, v.y, ar[r0 + rl]);
                    ai[r0 + rl] = st_fma(aj, v.x, ai[r0 + rl]);
                } else {
                    ar[r0 + rl] = st_fma(aj, v.x, ar[r0 + rl]);
                    ai[r0 + rl] = st_fma(aj, v.y, ai[r0 + rl]);
                }
            }
        } else {
            const float a0 = __uint_as_float(wg), a1 = __uint_as_float(wg ^ aux);
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                const int rl = 4 * g + j;
                const bool neg = (__builtin_popcount(j & ZJ) & 1) != 0;
                const float4 v = lds_el(pb + (((uint32_t)rl ^ xr_lo) * kSliceBytes), float());
                const float b0 = neg ? -a0 : a0, b1 = neg ? -a1 : a1;
                const float s0x = SWAP ? v.z : v.x, s0y = SWAP ? v.w : v.y, s1x = SWAP ? v.x : v.z, s1y = SWAP ? v.y : v.w;
                const int k0 = 2 * (r0 + rl), k1 = k0 + 1;
                if constexpr (IMAG) {
                    ar[k0] = st_fma(-b0, s0y, ar[k0]);
                    ai[k0] = st_fma(b0, s0x, ai[k0]);
                    ar[k1] = st_fma(-b1, s1y, ar[k1]);
                    ai[k1] = st_fma(b1, s1x, ai[k1]);
                } else {
                    ar[k0] = st_fma(b0, s0x, ar[k0]);
                    ai[k0] = st_fma(b0, s0y, ai[k0]);
                    ar[k1] = st_fma(b1, s1x, ar[k1]);
                    ai[k1] = st_fma(b1, s1y, ai[k1]);
                }
            }
        }
    }
}

// Uniform branch to the instantiation for (variant, output chunk): variant = ZJ | IMAG << 2 | SWAP << 3.
template <typename T, int R, int RC, int OC, int V>
__device__ __forceinline__ void dispatch_variant(uint32_t variant, uint32_t pb, uint32_t xr_lo, uint32_t zg, uint32_t aux,
                                                 uint32_t w, T (&ar)[R * El<T>::PAIR], T (&ai)[R * El<T>::PAIR]) {
    constexpr int NV = sizeof(T) == 8 ? 8 : 16;
    if constexpr (V + 1 == NV) {
        accumulate_chunk<T, R, RC, OC, (V & 4) != 0, (V & 8) != 0, V & 3>(pb, xr_lo, zg, aux, w, ar, ai);
    } else {
        if (variant == (uint32_t)V) accumulate_chunk<T, R, RC, OC, (V & 4) != 0, (V & 8) != 0, V & 3>(pb, xr_lo, zg, aux, w, ar, ai);
        else dispatch_variant<T, R, RC, OC, V + 1>(variant, pb, xr_lo, zg, aux, w, ar, ai);
    }
}

template <typename T, int R, int RC, int OC>
__device__ __forceinline__ void dispatch_chunk(uint32_t oc, uint32_t variant, uint32_t pb, uint32_t xr_lo, uint32_t zg,
                                               uint32_t aux, uint32_t w, T (&ar)[R * El<T>::PAIR],
                                               T (&ai)[R * El<T>::PAIR]) {
    if constexpr (OC + 1 == R / RC) {
        dispatch_variant<T, R, RC, OC, 0>(variant, pb, xr_lo, zg, aux, w, ar, ai);
    } else {
        if (oc == (uint32_t)OC) dispatch_variant<T, R, RC, OC, 0>(variant, pb, xr_lo, zg, aux, w, ar, ai);
        else dispatch_chunk<T, R, RC, OC + 1>(oc, variant, pb, xr_lo, zg, aux, w, ar, ai);
    }
}

template <typename T, int NR, int LRC, bool FUSED, int TRACE = 0>   // TRACE: 0 off, 1 three stamps per chunk, 2 seven
__global__ void __launch_bounds__(kThreads, 1)
apply_h_scatter_kernel(const __grid_constant__ StTable tab, const StParams<T> p) {
    using C = typename Cx<T>::type;
    constexpr int R = 1 << NR;
    constexpr int RC = 1 << LRC;                                  // slices per ring chunk
    constexpr int NC = R / RC;                                    // chunks per tile
    constexpr uint32_t SLICE_BYTES = kSliceBytes;                 // 256 elements of 16 bytes
    constexpr int PAIR = El<T>::PAIR, TB = El<T>::TB;
    constexpr uint32_t RUN_BYTES = kRun * SLICE_BYTES;
    constexpr uint32_t CHUNK_BYTES = RC * SLICE_BYTES;
    static_assert(R % RC == 0 && RC % kRun == 0 && LRC >= kFixedR, "tile = whole chunks = whole runs");

    extern __shared__ __align__(128) unsigned char smem_raw[];
    // the ring starts on a 4 KiB boundary of the shared window: a consumer's element address inside a staged slice is then
    // chunk address | (tid ^ xt) * 16 -- one XOR with a warp-uniform value, no carry into the slice bits
    unsigned char* smem = smem_raw + ((kRingAlign - (smem_u32(smem_raw) & (kRingAlign - 1u))) & (kRingAlign - 1u));
    unsigned char* q = smem + (size_t)p.nring * CHUNK_BYTES;
    uint64_t* bars = reinterpret_cast<uint64_t*>(q);
    q += 2 * kMaxRing * 8;
    double* red = reinterpret_cast<double*>(q);

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const uint32_t bar_full = smem_u32(bars), bar_empty = smem_u32(bars + kMaxRing);
    if (tid == 0) {
        for (int s = 0; s < p.nring; ++s) {
            mbar_init(bar_full + 8 * s, 1);
            mbar_init(bar_empty + 8 * s, kConsumerWarps);
        }
        mbar_fence_init();
    }
    __syncthreads();

    double s_in = 1.0, s_prev = 0.0;
    if (FUSED) st_fused_scalars(p.sc, p.j, red, s_in, s_prev);

    const uint32_t n_tiles = 1u << tab.n_outer;
    const int nring = p.nring, n_loads = tab.n_loads, n_outer = tab.n_outer;
    // Staggered start (round 2): the CTAs walk the same load list in lock step, so the loads that must come from DRAM (the
    // first of each run of masks that agree outside tile + window bits) would reach all of them at once.  Rotating the list
    // by a few places per CTA spreads those misses over time while every tile is still re-read within a few loads of its
    // first use (measured: -6 % at N = 64, neutral at N = 56; rotations beyond ~12 places lose the L2 reuse).  The order in
    // which the terms of an output are added then depends on the CTA that owns its tile: results are reproducible for a
    // given grid size, and equal across kernels only to rounding.
    const int rot = p.stagger > 0 ? (int)((blockIdx.x * 37u) % (uint32_t)p.stagger) % n_loads : 0;
    double dot = 0.0;

    if (warp >= kConsumerWarps) {
        asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(kProducerRegs));
        if (warp != kConsumerWarps || lane != 0) return;
        // ---------------- producer: one lane streams the chunks (8 consecutive slices = one bulk copy) ----------
        int pos = 0;
        uint32_t phase = 0;
        const uint32_t stage0 = smem_u32(smem);
        uint32_t g = 0, until_epoch = 0;   // loads issued; loads left in the current epoch
        for (uint32_t tile = blockIdx.x; tile < n_tiles; tile += gridDim.x) {
            uint32_t base = 0;
            for (int i = 0; i < n_outer; ++i) base |= ((tile >> i) & 1u) << tab.outer_pos[i];
            const bool tr = TRACE != 0 && p.trace && (int)blockIdx.x == p.trace_cta && (int)(tile / gridDim.x) == p.trace_round;
            for (int li = 0; li < n_loads; ++li) {
                int l = li + rot;
                if (l >= n_loads) l -= n_loads;
                if (p.sync) {
                    if (until_epoch == 0) {
                        lockstep_gate(p.sync, g / (uint32_t)p.epoch_len, (uint32_t)p.lag);
                        until_epoch = (uint32_t)p.epoch_len;
                    }
                    --until_epoch;
                    ++g;
                }
                const uint32_t src = base ^ tab.load_xo[l];
#pragma unroll
                for (int c = 0; c < NC; ++c) {
                    mbar_wait(bar_empty + 8 * pos, phase ^ 1u);
                    if constexpr (TRACE != 0) if (tr) p.trace[li * NC + c] = clock64();
                    mbar_arrive_expect_tx(bar_full + 8 * pos, CHUNK_BYTES);
#pragma unroll
                    for (int u = 0; u < RC / kRun; ++u)
                        bulk_load(stage0 + (uint32_t)pos * CHUNK_BYTES + (uint32_t)u * RUN_BYTES,
                                  p.in + (uint64_t)(src | tab.dep_r[c * RC + u * kRun]), RUN_BYTES, bar_full + 8 * pos);
                    if (++pos == nring) {
                        pos = 0;
                        phase ^= 1u;
                    }
                }
            }
            if (FUSED) {
                // operands of the fused epilogue, staged like source tiles so that their latency is hidden:
                // chunk c of in's own tile, then chunk c of prev's
#pragma unroll
                for (int c = 0; c < NC; ++c) {
                    for (int which = 0; which < (p.prev ? 2 : 1); ++which) {
                        const C* from = which ? p.prev : p.in;
                        mbar_wait(bar_empty + 8 * pos, phase ^ 1u);
                        mbar_arrive_expect_tx(bar_full + 8 * pos, CHUNK_BYTES);
#pragma unroll
                        for (int u = 0; u < RC / kRun; ++u)
                            bulk_load(stage0 + (uint32_t)pos * CHUNK_BYTES + (uint32_t)u * RUN_BYTES,
                                      from + (uint64_t)(base | tab.dep_r[c * RC + u * kRun]), RUN_BYTES,
                                      bar_full + 8 * pos);
                        if (++pos == nring) {
                            pos = 0;
                            phase ^= 1u;
                        }
                    }
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
    } else {
        // ---------------- consumers ----------------
        asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(kConsumerRegs));
        int pos = 0;
        uint32_t phase = 0;
        for (uint32_t tile = blockIdx.x; tile < n_tiles; tile += gridDim.x) {
            uint32_t base = 0;
            for (int i = 0; i < n_outer; ++i) base |= ((tile >> i) & 1u) << tab.outer_pos[i];
            const uint32_t bt = base | ((uint32_t)tid << (TB - 8));   // index of the element's first amplitude, r bits 0
            const uint32_t stage_base = smem_u32(smem), tid16 = (uint32_t)tid << 4;
            const bool tr = TRACE != 0 && p.trace && tid == 0 && (int)blockIdx.x == p.trace_cta && (int)(tile / gridDim.x) == p.trace_round;
            T ar[R * PAIR], ai[R * PAIR];
#pragma unroll
            for (int r = 0; r < R * PAIR; ++r) {
                ar[r] = 0;
                ai[r] = 0;
            }
            for (int li = 0; li < n_loads; ++li) {
                int l = li + rot;
                if (l >= n_loads) l -= n_loads;
                const int t0 = tab.load_t0[l], t1 = tab.load_t0[l + 1];
                for (uint32_t c = 0; c < (uint32_t)NC; ++c) {
                    if constexpr (TRACE != 0) if (tr) p.trace[(n_loads + li) * NC + c] = clock64();
                    mbar_wait(bar_full + 8 * pos, phase);
                    if constexpr (TRACE != 0) if (tr) p.trace[(2 * n_loads + li) * NC + c] = clock64();
                    const uint32_t cp = stage_base + (uint32_t)pos * CHUNK_BYTES + tid16;
                    uint4 e = tab.term[t0];
                    for (int t = t0; t < t1; ++t) {
                        const uint4 en = tab.term[t + 1 < t1 ? t + 1 : t];   // next entry: its constant-bank latency is hidden
                        // e.x: bits 0..8 in-slice bits of x | 9..13 r bits of x | 16..20 r bits of z | 31 imaginary coefficient
                        const uint32_t xr = (e.x >> 9) & 31u, zr = (e.x >> 16) & 31u;
                        const uint32_t oc = c ^ (xr >> LRC);
                        const uint32_t pb = cp ^ (((e.x & 511u) >> (TB - 8)) << 4);   // (tid ^ xt) * 16: bits 4..11 only
                        const uint32_t sgn = ((uint32_t)__popc(bt & e.y) + (uint32_t)__popc((oc << LRC) & zr)) << 31;
                        const uint32_t w = (sizeof(T) == 8 ? e.w : e.z) ^ sgn;
                        constexpr uint32_t lo = (uint32_t)RC - 1u;
                        uint32_t variant = (zr & 3u) | ((e.x >> 31) << 2);
                        uint32_t aux = e.z;
                        if constexpr (sizeof(T) == 4) {
                            variant |= (e.x & 1u) << 3;            // the mask flips index bit 0: the pair arrives swapped
                            aux = (e.y & 1u) << 31;                // second amplitude of the pair: index bit 0 set
                        }
                        if constexpr (TRACE == 2) if (tr && t == t0) p.trace[(3 * n_loads + li) * NC + c] = clock64();
                        dispatch_chunk<T, R, RC, 0>(oc, variant, pb, xr & lo, (zr & lo) >> 2, aux, w, ar, ai);
                        if constexpr (TRACE == 2) if (tr && t == t0) p.trace[(4 * n_loads + li) * NC + c] = clock64();
                        e = en;
                    }
                    if constexpr (TRACE == 2) if (tr) p.trace[(5 * n_loads + li) * NC + c] = clock64();
                    __syncwarp();
                    if (lane == 0) mbar_arrive(bar_empty + 8 * pos);
                    if constexpr (TRACE == 2) if (tr) p.trace[(6 * n_loads + li) * NC + c] = clock64();
                    if (++pos == nring) {
                        pos = 0;
                        phase ^= 1u;
                    }
                }
            }
            // epilogue: slice r of the tile is 256 consecutive elements; one 16-byte store per thread and slice
            using E = typename std::conditional<sizeof(T) == 8, double2, float4>::type;
            auto emit = [&](int r, const E* mine_p, const E* prev_p) {
                const uint64_t b = (uint64_t)(bt | tab.dep_r[r]);
                E o;
                if constexpr (sizeof(T) == 8) {
                    if constexpr (FUSED) {
                        const E mine = *mine_p;
                        double orr = ar[r] * s_in, oi = ai[r] * s_in;
                        if (prev_p) {
                            const E pv = *prev_p;
                            orr -= s_prev * pv.x;
                            oi -= s_prev * pv.y;
                        }
                        o.x = orr;
                        o.y = oi;
                        dot += mine.x * o.x + mine.y * o.y;
                    } else {
                        o.x = ar[r];
                        o.y = ai[r];
                    }
                } else {
                    if constexpr (FUSED) {
                        const E mine = *mine_p;
                        double o0r = (double)ar[2 * r] * s_in, o0i = (double)ai[2 * r] * s_in;
                        double o1r = (double)ar[2 * r + 1] * s_in, o1i = (double)ai[2 * r + 1] * s_in;
                        if (prev_p) {
                            const E pv = *prev_p;
                            o0r -= s_prev * (double)pv.x;
                            o0i -= s_prev * (double)pv.y;
                            o1r -= s_prev * (double)pv.z;
                            o1i -= s_prev * (double)pv.w;
                        }
                        o.x = (float)o0r;
                        o.y = (float)o0i;
                        o.z = (float)o1r;
                        o.w = (float)o1i;
                        dot += (double)mine.x * (double)o.x + (double)mine.y * (double)o.y +
                               (double)mine.z * (double)o.z + (double)mine.w * (double)o.w;
                    } else {
                        o.x = ar[2 * r];
                        o.y = ai[2 * r];
                        o.z = ar[2 * r + 1];
                        o.w = ai[2 * r + 1];
                    }
                }
                *reinterpret_cast<E*>(p.out + b) = o;
            };
            if constexpr (FUSED) {
#pragma unroll
                for (int c = 0; c < NC; ++c) {
                    mbar_wait(bar_full + 8 * pos, phase);
                    const E* mine_s = reinterpret_cast<const E*>(smem + (size_t)pos * CHUNK_BYTES) + tid;
                    const int pos_in = pos;
                    if (++pos == nring) {
                        pos = 0;
                        phase ^= 1u;
                    }
                    const E* prev_s = nullptr;
                    int pos_prev = 0;
                    if (p.prev) {
                        mbar_wait(bar_full + 8 * pos, phase);
                        prev_s = reinterpret_cast<const E*>(smem + (size_t)pos * CHUNK_BYTES) + tid;
                        pos_prev = pos;
                        if (++pos == nring) {
                            pos = 0;
                            phase ^= 1u;
                        }
                    }
#pragma unroll
                    for (int rl = 0; rl < RC; ++rl)
                        emit(c * RC + rl, mine_s + rl * kConsumerThreads, prev_s ? prev_s + rl * kConsumerThreads : nullptr);
                    __syncwarp();
                    if (lane == 0) {
                        mbar_arrive(bar_empty + 8 * pos_in);
                        if (prev_s) mbar_arrive(bar_empty + 8 * pos_prev);
                    }
                }
            } else {
#pragma unroll
                for (int r = 0; r < R; ++r) emit(r, nullptr, nullptr);
            }
        }
        if (FUSED) {
            // fixed-order sum over the 256 consumer threads (named barrier 1: the producer warpgroup has left)
            dot = warp_sum(dot);
            if (lane == 0) red[warp] = dot;
            asm volatile("bar.sync 1, %0;" ::"n"(kConsumerThreads) : "memory");
            if (warp == 0) {
                double s = lane < kConsumerWarps ? red[lane] : 0.0;
                s = warp_sum(s);
                if (lane == 0) {
                    p.sc->partial_dot[blockIdx.x] = s;
                    if (blockIdx.x == 0) p.sc->n_partial_dot = gridDim.x;
                }
            }
        }
    }
}

// Per dtype index (SYK_C64 = 0, SYK_C128 = 1): index bits inside a slice (a complex64 element is a pair of amplitudes),
// NR = log2 slices per tile, LRC = log2 slices per ring chunk: 128 KiB tiles in two 64 KiB chunks for both
constexpr int kStTB[2] = {9, 8};
constexpr int kStNR[2] = {5, 5};
constexpr int kStLRC[2] = {4, 4};

uint32_t extract_bits(uint32_t v, const int* pos, int n) {
    uint32_t r = 0;
    for (int i = 0; i < n; ++i) r |= ((v >> pos[i]) & 1u) << i;
    return r;
}
uint32_t deposit_bits(uint32_t v, const int* pos, int n) {
    uint32_t r = 0;
    for (int i = 0; i < n; ++i) r |= ((v >> i) & 1u) << pos[i];
    return r;
}

struct LayoutCost {
    int loads, passes;
    int total() const { return loads + 2 * passes; }
};

// #loads = distinct x outside the tile bits; #passes = distinct x outside tile + window bits.  seq = the free
// positions (index bits >= 11): seq[0..nr) are the free r bits, seq[nr..nr+kWindowBits) the window bits.
LayoutCost layout_cost(const std::vector<uint32_t>& xs, const std::vector<int>& seq, int nr, std::vector<uint32_t>& tmp,
                       int tb) {
    uint32_t tile = (1u << (tb + kFixedR)) - 1u;
    for (int i = 0; i < nr; ++i) tile |= 1u << seq[i];
    uint32_t win = tile;
    for (int i = nr; i < nr + kWindowBits && i < (int)seq.size(); ++i) win |= 1u << seq[i];
    LayoutCost c;
    tmp.resize(xs.size());
    for (size_t i = 0; i < xs.size(); ++i) tmp[i] = xs[i] & ~tile;
    std::sort(tmp.begin(), tmp.end());
    c.loads = (int)(std::unique(tmp.begin(), tmp.end()) - tmp.begin());
    for (size_t i = 0; i < xs.size(); ++i) tmp[i] = xs[i] & ~win;
    std::sort(tmp.begin(), tmp.end());
    c.passes = (int)(std::unique(tmp.begin(), tmp.end()) - tmp.begin());
    return c;
}

// Deterministic first-improvement hill climbing over swaps that move a bit between the classes r / window / rest,
// started from the identity layout (free r bits = 11.., window = the next 7).  nr = number of FREE r bits.
void choose_layout(const std::vector<uint32_t>& xs, int L, int nr, std::vector<int>& seq, int tb) {
    seq.clear();
    for (int q = tb + kFixedR; q < L; ++q) seq.push_back(q);
    const int n = (int)seq.size();
    const int nw = std::min(kWindowBits, n - nr);
    std::vector<uint32_t> tmp;
    int cur = layout_cost(xs, seq, nr, tmp, tb).total();
    auto cls = [&](int i) { return i < nr ? 0 : (i < nr + nw ? 1 : 2); };
    for (int sweep = 0; sweep < 16; ++sweep) {
        bool improved = false;
        for (int i = 0; i < nr + nw; ++i)
            for (int j = i + 1; j < n; ++j) {
                if (cls(i) == cls(j)) continue;
                std::swap(seq[i], seq[j]);
                const int c = layout_cost(xs, seq, nr, tmp, tb).total();
                if (c < cur) {
                    cur = c;
                    improved = true;
                } else {
                    std::swap(seq[i], seq[j]);
                }
            }
        if (!improved) break;
    }
    // canonical order inside each class (the cost does not depend on it): ascending bit positions
    std::sort(seq.begin(), seq.begin() + nr);
    std::sort(seq.begin() + nr, seq.begin() + nr + nw);
    std::sort(seq.begin() + nr + nw, seq.end());
}

bool build_st_table(const syk_ham* h, int dtype, StTable& tab) {
    const int k = dtype == SYK_C128 ? 1 : 0;
    const int nr = kStNR[k], tb = kStTB[k];
    const size_t nt = h->z.size();
    if (nt == 0 || nt > (size_t)kStMaxTerms || h->L < tb + nr) return false;
    std::vector<uint32_t> xs;
    for (size_t g = 0; g < h->x.size(); ++g) xs.push_back((uint32_t)h->x[g]);
    std::vector<int> seq;
    choose_layout(xs, h->L, nr - kFixedR, seq, tb);
    const int n_outer = h->L - tb - nr;
    std::vector<int> pvec;
    for (int i = 0; i < kFixedR; ++i) pvec.push_back(tb + i);
    for (int i = 0; i < nr - kFixedR; ++i) pvec.push_back(seq[i]);
    const int* P = pvec.data();
    const int* O = seq.data() + (nr - kFixedR);
    uint32_t omask = 0;
    for (int i = 0; i < n_outer; ++i) omask |= 1u << O[i];

    struct Item { uint32_t key, xo; uint32_t order; uint4 e; };
    std::vector<Item> items;
    items.reserve(nt);
    for (size_t g = 0; g < h->x.size(); ++g) {
        const uint32_t x = (uint32_t)h->x[g];
        for (uint32_t t = h->group_off[g]; t < h->group_off[g + 1]; ++t) {
            const std::complex<double> c = h->c[t];
            const bool imag = c.imag() != 0.0;
            if (imag && c.real() != 0.0) return false;   // never for SYK strings (c = J s^4 {1,-1,i,-i})
            const double a = imag ? c.imag() : c.real();
            const uint32_t z = (uint32_t)h->z[t];
            Item it;
            it.key = extract_bits(x, O, n_outer);
            it.xo = x & omask;
            it.order = (uint32_t)items.size();
            it.e.x = (x & ((1u << tb) - 1u)) | (extract_bits(x, P, nr) << 9) | (extract_bits(z, P, nr) << 16) |
                     (imag ? 0x80000000u : 0u);
            it.e.y = z;
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
    std::sort(items.begin(), items.end(), [](const Item& a, const Item& b) {
        return a.key != b.key ? a.key < b.key : a.order < b.order;
    });
    int n_loads = 0;
    for (size_t i = 0; i < items.size(); ++i) {
        if (i == 0 || items[i].key != items[i - 1].key) {
            if (n_loads >= kStMaxLoads) return false;
            tab.load_xo[n_loads] = items[i].xo;
            tab.load_t0[n_loads] = (uint16_t)i;
            ++n_loads;
        }
        tab.term[i] = items[i].e;
    }
    tab.load_t0[n_loads] = (uint16_t)items.size();
    tab.n_loads = n_loads;
    tab.n_outer = n_outer;
    tab.nr = nr;
    for (int s = 0; s < 64; ++s) tab.dep_r[s] = s < (1 << nr) ? deposit_bits((uint32_t)s, P, nr) : 0u;
    for (int i = 0; i < 32; ++i) tab.outer_pos[i] = i < n_outer ? (uint8_t)O[i] : 0;
    uint32_t tile = (1u << tb) - 1u;
    for (int i = 0; i < nr; ++i) tile |= 1u << P[i];
    tab.tile_mask = tile;
    return true;
}

const StTable* get_st_table(const syk_ham* h, int dtype) {
    const int k = dtype == SYK_C128 ? 1 : 0;
    if (!h->st[k]) h->st[k] = new (std::nothrow) StCache();
    if (!h->st[k]) return nullptr;
    if (!h->st[k]->valid) {
        if (!build_st_table(h, dtype, h->st[k]->tab)) return nullptr;
        h->st[k]->valid = true;
    }
    return &h->st[k]->tab;
}

template <typename T, int NR, int LRC>
int launch_st(const syk_ham* h, const StTable& tab, const void* d_in, void* d_out, const FusedArgs& fa,
              cudaStream_t stream) {
    using C = typename Cx<T>::type;
    constexpr size_t kChunkBytes = ((size_t)1 << LRC) * kSliceBytes;
    StParams<T> p;
    p.in = (const C*)d_in;
    p.out = (C*)d_out;
    p.prev = (const C*)fa.prev;
    p.sc = fa.sc;
    p.j = fa.j;
    p.nring = (int)((kSmemLimit - kMiscBytes - kRingAlign) / kChunkBytes);
    if (p.nring > kMaxRing) p.nring = kMaxRing;
    const size_t smem = (size_t)p.nring * kChunkBytes + kMiscBytes + kRingAlign;
    const int sms = num_sms();
    if (sms <= 0) return SYK_ECUDA;
    const uint64_t n_tiles = 1ull << tab.n_outer;
    const int grid = (int)(n_tiles < (uint64_t)sms ? n_tiles : (uint64_t)sms);
    // lock-step only where it pays: the vector does not fit in L2 and there are several rounds of tiles
    int epoch_len = 0, lag = 0;
    get_lockstep(&epoch_len, &lag);
    p.trace = fa.trace;
    p.trace_cta = fa.trace_cta;
    p.trace_round = fa.trace_round;
    p.sync = nullptr;
    p.epoch_len = epoch_len;
    p.lag = lag;
    p.stagger = (((uint64_t)sizeof(C) << h->L) > ((uint64_t)64 << 20) && n_tiles >= 4 * (uint64_t)grid && tab.n_loads >= 2 * kStagger)
                    ? kStagger : 0;
    if (epoch_len > 0 && ((uint64_t)sizeof(C) << h->L) > ((uint64_t)64 << 20) && n_tiles >= 4 * (uint64_t)grid) {
        p.sync = h->dev.sync;
        SYK_CUDA(cudaMemsetAsync(p.sync, 0, kSyncRing * sizeof(uint32_t), stream));
    }
    if (fa.sc) {
        SYK_CUDA(cudaFuncSetAttribute(apply_h_scatter_kernel<T, NR, LRC, true>,
                                      cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        apply_h_scatter_kernel<T, NR, LRC, true><<<grid, kThreads, smem, stream>>>(tab, p);
    } else if (fa.trace && fa.trace_detail) {   // diagnostic builds of the plain kernel (syk_apply_H_trace): clock stamps per ring chunk
        SYK_CUDA(cudaFuncSetAttribute(apply_h_scatter_kernel<T, NR, LRC, false, 2>,
                                      cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        apply_h_scatter_kernel<T, NR, LRC, false, 2><<<grid, kThreads, smem, stream>>>(tab, p);
    } else if (fa.trace) {
        SYK_CUDA(cudaFuncSetAttribute(apply_h_scatter_kernel<T, NR, LRC, false, 1>,
                                      cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        apply_h_scatter_kernel<T, NR, LRC, false, 1><<<grid, kThreads, smem, stream>>>(tab, p);
    } else {
        SYK_CUDA(cudaFuncSetAttribute(apply_h_scatter_kernel<T, NR, LRC, false>,
                                      cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        apply_h_scatter_kernel<T, NR, LRC, false><<<grid, kThreads, smem, stream>>>(tab, p);
    }
    count_launch();
    SYK_CUDA(cudaGetLastError());
    return SYK_OK;
}

}  // namespace

// 0 if the handle cannot use the kernel, else log2 of its tile size in amplitudes
int scatter_tile_log2(const syk_ham* h, int dtype, bool forced) {
    const int k = dtype == SYK_C128 ? 1 : 0;
    const int tl = kStTB[k] + kStNR[k];
    if (h->n_terms() == 0 || h->n_terms() > kStMaxTerms || h->L < tl) return 0;
    // automatic choice: at least ~4 rounds of 128 KiB tiles on 148 SMs
    if (!forced && h->L < tl + 10) return 0;
    return get_st_table(h, dtype) ? tl : 0;
}

int launch_apply_h_scatter(const syk_ham* h, int dtype, const void* d_in, void* d_out, const FusedArgs& fa,
                           cudaStream_t stream) {
    const StTable* tab = get_st_table(h, dtype);
    if (!tab) return SYK_EINVAL;
    if (dtype == SYK_C128) return launch_st<double, kStNR[1], kStLRC[1]>(h, *tab, d_in, d_out, fa, stream);
    return launch_st<float, kStNR[0], kStLRC[0]>(h, *tab, d_in, d_out, fa, stream);
}

int scatter_layout_info(const syk_ham* h, int dtype, int* n_loads, int* n_passes, uint32_t* tile_mask, uint32_t* window_mask) {
    const StTable* tab = get_st_table(h, dtype);
    if (!tab) return SYK_EINVAL;
    uint32_t win = tab->tile_mask;
    for (int i = 0; i < kWindowBits && i < tab->n_outer; ++i) win |= 1u << tab->outer_pos[i];
    std::vector<uint32_t> v;
    for (size_t g = 0; g < h->x.size(); ++g) v.push_back((uint32_t)h->x[g] & ~win);
    std::sort(v.begin(), v.end());
    if (n_loads) *n_loads = tab->n_loads;
    if (n_passes) *n_passes = (int)(std::unique(v.begin(), v.end()) - v.begin());
    if (tile_mask) *tile_mask = tab->tile_mask;
    if (window_mask) *window_mask = win;
    return SYK_OK;
}

int scatter_tile_bits(int dtype) {
    const int k = dtype == SYK_C128 ? 1 : 0;
    return kStTB[k] + kStNR[k];
}
int scatter_window_bits() { return kWindowBits; }

// syk_apply_H_trace (include/syk.h): one plain product with the timeline of one CTA and the load list it walked
int scatter_trace(const syk_ham* h, int dtype, const void* d_in, void* d_out, int cta, int round, int detail, uint64_t* clk,
                  int clk_capacity, int32_t* load_terms, uint32_t* load_xo, int load_capacity, int* n_loads, int* rot,
                  cudaStream_t stream) {
    const StTable* tab = get_st_table(h, dtype);
    if (!tab) return SYK_EINVAL;
    const int k = dtype == SYK_C128 ? 1 : 0;
    const int nc = 1 << (kStNR[k] - kStLRC[k]);
    const int n = tab->n_loads * nc;
    const int sms = num_sms();
    if (sms <= 0) return SYK_ECUDA;
    const uint64_t n_tiles = 1ull << tab->n_outer;
    const uint64_t grid = n_tiles < (uint64_t)sms ? n_tiles : (uint64_t)sms;
    if (cta < 0 || (uint64_t)cta >= grid || round < 0 || (uint64_t)round * grid + (uint64_t)cta >= n_tiles ||
        clk_capacity < 7 * n || load_capacity < tab->n_loads)
        return SYK_EINVAL;
    unsigned long long* d_trace = nullptr;
    SYK_CUDA(cudaMalloc(&d_trace, (size_t)7 * n * sizeof(unsigned long long)));
    cudaMemsetAsync(d_trace, 0, (size_t)7 * n * sizeof(unsigned long long), stream);
    FusedArgs fa;
    fa.trace = d_trace;
    fa.trace_cta = cta;
    fa.trace_round = round;
    fa.trace_detail = detail;
    int rc = launch_apply_h_scatter(h, dtype, d_in, d_out, fa, stream);
    if (rc == SYK_OK && cudaMemcpyAsync(clk, d_trace, (size_t)7 * n * sizeof(unsigned long long), cudaMemcpyDeviceToHost,
                                        stream) != cudaSuccess)
        rc = SYK_ECUDA;
    if (cudaStreamSynchronize(stream) != cudaSuccess) rc = SYK_ECUDA;
    cudaFree(d_trace);
    SYK_TRY(rc);
    for (int l = 0; l < tab->n_loads; ++l) {
        load_terms[l] = (int32_t)tab->load_t0[l + 1] - (int32_t)tab->load_t0[l];
        load_xo[l] = tab->load_xo[l];
    }
    *n_loads = tab->n_loads;
    // the rotation launch_st gives this CTA (same conditions)
    const bool big = ((uint64_t)elem_bytes(dtype) << h->L) > ((uint64_t)64 << 20) && n_tiles >= 4 * grid;
    const int stagger = big && tab->n_loads >= 2 * kStagger ? kStagger : 0;
    *rot = stagger > 0 ? (int)(((uint32_t)cta * 37u) % (uint32_t)stagger) % tab->n_loads : 0;
    return SYK_OK;
}

void free_scatter_tables(const syk_ham* h) {
    for (int k = 0; k < 2; ++k) {
        delete h->st[k];
        h->st[k] = nullptr;
    }
}

}  // namespace syk
