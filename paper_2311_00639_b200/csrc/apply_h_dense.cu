// a-2  apply_H, dense-table kernel: the gather form of Algorithm 1 for Hamiltonians with MANY terms
// per X-mask (dense p = 1: T = 194 580 terms on D_x = 10 903 masks at N = 48, 17.8 terms per mask).
//
//     out[b] = sum_g in[b ^ x_g] * S_g(b),      S_g(b) = sum_{t in g} c_t (-1)^popcount(b & z_t)
//
// Here the vector traffic is negligible (a few hundred source tiles per output tile, all L2 hits) and the work is
// the T sign-accumulates per amplitude: plain ALU.  Three things keep that cheap:
//   * the thread owns R = 8 amplitudes  base | tid | r << 9  (r = index bits 9..11), so everything that depends on
//     the term only (table read, popcount of the tile/thread part of the sign) is paid once per 8 amplitudes;
//   * the r-dependence of the sign is a WALSH FUNCTION of r:  (-1)^popcount(r & zr),  zr = bits 9..11 of z.  So the
//     terms of a group are first binned by zr -- one add per TERM into one of 8 registers (terms come sorted by
//     bin, so the register is a compile-time index of an unrolled walk over the bins that occur) -- and
//     S_g(r) for the 8 r is the Walsh-Hadamard transform of the bins: 24 adds per group instead of 8 per term;
//   * c_t is exactly real or exactly imaginary (J s^4 times 1, -1, i, -i): two real bin arrays, no complex adds.
// Then one complex multiply-add per (group, amplitude) with the source read from the staged tile.
//
// Source tiles (2^12 amplitudes: 64 / 32 KiB) come by cp.async.bulk into a double buffer (thread 0 issues the next
// one, mbarrier completion); the table (a few MB, streamed once per output tile) is staged chunk by chunk in shared
// memory by the threads themselves, double buffered, so the inner loops read it with broadcast LDS (read from global
// with warp-uniform addresses, each term cost an exposed L2 latency: 1120 ms per N = 48 matvec).
// Groups whose Z-masks agree outside their own X-mask (every four-qubit X-mask of a dense SYK Hamiltonian) skip the binning
// altogether: one table of 2^popcount(x) coefficient sums per group, one lookup and one complex multiply-add per amplitude
// (local_group below).
// History at N = 48 dense complex128: generic kernel 2390 ms; 8 warps x 16 amplitudes 692 ms; this shape 450 ms; with the
// x-local groups 178 ms (0.24 of the FP64 issue rate: latency-bound, profiles/r2_N48_dense_c128.md).
// No atomics on data, one write per output: bitwise reproducible.  Fused Lanczos epilogue as in apply_h.cu.
#include <algorithm>
#include <cstring>
#include <new>
#include <vector>

#include "device_utils.cuh"

namespace syk {

namespace {

// 16 warps, every thread a consumer (four warps per scheduler hide the dependent chain of a term: table LDS ->
// popcount -> sign -> add; with 8 warps and 16 amplitudes per thread the schedulers were 35 % busy); thread 0 also
// issues the bulk copies -- a source tile is consumed over ~10^5 cycles, so a plain double buffer is enough.
#ifndef SYK_DENSE_RBITS
#define SYK_DENSE_RBITS 3
#endif
// Index bits of a tile inside a thread (amplitudes per thread = 2^kRBits; 2^(12 - kRBits) threads).  Measured at N = 48 dense
// complex128 (plain product): 3 -> 170 ms (16 warps x 8 amplitudes), 2 -> 200 ms (32 warps x 4: twice the warps to hide the
// per-group chain, but twice the per-group instructions per amplitude).
constexpr int kRBits = SYK_DENSE_RBITS;
static_assert(kRBits == 2 || kRBits == 3, "tested shapes: 1024 threads x 4 amplitudes, 512 threads x 8 amplitudes");
constexpr int kThreadBitsD = 12 - kRBits;
constexpr int kConsumerThreads = 1 << kThreadBitsD;
constexpr int kThreads = kConsumerThreads;
constexpr int kR = 1 << kRBits;                              // amplitudes per thread
constexpr int kTileLog2D = 12;                     // 512 threads x 8
constexpr int kTile = 1 << kTileLog2D;
constexpr int kMiscBytes = 2 * 8 + 40 * 8 + 128 + 2 * 512 * 16;   // barriers, reduction scratch, table buffers

// The table is ONE stream of 16-byte entries, cut into chunks of <= kChunkEntries entries that hold whole groups:
//   group header : .x = tile-local X-mask, .y = number of terms that follow, .z = 1 real / 2 imaginary / 3 both,
//                  .w = which of the 16 bins occur
//   term         : .x = Z-mask, .y = bin = zr (bits 9..11 of z) + 8 if the coefficient is imaginary; terms of a
//                  group are sorted by bin and bit 8 of .y marks the last term of a bin,
//                  (.z, .w) = bits of the signed magnitude a (double) or .z = bits of (float) a
// The consumers copy chunk k+1 into shared memory while they work on chunk k (double buffer), so every table read
// in the inner loops is a broadcast LDS instead of a dependent global load.
constexpr int kChunkEntries = 512;
constexpr int kLocalMaxBits = 4;                   // x-local groups: popcount(x) <= 4 (a table of <= 16 values)
constexpr int kLocalMinTerms = 4;                  // ... and at least this many terms (else the per-term walk is cheaper)
struct DenseLoad { uint32_t hi, c0, c1, pad; };    // source tile = tile ^ hi; chunks [c0, c1)
struct DenseChunk { uint32_t e0, ne, pad0, pad1; };// entries [e0, e0 + ne)

template <typename T>
struct DnParams {
    using C = typename Cx<T>::type;
    const C* in;
    C* out;
    const C* prev;
    LanczosScalars* sc;
    int j;
    int L;
    int nslot;
    const DenseLoad* loads;
    const DenseChunk* chunks;
    const uint4* entries;
    int n_loads;
    int n_chunks;
};

__device__ __forceinline__ void dn_fused_scalars(LanczosScalars* sc, int j, double* red, double& s_in, double& s_prev) {
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

__device__ __forceinline__ double dn_fma(double a, double b, double c) { return __fma_rn(a, b, c); }
__device__ __forceinline__ float dn_fma(float a, float b, float c) { return __fmaf_rn(a, b, c); }

// in-place Walsh-Hadamard transform: s[r] = sum_z c[z] (-1)^popcount(r & z)
template <typename T>
__device__ __forceinline__ void wht(T (&c)[kR]) {
#pragma unroll
    for (int h = 1; h < kR; h <<= 1) {
#pragma unroll
        for (int i = 0; i < kR; ++i) {
            if ((i & h) == 0) {
                const T a = c[i], b = c[i | h];
                c[i] = a + b;
                c[i | h] = a - b;
            }
        }
    }
}

// bins B, B+1, ... of one group: for every bin that occurs, add its run of terms (closed by bit 8 of .y) to the register
// that owns it.  `e` always holds entry `t`, loaded one step ahead.
template <typename T, int B>
__device__ __forceinline__ void walk_bins(const uint4* __restrict__ ent, uint32_t& t, uint4& e, uint32_t occ, uint32_t bt,
                                          T (&cr)[kR], T (&ci)[kR]) {
    if constexpr (B < 2 * kR) {
        if (occ & (1u << B)) {
            uint32_t last;
            do {
                const uint32_t sgn = (uint32_t)__popc(bt & e.x) << 31;
                T a;
                if constexpr (sizeof(T) == 8) a = __hiloint2double((int)(e.w ^ sgn), (int)e.z);
                else a = __uint_as_float(e.z ^ sgn);
                if constexpr (B < kR) cr[B] += a;
                else ci[B - kR] += a;
                last = e.y & 256u;
                ++t;
                e = ent[t];   // t <= ne <= kChunkEntries - 1: always inside the buffer; four warps per scheduler hide it
            } while (!last);
        }
        walk_bins<T, B + 1>(ent, t, e, occ, bt, cr, ci);
    }
}

// ---------------------------------------------------------------------------------------------------------
// X-LOCAL groups.  If the Z-masks of a group agree outside the bits of its X-mask x (popcount(x) = k <= 4) -- true for every
// group of a dense SYK Hamiltonian whose x has four bits: its 16 terms are the X / Y choices on the four flipped qubits, the
// Jordan-Wigner strings are common -- then the whole group is ONE function of k bits of b:
//     S_g(b) = (-1)^popcount(b & zb) F[pext(b, x)],   zb = the common part of z outside x,
//     F[i]   = sum_t c_t (-1)^popcount(pdep(i, x) & z_t)                     (2^k complex numbers, summed on the host).
// Per (group, amplitude) that is one table read and one complex multiply-add instead of one sign-accumulate per term: 16 terms
// cost what ~3 cost before.  The table index of the thread's 8 amplitudes differs only through the r bits (index bits 9..11)
// that x contains, XR = (x >> 9) & 7: 2^popcount(XR) table reads per thread (1.6 on average for random x), and the source
// slice r ^ XR is a compile-time offset of the variant the (uniform) switch on XR selects.
// Stream format of such a group: header A {x & (tile - 1), 1 + 2^k, 4, zb}, header B {.x = positions of the bits of x, 5 bits
// each (unused: 9, an r bit, always 0 in the thread's base index), .y = index bit of r bit j in bits 2j..2j+1, .z = Walsh mask
// of zb's r bits}, then F[0 .. 2^k)
// as (re, im) doubles or floats at a 16-byte stride.
// ---------------------------------------------------------------------------------------------------------
template <typename T, int XR>
__device__ __forceinline__ void local_group(const uint4* __restrict__ F, uint32_t idx0, uint32_t mpos, uint32_t W,
                                            const typename Cx<T>::type* pb, T (&ar)[kR], T (&ai)[kR]) {
    using C = typename Cx<T>::type;
    constexpr int ND = 1 << ((XR & 1) + ((XR >> 1) & 1) + ((XR >> 2) & 1));
    static_assert(XR < kR, "XR = the r bits of x");
    T fr[ND], fi[ND];
#pragma unroll
    for (int d = 0; d < ND; ++d) {
        // bits of d go to the index-bit positions of the r bits that x contains (ascending r bit)
        uint32_t delta = 0;
        int dj = 0;
#pragma unroll
        for (int j = 0; j < kRBits; ++j) {
            if (XR & (1 << j)) {
                if (d & (1 << dj)) delta |= 1u << ((mpos >> (2 * j)) & 3u);
                ++dj;
            }
        }
        const uint4 e = F[idx0 ^ delta];
        if constexpr (sizeof(T) == 8) {
            fr[d] = __hiloint2double((int)e.y, (int)e.x);
            fi[d] = __hiloint2double((int)e.w, (int)e.z);
        } else {
            fr[d] = __uint_as_float(e.x);
            fi[d] = __uint_as_float(e.y);
        }
    }
#pragma unroll
    for (int r = 0; r < kR; ++r) {
        // which of the ND table values: the bits of r inside XR, compacted (compile time)
        int d = 0, dj = 0;
#pragma unroll
        for (int j = 0; j < kRBits; ++j) {
            if (XR & (1 << j)) {
                if (r & (1 << j)) d |= 1 << dj;
                ++dj;
            }
        }
        // sign of amplitude r = bit r of W (Walsh function of r for the group's zb, times the thread's own sign), applied to
        // the loaded source value in place: one shift and two LOP3 per amplitude; then four FMAs
        const uint32_t sg = (W << (31 - r)) & 0x80000000u;
        C v = pb[(uint32_t)(r ^ XR) << kThreadBitsD];
        if constexpr (sizeof(T) == 8) {
            v.x = __hiloint2double(__double2hiint(v.x) ^ (int)sg, __double2loint(v.x));
            v.y = __hiloint2double(__double2hiint(v.y) ^ (int)sg, __double2loint(v.y));
            ar[r] = __fma_rn(fr[d], v.x, ar[r]);
            ar[r] = __fma_rn(-fi[d], v.y, ar[r]);
            ai[r] = __fma_rn(fr[d], v.y, ai[r]);
            ai[r] = __fma_rn(fi[d], v.x, ai[r]);
        } else {
            v.x = __uint_as_float(__float_as_uint(v.x) ^ sg);
            v.y = __uint_as_float(__float_as_uint(v.y) ^ sg);
            ar[r] = __fmaf_rn(fr[d], v.x, ar[r]);
            ar[r] = __fmaf_rn(-fi[d], v.y, ar[r]);
            ai[r] = __fmaf_rn(fr[d], v.y, ai[r]);
            ai[r] = __fmaf_rn(fi[d], v.x, ai[r]);
        }
    }
}

// uniform branch to the variant for XR = the r bits of x
template <typename T, int XR>
__device__ __forceinline__ void dispatch_local(uint32_t xr, const uint4* __restrict__ F, uint32_t idx0, uint32_t mpos,
                                               uint32_t W, const typename Cx<T>::type* pb, T (&ar)[kR], T (&ai)[kR]) {
    if constexpr (XR + 1 == kR) {
        local_group<T, XR>(F, idx0, mpos, W, pb, ar, ai);
    } else {
        if (xr == (uint32_t)XR) local_group<T, XR>(F, idx0, mpos, W, pb, ar, ai);
        else dispatch_local<T, XR + 1>(xr, F, idx0, mpos, W, pb, ar, ai);
    }
}

// All groups of one staged table chunk applied to the thread's kR accumulators; `sp` = the staged source tile.
template <typename T>
__device__ __forceinline__ void process_chunk(const uint4* __restrict__ ent, uint32_t ne, const typename Cx<T>::type* sp,
                                              uint32_t bt, int tid, T (&ar)[kR], T (&ai)[kR]) {
    using C = typename Cx<T>::type;
    uint32_t i = 0;
    while (i < ne) {
        const uint4 gh = ent[i];   // group header
        const uint32_t i_end = i + 1 + gh.y;
        if (gh.z == 4u) {          // x-local group: one table value per amplitude
            const uint4 hb = ent[i + 1];
            const uint4* F = ent + i + 2;
            uint32_t idx0 = 0;
#pragma unroll
            for (int k = 0; k < 4; ++k) idx0 |= ((bt >> ((hb.x >> (5 * k)) & 31u)) & 1u) << k;
            // hb.z = Walsh mask of the r bits of zb: bit r = parity(r & zb's bits 9..11); times the thread's own sign
            const uint32_t W = hb.z ^ (0u - ((uint32_t)__popc(bt & gh.w) & 1u));
            const C* pbl = sp + ((uint32_t)tid ^ (gh.x & (uint32_t)(kConsumerThreads - 1)));
            dispatch_local<T, 0>(gh.x >> kThreadBitsD, F, idx0, hb.y, W, pbl, ar, ai);
            i = i_end;
            continue;
        }
        T cr[kR], ci[kR];
#pragma unroll
        for (int r = 0; r < kR; ++r) {
            cr[r] = 0;
            ci[r] = 0;
        }
        // terms are sorted by bin; .w of the header says which bins occur, bit 8 of a term's .y closes its bin
        uint32_t t = i + 1;
        uint4 e = ent[t];
        walk_bins<T, 0>(ent, t, e, gh.w, bt, cr, ci);
        i = i_end;
        const C* pb = sp + ((uint32_t)tid ^ (gh.x & (uint32_t)(kConsumerThreads - 1)));
        const uint32_t xr = gh.x >> kThreadBitsD;
        if (gh.z == 1u) {          // real coefficients only
            wht(cr);
#pragma unroll
            for (int r = 0; r < kR; ++r) {
                const C v = pb[((uint32_t)r ^ xr) << kThreadBitsD];
                ar[r] = dn_fma(cr[r], v.x, ar[r]);
                ai[r] = dn_fma(cr[r], v.y, ai[r]);
            }
        } else if (gh.z == 2u) {   // imaginary coefficients only
            wht(ci);
#pragma unroll
            for (int r = 0; r < kR; ++r) {
                const C v = pb[((uint32_t)r ^ xr) << kThreadBitsD];
                ar[r] = dn_fma(-ci[r], v.y, ar[r]);
                ai[r] = dn_fma(ci[r], v.x, ai[r]);
            }
        } else {
            wht(cr);
            wht(ci);
#pragma unroll
            for (int r = 0; r < kR; ++r) {
                const C v = pb[((uint32_t)r ^ xr) << kThreadBitsD];
                ar[r] = dn_fma(-ci[r], v.y, dn_fma(cr[r], v.x, ar[r]));
                ai[r] = dn_fma(ci[r], v.x, dn_fma(cr[r], v.y, ai[r]));
            }
        }
    }
}

// ---------------------------------------------------------------------------------------------------------
// Small vectors (fewer tiles than SMs: dense N <= 38 in a parity block, N <= 36 in the full space): the table is cut
// into `split` contiguous ranges of chunks and work item (tile, s) applies range s to tile `tile`, writing its partial
// sums to scratch; a second kernel adds the `split` partials in a fixed order and does the (fused) epilogue.  No
// atomics: still bitwise reproducible.
// ---------------------------------------------------------------------------------------------------------
template <typename T>
struct DnSplitParams {
    using C = typename Cx<T>::type;
    const C* in;
    C* partial;                 // [split][D]
    int L;
    int split;
    const uint32_t* range;      // [split + 1] chunk indices
    const DenseChunk* chunks;   // .pad0 = hi of the load the chunk belongs to
    const uint4* entries;
};

template <typename T>
__global__ void __launch_bounds__(kThreads, 1) apply_h_dense_split_kernel(const DnSplitParams<T> p) {
    using C = typename Cx<T>::type;
    constexpr uint32_t TILE_BYTES = kTile * sizeof(C);
    constexpr uint32_t kChunk = 16384;
    extern __shared__ __align__(128) unsigned char smem[];
    C* stage = reinterpret_cast<C*>(smem);
    uint4* tbuf = reinterpret_cast<uint4*>(smem + TILE_BYTES);
    uint64_t* bar = reinterpret_cast<uint64_t*>(smem + TILE_BYTES + kChunkEntries * sizeof(uint4));
    const int tid = threadIdx.x;
    const uint32_t bar_full = smem_u32(bar);
    if (tid == 0) {
        mbar_init(bar_full, 1);
        mbar_fence_init();
    }
    __syncthreads();
    const uint32_t tile = blockIdx.x / (uint32_t)p.split, s = blockIdx.x % (uint32_t)p.split;
    const uint32_t base = tile << kTileLog2D;
    const uint32_t bt = base | (uint32_t)tid;
    T ar[kR], ai[kR];
#pragma unroll
    for (int r = 0; r < kR; ++r) {
        ar[r] = 0;
        ai[r] = 0;
    }
    uint32_t cur_hi = 0xffffffffu, n_loaded = 0;
    const uint32_t cA = __ldg(p.range + s), cB = __ldg(p.range + s + 1);
    for (uint32_t c = cA; c < cB; ++c) {
        const uint32_t e0 = __ldg(&p.chunks[c].e0), ne = __ldg(&p.chunks[c].ne), hi = __ldg(&p.chunks[c].pad0);
        __syncthreads();   // everyone is done with the staged tile and the staged table chunk
        const bool new_tile = hi != cur_hi;
        if (new_tile) {
            if (tid == 0) {
                mbar_arrive_expect_tx(bar_full, TILE_BYTES);
                const unsigned char* src = reinterpret_cast<const unsigned char*>(p.in + ((uint64_t)(tile ^ hi) << kTileLog2D));
#pragma unroll
                for (uint32_t k = 0; k < TILE_BYTES; k += kChunk) bulk_load(smem_u32(stage) + k, src + k, kChunk, bar_full);
            }
            cur_hi = hi;
        }
        for (uint32_t t = (uint32_t)tid; t < (uint32_t)kChunkEntries; t += kThreads)
            tbuf[t] = t < ne ? __ldg(p.entries + e0 + t) : make_uint4(0, 0, 0, 0);
        __syncthreads();
        if (new_tile) {
            mbar_wait(bar_full, n_loaded & 1u);
            ++n_loaded;
        }
        process_chunk<T>(tbuf, ne, stage, bt, tid, ar, ai);
    }
#pragma unroll
    for (int r = 0; r < kR; ++r) {
        C o;
        o.x = ar[r];
        o.y = ai[r];
        p.partial[((uint64_t)s << p.L) + (uint64_t)base + (uint32_t)tid + r * kConsumerThreads] = o;
    }
}

// out[b] = sum_s partial[s][b] (fixed order) with the epilogue of the other apply_H kernels
template <typename T, bool FUSED>
__global__ void __launch_bounds__(256) dense_reduce_kernel(const typename Cx<T>::type* partial, int split, int L,
                                                           const typename Cx<T>::type* in, typename Cx<T>::type* out,
                                                           const typename Cx<T>::type* prev, LanczosScalars* sc, int j) {
    using C = typename Cx<T>::type;
    __shared__ double red[40];
    double s_in = 1.0, s_prev = 0.0;
    if (FUSED) dn_fused_scalars(sc, j, red, s_in, s_prev);
    const uint64_t D = 1ull << L;
    double dot = 0.0;
    for (uint64_t b = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; b < D; b += (uint64_t)gridDim.x * blockDim.x) {
        T ar = 0, ai = 0;
        for (int s = 0; s < split; ++s) {
            const C v = partial[((uint64_t)s << L) + b];
            ar += v.x;
            ai += v.y;
        }
        C o;
        if (FUSED) {
            const C mine = in[b];
            double orr = (double)ar * s_in, oi = (double)ai * s_in;
            if (prev) {
                const C pv = prev[b];
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
        out[b] = o;
    }
    if (FUSED) {
        double s = block_sum(dot, red);
        if (threadIdx.x == 0) {
            sc->partial_dot[blockIdx.x] = s;
            if (blockIdx.x == 0) sc->n_partial_dot = gridDim.x;
        }
    }
}

template <typename T, bool FUSED>
__global__ void __launch_bounds__(kThreads, 1) apply_h_dense_kernel(const DnParams<T> p) {
    using C = typename Cx<T>::type;
    constexpr uint32_t TILE_BYTES = kTile * sizeof(C);
    constexpr uint32_t kChunk = 16384;

    extern __shared__ __align__(128) unsigned char smem[];
    C* stages = reinterpret_cast<C*>(smem);                       // 2 tile slots
    unsigned char* q = smem + (size_t)2 * TILE_BYTES;
    uint4* tbuf = reinterpret_cast<uint4*>(q);                    // 2 x kChunkEntries table entries
    q += 2 * kChunkEntries * sizeof(uint4);
    uint64_t* bars = reinterpret_cast<uint64_t*>(q);
    q += 2 * 8;
    double* red = reinterpret_cast<double*>(q);

    const int tid = threadIdx.x;
    const uint32_t bar_full = smem_u32(bars);
    if (tid == 0) {
        mbar_init(bar_full, 1);
        mbar_init(bar_full + 8, 1);
        mbar_fence_init();
    }
    __syncthreads();

    double s_in = 1.0, s_prev = 0.0;
    if (FUSED) dn_fused_scalars(p.sc, p.j, red, s_in, s_prev);

    const uint32_t n_tiles = 1u << (p.L - kTileLog2D);
    const int n_loads = p.n_loads;
    double dot = 0.0;

    // source tile of load l of output tile `tile` into slot s (thread 0 only; completion on full[s])
    auto issue = [&](uint32_t tile, int l, uint32_t s) {
        const uint32_t hi = __ldg(&p.loads[l].hi);
        mbar_arrive_expect_tx(bar_full + 8 * s, TILE_BYTES);
        const unsigned char* src = reinterpret_cast<const unsigned char*>(p.in + ((uint64_t)(tile ^ hi) << kTileLog2D));
        const uint32_t dst = smem_u32(stages) + s * TILE_BYTES;
#pragma unroll
        for (uint32_t c = 0; c < TILE_BYTES; c += kChunk) bulk_load(dst + c, src + c, kChunk, bar_full + 8 * s);
    };

    // table stream: this thread's entry of the chunk being prefetched
    uint32_t ck = 0;                           // chunk whose copy sits in tbuf[ck & 1] after the next barrier
    constexpr int kPre = (kChunkEntries + kThreads - 1) / kThreads;   // table entries per thread and chunk
    uint4 pre[kPre];
    auto fetch = [&](uint32_t c) {             // global -> register (chunk c)
        const uint32_t e0 = __ldg(&p.chunks[c].e0), ne = __ldg(&p.chunks[c].ne);
#pragma unroll
        for (int k = 0; k < kPre; ++k) {
            const uint32_t t = (uint32_t)tid + (uint32_t)k * kThreads;
            pre[k] = t < ne ? __ldg(p.entries + e0 + t) : make_uint4(0, 0, 0, 0);
        }
    };
    auto stash = [&](uint32_t c) {
#pragma unroll
        for (int k = 0; k < kPre; ++k)
            if (tid + k * kThreads < kChunkEntries) tbuf[(c & 1u) * kChunkEntries + tid + k * kThreads] = pre[k];
    };
    fetch(0);
    stash(0);
    uint32_t g = 0;                            // loads consumed by this CTA: slot g & 1, parity (g >> 1) & 1
    if (tid == 0 && blockIdx.x < n_tiles) issue(blockIdx.x, 0, 0);
    for (uint32_t tile = blockIdx.x; tile < n_tiles; tile += gridDim.x) {
        const uint32_t base = tile << kTileLog2D;
        const uint32_t bt = base | (uint32_t)tid;
        T ar[kR], ai[kR];
#pragma unroll
        for (int r = 0; r < kR; ++r) {
            ar[r] = 0;
            ai[r] = 0;
        }
        for (int l = 0; l < n_loads; ++l, ++g) {
            const uint32_t slot = g & 1u;
            __syncthreads();                   // everyone has finished with the other slot (load g - 1)
            if (tid == 0) {                    // prefetch the next load: a load is ~10^5 cycles of arithmetic
                if (l + 1 < n_loads) issue(tile, l + 1, slot ^ 1u);
                else if (tile + gridDim.x < n_tiles) issue(tile + gridDim.x, 0, slot ^ 1u);
            }
            const uint32_t c0 = __ldg(&p.loads[l].c0), c1 = __ldg(&p.loads[l].c1);
            mbar_wait(bar_full + 8 * slot, (g >> 1) & 1u);
            const C* sp = stages + (size_t)slot * kTile;
            for (uint32_t c = c0; c < c1; ++c, ++ck) {
                // chunk c is in tbuf[ck & 1] once every thread has stashed it; the other buffer is free again
                __syncthreads();
                const uint32_t cn = c + 1 == (uint32_t)p.n_chunks ? 0u : c + 1;
                fetch(cn);
                const uint32_t ne = __ldg(&p.chunks[c].ne);
                const uint4* ent = tbuf + (ck & 1u) * kChunkEntries;
                process_chunk<T>(ent, ne, sp, bt, tid, ar, ai);
                stash(ck + 1);
            }
        }
        // epilogue (a tile takes milliseconds of arithmetic here: the latency of these global reads is nothing)
#pragma unroll
        for (int r = 0; r < kR; ++r) {
            const uint64_t b = (uint64_t)base + (uint32_t)tid + r * kConsumerThreads;
            C o;
            if (FUSED) {
                const C mine = __ldg(p.in + b);
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
    if (FUSED) {
        double s = block_sum(dot, red);
        if (tid == 0) {
            p.sc->partial_dot[blockIdx.x] = s;
            if (blockIdx.x == 0) p.sc->n_partial_dot = gridDim.x;
        }
    }
}

// Host: the entry stream (group header + its terms, canonical order), cut into chunks of whole groups that do not
// cross a load (run of equal x >> 12, ascending); uploaded once per handle and dtype.
int build_dense_tables(const syk_ham* h, int dtype, DenseCache& dc) {
    const size_t ng = h->x.size();
    std::vector<DenseLoad> loads;
    std::vector<DenseChunk> chunks;
    std::vector<uint4> entries;
    entries.reserve(h->z.size() + ng);
    int n_local = 0;
    for (size_t g = 0; g < ng; ++g) {
        const uint32_t x = (uint32_t)h->x[g];
        const uint32_t hi = x >> kTileLog2D;
        const uint32_t nt = h->group_off[g + 1] - h->group_off[g];
        if (nt + 1 > (uint32_t)kChunkEntries - 1) return SYK_EINVAL;   // a group must fit one chunk (dense N <= 64: 497)
        const bool new_load = loads.empty() || loads.back().hi != hi;
        if (new_load) {
            if (!loads.empty()) loads.back().c1 = (uint32_t)chunks.size();
            loads.push_back(DenseLoad{hi, (uint32_t)chunks.size(), 0u, 0u});
        }
        // x-local group (see local_group): all Z-masks agree outside x, popcount(x) <= 4, enough terms to pay for the table
        const int kx = __builtin_popcount(x);
        bool local = kx <= kLocalMaxBits && nt >= (uint32_t)kLocalMinTerms;
        const uint32_t z_first = (uint32_t)h->z[h->group_off[g]];
        for (uint32_t t = h->group_off[g]; t < h->group_off[g + 1] && local; ++t)
            if ((((uint32_t)h->z[t]) ^ z_first) & ~x) local = false;
        const uint32_t n_follow = local ? 1u + (1u << kx) : nt;
        if (new_load || chunks.back().ne + n_follow + 1 > (uint32_t)kChunkEntries - 1)   // one spare entry: read-ahead
            chunks.push_back(DenseChunk{(uint32_t)entries.size(), 0u, hi, 0u});
        if (local) {
            int pos[4] = {kThreadBitsD, kThreadBitsD, kThreadBitsD, kThreadBitsD};   // unused: an r bit (0 in the base index)
            int np = 0;
            for (int q = 0; q < 32; ++q)
                if (x & (1u << q)) pos[np++] = q;
            uint32_t mpos = 0;   // index bit of r bit j (index bit 9 + j of the vector), if x contains it
            for (int j = 0; j < kRBits; ++j) {
                const uint32_t bit = 1u << (kThreadBitsD + j);
                if (x & bit) mpos |= (uint32_t)__builtin_popcount(x & (bit - 1u)) << (2 * j);
            }
            uint32_t walsh = 0;   // bit r = parity of r & (bits 9..11 of the common Z part)
            for (uint32_t r = 0; r < (uint32_t)kR; ++r)
                walsh |= (uint32_t)(__builtin_popcount(r & (((z_first & ~x) >> kThreadBitsD) & (uint32_t)(kR - 1))) & 1) << r;
            entries.push_back(make_uint4(x & (uint32_t)(kTile - 1), n_follow, 4u, z_first & ~x));
            entries.push_back(make_uint4((uint32_t)pos[0] | (uint32_t)pos[1] << 5 | (uint32_t)pos[2] << 10 | (uint32_t)pos[3] << 15,
                                         mpos, walsh, 0u));
            for (uint32_t i = 0; i < (1u << kx); ++i) {
                uint32_t dep = 0;   // pdep(i, x)
                for (int q = 0; q < np; ++q)
                    if (i & (1u << q)) dep |= 1u << pos[q];
                double fr = 0.0, fi = 0.0;
                for (uint32_t t = h->group_off[g]; t < h->group_off[g + 1]; ++t) {
                    const std::complex<double> c = h->c[t];
                    if (c.imag() != 0.0 && c.real() != 0.0) return SYK_EINVAL;
                    double re = c.real(), im = c.imag();
                    if (dtype != SYK_C128) {   // R-C64: coefficients rounded once to fp32, summed exactly enough in fp64
                        re = (double)(float)re;
                        im = (double)(float)im;
                    }
                    const double sg = (__builtin_popcount(dep & (uint32_t)h->z[t]) & 1) ? -1.0 : 1.0;
                    fr += sg * re;
                    fi += sg * im;
                }
                uint4 e = make_uint4(0u, 0u, 0u, 0u);
                if (dtype == SYK_C128) {
                    uint64_t b0, b1;
                    std::memcpy(&b0, &fr, 8);
                    std::memcpy(&b1, &fi, 8);
                    e = make_uint4((uint32_t)b0, (uint32_t)(b0 >> 32), (uint32_t)b1, (uint32_t)(b1 >> 32));
                } else {
                    const float f0 = (float)fr, f1 = (float)fi;
                    std::memcpy(&e.x, &f0, 4);
                    std::memcpy(&e.y, &f1, 4);
                }
                entries.push_back(e);
            }
            chunks.back().ne += n_follow + 1;
            ++n_local;
            continue;
        }
        uint32_t flags = 0, occ = 0;
        const size_t header_at = entries.size();
        entries.push_back(make_uint4(x & (uint32_t)(kTile - 1), nt, 0u, 0u));
        std::vector<uint4> run;
        run.reserve(nt);
        for (uint32_t t = h->group_off[g]; t < h->group_off[g + 1]; ++t) {
            const std::complex<double> c = h->c[t];
            const bool imag = c.imag() != 0.0;
            if (imag && c.real() != 0.0) return SYK_EINVAL;   // never for SYK strings
            const double a = imag ? c.imag() : c.real();
            const uint32_t z = (uint32_t)h->z[t];
            uint4 e;
            e.x = z;
            e.y = ((z >> kThreadBitsD) & (uint32_t)(kR - 1)) | (imag ? (uint32_t)kR : 0u);
            if (dtype == SYK_C128) {
                uint64_t bits;
                std::memcpy(&bits, &a, 8);
                e.z = (uint32_t)bits;
                e.w = (uint32_t)(bits >> 32);
            } else {
                const float af = (float)a;   // R-C64: rounded once
                uint32_t bits;
                std::memcpy(&bits, &af, 4);
                e.z = bits;
                e.w = 0;
            }
            run.push_back(e);
            flags |= imag ? 2u : 1u;
            occ |= 1u << (e.y & 31u);
        }
        std::stable_sort(run.begin(), run.end(), [](const uint4& p, const uint4& q) { return (p.y & 31u) < (q.y & 31u); });
        for (size_t i = 0; i < run.size(); ++i) {
            if (i + 1 == run.size() || (run[i + 1].y & 31u) != (run[i].y & 31u)) run[i].y |= 256u;   // closes its bin
            entries.push_back(run[i]);
        }
        entries[header_at].w = occ;
        entries[header_at].z = flags;
        chunks.back().ne += nt + 1;
    }
    if (!loads.empty()) loads.back().c1 = (uint32_t)chunks.size();
    auto align = [](size_t v) { return (v + 255) & ~(size_t)255; };
    const size_t off_c = align(loads.size() * sizeof(DenseLoad));
    const size_t off_e = off_c + align(chunks.size() * sizeof(DenseChunk));
    const size_t total = off_e + align(entries.size() * sizeof(uint4)) + 256;
    std::vector<unsigned char> host(total, 0);
    std::memcpy(host.data(), loads.data(), loads.size() * sizeof(DenseLoad));
    std::memcpy(host.data() + off_c, chunks.data(), chunks.size() * sizeof(DenseChunk));
    std::memcpy(host.data() + off_e, entries.data(), entries.size() * sizeof(uint4));
    int dev = 0;
    SYK_CUDA(cudaGetDevice(&dev));
    void* blob = nullptr;
    SYK_CUDA(cudaMalloc(&blob, total));
    cudaError_t e = cudaMemcpy(blob, host.data(), total, cudaMemcpyHostToDevice);
    if (e != cudaSuccess) {
        cudaFree(blob);
        set_cuda_error(e, "cudaMemcpy(dense term tables)");
        return SYK_ECUDA;
    }
    dc.blob = blob;
    dc.device = dev;
    dc.off_groups = off_c;
    dc.off_terms = off_e;
    dc.n_loads = (int)loads.size();
    dc.n_chunks = (int)chunks.size();
    dc.n_local_groups = n_local;
    // small vectors: split the chunk list over several CTAs per tile (apply_h_dense_split_kernel)
    dc.split = 1;
    const int sms = num_sms();
    const uint64_t n_tiles = 1ull << (h->L - kTileLog2D);
    if (sms > 0 && n_tiles * 2 <= (uint64_t)sms && chunks.size() >= 2) {
        int split = (int)((uint64_t)(2 * sms) / n_tiles);
        if (split > (int)chunks.size()) split = (int)chunks.size();
        if (split > 64) split = 64;
        std::vector<uint32_t> range((size_t)split + 1);
        for (int s2 = 0; s2 <= split; ++s2) range[(size_t)s2] = (uint32_t)((uint64_t)chunks.size() * s2 / split);
        const size_t pbytes = (size_t)split * ((size_t)elem_bytes(dtype) << h->L);
        void* scratch = nullptr;
        SYK_CUDA(cudaMalloc(&scratch, pbytes + 4096));
        cudaError_t e2 = cudaMemcpy((char*)scratch + pbytes, range.data(), range.size() * 4, cudaMemcpyHostToDevice);
        if (e2 != cudaSuccess) {
            cudaFree(scratch);
            set_cuda_error(e2, "cudaMemcpy(dense split ranges)");
            return SYK_ECUDA;
        }
        dc.partial = scratch;
        dc.range = (const uint32_t*)((char*)scratch + pbytes);
        dc.split = split;
    }
    return SYK_OK;
}

int get_dense_tables(const syk_ham* h, int dtype, const DenseCache** out) {
    const int k = dtype == SYK_C128 ? 1 : 0;
    int dev = 0;
    SYK_CUDA(cudaGetDevice(&dev));
    if (!h->dn[k]) h->dn[k] = new (std::nothrow) DenseCache();
    if (!h->dn[k]) return SYK_ENOMEM;
    DenseCache& dc = *h->dn[k];
    if (dc.blob && dc.device != dev) {
        cudaFree(dc.blob);
        if (dc.partial) cudaFree(dc.partial);
        dc = DenseCache();
    }
    if (!dc.blob) SYK_TRY(build_dense_tables(h, dtype, dc));
    *out = &dc;
    return SYK_OK;
}

template <typename T>
int launch_dn(const syk_ham* h, const DenseCache& dc, const void* d_in, void* d_out, const FusedArgs& fa,
              cudaStream_t stream) {
    using C = typename Cx<T>::type;
    constexpr size_t kTileBytes = (size_t)kTile * sizeof(C);
    DnParams<T> p;
    p.in = (const C*)d_in;
    p.out = (C*)d_out;
    p.prev = (const C*)fa.prev;
    p.sc = fa.sc;
    p.j = fa.j;
    p.L = h->L;
    p.nslot = 2;
    p.loads = (const DenseLoad*)dc.blob;
    p.chunks = (const DenseChunk*)((const unsigned char*)dc.blob + dc.off_groups);
    p.entries = (const uint4*)((const unsigned char*)dc.blob + dc.off_terms);
    p.n_loads = dc.n_loads;
    p.n_chunks = dc.n_chunks;
    const size_t smem = 2 * kTileBytes + kMiscBytes;
    const int sms = num_sms();
    if (sms <= 0) return SYK_ECUDA;
    if (dc.split > 1) {
        DnSplitParams<T> sp;
        sp.in = (const C*)d_in;
        sp.partial = (C*)dc.partial;
        sp.L = h->L;
        sp.split = dc.split;
        sp.range = dc.range;
        sp.chunks = p.chunks;
        sp.entries = p.entries;
        const size_t smem2 = kTileBytes + (size_t)kChunkEntries * sizeof(uint4) + 64;
        const unsigned n_items = (unsigned)((1ull << (h->L - kTileLog2D)) * (uint64_t)dc.split);
        SYK_CUDA(cudaFuncSetAttribute(apply_h_dense_split_kernel<T>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem2));
        apply_h_dense_split_kernel<T><<<n_items, kThreads, smem2, stream>>>(sp);
        const uint64_t D = 1ull << h->L;
        const unsigned gr = (unsigned)std::min<uint64_t>((D + 255) / 256, (uint64_t)sms * 4);
        if (fa.sc)
            dense_reduce_kernel<T, true><<<gr, 256, 0, stream>>>((const C*)dc.partial, dc.split, h->L, (const C*)d_in, (C*)d_out,
                                                                (const C*)fa.prev, fa.sc, fa.j);
        else
            dense_reduce_kernel<T, false><<<gr, 256, 0, stream>>>((const C*)dc.partial, dc.split, h->L, (const C*)d_in, (C*)d_out,
                                                                 nullptr, nullptr, 0);
        count_launch(2);
        SYK_CUDA(cudaGetLastError());
        return SYK_OK;
    }
    const uint64_t n_tiles = 1ull << (h->L - kTileLog2D);
    const int grid = (int)(n_tiles < (uint64_t)sms ? n_tiles : (uint64_t)sms);
    if (fa.sc) {
        SYK_CUDA(cudaFuncSetAttribute(apply_h_dense_kernel<T, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        apply_h_dense_kernel<T, true><<<grid, kThreads, smem, stream>>>(p);
    } else {
        SYK_CUDA(cudaFuncSetAttribute(apply_h_dense_kernel<T, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        apply_h_dense_kernel<T, false><<<grid, kThreads, smem, stream>>>(p);
    }
    count_launch();
    SYK_CUDA(cudaGetLastError());
    return SYK_OK;
}

}  // namespace

// Can the handle use the dense-table kernel?  Automatic choice: many terms per X-mask (vectors with fewer tiles than SMs
// take the split form: the table is shared out over several CTAs per tile).
bool dense_kernel_ok(const syk_ham* h, bool forced) {
    if (h->n_terms() == 0 || h->L < kTileLog2D) return false;
    if (!forced && !(h->n_terms() >= 4 * h->n_groups() && h->n_terms() > kRtMaxTerms)) return false;
    // what build_dense_tables cannot represent: a group larger than one table chunk (generic Pauli sums with very many
    // diagonal terms), a coefficient that is neither real nor imaginary (non-Hermitian sums) -> another kernel
    if (h->dense_representable < 0) {   // tables are immutable after the build: checked once
        int ok = 1;
        for (size_t g = 0; g < h->x.size() && ok; ++g)
            if (h->group_off[g + 1] - h->group_off[g] + 1 > (uint32_t)kChunkEntries - 1) ok = 0;
        for (size_t t = 0; t < h->c.size() && ok; ++t)
            if (h->c[t].real() != 0.0 && h->c[t].imag() != 0.0) ok = 0;
        h->dense_representable = ok;
    }
    return h->dense_representable == 1;
}

int prepare_dense_tables(const syk_ham* h, int dtype) {
    const DenseCache* dc = nullptr;
    return get_dense_tables(h, dtype, &dc);
}

int dense_tables_info(const syk_ham* h, int dtype, int* n_loads, int* n_chunks, int* split, int* n_local_groups) {
    const DenseCache* dc = nullptr;
    SYK_TRY(get_dense_tables(h, dtype, &dc));
    if (n_loads) *n_loads = dc->n_loads;
    if (n_chunks) *n_chunks = dc->n_chunks;
    if (split) *split = dc->split;
    if (n_local_groups) *n_local_groups = dc->n_local_groups;
    return SYK_OK;
}

int launch_apply_h_dense(const syk_ham* h, int dtype, const void* d_in, void* d_out, const FusedArgs& fa,
                         cudaStream_t stream) {
    const DenseCache* dc = nullptr;
    SYK_TRY(get_dense_tables(h, dtype, &dc));
    if (dtype == SYK_C128) return launch_dn<double>(h, *dc, d_in, d_out, fa, stream);
    return launch_dn<float>(h, *dc, d_in, d_out, fa, stream);
}

void free_dense_tables(const syk_ham* h) {
    for (int k = 0; k < 2; ++k) {
        if (h->dn[k]) {
            if (h->dn[k]->blob) cudaFree(h->dn[k]->blob);
            if (h->dn[k]->partial) cudaFree(h->dn[k]->partial);
            delete h->dn[k];
            h->dn[k] = nullptr;
        }
    }
}

}  // namespace syk
