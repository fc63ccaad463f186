// a-3  Fused Krylov vector kernels (the Krylov method's vector work and its memory count).
//
// Each Lanczos step is two kernels: apply_H with the fused epilogue (apply_h.cu) and `axpy_norm_kernel` here:
//     u_{j+1} = w - (alpha_j/|u_j|) u_j   and   sum |u_{j+1}|^2   in one pass (2 reads + 1 write),
// with alpha_j finalised from apply_H's per-CTA partial sums in this kernel's prologue, so no scalar crosses to
// the host during a Lanczos run.  Vectors are kept un-normalised (u_j = |u_j| v_j); the normalisation is folded
// into the scalars of the next kernel.  All reductions: fp64, per-thread serial -> warp shuffle tree -> per-CTA
// partial -> fixed-order sum of partials; no atomics, bitwise reproducible.
//
// Vectors are processed in 16-byte units (one complex128 or two complex64) with grid-stride loops.
#include <cstddef>

#include "device_utils.cuh"

namespace syk {

namespace {

constexpr int kThreads = 256;

template <typename T> struct Unit;
template <> struct Unit<double> {
    using V = double2;
    static constexpr int NS = 2;   // scalars per unit
    static __device__ __forceinline__ void load(const V* p, uint64_t i, double* a) {
        V v = p[i];
        a[0] = v.x; a[1] = v.y;
    }
    static __device__ __forceinline__ void store(V* p, uint64_t i, const double* a) { p[i] = make_double2(a[0], a[1]); }
};
template <> struct Unit<float> {
    using V = float4;
    static constexpr int NS = 4;
    static __device__ __forceinline__ void load(const V* p, uint64_t i, double* a) {
        V v = p[i];
        a[0] = v.x; a[1] = v.y; a[2] = v.z; a[3] = v.w;
    }
    static __device__ __forceinline__ void store(V* p, uint64_t i, const double* a) {
        p[i] = make_float4((float)a[0], (float)a[1], (float)a[2], (float)a[3]);
    }
    // rounds a[] to fp32 in place so that reductions see the stored values
};

template <typename T> __device__ __forceinline__ double stored(double v);
template <> __device__ __forceinline__ double stored<double>(double v) { return v; }
template <> __device__ __forceinline__ double stored<float>(double v) { return (double)(float)v; }

inline uint64_t n_units(int dtype, uint64_t D) { return dtype == SYK_C128 ? D : D / 2; }

inline int grid_for(uint64_t units) {
    const int sms = num_sms();
    uint64_t blocks = (units + kThreads - 1) / kThreads;
    uint64_t cap = (uint64_t)(sms > 0 ? sms : 1) * 8;
    if (cap > (uint64_t)kMaxPartials) cap = kMaxPartials;
    if (blocks < 1) blocks = 1;
    return (int)(blocks < cap ? blocks : cap);
}

// Batched launches (grid.y = realization): argument k of realization r lives at base_k + r * stride_k bytes.
template <typename P>
__device__ __forceinline__ P* at_batch(P* p, size_t stride) {
    return p ? reinterpret_cast<P*>(reinterpret_cast<uintptr_t>(p) + (size_t)blockIdx.y * stride) : p;
}

#define GRID_STRIDE(i, n) \
    for (uint64_t i = (uint64_t)blockIdx.x * kThreads + threadIdx.x; i < (n); i += (uint64_t)gridDim.x * kThreads)

template <typename T>
__global__ void __launch_bounds__(kThreads) norm2_kernel(const typename Unit<T>::V* __restrict__ v, uint64_t n,
                                                         LanczosScalars* sc, BatchStride bs) {
    __shared__ double red[40];
    v = at_batch(v, bs.a);
    sc = at_batch(sc, bs.sc);
    double s = 0.0;
    GRID_STRIDE(i, n) {
        double a[4];
        Unit<T>::load(v, i, a);
#pragma unroll
        for (int k = 0; k < Unit<T>::NS; ++k) s += a[k] * a[k];
    }
    s = block_sum(s, red);
    if (threadIdx.x == 0) {
        sc->partial_nrm[blockIdx.x] = s;
        if (blockIdx.x == 0) sc->n_partial_nrm = gridDim.x;
    }
}

// w <- w - (alpha_j/|u_j|) u ; partial |w|^2 ; optionally y <- ys*y + cy*u (complex scalars)
template <typename T, bool WITH_Y>
__global__ void __launch_bounds__(kThreads) axpy_norm_kernel(typename Unit<T>::V* __restrict__ w,
                                                             const typename Unit<T>::V* __restrict__ u,
                                                             typename Unit<T>::V* y, uint64_t n, int j, int first_y,
                                                             LanczosScalars* sc, BatchStride bs) {
    __shared__ double red[40];
    w = at_batch(w, bs.a);
    u = at_batch(u, bs.b);
    y = at_batch(y, bs.c);
    sc = at_batch(sc, bs.sc);
    const double nj = sc->nrm[j];
    const double dotsum = reduce_partials(sc->partial_dot, sc->n_partial_dot, red);
    const double alpha = nj > 0.0 ? dotsum / nj : 0.0;
    if (blockIdx.x == 0 && threadIdx.x == 0) sc->alpha[j] = alpha;
    const double a = nj > 0.0 ? alpha / nj : 0.0;
    double cyr = 0.0, cyi = 0.0, ysr = 1.0, ysi = 0.0;
    if (WITH_Y) {
        const double inv = nj > 0.0 ? 1.0 / nj : 0.0;
        cyr = sc->coef[j].x * inv;
        cyi = sc->coef[j].y * inv;
        if (first_y) {
            const double n1 = sc->nrm[1];
            const double inv1 = n1 > 0.0 ? 1.0 / n1 : 0.0;
            ysr = sc->coef[1].x * inv1;
            ysi = sc->coef[1].y * inv1;
        }
    }
    double s = 0.0;
    GRID_STRIDE(i, n) {
        double wv[4], uv[4];
        Unit<T>::load(w, i, wv);
        Unit<T>::load(u, i, uv);
#pragma unroll
        for (int k = 0; k < Unit<T>::NS; ++k) {
            wv[k] = stored<T>(wv[k] - a * uv[k]);
            s += wv[k] * wv[k];
        }
        Unit<T>::store(w, i, wv);
        if (WITH_Y) {
            double yv[4];
            Unit<T>::load(y, i, yv);
#pragma unroll
            for (int k = 0; k < Unit<T>::NS; k += 2) {
                const double yr = ysr * yv[k] - ysi * yv[k + 1] + cyr * uv[k] - cyi * uv[k + 1];
                const double yi = ysr * yv[k + 1] + ysi * yv[k] + cyr * uv[k + 1] + cyi * uv[k];
                yv[k] = yr;
                yv[k + 1] = yi;
            }
            Unit<T>::store(y, i, yv);
        }
    }
    s = block_sum(s, red);
    if (threadIdx.x == 0) {
        sc->partial_nrm[blockIdx.x] = s;
        if (blockIdx.x == 0) sc->n_partial_nrm = gridDim.x;
    }
}

__global__ void __launch_bounds__(kThreads) finalize_nrm_kernel(int j, LanczosScalars* sc, BatchStride bs) {
    __shared__ double red[40];
    sc = at_batch(sc, bs.sc);
    const double n2 = reduce_partials(sc->partial_nrm, sc->n_partial_nrm, red);
    if (threadIdx.x == 0) sc->nrm[j] = sqrt(n2);
}

// psi <- sum_{j=1..m} (coef[j]/nrm[j]) u_j ; u_1 = psi, u_j (j >= 2) = vecs + (j-2)*stride units
template <typename T>
__global__ void __launch_bounds__(kThreads) combine_kernel(typename Unit<T>::V* psi, const typename Unit<T>::V* vecs,
                                                           uint64_t stride, uint64_t n, int m,
                                                           const LanczosScalars* __restrict__ sc, BatchStride bs) {
    __shared__ double cr[kMaxKrylov + 2], ci[kMaxKrylov + 2];
    psi = at_batch(psi, bs.a);
    vecs = at_batch(vecs, bs.b);
    sc = at_batch(sc, bs.sc);
    if (m < 0) m = sc->m_eff;   // batched: every realization has its own effective Krylov dimension
    for (int j = 1 + threadIdx.x; j <= m; j += kThreads) {
        const double nj = sc->nrm[j];
        const double inv = nj > 0.0 ? 1.0 / nj : 0.0;
        cr[j] = sc->coef[j].x * inv;
        ci[j] = sc->coef[j].y * inv;
    }
    __syncthreads();
    GRID_STRIDE(i, n) {
        double acc[4], uv[4];
        Unit<T>::load(psi, i, uv);
#pragma unroll
        for (int k = 0; k < Unit<T>::NS; k += 2) {
            acc[k] = cr[1] * uv[k] - ci[1] * uv[k + 1];
            acc[k + 1] = cr[1] * uv[k + 1] + ci[1] * uv[k];
        }
        for (int j = 2; j <= m; ++j) {
            Unit<T>::load(vecs + (uint64_t)(j - 2) * stride, i, uv);
#pragma unroll
            for (int k = 0; k < Unit<T>::NS; k += 2) {
                acc[k] += cr[j] * uv[k] - ci[j] * uv[k + 1];
                acc[k + 1] += cr[j] * uv[k + 1] + ci[j] * uv[k];
            }
        }
        Unit<T>::store(psi, i, acc);
    }
}

// y <- ys*y + cy*u with ys = first_y ? coef[1]/nrm[1] : 1, cy = (u ? coef[j]/nrm[j] : 0)
template <typename T>
__global__ void __launch_bounds__(kThreads) axpy_coef_kernel(typename Unit<T>::V* y, const typename Unit<T>::V* u,
                                                             uint64_t n, int j, int first_y,
                                                             const LanczosScalars* __restrict__ sc) {
    double cyr = 0.0, cyi = 0.0, ysr = 1.0, ysi = 0.0;
    if (u) {
        const double nj = sc->nrm[j];
        const double inv = nj > 0.0 ? 1.0 / nj : 0.0;
        cyr = sc->coef[j].x * inv;
        cyi = sc->coef[j].y * inv;
    }
    if (first_y) {
        const double n1 = sc->nrm[1];
        const double inv1 = n1 > 0.0 ? 1.0 / n1 : 0.0;
        ysr = sc->coef[1].x * inv1;
        ysi = sc->coef[1].y * inv1;
    }
    GRID_STRIDE(i, n) {
        double yv[4], uv[4] = {0, 0, 0, 0};
        Unit<T>::load(y, i, yv);
        if (u) Unit<T>::load(u, i, uv);
#pragma unroll
        for (int k = 0; k < Unit<T>::NS; k += 2) {
            const double yr = ysr * yv[k] - ysi * yv[k + 1] + cyr * uv[k] - cyi * uv[k + 1];
            const double yi = ysr * yv[k + 1] + ysi * yv[k] + cyr * uv[k + 1] + cyi * uv[k];
            yv[k] = yr;
            yv[k + 1] = yi;
        }
        Unit<T>::store(y, i, yv);
    }
}

template <typename T>
__global__ void __launch_bounds__(kThreads) cdot_kernel(const typename Unit<T>::V* __restrict__ a,
                                                        const typename Unit<T>::V* __restrict__ b, uint64_t n,
                                                        LanczosScalars* sc, BatchStride bs) {
    __shared__ double red[40];
    a = at_batch(a, bs.a);
    b = at_batch(b, bs.b);
    sc = at_batch(sc, bs.sc);
    double sr = 0.0, si = 0.0;
    GRID_STRIDE(i, n) {
        double av[4], bv[4];
        Unit<T>::load(a, i, av);
        Unit<T>::load(b, i, bv);
#pragma unroll
        for (int k = 0; k < Unit<T>::NS; k += 2) {   // conj(a) * b
            sr += av[k] * bv[k] + av[k + 1] * bv[k + 1];
            si += av[k] * bv[k + 1] - av[k + 1] * bv[k];
        }
    }
    sr = block_sum(sr, red);
    si = block_sum(si, red);
    if (threadIdx.x == 0) {
        sc->partial_cdot[blockIdx.x] = make_double2(sr, si);
        if (blockIdx.x == 0) sc->n_partial_cdot = gridDim.x;
    }
}

// coef[0] <- sum of the complex partials (fixed order): the result slot of a batched inner product
__global__ void __launch_bounds__(kThreads) finalize_cdot_kernel(LanczosScalars* sc, BatchStride bs) {
    __shared__ double red[40];
    sc = at_batch(sc, bs.sc);
    double sr = 0.0, si = 0.0;
    for (int i = threadIdx.x; i < sc->n_partial_cdot; i += kThreads) {
        sr += sc->partial_cdot[i].x;
        si += sc->partial_cdot[i].y;
    }
    sr = block_sum(sr, red);
    si = block_sum(si, red);
    if (threadIdx.x == 0) sc->coef[0] = make_double2(sr, si);
}

// v <- v / sqrt(sum partial_nrm)
template <typename T>
__global__ void __launch_bounds__(kThreads) normalise_kernel(typename Unit<T>::V* v, uint64_t n, LanczosScalars* sc) {
    __shared__ double red[40];
    const double n2 = reduce_partials(sc->partial_nrm, sc->n_partial_nrm, red);
    const double inv = n2 > 0.0 ? 1.0 / sqrt(n2) : 0.0;
    GRID_STRIDE(i, n) {
        double a[4];
        Unit<T>::load(v, i, a);
#pragma unroll
        for (int k = 0; k < Unit<T>::NS; ++k) a[k] *= inv;
        Unit<T>::store(v, i, a);
    }
}

// R-PSI: amplitude b = rho (cos, sin)(2 pi u2), rho = sqrt(-2 ln u1), from stream 2 of R-RNG; partial |.|^2
// A bit permutation of basis indices: index bit j moves to bit src_bit[j] (n_bits = 0: identity).
struct BitPerm {
    uint8_t src_bit[32];
    int n_bits;
};
__device__ __forceinline__ uint64_t bit_permute(const BitPerm& bp, uint64_t i) {
    if (bp.n_bits == 0) return i;
    uint64_t r = 0;
    for (int j = 0; j < bp.n_bits; ++j) r |= ((i >> j) & 1ull) << bp.src_bit[j];
    return r;
}

// The stored amplitude i is the amplitude of the canonical basis state bit_permute(to_canonical, i) (qubit layout of
// a handle), so a state is the same physical state in every layout.
template <typename T>
__global__ void __launch_bounds__(kThreads) random_fill_kernel(typename Cx<T>::type* psi, uint64_t D, uint64_t key,
                                                               LanczosScalars* sc, const BitPerm to_canonical) {
    __shared__ double red[40];
    double s = 0.0;
    GRID_STRIDE(i, D) {
        const uint64_t b = bit_permute(to_canonical, i);
        const double u1 = (double)(rng_draw(key, b, 0) + 1) * 0x1.0p-53;
        const double u2 = (double)rng_draw(key, b, 1) * 0x1.0p-53;
        const double rho = sqrt(-2.0 * log(u1));
        double sn, cs;
        sincos(6.283185307179586476925286766559 * u2, &sn, &cs);
        typename Cx<T>::type o;
        o.x = (T)(rho * cs);
        o.y = (T)(rho * sn);
        psi[i] = o;
        s += (double)o.x * (double)o.x + (double)o.y * (double)o.y;
    }
    s = block_sum(s, red);
    if (threadIdx.x == 0) {
        sc->partial_nrm[blockIdx.x] = s;
        if (blockIdx.x == 0) sc->n_partial_nrm = gridDim.x;
    }
}

// out = gamma_n in, one thread per pair (b0, b0 | bit); works in place.
//   gamma_{2q}   = s Z^{bit-1} X^{bit};  gamma_{2q+1} = -i s Z^{2 bit - 1} X^{bit}   (R-JW, R-SIGN)
// given as the index bit q that is flipped and the Z-mask over index bits (both already mapped through the qubit layout).
template <typename T>
__global__ void __launch_bounds__(kThreads) gamma_kernel(const typename Cx<T>::type* in, typename Cx<T>::type* out,
                                                         uint64_t half, int q, uint32_t zmask, int odd, T s, BatchStride bs) {
    using C = typename Cx<T>::type;
    in = at_batch(in, bs.a);
    out = at_batch(out, bs.b);
    const uint64_t bit = 1ull << q;
    GRID_STRIDE(pidx, half) {
        const uint64_t b0 = ((pidx >> q) << (q + 1)) | (pidx & (bit - 1));
        const uint64_t b1 = b0 | bit;
        const C v0 = in[b0], v1 = in[b1];
        const T s0 = (__popc((uint32_t)b0 & zmask) & 1) ? -s : s;
        const T s1 = (__popc((uint32_t)b1 & zmask) & 1) ? -s : s;
        C o0, o1;
        if (odd) {   // times -i: (x, y) -> (y, -x)
            o0.x = s0 * v1.y; o0.y = -s0 * v1.x;
            o1.x = s1 * v0.y; o1.y = -s1 * v0.x;
        } else {
            o0.x = s0 * v1.x; o0.y = s0 * v1.y;
            o1.x = s1 * v0.x; o1.y = s1 * v0.y;
        }
        out[b0] = o0;
        out[b1] = o1;
    }
}

// Blocks of the two gammas of the dropped top qubit between parity sectors (R-BLOCK): no gather.
//   mode 0: gamma_{N-2}: out[b'] = s (-1)^popcount(b') in[b']        mode 1: gamma_{N-1}: out[b'] = -i s sigma in[b']
template <typename T>
__global__ void __launch_bounds__(kThreads) gamma_top_kernel(const typename Cx<T>::type* in, typename Cx<T>::type* out,
                                                             uint64_t n, int mode, T s_sigma) {
    using C = typename Cx<T>::type;
    GRID_STRIDE(b, n) {
        const C v = in[b];
        C o;
        if (mode == 0) {
            const T s = (__popc((uint32_t)b) & 1) ? -s_sigma : s_sigma;
            o.x = s * v.x;
            o.y = s * v.y;
        } else {   // times -i: (x, y) -> (y, -x)
            o.x = s_sigma * v.y;
            o.y = -s_sigma * v.x;
        }
        out[b] = o;
    }
}

// out[i] = in[bit_permute(bp, i)]: change of qubit layout of a whole vector (writes coalesced, reads gathered)
template <typename T>
__global__ void __launch_bounds__(kThreads) bit_permute_kernel(const typename Cx<T>::type* in, typename Cx<T>::type* out,
                                                               uint64_t D, const BitPerm bp) {
    GRID_STRIDE(i, D) { out[i] = in[bit_permute(bp, i)]; }
}

#define DISPATCH(dtype, CALL_D, CALL_F) \
    do {                                \
        if ((dtype) == SYK_C128) {      \
            CALL_D;                     \
        } else {                        \
            CALL_F;                     \
        }                               \
        count_launch();                 \
        SYK_CUDA(cudaGetLastError());   \
    } while (0)

}  // namespace

int launch_norm2(int dtype, uint64_t D, const void* v, LanczosScalars* sc, cudaStream_t st, const Batch& bt) {
    const uint64_t n = n_units(dtype, D);
    const int g = grid_for(n);
    const dim3 gb(g, bt.n);
    DISPATCH(dtype, (norm2_kernel<double><<<gb, kThreads, 0, st>>>((const double2*)v, n, sc, bt.s)),
             (norm2_kernel<float><<<gb, kThreads, 0, st>>>((const float4*)v, n, sc, bt.s)));
    return SYK_OK;
}

int launch_axpy_norm(int dtype, uint64_t D, void* w, const void* u, int j, LanczosScalars* sc, void* y, int first_y,
                     cudaStream_t st, const Batch& bt) {
    const uint64_t n = n_units(dtype, D);
    const dim3 g(grid_for(n), bt.n);
    if (y) {
        DISPATCH(dtype,
                 (axpy_norm_kernel<double, true><<<g, kThreads, 0, st>>>((double2*)w, (const double2*)u, (double2*)y, n,
                                                                        j, first_y, sc, bt.s)),
                 (axpy_norm_kernel<float, true><<<g, kThreads, 0, st>>>((float4*)w, (const float4*)u, (float4*)y, n, j,
                                                                       first_y, sc, bt.s)));
    } else {
        DISPATCH(dtype,
                 (axpy_norm_kernel<double, false><<<g, kThreads, 0, st>>>((double2*)w, (const double2*)u, nullptr, n, j,
                                                                         0, sc, bt.s)),
                 (axpy_norm_kernel<float, false><<<g, kThreads, 0, st>>>((float4*)w, (const float4*)u, nullptr, n, j, 0,
                                                                        sc, bt.s)));
    }
    return SYK_OK;
}

int launch_finalize_nrm(int j, LanczosScalars* sc, cudaStream_t st, const Batch& bt) {
    finalize_nrm_kernel<<<dim3(1, bt.n), kThreads, 0, st>>>(j, sc, bt.s);
    count_launch();
    SYK_CUDA(cudaGetLastError());
    return SYK_OK;
}

int launch_combine(int dtype, uint64_t D, void* psi, const void* vecs, uint64_t stride_elems, int m,
                   LanczosScalars* sc, cudaStream_t st, const Batch& bt) {
    const uint64_t n = n_units(dtype, D), stride = n_units(dtype, stride_elems);
    const dim3 g(grid_for(n), bt.n);
    DISPATCH(dtype,
             (combine_kernel<double><<<g, kThreads, 0, st>>>((double2*)psi, (const double2*)vecs, stride, n, m, sc, bt.s)),
             (combine_kernel<float><<<g, kThreads, 0, st>>>((float4*)psi, (const float4*)vecs, stride, n, m, sc, bt.s)));
    return SYK_OK;
}

int launch_axpy_coef(int dtype, uint64_t D, void* y, const void* u, int j, int first_y, LanczosScalars* sc,
                     cudaStream_t st) {
    const uint64_t n = n_units(dtype, D);
    const int g = grid_for(n);
    DISPATCH(dtype, (axpy_coef_kernel<double><<<g, kThreads, 0, st>>>((double2*)y, (const double2*)u, n, j, first_y, sc)),
             (axpy_coef_kernel<float><<<g, kThreads, 0, st>>>((float4*)y, (const float4*)u, n, j, first_y, sc)));
    return SYK_OK;
}

int launch_cdot(int dtype, uint64_t D, const void* a, const void* b, LanczosScalars* sc, cudaStream_t st,
                const Batch& bt) {
    const uint64_t n = n_units(dtype, D);
    const int g = grid_for(n);
    const dim3 gb(g, bt.n);
    DISPATCH(dtype, (cdot_kernel<double><<<gb, kThreads, 0, st>>>((const double2*)a, (const double2*)b, n, sc, bt.s)),
             (cdot_kernel<float><<<gb, kThreads, 0, st>>>((const float4*)a, (const float4*)b, n, sc, bt.s)));
    return SYK_OK;
}

int launch_normalise(int dtype, uint64_t D, void* v, LanczosScalars* sc, cudaStream_t st) {
    const uint64_t n = n_units(dtype, D);
    const int g = grid_for(n);
    DISPATCH(dtype, (normalise_kernel<double><<<g, kThreads, 0, st>>>((double2*)v, n, sc)),
             (normalise_kernel<float><<<g, kThreads, 0, st>>>((float4*)v, n, sc)));
    return SYK_OK;
}

// index bit j of a vector stored in the layout of `h` is qubit inv[j]: stored index -> canonical index
static BitPerm to_canonical_perm(const syk_ham* h) {
    BitPerm bp;
    bp.n_bits = 0;
    for (int j = 0; j < 32; ++j) bp.src_bit[j] = (uint8_t)j;
    if (h && !h->identity_layout()) {
        bp.n_bits = h->L;
        for (int q = 0; q < h->L; ++q) bp.src_bit[h->perm[(size_t)q]] = (uint8_t)q;
    }
    return bp;
}

int launch_random_fill(int N, uint64_t seed, uint32_t realization, int dtype, void* psi, LanczosScalars* sc,
                       cudaStream_t st, const syk_ham* layout_of) {
    const uint64_t D = 1ull << (N / 2);
    const uint64_t key = rng_key(seed, realization, kStreamState);
    const int g = grid_for(D);
    const BitPerm bp = to_canonical_perm(layout_of);
    DISPATCH(dtype, (random_fill_kernel<double><<<g, kThreads, 0, st>>>((double2*)psi, D, key, sc, bp)),
             (random_fill_kernel<float><<<g, kThreads, 0, st>>>((float2*)psi, D, key, sc, bp)));
    return SYK_OK;
}

static int launch_gamma_masks(int L, int qbit, uint32_t zmask, int odd, int gamma_norm, int dtype, const void* in, void* out,
                              cudaStream_t st, const Batch& bt) {
    const uint64_t half = 1ull << (L - 1);
    const dim3 g(grid_for(half), bt.n);
    const double s = gamma_norm == SYK_GAMMA_HALF ? 0.70710678118654752440 : 1.0;
    DISPATCH(dtype,
             (gamma_kernel<double><<<g, kThreads, 0, st>>>((const double2*)in, (double2*)out, half, qbit, zmask, odd, s,
                                                          bt.s)),
             (gamma_kernel<float><<<g, kThreads, 0, st>>>((const float2*)in, (float2*)out, half, qbit, zmask, odd,
                                                         (float)s, bt.s)));
    return SYK_OK;
}

int launch_gamma(int N, int n, int gamma_norm, int dtype, const void* in, void* out, cudaStream_t st, const Batch& bt) {
    const int q = n >> 1, odd = n & 1;
    const uint64_t bit = 1ull << q;
    return launch_gamma_masks(N / 2, q, (uint32_t)(odd ? ((bit << 1) - 1) : (bit - 1)), odd, gamma_norm, dtype, in, out, st, bt);
}

// gamma_n on vectors stored in the qubit layout of `h` (h spans the vector: L qubits): the same string with the flipped
// qubit and the Z-mask mapped to index bits
int launch_gamma_h(const syk_ham* h, int n, int dtype, const void* in, void* out, cudaStream_t st, const Batch& bt) {
    const int q = n >> 1, odd = n & 1;
    if (q >= h->L) return SYK_EINVAL;
    const uint64_t bit = 1ull << q;
    const uint64_t zq = odd ? ((bit << 1) - 1) : (bit - 1);
    return launch_gamma_masks(h->L, h->bit_of_qubit(q), (uint32_t)h->to_storage(zq), odd, h->gamma_norm, dtype, in, out, st, bt);
}

int launch_bit_permute(int L, const uint8_t* src_bit, int dtype, const void* in, void* out, cudaStream_t st) {
    BitPerm bp;
    bp.n_bits = L;
    for (int j = 0; j < 32; ++j) bp.src_bit[j] = j < L ? src_bit[j] : (uint8_t)j;
    const uint64_t D = 1ull << L;
    const int g = grid_for(D);
    DISPATCH(dtype, (bit_permute_kernel<double><<<g, kThreads, 0, st>>>((const double2*)in, (double2*)out, D, bp)),
             (bit_permute_kernel<float><<<g, kThreads, 0, st>>>((const float2*)in, (float2*)out, D, bp)));
    return SYK_OK;
}

int permute_vector(const syk_ham* h, int dtype, bool to_layout, const void* in, void* out, cudaStream_t st) {
    uint8_t src[32];
    for (int j = 0; j < 32; ++j) src[j] = (uint8_t)j;
    if (!h->identity_layout()) {
        // to_layout: out[i] = in[canonical(i)], index bit perm[q] <- qubit q;  back: out[b] = in[storage(b)], bit q <- perm[q]
        for (int q = 0; q < h->L; ++q) {
            if (to_layout) src[h->perm[(size_t)q]] = (uint8_t)q;
            else src[q] = h->perm[(size_t)q];
        }
    }
    return launch_bit_permute(h->L, src, dtype, in, out, st);
}

int launch_gamma_block(int N, int n, int gamma_norm, int sector_out, int dtype, const void* in, void* out,
                       cudaStream_t st, const syk_ham* layout_of) {
    if (n < N - 2) {   // string lives on the kept qubits
        if (layout_of) return launch_gamma_h(layout_of, n, dtype, in, out, st);
        return launch_gamma(N - 2, n, gamma_norm, dtype, in, out, st);
    }
    // gamma_{N-2}: (-1)^popcount(b') and gamma_{N-1}: a constant -- both invariant under a relabelling of the kept qubits
    const uint64_t Dr = 1ull << (N / 2 - 1);
    const int g = grid_for(Dr);
    double s = gamma_norm == SYK_GAMMA_HALF ? 0.70710678118654752440 : 1.0;
    const int mode = n - (N - 2);
    if (mode == 1 && sector_out) s = -s;
    DISPATCH(dtype, (gamma_top_kernel<double><<<g, kThreads, 0, st>>>((const double2*)in, (double2*)out, Dr, mode, s)),
             (gamma_top_kernel<float><<<g, kThreads, 0, st>>>((const float2*)in, (float2*)out, Dr, mode, (float)s)));
    return SYK_OK;
}

// Batched inner products: results[r] = <a_r|b_r>; synchronises the stream.
int cdot_batched(int dtype, uint64_t D, const void* a, const void* b, LanczosScalars* sc, const Batch& bt, double* re_im,
                 cudaStream_t st) {
    SYK_TRY(launch_cdot(dtype, D, a, b, sc, st, bt));
    finalize_cdot_kernel<<<dim3(1, bt.n), kThreads, 0, st>>>(sc, bt.s);
    count_launch();
    SYK_CUDA(cudaGetLastError());
    SYK_CUDA(cudaMemcpy2DAsync(re_im, sizeof(double2), (const char*)sc + offsetof(LanczosScalars, coef), bt.s.sc,
                               sizeof(double2), (size_t)bt.n, cudaMemcpyDeviceToHost, st));
    SYK_CUDA(cudaStreamSynchronize(st));
    return SYK_OK;
}

// Sum of the complex partials on the host (fixed order); synchronises the stream.
int fetch_cdot(LanczosScalars* sc, double* re_im, cudaStream_t st) {
    static thread_local std::vector<double2> host;
    int n = 0;
    SYK_CUDA(cudaMemcpyAsync(&n, &sc->n_partial_cdot, sizeof(int), cudaMemcpyDeviceToHost, st));
    SYK_CUDA(cudaStreamSynchronize(st));
    if (n < 0 || n > kMaxPartials) return SYK_ECUDA;
    host.resize((size_t)n);
    SYK_CUDA(cudaMemcpyAsync(host.data(), sc->partial_cdot, sizeof(double2) * (size_t)n, cudaMemcpyDeviceToHost, st));
    SYK_CUDA(cudaStreamSynchronize(st));
    double sr = 0.0, si = 0.0;
    for (int i = 0; i < n; ++i) {
        sr += host[(size_t)i].x;
        si += host[(size_t)i].y;
    }
    re_im[0] = sr;
    re_im[1] = si;
    return SYK_OK;
}

}  // namespace syk

extern "C" {

size_t syk_reduce_scratch_bytes(void) { return (sizeof(syk::LanczosScalars) + 4095) & ~(size_t)4095; }

static bool ok_vec(int N, int dtype, const void* p) {
    return N >= 4 && N <= 64 && (N % 2) == 0 && (dtype == SYK_C64 || dtype == SYK_C128) && p &&
           ((uintptr_t)p & 15) == 0;
}

int syk_apply_gamma_block(int N, int n, int gamma_norm, int sector_out, int dtype, const void* d_in, void* d_out,
                          void* stream) {
    if (N < 6 || N > 66 || (N & 1) || n < 0 || n >= N || (dtype != SYK_C64 && dtype != SYK_C128) || !d_in || !d_out ||
        (gamma_norm != SYK_GAMMA_PAULI && gamma_norm != SYK_GAMMA_HALF) || (sector_out != 0 && sector_out != 1))
        return SYK_EINVAL;
    if (((uintptr_t)d_in & 15) || ((uintptr_t)d_out & 15)) return SYK_EINVAL;
    return syk::launch_gamma_block(N, n, gamma_norm, sector_out, dtype, d_in, d_out, (cudaStream_t)stream);
}

int syk_apply_gamma(int N, int n, int gamma_norm, int dtype, const void* d_in, void* d_out, void* stream) {
    if (!ok_vec(N, dtype, d_in) || !ok_vec(N, dtype, d_out) || n < 0 || n >= N ||
        (gamma_norm != SYK_GAMMA_PAULI && gamma_norm != SYK_GAMMA_HALF))
        return SYK_EINVAL;
    if (d_in != d_out) {   // partial overlap is not allowed
        const size_t bytes = ((size_t)1 << (N / 2)) * syk::elem_bytes(dtype);
        const uintptr_t a = (uintptr_t)d_in, b = (uintptr_t)d_out;
        if (a < b + bytes && b < a + bytes) return SYK_EINVAL;
    }
    return syk::launch_gamma(N, n, gamma_norm, dtype, d_in, d_out, (cudaStream_t)stream);
}

int syk_apply_gamma_h(const syk_ham* h, int n, int dtype, const void* d_in, void* d_out, void* stream) {
    if (!h || h->generic || h->block_of_N || !ok_vec(h->N, dtype, d_in) || !ok_vec(h->N, dtype, d_out) || n < 0 || n >= h->N)
        return SYK_EINVAL;
    if (d_in != d_out) {
        const size_t bytes = ((size_t)1 << h->L) * syk::elem_bytes(dtype);
        const uintptr_t a = (uintptr_t)d_in, b = (uintptr_t)d_out;
        if (a < b + bytes && b < a + bytes) return SYK_EINVAL;
    }
    return syk::launch_gamma_h(h, n, dtype, d_in, d_out, (cudaStream_t)stream);
}

int syk_apply_gamma_block_h(const syk_ham* h_block, int n, int sector_out, int dtype, const void* d_in, void* d_out,
                            void* stream) {
    if (!h_block || h_block->block_of_N < 6 || n < 0 || n >= h_block->block_of_N || (dtype != SYK_C64 && dtype != SYK_C128) ||
        !d_in || !d_out || (sector_out != 0 && sector_out != 1) || ((uintptr_t)d_in & 15) || ((uintptr_t)d_out & 15))
        return SYK_EINVAL;
    return syk::launch_gamma_block(h_block->block_of_N, n, h_block->gamma_norm, sector_out, dtype, d_in, d_out,
                                   (cudaStream_t)stream, h_block);
}

int syk_random_state_h(const syk_ham* h, uint64_t seed, uint32_t realization, int dtype, void* d_psi, void* d_scratch,
                       void* stream) {
    if (!h || h->L > 32 || !ok_vec(2 * h->L, dtype, d_psi) || !d_scratch || ((uintptr_t)d_scratch & 15)) return SYK_EINVAL;
    auto* sc = (syk::LanczosScalars*)d_scratch;
    SYK_TRY(syk::launch_random_fill(2 * h->L, seed, realization, dtype, d_psi, sc, (cudaStream_t)stream, h));
    return syk::launch_normalise(dtype, 1ull << h->L, d_psi, sc, (cudaStream_t)stream);
}

int syk_permute_vector(const syk_ham* h, int dtype, int to_layout, const void* d_in, void* d_out, void* stream) {
    if (!h || h->L > 32 || !ok_vec(2 * h->L, dtype, d_in) || !ok_vec(2 * h->L, dtype, d_out)) return SYK_EINVAL;
    const size_t bytes = ((size_t)1 << h->L) * syk::elem_bytes(dtype);
    const uintptr_t a = (uintptr_t)d_in, b = (uintptr_t)d_out;
    if (a < b + bytes && b < a + bytes) return SYK_EINVAL;
    return syk::permute_vector(h, dtype, to_layout != 0, d_in, d_out, (cudaStream_t)stream);
}

int syk_random_state(int N, uint64_t seed, uint32_t realization, int dtype, void* d_psi, void* d_scratch,
                     void* stream) {
    if (!ok_vec(N, dtype, d_psi) || !d_scratch || ((uintptr_t)d_scratch & 15)) return SYK_EINVAL;
    auto* sc = (syk::LanczosScalars*)d_scratch;
    SYK_TRY(syk::launch_random_fill(N, seed, realization, dtype, d_psi, sc, (cudaStream_t)stream));
    return syk::launch_normalise(dtype, 1ull << (N / 2), d_psi, sc, (cudaStream_t)stream);
}

int syk_dot(int N, int dtype, const void* d_a, const void* d_b, void* d_scratch, double* re_im, void* stream) {
    if (!ok_vec(N, dtype, d_a) || !ok_vec(N, dtype, d_b) || !d_scratch || !re_im) return SYK_EINVAL;
    auto* sc = (syk::LanczosScalars*)d_scratch;
    SYK_TRY(syk::launch_cdot(dtype, 1ull << (N / 2), d_a, d_b, sc, (cudaStream_t)stream));
    return syk::fetch_cdot(sc, re_im, (cudaStream_t)stream);
}

}  // extern "C"
