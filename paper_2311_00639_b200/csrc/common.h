// Internal declarations of libsyk_b200 (not part of the C ABI; see include/syk.h).
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

#include <complex>
#include <vector>

#include "../../include/syk.h"

namespace syk {

// ---------------------------------------------------------------------------------------------------------
// Host tables of one Hamiltonian in canonical order (a-1) and their device copy.
// ---------------------------------------------------------------------------------------------------------
constexpr int kSyncRing = 32;      // epoch counters of the register-tile kernel's lock-step (apply_h_regtile.cu)
struct DeviceTables {
    uint32_t* gx = nullptr;        // [n_groups]    X-mask of each group
    uint32_t* goff = nullptr;      // [n_groups+1]  first term of each group
    uint32_t* tz = nullptr;        // [n_terms]     Z-mask of each term
    double2* tc128 = nullptr;      // [n_terms]     coefficient (re, im), fp64
    float2* tc64 = nullptr;        // [n_terms]     coefficient rounded once to fp32 (R-C64)
    // tile-load lists of the TMA kernel, one per tile size: distinct values of x >> tile_log2 in ascending
    // order, each with the range of groups it serves
    uint32_t* load_hi[2] = {nullptr, nullptr};     // [n_loads]    x >> tile_log2
    uint32_t* load_g0[2] = {nullptr, nullptr};     // [n_loads+1]  first group of each load
    int n_loads[2] = {0, 0};
    uint32_t* sync = nullptr;      // [kSyncRing] epoch counters of the register-tile kernel's lock-step (zeroed per launch)
    int device = -1;
    void* blob = nullptr;          // single allocation holding all of the above
};

}  // namespace syk

namespace syk {
// Term/load table of the register-tile kernel (apply_h_regtile.cu), passed BY VALUE as a __grid_constant__ kernel
// parameter so that every per-term quantity is warp-uniform by construction (constant bank, uniform datapath).
constexpr int kRtMaxTerms = 1024;
constexpr int kRtMaxLoads = 1024;
struct RtTable {
    // term t: .x = tile-local X-mask | (coefficient is imaginary) << 31 ; .y = Z-mask ;
    //         (.z, .w) = bits of the signed magnitude a (double), or .z = bits of (float) a for complex64
    uint4 term[kRtMaxTerms];
    uint32_t load_hi[kRtMaxLoads];         // x >> tile_log2 of each load; the hi == 0 load is LAST
    uint16_t load_t0[kRtMaxLoads + 2];     // first term of each load
    int n_loads;
    int tile_log2;
};
struct RtCache {
    RtTable tab;
    int valid_for = -1;                    // dtype * 64 + tile_log2 the table was built for
};
// Term/load table of the scatter-tile kernel (apply_h_scatter.cu), also a __grid_constant__ parameter.
constexpr int kStMaxTerms = 1024;
constexpr int kStMaxLoads = 1024;
struct StTable {
    // term t: .x = in-slice bits of x (8 / 9 for complex128 / complex64) | (r bits of x) << 9 | (r bits of z) << 16 |
    //         (coefficient is imaginary) << 31 ;
    //         .y = Z-mask ; (.z, .w) = bits of the signed magnitude a (double), or .z = bits of (float) a
    uint4 term[kStMaxTerms];
    uint32_t load_xo[kStMaxLoads];         // x restricted to the outer bit positions, per load (sorted by tile counter)
    uint16_t load_t0[kStMaxLoads + 2];     // first term of each load
    uint32_t dep_r[64];                    // r -> its bits deposited at the tile's r-bit positions
    uint8_t outer_pos[32];                 // outer bit positions, [0] = fastest bit of the tile counter
    uint32_t tile_mask;                    // thread bits | r bits
    int n_loads, n_outer, nr;
};
struct StCache {
    StTable tab;
    bool valid = false;
};
// Device tables of the dense-table kernel (apply_h_dense.cu): one allocation holding loads | groups | terms.
struct DenseCache {
    void* blob = nullptr;
    int device = -1;
    size_t off_groups = 0, off_terms = 0;   // byte offsets of the chunk list and of the entry stream
    int n_loads = 0, n_chunks = 0;
    int n_local_groups = 0;                 // groups applied through a table of 2^popcount(x) values (x-local groups)
    // small vectors: `split` CTAs per tile, each with a range of chunks; partial sums in `partial` ([split][D], owned)
    int split = 1;
    void* partial = nullptr;
    const uint32_t* range = nullptr;
};
}  // namespace syk

struct syk_ham {
    int N = 0;
    int L = 0;
    int gamma_norm = 0;
    // Tables in the STORAGE basis: what every kernel table is built from.  Index bit perm[q] of a stored vector is qubit q
    // (qubit relabelling); with the identity layout they equal the canonical tables below.
    std::vector<uint64_t> x;                   // [n_groups]
    std::vector<uint32_t> group_off;           // [n_groups+1]
    std::vector<uint64_t> z;                   // [n_terms]
    std::vector<std::complex<double>> c;       // [n_terms]
    // Canonical tables (a-1, qubit q = index bit q): what syk_ham_tables exports; fixed at build time.
    std::vector<uint64_t> can_x;               // [n_groups]
    std::vector<uint32_t> can_group_off;       // [n_groups+1]
    std::vector<uint64_t> can_z;               // [n_terms]
    std::vector<std::complex<double>> can_c;   // [n_terms]
    std::vector<int32_t> quartet;              // [n_terms*4]  canonical term order
    std::vector<double> J;                     // [n_terms]    canonical term order
    std::vector<uint8_t> perm;                 // [L] qubit -> index bit of stored vectors; empty = identity
    int block_of_N = 0;                        // parity block (syk_build_parity_block): N of the full Hamiltonian, else 0
    int sector = -1;                           // parity block: 0 even / 1 odd popcount sector
    bool generic = false;                      // built from caller-supplied Pauli strings (no Majorana meaning)
    bool hermitian = true;                     // false: complex couplings / strings with a non-Hermitian coefficient (Arnoldi)
    uint64_t uid = 0;                          // unique per handle (never reused): key of cached CUDA graphs
    mutable uint64_t table_epoch = 0;          // bumped whenever the kernel tables are dropped (layout change)
    int forced_kernel = -1;                    // syk_set_apply_H_kernel
    mutable int dense_representable = -1;      // dense-table kernel: -1 not checked yet, 0 / 1
    mutable syk::DeviceTables dev;             // created on first device use
    mutable syk::RtCache* rt[2] = {nullptr, nullptr};   // register-tile kernel tables per dtype (host, lazily built)
    mutable syk::StCache* st[2] = {nullptr, nullptr};   // scatter-tile kernel tables per dtype (host, lazily built)
    mutable syk::DenseCache* dn[2] = {nullptr, nullptr};   // dense-table kernel tables per dtype (device, lazily built)
    bool identity_layout() const { return perm.empty(); }
    int bit_of_qubit(int q) const { return perm.empty() ? q : (int)perm[(size_t)q]; }
    uint64_t to_storage(uint64_t mask) const {   // a mask over qubits -> the same mask over index bits
        if (perm.empty()) return mask;
        uint64_t r = 0;
        for (int q = 0; q < L; ++q) r |= ((mask >> q) & 1ull) << perm[(size_t)q];
        return r;
    }
    int64_t n_terms() const { return (int64_t)z.size(); }
    int64_t n_groups() const { return (int64_t)x.size(); }
};

namespace syk {

// tile sizes of the TMA kernel (amplitudes per tile), index by dtype (SYK_C64 = 0, SYK_C128 = 1): 16 KiB tiles
constexpr int kTileLog2[2] = {11, 10};
constexpr int kMaxKrylov = 128;
constexpr int kMaxPartials = 4096;            // upper bound on the grid size of any reducing kernel

inline size_t elem_bytes(int dtype) { return dtype == SYK_C128 ? 16 : 8; }

// error plumbing ------------------------------------------------------------------------------------------
void set_cuda_error(cudaError_t e, const char* what);
#define SYK_CUDA(call)                                          \
    do {                                                        \
        cudaError_t e__ = (call);                               \
        if (e__ != cudaSuccess) {                               \
            ::syk::set_cuda_error(e__, #call);                  \
            return SYK_ECUDA;                                   \
        }                                                       \
    } while (0)
#define SYK_TRY(call)                   \
    do {                                \
        int r__ = (call);               \
        if (r__ != SYK_OK) return r__;  \
    } while (0)

void count_launch(int n = 1);
// benchmark timing of apply_H launches (syk_profile_*): no-ops unless enabled
bool profile_enabled();
uint64_t next_handle_uid();
void profile_begin(cudaStream_t st);
void profile_end(cudaStream_t st);
int num_sms();                                 // SM count of the current device (cached); <= 0 on error

// device table management (device_tables.cu)
int ensure_device_tables(const syk_ham* h);
void free_device_tables(const syk_ham* h);

// ---------------------------------------------------------------------------------------------------------
// Scalars of a Lanczos run, resident on the device (a-3): everything the fused kernels need between steps.
// ---------------------------------------------------------------------------------------------------------
struct LanczosScalars {
    double alpha[kMaxKrylov + 2];   // alpha[j], j = 1..m
    double nrm[kMaxKrylov + 2];     // nrm[j] = |u_j|, u_1 = psi, u_{j+1} = w - alpha_j v_j  (nrm[j+1] = beta_{j+1})
    double2 coef[kMaxKrylov + 2];   // coef[j] = [exp(-i tau T_m) e_1]_j * nrm[1], uploaded by the host
    double partial_dot[kMaxPartials];   // per-CTA partial sums of Re<u_j|w> written by apply_H
    double partial_nrm[kMaxPartials];   // per-CTA partial sums of |.|^2 written by the vector kernels
    double2 partial_cdot[kMaxPartials]; // per-CTA partial sums of a complex dot product
    int n_partial_dot;              // how many entries of partial_dot are valid
    int n_partial_nrm;
    int n_partial_cdot;
    int m_eff;                      // batched combine: effective Krylov dimension of this realization
};

// What the fused epilogue of apply_H does (all pointers device):
//   plain : out[b] = acc
//   fused : out[b] = acc / nrm[j] - (nrm[j]/nrm[j-1]) prev[b]   (second term absent when j == 1)
//           and partial_dot[cta] = sum_b Re(conj(in[b]) out[b]);
//           nrm[j] is first reduced from partial_nrm (written by the preceding vector kernel).
struct FusedArgs {
    LanczosScalars* sc = nullptr;   // nullptr = plain
    const void* prev = nullptr;     // u_{j-1}; may alias out; nullptr when j == 1
    int j = 0;
    unsigned long long* trace = nullptr;   // scatter-tile kernel only: timeline of one CTA (syk_apply_H_trace)
    int trace_cta = 0, trace_round = 0, trace_detail = 0;
};

// register-tile kernel (apply_h_regtile.cu): 0 if the handle cannot use it, else the tile_log2 it would use
int regtile_tile_log2(const syk_ham* h, int dtype, bool forced);
int launch_apply_h_regtile(const syk_ham* h, int dtype, const void* d_in, void* d_out, const FusedArgs& fa,
                           cudaStream_t stream);
void free_regtile_tables(const syk_ham* h);
void set_lockstep(int epoch_len, int lag);
void get_lockstep(int* epoch_len, int* lag);

// scatter-tile kernel (apply_h_scatter.cu)
int scatter_tile_log2(const syk_ham* h, int dtype, bool forced);
int launch_apply_h_scatter(const syk_ham* h, int dtype, const void* d_in, void* d_out, const FusedArgs& fa,
                           cudaStream_t stream);
int scatter_trace(const syk_ham* h, int dtype, const void* d_in, void* d_out, int cta, int round, int detail, uint64_t* clk,
                  int clk_capacity, int32_t* load_terms, uint32_t* load_xo, int load_capacity, int* n_loads, int* rot,
                  cudaStream_t stream);
int scatter_layout_info(const syk_ham* h, int dtype, int* n_loads, int* n_passes, uint32_t* tile_mask,
                        uint32_t* window_mask);
void free_scatter_tables(const syk_ham* h);
int scatter_tile_bits(int dtype);      // index bits of one tile (13 complex128 / 14 complex64)
int scatter_window_bits();             // ~log2(tiles in flight)

// dense-table kernel (apply_h_dense.cu)
bool dense_kernel_ok(const syk_ham* h, bool forced);
int launch_apply_h_dense(const syk_ham* h, int dtype, const void* d_in, void* d_out, const FusedArgs& fa,
                         cudaStream_t stream);
void free_dense_tables(const syk_ham* h);
int prepare_dense_tables(const syk_ham* h, int dtype);   // builds / uploads the device table and the split scratch
int dense_tables_info(const syk_ham* h, int dtype, int* n_loads, int* n_chunks, int* split, int* n_local_groups);

// apply_H launcher shared by syk_apply_H and the Krylov driver (apply_h.cu)
int launch_apply_h(const syk_ham* h, int dtype, const void* d_in, void* d_out, const FusedArgs& fa,
                   cudaStream_t stream);

// Batched launches over disorder realizations (grid.y = realization): pointer argument k of realization r is
// base_k + r * stride_k bytes (a, b, c in the launcher's argument order), its LanczosScalars base + r * sc bytes.
struct BatchStride { size_t a = 0, b = 0, c = 0, sc = 0; };
struct Batch {
    int n = 1;
    BatchStride s;
};

// batched apply_H over realizations with the 16 KiB-tile kernel (apply_h.cu): d_tab = device array of
// batched_table_bytes(nb) bytes that receives the per-realization table descriptors when `upload` is set
size_t batched_table_bytes(int nb);
bool batched_apply_ok(const syk_ham* const* hams, int nb, int dtype);
int launch_apply_h_batched(const syk_ham* const* hams, int nb, int dtype, void* d_tab, bool upload, const void* in,
                           size_t s_in, void* out, size_t s_out, const void* prev, size_t s_prev, void* sc, size_t s_sc,
                           int j, cudaStream_t stream);

// vector kernels (vector_ops.cu); all reductions go through LanczosScalars partial arrays
int launch_norm2(int dtype, uint64_t D, const void* d_v, LanczosScalars* sc, cudaStream_t stream,
                 const Batch& bt = Batch());
// u_next = w - (alpha_j / nrm[j]) u_j in place on w, |u_next|^2 partials; alpha_j reduced from partial_dot.
// When y != nullptr also y = y_scale * y + (coef[j]/nrm[j]) u_j  with y_scale = coef[1]/nrm[1] if first_y else 1.
int launch_axpy_norm(int dtype, uint64_t D, void* d_w, const void* d_u, int j, LanczosScalars* sc, void* d_y,
                     int first_y, cudaStream_t stream, const Batch& bt = Batch());   // strides: w, u, y
// finalises nrm[j] from partial_nrm (used after the last vector kernel of a run); 1 block
int launch_finalize_nrm(int j, LanczosScalars* sc, cudaStream_t stream, const Batch& bt = Batch());
// psi = sum_{j=1..m} (coef[j]/nrm[j]) u_j, u_1 = psi itself (in place), u_j (j >= 2) = vecs + (j-2)*stride_elems
int launch_combine(int dtype, uint64_t D, void* d_psi, const void* d_vecs, uint64_t stride_elems, int m,
                   LanczosScalars* sc, cudaStream_t stream, const Batch& bt = Batch());   // m < 0: sc->m_eff; strides: psi, vecs
// y = ys*y + (coef[j]/nrm[j]) u, ys = first_y ? coef[1]/nrm[1] : 1; u == nullptr drops the second term
int launch_axpy_coef(int dtype, uint64_t D, void* d_y, const void* d_u, int j, int first_y, LanczosScalars* sc,
                     cudaStream_t stream);
int launch_cdot(int dtype, uint64_t D, const void* d_a, const void* d_b, LanczosScalars* sc, cudaStream_t stream,
                const Batch& bt = Batch());
int fetch_cdot(LanczosScalars* sc, double* re_im, cudaStream_t stream);   // host sum of the partials; synchronises
int cdot_batched(int dtype, uint64_t D, const void* d_a, const void* d_b, LanczosScalars* sc, const Batch& bt,
                 double* re_im /* [bt.n][2] */, cudaStream_t stream);
int launch_normalise(int dtype, uint64_t D, void* d_v, LanczosScalars* sc, cudaStream_t stream);
int launch_gamma(int N, int n, int gamma_norm, int dtype, const void* d_in, void* d_out, cudaStream_t stream,
                 const Batch& bt = Batch());
// gamma_n in the storage basis of `h` (a full-space handle, or a parity block for n < N_full - 2): the Jordan-Wigner string
// with its masks mapped through the handle's qubit layout
int launch_gamma_h(const syk_ham* h, int n, int dtype, const void* d_in, void* d_out, cudaStream_t stream,
                   const Batch& bt = Batch());
// out[i] = in[sigma(i)], sigma = the bit permutation that moves index bit j to bit src_bit[j]
int launch_bit_permute(int L, const uint8_t* src_bit, int dtype, const void* d_in, void* d_out, cudaStream_t stream);
// canonical -> storage basis of h (to_layout) or back; in != out
int permute_vector(const syk_ham* h, int dtype, bool to_layout, const void* d_in, void* d_out, cudaStream_t stream);
// drops every cached kernel table of the handle (after a change of layout)
void invalidate_kernel_tables(const syk_ham* h);
// gamma_n of the FULL space (N Majoranas) between parity blocks on N/2-1 qubits; the result lies in sector_out
int launch_gamma_block(int N, int n, int gamma_norm, int sector_out, int dtype, const void* d_in, void* d_out,
                       cudaStream_t stream, const syk_ham* layout_of = nullptr);
int launch_random_fill(int N, uint64_t seed, uint32_t realization, int dtype, void* d_psi, LanczosScalars* sc,
                       cudaStream_t stream, const syk_ham* layout_of = nullptr);
int apply_h_kernel_kind(const syk_ham* h, int dtype);

// Krylov driver internals shared with the OTOC pipeline (krylov.cu)
int krylov_evolve_impl(const syk_ham* h, int dtype, void* d_psi, double tau_re, double tau_im,
                       const syk_krylov_opts* opts, void* d_work, size_t work_bytes, syk_stats* stats,
                       cudaStream_t stream);
size_t krylov_header_bytes();
size_t krylov_batched_bytes(const syk_ham* h0, int nb, int dtype, int m);
int krylov_evolve_batched_impl(const syk_ham* const* hams, int nb, int dtype, void* d_psi, size_t psi_stride_bytes,
                               double tau_re, double tau_im, const syk_krylov_opts* opts, void* d_work,
                               size_t work_bytes, syk_stats* stats, bool* tables_uploaded, cudaStream_t stream);
int resolve_krylov_dim(const syk_ham* h, const syk_krylov_opts* o);
void set_graphs(int on);
// the same call for a non-Hermitian operator: Arnoldi + host exponential of the Hessenberg matrix (arnoldi.cu)
int arnoldi_evolve_impl(const syk_ham* h, int dtype, void* d_psi, double tau_re, double tau_im, const syk_krylov_opts* opts,
                        void* d_work, size_t work_bytes, syk_stats* stats, cudaStream_t stream);

// ---------------------------------------------------------------------------------------------------------
// The counter-based generator R-RNG, host and device.
// ---------------------------------------------------------------------------------------------------------
#ifdef __CUDACC__
#define SYK_HD __host__ __device__ __forceinline__
#else
#define SYK_HD inline
#endif
constexpr uint64_t kGold = 0x9E3779B97F4A7C15ull;
SYK_HD uint64_t rng_fmix(uint64_t z) {
    z ^= z >> 30; z *= 0xBF58476D1CE4E5B9ull;
    z ^= z >> 27; z *= 0x94D049BB133111EBull;
    z ^= z >> 31;
    return z;
}
SYK_HD uint64_t rng_absorb(uint64_t h, uint64_t w) { return rng_fmix((h ^ w) + kGold); }
SYK_HD uint64_t rng_key(uint64_t seed, uint64_t realization, uint64_t stream) {
    return rng_absorb(rng_absorb(rng_absorb(0, seed), realization), stream);
}
SYK_HD uint64_t rng_draw(uint64_t key, uint64_t index, uint64_t d) {
    return rng_absorb(rng_absorb(key, index), d) >> 11;
}
constexpr uint64_t kStreamHamiltonian = 1, kStreamState = 2;

}  // namespace syk
