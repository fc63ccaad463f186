/* syk.h -- C ABI of libsyk_b200: the data-parallel hot path of the sparse-SYK OTOC method of
 * arXiv 2311.00639 on one NVIDIA B200 (sm_100a).
 *
 * Citations "PAPER.md:<line>" refer to the paper text; "R-xxx" to the readings listed in DESIGN.md section 2.
 *
 * Conventions common to every call
 *   - Every function returns an int: SYK_OK (0) or a negative error code.  Nothing throws, prints or exits.
 *   - N = number of Majorana fermions, even, 4 <= N <= 64.  L = N/2 qubits, D = 2^L amplitudes.  (N = 66 can be built
 *     and cut into parity blocks of 32 qubits, which every call accepts; the full N = 66 handle itself only serves
 *     syk_ham_info / syk_ham_tables / syk_build_parity_block.)
 *   - A state vector is a contiguous array of D complex numbers, interleaved (re, im); `dtype` says whether the
 *     components are float (SYK_C64, 8 bytes per amplitude) or double (SYK_C128, 16 bytes per amplitude).
 *     Basis index b = sum_q bit_q 2^q, qubit 0 = least significant bit (R-ENDIAN).
 *   - Pointers named d_* are DEVICE pointers owned by the caller, 16-byte aligned; pointers named h_* and all
 *     other pointers are HOST pointers.  The library never allocates device vectors: work space is passed in
 *     (the memory discipline is part of the method).  The only device memory the library
 *     owns belongs to a handle and is released by syk_free_hamiltonian: the term table (a few KB for sparse H,
 *     <= ~8 MB for dense N=48) and, for the dense-table kernel on vectors with fewer tiles than SMs, a scratch
 *     buffer of partial sums (<= 64 vectors of <= 2^19 amplitudes).  syk_ham_prepare allocates and uploads all
 *     of it; after that no compute call allocates.  A handle that was not prepared does the same lazily inside
 *     its first compute call (one synchronous cudaMalloc + copy).  (The CUDA graphs of the latency path for small
 *     vectors, syk_set_cuda_graphs, are instantiated by the driver on first use, which may take device memory of its own.)
 *   - A handle is not thread-safe and must not be used by two launches that are in flight at the same time
 *     (different streams or threads): the lazily built table caches, the split scratch and the pacing counters
 *     of the tile kernels belong to the handle.  Different handles are independent.
 *   - `stream` is a cudaStream_t passed as void* (NULL = default stream).  Calls enqueue work and return, except
 *     where they hand back host scalars (syk_krylov_evolve, syk_otoc, syk_lanczos_run, *_host): those
 *     synchronise that stream only.
 *   - There is no CPU fallback: a compute call on a machine without a CUDA device returns SYK_ECUDA.
 *   - Results are bitwise reproducible run to run on the same GPU model: no atomics on data, fixed reduction trees
 *     (per-CTA partial sums and, in the large-vector kernel, a per-CTA order of the terms: both fixed by the SM count).
 */
#ifndef SYK_B200_H
#define SYK_B200_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

enum { SYK_OK = 0,
       SYK_EINVAL = -1,   /* bad argument: N odd / out of range, p outside (0,1], index >= N, i == j, null or
                             unaligned pointer, in == out where forbidden, unsorted quartet or t_grid */
       SYK_ENOMEM = -2,   /* work space too small (ask the *_workspace_bytes query) or host allocation failed */
       SYK_ECUDA = -3,    /* CUDA runtime error or no device; text via syk_last_cuda_error() */
       SYK_ENOCONV = -4,  /* Krylov sub-step limit reached; the result is written, stats->err_est says how bad */
       SYK_ELIMIT = -5    /* size beyond the fixed device scratch of a *_static entry point (syk_dot_static_max_N) */ };

enum { SYK_C64 = 0, SYK_C128 = 1 };
enum { SYK_GAMMA_PAULI = 0,  /* gamma_n = Pauli string, {g_m,g_n} = 2 delta; benchmark default */
       SYK_GAMMA_HALF = 1    /* gamma_n = Pauli string / sqrt(2), {g_m,g_n} = delta; R-NORM      */ };

typedef struct syk_ham syk_ham;   /* opaque, library-owned: host term tables + lazily created device copy */

const char* syk_strerror(int code);
const char* syk_last_cuda_error(void);           /* text of the last CUDA error seen by this thread ("" if none) */
int syk_version(void);

/* ------------------------------------------------------------------------------------------------------------
 * a-1  Term compiler (host).  Eq. (1); <bits, coeff> encoding PAPER.md:257-267; operator
 *      product and sum PAPER.md:299.
 *
 * syk_build_hamiltonian samples H = sum_{i<j<k<l} p_ijkl J_ijkl g_i g_j g_k g_l: each quartet (lexicographic rank
 * r) is kept with probability p and gets J ~ N(0, 3/(8 p N^3)) from the counter-based generator R-RNG keyed
 * (seed, realization, r).  Each kept quartet becomes one Pauli string c Z^z X^x (Jordan-Wigner, R-JW; acting as
 * (O v)[b] = c (-1)^popcount(b & z) v[b xor x], R-SIGN) with c = J s^4 times a phase in {1,-1,i,-i}; strings
 * are grouped by X-mask; canonical order: groups by ascending x, terms inside a group by ascending z.
 * syk_build_from_terms does the same for caller-supplied quartets (each i<j<k<l, all distinct) and couplings.
 * *out receives a new handle; release it with syk_free_hamiltonian.  No device is needed for these calls.
 */
int syk_build_hamiltonian(int N, double p, uint64_t seed, uint32_t realization, int gamma_norm, syk_ham** out);
int syk_build_from_terms(int N, int64_t n_terms, const int32_t* quartets /* [n_terms][4] */,
                         const double* J /* [n_terms] */, int gamma_norm, syk_ham** out);
/* Generic sum of Pauli strings on L qubits (2 <= L <= 32; spin chains, Ising-type models and
 * non-Hermitian operators through the same operator action).  String t is c_t Z^{z_t} X^{x_t} acting as
 * (O v)[b] = c_t (-1)^popcount(b & z_t) v[b xor x_t] (R-SIGN; Y = -i Z X), c_t any finite complex number.  Equal (x, z)
 * are combined.  A string is Hermitian iff c_t is real when popcount(x_t & z_t) is even and imaginary when it is odd; if
 * every string is, the handle is Hermitian and evolves by Lanczos, otherwise it is NON-HERMITIAN: syk_apply_H works as
 * for any handle (strings whose coefficient is neither real nor imaginary use the generic / 16 KiB-tile kernels),
 * syk_krylov_evolve runs the Arnoldi process with the exponential of the m x m Hessenberg matrix on the host (one-pass
 * only: two_pass -> SYK_EINVAL), syk_lanczos_run and the batched lock-step calls return SYK_EINVAL.  The handle works with
 * syk_apply_H, syk_krylov_evolve and the work-space queries (dim = 2^L; syk_ham_info reports N = 2L); the Majorana calls
 * (syk_otoc, syk_green, syk_build_parity_block) reject it. */
int syk_build_from_pauli_strings(int L, int64_t n_terms, const uint64_t* x, const uint64_t* z, const double* c_re_im,
                                 syk_ham** out);
/* syk_build_from_terms with COMPLEX couplings J_t = J_re_im[t][0] + i J_re_im[t][1]: the non-Hermitian SYK model named in
 * PAPER.md:108.  It is Hermitian iff all imaginary parts are zero; a non-Hermitian handle works with syk_apply_H,
 * syk_krylov_evolve (Arnoldi), syk_build_parity_block and the layout calls, while syk_otoc / syk_green (defined through
 * thermal factors of a Hermitian H) return SYK_EINVAL.  syk_ham_tables reports Re J in J_of_term; the coefficients c carry the full coupling. */
int syk_build_from_terms_complex(int N, int64_t n_terms, const int32_t* quartets /* [n_terms][4] */,
                                 const double* J_re_im /* [n_terms][2] */, int gamma_norm, syk_ham** out);
/* 1 if the handle is Hermitian (Lanczos), 0 if not (Arnoldi). */
int syk_ham_is_hermitian(const syk_ham* h);
void syk_free_hamiltonian(syk_ham* h);

/* Sizes: any output pointer may be NULL. dim = 2^(N/2). */
int syk_ham_info(const syk_ham* h, int* N, int64_t* n_terms, int64_t* n_xmasks, int64_t* dim);

/* Copies the canonical tables to caller arrays (any may be NULL): x[n_xmasks], group_off[n_xmasks+1],
 * z[n_terms], c_re_im[n_terms][2], quartet_of_term[n_terms][4], J_of_term[n_terms]. */
int syk_ham_tables(const syk_ham* h, uint64_t* x, uint32_t* group_off, uint64_t* z, double* c_re_im,
                   int32_t* quartet_of_term, double* J_of_term);

/* ------------------------------------------------------------------------------------------------------------
 * Qubit layout of a handle (the fewer and the more local the terms, the cheaper
 * Algorithm 1).  Which qubit sits on which bit of the basis index is physically free -- a relabelling of the Jordan-
 * Wigner qubits is a permutation of the basis -- but it decides how often the tile kernels of apply_H move the vector:
 * once from L2 into the SMs per distinct X-mask outside the low "tile" bits, once from DRAM per distinct X-mask outside
 * tile + "window" bits.  A handle therefore carries a layout perm[q] = index bit of qubit q (identity after a build).
 *   syk_ham_optimize_layout : chooses perm for the tile geometry of `dtype` (deterministic hill climbing on
 *                             loads + 2 passes over the partition of the qubits into tile / window / rest) and sets it;
 *                             Hamiltonians with more than 1024 terms keep the identity.
 *   syk_ham_set_layout      : sets a caller-chosen permutation (NULL = identity).  SYK_EINVAL if perm is not one.
 *   syk_ham_layout          : exports perm[N/2] and whether it is the identity.
 * Setting a layout rewrites the handle's kernel tables (every string c Z^z X^x becomes c Z^{Pz} X^{Px}) and drops its
 * device copies: do it before syk_ham_prepare and before any vector exists.  The CANONICAL tables exported by
 * syk_ham_tables never change.  From then on every DEVICE vector passed with this handle (syk_apply_H, syk_lanczos_run,
 * syk_krylov_evolve, syk_otoc, syk_green, ...) is stored in the handle's layout: amplitude of basis state b at index
 * sum_q bit_q(b) 2^perm[q].  The calls below produce / convert such vectors; the *_host entry points take canonical host
 * vectors and convert on the device; results that do not depend on the basis (F(t), G(t), Lanczos coefficients, dots)
 * are the same in every layout up to rounding order.  The two parity blocks of a Hamiltonian must share one layout.
 */
int syk_ham_optimize_layout(syk_ham* h, int dtype);
int syk_ham_set_layout(syk_ham* h, const int32_t* perm /* [N/2] or NULL */);
int syk_ham_layout(const syk_ham* h, int32_t* perm /* [N/2], may be NULL */, int* is_identity /* may be NULL */);
/* d_out = the vector d_in converted from the canonical basis to the handle's layout (to_layout != 0) or back; d_in and
 * d_out must not overlap. */
int syk_permute_vector(const syk_ham* h, int dtype, int to_layout, const void* d_in, void* d_out, void* stream);
/* syk_random_state / syk_apply_gamma / syk_apply_gamma_block for vectors in the layout of a handle: the same physical
 * state / operator (the Haar-random amplitude of canonical basis state b lands on its stored index; the Jordan-Wigner
 * string of gamma_n has its masks mapped through perm).  syk_random_state_h and syk_permute_vector accept any handle,
 * syk_apply_gamma_h a full-space Majorana handle, syk_apply_gamma_block_h a parity block (N, gamma_norm taken from it). */
int syk_random_state_h(const syk_ham* h, uint64_t seed, uint32_t realization, int dtype, void* d_psi, void* d_scratch,
                       void* stream);
int syk_apply_gamma_h(const syk_ham* h, int n, int dtype, const void* d_in, void* d_out, void* stream);
int syk_apply_gamma_block_h(const syk_ham* h_block, int n, int sector_out, int dtype, const void* d_in, void* d_out,
                            void* stream);

/* Creates the device copy of the term tables of `h` on the current device for `dtype` (and, for the dense-table
 * kernel, its entry stream and split scratch): after this call syk_apply_H / syk_lanczos_run / syk_krylov_evolve /
 * syk_otoc / syk_green on this handle and dtype allocate nothing (few allocation calls).  Synchronous
 * (cudaMalloc + cudaMemcpy).  Call again after syk_set_apply_H_kernel or after switching devices. */
int syk_ham_prepare(const syk_ham* h, int dtype);

/* ------------------------------------------------------------------------------------------------------------
 * a-2  apply_H (device).  Algorithm 1, in gather form:
 *        out[b] = sum_g in[b xor x_g] * sum_{t in g} c_t (-1)^popcount(b & z_t),      0 <= b < D.
 * d_in and d_out are distinct, non-overlapping device vectors of `dtype`.  SYK_C64 multiplies and accumulates
 * in fp32 (R-C64), SYK_C128 in fp64.  An empty Hamiltonian (no terms) gives out = 0.
 */
int syk_apply_H(const syk_ham* h, int dtype, const void* d_in, void* d_out, void* stream);

/* Batched over disorder realizations: n_batch handles with the same N; vector r of the batch
 * starts at element offset r*batch_stride (batch_stride >= D) of d_in / d_out. */
int syk_apply_H_batched(const syk_ham* const* hams, int n_batch, int dtype, const void* d_in, void* d_out,
                        int64_t batch_stride, void* stream);

/* The same product with HOST vectors: copies h_in to the device work space, applies H, copies the result to
 * h_out; synchronises.  d_work must hold 2*D amplitudes of `dtype`. */
int syk_apply_H_host(const syk_ham* h, int dtype, const void* h_in, void* h_out, void* d_work, size_t work_bytes,
                     void* stream);

/* out = gamma_n in (one Pauli string: flip qubit n/2, sign from the lower qubits, R-JW).
 * d_out may equal d_in (in place). */
int syk_apply_gamma(int N, int n, int gamma_norm, int dtype, const void* d_in, void* d_out, void* stream);

/* ------------------------------------------------------------------------------------------------------------
 * a-5 (input)  Normalised complex Gaussian ("Haar-random") state from R-RNG stream 2, written to
 * d_psi.  d_scratch: at least syk_reduce_scratch_bytes() bytes of device memory. */
size_t syk_reduce_scratch_bytes(void);
int syk_random_state(int N, uint64_t seed, uint32_t realization, int dtype, void* d_psi, void* d_scratch,
                     void* stream);

/* <a|b> = sum conj(a[k]) b[k] in fp64 (deterministic); synchronises; result to host re_im[2]. */
int syk_dot(int N, int dtype, const void* d_a, const void* d_b, void* d_scratch, double* re_im, void* stream);

/* The same inner product for callers that cannot allocate or synchronise (CUDA graph capture, serving loops, harnesses
 * that forbid cudaMalloc): d_result[0..1] (DEVICE memory, 8-byte aligned) <- (Re, Im) <a|b>, by two kernel launches on
 * `stream`; no scratch argument, no cudaMalloc / cudaFree / allocating routine, no synchronisation, no host copy.  The
 * per-CTA partial sums live in one file-scope __device__ array of 64 KiB that every GPU loading the library holds until
 * exit; its device address is resolved once per device (syk_dot_static_prepare, or the first call on that device: call
 * prepare before starting a capture).  Limit: 2^25 16-byte units, i.e. N <= syk_dot_static_max_N(dtype) = 50 (complex128) /
 * 52 (complex64); larger N returns SYK_ELIMIT and launches nothing.  Every CTA sums a fixed stretch of the vector, so the
 * result depends on the data only (bitwise equal on every GPU; equal to syk_dot to rounding).  All calls of a process on a
 * device SHARE the array: calls that overlap on the GPU (two streams, independent graph branches) race and give wrong
 * results -- order them.  Nothing in the array needs clearing between calls. */
int syk_dot_static_max_N(int dtype);
int syk_dot_static_prepare(void);
int syk_dot_static(int N, int dtype, const void* d_a, const void* d_b, double* d_result, void* stream);

/* ------------------------------------------------------------------------------------------------------------
 * a-3 / a-4  Lanczos and the Krylov exponential, PAPER.md:301 ("restarted Krylov subspace method for
 * exp(-iHt)|Psi>"), R-KRYLOV.
 *
 * syk_lanczos_run: m steps of the Hermitian Lanczos recurrence from v_1 = psi/|psi| with the fused kernels
 * (apply_H with the -beta_j v_{j-1} term and the <v_j|w> partial sums fused; then w - alpha_j v_j with |.|^2
 * fused; scalars stay on the device between steps).  Outputs (host): alpha[m], beta[m+1] with beta[0] = |psi|
 * and beta[j] (j>=1) the off-diagonal element / residual norm after step j.  d_psi is not modified.  Work
 * space: syk_krylov_workspace_bytes with two_pass = 0 and krylov_dim = m.  Synchronises.
 */
typedef struct {
    int krylov_dim;     /* m: Lanczos steps per sub-step (2..128); 0 = default 24 */
    double tol;         /* relative error target for the whole call; 0 = default 1e-12 (C128) / 1e-6 (C64) */
    int two_pass;       /* 0: store the m Lanczos vectors (m work vectors); 1: two-pass Lanczos (2 work vectors) */
    int max_substeps;   /* 0 = default 100000 */
    int renormalize;    /* 1: carry the norm separately: every sub-step rescales its result to the norm
                           of its input, so |psi| is unchanged by the call and stats->log_norm receives
                           ln(|exp(-i tau H) psi| / |psi|); the true result is exp(log_norm) times the returned vector.
                           Needed in complex64 for imaginary times whose growth exp(-beta E_0) leaves the fp32 range
                           (PAPER.md:363 runs beta = 20 in single precision).  0: the result carries its norm. */
} syk_krylov_opts;

typedef struct {
    int64_t n_matvec;   /* apply_H launches */
    int n_substeps;     /* time sub-steps taken */
    int krylov_dim_used;/* smallest effective m over sub-steps (happy breakdown shortens it) */
    double err_est;     /* accumulated a-posteriori error estimate, relative */
    double model_bytes; /* bytes the byte model of DESIGN.md section 6 attributes to the call */
    double elapsed_ms;  /* device time of the call (CUDA events on `stream`) */
    double log_norm;    /* opts->renormalize: ln of the factor taken out of the result (summed over sub-steps); else 0 */
} syk_stats;

int syk_krylov_workspace_bytes(const syk_ham* h, int dtype, const syk_krylov_opts* opts, size_t* bytes);

int syk_lanczos_run(const syk_ham* h, int dtype, const void* d_psi, int m, double* alpha, double* beta,
                    void* d_work, size_t work_bytes, syk_stats* stats, void* stream);

/* psi <- exp(-i (tau_re + i tau_im) H) psi, in place (R-TAU).  Real time t: (t, 0).  exp(-beta H/4): (0, -beta/4).
 * exp(-(it + beta/4)H): (t, -beta/4).  The result is NOT renormalised.  opts/stats may be NULL. */
int syk_krylov_evolve(const syk_ham* h, int dtype, void* d_psi, double tau_re, double tau_im,
                      const syk_krylov_opts* opts, void* d_work, size_t work_bytes, syk_stats* stats, void* stream);

/* Lock-step batched evolution: psi_r <- exp(-i tau H_r) psi_r for r < n_batch, psi_r at d_psi + r*batch_stride elements.
 * Same conditions as the lock-step mode of syk_otoc_batched (else SYK_EINVAL); opts->two_pass must be 0.  Work space:
 * syk_krylov_workspace_bytes_batched.  stats: n_matvec counts realization-matvecs, n_substeps the rounds, err_est the
 * largest per-realization estimate. */
int syk_krylov_workspace_bytes_batched(const syk_ham* h, int n_batch, int dtype, const syk_krylov_opts* opts,
                                       size_t* bytes);
int syk_krylov_evolve_batched(const syk_ham* const* hams, int n_batch, int dtype, void* d_psi, int64_t batch_stride,
                              double tau_re, double tau_im, const syk_krylov_opts* opts, void* d_work, size_t work_bytes,
                              syk_stats* stats, void* stream);

/* Same with a HOST vector (in/out): d_work must hold one extra vector in front of the Krylov work space, i.e.
 * D*elem_bytes + syk_krylov_workspace_bytes(). */
int syk_krylov_evolve_host(const syk_ham* h, int dtype, void* h_psi, double tau_re, double tau_im,
                           const syk_krylov_opts* opts, void* d_work, size_t work_bytes, syk_stats* stats,
                           void* stream);

/* ------------------------------------------------------------------------------------------------------------
 * a-5  Regularised OTOC, PAPER.md:230 (R-EQ2, R-WV, R-F):
 *   F(t) = <psi| e^{(it-b/8)H} g_W e^{-(it+b/4)H} g_V e^{(it-b/4)H} g_W e^{-(it+b/4)H} g_V e^{-bH/8} |psi>
 * for t in t_grid (non-decreasing, >= 0), W = gamma_{i_W}, V = gamma_{j_V}, b = beta >= 0.  F_out[n_t][2] (host)
 * receives the un-normalised complex values; OTOC(t) = F(t)/F(0) is the caller's division.
 * d_psi is used as work space and destroyed.  Work space: syk_otoc_workspace_bytes (2 vectors + Krylov work).
 * stats (may be NULL) accumulates over all evolutions. */
int syk_otoc_workspace_bytes(const syk_ham* h, int dtype, const syk_krylov_opts* opts, size_t* bytes);
int syk_otoc(const syk_ham* h, int dtype, int i_W, int j_V, double beta, const double* t_grid, int n_t,
             void* d_psi, double* F_out, const syk_krylov_opts* opts, void* d_work, size_t work_bytes,
             syk_stats* stats, void* stream);

/* Retarded Green function:  G(t) = <psi| e^{(it-b/2)H} g_n e^{-iHt} g_n e^{-bH/2} |psi>  for t in
 * t_grid (non-decreasing, >= 0); G_out[n_t][2] (host) receives the un-normalised complex values, G_R(t) =
 * Re G(t)/G(0) is the caller's division.  Same work space, ownership and error rules as syk_otoc (d_psi is
 * destroyed; syk_otoc_workspace_bytes). */
int syk_green(const syk_ham* h, int dtype, int n, double beta, const double* t_grid, int n_t, void* d_psi,
              double* G_out, const syk_krylov_opts* opts, void* d_work, size_t work_bytes, syk_stats* stats,
              void* stream);

/* ------------------------------------------------------------------------------------------------------------
 * Parity blocks, PAPER.md:220-247 (reading R-BLOCK of DESIGN.md).  H commutes with the fermion
 * parity Z^{(x)L}: H = H_UU (+) H_DD with sector 0 = even, 1 = odd popcount of the basis index.  A block acts on
 * D/2 = 2^(L-1) amplitudes: reduced index b' = low L-1 bits of b, the dropped top bit is parity(b') xor sector.
 *
 * syk_build_parity_block: the block of a FULL handle (N >= 6) as a handle of its own on L-1 qubits -- every call that
 * takes a handle (syk_apply_H, syk_lanczos_run, syk_krylov_evolve, work-space queries, ...) works on it with vectors
 * of D/2 amplitudes; syk_ham_info reports N-2 and D/2; quartet_of_term / J_of_term still name the original quartets.
 * syk_apply_gamma_block: gamma_n of the full space (0 <= n < N) as a map from sector 1-sector_out to sector_out on
 * reduced vectors (in place allowed); gamma_{N-2} is a diagonal sign and gamma_{N-1} = -/+ i s 1: no gather
 * (PAPER.md:238-242).  syk_otoc_block / syk_green_block: the term of F(t) / G(t) (PAPER.md:232 / 220) that starts
 * from the reduced state d_psi in `sector`; the full-space value for psi = psi_U (+) psi_D is the sum of the two
 * sectors' results.  Same work space (syk_otoc_workspace_bytes of either block), ownership and errors as syk_otoc. */
int syk_build_parity_block(const syk_ham* h, int sector, syk_ham** out);
int syk_apply_gamma_block(int N, int n, int gamma_norm, int sector_out, int dtype, const void* d_in, void* d_out,
                          void* stream);
int syk_otoc_block(const syk_ham* h_even, const syk_ham* h_odd, int sector, int dtype, int i_W, int j_V, double beta,
                   const double* t_grid, int n_t, void* d_psi, double* F_out, const syk_krylov_opts* opts, void* d_work,
                   size_t work_bytes, syk_stats* stats, void* stream);
int syk_green_block(const syk_ham* h_even, const syk_ham* h_odd, int sector, int dtype, int n, double beta,
                    const double* t_grid, int n_t, void* d_psi, double* G_out, const syk_krylov_opts* opts, void* d_work,
                    size_t work_bytes, syk_stats* stats, void* stream);

/* Batched over disorder realizations: realization r uses hams[r], state d_psi + r*batch_stride
 * elements, and writes F_out[r][n_t][2].  Two modes, chosen by the work space the caller passes:
 *  - lock-step: work_bytes >= syk_otoc_batched_workspace_bytes(hams[0], n_batch, ...), all realizations have the same N,
 *    one-pass Lanczos, and every term table fits the shared-memory budget of the 16 KiB-tile kernel (sparse H, small
 *    and medium N).  Every kernel then runs with grid.y = realization: one launch per Lanczos step for the whole
 *    batch, the host does the n_batch small exponentials between rounds.  batch_stride * element size must be a
 *    multiple of 16 bytes.
 *  - otherwise: one work space of syk_otoc_workspace_bytes is shared and the realizations run back to back.
 * Results of the two modes agree to the Krylov tolerance (sub-steps are chosen per realization in both). */
int syk_otoc_batched_workspace_bytes(const syk_ham* h, int n_batch, int dtype, const syk_krylov_opts* opts,
                                     size_t* bytes);
int syk_otoc_batched(const syk_ham* const* hams, int n_batch, int dtype, int i_W, int j_V, double beta,
                     const double* t_grid, int n_t, void* d_psi, int64_t batch_stride, double* F_out,
                     const syk_krylov_opts* opts, void* d_work, size_t work_bytes, syk_stats* stats, void* stream);

/* The Green function of gamma_n for a batch of realizations, same two modes, buffers and work-space query
 * (syk_otoc_batched_workspace_bytes) as syk_otoc_batched; G_out[r][n_t][2]. */
int syk_green_batched(const syk_ham* const* hams, int n_batch, int dtype, int n, double beta, const double* t_grid, int n_t,
                      void* d_psi, int64_t batch_stride, double* G_out, const syk_krylov_opts* opts, void* d_work,
                      size_t work_bytes, syk_stats* stats, void* stream);

/* ------------------------------------------------------------------------------------------------------------
 * Introspection for tests and the benchmark. */
/* Which apply_H kernel a handle would use for `dtype`: 0 = generic gather, 1 = TMA-pipelined 16 KiB-tile gather,
 * 2 = TMA-pipelined register-tile gather (64 KiB tiles; sparse H with <= 1024 terms and D >= 2^22 / 2^23),
 * 3 = TMA-pipelined scatter-tile gather (128 KiB tiles on index bits chosen per Hamiltonian; sparse H with
 *     1..1024 terms and D >= 2^23 / 2^24),
 * 4 = dense-table kernel (many terms per X-mask: an X-mask whose Z-masks agree outside its own bits is one table lookup per
 *     amplitude, the others have their terms binned by the Walsh index of the Z-mask and transformed once per X-mask; chosen for > 1024 terms with >= 4 terms per X-mask and D >= 2^12; holds its own device table and, for
 *     vectors with fewer tiles than SMs, a scratch buffer for partial sums). */
int syk_apply_H_kernel_kind(const syk_ham* h, int dtype);
/* Force the kernel choice for subsequent syk_apply_H calls on this handle: -1 = automatic, 0 / 1 / 2 / 3 / 4 as above
 * (a kind the handle cannot use falls back to the next lower one). */
int syk_set_apply_H_kernel(syk_ham* h, int kind);
/* Shape of the dense-table kernel's (kind 4) device table for this handle: n_loads source tiles per output tile,
 * n_chunks table chunks of <= 512 entries streamed per output tile, split = CTAs that share one output tile (1 = the
 * persistent one-CTA-per-tile form; > 1 = the split form for vectors with fewer tiles than SMs), n_local_groups =
 * X-masks whose terms are applied through ONE table of 2^popcount(x) values instead of term by term (their Z-masks agree
 * outside the bits of x, popcount(x) <= 4, >= 4 terms: every four-qubit X-mask of a dense SYK Hamiltonian).  Builds the
 * table if needed.  Any output pointer may be NULL.  SYK_EINVAL if the handle cannot use kind 4. */
int syk_apply_H_dense_info(const syk_ham* h, int dtype, int* n_loads, int* n_chunks, int* split, int* n_local_groups);
/* Tile layout the scatter-tile kernel (kind 3) uses for this Hamiltonian in its current qubit layout: n_loads = source tiles fetched per
 * output tile (L2 -> SM transfers of the whole vector per product), n_passes = distinct X-masks outside tile and
 * L2-window bits (DRAM reads of the whole vector per product, if L2 reuse were perfect), tile_mask / window_mask =
 * the index bits of a tile / of tile + window.  Any output pointer may be NULL.  SYK_EINVAL if kind 3 cannot be used. */
int syk_apply_H_layout(const syk_ham* h, int dtype, int* n_loads, int* n_passes, uint32_t* tile_mask,
                       uint32_t* window_mask);
/* Diagnostic (measure, don't guess): one plain product out = H in through the scatter-tile kernel (kind 3, else SYK_EINVAL)
 * in which persistent CTA `cta` records, for the `round`-th output tile it owns, seven SM-clock stamps per ring chunk:
 * clk[v] = the producer issued the bulk copies of chunk v, clk[n + v] = the first consumer warp asked for chunk v,
 * clk[2 n + v] = it got it, clk[3 n + v] = it had decoded the chunk's first term (the LDS stream follows), clk[4 n + v] = it
 * had issued the first term, clk[5 n + v] = all terms, clk[6 n + v] = it had arrived on the chunk's empty-barrier;
 * v = list position * 2 + chunk, n = 2 * n_loads (clk_capacity >= 7 n).  detail = 0 records the first three only (the others
 * stay 0): every stamp costs the traced warp time, and the seven-stamp build lengthens a chunk by ~200 clocks.  So
 * clk[2n + v] - clk[n + v] is the time the consumers waited for data and clk[n + v + 1] - clk[2n + v] the time they
 * worked on chunk v.  List position li of this CTA holds load (li + rot) % n_loads; load_terms[l] / load_xo[l] = number of
 * terms / the part of the X-mask outside the tile bits of load l (load_capacity >= n_loads).  Unlike every other compute
 * call this one allocates (and frees) a small device buffer and synchronises `stream`.  Results of `out` are those of
 * syk_apply_H. */
int syk_apply_H_trace(const syk_ham* h, int dtype, const void* d_in, void* d_out, int cta, int round, int detail, uint64_t* clk,
                      int clk_capacity, int32_t* load_terms, uint32_t* load_xo, int load_capacity, int* n_loads, int* rot,
                      void* stream);
/* Pacing of the register-tile / scatter-tile kernels' persistent CTAs (process-wide; a tuning knob, results do not depend on it):
 * producers count their tile loads in epochs of `epoch_len` loads and may start an epoch only when every CTA has
 * issued the epoch `lag`+1 before it, which keeps the CTAs at the same place of the sorted load list so that source
 * tiles shared between neighbouring output tiles are still in L2.  epoch_len = 0 lets the CTAs run free.
 * Default (8, 1).  Used only for vectors larger than L2.  0 <= lag <= 30. */
int syk_set_lockstep(int epoch_len, int lag);
/* Latency path of the Krylov driver (process-wide switch, default on; results do not depend on it): for vectors of at most
 * 8 MB one Lanczos round (norm, m fused apply_H + m fused vector kernels, final norm) is captured once per (handle, dtype,
 * m, buffers) into a CUDA graph and replayed with one launch per round; a per-thread cache holds the 24 most recent
 * graphs.  Off while syk_profile_enable is on.  Replayed kernels count in syk_launch_count. */
int syk_set_cuda_graphs(int on);
/* Number of kernels launched by this library on the calling thread since the last reset. */
int64_t syk_launch_count(int reset);
/* Per-kernel device timing for the benchmark's roofline line.  While enabled, every apply_H launch made by the
 * calling thread (direct or inside syk_lanczos_run / syk_krylov_evolve / syk_otoc) is bracketed by two CUDA
 * events on its stream (at most 65536 launches are recorded; later ones are counted but not timed).
 * syk_profile_read synchronises those events and returns their summed duration, the number of timed launches
 * and, when `reset` is non-zero, forgets them.  Any output pointer may be NULL. */
int syk_profile_enable(int on);
int syk_profile_read(double* apply_h_ms, int64_t* apply_h_launches, int reset);

/* ------------------------------------------------------------------------------------------------------------
 * On-chip peak measurements (denominators of the benchmark's roofline; SURVEY section 7 "hard parts": the HBM copy
 * peak is known, the L2 -> SM, shared-memory and ALU-issue peaks of this box are not).  One launch of 1 CTA per SM:
 *   kind 0: every CTA streams arg0 chunks of 64 KiB from d_buf (walked pseudo-randomly; a buffer of <= 32 MB stays in
 *           L2, a multi-GB one streams from DRAM) into the 3-chunk shared-memory ring of the scatter-tile kernel with
 *           cp.async.bulk, no arithmetic; arg1 > 0: only arg1 CTAs (SMs) stream (per-SM rate below the chip-wide L2 limit);
 *   kind 1: no copies; the 8 consumer warps make arg1 passes over each of arg0 staged chunks with the kernel's
 *           XOR-permuted LDS.128 + 2 FP64 FMA per element;
 *   kind 2: both at once (arg1 passes over every chunk that arrives);
 *   kind 3: arg0 x 64 FP64 adds per thread in 8 independent chains, 512 threads per SM;
 *   kind 4: arg0 x 64 times the per-term sequence of the dense-table kernel (broadcast LDS of a table entry, AND, POPC,
 *           shift, XOR into the sign bit, FP64 add into one of 8 bin registers), 512 threads per SM.
 *   kind 5: as kind 0 in two groups at once: even CTAs walk the whole of d_buf (DRAM for a multi-GB buffer), odd CTAs only
 *           its first 32 MB (L2 resident) and stream arg1 times as many chunks: do the DRAM and the L2 supply overlap?
 *   kind 6: do global loads share the shared-memory data path?  256 threads per SM; per iteration (arg0 of them) every
 *           thread issues 16 LDG.128 (ld.global.cg, 64 KiB of d_buf per CTA and iteration; d_buf = NULL: none) and arg1 x 16
 *           LDS.128 over a staged 64 KiB chunk, one FP64 FMA pair per value.
 *   kind 7: distributed shared memory: clusters of two CTAs, 256 threads each; per iteration (arg0 of them) every thread reads 16
 *           16-byte elements of a staged 64 KiB chunk through the shared::cluster window of its own CTA (arg1 = 0) or of the
 *           peer CTA (arg1 = 1: SM-to-SM).  [3] = bytes read; rate per SM = [3] / SMs used (an even number) / [1].
 * result[6]: [0] = device time in ms (CUDA events), [1] = SM cycles of the slowest CTA (clock64), [2] = bytes copied
 * into shared memory (kinds 0, 2; kind 5: by the even CTAs), thread-level adds (kinds 3, 4) or bytes loaded by LDG (kind 6),
 * [3] = bytes read by LDS (kinds 1, 2, 6; kind 5: bytes copied by the odd CTAs), [4] / [5] = cycles of the slowest even / odd CTA.
 * d_work: >= syk_microbench_workspace_bytes() of device memory; d_buf (kinds 0, 2): 128-byte aligned, buf_bytes >= 128 KiB
 * (rounded down to a power of two).  Synchronises. */
size_t syk_microbench_workspace_bytes(void);
int syk_microbench(int kind, int arg0, int arg1, const void* d_buf, size_t buf_bytes, void* d_work, size_t work_bytes,
                   double* result, void* stream);

#ifdef __cplusplus
}
#endif
#endif /* SYK_B200_H */
