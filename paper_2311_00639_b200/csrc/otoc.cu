// a-5  OTOC pipeline (R-EQ2; random state -> Krylov evolution -> inner product).
//
//   F(t) = <psi| E(-t - ib/8) g_W E(t - ib/4) g_V E(-t - ib/4) g_W E(t - ib/4) g_V E(-ib/8) |psi>,  E(tau) = exp(-i tau H)
//
// Right to left on the ket, with the bra side l(t) = E(t - ib/8) psi.  Both l(t) and phi(t) = E(t - ib/4) g_V E(-ib/8) psi
// are advanced incrementally along the (non-decreasing) t grid by E(dt); the two middle evolutions of length t act on
// t-dependent states and are redone for every grid point:
//   l    <- E(-ib/8) psi                     (in psi's own buffer; psi is destroyed)
//   phi  <- E(-ib/4) g_V l
//   for each t_k:  l <- E(dt) l ; phi <- E(dt) phi
//                  r <- g_W phi ; r <- E(-t - ib/4) r ; r <- g_V r ; r <- E(t - ib/4) r ; r <- g_W r ;  F_k = <l|r>
// Resident vectors: l, phi, r + Krylov work (2 in two-pass mode: 5 in total, PAPER.md:249's v+3 with v = 2).
#include <cmath>
#include <vector>

#include "common.h"

namespace syk {

// The space the pipelines run in: the full 2^(N/2) space (sector < 0: one Hamiltonian, JW gammas) or parity blocks
// on N/2-1 qubits (R-BLOCK: hs[0] / hs[1] = even / odd block, a state in sector s evolves under
// hs[s] and every gamma moves it to the other sector).
struct Space {
    const syk_ham* hs[2];
    int sector;    // sector of the initial state; < 0 = full space
    int N;         // Majoranas of the FULL Hamiltonian
    int gamma_norm;
    const syk_ham* ham(int sec) const { return sector < 0 ? hs[0] : hs[sec]; }
    // vectors live in the qubit layout of the handles (both blocks share one layout: a gamma maps between them)
    int gamma(int n, int sec_out, int dtype, const void* in, void* out, cudaStream_t st) const {
        return sector < 0 ? launch_gamma_h(hs[0], n, dtype, in, out, st)
                          : launch_gamma_block(N, n, gamma_norm, sec_out, dtype, in, out, st, hs[0]);
    }
};

// One evolution inside a pipeline: accumulates the call's statistics into `stats` and its log-norm (opts->renormalize:
// the factor taken out of the vector) into the accumulator of the vector that was evolved.
static int evolve_tracked(const syk_ham* h, int dtype, void* v, double tre, double tim, const syk_krylov_opts* opts,
                          void* kwork, size_t kbytes, syk_stats* stats, double* log_norm, cudaStream_t st) {
    syk_stats loc{};
    const int rc = krylov_evolve_impl(h, dtype, v, tre, tim, opts, kwork, kbytes, &loc, st);
    if (stats) {
        stats->n_matvec += loc.n_matvec;
        stats->n_substeps += loc.n_substeps;
        stats->err_est += loc.err_est;
        stats->model_bytes += loc.model_bytes;
        if (loc.krylov_dim_used > 0)
            stats->krylov_dim_used = stats->krylov_dim_used == 0 ? loc.krylov_dim_used
                                                                 : (loc.krylov_dim_used < stats->krylov_dim_used ? loc.krylov_dim_used : stats->krylov_dim_used);
        stats->log_norm += loc.log_norm;
    }
    *log_norm += loc.log_norm;
    return rc;
}

static int otoc_one(const Space& sp, int dtype, int i_W, int j_V, double beta, const double* t_grid, int n_t,
                    void* d_psi, double* F_out, const syk_krylov_opts* opts, void* d_work, size_t work_bytes,
                    syk_stats* stats, cudaStream_t st) {
    const syk_ham* h = sp.hs[0];
    const int s0 = sp.sector < 0 ? 0 : sp.sector, s1 = sp.sector < 0 ? 0 : 1 - sp.sector;
    const uint64_t D = 1ull << h->L;
    const size_t vbytes = (size_t)D * elem_bytes(dtype);
    size_t kbytes = 0;
    SYK_TRY(syk_krylov_workspace_bytes(h, dtype, opts, &kbytes));
    if (work_bytes < 2 * vbytes + kbytes) return SYK_ENOMEM;
    char* l = (char*)d_psi;
    char* phi = (char*)d_work;
    char* r = phi + vbytes;
    char* kwork = r + vbytes;
    LanczosScalars* sc = (LanczosScalars*)kwork;   // the Krylov header doubles as reduction scratch between evolutions
    int rc_soft = SYK_OK;
    // opts->renormalize: every vector keeps the norm it had and carries the logarithm of the factor taken out of it
    double ln_l = 0.0, ln_phi = 0.0, ln_r = 0.0;
    auto evolve = [&](void* v, int sec, double tre, double tim, double* ln) -> int {
        int rc = evolve_tracked(sp.ham(sec), dtype, v, tre, tim, opts, kwork, kbytes, stats, ln, st);
        if (rc == SYK_ENOCONV) {
            rc_soft = rc;
            return SYK_OK;
        }
        return rc;
    };
    // l lives in sector s0, phi in s1; r goes s0 -> s1 -> s0
    SYK_TRY(evolve(l, s0, 0.0, -beta / 8.0, &ln_l));
    SYK_TRY(sp.gamma(j_V, s1, dtype, l, phi, st));
    ln_phi = ln_l;
    SYK_TRY(evolve(phi, s1, 0.0, -beta / 4.0, &ln_phi));
    double t_prev = 0.0;
    for (int k = 0; k < n_t; ++k) {
        const double t = t_grid[k], dt = t - t_prev;
        if (dt > 0.0) {
            SYK_TRY(evolve(l, s0, dt, 0.0, &ln_l));
            SYK_TRY(evolve(phi, s1, dt, 0.0, &ln_phi));
        }
        t_prev = t;
        SYK_TRY(sp.gamma(i_W, s0, dtype, phi, r, st));
        ln_r = ln_phi;
        SYK_TRY(evolve(r, s0, -t, -beta / 4.0, &ln_r));
        SYK_TRY(sp.gamma(j_V, s1, dtype, r, r, st));
        SYK_TRY(evolve(r, s1, t, -beta / 4.0, &ln_r));
        SYK_TRY(sp.gamma(i_W, s0, dtype, r, r, st));
        SYK_TRY(launch_cdot(dtype, D, l, r, sc, st));
        SYK_TRY(fetch_cdot(sc, F_out + 2 * k, st));
        const double scale = std::exp(ln_l + ln_r);   // 1 unless opts->renormalize
        F_out[2 * k] *= scale;
        F_out[2 * k + 1] *= scale;
    }
    return rc_soft;
}

// Retarded Green function:
//   G(t) = <psi| e^{(it-b/2)H} g_n e^{-iHt} g_n e^{-bH/2} |psi> = < E(t) l0 | g_n E(t) g_n l0 >,  l0 = E(-ib/2) psi,
// so both sides advance incrementally along the t grid: two evolutions by dt per grid point, one gamma insertion,
// one inner product.  Resident: l (in psi's buffer), phi, r + Krylov work.
static int green_one(const Space& sp, int dtype, int n, double beta, const double* t_grid, int n_t, void* d_psi,
                     double* G_out, const syk_krylov_opts* opts, void* d_work, size_t work_bytes, syk_stats* stats,
                     cudaStream_t st) {
    const syk_ham* h = sp.hs[0];
    const int s0 = sp.sector < 0 ? 0 : sp.sector, s1 = sp.sector < 0 ? 0 : 1 - sp.sector;
    const uint64_t D = 1ull << h->L;
    const size_t vbytes = (size_t)D * elem_bytes(dtype);
    size_t kbytes = 0;
    SYK_TRY(syk_krylov_workspace_bytes(h, dtype, opts, &kbytes));
    if (work_bytes < 2 * vbytes + kbytes) return SYK_ENOMEM;
    char* l = (char*)d_psi;
    char* phi = (char*)d_work;
    char* r = phi + vbytes;
    char* kwork = r + vbytes;
    LanczosScalars* sc = (LanczosScalars*)kwork;
    int rc_soft = SYK_OK;
    double ln_l = 0.0, ln_phi = 0.0;
    auto evolve = [&](void* v, int sec, double tre, double tim, double* ln) -> int {
        int rc = evolve_tracked(sp.ham(sec), dtype, v, tre, tim, opts, kwork, kbytes, stats, ln, st);
        if (rc == SYK_ENOCONV) {
            rc_soft = rc;
            return SYK_OK;
        }
        return rc;
    };
    SYK_TRY(evolve(l, s0, 0.0, -beta / 2.0, &ln_l));
    SYK_TRY(sp.gamma(n, s1, dtype, l, phi, st));
    ln_phi = ln_l;
    double t_prev = 0.0;
    for (int k = 0; k < n_t; ++k) {
        const double dt = t_grid[k] - t_prev;
        if (dt > 0.0) {
            SYK_TRY(evolve(l, s0, dt, 0.0, &ln_l));
            SYK_TRY(evolve(phi, s1, dt, 0.0, &ln_phi));
        }
        t_prev = t_grid[k];
        SYK_TRY(sp.gamma(n, s0, dtype, phi, r, st));
        SYK_TRY(launch_cdot(dtype, D, l, r, sc, st));
        SYK_TRY(fetch_cdot(sc, G_out + 2 * k, st));
        const double scale = std::exp(ln_l + ln_phi);   // 1 unless opts->renormalize
        G_out[2 * k] *= scale;
        G_out[2 * k + 1] *= scale;
    }
    return rc_soft;
}

// The OTOC pipeline of otoc_one with every kernel batched over the realizations (grid.y) and the realizations advancing
// through each evolution in lock step.  Work space: phi[nb] | r[nb] | batched Krylov work space.
static size_t otoc_batched_bytes(const syk_ham* h0, int nb, int dtype, const syk_krylov_opts* opts) {
    const size_t v = ((size_t)1 << h0->L) * elem_bytes(dtype);
    return 2 * (size_t)nb * v + krylov_batched_bytes(h0, nb, dtype, resolve_krylov_dim(h0, opts));
}

// green = true: the Green function of gamma_{i_W} (j_V unused), same buffers: l = E(-ib/2) psi, phi = g l, per grid point both
// advance by E(dt) and G = <l | g phi>
static int otoc_batched_impl(const syk_ham* const* hams, int nb, int dtype, int i_W, int j_V, double beta,
                             const double* t_grid, int n_t, void* d_psi, size_t psi_stride, double* F_out,
                             const syk_krylov_opts* opts, void* d_work, size_t work_bytes, syk_stats* stats,
                             cudaStream_t st, bool green = false) {
    const syk_ham* h0 = hams[0];
    const uint64_t D = 1ull << h0->L;
    const size_t v = (size_t)D * elem_bytes(dtype);
    const int m = resolve_krylov_dim(h0, opts);
    if (work_bytes < otoc_batched_bytes(h0, nb, dtype, opts)) return SYK_ENOMEM;
    {   // the states must not overlap the work space
        const uintptr_t a = (uintptr_t)d_psi, b = (uintptr_t)d_work;
        if (a < b + otoc_batched_bytes(h0, nb, dtype, opts) && b < a + (size_t)(nb - 1) * psi_stride + v) return SYK_EINVAL;
    }
    char* l = (char*)d_psi;
    char* phi = (char*)d_work;
    char* r = phi + (size_t)nb * v;
    char* kwork = r + (size_t)nb * v;
    const size_t kbytes = krylov_batched_bytes(h0, nb, dtype, m);
    const size_t ws_stride = krylov_header_bytes() + (size_t)m * v;
    LanczosScalars* sc = (LanczosScalars*)(kwork + batched_table_bytes(nb));   // realization 0's header
    bool uploaded = false;
    int rc_soft = SYK_OK;
    auto evolve = [&](void* vec, size_t stride, double tre, double tim) -> int {
        int rc = krylov_evolve_batched_impl(hams, nb, dtype, vec, stride, tre, tim, opts, kwork, kbytes, stats, &uploaded,
                                            st);
        if (rc == SYK_ENOCONV) {
            rc_soft = rc;
            return SYK_OK;
        }
        return rc;
    };
    auto gamma = [&](int n, const void* in, size_t s_in, void* out, size_t s_out) -> int {
        Batch b;
        b.n = nb;
        b.s.a = s_in;
        b.s.b = s_out;
        return launch_gamma_h(h0, n, dtype, in, out, st, b);   // one layout for the whole batch (batched_apply_ok)
    };
    std::vector<double> dots((size_t)2 * nb);
    if (green) {
        SYK_TRY(evolve(l, psi_stride, 0.0, -beta / 2.0));
        SYK_TRY(gamma(i_W, l, psi_stride, phi, v));
    } else {
        SYK_TRY(evolve(l, psi_stride, 0.0, -beta / 8.0));
        SYK_TRY(gamma(j_V, l, psi_stride, phi, v));
        SYK_TRY(evolve(phi, v, 0.0, -beta / 4.0));
    }
    double t_prev = 0.0;
    for (int k = 0; k < n_t; ++k) {
        const double t = t_grid[k], dt = t - t_prev;
        if (dt > 0.0) {
            SYK_TRY(evolve(l, psi_stride, dt, 0.0));
            SYK_TRY(evolve(phi, v, dt, 0.0));
        }
        t_prev = t;
        SYK_TRY(gamma(i_W, phi, v, r, v));
        if (!green) {
            SYK_TRY(evolve(r, v, -t, -beta / 4.0));
            SYK_TRY(gamma(j_V, r, v, r, v));
            SYK_TRY(evolve(r, v, t, -beta / 4.0));
            SYK_TRY(gamma(i_W, r, v, r, v));
        }
        Batch b;
        b.n = nb;
        b.s.a = psi_stride;
        b.s.b = v;
        b.s.sc = ws_stride;
        SYK_TRY(cdot_batched(dtype, D, l, r, sc, b, dots.data(), st));
        for (int rr = 0; rr < nb; ++rr) {
            F_out[((size_t)rr * n_t + k) * 2] = dots[2 * (size_t)rr];
            F_out[((size_t)rr * n_t + k) * 2 + 1] = dots[2 * (size_t)rr + 1];
        }
    }
    return rc_soft;
}

static Space full_space(const syk_ham* h) { return Space{{h, h}, -1, h->N, h->gamma_norm}; }

// the two blocks of one Hamiltonian: same N, same normalisation, sectors 0 and 1
static bool blocks_ok(const syk_ham* he, const syk_ham* ho, int sector) {
    return he && ho && (sector == 0 || sector == 1) && he->block_of_N >= 6 && he->block_of_N == ho->block_of_N &&
           he->sector == 0 && ho->sector == 1 && he->gamma_norm == ho->gamma_norm && he->perm == ho->perm;
}

static bool otoc_args_ok(const syk_ham* h, int dtype, int i_W, int j_V, double beta, const double* t_grid, int n_t,
                         const void* d_psi, const double* F_out, const void* d_work) {
    if (!h || (dtype != SYK_C64 && dtype != SYK_C128) || !d_psi || !d_work || n_t < 0 || (n_t > 0 && (!t_grid || !F_out)))
        return false;
    if (((uintptr_t)d_psi & 15) || ((uintptr_t)d_work & 15)) return false;
    if (h->generic) return false;                         // gamma insertions mean nothing for a spin-chain operator
    if (!h->hermitian) return false;                      // the regularised OTOC / Green function are defined for H = H^+
    const int N = h->block_of_N ? h->block_of_N : h->N;   // operator indices refer to the full Hamiltonian
    if (i_W < 0 || i_W >= N || j_V < 0 || j_V >= N || i_W == j_V || !(beta >= 0.0)) return false;
    double prev = 0.0;
    for (int k = 0; k < n_t; ++k) {
        if (!(t_grid[k] >= prev)) return false;
        prev = t_grid[k];
    }
    return true;
}

}  // namespace syk

extern "C" {

int syk_otoc_workspace_bytes(const syk_ham* h, int dtype, const syk_krylov_opts* opts, size_t* bytes) {
    size_t k = 0;
    SYK_TRY(syk_krylov_workspace_bytes(h, dtype, opts, &k));
    *bytes = k + 2 * ((size_t)1 << h->L) * syk::elem_bytes(dtype);
    return SYK_OK;
}

int syk_otoc(const syk_ham* h, int dtype, int i_W, int j_V, double beta, const double* t_grid, int n_t, void* d_psi,
             double* F_out, const syk_krylov_opts* opts, void* d_work, size_t work_bytes, syk_stats* stats,
             void* stream) {
    if (!syk::otoc_args_ok(h, dtype, i_W, j_V, beta, t_grid, n_t, d_psi, F_out, d_work) || h->block_of_N)
        return SYK_EINVAL;
    if (stats) *stats = syk_stats{};
    return syk::otoc_one(syk::full_space(h), dtype, i_W, j_V, beta, t_grid, n_t, d_psi, F_out, opts, d_work, work_bytes, stats,
                         (cudaStream_t)stream);
}

int syk_green(const syk_ham* h, int dtype, int n, double beta, const double* t_grid, int n_t, void* d_psi,
              double* G_out, const syk_krylov_opts* opts, void* d_work, size_t work_bytes, syk_stats* stats,
              void* stream) {
    // same argument rules as syk_otoc with a single operator index
    if (!h || n < 0 || n >= h->N || h->block_of_N) return SYK_EINVAL;
    if (!syk::otoc_args_ok(h, dtype, n, n == 0 ? 1 : 0, beta, t_grid, n_t, d_psi, G_out, d_work)) return SYK_EINVAL;
    if (stats) *stats = syk_stats{};
    return syk::green_one(syk::full_space(h), dtype, n, beta, t_grid, n_t, d_psi, G_out, opts, d_work, work_bytes, stats,
                          (cudaStream_t)stream);
}

// Parity-block forms (R-BLOCK): one of the two terms of F / G, for a reduced state in `sector`.
int syk_otoc_block(const syk_ham* h_even, const syk_ham* h_odd, int sector, int dtype, int i_W, int j_V, double beta,
                   const double* t_grid, int n_t, void* d_psi, double* F_out, const syk_krylov_opts* opts, void* d_work,
                   size_t work_bytes, syk_stats* stats, void* stream) {
    if (!syk::blocks_ok(h_even, h_odd, sector)) return SYK_EINVAL;
    if (!syk::otoc_args_ok(h_even, dtype, i_W, j_V, beta, t_grid, n_t, d_psi, F_out, d_work)) return SYK_EINVAL;
    if (stats) *stats = syk_stats{};
    const syk::Space sp{{h_even, h_odd}, sector, h_even->block_of_N, h_even->gamma_norm};
    return syk::otoc_one(sp, dtype, i_W, j_V, beta, t_grid, n_t, d_psi, F_out, opts, d_work, work_bytes, stats,
                         (cudaStream_t)stream);
}

int syk_green_block(const syk_ham* h_even, const syk_ham* h_odd, int sector, int dtype, int n, double beta,
                    const double* t_grid, int n_t, void* d_psi, double* G_out, const syk_krylov_opts* opts, void* d_work,
                    size_t work_bytes, syk_stats* stats, void* stream) {
    if (!syk::blocks_ok(h_even, h_odd, sector) || n < 0 || n >= h_even->block_of_N) return SYK_EINVAL;
    if (!syk::otoc_args_ok(h_even, dtype, n, n == 0 ? 1 : 0, beta, t_grid, n_t, d_psi, G_out, d_work)) return SYK_EINVAL;
    if (stats) *stats = syk_stats{};
    const syk::Space sp{{h_even, h_odd}, sector, h_even->block_of_N, h_even->gamma_norm};
    return syk::green_one(sp, dtype, n, beta, t_grid, n_t, d_psi, G_out, opts, d_work, work_bytes, stats,
                          (cudaStream_t)stream);
}

int syk_otoc_batched_workspace_bytes(const syk_ham* h, int n_batch, int dtype, const syk_krylov_opts* opts,
                                     size_t* bytes) {
    if (!h || !bytes || n_batch < 1 || (dtype != SYK_C64 && dtype != SYK_C128)) return SYK_EINVAL;
    if (opts && (opts->krylov_dim < 0 || opts->krylov_dim == 1)) return SYK_EINVAL;
    *bytes = syk::otoc_batched_bytes(h, n_batch, dtype, opts);
    return SYK_OK;
}

int syk_otoc_batched(const syk_ham* const* hams, int n_batch, int dtype, int i_W, int j_V, double beta,
                     const double* t_grid, int n_t, void* d_psi, int64_t batch_stride, double* F_out,
                     const syk_krylov_opts* opts, void* d_work, size_t work_bytes, syk_stats* stats, void* stream) {
    if (!hams || n_batch < 0) return SYK_EINVAL;
    if (stats) *stats = syk_stats{};
    // lock-step batched pipeline when the realizations qualify (small N, tables in shared memory, one-pass) and the work
    // space is large enough for it (syk_otoc_batched_workspace_bytes); else one realization after the other
    if (n_batch >= 2 && hams[0] && !(opts && (opts->two_pass || opts->renormalize)) && syk::batched_apply_ok(hams, n_batch, dtype) &&
        work_bytes >= syk::otoc_batched_bytes(hams[0], n_batch, dtype, opts)) {
        for (int r = 0; r < n_batch; ++r) {
            if (hams[r]->block_of_N || batch_stride < ((int64_t)1 << hams[r]->L)) return SYK_EINVAL;
            char* psi = (char*)d_psi + (size_t)r * (size_t)batch_stride * syk::elem_bytes(dtype);
            if (!syk::otoc_args_ok(hams[r], dtype, i_W, j_V, beta, t_grid, n_t, psi, F_out, d_work)) return SYK_EINVAL;
        }
        if (((size_t)batch_stride * syk::elem_bytes(dtype)) % 16) return SYK_EINVAL;
        return syk::otoc_batched_impl(hams, n_batch, dtype, i_W, j_V, beta, t_grid, n_t, d_psi,
                                      (size_t)batch_stride * syk::elem_bytes(dtype), F_out, opts, d_work, work_bytes, stats,
                                      (cudaStream_t)stream);
    }
    int rc_soft = SYK_OK;
    for (int r = 0; r < n_batch; ++r) {
        if (!hams[r] || hams[r]->N != hams[0]->N || batch_stride < ((int64_t)1 << hams[r]->L)) return SYK_EINVAL;
        char* psi = (char*)d_psi + (size_t)r * (size_t)batch_stride * syk::elem_bytes(dtype);
        if (!syk::otoc_args_ok(hams[r], dtype, i_W, j_V, beta, t_grid, n_t, psi, F_out, d_work) || hams[r]->block_of_N)
            return SYK_EINVAL;
        int rc = syk::otoc_one(syk::full_space(hams[r]), dtype, i_W, j_V, beta, t_grid, n_t, psi, F_out + (size_t)r * 2 * n_t, opts,
                               d_work, work_bytes, stats, (cudaStream_t)stream);
        if (rc == SYK_ENOCONV) rc_soft = rc;
        else if (rc != SYK_OK) return rc;
    }
    return rc_soft;
}

int syk_green_batched(const syk_ham* const* hams, int n_batch, int dtype, int n, double beta, const double* t_grid, int n_t,
                      void* d_psi, int64_t batch_stride, double* G_out, const syk_krylov_opts* opts, void* d_work,
                      size_t work_bytes, syk_stats* stats, void* stream) {
    if (!hams || n_batch < 1 || !hams[0]) return SYK_EINVAL;
    if (stats) *stats = syk_stats{};
    const int other = n == 0 ? 1 : 0;   // otoc_args_ok wants two different operator indices
    const bool lockstep = n_batch >= 2 && !(opts && (opts->two_pass || opts->renormalize)) &&
                          syk::batched_apply_ok(hams, n_batch, dtype) &&
                          work_bytes >= syk::otoc_batched_bytes(hams[0], n_batch, dtype, opts);
    for (int r = 0; r < n_batch; ++r) {
        if (!hams[r] || hams[r]->N != hams[0]->N || hams[r]->block_of_N || batch_stride < ((int64_t)1 << hams[r]->L) ||
            n < 0 || n >= hams[r]->N)
            return SYK_EINVAL;
        char* psi = (char*)d_psi + (size_t)r * (size_t)batch_stride * syk::elem_bytes(dtype);
        if (!syk::otoc_args_ok(hams[r], dtype, n, other, beta, t_grid, n_t, psi, G_out, d_work)) return SYK_EINVAL;
    }
    if (lockstep) {
        if (((size_t)batch_stride * syk::elem_bytes(dtype)) % 16) return SYK_EINVAL;
        return syk::otoc_batched_impl(hams, n_batch, dtype, n, other, beta, t_grid, n_t, d_psi,
                                      (size_t)batch_stride * syk::elem_bytes(dtype), G_out, opts, d_work, work_bytes, stats,
                                      (cudaStream_t)stream, true);
    }
    int rc_soft = SYK_OK;
    for (int r = 0; r < n_batch; ++r) {
        char* psi = (char*)d_psi + (size_t)r * (size_t)batch_stride * syk::elem_bytes(dtype);
        int rc = syk::green_one(syk::full_space(hams[r]), dtype, n, beta, t_grid, n_t, psi, G_out + (size_t)r * 2 * n_t, opts,
                                d_work, work_bytes, stats, (cudaStream_t)stream);
        if (rc == SYK_ENOCONV) rc_soft = rc;
        else if (rc != SYK_OK) return rc;
    }
    return rc_soft;
}

// ---- HOST-buffer entry points: the same calls with the host<->device copies inside ---------------------------
int syk_apply_H_host(const syk_ham* h, int dtype, const void* h_in, void* h_out, void* d_work, size_t work_bytes,
                     void* stream) {
    if (!h || !h_in || !h_out || !d_work || (dtype != SYK_C64 && dtype != SYK_C128)) return SYK_EINVAL;
    const size_t v = ((size_t)1 << h->L) * syk::elem_bytes(dtype);
    if (work_bytes < 2 * v) return SYK_ENOMEM;
    cudaStream_t st = (cudaStream_t)stream;
    char* din = (char*)d_work;
    char* dout = din + v;
    if (h->identity_layout()) {
        SYK_CUDA(cudaMemcpyAsync(din, h_in, v, cudaMemcpyHostToDevice, st));
        SYK_TRY(syk_apply_H(h, dtype, din, dout, stream));
        SYK_CUDA(cudaMemcpyAsync(h_out, dout, v, cudaMemcpyDeviceToHost, st));
    } else {   // host vectors are canonical: one gather pass into / out of the handle's qubit layout
        SYK_CUDA(cudaMemcpyAsync(dout, h_in, v, cudaMemcpyHostToDevice, st));
        SYK_TRY(syk::permute_vector(h, dtype, true, dout, din, st));
        SYK_TRY(syk_apply_H(h, dtype, din, dout, stream));
        SYK_TRY(syk::permute_vector(h, dtype, false, dout, din, st));
        SYK_CUDA(cudaMemcpyAsync(h_out, din, v, cudaMemcpyDeviceToHost, st));
    }
    SYK_CUDA(cudaStreamSynchronize(st));
    return SYK_OK;
}

int syk_krylov_evolve_host(const syk_ham* h, int dtype, void* h_psi, double tau_re, double tau_im,
                           const syk_krylov_opts* opts, void* d_work, size_t work_bytes, syk_stats* stats,
                           void* stream) {
    if (!h || !h_psi || !d_work || (dtype != SYK_C64 && dtype != SYK_C128)) return SYK_EINVAL;
    const size_t v = ((size_t)1 << h->L) * syk::elem_bytes(dtype);
    if (work_bytes < v) return SYK_ENOMEM;
    cudaStream_t st = (cudaStream_t)stream;
    // host vectors are canonical; with a relabelled handle the first Krylov work vector stages the copy (one gather pass
    // into / out of the handle's qubit layout on either side)
    char* stage = (char*)d_work + v + syk::krylov_header_bytes();
    const bool relabelled = !h->identity_layout();
    if (relabelled && work_bytes < 2 * v + syk::krylov_header_bytes()) return SYK_ENOMEM;
    SYK_CUDA(cudaMemcpyAsync(relabelled ? (void*)stage : d_work, h_psi, v, cudaMemcpyHostToDevice, st));
    if (relabelled) SYK_TRY(syk::permute_vector(h, dtype, true, stage, d_work, st));
    int rc = syk_krylov_evolve(h, dtype, d_work, tau_re, tau_im, opts, (char*)d_work + v, work_bytes - v, stats, stream);
    if (rc != SYK_OK && rc != SYK_ENOCONV) return rc;
    if (relabelled) SYK_TRY(syk::permute_vector(h, dtype, false, d_work, stage, st));
    SYK_CUDA(cudaMemcpyAsync(h_psi, relabelled ? (const void*)stage : (const void*)d_work, v, cudaMemcpyDeviceToHost, st));
    SYK_CUDA(cudaStreamSynchronize(st));
    return rc;
}

}  // extern "C"
