// a-4  Krylov driver: psi <- exp(-i tau H) psi for complex tau (R-TAU, R-KRYLOV).
//
// Hermitian Lanczos builds T_m (real symmetric tridiagonal; alpha_j, beta_j) with the fused kernels; the small
// exponential exp(-i tau T_m) e_1 is taken on the host through a Jacobi eigen-decomposition of T_m; the result is
// |psi| V_m exp(-i tau T_m) e_1.  T_m does not depend on tau, so after one build the driver picks the longest
// sub-step h along the ray tau = |tau| e^{i phi} whose a-posteriori error estimate
//        err(h) = int_0^h beta_{m+1} |e_m^T exp(-i e^{i phi} s T_m) e_1| ds / |exp(-i e^{i phi} h T_m) e_1|
// (the time integral of the residual norm of y' = -iHy, relative to the result) stays below its share
// tol * h/|tau| of the budget, applies it, and repeats on the remainder.
//
//  one-pass : keeps u_2..u_{m+1} (m work vectors), then psi = sum_j c_j v_j in one fused pass.
//  two-pass : 2 work vectors P, Q.  Pass 1 runs the recurrence for T_m only; from step 3 on the new vector
//             overwrites u_{j-1} in place (out aliases prev in the fused apply_H), so psi is untouched.  Pass 2
//             repeats the identical recurrence (bitwise: fixed reduction trees) and accumulates
//             y += c_j v_j into psi's own buffer as soon as u_1 is no longer needed.  Replaces the restarted
//             scheme of PAPER.md:301 as the bounded-memory mode (PAPER.md:249 counts v+3 vectors; this is 3).
#include <algorithm>
#include <atomic>
#include <cmath>
#include <complex>
#include <cstddef>
#include <thread>

#include "common.h"

namespace syk {

size_t krylov_header_bytes() { return (sizeof(LanczosScalars) + 4095) & ~(size_t)4095; }

namespace {

using cplx = std::complex<double>;

// Cyclic Jacobi for a real symmetric matrix A (m x m, row-major, destroyed): eigenvalues theta, eigenvectors in
// the columns of Q (row-major).  Small m only (<= 128).
void jacobi_eig(int m, std::vector<double>& A, std::vector<double>& theta, std::vector<double>& Q) {
    Q.assign((size_t)m * m, 0.0);
    for (int i = 0; i < m; ++i) Q[(size_t)i * m + i] = 1.0;
    auto a = [&](int i, int j) -> double& { return A[(size_t)i * m + j]; };
    for (int sweep = 0; sweep < 100; ++sweep) {
        double off = 0.0, diag = 0.0;
        for (int i = 0; i < m; ++i) {
            diag += a(i, i) * a(i, i);
            for (int j = i + 1; j < m; ++j) off += a(i, j) * a(i, j);
        }
        if (off <= 1e-34 * (diag + off) || off == 0.0) break;
        for (int p = 0; p < m - 1; ++p)
            for (int q = p + 1; q < m; ++q) {
                const double apq = a(p, q);
                if (apq == 0.0) continue;
                const double th = (a(q, q) - a(p, p)) / (2.0 * apq);
                const double t = (th >= 0.0 ? 1.0 : -1.0) / (std::fabs(th) + std::sqrt(th * th + 1.0));
                const double c = 1.0 / std::sqrt(t * t + 1.0), s = t * c;
                for (int k = 0; k < m; ++k) {   // columns p, q
                    const double akp = a(k, p), akq = a(k, q);
                    a(k, p) = c * akp - s * akq;
                    a(k, q) = s * akp + c * akq;
                }
                for (int k = 0; k < m; ++k) {   // rows p, q
                    const double apk = a(p, k), aqk = a(q, k);
                    a(p, k) = c * apk - s * aqk;
                    a(q, k) = s * apk + c * aqk;
                }
                for (int k = 0; k < m; ++k) {
                    const double qkp = Q[(size_t)k * m + p], qkq = Q[(size_t)k * m + q];
                    Q[(size_t)k * m + p] = c * qkp - s * qkq;
                    Q[(size_t)k * m + q] = s * qkp + c * qkq;
                }
            }
    }
    theta.resize(m);
    for (int i = 0; i < m; ++i) theta[i] = a(i, i);
}

struct SmallExp {
    int m = 0;
    std::vector<double> theta, Q;
    double beta_next = 0.0;   // beta_{m+1}
    cplx dir;                 // tau / |tau|
    // component j (0-based) of exp(-i dir s T) e_1
    cplx comp(int j, double s) const {
        cplx acc = 0.0;
        for (int k = 0; k < m; ++k)
            acc += Q[(size_t)j * m + k] * std::exp(cplx(0.0, -1.0) * dir * (s * theta[k])) * Q[k];
        return acc;
    }
    // |exp(-i dir s T) e_1|: Q is orthogonal, so the norm is that of the coefficient vector in the eigenbasis
    double result_norm(double s) const {
        double n2 = 0.0;
        for (int k = 0; k < m; ++k) n2 += std::norm(std::exp(cplx(0.0, -1.0) * dir * (s * theta[k]))) * Q[k] * Q[k];
        return std::sqrt(n2);
    }
    double residual(double s) const { return beta_next * std::abs(comp(m - 1, s)); }
    // Simpson estimate of int_0^h residual ds / |result(h)|
    double err(double h) const {
        if (beta_next == 0.0 || h == 0.0) return 0.0;
        const int n = 32;
        double sum = residual(0.0) + residual(h);
        for (int i = 1; i < n; ++i) sum += residual(h * i / n) * ((i & 1) ? 4.0 : 2.0);
        const double rn = result_norm(h);
        return (sum * h / (3.0 * n)) / (rn > 0.0 ? rn : 1.0);
    }
};

struct Ctx {
    const syk_ham* h;
    int dtype;
    uint64_t D;
    size_t vbytes;
    char* psi;
    char* vecs;
    LanczosScalars* sc;
    bool two_pass;
    cudaStream_t st;
    syk_stats* stats;
    char* buf(int j) const {   // buffer holding u_j
        if (j == 1) return psi;
        if (two_pass) return vecs + ((j & 1) ? vbytes : 0);
        return vecs + (size_t)(j - 2) * vbytes;
    }
};

// steps j = 1..n_steps of the recurrence; with_y: two-pass second pass, accumulate y into psi's buffer
int run_recurrence(const Ctx& c, int n_steps, bool with_y) {
    SYK_TRY(launch_norm2(c.dtype, c.D, c.psi, c.sc, c.st));
    for (int j = 1; j <= n_steps; ++j) {
        FusedArgs fa;
        fa.sc = c.sc;
        fa.j = j;
        fa.prev = j > 1 ? c.buf(j - 1) : nullptr;
        SYK_TRY(launch_apply_h(c.h, c.dtype, c.buf(j), c.buf(j + 1), fa, c.st));
        void* y = (with_y && j >= 2) ? c.psi : nullptr;
        SYK_TRY(launch_axpy_norm(c.dtype, c.D, c.buf(j + 1), c.buf(j), j, c.sc, y, j == 2, c.st));
        if (c.stats) c.stats->n_matvec += 1;
    }
    return SYK_OK;
}

// ---------------------------------------------------------------------------------------------------------
// Latency path for small vectors ("hard parts": configs[0], [1] are launch bound): the
// 2 n + 2 launches of one Lanczos round have the same arguments every time they are issued for the same (handle, buffers),
// so the round is captured ONCE into a CUDA graph (on an internal stream) and replayed with one cudaGraphLaunch on the
// caller's stream.  Keyed by everything that is baked into the kernel arguments; a small per-thread LRU cache.
// ---------------------------------------------------------------------------------------------------------
struct GraphKey {
    uint64_t uid, epoch;
    int dtype, n_steps, with_y, finalize, forced;
    const void* psi;
    const void* work;
    bool operator==(const GraphKey& o) const {
        return uid == o.uid && epoch == o.epoch && dtype == o.dtype && n_steps == o.n_steps && with_y == o.with_y &&
               finalize == o.finalize && forced == o.forced && psi == o.psi && work == o.work;
    }
};
struct GraphEntry {
    GraphKey key;
    cudaGraphExec_t exec = nullptr;   // nullptr: capture failed for this key, use direct launches
    int n_kernels = 0;
    uint64_t last_use = 0;
    int device = -1;
};
struct GraphCache {
    std::vector<GraphEntry> e;
    cudaStream_t cap = nullptr;
    int cap_device = -1;
    uint64_t clock = 0;
    ~GraphCache() {   // process exit: the context may be gone, do not touch CUDA
    }
};
thread_local GraphCache g_graphs;
constexpr size_t kMaxGraphs = 24;
constexpr size_t kGraphMaxVectorBytes = (size_t)8 << 20;   // larger vectors are not launch bound
std::atomic<int> g_graphs_on{1};

int run_recurrence_direct(const Ctx& c, int n_steps, bool with_y, bool finalize) {
    SYK_TRY(run_recurrence(c, n_steps, with_y));
    if (finalize) SYK_TRY(launch_finalize_nrm(n_steps + 1, c.sc, c.st));
    return SYK_OK;
}

// the round of run_recurrence (+ finalize_nrm) through a cached graph when the vector is small; else direct launches
int run_round(const Ctx& c, int n_steps, bool with_y, bool finalize) {
    if (!g_graphs_on.load() || c.vbytes > kGraphMaxVectorBytes || profile_enabled())
        return run_recurrence_direct(c, n_steps, with_y, finalize);
    int dev = 0;
    SYK_CUDA(cudaGetDevice(&dev));
    GraphCache& gc = g_graphs;
    const GraphKey key{c.h->uid, c.h->table_epoch, c.dtype, n_steps, with_y ? 1 : 0, finalize ? 1 : 0, c.h->forced_kernel,
                       c.psi, c.vecs};
    GraphEntry* hit = nullptr;
    for (GraphEntry& g : gc.e)
        if (g.key == key && g.device == dev) hit = &g;
    if (!hit) {
        SYK_TRY(ensure_device_tables(c.h));   // allocations cannot happen inside a capture
        if (apply_h_kernel_kind(c.h, c.dtype) == 4) SYK_TRY(prepare_dense_tables(c.h, c.dtype));
        if (gc.cap && gc.cap_device != dev) {
            cudaStreamDestroy(gc.cap);
            gc.cap = nullptr;
        }
        if (!gc.cap) {
            SYK_CUDA(cudaStreamCreateWithFlags(&gc.cap, cudaStreamNonBlocking));
            gc.cap_device = dev;
        }
        if (gc.e.size() >= kMaxGraphs) {   // evict the least recently used
            size_t lru = 0;
            for (size_t i = 1; i < gc.e.size(); ++i)
                if (gc.e[i].last_use < gc.e[lru].last_use) lru = i;
            if (gc.e[lru].exec) cudaGraphExecDestroy(gc.e[lru].exec);
            gc.e.erase(gc.e.begin() + (long)lru);
        }
        GraphEntry ne;
        ne.key = key;
        ne.device = dev;
        Ctx cc = c;
        cc.st = gc.cap;
        cc.stats = nullptr;
        const int64_t before = syk_launch_count(0);
        cudaGraph_t graph = nullptr;
        if (cudaStreamBeginCapture(gc.cap, cudaStreamCaptureModeRelaxed) == cudaSuccess) {
            const int rc = run_recurrence_direct(cc, n_steps, with_y, finalize);
            const cudaError_t e = cudaStreamEndCapture(gc.cap, &graph);
            if (rc == SYK_OK && e == cudaSuccess && graph) {
                if (cudaGraphInstantiate(&ne.exec, graph, 0) != cudaSuccess) ne.exec = nullptr;
            }
            if (graph) cudaGraphDestroy(graph);
        }
        cudaGetLastError();
        ne.n_kernels = (int)(syk_launch_count(0) - before);
        count_launch(-ne.n_kernels);   // nothing ran during the capture
        gc.e.push_back(ne);
        hit = &gc.e.back();
    }
    hit->last_use = ++gc.clock;
    if (!hit->exec) return run_recurrence_direct(c, n_steps, with_y, finalize);
    SYK_CUDA(cudaGraphLaunch(hit->exec, c.st));
    count_launch(hit->n_kernels);
    if (c.stats) c.stats->n_matvec += n_steps;
    return SYK_OK;
}

int fetch_scalars(const Ctx& c, int m, double* alpha, double* nrm) {
    SYK_CUDA(cudaMemcpyAsync(alpha, c.sc->alpha, sizeof(double) * (size_t)(m + 2), cudaMemcpyDeviceToHost, c.st));
    SYK_CUDA(cudaMemcpyAsync(nrm, c.sc->nrm, sizeof(double) * (size_t)(m + 2), cudaMemcpyDeviceToHost, c.st));
    SYK_CUDA(cudaStreamSynchronize(c.st));
    return SYK_OK;
}

int effective_dim(int m, const double* alpha, const double* nrm, double eps) {
    double scale = 0.0;
    for (int j = 1; j <= m; ++j) {
        scale = std::max(scale, std::fabs(alpha[j]));
        if (j >= 2) scale = std::max(scale, nrm[j]);
        const double b = nrm[j + 1];
        if (!(b > eps * scale) || !std::isfinite(b)) return j;   // happy breakdown: invariant subspace reached
    }
    return m;
}

// Host part of one sub-step: T_m from (alpha, nrm) -> effective dimension (happy breakdown), the longest sub-step hs
// along the ray `dir` whose error estimate fits its share of the budget, and the coefficients coef[j] =
// [exp(-i dir hs T) e_1]_j * nrm[1] (j = 1..me) of the result in the Lanczos basis.
struct StepChoice {
    int me;
    double hs;
    double err;
    bool noconv;
    double growth;   // |exp(-i dir hs T) e_1| = |result| / |input| of the sub-step
};

StepChoice choose_step(int m, const double* alpha, const double* nrm, cplx dir, double tol, double len, double remaining,
                       double eps_break, bool last_allowed, double2* coef, bool renormalize = false) {
    StepChoice ch{};
    const int me = effective_dim(m, alpha, nrm, eps_break);
    SmallExp se;
    se.m = me;
    se.dir = dir;
    se.beta_next = me < m ? 0.0 : nrm[m + 1];
    std::vector<double> A((size_t)me * me, 0.0);
    for (int j = 1; j <= me; ++j) {
        A[(size_t)(j - 1) * me + (j - 1)] = alpha[j];
        if (j < me) A[(size_t)(j - 1) * me + j] = A[(size_t)j * me + (j - 1)] = nrm[j + 1];
    }
    jacobi_eig(me, A, se.theta, se.Q);
    // longest sub-step whose error estimate fits its share of the budget
    auto fits = [&](double hs) { return se.err(hs) <= tol * hs / len; };
    double hs = remaining;
    if (!fits(hs)) {
        if (last_allowed) {
            ch.noconv = true;   // forced: take the remainder in one step
        } else {
            double lo = 0.0, hi = remaining;
            for (int it = 0; it < 14; ++it) {   // the step length needs no precision: `lo` always fits the budget
                const double mid = 0.5 * (lo + hi);
                if (fits(mid)) lo = mid; else hi = mid;
            }
            hs = lo;
            if (!(hs > 1e-9 * len)) {   // estimate never fits: Krylov space too small for this tolerance
                ch.noconv = true;
                hs = std::min(remaining, std::max(hi, 1e-6 * len));
            }
        }
    }
    ch.me = me;
    ch.hs = hs;
    ch.err = se.err(hs);
    ch.growth = se.result_norm(hs);
    // renormalize: the result keeps the norm of the input, the factor goes to log_norm
    const double keep = (renormalize && ch.growth > 0.0) ? 1.0 / ch.growth : 1.0;
    for (int j = 1; j <= me; ++j) {
        const cplx v = se.comp(j - 1, hs) * (nrm[1] * keep);
        coef[j] = make_double2(v.real(), v.imag());
    }
    return ch;
}

bool valid_args(const syk_ham* h, int dtype, const void* psi, const void* work) {
    return h && h->L <= 32 && (dtype == SYK_C64 || dtype == SYK_C128) && psi && work && ((uintptr_t)psi & 15) == 0 &&
           ((uintptr_t)work & 15) == 0;
}

int resolve_dim(const syk_ham* h, const syk_krylov_opts* o) {
    int m = (o && o->krylov_dim > 0) ? o->krylov_dim : 24;
    const uint64_t D = 1ull << h->L;
    if (m > kMaxKrylov) m = kMaxKrylov;
    if ((uint64_t)m > D) m = (int)D;
    return m;
}

}  // namespace

int krylov_evolve_impl(const syk_ham* h, int dtype, void* d_psi, double tau_re, double tau_im,
                       const syk_krylov_opts* opts, void* d_work, size_t work_bytes, syk_stats* stats,
                       cudaStream_t st) {
    if (!valid_args(h, dtype, d_psi, d_work) || !std::isfinite(tau_re) || !std::isfinite(tau_im)) return SYK_EINVAL;
    if (opts && (opts->krylov_dim < 0 || opts->krylov_dim == 1 || opts->tol < 0 || opts->max_substeps < 0))
        return SYK_EINVAL;
    if (!h->hermitian)   // no three-term recurrence without H = H^+: Arnoldi (NEXT-4)
        return arnoldi_evolve_impl(h, dtype, d_psi, tau_re, tau_im, opts, d_work, work_bytes, stats, st);
    const int m = resolve_dim(h, opts);
    const bool two_pass = opts && opts->two_pass;
    const double tol = (opts && opts->tol > 0) ? opts->tol : (dtype == SYK_C128 ? 1e-12 : 1e-6);
    const int max_sub = (opts && opts->max_substeps > 0) ? opts->max_substeps : 100000;
    const bool renorm = opts && opts->renormalize;

    Ctx c;
    c.h = h;
    c.dtype = dtype;
    c.D = 1ull << h->L;
    c.vbytes = (size_t)c.D * elem_bytes(dtype);
    c.psi = (char*)d_psi;
    c.sc = (LanczosScalars*)d_work;
    c.vecs = (char*)d_work + krylov_header_bytes();
    c.two_pass = two_pass;
    c.st = st;
    c.stats = stats;
    const size_t need = krylov_header_bytes() + (size_t)(two_pass ? 2 : m) * c.vbytes;
    if (work_bytes < need) return SYK_ENOMEM;
    {   // psi must not overlap the work space
        const uintptr_t a = (uintptr_t)d_psi, b = (uintptr_t)d_work;
        if (a < b + need && b < a + c.vbytes) return SYK_EINVAL;
    }

    const double len = std::hypot(tau_re, tau_im);
    if (len == 0.0 || h->n_terms() == 0) return SYK_OK;
    const cplx dir(tau_re / len, tau_im / len);
    const double eps_break = dtype == SYK_C128 ? 1e-13 : 2e-6;
    const double V = (double)c.vbytes, Dx = (double)h->n_groups();

    double remaining = len;
    int rc = SYK_OK;
    std::vector<double> alpha(kMaxKrylov + 2), nrm(kMaxKrylov + 2);
    std::vector<double2> coef(kMaxKrylov + 2);
    int n_sub = 0;
    while (remaining > 1e-15 * len) {
        ++n_sub;
        SYK_TRY(run_round(c, m, false, true));
        SYK_TRY(fetch_scalars(c, m, alpha.data(), nrm.data()));
        if (!(nrm[1] > 0.0)) return SYK_OK;   // zero vector stays zero
        const StepChoice ch = choose_step(m, alpha.data(), nrm.data(), dir, tol, len, remaining, eps_break,
                                          n_sub >= max_sub, coef.data(), renorm);
        if (renorm && stats && ch.growth > 0.0) stats->log_norm += std::log(ch.growth);
        const int me = ch.me;
        const double hs = ch.hs;
        if (ch.noconv) rc = SYK_ENOCONV;
        if (stats) {
            stats->err_est += ch.err;
            stats->krylov_dim_used = stats->krylov_dim_used == 0 ? me : std::min(stats->krylov_dim_used, me);
            stats->n_substeps += 1;
        }
        SYK_CUDA(cudaMemcpyAsync(c.sc->coef, coef.data(), sizeof(double2) * (size_t)(me + 1), cudaMemcpyHostToDevice, st));
        if (!two_pass) {
            SYK_TRY(launch_combine(dtype, c.D, c.psi, c.vecs, c.D, me, c.sc, st));
            if (stats) stats->model_bytes += m * ((Dx + 3.0) * V + 3.0 * V) + V + (me + 1.0) * V;
        } else {
            if (me == 1) {
                SYK_TRY(launch_axpy_coef(dtype, c.D, c.psi, nullptr, 1, 1, c.sc, st));
            } else {
                SYK_TRY(run_round(c, me - 1, true, false));
                SYK_TRY(launch_axpy_coef(dtype, c.D, c.psi, c.buf(me), me, me == 2, c.sc, st));
            }
            if (stats) stats->model_bytes += (m + me - 1) * ((Dx + 3.0) * V + 3.0 * V) + 2.0 * V + 2.0 * me * V;
        }
        remaining -= hs;
    }
    return rc;
}

// ---------------------------------------------------------------------------------------------------------
// Batched over disorder realizations (BASELINE configs[1]): every kernel runs with grid.y = realization,
// so the nb realizations advance through the Lanczos recurrence in lock step and share launches; the host does the nb
// small exponentials between two rounds.  One-pass only.  Work space: table descriptors | nb x (scalars header + m
// vectors).  A realization that has reached its target time keeps coef = identity (psi unchanged) while the others
// finish.
// ---------------------------------------------------------------------------------------------------------
int resolve_krylov_dim(const syk_ham* h, const syk_krylov_opts* o) { return resolve_dim(h, o); }
void set_graphs(int on) { g_graphs_on.store(on); }

size_t krylov_batched_bytes(const syk_ham* h0, int nb, int dtype, int m) {
    const size_t v = ((size_t)1 << h0->L) * elem_bytes(dtype);
    return batched_table_bytes(nb) + (size_t)nb * (krylov_header_bytes() + (size_t)m * v);
}

int krylov_evolve_batched_impl(const syk_ham* const* hams, int nb, int dtype, void* d_psi, size_t psi_stride_bytes,
                               double tau_re, double tau_im, const syk_krylov_opts* opts, void* d_work,
                               size_t work_bytes, syk_stats* stats, bool* tables_uploaded, cudaStream_t st) {
    const syk_ham* h0 = hams[0];
    const int m = resolve_dim(h0, opts);
    const double tol = (opts && opts->tol > 0) ? opts->tol : (dtype == SYK_C128 ? 1e-12 : 1e-6);
    const int max_sub = (opts && opts->max_substeps > 0) ? opts->max_substeps : 100000;
    const uint64_t D = 1ull << h0->L;
    const size_t vbytes = (size_t)D * elem_bytes(dtype);
    const size_t ws_stride = krylov_header_bytes() + (size_t)m * vbytes;
    if (work_bytes < krylov_batched_bytes(h0, nb, dtype, m)) return SYK_ENOMEM;
    {   // the states must not overlap the work space
        const uintptr_t a = (uintptr_t)d_psi, b = (uintptr_t)d_work;
        const size_t span = (size_t)(nb - 1) * psi_stride_bytes + vbytes;
        if (a < b + krylov_batched_bytes(h0, nb, dtype, m) && b < a + span) return SYK_EINVAL;
    }
    char* tab = (char*)d_work;
    char* ws = tab + batched_table_bytes(nb);                 // realization r: header at ws + r ws_stride, then m vectors
    char* vecs = ws + krylov_header_bytes();
    char* psi = (char*)d_psi;
    const double len = std::hypot(tau_re, tau_im);
    if (len == 0.0) return SYK_OK;
    const cplx dir(tau_re / len, tau_im / len);
    const double eps_break = dtype == SYK_C128 ? 1e-13 : 2e-6;
    // buffer of u_j: j == 1 -> psi (user stride), else work vector j-2 (work-space stride)
    auto buf = [&](int j) { return j == 1 ? psi : vecs + (size_t)(j - 2) * vbytes; };
    auto stride = [&](int j) { return j == 1 ? psi_stride_bytes : ws_stride; };

    std::vector<double> remaining((size_t)nb, len);
    std::vector<double> alpha((size_t)nb * (kMaxKrylov + 2)), nrm((size_t)nb * (kMaxKrylov + 2));
    std::vector<double2> coef((size_t)nb * (kMaxKrylov + 2));
    std::vector<int> meff((size_t)nb, 1);
    const size_t row = sizeof(double) * (kMaxKrylov + 2);
    int rc = SYK_OK;
    for (int n_sub = 1;; ++n_sub) {
        bool any = false;
        for (int r = 0; r < nb; ++r) any |= remaining[(size_t)r] > 1e-15 * len;
        if (!any) break;
        Batch b;
        b.n = nb;
        b.s.sc = ws_stride;
        b.s.a = psi_stride_bytes;
        SYK_TRY(launch_norm2(dtype, D, psi, (LanczosScalars*)ws, st, b));
        for (int j = 1; j <= m; ++j) {
            SYK_TRY(launch_apply_h_batched(hams, nb, dtype, tab, !*tables_uploaded, buf(j), stride(j), buf(j + 1),
                                           stride(j + 1), j > 1 ? buf(j - 1) : nullptr, j > 1 ? stride(j - 1) : 0, ws,
                                           ws_stride, j, st));
            *tables_uploaded = true;
            Batch ba;
            ba.n = nb;
            ba.s.a = stride(j + 1);
            ba.s.b = stride(j);
            ba.s.sc = ws_stride;
            SYK_TRY(launch_axpy_norm(dtype, D, buf(j + 1), buf(j), j, (LanczosScalars*)ws, nullptr, 0, st, ba));
            if (stats) stats->n_matvec += nb;
        }
        Batch bf;
        bf.n = nb;
        bf.s.sc = ws_stride;
        SYK_TRY(launch_finalize_nrm(m + 1, (LanczosScalars*)ws, st, bf));
        SYK_CUDA(cudaMemcpy2DAsync(alpha.data(), row, ws + offsetof(LanczosScalars, alpha), ws_stride, row, (size_t)nb,
                                   cudaMemcpyDeviceToHost, st));
        SYK_CUDA(cudaMemcpy2DAsync(nrm.data(), row, ws + offsetof(LanczosScalars, nrm), ws_stride, row, (size_t)nb,
                                   cudaMemcpyDeviceToHost, st));
        SYK_CUDA(cudaStreamSynchronize(st));
        // the nb small exponentials are independent: spread them over a few host threads
        std::vector<StepChoice> choice((size_t)nb);
        std::vector<char> active((size_t)nb, 0);
        auto work = [&](int r0, int r1) {
            for (int r = r0; r < r1; ++r) {
                const double* a = alpha.data() + (size_t)r * (kMaxKrylov + 2);
                const double* nr = nrm.data() + (size_t)r * (kMaxKrylov + 2);
                double2* cf = coef.data() + (size_t)r * (kMaxKrylov + 2);
                for (int j = 0; j < kMaxKrylov + 2; ++j) cf[j] = make_double2(0.0, 0.0);
                if (!(remaining[(size_t)r] > 1e-15 * len) || !(nr[1] > 0.0)) {
                    cf[1] = make_double2(nr[1], 0.0);   // identity: psi stays what it is
                    continue;
                }
                active[(size_t)r] = 1;
                choice[(size_t)r] = choose_step(m, a, nr, dir, tol, len, remaining[(size_t)r], eps_break,
                                                n_sub >= max_sub, cf);
            }
        };
        {
            const int n_thr = std::max(1, std::min({nb, 8, (int)std::thread::hardware_concurrency()}));
            std::vector<std::thread> pool;
            const int per = (nb + n_thr - 1) / n_thr;
            for (int k = 1; k < n_thr; ++k)
                if (k * per < nb) pool.emplace_back(work, k * per, std::min(nb, (k + 1) * per));
            work(0, std::min(nb, per));
            for (auto& th : pool) th.join();
        }
        for (int r = 0; r < nb; ++r) {
            meff[(size_t)r] = 1;
            if (!active[(size_t)r]) {
                remaining[(size_t)r] = 0.0;
                continue;
            }
            const StepChoice& ch = choice[(size_t)r];
            if (ch.noconv) rc = SYK_ENOCONV;
            meff[(size_t)r] = ch.me;
            remaining[(size_t)r] -= ch.hs;
            if (stats) {
                stats->err_est = std::max(stats->err_est, ch.err);
                stats->krylov_dim_used = stats->krylov_dim_used == 0 ? ch.me : std::min(stats->krylov_dim_used, ch.me);
            }
        }
        if (stats) {
            stats->n_substeps += 1;
            const double V = (double)vbytes;
            for (int r = 0; r < nb; ++r)
                stats->model_bytes += m * (((double)hams[r]->n_groups() + 3.0) * V + 3.0 * V) + V + (m + 1.0) * V;
        }
        SYK_CUDA(cudaMemcpy2DAsync(ws + offsetof(LanczosScalars, coef), ws_stride, coef.data(),
                                   sizeof(double2) * (kMaxKrylov + 2), sizeof(double2) * (kMaxKrylov + 2), (size_t)nb,
                                   cudaMemcpyHostToDevice, st));
        SYK_CUDA(cudaMemcpy2DAsync(ws + offsetof(LanczosScalars, m_eff), ws_stride, meff.data(), sizeof(int), sizeof(int),
                                   (size_t)nb, cudaMemcpyHostToDevice, st));
        Batch bc;
        bc.n = nb;
        bc.s.a = psi_stride_bytes;
        bc.s.b = ws_stride;
        bc.s.sc = ws_stride;
        SYK_TRY(launch_combine(dtype, D, psi, vecs, D, -1, (LanczosScalars*)ws, st, bc));
        SYK_CUDA(cudaStreamSynchronize(st));   // coef / meff host buffers are reused in the next round
    }
    return rc;
}

}  // namespace syk

extern "C" {

int syk_set_cuda_graphs(int on) {
    syk::set_graphs(on != 0);
    return SYK_OK;
}

int syk_krylov_workspace_bytes_batched(const syk_ham* h, int n_batch, int dtype, const syk_krylov_opts* opts,
                                       size_t* bytes) {
    if (!h || !bytes || n_batch < 1 || (dtype != SYK_C64 && dtype != SYK_C128)) return SYK_EINVAL;
    if (opts && (opts->krylov_dim < 0 || opts->krylov_dim == 1 || opts->two_pass)) return SYK_EINVAL;
    *bytes = syk::krylov_batched_bytes(h, n_batch, dtype, syk::resolve_dim(h, opts));
    return SYK_OK;
}

int syk_krylov_evolve_batched(const syk_ham* const* hams, int n_batch, int dtype, void* d_psi, int64_t batch_stride,
                              double tau_re, double tau_im, const syk_krylov_opts* opts, void* d_work, size_t work_bytes,
                              syk_stats* stats, void* stream) {
    if (!hams || n_batch < 1 || !hams[0] || !syk::valid_args(hams[0], dtype, d_psi, d_work) || !std::isfinite(tau_re) ||
        !std::isfinite(tau_im))
        return SYK_EINVAL;
    if (opts && (opts->krylov_dim < 0 || opts->krylov_dim == 1 || opts->tol < 0 || opts->max_substeps < 0 || opts->two_pass ||
                 opts->renormalize))
        return SYK_EINVAL;
    if (batch_stride < ((int64_t)1 << hams[0]->L) || ((size_t)batch_stride * syk::elem_bytes(dtype)) % 16) return SYK_EINVAL;
    if (!syk::batched_apply_ok(hams, n_batch, dtype)) return SYK_EINVAL;
    if (stats) *stats = syk_stats{};
    bool uploaded = false;
    return syk::krylov_evolve_batched_impl(hams, n_batch, dtype, d_psi, (size_t)batch_stride * syk::elem_bytes(dtype),
                                           tau_re, tau_im, opts, d_work, work_bytes, stats, &uploaded,
                                           (cudaStream_t)stream);
}

int syk_krylov_workspace_bytes(const syk_ham* h, int dtype, const syk_krylov_opts* opts, size_t* bytes) {
    if (!h || h->L > 32 || !bytes || (dtype != SYK_C64 && dtype != SYK_C128)) return SYK_EINVAL;
    if (opts && (opts->krylov_dim < 0 || opts->krylov_dim == 1)) return SYK_EINVAL;
    const int m = syk::resolve_dim(h, opts);
    const size_t v = ((size_t)1 << h->L) * syk::elem_bytes(dtype);
    *bytes = syk::krylov_header_bytes() + (size_t)((opts && opts->two_pass) ? 2 : m) * v;
    return SYK_OK;
}

int syk_krylov_evolve(const syk_ham* h, int dtype, void* d_psi, double tau_re, double tau_im,
                      const syk_krylov_opts* opts, void* d_work, size_t work_bytes, syk_stats* stats, void* stream) {
    cudaStream_t st = (cudaStream_t)stream;
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    if (stats) {
        *stats = syk_stats{};
        SYK_CUDA(cudaEventCreate(&e0));
        SYK_CUDA(cudaEventCreate(&e1));
        SYK_CUDA(cudaEventRecord(e0, st));
    }
    int rc = syk::krylov_evolve_impl(h, dtype, d_psi, tau_re, tau_im, opts, d_work, work_bytes, stats, st);
    if (stats) {
        if (rc == SYK_OK || rc == SYK_ENOCONV) {
            float ms = 0.f;
            if (cudaEventRecord(e1, st) == cudaSuccess && cudaEventSynchronize(e1) == cudaSuccess &&
                cudaEventElapsedTime(&ms, e0, e1) == cudaSuccess)
                stats->elapsed_ms = ms;
        }
        cudaEventDestroy(e0);
        cudaEventDestroy(e1);
    }
    return rc;
}

int syk_lanczos_run(const syk_ham* h, int dtype, const void* d_psi, int m, double* alpha, double* beta,
                    void* d_work, size_t work_bytes, syk_stats* stats, void* stream) {
    if (!syk::valid_args(h, dtype, d_psi, d_work) || !alpha || !beta || m < 1 || m > syk::kMaxKrylov || !h->hermitian)
        return SYK_EINVAL;
    cudaStream_t st = (cudaStream_t)stream;
    syk::Ctx c;
    c.h = h;
    c.dtype = dtype;
    c.D = 1ull << h->L;
    c.vbytes = (size_t)c.D * syk::elem_bytes(dtype);
    c.psi = (char*)const_cast<void*>(d_psi);
    c.sc = (syk::LanczosScalars*)d_work;
    c.vecs = (char*)d_work + syk::krylov_header_bytes();
    c.two_pass = false;
    c.st = st;
    c.stats = stats;
    if (work_bytes < syk::krylov_header_bytes() + (size_t)m * c.vbytes) return SYK_ENOMEM;
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    if (stats) {
        *stats = syk_stats{};
        SYK_CUDA(cudaEventCreate(&e0));
        SYK_CUDA(cudaEventCreate(&e1));
        SYK_CUDA(cudaEventRecord(e0, st));
    }
    int rc = syk::run_recurrence(c, m, false);
    if (rc == SYK_OK) rc = syk::launch_finalize_nrm(m + 1, c.sc, st);
    if (rc == SYK_OK && stats) {
        float ms = 0.f;
        if (cudaEventRecord(e1, st) == cudaSuccess && cudaEventSynchronize(e1) == cudaSuccess &&
            cudaEventElapsedTime(&ms, e0, e1) == cudaSuccess)
            stats->elapsed_ms = ms;
        const double V = (double)c.vbytes;
        stats->model_bytes = m * ((double)h->n_groups() + 6.0) * V + V;
        stats->krylov_dim_used = m;
    }
    if (stats) {
        cudaEventDestroy(e0);
        cudaEventDestroy(e1);
    }
    SYK_TRY(rc);
    std::vector<double> a(syk::kMaxKrylov + 2), n(syk::kMaxKrylov + 2);
    SYK_TRY(syk::fetch_scalars(c, m, a.data(), n.data()));
    for (int j = 1; j <= m; ++j) alpha[j - 1] = a[j];
    for (int j = 0; j <= m; ++j) beta[j] = n[j + 1];
    return SYK_OK;
}

}  // extern "C"
