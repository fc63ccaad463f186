// a-4 for NON-HERMITIAN operators ("non-Hermitian SYK"): psi <- exp(-i tau H) psi by the
// Arnoldi process.  Without H = H^+ the three-term recurrence of krylov.cu does not hold: the new vector is orthogonalised
// against ALL previous ones (classical Gram-Schmidt, applied twice), the projected matrix is an upper Hessenberg matrix
//     H_m = V_m^+ H V_m   (complex, m x m),      H V_m = V_m H_m + h_{m+1,m} v_{m+1} e_m^T,
// and the small exponential exp(-i tau H_m) e_1 is taken on the host by scaling and squaring.  Same a-posteriori
// estimate and sub-stepping as the Lanczos driver: the longest step h along the ray of tau with
//     int_0^h h_{m+1,m} |e_m^T exp(-i dir s H_m) e_1| ds / |exp(-i dir h H_m) e_1|  <=  tol h / |tau|.
// One-pass only (m work vectors: v_2 .. v_{m+1}; v_1 lives in psi's buffer).  Every product is a plain apply_H launch
// (any kernel kind; the fused Lanczos epilogue is not used); dots and norms are the deterministic fp64 reductions of
// vector_ops.cu.  This path is about generality, not speed: 2 j inner products per step, each fetched to the host.
#include <algorithm>
#include <cmath>
#include <complex>
#include <vector>

#include "common.h"

namespace syk {

namespace {

using cplx = std::complex<double>;

// C = A B for n x n row-major complex matrices
void matmul(int n, const std::vector<cplx>& A, const std::vector<cplx>& B, std::vector<cplx>& C) {
    C.assign((size_t)n * n, cplx(0.0));
    for (int i = 0; i < n; ++i)
        for (int k = 0; k < n; ++k) {
            const cplx a = A[(size_t)i * n + k];
            if (a == cplx(0.0)) continue;
            for (int j = 0; j < n; ++j) C[(size_t)i * n + j] += a * B[(size_t)k * n + j];
        }
}

// exp(A) by scaling and squaring with a Taylor series (|A / 2^s|_1 <= 1/4, 20 terms: remainder < 1e-30)
void expm(int n, const std::vector<cplx>& A, std::vector<cplx>& E) {
    double norm1 = 0.0;
    for (int j = 0; j < n; ++j) {
        double col = 0.0;
        for (int i = 0; i < n; ++i) col += std::abs(A[(size_t)i * n + j]);
        norm1 = std::max(norm1, col);
    }
    int s = 0;
    while (std::ldexp(norm1, -s) > 0.25 && s < 60) ++s;
    std::vector<cplx> B(A), term, tmp;
    const double scale = std::ldexp(1.0, -s);
    for (cplx& v : B) v *= scale;
    E.assign((size_t)n * n, cplx(0.0));
    for (int i = 0; i < n; ++i) E[(size_t)i * n + i] = 1.0;
    term = E;
    for (int k = 1; k <= 20; ++k) {
        matmul(n, term, B, tmp);
        for (cplx& v : tmp) v /= (double)k;
        term.swap(tmp);
        for (size_t i = 0; i < E.size(); ++i) E[i] += term[i];
    }
    for (int q = 0; q < s; ++q) {
        matmul(n, E, E, tmp);
        E.swap(tmp);
    }
}

// exp(-i dir s H_m) e_1 sampled along the ray: y(s + ds) = exp(-i dir ds H_m) y(s), ds = h / n
struct HessExp {
    int m = 0;
    std::vector<cplx> H;       // m x m, row-major
    double h_next = 0.0;       // h_{m+1,m}
    cplx dir;
    // Simpson estimate of int_0^h residual ds / |y(h)| and the coefficient vector y(h)
    double err(double h, std::vector<cplx>* y_out) const {
        const int n = 32;
        std::vector<cplx> A((size_t)m * m), E;
        const cplx f = cplx(0.0, -1.0) * dir * (h / n);
        for (size_t i = 0; i < A.size(); ++i) A[i] = f * H[i];
        expm(m, A, E);
        std::vector<cplx> y((size_t)m, cplx(0.0)), z((size_t)m);
        y[0] = 1.0;
        double sum = h_next * std::abs(y[(size_t)m - 1]);
        for (int i = 1; i <= n; ++i) {
            for (int r = 0; r < m; ++r) {
                cplx acc = 0.0;
                for (int c = 0; c < m; ++c) acc += E[(size_t)r * m + c] * y[(size_t)c];
                z[(size_t)r] = acc;
            }
            y.swap(z);
            const double res = h_next * std::abs(y[(size_t)m - 1]);
            sum += res * (i == n ? 1.0 : ((i & 1) ? 4.0 : 2.0));
        }
        double n2 = 0.0;
        for (const cplx& v : y) n2 += std::norm(v);
        if (y_out) *y_out = y;
        if (h_next == 0.0 || h == 0.0) return 0.0;
        const double rn = std::sqrt(n2);
        return (sum * h / (3.0 * n)) / (rn > 0.0 ? rn : 1.0);
    }
};

}  // namespace

int arnoldi_evolve_impl(const syk_ham* h, int dtype, void* d_psi, double tau_re, double tau_im, const syk_krylov_opts* opts,
                        void* d_work, size_t work_bytes, syk_stats* stats, cudaStream_t st) {
    if (opts && opts->two_pass) return SYK_EINVAL;   // the two-pass scheme relies on the three-term recurrence
    const int m = resolve_krylov_dim(h, opts);
    const double tol = (opts && opts->tol > 0) ? opts->tol : (dtype == SYK_C128 ? 1e-12 : 1e-6);
    const int max_sub = (opts && opts->max_substeps > 0) ? opts->max_substeps : 100000;
    const uint64_t D = 1ull << h->L;
    const size_t vbytes = (size_t)D * elem_bytes(dtype);
    const size_t need = krylov_header_bytes() + (size_t)m * vbytes;
    if (work_bytes < need) return SYK_ENOMEM;
    {
        const uintptr_t a = (uintptr_t)d_psi, b = (uintptr_t)d_work;
        if (a < b + need && b < a + vbytes) return SYK_EINVAL;
    }
    LanczosScalars* sc = (LanczosScalars*)d_work;
    char* vecs = (char*)d_work + krylov_header_bytes();
    auto vec = [&](int j) -> char* { return j == 1 ? (char*)d_psi : vecs + (size_t)(j - 2) * vbytes; };   // v_j, j = 1..m+1

    const double len = std::hypot(tau_re, tau_im);
    if (len == 0.0 || h->n_terms() == 0) return SYK_OK;
    const cplx dir(tau_re / len, tau_im / len);
    const double eps_break = dtype == SYK_C128 ? 1e-13 : 2e-6;
    const double V = (double)vbytes, Dx = (double)h->n_groups();

    std::vector<double> ones(kMaxKrylov + 2, 1.0);
    std::vector<double2> coef(kMaxKrylov + 2);
    auto fetch_norm = [&](int j, double* out) -> int {   // |v| from the partial sums left by launch_norm2
        SYK_TRY(launch_finalize_nrm(j, sc, st));
        SYK_CUDA(cudaMemcpyAsync(out, &sc->nrm[j], sizeof(double), cudaMemcpyDeviceToHost, st));
        SYK_CUDA(cudaStreamSynchronize(st));
        return SYK_OK;
    };
    auto upload_unit_norms = [&]() -> int {
        SYK_CUDA(cudaMemcpyAsync(sc->nrm, ones.data(), sizeof(double) * (size_t)(m + 2), cudaMemcpyHostToDevice, st));
        return SYK_OK;
    };

    double remaining = len;
    int rc = SYK_OK, n_sub = 0;
    while (remaining > 1e-15 * len) {
        ++n_sub;
        double beta0 = 0.0;
        SYK_TRY(launch_norm2(dtype, D, vec(1), sc, st));
        SYK_TRY(fetch_norm(1, &beta0));
        if (!(beta0 > 0.0)) return SYK_OK;   // zero vector stays zero
        SYK_TRY(launch_normalise(dtype, D, vec(1), sc, st));
        HessExp he;
        he.dir = dir;
        std::vector<cplx> Hfull((size_t)(m + 1) * m, cplx(0.0));   // (m+1) x m
        int me = m;
        double scale_seen = 0.0;
        for (int j = 1; j <= m; ++j) {
            FusedArgs plain;
            SYK_TRY(launch_apply_h(h, dtype, vec(j), vec(j + 1), plain, st));
            if (stats) stats->n_matvec += 1;
            for (int pass = 0; pass < 2; ++pass) {   // classical Gram-Schmidt, twice
                for (int i = 1; i <= j; ++i) {
                    double d[2];
                    SYK_TRY(launch_cdot(dtype, D, vec(i), vec(j + 1), sc, st));
                    SYK_TRY(fetch_cdot(sc, d, st));
                    Hfull[(size_t)(i - 1) * m + (j - 1)] += cplx(d[0], d[1]);
                    coef[(size_t)i] = make_double2(-d[0], -d[1]);
                }
                SYK_CUDA(cudaMemcpyAsync(sc->coef, coef.data(), sizeof(double2) * (size_t)(j + 1), cudaMemcpyHostToDevice, st));
                SYK_TRY(upload_unit_norms());
                for (int i = 1; i <= j; ++i) SYK_TRY(launch_axpy_coef(dtype, D, vec(j + 1), vec(i), i, 0, sc, st));
                SYK_CUDA(cudaStreamSynchronize(st));   // coef is reused
            }
            double hn = 0.0;
            SYK_TRY(launch_norm2(dtype, D, vec(j + 1), sc, st));
            SYK_TRY(fetch_norm(j + 1, &hn));
            for (int i = 1; i <= j; ++i) scale_seen = std::max(scale_seen, std::abs(Hfull[(size_t)(i - 1) * m + (j - 1)]));
            Hfull[(size_t)j * m + (j - 1)] = hn;
            if (!(hn > eps_break * scale_seen) || !std::isfinite(hn)) {   // invariant subspace reached: exact in j steps
                me = j;
                he.h_next = 0.0;
                break;
            }
            he.h_next = hn;
            if (j < m) SYK_TRY(launch_normalise(dtype, D, vec(j + 1), sc, st));
        }
        he.m = me;
        he.H.assign((size_t)me * me, cplx(0.0));
        for (int i = 0; i < me; ++i)
            for (int k = 0; k < me; ++k) he.H[(size_t)i * me + k] = Hfull[(size_t)i * m + k];
        // longest sub-step whose error estimate fits its share of the budget
        std::vector<cplx> y;
        auto fits = [&](double hs) { return he.err(hs, &y) <= tol * hs / len; };
        double hs = remaining;
        bool noconv = false;
        if (!fits(hs)) {
            if (n_sub >= max_sub) {
                noconv = true;
            } else {
                double lo = 0.0, hi = remaining;
                for (int it = 0; it < 14; ++it) {
                    const double mid = 0.5 * (lo + hi);
                    if (fits(mid)) lo = mid; else hi = mid;
                }
                hs = lo;
                if (!(hs > 1e-9 * len)) {
                    noconv = true;
                    hs = std::min(remaining, std::max(hi, 1e-6 * len));
                }
            }
        }
        const double err = he.err(hs, &y);
        if (noconv) rc = SYK_ENOCONV;
        if (stats) {
            stats->err_est += err;
            stats->krylov_dim_used = stats->krylov_dim_used == 0 ? me : std::min(stats->krylov_dim_used, me);
            stats->n_substeps += 1;
            stats->model_bytes += me * ((Dx + 2.0) * V) + (double)me * (me + 1) * 5.0 * V + (me + 1.0) * V;
        }
        double scale = beta0;
        if (opts && opts->renormalize) {   // the result keeps the norm of the input, the factor goes to log_norm
            double n2 = 0.0;
            for (int j = 0; j < me; ++j) n2 += std::norm(y[(size_t)j]);
            if (n2 > 0.0) {
                scale = beta0 / std::sqrt(n2);
                if (stats) stats->log_norm += 0.5 * std::log(n2);
            }
        }
        for (int j = 1; j <= me; ++j) coef[(size_t)j] = make_double2(scale * y[(size_t)j - 1].real(), scale * y[(size_t)j - 1].imag());
        SYK_CUDA(cudaMemcpyAsync(sc->coef, coef.data(), sizeof(double2) * (size_t)(me + 1), cudaMemcpyHostToDevice, st));
        SYK_TRY(upload_unit_norms());
        SYK_TRY(launch_combine(dtype, D, vec(1), vecs, D, me, sc, st));
        SYK_CUDA(cudaStreamSynchronize(st));
        remaining -= hs;
    }
    return rc;
}

}  // namespace syk
