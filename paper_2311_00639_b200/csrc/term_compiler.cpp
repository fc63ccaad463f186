// a-1  Host term compiler: Eq. (1) -> Pauli strings c Z^z X^x grouped by X-mask.
//
// Every Jordan-Wigner Majorana (R-JW) is one string:  gamma_{2q}   = s   Z^{(1<<q)-1}     X^{1<<q}
//                                                     gamma_{2q+1} = -is Z^{(1<<(q+1))-1} X^{1<<q}   (Y = -i Z X)
// and strings multiply by XOR of the masks plus a sign ("the product of two sigma matrices
// coincides with the XOR of their bit strings up to a sign"):
//     (i^a Z^{z1} X^{x1}) (i^b Z^{z2} X^{x2}) = i^{a+b+2 popcount(x1 & z2)} Z^{z1^z2} X^{x1^x2}
// because moving X^{x1} through Z^{z2} costs (-1)^{popcount(x1 & z2)}.  Phases are tracked as powers of i, so
// the coefficient of a term is exactly real or exactly imaginary.  Operator sum = merge of lists with equal
// (x, z) combined.
#include <algorithm>
#include <cmath>
#include <new>
#include <numeric>

#include "common.h"

namespace {

struct PauliString {
    uint64_t x, z;
    int ipow;   // phase i^ipow
};

inline PauliString jw_gamma(int n) {
    int q = n >> 1;
    PauliString s;
    s.x = 1ull << q;
    if ((n & 1) == 0) {
        s.z = (1ull << q) - 1;
        s.ipow = 0;
    } else {
        s.z = (1ull << (q + 1)) - 1;   // q + 1 <= N/2 <= 32
        s.ipow = 3;   // -i
    }
    return s;
}

inline PauliString mul(const PauliString& a, const PauliString& b) {
    PauliString r;
    r.x = a.x ^ b.x;
    r.z = a.z ^ b.z;
    r.ipow = (a.ipow + b.ipow + 2 * __builtin_popcountll(a.x & b.z)) & 3;
    return r;
}

struct RawTerm {
    uint64_t x, z;
    std::complex<double> c;
    int32_t q[4];
    double J;
};

int compile(int N, int gamma_norm, std::vector<RawTerm>& raw, syk_ham** out) {
    // canonical order: ascending x, then ascending z; equal (x, z) are combined
    std::stable_sort(raw.begin(), raw.end(), [](const RawTerm& a, const RawTerm& b) {
        return a.x != b.x ? a.x < b.x : a.z < b.z;
    });
    syk_ham* h = new (std::nothrow) syk_ham();
    if (!h) return SYK_ENOMEM;
    h->N = N;
    h->L = N / 2;
    h->gamma_norm = gamma_norm;
    try {
        for (size_t t = 0; t < raw.size(); ++t) {
            const RawTerm& r = raw[t];
            if (!h->z.empty() && h->x.back() == r.x && h->z.back() == r.z) {   // duplicate string: add
                h->c.back() += r.c;
                h->J.back() += r.J;
                continue;
            }
            if (h->x.empty() || h->x.back() != r.x) {
                h->x.push_back(r.x);
                h->group_off.push_back((uint32_t)h->z.size());
            }
            h->z.push_back(r.z);
            h->c.push_back(r.c);
            h->J.push_back(r.J);
            h->quartet.insert(h->quartet.end(), r.q, r.q + 4);
        }
        h->group_off.push_back((uint32_t)h->z.size());
    } catch (const std::bad_alloc&) {
        delete h;
        return SYK_ENOMEM;
    }
    *out = h;
    return SYK_OK;
}

bool make_term(int N, int gamma_norm, const int32_t* q, double J, RawTerm* t) {
    if (!(0 <= q[0] && q[0] < q[1] && q[1] < q[2] && q[2] < q[3] && q[3] < N)) return false;
    PauliString s = mul(mul(mul(jw_gamma(q[0]), jw_gamma(q[1])), jw_gamma(q[2])), jw_gamma(q[3]));
    t->x = s.x;
    t->z = s.z;
    double s4 = (gamma_norm == SYK_GAMMA_HALF) ? 0.25 : 1.0;   // (1/sqrt 2)^4, exact
    double a = J * s4;
    switch (s.ipow) {
        case 0: t->c = {a, 0.0}; break;
        case 1: t->c = {0.0, a}; break;
        case 2: t->c = {-a, 0.0}; break;
        default: t->c = {0.0, -a}; break;
    }
    for (int k = 0; k < 4; ++k) t->q[k] = q[k];
    t->J = J;
    return true;
}

bool valid_common(int N, int gamma_norm, syk_ham** out) {
    return out && N >= 4 && N <= 66 && (N % 2) == 0 &&   // N = 66: only its parity blocks (32 qubits) can be applied
           (gamma_norm == SYK_GAMMA_PAULI || gamma_norm == SYK_GAMMA_HALF);
}

}  // namespace

extern "C" {

int syk_build_hamiltonian(int N, double p, uint64_t seed, uint32_t realization, int gamma_norm, syk_ham** out) {
    if (!valid_common(N, gamma_norm, out) || !(p > 0.0 && p <= 1.0)) return SYK_EINVAL;
    *out = nullptr;
    const uint64_t key = syk::rng_key(seed, realization, syk::kStreamHamiltonian);
    const uint64_t threshold = (uint64_t)std::floor(p * 9007199254740992.0);   // floor(p 2^53)
    const double sigma = std::sqrt(3.0 / (8.0 * p * (double)N * (double)N * (double)N));
    const double two_pi = 6.283185307179586476925286766559;
    std::vector<RawTerm> raw;
    try {
        uint64_t r = 0;
        for (int i = 0; i < N; ++i)
            for (int j = i + 1; j < N; ++j)
                for (int k = j + 1; k < N; ++k)
                    for (int l = k + 1; l < N; ++l, ++r) {
                        if (syk::rng_draw(key, r, 0) >= threshold) continue;
                        double u1 = (double)(syk::rng_draw(key, r, 1) + 1) * 0x1.0p-53;
                        double u2 = (double)syk::rng_draw(key, r, 2) * 0x1.0p-53;
                        double J = sigma * std::sqrt(-2.0 * std::log(u1)) * std::cos(two_pi * u2);
                        int32_t q[4] = {i, j, k, l};
                        RawTerm t;
                        make_term(N, gamma_norm, q, J, &t);
                        raw.push_back(t);
                    }
    } catch (const std::bad_alloc&) {
        return SYK_ENOMEM;
    }
    return compile(N, gamma_norm, raw, out);
}

int syk_build_from_terms(int N, int64_t n_terms, const int32_t* quartets, const double* J, int gamma_norm,
                         syk_ham** out) {
    if (!valid_common(N, gamma_norm, out) || n_terms < 0 || (n_terms > 0 && (!quartets || !J))) return SYK_EINVAL;
    if (n_terms > 0xFFFFFFF0ll) return SYK_EINVAL;
    *out = nullptr;
    std::vector<RawTerm> raw;
    try {
        raw.resize((size_t)n_terms);
    } catch (const std::bad_alloc&) {
        return SYK_ENOMEM;
    }
    for (int64_t t = 0; t < n_terms; ++t)
        if (!make_term(N, gamma_norm, quartets + 4 * t, J[t], &raw[(size_t)t])) return SYK_EINVAL;
    return compile(N, gamma_norm, raw, out);
}

int syk_build_from_pauli_strings(int L, int64_t n_terms, const uint64_t* x, const uint64_t* z, const double* c_re_im,
                                 syk_ham** out) {
    if (!out || L < 2 || L > 32 || n_terms < 0 || (n_terms > 0 && (!x || !z || !c_re_im))) return SYK_EINVAL;
    if (n_terms > 0xFFFFFFF0ll) return SYK_EINVAL;
    *out = nullptr;
    const uint64_t mask = L == 64 ? ~0ull : ((1ull << L) - 1);
    std::vector<RawTerm> raw;
    try {
        raw.resize((size_t)n_terms);
    } catch (const std::bad_alloc&) {
        return SYK_ENOMEM;
    }
    for (int64_t t = 0; t < n_terms; ++t) {
        if ((x[t] | z[t]) & ~mask) return SYK_EINVAL;
        const double re = c_re_im[2 * t], im = c_re_im[2 * t + 1];
        // Hermitian sum of independent strings: (c Z^z X^x)^+ = conj(c) (-1)^popcount(x & z) Z^z X^x, so c must be
        // real when popcount(x & z) is even and imaginary when it is odd (the Lanczos driver needs H = H^+)
        const bool odd = __builtin_popcountll(x[t] & z[t]) & 1;
        if (!std::isfinite(re) || !std::isfinite(im) || (odd ? re != 0.0 : im != 0.0)) return SYK_EINVAL;
        RawTerm& r = raw[(size_t)t];
        r.x = x[t];
        r.z = z[t];
        r.c = {re, im};
        for (int k = 0; k < 4; ++k) r.q[k] = -1;
        r.J = 0.0;
    }
    int rc = compile(2 * L, SYK_GAMMA_PAULI, raw, out);
    if (rc == SYK_OK) (*out)->generic = true;
    return rc;
}

int syk_build_parity_block(const syk_ham* h, int sector, syk_ham** out) {
    if (!h || !out || (sector != 0 && sector != 1) || h->block_of_N != 0 || h->generic || h->N < 6) return SYK_EINVAL;
    *out = nullptr;
    const int L = h->L;
    const uint64_t low = (1ull << (L - 1)) - 1;
    std::vector<RawTerm> raw;
    try {
        raw.reserve(h->z.size());
        for (size_t g = 0; g < h->x.size(); ++g)
            for (uint32_t t = h->group_off[g]; t < h->group_off[g + 1]; ++t) {
                // c Z^z X^x restricted to the sector (R-BLOCK): the dropped top bit of the output index is
                // parity(b') xor sector, so a Z on it contributes (-1)^sector and complements the low Z-mask
                const bool z_top = (h->z[t] >> (L - 1)) & 1ull;
                RawTerm r;
                r.x = h->x[g] & low;
                r.z = z_top ? (~h->z[t]) & low : h->z[t] & low;
                r.c = (z_top && sector) ? -h->c[t] : h->c[t];
                for (int k = 0; k < 4; ++k) r.q[k] = h->quartet[4 * (size_t)t + k];
                r.J = h->J[t];
                raw.push_back(r);
            }
    } catch (const std::bad_alloc&) {
        return SYK_ENOMEM;
    }
    int rc = compile(h->N - 2, h->gamma_norm, raw, out);
    if (rc == SYK_OK) {
        (*out)->block_of_N = h->N;
        (*out)->sector = sector;
    }
    return rc;
}

void syk_free_hamiltonian(syk_ham* h) {
    if (!h) return;
    syk::free_device_tables(h);
    syk::free_regtile_tables(h);
    syk::free_scatter_tables(h);
    syk::free_dense_tables(h);
    delete h;
}

int syk_ham_info(const syk_ham* h, int* N, int64_t* n_terms, int64_t* n_xmasks, int64_t* dim) {
    if (!h) return SYK_EINVAL;
    if (N) *N = h->N;
    if (n_terms) *n_terms = h->n_terms();
    if (n_xmasks) *n_xmasks = h->n_groups();
    if (dim) *dim = (int64_t)1 << h->L;
    return SYK_OK;
}

int syk_ham_tables(const syk_ham* h, uint64_t* x, uint32_t* group_off, uint64_t* z, double* c_re_im,
                   int32_t* quartet_of_term, double* J_of_term) {
    if (!h) return SYK_EINVAL;
    if (x) std::copy(h->x.begin(), h->x.end(), x);
    if (group_off) std::copy(h->group_off.begin(), h->group_off.end(), group_off);
    if (z) std::copy(h->z.begin(), h->z.end(), z);
    if (c_re_im)
        for (size_t t = 0; t < h->c.size(); ++t) {
            c_re_im[2 * t] = h->c[t].real();
            c_re_im[2 * t + 1] = h->c[t].imag();
        }
    if (quartet_of_term) std::copy(h->quartet.begin(), h->quartet.end(), quartet_of_term);
    if (J_of_term) std::copy(h->J.begin(), h->J.end(), J_of_term);
    return SYK_OK;
}

}  // extern "C"
