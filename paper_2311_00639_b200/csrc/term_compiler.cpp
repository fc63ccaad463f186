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
    h->uid = syk::next_handle_uid();
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
        // the canonical tables are what syk_ham_tables exports; the storage-basis tables start out equal to them
        h->can_x = h->x;
        h->can_group_off = h->group_off;
        h->can_z = h->z;
        h->can_c = h->c;
    } catch (const std::bad_alloc&) {
        delete h;
        return SYK_ENOMEM;
    }
    *out = h;
    return SYK_OK;
}

// Storage-basis tables of a handle for the qubit layout `perm` (qubit q = index bit perm[q]): every canonical string
// c Z^z X^x becomes c Z^{P z} X^{P x}; groups by ascending P x, terms by ascending P z.  Drops all cached kernel tables.
int apply_layout(syk_ham* h, const std::vector<uint8_t>& perm) {
    const int L = h->L;
    auto map = [&](uint64_t m) {
        uint64_t r = 0;
        for (int q = 0; q < L; ++q) r |= ((m >> q) & 1ull) << perm[(size_t)q];
        return r;
    };
    struct T3 { uint64_t x, z; std::complex<double> c; };
    try {
        std::vector<T3> t;
        t.reserve(h->can_z.size());
        for (size_t g = 0; g < h->can_x.size(); ++g)
            for (uint32_t k = h->can_group_off[g]; k < h->can_group_off[g + 1]; ++k)
                t.push_back(T3{map(h->can_x[g]), map(h->can_z[k]), h->can_c[k]});
        std::sort(t.begin(), t.end(), [](const T3& a, const T3& b) { return a.x != b.x ? a.x < b.x : a.z < b.z; });
        std::vector<uint64_t> x, z;
        std::vector<uint32_t> off;
        std::vector<std::complex<double>> c;
        for (const T3& e : t) {
            if (x.empty() || x.back() != e.x) {
                x.push_back(e.x);
                off.push_back((uint32_t)z.size());
            }
            z.push_back(e.z);
            c.push_back(e.c);
        }
        off.push_back((uint32_t)z.size());
        bool identity = true;
        for (int q = 0; q < L; ++q) identity &= perm[(size_t)q] == q;
        syk::invalidate_kernel_tables(h);
        h->x.swap(x);
        h->group_off.swap(off);
        h->z.swap(z);
        h->c.swap(c);
        h->perm = identity ? std::vector<uint8_t>() : perm;
    } catch (const std::bad_alloc&) {
        return SYK_ENOMEM;
    }
    return SYK_OK;
}

// ---- choice of the layout -------------------------------------------------------------------
// The tile kernels move the vector once from L2 into the SMs per distinct value of (x outside the TILE bits) and once
// from DRAM per distinct value of (x outside TILE + WINDOW bits) (apply_h_scatter.cu).  The X-masks of a sparse SYK
// Hamiltonian are random 2- and 4-subsets of the qubits, so WHICH qubits sit on the low index bits decides both counts:
// minimise  loads + 2 passes  over the partition of the qubits into tile / window / rest by deterministic hill climbing
// from a few starting points.
struct DistinctCounter {
    std::vector<uint32_t> key, stamp;
    uint32_t gen = 0, mask = 0;
    explicit DistinctCounter(size_t n) {
        size_t cap = 64;
        while (cap < 4 * n) cap <<= 1;
        key.assign(cap, 0);
        stamp.assign(cap, 0);
        mask = (uint32_t)cap - 1;
    }
    int count(const std::vector<uint32_t>& xs, uint32_t keep) {
        ++gen;
        int n = 0;
        for (uint32_t x : xs) {
            const uint32_t v = x & keep;
            uint32_t slot = (v * 0x9E3779B1u) >> 7 & mask;
            for (;;) {
                if (stamp[slot] != gen) {
                    stamp[slot] = gen;
                    key[slot] = v;
                    ++n;
                    break;
                }
                if (key[slot] == v) break;
                slot = (slot + 1) & mask;
            }
        }
        return n;
    }
};

void choose_permutation(const syk_ham* h, int n_tile, int n_window, std::vector<uint8_t>& perm) {
    const int L = h->L;
    std::vector<uint32_t> xs;
    for (uint64_t x : h->can_x) xs.push_back((uint32_t)x);
    DistinctCounter dc(xs.size());
    const int nt = std::min(n_tile, L), nw = std::min(n_window, L - nt);
    // seq[0..nt) = qubits of the tile, seq[nt..nt+nw) = window qubits, the rest above
    auto cost = [&](const std::vector<int>& seq) {
        uint32_t tile = 0, win = 0;
        for (int i = 0; i < nt; ++i) tile |= 1u << seq[(size_t)i];
        win = tile;
        for (int i = nt; i < nt + nw; ++i) win |= 1u << seq[(size_t)i];
        return dc.count(xs, ~tile) + 2 * dc.count(xs, ~win);
    };
    auto cls = [&](int i) { return i < nt ? 0 : (i < nt + nw ? 1 : 2); };
    std::vector<int> best;
    int best_cost = 0;
    uint64_t rng = 0x243F6A8885A308D3ull;   // fixed: the choice is a deterministic function of the tables
    for (int start = 0; start < 4; ++start) {
        std::vector<int> seq((size_t)L);
        std::iota(seq.begin(), seq.end(), 0);
        if (start > 0)
            for (int i = L - 1; i > 0; --i) {   // Fisher-Yates with a 64-bit LCG
                rng = rng * 6364136223846793005ull + 1442695040888963407ull;
                std::swap(seq[(size_t)i], seq[(size_t)((rng >> 33) % (uint64_t)(i + 1))]);
            }
        int cur = cost(seq);
        for (int sweep = 0; sweep < 32; ++sweep) {
            bool improved = false;
            for (int i = 0; i < nt + nw; ++i)
                for (int j = i + 1; j < L; ++j) {
                    if (cls(i) == cls(j)) continue;
                    std::swap(seq[(size_t)i], seq[(size_t)j]);
                    const int c = cost(seq);
                    if (c < cur) {
                        cur = c;
                        improved = true;
                    } else {
                        std::swap(seq[(size_t)i], seq[(size_t)j]);
                    }
                }
            if (!improved) break;
        }
        if (best.empty() || cur < best_cost) {
            best = seq;
            best_cost = cur;
        }
    }
    // canonical order inside each class (the cost does not depend on it): ascending qubit numbers
    std::sort(best.begin(), best.begin() + nt);
    std::sort(best.begin() + nt, best.begin() + nt + nw);
    std::sort(best.begin() + nt + nw, best.end());
    perm.assign((size_t)L, 0);
    for (int i = 0; i < L; ++i) perm[(size_t)best[(size_t)i]] = (uint8_t)i;
}

bool make_term(int N, int gamma_norm, const int32_t* q, double J, RawTerm* t, double J_im = 0.0) {
    if (!(0 <= q[0] && q[0] < q[1] && q[1] < q[2] && q[2] < q[3] && q[3] < N)) return false;
    PauliString s = mul(mul(mul(jw_gamma(q[0]), jw_gamma(q[1])), jw_gamma(q[2])), jw_gamma(q[3]));
    t->x = s.x;
    t->z = s.z;
    double s4 = (gamma_norm == SYK_GAMMA_HALF) ? 0.25 : 1.0;   // (1/sqrt 2)^4, exact
    double a = J * s4, b = J_im * s4;   // (a + i b) i^ipow, exactly: multiplication by i is a swap and a sign
    switch (s.ipow) {
        case 0: t->c = {a, b}; break;
        case 1: t->c = {-b, a}; break;
        case 2: t->c = {-a, -b}; break;
        default: t->c = {b, -a}; break;
    }
    if (J_im == 0.0) {   // keep exact zeros (not -0.0 + 0.0 artefacts): the tile kernels test c for real / imaginary
        if (s.ipow & 1) t->c = {0.0, t->c.imag()};
        else t->c = {t->c.real(), 0.0};
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

int syk_build_from_terms_complex(int N, int64_t n_terms, const int32_t* quartets, const double* J_re_im, int gamma_norm,
                                 syk_ham** out) {
    if (!valid_common(N, gamma_norm, out) || n_terms < 0 || (n_terms > 0 && (!quartets || !J_re_im))) return SYK_EINVAL;
    if (n_terms > 0xFFFFFFF0ll) return SYK_EINVAL;
    *out = nullptr;
    std::vector<RawTerm> raw;
    try {
        raw.resize((size_t)n_terms);
    } catch (const std::bad_alloc&) {
        return SYK_ENOMEM;
    }
    bool hermitian = true;
    for (int64_t t = 0; t < n_terms; ++t) {
        const double re = J_re_im[2 * t], im = J_re_im[2 * t + 1];
        if (!std::isfinite(re) || !std::isfinite(im)) return SYK_EINVAL;
        if (!make_term(N, gamma_norm, quartets + 4 * t, re, &raw[(size_t)t], im)) return SYK_EINVAL;
        hermitian &= im == 0.0;   // a product of four distinct Majoranas is Hermitian: H = H^+ iff every J is real
    }
    int rc = compile(N, gamma_norm, raw, out);
    if (rc == SYK_OK) (*out)->hermitian = hermitian;
    return rc;
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
    bool hermitian = true;
    for (int64_t t = 0; t < n_terms; ++t) {
        if ((x[t] | z[t]) & ~mask) return SYK_EINVAL;
        const double re = c_re_im[2 * t], im = c_re_im[2 * t + 1];
        // (c Z^z X^x)^+ = conj(c) (-1)^popcount(x & z) Z^z X^x: a string is Hermitian iff c is real when
        // popcount(x & z) is even and imaginary when it is odd.  Any other coefficient makes the sum non-Hermitian
        // (checked string by string): such a handle is evolved by Arnoldi instead of Lanczos.
        const bool odd = __builtin_popcountll(x[t] & z[t]) & 1;
        if (!std::isfinite(re) || !std::isfinite(im)) return SYK_EINVAL;
        hermitian &= odd ? re == 0.0 : im == 0.0;
        RawTerm& r = raw[(size_t)t];
        r.x = x[t];
        r.z = z[t];
        r.c = {re, im};
        for (int k = 0; k < 4; ++k) r.q[k] = -1;
        r.J = 0.0;
    }
    int rc = compile(2 * L, SYK_GAMMA_PAULI, raw, out);
    if (rc == SYK_OK) {
        (*out)->generic = true;
        (*out)->hermitian = hermitian;
    }
    return rc;
}

int syk_build_parity_block(const syk_ham* h, int sector, syk_ham** out) {
    if (!h || !out || (sector != 0 && sector != 1) || h->block_of_N != 0 || h->generic || h->N < 6) return SYK_EINVAL;
    *out = nullptr;
    const int L = h->L;
    const uint64_t low = (1ull << (L - 1)) - 1;
    std::vector<RawTerm> raw;
    try {
        raw.reserve(h->can_z.size());
        for (size_t g = 0; g < h->can_x.size(); ++g)
            for (uint32_t t = h->can_group_off[g]; t < h->can_group_off[g + 1]; ++t) {
                // c Z^z X^x restricted to the sector (R-BLOCK): the dropped top bit of the output index is
                // parity(b') xor sector, so a Z on it contributes (-1)^sector and complements the low Z-mask
                // (canonical tables: a block is cut from the canonical Hamiltonian and starts with the identity layout)
                const bool z_top = (h->can_z[t] >> (L - 1)) & 1ull;
                RawTerm r;
                r.x = h->can_x[g] & low;
                r.z = z_top ? (~h->can_z[t]) & low : h->can_z[t] & low;
                r.c = (z_top && sector) ? -h->can_c[t] : h->can_c[t];
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
        (*out)->hermitian = h->hermitian;
    }
    return rc;
}

void syk_free_hamiltonian(syk_ham* h) {
    if (!h) return;
    syk::invalidate_kernel_tables(h);
    delete h;
}

int syk_ham_set_layout(syk_ham* h, const int32_t* perm) {
    if (!h || h->L > 32) return SYK_EINVAL;
    std::vector<uint8_t> p((size_t)h->L);
    uint64_t seen = 0;
    for (int q = 0; q < h->L; ++q) {
        const int32_t b = perm ? perm[q] : q;
        if (b < 0 || b >= h->L || ((seen >> b) & 1ull)) return SYK_EINVAL;
        seen |= 1ull << b;
        p[(size_t)q] = (uint8_t)b;
    }
    return apply_layout(h, p);
}

int syk_ham_optimize_layout(syk_ham* h, int dtype) {
    if (!h || h->L > 32 || (dtype != SYK_C64 && dtype != SYK_C128)) return SYK_EINVAL;
    // only the tile kernels for sparse H gain (<= 1024 terms); anything else keeps the identity layout
    if (h->n_terms() == 0 || h->n_terms() > syk::kStMaxTerms) return syk_ham_set_layout(h, nullptr);
    std::vector<uint8_t> p;
    try {
        choose_permutation(h, syk::scatter_tile_bits(dtype), syk::scatter_window_bits(), p);
    } catch (const std::bad_alloc&) {
        return SYK_ENOMEM;
    }
    return apply_layout(h, p);
}

int syk_ham_layout(const syk_ham* h, int32_t* perm, int* is_identity) {
    if (!h) return SYK_EINVAL;
    if (perm)
        for (int q = 0; q < h->L; ++q) perm[q] = h->bit_of_qubit(q);
    if (is_identity) *is_identity = h->identity_layout() ? 1 : 0;
    return SYK_OK;
}

int syk_ham_is_hermitian(const syk_ham* h) { return h ? (h->hermitian ? 1 : 0) : SYK_EINVAL; }

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
    if (x) std::copy(h->can_x.begin(), h->can_x.end(), x);
    if (group_off) std::copy(h->can_group_off.begin(), h->can_group_off.end(), group_off);
    if (z) std::copy(h->can_z.begin(), h->can_z.end(), z);
    if (c_re_im)
        for (size_t t = 0; t < h->can_c.size(); ++t) {
            c_re_im[2 * t] = h->can_c[t].real();
            c_re_im[2 * t + 1] = h->can_c[t].imag();
        }
    if (quartet_of_term) std::copy(h->quartet.begin(), h->quartet.end(), quartet_of_term);
    if (J_of_term) std::copy(h->J.begin(), h->J.end(), J_of_term);
    return SYK_OK;
}

}  // extern "C"
