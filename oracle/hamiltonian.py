"""Oracle O3-O5: the sparse SYK Hamiltonian of Eq. (1), dense and row-by-row.

Test infrastructure only (see oracle/__init__.py).

    H = sum_{i<j<k<l kept} J_ijkl gamma_i gamma_j gamma_k gamma_l

Three routes to the same operator, none of which multiplies bit-mask "Pauli strings":

* `dense_hamiltonian`  : dense matrix products of the Kronecker-built gammas (O3; N <= ~16).
* `gamma_row`          : each Jordan-Wigner gamma_n is a monomial matrix (one non-zero per row); its
                         row b is read off the Kronecker product entry by entry.  Chaining four rows gives
                         row b of a term (`term_row`), summing terms gives rows of H (`hamiltonian_rows`),
                         applying one gamma at a time gives H.v at any N that fits in RAM
                         (`matvec_sequential`, O5).
* `derive_tables`      : the integer tables the CUDA library exports (X-mask, Z-mask, coefficient),
                         *derived from rows of the term matrix* (O4), for the bit-exact comparison.

Conventions: DESIGN.md R-JW, R-Y, R-ENDIAN, R-SIGN (operator c Z^z X^x acts as
(O v)[b] = c (-1)^popcount(b & z) v[b xor x]: the sign is read at the OUTPUT index b).
"""
import numpy as np

from . import majorana


# ------------------------------------------------------------------------------------------------
# O3: dense
# ------------------------------------------------------------------------------------------------
def dense_hamiltonian(N, quartets, J, gamma_norm=majorana.GAMMA_PAULI):
    """Eq. (1) by dense matrix products.  quartets: (T,4) ints with i<j<k<l; J: (T,) floats."""
    g = majorana.jw_gammas(N, gamma_norm)
    D = 1 << (N // 2)
    H = np.zeros((D, D), dtype=np.complex128)
    for (i, j, k, l), Jt in zip(np.asarray(quartets).reshape(-1, 4), np.asarray(J, dtype=np.float64)):
        H += Jt * (g[i] @ g[j] @ g[k] @ g[l])
    return H


# ------------------------------------------------------------------------------------------------
# monomial rows of a single Jordan-Wigner gamma
# ------------------------------------------------------------------------------------------------
def _popcount_parity(a):
    """Parity (0/1) of the number of set bits of each uint64 in a."""
    a = np.asarray(a, dtype=np.uint64).copy()
    for sh in (32, 16, 8, 4, 2, 1):
        a ^= a >> np.uint64(sh)
    return (a & np.uint64(1)).astype(np.int64)


def gamma_row(n, b, gamma_norm=majorana.GAMMA_PAULI):
    """Row(s) b of the Jordan-Wigner gamma_n: returns (col, val) with gamma_n[b, col] = val the only
    non-zero of that row.  Entry of a Kronecker product = product of the factors' entries:
    Z on qubits j<q gives (-1)^{b_j}; X_q (n even) gives 1 at column b with bit q flipped;
    Y_q (n odd) gives Y[b_q, 1-b_q] = -i if b_q = 0, +i if b_q = 1 (textbook Y, R-Y)."""
    b = np.asarray(b, dtype=np.uint64)
    q = n // 2
    s = majorana.gamma_scale(gamma_norm)
    col = b ^ np.uint64(1 << q)
    below = b & np.uint64((1 << q) - 1)
    val = (1.0 - 2.0 * _popcount_parity(below)).astype(np.complex128) * s
    if n % 2 == 1:
        bq = ((b >> np.uint64(q)) & np.uint64(1)).astype(np.int64)
        val = val * np.where(bq == 0, -1j, 1j)
    return col, val


def term_row(quartet, b, gamma_norm=majorana.GAMMA_PAULI):
    """Row(s) b of gamma_i gamma_j gamma_k gamma_l: (col, val).  Row b of a product A.B of monomial
    matrices is A[b,c] times row c of B, so the chain runs left to right."""
    col = np.asarray(b, dtype=np.uint64)
    val = np.ones(col.shape, dtype=np.complex128)
    for n in quartet:
        col, a = gamma_row(int(n), col, gamma_norm)
        val = val * a
    return col, val


def hamiltonian_rows(N, quartets, J, b, gamma_norm=majorana.GAMMA_PAULI):
    """Rows b of H as (cols[T, len(b)], vals[T, len(b)]); H[b, cols[t,.]] += vals[t,.] (pin P13 uses it)."""
    b = np.asarray(b, dtype=np.uint64)
    quartets = np.asarray(quartets).reshape(-1, 4)
    cols = np.empty((len(quartets),) + b.shape, dtype=np.uint64)
    vals = np.empty((len(quartets),) + b.shape, dtype=np.complex128)
    for t, (q, Jt) in enumerate(zip(quartets, np.asarray(J, dtype=np.float64))):
        c, v = term_row(q, b, gamma_norm)
        cols[t], vals[t] = c, Jt * v
    return cols, vals


# ------------------------------------------------------------------------------------------------
# O5: H.v applying one gamma at a time
# ------------------------------------------------------------------------------------------------
def apply_gamma(N, n, v, gamma_norm=majorana.GAMMA_PAULI):
    """gamma_n v for a state v of dimension 2^(N/2): (gamma v)[b] = val(b) v[col(b)]."""
    v = np.asarray(v)
    D = 1 << (N // 2)
    assert v.shape == (D,)
    col, val = gamma_row(n, np.arange(D, dtype=np.uint64), gamma_norm)
    return val * v[col.astype(np.int64)]


def matvec_sequential(N, quartets, J, v, gamma_norm=majorana.GAMMA_PAULI):
    """H v = sum_t J_t gamma_i (gamma_j (gamma_k (gamma_l v)))  -- never forms a product string."""
    v = np.asarray(v, dtype=np.complex128)
    out = np.zeros_like(v)
    for (i, j, k, l), Jt in zip(np.asarray(quartets).reshape(-1, 4), np.asarray(J, dtype=np.float64)):
        w = apply_gamma(N, int(l), v, gamma_norm)
        w = apply_gamma(N, int(k), w, gamma_norm)
        w = apply_gamma(N, int(j), w, gamma_norm)
        w = apply_gamma(N, int(i), w, gamma_norm)
        out += Jt * w
    return out


def sparse_hamiltonian(N, quartets, J, gamma_norm=majorana.GAMMA_PAULI):
    """H as a scipy CSR matrix assembled from monomial rows (N <= ~28)."""
    import scipy.sparse as sp
    D = 1 << (N // 2)
    rows = np.arange(D, dtype=np.uint64)
    H = sp.csr_matrix((D, D), dtype=np.complex128)
    for q, Jt in zip(np.asarray(quartets).reshape(-1, 4), np.asarray(J, dtype=np.float64)):
        col, val = term_row(q, rows, gamma_norm)
        H = H + sp.csr_matrix((Jt * val, (rows.astype(np.int64), col.astype(np.int64))), shape=(D, D))
    return H


# ------------------------------------------------------------------------------------------------
# O4: integer tables derived from the term matrix
# ------------------------------------------------------------------------------------------------
def derive_tables(N, quartets, J, gamma_norm=majorana.GAMMA_PAULI, verify_rows=0, rng=None):
    """Tables (x, group_off, z, c, quartet_of_term) in the canonical order: groups by ascending x,
    terms inside a group by ascending z.

    For each term M = gamma_i gamma_j gamma_k gamma_l (a monomial matrix):
        x = column of the non-zero in row 0;  c0 = M[0, x];
        bit q of z = 1  iff  M[2^q, 2^q xor x] = -c0         (it must be +c0 or -c0);
        c = J * c0.
    `verify_rows` > 0 additionally checks M[b, b xor x] = c0 (-1)^popcount(b & z) on that many random rows.
    """
    L = N // 2
    quartets = np.asarray(quartets, dtype=np.int64).reshape(-1, 4)
    J = np.asarray(J, dtype=np.float64)
    T = len(quartets)
    xs = np.zeros(T, dtype=np.uint64)
    zs = np.zeros(T, dtype=np.uint64)
    cs = np.zeros(T, dtype=np.complex128)
    unit_rows = np.array([0] + [1 << q for q in range(L)], dtype=np.uint64)
    for t in range(T):
        col, val = term_row(quartets[t], unit_rows, gamma_norm)
        x = int(col[0])
        c0 = complex(val[0])
        z = 0
        for q in range(L):
            assert int(col[1 + q]) == (1 << q) ^ x, "term is not a permutation by XOR"
            if val[1 + q] == -c0:
                z |= 1 << q
            else:
                assert val[1 + q] == c0, "term is not a signed permutation"
        if verify_rows:
            D = 1 << L
            r = rng if rng is not None else np.random.default_rng(12345 + t)
            b = r.integers(0, D, size=verify_rows, dtype=np.uint64)
            cb, vb = term_row(quartets[t], b, gamma_norm)
            assert np.array_equal(cb, b ^ np.uint64(x))
            assert np.array_equal(vb, c0 * (1.0 - 2.0 * _popcount_parity(b & np.uint64(z))))
        xs[t], zs[t], cs[t] = x, z, J[t] * c0
    order = np.lexsort((zs, xs))                      # primary key x, secondary z
    xs, zs, cs, quartets = xs[order], zs[order], cs[order], quartets[order]
    ux, first = np.unique(xs, return_index=True)
    group_off = np.concatenate([first, [T]]).astype(np.uint32)
    return {"x": ux.astype(np.uint64), "group_off": group_off, "z": zs, "c": cs,
            "quartet_of_term": quartets.astype(np.int32)}


def matvec_from_tables(tables, v):
    """(H v)[b] = sum_g v[b xor x_g] sum_{t in g} c_t (-1)^popcount(b & z_t)   (SURVEY 8a-2 form).
    Only used to pin `derive_tables` against the dense product; not a reference for the GPU tables."""
    v = np.asarray(v, dtype=np.complex128)
    D = len(v)
    b = np.arange(D, dtype=np.uint64)
    out = np.zeros_like(v)
    x, off, z, c = tables["x"], tables["group_off"], tables["z"], tables["c"]
    for g in range(len(x)):
        coef = np.zeros(D, dtype=np.complex128)
        for t in range(int(off[g]), int(off[g + 1])):
            coef += c[t] * (1.0 - 2.0 * _popcount_parity(b & z[t]))
        out += coef * v[(b ^ x[g]).astype(np.int64)]
    return out
