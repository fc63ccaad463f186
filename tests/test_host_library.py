"""Host-side checks of libsyk_b200 that need no GPU: the C ABI surface and the term compiler (a-1).

The integer tables of the library are compared BIT-EXACTLY with the oracle's tables, which are derived from rows
of Kronecker-built term matrices (oracle/hamiltonian.py: derive_tables), never from mask arithmetic.
"""
import ctypes
import math
import os
import re

import numpy as np
import pytest

from oracle import hamiltonian as ohm
from oracle import majorana, rng as orng
from paper_2311_00639_b200 import build as pkg_build
from paper_2311_00639_b200 import inputs

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def B():
    pkg_build.build()
    from paper_2311_00639_b200 import binding
    return binding


def declared_symbols():
    text = open(os.path.join(ROOT, "include", "syk.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(syk_[a-zA-Z0-9_]+)\s*\(", text)))


def assert_coeff_equal(c_lib, c_ref, gamma_norm):
    """Phase class (which of re/im is non-zero, and its sign) exactly; magnitude exactly for s = 1.  For
    s = 1/sqrt(2) the oracle multiplies four Kronecker factors of 0.7071... (s^4 = 0.25 up to 2 ulp) while the
    library uses the exact 0.25, so the magnitude is compared to 4 ulp there."""
    assert np.array_equal(np.sign(c_lib.real), np.sign(c_ref.real))
    assert np.array_equal(np.sign(c_lib.imag), np.sign(c_ref.imag))
    if gamma_norm == majorana.GAMMA_PAULI:
        assert np.array_equal(c_lib, c_ref)
    else:
        assert np.allclose(c_lib, c_ref, rtol=1e-15, atol=0.0)


def test_library_exports_every_declared_symbol(B):
    names = declared_symbols()
    assert len(names) >= 25
    lib = ctypes.CDLL(B.LIB_PATH)
    for n in names:
        assert hasattr(lib, n), f"{n} declared in include/syk.h but not exported"
    # and the binding wraps the same names
    for n in names:
        assert n in B.EXPORTED, f"{n} has no ctypes signature in binding.py"


def test_strerror_and_version(B):
    assert B.syk_version() >= 100
    assert B._lib.syk_strerror(0) == b"ok"
    assert b"invalid" in B._lib.syk_strerror(B.SYK_EINVAL)


@pytest.mark.parametrize("N,k,seed,realization,gn", [
    (8, None, 0, 0, 0), (8, None, 3, 1, 1), (12, 2, 1, 0, 0), (16, None, 0, 0, 0), (16, 4, 7, 5, 1),
    (24, 4, 0, 2, 0), (32, 4, 0, 0, 0), (32, 4, 0, 99, 0),
])
def test_sampler_and_tables_bit_exact(B, N, k, seed, realization, gn):
    """a-1: same quartets kept (integer compare), J to 1 ulp, tables (x, group_off, z, phase class) bit-exact."""
    p = inputs.bernoulli_p(N, k)
    q_ref, J_ref, _ = orng.sample_couplings(N, p, seed, realization)
    h = B.syk_build_hamiltonian(N, p, seed, realization, gn)
    info = h.info()
    tab = h.tables()
    assert info["N"] == N and info["dim"] == 1 << (N // 2)
    assert info["n_terms"] == len(J_ref)
    # library terms are in canonical order; compare as sets keyed by quartet
    lib_q = [tuple(r) for r in tab["quartet_of_term"]]
    assert sorted(lib_q) == sorted(tuple(r) for r in q_ref)
    J_by_q = {tuple(r): j for r, j in zip(q_ref, J_ref)}
    J_lib = tab["J"]
    J_exp = np.array([J_by_q[r] for r in lib_q])
    assert np.allclose(J_lib, J_exp, rtol=4e-16, atol=0.0)
    # tables derived by the oracle from dense rows, using the LIBRARY's J so that c compares exactly
    ref = ohm.derive_tables(N, np.array(lib_q), J_lib, gn, verify_rows=4)
    assert np.array_equal(tab["x"], ref["x"])
    assert np.array_equal(tab["group_off"], ref["group_off"])
    assert np.array_equal(tab["z"], ref["z"])
    assert np.array_equal(tab["quartet_of_term"], ref["quartet_of_term"])
    assert_coeff_equal(tab["c"], ref["c"], gn)
    assert info["n_xmasks"] == len(ref["x"])


def test_build_from_terms_matches_oracle_tables(B):
    N = 20
    q, J = inputs.random_quartets(N, 300, seed=11)
    h = B.syk_build_from_terms(N, q, J, B.SYK_GAMMA_HALF)
    tab = h.tables()
    ref = ohm.derive_tables(N, q, J, majorana.GAMMA_HALF)
    for key in ("x", "group_off", "z", "quartet_of_term"):
        assert np.array_equal(tab[key], ref[key]), key
    assert_coeff_equal(tab["c"], ref["c"], majorana.GAMMA_HALF)


def test_dense_N16_mask_statistics(B):
    """SURVEY 8a-1 / pin P7: dense N=16 has 1820 terms on 99 X-masks (1 + C(8,2) + C(8,4))."""
    h = B.syk_build_hamiltonian(16, 1.0, 0, 0, 0)
    info = h.info()
    assert info["n_terms"] == 1820 and info["n_xmasks"] == 99
    x = h.tables()["x"]
    pc = np.array([bin(int(v)).count("1") for v in x])
    assert sorted(set(pc)) == [0, 2, 4]
    assert (pc == 0).sum() == 1 and (pc == 2).sum() == 28 and (pc == 4).sum() == 70


def test_hand_worked_terms(B):
    """Pin P4 through the library: tests/golden/pauli_products_by_hand.txt."""
    path = os.path.join(ROOT, "tests", "golden", "pauli_products_by_hand.txt")
    rows = [l.split() for l in open(path) if l.strip() and not l.startswith("#")]
    assert rows
    for r in rows:
        N, quartet, x, z = int(r[0]), [int(a) for a in r[1:5]], int(r[5], 2), int(r[6], 2)
        c = complex(float(r[7]), float(r[8]))
        h = B.syk_build_from_terms(N, [quartet], [1.0], B.SYK_GAMMA_PAULI)
        t = h.tables()
        assert int(t["x"][0]) == x and int(t["z"][0]) == z and complex(t["c"][0]) == c, r


def test_large_N_tables_structure(B):
    """N=48 (configs[2] sparsities), N=56, k=4 and N=64, k=2 (bench configs): structure that holds at any size, and EVERY
    term against the oracle's dense-row derivation (integer tables bit-exact)."""
    for N, k in ((48, 1), (48, 8), (56, 4), (64, 2)):
        p = inputs.bernoulli_p(N, k)
        h = B.syk_build_hamiltonian(N, p, 0, 0, 0)
        info, t = h.info(), h.tables()
        T = info["n_terms"]
        assert abs(T - k * N) < 6 * math.sqrt(k * N)
        assert np.all(np.diff(t["x"].astype(np.int64)) > 0)
        assert t["group_off"][0] == 0 and t["group_off"][-1] == T
        pc = np.array([bin(int(v)).count("1") for v in t["x"]])
        assert set(pc) <= {0, 2, 4}
        # c is real iff popcount(x & z) is even
        xs = np.repeat(t["x"], np.diff(t["group_off"]).astype(np.int64))
        par = np.array([bin(int(a & b)).count("1") & 1 for a, b in zip(xs, t["z"])])
        assert np.all((t["c"].imag == 0) == (par == 0))
        assert np.all((t["c"].real == 0) == (par == 1))
        assert np.all(t["x"] < (1 << (N // 2))) and np.all(t["z"] < (1 << (N // 2)))
        # all terms against the oracle's dense-row derivation: whole tables, canonical order included
        ref = ohm.derive_tables(N, t["quartet_of_term"], t["J"], 0)
        for key in ("x", "group_off", "z"):
            assert np.array_equal(t[key], ref[key]), (N, k, key)
        assert_coeff_equal(t["c"], ref["c"], 0)


def test_argument_errors(B):
    out = ctypes.c_void_p()
    f = B._lib.syk_build_hamiltonian
    assert f(7, 0.5, 0, 0, 0, ctypes.byref(out)) == B.SYK_EINVAL       # odd N
    assert f(2, 0.5, 0, 0, 0, ctypes.byref(out)) == B.SYK_EINVAL       # N < 4
    assert f(68, 0.5, 0, 0, 0, ctypes.byref(out)) == B.SYK_EINVAL      # N > 66 (66 only for parity blocks)
    assert f(8, 0.0, 0, 0, 0, ctypes.byref(out)) == B.SYK_EINVAL       # p = 0
    assert f(8, 1.5, 0, 0, 0, ctypes.byref(out)) == B.SYK_EINVAL       # p > 1
    assert f(8, 0.5, 0, 0, 2, ctypes.byref(out)) == B.SYK_EINVAL       # gamma_norm
    with pytest.raises(B.SykError):
        B.syk_build_from_terms(8, [[0, 0, 1, 2]], [1.0])                # not strictly increasing
    with pytest.raises(B.SykError):
        B.syk_build_from_terms(8, [[0, 1, 2, 8]], [1.0])                # index >= N
    h = B.syk_build_from_terms(8, np.zeros((0, 4), dtype=np.int32), np.zeros(0))   # empty H is valid
    assert h.info()["n_terms"] == 0 and h.info()["n_xmasks"] == 0
    assert list(h.tables()["group_off"]) == [0]


def test_duplicate_quartets_are_merged(B):
    """Operator sum: equal strings are combined."""
    h = B.syk_build_from_terms(8, [[0, 1, 2, 3], [0, 1, 2, 3]], [0.25, 0.5])
    t = h.tables()
    assert h.info()["n_terms"] == 1 and abs(t["c"][0]) == 0.75


def test_workspace_queries_without_gpu(B):
    h = B.syk_build_hamiltonian(16, 1.0, 0, 0, 0)
    V = 256 * 16
    hdr = B.syk_krylov_workspace_bytes(h, B.SYK_C128, {"krylov_dim": 20}) - 20 * V
    assert hdr > 0 and hdr % 4096 == 0
    assert B.syk_krylov_workspace_bytes(h, B.SYK_C128, {"krylov_dim": 20, "two_pass": 1}) == hdr + 2 * V
    assert B.syk_otoc_workspace_bytes(h, B.SYK_C64, {"krylov_dim": 20, "two_pass": 1}) == hdr + 4 * 256 * 8
    assert B.syk_reduce_scratch_bytes() == hdr


def test_no_cpu_fallback_without_device(B):
    """On a machine without a CUDA device every compute entry point must fail loudly (SYK_ECUDA)."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    h = B.syk_build_hamiltonian(8, 1.0, 0, 0, 0)
    buf = (ctypes.c_double * 64)()
    a = ctypes.addressof(buf)
    a = (a + 15) & ~15
    rc = B._lib.syk_apply_H(h.handle, B.SYK_C128, a, a + 256, None)
    assert rc == B.SYK_ECUDA
    assert B._lib.syk_last_cuda_error() != b""


# ------------------------------------------------------------------------------------------------------------
# NEXT-1 parity blocks (DESIGN.md R-BLOCK)
# ------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("gamma_norm", [0, 1])
def test_parity_block_tables_bit_exact(B, gamma_norm):
    """Tables of syk_build_parity_block against tables DERIVED from the dense block of every term matrix (the O4
    recipe on the reduced basis: x' = column of the non-zero of row 0, c = that entry, bit q of z = 1 iff the
    entry of row 2^q has the opposite sign), for both sectors."""
    from oracle import parity as opar
    N, L = 10, 5
    q, J, _ = orng.sample_couplings(N, 0.5, seed=3, realization=1)
    h = B.syk_build_from_terms(N, q, J, gamma_norm)
    g = majorana.jw_gammas(N, gamma_norm)
    for sector in (0, 1):
        hb = B.syk_build_parity_block(h, sector)
        info = hb.info()
        assert info["N"] == N - 2 and info["dim"] == 1 << (L - 1) and info["n_terms"] == len(J)
        tab = hb.tables()
        idx = opar.sector_indices(L, sector).astype(np.int64)
        ref = []
        for (i, j, k, l), Jt in zip(q, J):
            M = (Jt * (g[i] @ g[j] @ g[k] @ g[l]))[np.ix_(idx, idx)]
            x = int(np.nonzero(M[0])[0][0])
            c = M[0, x]
            z = 0
            for bit in range(L - 1):
                e = M[1 << bit, (1 << bit) ^ x]
                assert abs(abs(e) - abs(c)) <= 1e-15
                if abs(e + c) <= 1e-15:
                    z |= 1 << bit
            ref.append((x, z, c, (int(i), int(j), int(k), int(l))))
        ref.sort(key=lambda r: (r[0], r[1]))
        xs = np.repeat(tab["x"], np.diff(tab["group_off"].astype(np.int64)))
        assert [int(v) for v in xs] == [r[0] for r in ref]
        assert [int(v) for v in tab["z"]] == [r[1] for r in ref]
        assert [tuple(int(a) for a in row) for row in tab["quartet_of_term"]] == [r[3] for r in ref]
        assert_coeff_equal(tab["c"], np.array([r[2] for r in ref]), gamma_norm)
        # and the table form reproduces the block matrix on a vector
        v = np.random.default_rng(5).normal(size=1 << (L - 1)) + 0j
        Hs = opar.block_hamiltonian(N, q, J, sector, gamma_norm)
        assert np.allclose(ohm.matvec_from_tables(tab, v), Hs @ v, atol=1e-13)
        # a block of a block, bad sector, too small N
        for bad in (lambda: B.syk_build_parity_block(hb, 0), lambda: B.syk_build_parity_block(h, 2)):
            with pytest.raises(B.SykError):
                bad()
    h4 = B.syk_build_from_terms(4, np.array([[0, 1, 2, 3]], dtype=np.int32), np.array([1.0]))
    with pytest.raises(B.SykError):
        B.syk_build_parity_block(h4, 0)


def test_pauli_string_builder(B):
    """syk_build_from_pauli_strings: canonical tables, duplicates combined, Hermiticity rule, range checks; the
    table form applied on the host reproduces the oracle's Kronecker-product matrix."""
    from oracle import pauli as opauli
    L = 6
    terms = opauli.heisenberg_terms(L, 0.7, -0.4, 1.1, periodic=True) + opauli.transverse_ising_terms(L, 0.3, 0.9)
    h = B.syk_build_from_pauli_strings(L, terms)
    info = h.info()
    assert info["N"] == 2 * L and info["dim"] == 1 << L
    tab = h.tables()
    assert info["n_terms"] == len(terms) - L            # the ZZ bonds occur twice and are combined
    xs = np.repeat(tab["x"], np.diff(tab["group_off"].astype(np.int64)))
    assert np.all(np.diff(xs.astype(np.int64)) >= 0)
    H = opauli.sum_matrix(L, terms)
    v = np.random.default_rng(1).normal(size=1 << L) + 1j * np.random.default_rng(2).normal(size=1 << L)
    assert np.allclose(ohm.matvec_from_tables(tab, v), H @ v, atol=1e-13)
    assert B.syk_ham_is_hermitian(h)
    # the Hermiticity rule, string by string: such sums are accepted and flagged non-Hermitian (Arnoldi, NEXT-4)
    for nonherm in ([(1, 1, 1.0)],            # a Y-like string is Hermitian only with an imaginary coefficient
                    [(1, 0, 1j)],             # X only with a real one
                    [(1, 0, 0.3 - 0.2j), (0, 3, 1.0)]):
        hn = B.syk_build_from_pauli_strings(L, nonherm)
        assert not B.syk_ham_is_hermitian(hn)
        tn = hn.tables()
        Hn = opauli.sum_matrix(L, nonherm)
        assert not np.allclose(Hn, Hn.conj().T)
        assert np.allclose(ohm.matvec_from_tables(tn, v), Hn @ v, atol=1e-13)
    for bad in ([(1 << L, 0, 1.0)],           # bit outside the chain
                [(0, 1 << L, 1.0)],
                [(1, 0, float("nan"))]):
        with pytest.raises(B.SykError):
            B.syk_build_from_pauli_strings(L, bad)
    with pytest.raises(B.SykError):
        B.syk_build_from_pauli_strings(1, [(1, 0, 1.0)])
    with pytest.raises(B.SykError):
        B.syk_build_parity_block(h, 0)


def test_N66_only_through_parity_blocks(B):
    """N = 66 (33 qubits) can be built and cut into parity blocks of 32 qubits; the block tables obey the same structure
    rules as any table (sorted, even-popcount X-masks inside 32 bits, coefficient real iff popcount(x & z) even)."""
    N = 66
    h = B.syk_build_hamiltonian(N, inputs.bernoulli_p(N, 2), 0, 0)
    info = h.info()
    assert info["N"] == 66 and info["dim"] == 1 << 33 and info["n_terms"] > 60
    for sector in (0, 1):
        hb = B.syk_build_parity_block(h, sector)
        ib = hb.info()
        assert ib["N"] == 64 and ib["dim"] == 1 << 32 and ib["n_terms"] == info["n_terms"]
        tab = hb.tables()
        assert np.all(tab["x"] < (1 << 32)) and np.all(tab["z"] < (1 << 32))
        assert np.all(np.diff(tab["x"].astype(np.int64)) > 0)
        xs = np.repeat(tab["x"], np.diff(tab["group_off"].astype(np.int64)))
        par = np.array([bin(int(a) & int(b)).count("1") & 1 for a, b in zip(xs, tab["z"])])
        assert np.all((tab["c"].imag != 0) == (par == 1)) and np.all((tab["c"].real != 0) == (par == 0))
    with pytest.raises(B.SykError):
        B.syk_krylov_workspace_bytes(h, B.SYK_C64, {"krylov_dim": 4})
    with pytest.raises(B.SykError):
        B.syk_build_hamiltonian(68, 1e-4, 0, 0)


def test_scatter_layout_choice_on_host(B):
    """The per-Hamiltonian tile layout of the scatter-tile kernel (host-side hill climbing): deterministic, never worse
    than the identity layout (tile = low bits), consistent with a direct count from the X-masks, and it does reduce
    loads and passes for the two headline Hamiltonians."""
    for N, k, code, tb in ((56, 4, B.SYK_C128, 8), (64, 2, B.SYK_C64, 9), (48, 4, B.SYK_C128, 8)):
        p = inputs.bernoulli_p(N, k)
        h = B.syk_build_hamiltonian(N, p, 0, 0)
        lay = B.syk_apply_H_layout(h, code)
        lay2 = B.syk_apply_H_layout(B.syk_build_hamiltonian(N, p, 0, 0), code)
        assert lay == lay2
        x = [int(v) for v in h.tables()["x"]]
        tile, win = lay["tile_mask"], lay["window_mask"]
        assert bin(tile).count("1") == tb + 5 and tile & ((1 << (tb + 3)) - 1) == (1 << (tb + 3)) - 1
        assert win & tile == tile and bin(win).count("1") == min(tb + 5 + 7, N // 2)
        assert lay["n_loads"] == len({v & ~tile for v in x})
        assert lay["n_passes"] == len({v & ~win for v in x})
        ident_tile = (1 << (tb + 5)) - 1
        ident_win = (1 << min(tb + 12, N // 2)) - 1
        assert lay["n_loads"] + 2 * lay["n_passes"] <= len({v & ~ident_tile for v in x}) + 2 * len({v & ~ident_win for v in x})
        if N >= 56:
            assert lay["n_loads"] < len({v & ~ident_tile for v in x}) and lay["n_passes"] < len({v & ~ident_win for v in x})


def _permute_mask(m, perm):
    return sum(((int(m) >> q) & 1) << int(perm[q]) for q in range(len(perm)))


def test_qubit_layout_api_on_host(B):
    """NEXT-3: the exported qubit relabelling.  syk_ham_optimize_layout returns a permutation, is
    deterministic, never changes the canonical tables, and cuts the loads / passes of the tile kernel below what the
    canonical layout (with the kernel's own choice of 2 free tile bits) reaches; the counts the library reports equal a
    direct count from the permuted X-masks; set_layout validates its argument and NULL restores the identity."""
    for N, k, code in ((56, 4, B.SYK_C128), (64, 2, B.SYK_C64)):
        L = N // 2
        p = inputs.bernoulli_p(N, k)
        h = B.syk_build_hamiltonian(N, p, 0, 0)
        t0 = h.tables()
        lay0 = B.syk_apply_H_layout(h, code)
        assert B.syk_ham_layout(h)["identity"] and list(B.syk_ham_layout(h)["perm"]) == list(range(L))
        res = B.syk_ham_optimize_layout(h, code)
        perm = res["perm"]
        assert sorted(perm) == list(range(L)) and not res["identity"]
        h2 = B.syk_build_hamiltonian(N, p, 0, 0)
        assert list(B.syk_ham_optimize_layout(h2, code)["perm"]) == list(perm)          # deterministic
        t1 = h.tables()
        for key in ("x", "group_off", "z", "c", "quartet_of_term", "J"):
            assert np.array_equal(t0[key], t1[key]), key                                 # canonical tables untouched
        lay1 = B.syk_apply_H_layout(h, code)
        xs = [_permute_mask(v, perm) for v in t0["x"]]
        assert lay1["n_loads"] == len({v & ~lay1["tile_mask"] for v in xs})
        assert lay1["n_passes"] == len({v & ~lay1["window_mask"] for v in xs})
        assert lay1["n_loads"] < lay0["n_loads"] and lay1["n_passes"] <= lay0["n_passes"], (lay0, lay1)
        assert lay1["n_loads"] <= 0.93 * lay0["n_loads"]                                 # N=56: 137 -> ~124, N=64: 100 -> ~92
        # explicit layouts
        B.syk_ham_set_layout(h, None)
        assert B.syk_ham_layout(h)["identity"] and B.syk_apply_H_layout(h, code) == lay0
        rev = list(range(L - 1, -1, -1))
        B.syk_ham_set_layout(h, rev)
        assert list(B.syk_ham_layout(h)["perm"]) == rev
        for bad in ([0] * L, list(range(1, L + 1)), list(range(L - 1))):
            with pytest.raises(B.SykError):
                B.syk_ham_set_layout(h, bad)
    # dense Hamiltonians (more than 1024 terms) keep the identity
    hd = B.syk_build_hamiltonian(24, 1.0, 0, 0)
    assert B.syk_ham_optimize_layout(hd, B.SYK_C128)["identity"]


def test_complex_coupling_builder(B):
    """syk_build_from_terms_complex (non-Hermitian SYK): the tables are those of the real-coupling builder
    with every coefficient multiplied by its complex J (Eq. 1 is linear in J); real J gives the identical Hermitian handle."""
    N = 16
    q, J, _ = orng.sample_couplings(N, inputs.bernoulli_p(N, 4), 5, 0)
    Jc = J * np.exp(1j * np.linspace(0.1, 2.9, len(J)))
    hc = B.syk_build_from_terms_complex(N, q, Jc)
    h1 = B.syk_build_from_terms(N, q, np.ones(len(J)))
    assert not B.syk_ham_is_hermitian(hc) and B.syk_ham_is_hermitian(h1)
    tc, t1 = hc.tables(), h1.tables()
    for key in ("x", "group_off", "z", "quartet_of_term"):
        assert np.array_equal(tc[key], t1[key]), key
    order = {tuple(qq): k for k, qq in enumerate(np.asarray(q).reshape(-1, 4).tolist())}
    Jsorted = np.array([Jc[order[tuple(qq)]] for qq in tc["quartet_of_term"].tolist()])
    assert np.allclose(tc["c"], t1["c"] * Jsorted, rtol=1e-15, atol=0)
    hr = B.syk_build_from_terms_complex(N, q, J.astype(np.complex128))
    h0 = B.syk_build_from_terms(N, q, J)
    assert B.syk_ham_is_hermitian(hr)
    assert all(np.array_equal(hr.tables()[k], h0.tables()[k]) for k in ("x", "z", "c", "group_off"))
