"""Pins of the CPU oracle against what the paper and the mathematics fix (no GPU, no CUDA library).

Pin numbering follows SURVEY.md 8(c) / DESIGN.md "Oracle pins".  Every test here must fail for a
plausible mistake in oracle/ (dropped term, wrong sign or index, transposed operand).
"""
import itertools
import math
import os

import numpy as np
import pytest

from oracle import alg1, evolve, green, hamiltonian, majorana, otoc, parity, pauli, rng

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def _random_state(D, seed):
    r = np.random.default_rng(seed)
    v = r.normal(size=D) + 1j * r.normal(size=D)
    return v / np.linalg.norm(v)


def _all_quartets(N):
    return np.array(list(itertools.combinations(range(N), 4)), dtype=np.int32)


# ---------------------------------------------------------------- RNG (O1)
def test_mixer_is_splitmix64():
    # absorb(0,0) = fmix(GOLD) is the first output of SplitMix64 seeded with 0; the second is fmix(2*GOLD).
    # Published test vector of that generator (Steele, Lea, Flood 2014; used to seed xoshiro).
    assert rng.absorb(0, 0) == 0xE220A8397B1DCDAF
    assert rng.fmix((2 * rng.GOLD) & rng.MASK64) == 0x6E789E6AA1B965F4


def test_vector_draw_equals_scalar_draw():
    key = rng.make_key(7, 3, rng.STREAM_STATE)
    idx = np.array([0, 1, 2, 12345, 2 ** 32 - 1, 2 ** 40 + 17], dtype=np.uint64)
    for d in (0, 1, 2):
        assert [int(a) for a in rng.draw_np(key, idx, d)] == [rng.draw(key, int(i), d) for i in idx]


def test_sparsity_definition():
    # k = (p/N) C(N,4)  =>  <#terms> = p C(N,4) = k N
    for N, k in ((32, 4), (56, 4), (64, 2)):
        p = rng.sparsity_p(N, k)
        assert math.isclose(p * math.comb(N, 4) / N, k, rel_tol=1e-15)


def test_dense_keeps_all_and_variance():
    N = 24
    q, J, ranks = rng.sample_couplings(N, 1.0, seed=0, realization=0)
    assert len(J) == math.comb(N, 4) and np.array_equal(ranks, np.arange(len(J)))
    assert np.array_equal(q, _all_quartets(N))                      # lexicographic order
    var = 3.0 / (8.0 * 1.0 * N ** 3)
    assert abs(J.mean()) < 4 * math.sqrt(var / len(J))
    assert abs(J.var() / var - 1.0) < 0.03                          # 10626 draws: sigma(var)/var ~ 1.4 %


def test_sparse_statistics():
    N, k = 32, 4
    p = rng.sparsity_p(N, k)
    counts, allJ = [], []
    for r in range(40):
        q, J, ranks = rng.sample_couplings(N, p, seed=1, realization=r)
        assert np.all(q[:, 0] < q[:, 1]) and np.all(q[:, 1] < q[:, 2]) and np.all(q[:, 2] < q[:, 3])
        assert np.all(np.diff(ranks) > 0)
        counts.append(len(J))
        allJ.append(J)
    allJ = np.concatenate(allJ)
    assert abs(np.mean(counts) - k * N) < 4 * math.sqrt(k * N / 40)          # Binomial, mean kN
    var = 3.0 / (8.0 * p * N ** 3)
    assert abs(allJ.var() / var - 1.0) < 0.08                                # ~5000 draws
    kurt = np.mean(allJ ** 4) / allJ.var() ** 2
    assert abs(kurt - 3.0) < 0.35                                            # Gaussian


def test_random_state_is_normalised_gaussian():
    psi = rng.random_state(24, seed=0, realization=5)
    assert psi.shape == (4096,) and math.isclose(np.vdot(psi, psi).real, 1.0, rel_tol=1e-14)
    x = np.concatenate([psi.real, psi.imag]) * math.sqrt(2 * 4096)
    assert abs(x.mean()) < 0.05 and abs(x.var() - 1) < 0.06 and abs(np.mean(x ** 4) / x.var() ** 2 - 3) < 0.25
    assert not np.allclose(psi, rng.random_state(24, seed=0, realization=6))


# ---------------------------------------------------------------- P1 Clifford algebra
@pytest.mark.parametrize("N", [4, 6, 8, 10])
@pytest.mark.parametrize("gamma_norm", [majorana.GAMMA_PAULI, majorana.GAMMA_HALF])
def test_P1_clifford(N, gamma_norm):
    g = majorana.jw_gammas(N, gamma_norm)
    s2 = majorana.gamma_scale(gamma_norm) ** 2
    eye = np.eye(1 << (N // 2))
    for m in range(N):
        assert np.allclose(g[m], g[m].conj().T)
        for n in range(N):
            anti = g[m] @ g[n] + g[n] @ g[m]
            assert np.allclose(anti, (2 * s2 if m == n else 0) * eye, atol=1e-15)   # PAPER.md:30 / 178


def test_P1_gamma_row_matches_kron():
    N = 8
    D = 16
    for gamma_norm in (0, 1):
        g = majorana.jw_gammas(N, gamma_norm)
        for n in range(N):
            col, val = hamiltonian.gamma_row(n, np.arange(D, dtype=np.uint64), gamma_norm)
            M = np.zeros((D, D), dtype=complex)
            M[np.arange(D), col.astype(int)] = val
            assert np.array_equal(M, g[n])


# ---------------------------------------------------------------- P2 Hermiticity, trace, parity
@pytest.mark.parametrize("N", [8, 12])
def test_P2_hermitian_traceless_parity(N):
    q, J, _ = rng.sample_couplings(N, 0.5, seed=3, realization=0)
    H = hamiltonian.dense_hamiltonian(N, q, J)
    D = 1 << (N // 2)
    assert np.allclose(H, H.conj().T, atol=1e-15)
    assert abs(np.trace(H)) < 1e-13
    par = np.diag(1.0 - 2.0 * hamiltonian._popcount_parity(np.arange(D, dtype=np.uint64)))
    assert np.allclose(H @ par, par @ H, atol=1e-15)


# ---------------------------------------------------------------- P3 second moment
@pytest.mark.parametrize("gamma_norm", [0, 1])
def test_P3_second_moment(gamma_norm):
    N = 12
    q, J, _ = rng.sample_couplings(N, 1.0, seed=0, realization=1)
    H = hamiltonian.dense_hamiltonian(N, q, J, gamma_norm)
    s8 = majorana.gamma_scale(gamma_norm) ** 8
    assert math.isclose(np.trace(H @ H).real / 64, s8 * np.sum(J ** 2), rel_tol=1e-12)


# ---------------------------------------------------------------- P4 hand-worked products
def _golden_products():
    rows = []
    with open(os.path.join(GOLDEN, "pauli_products_by_hand.txt")) as f:
        for line in f:
            if line.startswith("#") or not line.strip():
                continue
            t = line.split()
            rows.append((int(t[0]), tuple(int(a) for a in t[1:5]), int(t[5], 2), int(t[6], 2),
                         complex(float(t[7]), float(t[8]))))
    return rows


@pytest.mark.parametrize("N,quartet,x,z,c", _golden_products())
def test_P4_hand_worked_products(N, quartet, x, z, c):
    Jt = 0.75
    tab = hamiltonian.derive_tables(N, [quartet], [Jt], verify_rows=8)
    assert int(tab["x"][0]) == x and int(tab["z"][0]) == z and tab["c"][0] == Jt * c
    # and the dense Kronecker product agrees with c Z^z X^x
    H = hamiltonian.dense_hamiltonian(N, [quartet], [Jt])
    D = 1 << (N // 2)
    M = np.zeros((D, D), dtype=complex)
    for b in range(D):
        M[b, b ^ x] = Jt * c * (-1) ** bin(b & z).count("1")
    assert np.array_equal(H, M)
    # the paper's encoding of the same string: X flags on even bits, Z flags on odd bits,
    # coeff_paper = c (-1)^popcount(x & z)  (DESIGN.md R-SIGN)
    bits, coeff = alg1.hamiltonian_tuples(N, [quartet], [Jt])
    want = sum(((x >> k) & 1) << (2 * k) | ((z >> k) & 1) << (2 * k + 1) for k in range(N // 2))
    assert int(bits[0]) == want
    assert coeff[0] == Jt * c * (-1) ** bin(x & z).count("1")


# ---------------------------------------------------------------- P5 two representations, one spectrum
@pytest.mark.parametrize("sigma_y", [majorana.SY_PRINTED, majorana.SY])
def test_P5_paper_representation(sigma_y):
    N = 8
    gp = majorana.paper_gammas(N, sigma_y)
    eye = np.eye(16)
    for m in range(N):
        for n in range(N):
            assert np.allclose(gp[m] @ gp[n] + gp[n] @ gp[m], (2 if m == n else 0) * eye)
    Dp = 8
    UD = lambda M: M[:Dp, Dp:]
    DU = lambda M: M[Dp:, :Dp]
    assert np.array_equal(UD(gp[N - 1]), -1j * np.eye(Dp)) and np.array_equal(DU(gp[N - 1]), 1j * np.eye(Dp))
    sz = majorana.site_operator(majorana.SZ, N // 2 - 2, N // 2 - 1)
    assert np.array_equal(UD(gp[N - 2]), sz) and np.array_equal(DU(gp[N - 2]), sz)
    q = _all_quartets(N)
    J = np.random.default_rng(0).normal(size=len(q))
    H_jw = hamiltonian.dense_hamiltonian(N, q, J)
    H_p = sum(Jt * gp[a] @ gp[b] @ gp[c] @ gp[d] for (a, b, c, d), Jt in zip(q, J))
    assert np.allclose(np.linalg.eigvalsh(H_jw), np.linalg.eigvalsh(H_p), atol=1e-12)
    assert np.allclose(H_p[:Dp, Dp:], 0) and np.allclose(H_p[Dp:, :Dp], 0)


# ---------------------------------------------------------------- P6 literal Algorithm 1
def test_P6_algorithm1_gives_textbook_pauli_matrices():
    # one site; coeff = lambda i^{#y}: sigma_x <01,1>, sigma_y <11,i>, sigma_z <10,1>
    e0, e1 = np.array([1, 0], dtype=complex), np.array([0, 1], dtype=complex)
    col = lambda bits, cf: np.stack([alg1.apply_python(1, [bits], [cf], e) for e in (e0, e1)], axis=1)
    assert np.array_equal(col(0b01, 1), majorana.SX)
    assert np.array_equal(col(0b10, 1), majorana.SZ)
    assert np.array_equal(col(0b11, 1j), majorana.SY)                  # DESIGN.md R-Y


@pytest.mark.parametrize("N,p", [(8, 1.0), (12, 0.2)])
def test_P6_algorithm1_equals_dense(N, p):
    q, J, _ = rng.sample_couplings(N, p, seed=11, realization=2)
    L = N // 2
    H = hamiltonian.dense_hamiltonian(N, q, J)
    psi = _random_state(1 << L, 5)
    bits, coeff = alg1.hamiltonian_tuples(N, q, J)
    want = H @ psi
    assert np.allclose(alg1.apply_python(L, bits, coeff, psi), want, atol=1e-14)
    got_c = alg1.apply_c(L, bits, coeff, psi)
    assert np.allclose(got_c, want, atol=1e-14)
    part = alg1.apply_c(L, bits, coeff, psi, 5, 13)
    assert np.array_equal(part, got_c[5:13])


# ---------------------------------------------------------------- P7 brute force: every route agrees
@pytest.mark.parametrize("N,p,gamma_norm", [(4, 1.0, 0), (6, 1.0, 1), (8, 1.0, 0), (12, 0.15, 0), (16, 0.05, 1)])
def test_P7_routes_agree(N, p, gamma_norm):
    q, J, _ = rng.sample_couplings(N, p, seed=2, realization=N)
    D = 1 << (N // 2)
    H = hamiltonian.dense_hamiltonian(N, q, J, gamma_norm)
    v = _random_state(D, N)
    want = H @ v
    assert np.allclose(hamiltonian.matvec_sequential(N, q, J, v, gamma_norm), want, atol=1e-14)
    assert np.allclose(hamiltonian.sparse_hamiltonian(N, q, J, gamma_norm).toarray(), H, atol=1e-15)
    tab = hamiltonian.derive_tables(N, q, J, gamma_norm, verify_rows=16)
    assert np.allclose(hamiltonian.matvec_from_tables(tab, v), want, atol=1e-14)
    rows = np.array([0, 1, D // 2, D - 1], dtype=np.uint64)
    cols, vals = hamiltonian.hamiltonian_rows(N, q, J, rows, gamma_norm)
    assert np.allclose((vals * v[cols.astype(int)]).sum(axis=0), want[rows.astype(int)], atol=1e-14)
    # canonical order and structure of the tables
    assert np.all(np.diff(tab["x"].astype(np.int64)) > 0)
    for g in range(len(tab["x"])):
        zs = tab["z"][tab["group_off"][g]:tab["group_off"][g + 1]].astype(np.int64)
        assert len(zs) >= 1 and np.all(np.diff(zs) > 0)
    pc = np.array([bin(int(x)).count("1") for x in tab["x"]])
    assert set(pc) <= {0, 2, 4}
    # Hermiticity rule: c real iff popcount(x & z) even
    xt = np.repeat(tab["x"], np.diff(tab["group_off"].astype(np.int64)))
    odd = hamiltonian._popcount_parity(xt & tab["z"]) == 1
    assert np.all(tab["c"].real[odd] == 0) and np.all(tab["c"].imag[~odd] == 0)
    if N <= 12:
        P = evolve.ExactPropagator(N, q, J, gamma_norm)
        assert np.allclose(P.eigenvalues(), np.linalg.eigvalsh(H), atol=1e-12)


def test_P7_dense_N16_mask_count():
    # N=16 dense has 1820 terms and 99 = 1 + C(8,2) + C(8,4) distinct X-masks
    q = _all_quartets(16)
    tab = hamiltonian.derive_tables(16, q, np.ones(len(q)))
    assert len(tab["z"]) == 1820 and len(tab["x"]) == 1 + math.comb(8, 2) + math.comb(8, 4)


# ---------------------------------------------------------------- P8 exactly solvable exponentials
@pytest.mark.parametrize("tau", [0.7, -1.3j, 0.4 - 0.9j])
def test_P8_single_term(tau):
    # H = J P with P^2 = s^8: exp(-i tau H) = cos(tau J s^4) - i sin(tau J s^4) P / s^4
    N, quartet, Jt = 8, (1, 2, 5, 7), 0.83
    for gamma_norm in (0, 1):
        s4 = majorana.gamma_scale(gamma_norm) ** 4
        v = _random_state(16, 1)
        Pv = hamiltonian.matvec_sequential(N, [quartet], [1.0], v, gamma_norm)
        want = np.cos(tau * Jt * s4) * v - 1j * np.sin(tau * Jt * s4) * Pv / s4
        prop = evolve.ExactPropagator(N, [quartet], [Jt], gamma_norm)
        assert np.allclose(prop.apply(tau, v), want, atol=1e-14)
        assert np.allclose(evolve.chebyshev_propagate(N, [quartet], [Jt], tau, v, gamma_norm), want, atol=1e-13)


def test_P8_diagonal_hamiltonian():
    # quartets (2a,2a+1,2b,2b+1) give -J Z_a Z_b: H is diagonal and exp is element-wise
    N = 10
    quartets = [(0, 1, 2, 3), (2, 3, 8, 9), (4, 5, 6, 7)]
    J = np.array([0.3, -0.7, 1.1])
    D = 32
    b = np.arange(D)
    bit = lambda a: 1 - 2 * ((b >> a) & 1)
    diag = -(J[0] * bit(0) * bit(1) + J[1] * bit(1) * bit(4) + J[2] * bit(2) * bit(3))
    v = _random_state(D, 2)
    tau = 0.9 - 0.5j
    prop = evolve.ExactPropagator(N, quartets, J)
    assert np.allclose(prop.apply(tau, v), np.exp(-1j * tau * diag) * v, atol=1e-14)
    assert np.allclose(hamiltonian.matvec_sequential(N, quartets, J, v), diag * v, atol=1e-15)


def test_P8_empty_hamiltonian_is_identity():
    v = _random_state(16, 3)
    empty_q, empty_J = np.zeros((0, 4), dtype=np.int32), np.zeros(0)
    assert np.array_equal(evolve.chebyshev_propagate(8, empty_q, empty_J, 1.0, v), v)
    assert np.array_equal(hamiltonian.matvec_sequential(8, empty_q, empty_J, v), np.zeros(16))


# ---------------------------------------------------------------- P9 group properties; two exponentials agree
def test_P9_group_properties_and_chebyshev():
    N = 12
    q, J, _ = rng.sample_couplings(N, 0.1, seed=4, realization=0)
    prop = evolve.ExactPropagator(N, q, J)
    v = _random_state(64, 4)
    a, b = 0.8 - 0.3j, -0.5 - 0.7j
    assert math.isclose(np.linalg.norm(prop.apply(2.5, v)), 1.0, rel_tol=1e-13)              # unitarity
    assert np.allclose(prop.apply(-2.5, prop.apply(2.5, v)), v, atol=1e-13)                   # E(t)E(-t) = 1
    assert np.allclose(prop.apply(a, prop.apply(b, v)), prop.apply(a + b, v), atol=1e-13)     # E(a)E(b) = E(a+b)
    for tau in (3.0, -2.0j, 1.5 - 1.0j):
        assert np.allclose(evolve.chebyshev_propagate(N, q, J, tau, v), prop.apply(tau, v), atol=1e-12)
    H = hamiltonian.dense_hamiltonian(N, q, J)
    assert np.allclose(evolve.dense_propagator(H, a) @ v, prop.apply(a, v), atol=1e-13)
    norms = [np.vdot(v, prop.apply(-1j * beta, v)).real for beta in (0.0, 0.5, 1.0, 2.0)]
    assert all(n > 0 for n in norms)                                                          # <v|e^{-bH}|v> > 0


# ---------------------------------------------------------------- P11 OTOC closed forms and the Eq. (2) reading
@pytest.mark.parametrize("gamma_norm", [0, 1])
def test_P11_otoc_closed_forms(gamma_norm):
    N = 8
    q, J, _ = rng.sample_couplings(N, 1.0, seed=5, realization=0)
    prop = evolve.ExactPropagator(N, q, J, gamma_norm)
    s4 = majorana.gamma_scale(gamma_norm) ** 4
    for seed in (1, 2):
        psi = _random_state(16, seed)
        F = otoc.otoc_same_psi(prop, N, N - 1, N - 2, 0.0, [0.0], psi, gamma_norm)
        assert abs(F[0] - (-s4)) < 1e-14                    # gWgVgWgV = -s^4 for W != V, for every psi
    H = hamiltonian.dense_hamiltonian(N, q, J, gamma_norm)
    g = majorana.jw_gammas(N, gamma_norm)
    t_grid = [0.0, 0.6, 1.7]
    Ftr = otoc.otoc_exact_trace(H, g[N - 1], g[N - 2], 2.0, t_grid)
    # R-EQ2: the supplement's operator order equals Tr[y W(t) y V y W(t) y V]
    for t, f in zip(t_grid, Ftr):
        assert abs(f - otoc.main_text_trace(H, g[N - 1], g[N - 2], 2.0, t)) < 1e-13
    assert np.all(np.abs(Ftr.imag) < 1e-13)                 # exact-trace F is real
    assert Ftr[0].real < 0 and abs(Ftr[1] / Ftr[0]) <= 1 + 1e-12
    # same-psi estimator: averaged over many psi it approaches the trace
    est = np.mean([otoc.otoc_same_psi(prop, N, N - 1, N - 2, 2.0, t_grid, _random_state(16, 100 + k), gamma_norm)
                   for k in range(300)], axis=0)
    assert np.allclose(est, Ftr, atol=0.12 * abs(Ftr[0]))


def test_P12_qualitative_decay():
    # PAPER.md:398 / Fig. 2: with s = 1 and beta = 5 the OTOC falls from 1 to ~0.8 at t* <~ 4 for N <= 54.
    # Smoke check on the normalisation reading R-NORM at N = 16 (dense), trace-estimated over a few states.
    N = 16
    q, J, _ = rng.sample_couplings(N, 1.0, seed=0, realization=0)
    prop = evolve.ExactPropagator(N, q, J)
    t_grid = [0.0, 2.0, 4.0]
    F = np.mean([otoc.otoc_same_psi(prop, N, N - 1, N - 2, 5.0, t_grid, rng.random_state(N, 0, r)) for r in range(8)],
                axis=0)
    ratio = (F / F[0]).real
    assert ratio[0] == 1.0 and 0.5 < ratio[1] < 1.0 and ratio[2] < 0.85


# ---------------------------------------------------------------- P13 Green function closed forms
@pytest.mark.parametrize("gamma_norm", [0, 1])
def test_P13_green_closed_forms(gamma_norm):
    """G(t) = <psi|e^{(it-b/2)H} g e^{-iHt} g e^{-bH/2}|psi>: (i) G(0) = s^2 <psi|e^{-bH}|psi> from the spectral
    sum; (ii) H = 0: G = s^2 for all t; (iii) one-term H = J P with g anticommuting with P: g e^{-iHt} g =
    s^2 e^{+iHt}, so G(t) = s^2 <psi|e^{(2it - b)H}|psi> = s^2 [cosh(zJs^4) + sinh(zJs^4) <P>/s^4], z = 2it - b;
    with g commuting with P the t-dependence cancels: G(t) = G(0); (iv) the same-psi value averaged over many psi
    approaches the exact trace, which is what PAPER.md:212 estimates."""
    s = majorana.gamma_scale(gamma_norm)
    s2, s4 = s * s, s ** 4
    N = 8
    q, J, _ = rng.sample_couplings(N, 1.0, seed=7, realization=0)
    prop = evolve.ExactPropagator(N, q, J, gamma_norm)
    H = hamiltonian.dense_hamiltonian(N, q, J, gamma_norm)
    w, U = np.linalg.eigh(H)
    psi = _random_state(16, 3)
    beta = 1.7
    G0 = green.green_same_psi(prop, N, N - 1, beta, [0.0], psi, gamma_norm)[0]
    assert abs(G0 - s2 * np.sum(np.abs(U.conj().T @ psi) ** 2 * np.exp(-beta * w))) < 1e-13
    # (ii) empty Hamiltonian
    empty = evolve.ExactPropagator(N, np.zeros((0, 4), dtype=np.int32), np.zeros(0), gamma_norm)
    assert np.allclose(green.green_same_psi(empty, N, 2, beta, [0.0, 1.0, 3.0], psi, gamma_norm), s2, atol=1e-14)
    # (iii) single term (0,1,2,3) = -s^4 Z0 Z1: gamma_0 (X on qubit 0) anticommutes with it, gamma_6 commutes
    Jq = 0.83
    one = evolve.ExactPropagator(N, np.array([[0, 1, 2, 3]], dtype=np.int32), np.array([Jq]), gamma_norm)
    P = hamiltonian.dense_hamiltonian(N, np.array([[0, 1, 2, 3]], dtype=np.int32), np.array([1.0]), gamma_norm)
    expP = np.vdot(psi, P @ psi).real / s4
    t_grid = np.array([0.0, 0.4, 1.3])
    z = 2j * t_grid - beta
    want = s2 * (np.cosh(z * Jq * s4) + np.sinh(z * Jq * s4) * expP)
    assert np.allclose(green.green_same_psi(one, N, 0, beta, t_grid, psi, gamma_norm), want, atol=1e-13)
    Gc = green.green_same_psi(one, N, 6, beta, t_grid, psi, gamma_norm)
    assert np.allclose(Gc, Gc[0], atol=1e-13)
    # (iv) trace estimator
    g = majorana.jw_gammas(N, gamma_norm)
    tg = [0.0, 0.7, 1.9]
    Gtr = green.green_exact_trace(H, g[N - 1], 1.0, tg)
    est = np.mean([green.green_same_psi(prop, N, N - 1, 1.0, tg, _random_state(16, 500 + k), gamma_norm)
                   for k in range(300)], axis=0)
    assert np.allclose(est, Gtr, atol=0.12 * abs(Gtr[0]))
    assert abs(Gtr[0].imag) < 1e-13 and Gtr[0].real > 0


# ---------------------------------------------------------------- P14 parity blocks
@pytest.mark.parametrize("gamma_norm", [0, 1])
def test_P14_parity_blocks(gamma_norm):
    """(i) spectrum(H) = spectrum(H_UU) u spectrum(H_DD); (ii) the paper's statements about the last two gammas hold
    for the Jordan-Wigner blocks too: the block of gamma_{N-1} is -i s (+1 | -1) times the identity with opposite signs
    for the two directions (g^{UD} = -g^{DU} = -i 1), the block of gamma_{N-2} is the same diagonal sign
    matrix in both directions; (iii) F(t) and G(t) of the full space are the sums of their two block
    terms ("+ swap UD"), for the sector components of the same psi; (iv) (H v) restricted = H_ss
    v_s, (gamma v) restricted = block times v restricted."""
    N, L = 10, 5
    s = majorana.gamma_scale(gamma_norm)
    q, J, _ = rng.sample_couplings(N, 0.4, seed=11, realization=0)
    H = hamiltonian.dense_hamiltonian(N, q, J, gamma_norm)
    blocks = [parity.block_hamiltonian(N, q, J, sec, gamma_norm) for sec in (0, 1)]
    w = np.sort(np.concatenate([np.linalg.eigvalsh(b) for b in blocks]))
    assert np.allclose(w, np.linalg.eigvalsh(H), atol=1e-12)
    # (ii)
    gl0, gl1 = parity.block_gamma(N, N - 1, 0, gamma_norm), parity.block_gamma(N, N - 1, 1, gamma_norm)
    eye = np.eye(1 << (L - 1))
    assert np.allclose(gl0, -gl1, atol=0) and np.allclose(np.abs(gl0), s * eye, atol=1e-15)
    assert np.allclose(gl0, gl0[0, 0] * eye, atol=0) and abs(gl0[0, 0].real) == 0.0 and abs(gl0[0, 0].imag) == s
    gm0, gm1 = parity.block_gamma(N, N - 2, 0, gamma_norm), parity.block_gamma(N, N - 2, 1, gamma_norm)
    assert np.array_equal(gm0, gm1) and np.allclose(np.abs(gm0), s * eye, atol=1e-15)
    assert np.count_nonzero(gm0 - np.diag(np.diag(gm0))) == 0 and set(np.unique(np.diag(gm0).real / s)) == {-1.0, 1.0}
    # (iv)
    v = _random_state(1 << L, 4)
    for sec in (0, 1):
        vs = parity.restrict(v, L, sec)
        full = parity.embed(vs, L, sec)
        assert np.allclose(parity.restrict(H @ full, L, sec), blocks[sec] @ vs, atol=1e-14)
        assert np.allclose(parity.restrict(H @ full, L, 1 - sec), 0, atol=0)
        for n in (0, 3, N - 2, N - 1):
            gv = hamiltonian.apply_gamma(N, n, full, gamma_norm)
            assert np.allclose(parity.restrict(gv, L, 1 - sec), parity.block_gamma(N, n, 1 - sec, gamma_norm) @ vs, atol=1e-15)
            assert np.allclose(parity.restrict(gv, L, sec), 0, atol=0)
    # (iii)
    prop = evolve.ExactPropagator(N, q, J, gamma_norm)
    props = [parity.BlockPropagator(N, q, J, sec, gamma_norm) for sec in (0, 1)]
    t_grid = [0.0, 0.8, 2.1]
    F = otoc.otoc_same_psi(prop, N, N - 1, N - 2, 1.5, t_grid, v, gamma_norm)
    Fb = sum(parity.otoc_block_same_psi(props, N, N - 1, N - 2, 1.5, t_grid, parity.restrict(v, L, sec), sec, gamma_norm)
             for sec in (0, 1))
    assert np.allclose(F, Fb, atol=1e-13)
    F2 = otoc.otoc_same_psi(prop, N, 2, 5, 1.5, t_grid, v, gamma_norm)
    F2b = sum(parity.otoc_block_same_psi(props, N, 2, 5, 1.5, t_grid, parity.restrict(v, L, sec), sec, gamma_norm)
              for sec in (0, 1))
    assert np.allclose(F2, F2b, atol=1e-13)
    G = green.green_same_psi(prop, N, N - 1, 1.5, t_grid, v, gamma_norm)
    Gb = sum(parity.green_block_same_psi(props, N, N - 1, 1.5, t_grid, parity.restrict(v, L, sec), sec, gamma_norm)
             for sec in (0, 1))
    assert np.allclose(G, Gb, atol=1e-13)


# ---------------------------------------------------------------- P15 generic Pauli sums
def test_P15_pauli_strings_and_spin_chains():
    """(i) Z X = i Y for the textbook Y (R-Y), so the string (x=1, z=1, c=-i) is Y; a JW Majorana is the string the
    term compiler uses; (ii) the periodic transverse-field Ising chain has the free-fermion ground energy
    E0 = -sum_m sqrt(J^2 + h^2 - 2 J h cos(pi (2m+1)/L)) (even-parity sector, textbook); (iii) the Heisenberg chain
    commutes with total S^z and two sites give the singlet/triplet levels -3J, +J."""
    Y = np.array([[0, -1j], [1j, 0]])
    assert np.allclose(pauli.string_matrix(1, 1, 1, -1j), Y, atol=0)
    assert np.allclose(pauli.string_matrix(2, 0b10, 0b01, 1.0), np.kron(majorana.SX, majorana.SZ), atol=0)
    g = majorana.jw_gammas(8)
    assert np.allclose(pauli.string_matrix(4, 0b0100, 0b0011, 1.0), g[4], atol=0)        # gamma_4 = Z0 Z1 X2
    assert np.allclose(pauli.string_matrix(4, 0b0100, 0b0111, -1j), g[5], atol=0)       # gamma_5 = Z0 Z1 Y2
    L, J, h = 8, 1.0, 0.7
    H = pauli.sum_matrix(L, pauli.transverse_ising_terms(L, J, h))
    assert np.allclose(H, H.conj().T, atol=0)
    k = np.pi * (2 * np.arange(L) + 1) / L
    assert abs(np.linalg.eigvalsh(H)[0] + np.sum(np.sqrt(J * J + h * h - 2 * J * h * np.cos(k)))) < 1e-12
    H2 = pauli.sum_matrix(2, pauli.heisenberg_terms(2, 1.0, 1.0, 1.0))
    assert np.allclose(np.linalg.eigvalsh(H2), [-3.0, 1.0, 1.0, 1.0], atol=1e-13)
    H6 = pauli.sum_matrix(6, pauli.heisenberg_terms(6, 1.0, 1.0, 0.5, periodic=True))
    Sz = sum(pauli.string_matrix(6, 0, 1 << q) for q in range(6))
    assert np.allclose(H6 @ Sz, Sz @ H6, atol=1e-13) and np.allclose(H6, H6.conj().T, atol=0)


# ------------------------------------------------------------------------------------------------------------
# P16: non-Hermitian operators (oracle/nonhermitian.py)
# ------------------------------------------------------------------------------------------------------------
def test_P16_nonhermitian_propagator_closed_forms():
    from oracle import nonhermitian as onh
    v = np.array([0.3 - 0.2j, 1.1 + 0.4j])
    # nilpotent: H^2 = 0, so exp(-i tau H) = 1 - i tau H exactly (no eigenbasis exists)
    Hn = np.array([[0.0, 2.5], [0.0, 0.0]], dtype=np.complex128)
    for tau in (0.7, -1.3 + 0.4j):
        assert np.allclose(onh.expm_propagate(Hn, tau, v), v - 1j * tau * (Hn @ v), rtol=0, atol=1e-15)
    # diagonal complex H: element-wise
    d = np.array([0.4 + 0.3j, -1.2 - 0.7j])
    assert np.allclose(onh.expm_propagate(np.diag(d), 0.9 - 0.2j, v), np.exp(-1j * (0.9 - 0.2j) * d) * v, atol=1e-15)
    # Hermitian H: the eigh propagator of oracle/evolve.py
    r = np.random.default_rng(3)
    A = r.normal(size=(8, 8)) + 1j * r.normal(size=(8, 8))
    Hh = A + A.conj().T
    w = r.normal(size=8) + 1j * r.normal(size=8)
    assert np.allclose(onh.expm_propagate(Hh, 0.6 - 0.3j, w), evolve.dense_propagator(Hh, 0.6 - 0.3j) @ w, atol=1e-12)
    # non-normal H: group law, and exp(-i t (i K)) = exp(t K) for Hermitian K
    assert np.linalg.norm(A @ A.conj().T - A.conj().T @ A) > 1.0
    one = onh.expm_propagate(A, 0.5, onh.expm_propagate(A, 0.2 - 0.1j, w))
    assert np.allclose(one, onh.expm_propagate(A, 0.7 - 0.1j, w), atol=1e-11)
    wk, Uk = np.linalg.eigh(Hh)
    assert np.allclose(onh.expm_propagate(1j * Hh, 0.3, w), Uk @ (np.exp(0.3 * wk) * (Uk.conj().T @ w)), atol=1e-10)


def test_P16_complex_syk_hamiltonian():
    """Complex couplings: linear in J (real J reproduces the dense Hermitian H of Eq. 1 built by matrix products); H - H^+ =
    2 i H[Im J]; a purely imaginary J gives an anti-Hermitian H."""
    from oracle import nonhermitian as onh
    N = 10
    q, J, _ = rng.sample_couplings(N, 0.3, 4, 0)
    H0 = hamiltonian.dense_hamiltonian(N, q, J)
    assert np.allclose(onh.complex_syk_hamiltonian(N, q, J.astype(np.complex128)), H0, atol=1e-15)
    Jc = J * np.exp(1j * np.linspace(0.2, 2.5, len(J)))
    Hc = onh.complex_syk_hamiltonian(N, q, Jc)
    assert np.allclose(Hc - Hc.conj().T, 2j * hamiltonian.dense_hamiltonian(N, q, Jc.imag.copy()), atol=1e-14)
    assert np.allclose(Hc, sum(Jt * M for Jt, M in zip(Jc, [hamiltonian.dense_hamiltonian(N, [qq], [1.0]) for qq in q])), atol=1e-14)
    Hi = onh.complex_syk_hamiltonian(N, q, 1j * J)
    assert np.allclose(Hi, -Hi.conj().T, atol=1e-15)


def test_paper_statements_fixture_is_what_the_oracle_uses():
    """tests/golden/paper_statements.txt lists values the paper prints, each with its PAPER.md line.  The ones that are
    numbers or tables are read here and compared with what the oracle computes with: the <bits> encoding of the four site
    operators against oracle/alg1.py, the coupling variance 3/(8 p N^3) against the sample
    variance of oracle/rng.py's couplings, k = (p/N) C(N,4) against the mean number of kept terms, and the two Clifford
    normalisations against the Kronecker-built gammas."""
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "paper_statements.txt")
    stm = {}
    for line in open(path):
        line = line.strip()
        if not line or line.startswith("#"):
            continue
        key, rest = line.split("=", 1)
        value, cite = rest.rsplit(";", 1)
        assert "PAPER.md:" in cite, line
        stm[key.strip()] = value.strip()
    enc = dict(tok.split("=") for tok in stm["encoding"].split())
    assert {int(k[1]): int(v, 2) for k, v in enc.items()} == alg1._CODE
    assert stm["coupling_variance"].replace(" ", "") == "3/(8pN^3)"
    N, k = 24, 6.0
    p = k * N / math.comb(N, 4)
    Js = np.concatenate([rng.sample_couplings(N, p, 11, r)[1] for r in range(400)])
    var = eval(stm["coupling_variance"].replace("^", "**").replace("8 p N", "8*p*N"), {"p": p, "N": N})
    assert abs(np.var(Js) / var - 1.0) < 0.03
    assert stm["sparsity"].replace(" ", "") == "k=(p/N)C(N,4)"
    assert abs(len(Js) / 400.0 - (p / N) * math.comb(N, 4) * N) < 0.05 * k * N          # mean kept terms = k N
    for key, gn, scale in (("clifford_main_text", majorana.GAMMA_HALF, 1.0), ("clifford_supplement", majorana.GAMMA_PAULI, 2.0)):
        assert ("2 delta" in stm[key]) == (scale == 2.0)
        g = majorana.jw_gammas(6, gn)
        assert np.allclose(g[1] @ g[1] + g[1] @ g[1], scale * np.eye(8)) and np.allclose(g[0] @ g[3] + g[3] @ g[0], 0)


def test_P15_apply_string_equals_string_matrix():
    """pauli.apply_string (site factors contracted one by one) against the Kronecker-product matrix of the same string, for
    every (x, z) on 3 qubits and random strings on 7 qubits; apply_sum against sum_matrix; Z X = iY on one site."""
    rs = np.random.default_rng(5)
    L = 3
    v = rs.standard_normal(8) + 1j * rs.standard_normal(8)
    for x in range(8):
        for z in range(8):
            assert np.allclose(pauli.apply_string(L, x, z, 0.5 - 2j, v), pauli.string_matrix(L, x, z, 0.5 - 2j) @ v, atol=1e-14)
    L = 7
    v = rs.standard_normal(128) + 1j * rs.standard_normal(128)
    terms = [(int(rs.integers(0, 128)), int(rs.integers(0, 128)), complex(rs.standard_normal(), rs.standard_normal()))
             for _ in range(12)]
    assert np.allclose(pauli.apply_sum(L, terms, v), pauli.sum_matrix(L, terms) @ v, atol=1e-13)
    e0, e1 = np.array([1.0, 0.0]), np.array([0.0, 1.0])
    assert np.allclose(pauli.apply_string(1, 1, 1, 1.0, e0), -e1)            # Z X |0> = Z |1> = -|1> = (iY)|0>
    assert np.allclose(pauli.apply_string(1, 1, 1, 1.0, e1), e0)             # Z X |1> = |0>     = (iY)|1>
