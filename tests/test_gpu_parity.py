"""Parity of the CUDA path (through the C ABI) against the CPU oracle, element by element.  Needs a B200.

Tolerances (BASELINE.json north_star): relative L2 error <= 1e-10 for complex128, <= 1e-5 for complex64;
integer tables bit-exact (tests/test_host_library.py).
"""
import math

import numpy as np
import pytest

from oracle import evolve as oev
from oracle import green as ogreen
from oracle import hamiltonian as ohm
from oracle import majorana
from oracle import otoc as ootoc
from oracle import rng as orng
from paper_2311_00639_b200 import inputs

pytestmark = pytest.mark.gpu

TOL = {"c128": 1e-10, "c64": 1e-5}


@pytest.fixture(scope="module")
def B():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2311_00639_b200 import binding   # raises if the library is not built: no CPU path
    return binding


@pytest.fixture(scope="module")
def torch():
    import torch
    return torch


def tdtype(torch, name):
    return torch.complex128 if name == "c128" else torch.complex64


def npdtype(name):
    return np.complex128 if name == "c128" else np.complex64


def relerr(a, b):
    a = np.asarray(a, dtype=np.complex128)
    b = np.asarray(b, dtype=np.complex128)
    nb = np.linalg.norm(b)
    return float(np.linalg.norm(a - b) / (nb if nb > 0 else 1.0))


def to_dev(torch, a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def work(torch, nbytes):
    return torch.empty(int(nbytes) + 256, dtype=torch.uint8, device="cuda")


def couplings(N, k, seed=0, realization=0):
    return orng.sample_couplings(N, inputs.bernoulli_p(N, k), seed, realization)[:2]


# ------------------------------------------------------------------------------------------------------------
# a-2 apply_H
# ------------------------------------------------------------------------------------------------------------
APPLY_CASES = [
    # N, k (None = dense), gamma_norm
    (4, None, 0), (6, None, 1), (8, None, 0), (12, None, 0), (16, None, 0), (16, 4, 1),
    (20, 4, 0), (22, 8, 0), (24, 4, 0), (26, 2, 0), (28, 4, 1), (30, 8, 0), (32, 4, 0),
    (24, None, 0), (28, None, 1),      # dense beyond the shared-memory table: generic and dense-table kernels
]


@pytest.mark.parametrize("dt", ["c128", "c64"])
@pytest.mark.parametrize("N,k,gn", APPLY_CASES)
def test_apply_H_vs_oracle(B, torch, N, k, gn, dt):
    """out = H.in against the oracle's sequential-gamma product (O5), every kernel the handle can use
    (0 generic, 1 16 KiB-tile TMA, 2 register-tile TMA, 3 scatter-tile TMA, 4 dense-table)."""
    q, J = couplings(N, k, seed=1)
    D = 1 << (N // 2)
    v = inputs.gaussian_state(D, seed=100 + N, dtype=npdtype(dt))
    ref = ohm.matvec_sequential(N, q, J, v.astype(np.complex128), gn)
    h = B.syk_build_from_terms(N, q, J, gn)
    d_in = to_dev(torch, v)
    kinds = {0}
    for want in (1, 2, 3, 4):
        B.syk_set_apply_H_kernel(h, want)
        kinds.add(B.syk_apply_H_kernel_kind(h, B.dtype_code(d_in)))
    if N >= 28 and k is not None:
        assert kinds == {0, 1, 2, 3, 4}
    if N >= 24 and k is None:
        assert kinds >= {0, 4}
    for kind in sorted(kinds):
        B.syk_set_apply_H_kernel(h, kind)
        assert B.syk_apply_H_kernel_kind(h, B.dtype_code(d_in)) == kind
        d_out = torch.full((D,), complex(float("nan"), float("nan")), dtype=tdtype(torch, dt), device="cuda")
        B.syk_apply_H(h, d_in, d_out)
        torch.cuda.synchronize()
        assert relerr(d_out.cpu().numpy(), ref) <= TOL[dt], (kind, N, dt)
        assert np.array_equal(d_in.cpu().numpy(), v), "apply_H modified its input"


def test_apply_H_tma_kernel_is_selected_for_sparse(B, torch):
    """The sm_100a tile kernel must be the default whenever the vector spans at least one tile."""
    q, J = couplings(32, 4)
    h = B.syk_build_from_terms(32, q, J)
    assert B.syk_apply_H_kernel_kind(h, B.SYK_C128) == 1
    assert B.syk_apply_H_kernel_kind(h, B.SYK_C64) == 1


@pytest.mark.parametrize("dt", ["c128", "c64"])
@pytest.mark.parametrize("qubits", [(0, 1, 2, 3, 4), (0, 3, 7, 9, 11), (10, 11, 12, 13), (5, 10, 11, 12, 13)])
def test_apply_H_structured_masks(B, torch, qubits, dt):
    """Mask sets confined to the warp-local bits, the tile-local bits, only bits above the tile, and mixed."""
    N = 28
    q, J = inputs.quartets_on_qubits(qubits, 40, seed=5, sigma=0.3)
    D = 1 << (N // 2)
    v = inputs.gaussian_state(D, seed=3, dtype=npdtype(dt))
    ref = ohm.matvec_sequential(N, q, J, v.astype(np.complex128))
    h = B.syk_build_from_terms(N, q, J)
    d_in = to_dev(torch, v)
    for kind in (0, 1, 2, 3, 4):
        B.syk_set_apply_H_kernel(h, kind)
        assert B.syk_apply_H_kernel_kind(h, B.dtype_code(d_in)) == kind
        d_out = torch.zeros(D, dtype=tdtype(torch, dt), device="cuda")
        B.syk_apply_H(h, d_in, d_out)
        assert relerr(d_out.cpu().numpy(), ref) <= TOL[dt], kind


def test_apply_H_literal_algorithm1(B, torch):
    """Third route (pin P6): the paper's Algorithm 1 transcribed literally in C equals the CUDA result."""
    from oracle import alg1
    N = 24
    q, J = couplings(N, 4, seed=2)
    D = 1 << (N // 2)
    v = inputs.gaussian_state(D, seed=9)
    bits, coeff = alg1.hamiltonian_tuples(N, q, J)
    ref = alg1.apply_c(N // 2, bits, coeff, v)
    h = B.syk_build_from_terms(N, q, J)
    d_out = torch.zeros(D, dtype=torch.complex128, device="cuda")
    B.syk_apply_H(h, to_dev(torch, v), d_out)
    assert relerr(d_out.cpu().numpy(), ref) <= 1e-13


def test_apply_H_edge_cases(B, torch):
    # empty Hamiltonian: out = 0
    h0 = B.syk_build_from_terms(16, np.zeros((0, 4), dtype=np.int32), np.zeros(0))
    v = to_dev(torch, inputs.gaussian_state(256, 1))
    out = torch.full((256,), 7.0 + 1j, dtype=torch.complex128, device="cuda")
    B.syk_apply_H(h0, v, out)
    assert float(out.abs().max()) == 0.0
    # in == out and overlapping buffers are refused
    h = B.syk_build_hamiltonian(16, 1.0, 0)
    with pytest.raises(B.SykError):
        B.syk_apply_H(h, v, v)
    big = torch.zeros(256 + 128, dtype=torch.complex128, device="cuda")
    with pytest.raises(B.SykError):
        B.syk_apply_H(h, big[:256], big[128:])
    # unaligned pointer
    raw = torch.zeros(2 * 258, dtype=torch.float64, device="cuda")
    with pytest.raises(B.SykError):
        B._check(B._lib.syk_apply_H(h.handle, B.SYK_C128, raw.data_ptr() + 8, out.data_ptr(), 0), "apply")
    # a CPU tensor is refused by the binding: there is no CPU path
    with pytest.raises(B.SykError):
        B.syk_apply_H(h, torch.zeros(256, dtype=torch.complex128), out)


def test_apply_H_bitwise_reproducible(B, torch):
    q, J = couplings(30, 4)
    h = B.syk_build_from_terms(30, q, J)
    D = 1 << 15
    v = to_dev(torch, inputs.gaussian_state(D, 2))
    a = torch.zeros(D, dtype=torch.complex128, device="cuda")
    b = torch.zeros(D, dtype=torch.complex128, device="cuda")
    B.syk_apply_H(h, v, a)
    B.syk_apply_H(h, v, b)
    assert torch.equal(torch.view_as_real(a), torch.view_as_real(b))


def test_apply_H_batched_and_host(B, torch):
    N, nb = 20, 5
    D = 1 << (N // 2)
    stride = D + 64
    hams, refs = [], []
    vin = np.zeros((nb, stride), dtype=np.complex128)
    for r in range(nb):
        q, J = couplings(N, 4, seed=0, realization=r)
        hams.append(B.syk_build_hamiltonian(N, inputs.bernoulli_p(N, 4), 0, r))
        vin[r, :D] = inputs.gaussian_state(D, seed=50 + r)
        refs.append(ohm.matvec_sequential(N, q, J, vin[r, :D]))
    d_in = to_dev(torch, vin.reshape(-1))
    d_out = torch.zeros(nb * stride, dtype=torch.complex128, device="cuda")
    B.syk_apply_H_batched(hams, d_in, d_out, stride)
    got = d_out.cpu().numpy().reshape(nb, stride)
    for r in range(nb):
        assert relerr(got[r, :D], refs[r]) <= 1e-10
        assert np.all(got[r, D:] == 0)
    # host entry point (copies inside)
    h_out = np.zeros(D, dtype=np.complex128)
    B.syk_apply_H_host(hams[0], np.ascontiguousarray(vin[0, :D]), h_out, work(torch, 2 * D * 16))
    assert relerr(h_out, refs[0]) <= 1e-10


# ------------------------------------------------------------------------------------------------------------
# gamma, dot, random state
# ------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("dt", ["c128", "c64"])
@pytest.mark.parametrize("gn", [0, 1])
def test_apply_gamma_all_n(B, torch, dt, gn):
    N = 12
    D = 1 << (N // 2)
    v = inputs.gaussian_state(D, 4, npdtype(dt))
    d_in = to_dev(torch, v)
    for n in range(N):
        ref = ohm.apply_gamma(N, n, v.astype(np.complex128), gn)
        d_out = torch.zeros(D, dtype=tdtype(torch, dt), device="cuda")
        B.syk_apply_gamma(N, n, d_in, d_out, gn)
        assert relerr(d_out.cpu().numpy(), ref) <= (1e-15 if dt == "c128" else 1e-7)
        inplace = d_in.clone()
        B.syk_apply_gamma(N, n, inplace, inplace, gn)
        assert torch.equal(torch.view_as_real(inplace), torch.view_as_real(d_out))


def test_apply_gamma_large_and_clifford(B, torch):
    """{g_m, g_n} = 2 delta at N = 44 on a random vector: the kernel's signs at high bits."""
    N = 44
    D = 1 << (N // 2)
    scratch = work(torch, B.syk_reduce_scratch_bytes())
    v = torch.empty(D, dtype=torch.complex128, device="cuda")
    B.syk_random_state(N, 0, 0, v, scratch)
    a, b = torch.empty_like(v), torch.empty_like(v)
    for m, n in ((0, 43), (43, 42), (21, 20), (7, 30)):
        B.syk_apply_gamma(N, n, v, a)
        B.syk_apply_gamma(N, m, a, a)
        B.syk_apply_gamma(N, m, v, b)
        B.syk_apply_gamma(N, n, b, b)
        assert float((a + b).abs().max()) == 0.0          # anticommute exactly
    B.syk_apply_gamma(N, 43, v, a)
    B.syk_apply_gamma(N, 43, a, a)
    assert torch.equal(torch.view_as_real(a), torch.view_as_real(v))   # g^2 = 1 exactly


@pytest.mark.parametrize("dt", ["c128", "c64"])
def test_dot(B, torch, dt):
    N = 22
    D = 1 << (N // 2)
    a = inputs.gaussian_state(D, 1, npdtype(dt))
    b = inputs.gaussian_state(D, 2, npdtype(dt))
    scratch = work(torch, B.syk_reduce_scratch_bytes())
    got = B.syk_dot(N, to_dev(torch, a), to_dev(torch, b), scratch)
    ref = np.vdot(a.astype(np.complex128), b.astype(np.complex128))
    assert abs(got - ref) <= 1e-13


@pytest.mark.parametrize("N", [8, 20, 24])
def test_random_state_vs_oracle(B, torch, N):
    """R-PSI / R-RNG implemented twice: counter-based draws are bit-identical, Box-Muller to libm rounding."""
    D = 1 << (N // 2)
    scratch = work(torch, B.syk_reduce_scratch_bytes())
    psi = torch.empty(D, dtype=torch.complex128, device="cuda")
    B.syk_random_state(N, 5, 3, psi, scratch)
    ref = orng.random_state(N, 5, 3)
    assert relerr(psi.cpu().numpy(), ref) <= 1e-13
    psi32 = torch.empty(D, dtype=torch.complex64, device="cuda")
    B.syk_random_state(N, 5, 3, psi32, scratch)
    assert relerr(psi32.cpu().numpy(), ref) <= 2e-7
    assert abs(float(torch.linalg.vector_norm(psi)) - 1.0) <= 1e-14


# ------------------------------------------------------------------------------------------------------------
# a-3 / a-4 Lanczos and the Krylov exponential
# ------------------------------------------------------------------------------------------------------------
def test_lanczos_identities(B, torch):
    """Pin P10: alpha_1 = <v|H|v>, beta_2^2 = <v|H^2|v> - alpha_1^2, Ritz values inside the spectrum; the
    matvecs on the right-hand sides are the oracle's."""
    N = 16
    q, J = couplings(N, None)
    D = 1 << (N // 2)
    psi = 3.0 * inputs.gaussian_state(D, 8)                      # un-normalised on purpose
    h = B.syk_build_from_terms(N, q, J)
    m = 24
    wk = work(torch, B.syk_krylov_workspace_bytes(h, B.SYK_C128, {"krylov_dim": m}))
    d_psi = to_dev(torch, psi)
    alpha, beta, st = B.syk_lanczos_run(h, d_psi, m, wk)
    assert np.array_equal(d_psi.cpu().numpy(), psi)
    v = psi / np.linalg.norm(psi)
    Hv = ohm.matvec_sequential(N, q, J, v)
    a1 = np.vdot(v, Hv).real
    assert abs(beta[0] - 3.0) <= 1e-13
    assert abs(alpha[0] - a1) <= 1e-13
    assert abs(beta[1] ** 2 - (np.vdot(Hv, Hv).real - a1 ** 2)) <= 1e-13
    T = np.diag(alpha) + np.diag(beta[1:m], 1) + np.diag(beta[1:m], -1)
    ritz = np.linalg.eigvalsh(T)
    w = np.linalg.eigvalsh(ohm.dense_hamiltonian(N, q, J))
    assert ritz.min() >= w.min() - 1e-10 and ritz.max() <= w.max() + 1e-10
    # extremal Ritz values converge first: after 24 of 256 steps the lowest one is within 1 % of the band width
    assert abs(ritz.min() - w.min()) < 1e-2 * (w.max() - w.min())
    assert st["n_matvec"] == m


@pytest.mark.parametrize("dt", ["c128", "c64"])
def test_fused_lanczos_every_kernel_kind(B, torch, dt):
    """The fused epilogue (out = acc/|u_j| - (|u_j|/|u_{j-1}|) prev, <u_j|out> partial sums) of every apply_H
    kernel: 6 Lanczos steps at N=28 (several tiles) against the textbook three-term recurrence run with the oracle's
    sequential-gamma matvec in fp64."""
    N, m = 28, 6
    q, J = couplings(N, 4, seed=2)
    D = 1 << (N // 2)
    psi = inputs.gaussian_state(D, 21, npdtype(dt))
    v = psi.astype(np.complex128)
    b0 = np.linalg.norm(v)
    v = v / b0
    v_prev = np.zeros_like(v)
    beta_prev = 0.0
    a_ref, b_ref = [], [b0]
    for _ in range(m):
        w = ohm.matvec_sequential(N, q, J, v) - beta_prev * v_prev
        a = np.vdot(v, w).real
        w = w - a * v
        bn = np.linalg.norm(w)
        a_ref.append(a)
        b_ref.append(bn)
        v_prev, v, beta_prev = v, w / bn, bn
    h = B.syk_build_from_terms(N, q, J)
    code = B.SYK_C128 if dt == "c128" else B.SYK_C64
    wk = work(torch, B.syk_krylov_workspace_bytes(h, code, {"krylov_dim": m}))
    d_psi = to_dev(torch, psi)
    tol = 1e-11 if dt == "c128" else 2e-5
    for kind in (0, 1, 2, 3, 4):
        B.syk_set_apply_H_kernel(h, kind)
        assert B.syk_apply_H_kernel_kind(h, code) == kind
        alpha, beta, st = B.syk_lanczos_run(h, d_psi, m, wk)
        assert np.max(np.abs(np.asarray(alpha) - np.asarray(a_ref))) <= tol, (kind, dt)
        assert np.max(np.abs(np.asarray(beta) - np.asarray(b_ref))) <= tol, (kind, dt)


EVOLVE_CASES = [
    # N, k, tau, opts
    (16, None, (1.0, 0.0), {"krylov_dim": 20}),
    (16, None, (0.0, -1.25), {"krylov_dim": 20}),
    (16, None, (3.0, -1.25), {"krylov_dim": 20}),
    (16, None, (-3.0, -1.25), {"krylov_dim": 12, "two_pass": 1}),
    (16, 4, (10.0, 0.0), {"krylov_dim": 30}),
    (20, 4, (2.0, -0.625), {"krylov_dim": 24, "two_pass": 1}),
    (24, 4, (1.5, -1.25), {"krylov_dim": 30}),
    (24, 4, (1.5, -1.25), {"krylov_dim": 5, "two_pass": 1}),      # the paper's restart dimension
]


@pytest.fixture(scope="module")
def propagators():
    cache = {}

    def get(N, k, gn=0):
        key = (N, k, gn)
        if key not in cache:
            q, J = couplings(N, k, seed=4)
            cache[key] = (q, J, oev.ExactPropagator(N, q, J, gn))
        return cache[key]
    return get


@pytest.mark.parametrize("dt", ["c128", "c64"])
@pytest.mark.parametrize("N,k,tau,opts", EVOLVE_CASES)
def test_krylov_evolve_vs_exact(B, torch, propagators, N, k, tau, opts, dt):
    """e^{-i tau H} psi against full diagonalisation (O6) for real, imaginary and complex tau."""
    q, J, prop = propagators(N, k)
    D = 1 << (N // 2)
    psi = inputs.gaussian_state(D, 21, npdtype(dt))
    ref = prop.apply(complex(*tau), psi.astype(np.complex128))
    h = B.syk_build_from_terms(N, q, J)
    code = B.SYK_C128 if dt == "c128" else B.SYK_C64
    wk = work(torch, B.syk_krylov_workspace_bytes(h, code, opts))
    d_psi = to_dev(torch, psi)
    st = B.syk_krylov_evolve(h, d_psi, tau[0], tau[1], wk, opts)
    assert relerr(d_psi.cpu().numpy(), ref) <= TOL[dt], st
    assert st["err_est"] <= TOL[dt] and st["n_substeps"] >= 1 and st["n_matvec"] >= 2


@pytest.mark.parametrize("dt", ["c128", "c64"])
def test_two_pass_every_tile_kernel_vs_chebyshev(B, torch, dt):
    """Two-pass Lanczos (bounded vector count) makes `out` alias `prev` in the fused epilogue from step 3
    on.  The register-tile, scatter-tile and dense-table kernels -- the ones that run the N = 64 two-pass workload --
    are forced at N = 28 (2..4 tiles, several ring chunks per tile) and compared with the oracle's Chebyshev propagator
    (O8: shares nothing with Lanczos), for real and complex tau, and with the one-pass result of the same kernel."""
    N = 28
    q, J = couplings(N, 4, seed=9)
    D = 1 << (N // 2)
    psi = inputs.gaussian_state(D, 41, npdtype(dt))
    code = B.SYK_C128 if dt == "c128" else B.SYK_C64
    h = B.syk_build_from_terms(N, q, J)
    o2 = {"krylov_dim": 6, "two_pass": 1}
    o1 = {"krylov_dim": 6}
    w2 = work(torch, B.syk_krylov_workspace_bytes(h, code, o2))
    w1 = work(torch, B.syk_krylov_workspace_bytes(h, code, o1))
    for tau in ((1.2, 0.0), (-0.7, -1.25)):
        ref = oev.chebyshev_propagate(N, q, J, complex(*tau), psi.astype(np.complex128))
        for kind in (1, 2, 3, 4):
            B.syk_set_apply_H_kernel(h, kind)
            assert B.syk_apply_H_kernel_kind(h, code) == kind
            d2 = to_dev(torch, psi)
            st2 = B.syk_krylov_evolve(h, d2, tau[0], tau[1], w2, o2)
            assert relerr(d2.cpu().numpy(), ref) <= TOL[dt], (kind, tau, st2)
            assert st2["n_substeps"] >= 2                              # several rounds: u_1 is rebuilt from psi each time
            d1 = to_dev(torch, psi)
            st1 = B.syk_krylov_evolve(h, d1, tau[0], tau[1], w1, o1)
            assert st1["n_substeps"] == st2["n_substeps"]              # the recurrence is repeated bit-identically
            assert relerr(d2.cpu().numpy(), d1.cpu().numpy()) <= (1e-13 if dt == "c128" else 2e-6), (kind, tau)


def test_krylov_dim2_two_pass(B, torch, propagators):
    """The paper's N >= 62 setting, Krylov dimension 2: a first-order scheme, so the sub-step
    count grows like 1/tol; checked at tol = 1e-6 against the exact exponential."""
    N = 24
    q, J, prop = propagators(N, 4)
    D = 1 << (N // 2)
    psi = inputs.gaussian_state(D, 22)
    h = B.syk_build_from_terms(N, q, J)
    o = {"krylov_dim": 2, "two_pass": 1, "tol": 1e-6}
    d = to_dev(torch, psi)
    st = B.syk_krylov_evolve(h, d, 0.05, 0.0, work(torch, B.syk_krylov_workspace_bytes(h, B.SYK_C128, o)), o)
    assert relerr(d.cpu().numpy(), prop.apply(0.05, psi)) <= 1e-6
    assert st["n_substeps"] > 1 and st["n_matvec"] == 3 * st["n_substeps"]


def test_krylov_one_pass_equals_two_pass_and_group_property(B, torch, propagators):
    """Pin P9: one-pass = two-pass to rounding; E(a)E(b) = E(a+b) incl. complex; round trip."""
    N = 20
    q, J, _ = propagators(N, 4)
    D = 1 << (N // 2)
    psi = inputs.gaussian_state(D, 33)
    h = B.syk_build_from_terms(N, q, J)
    o1, o2 = {"krylov_dim": 16}, {"krylov_dim": 16, "two_pass": 1}
    w1 = work(torch, B.syk_krylov_workspace_bytes(h, B.SYK_C128, o1))
    w2 = work(torch, B.syk_krylov_workspace_bytes(h, B.SYK_C128, o2))
    a, b = to_dev(torch, psi), to_dev(torch, psi)
    B.syk_krylov_evolve(h, a, 2.0, -0.5, w1, o1)
    B.syk_krylov_evolve(h, b, 2.0, -0.5, w2, o2)
    assert relerr(a.cpu().numpy(), b.cpu().numpy()) <= 1e-13
    c = to_dev(torch, psi)
    B.syk_krylov_evolve(h, c, 0.0, -0.5, w1, o1)
    B.syk_krylov_evolve(h, c, 2.0, 0.0, w1, o1)
    assert relerr(c.cpu().numpy(), a.cpu().numpy()) <= 1e-10     # single complex build = imaginary x real
    d = to_dev(torch, psi)
    B.syk_krylov_evolve(h, d, 5.0, 0.0, w1, o1)
    assert abs(float(torch.linalg.vector_norm(d)) - 1.0) <= 1e-11   # unitary
    B.syk_krylov_evolve(h, d, -5.0, 0.0, w1, o1)
    assert relerr(d.cpu().numpy(), psi) <= 1e-10                  # round trip


def test_krylov_closed_forms(B, torch):
    """Pin P8 on the GPU: single term (cos - i sin P), diagonal H, empty H, tau = 0."""
    N, D = 16, 256
    psi = inputs.gaussian_state(D, 5)
    # single term: H = J P with P^2 = 1
    qd, Jd = np.array([[1, 4, 6, 11]], dtype=np.int32), np.array([0.7])
    h = B.syk_build_from_terms(N, qd, Jd)
    P = ohm.matvec_sequential(N, qd, np.array([1.0]), psi)
    o = {"krylov_dim": 8}
    wk = work(torch, B.syk_krylov_workspace_bytes(h, B.SYK_C128, o))
    d = to_dev(torch, psi)
    st = B.syk_krylov_evolve(h, d, 2.5, 0.0, wk, o)
    ref = math.cos(2.5 * 0.7) * psi - 1j * math.sin(2.5 * 0.7) * P
    assert relerr(d.cpu().numpy(), ref) <= 1e-12
    assert st["krylov_dim_used"] == 2                              # happy breakdown after two steps
    # diagonal H: quartets (2a,2a+1,2b,2b+1) -> -J Z_a Z_b
    qz = np.array([[0, 1, 4, 5], [2, 3, 10, 11], [6, 7, 14, 15]], dtype=np.int32)
    Jz = np.array([0.3, -0.8, 0.5])
    h = B.syk_build_from_terms(N, qz, Jz)
    assert list(h.tables()["x"]) == [0]
    bidx = np.arange(D)
    zbit = lambda a: 1.0 - 2.0 * ((bidx >> a) & 1)
    diag = -(0.3 * zbit(0) * zbit(2) - 0.8 * zbit(1) * zbit(5) + 0.5 * zbit(3) * zbit(7))
    d = to_dev(torch, psi)
    B.syk_krylov_evolve(h, d, 1.0, -0.75, wk, o)
    assert relerr(d.cpu().numpy(), np.exp(-1j * (1.0 - 0.75j) * diag) * psi) <= 1e-11
    # empty H and tau = 0: identity
    h0 = B.syk_build_from_terms(N, np.zeros((0, 4), dtype=np.int32), np.zeros(0))
    d = to_dev(torch, psi)
    B.syk_krylov_evolve(h0, d, 3.0, -1.0, wk, o)
    assert np.array_equal(d.cpu().numpy(), psi)
    B.syk_krylov_evolve(h, d, 0.0, 0.0, wk, o)
    assert np.array_equal(d.cpu().numpy(), psi)


def test_krylov_argument_errors_and_host_entry(B, torch, propagators):
    N = 16
    q, J, prop = propagators(N, None)
    h = B.syk_build_from_terms(N, q, J)
    D = 256
    psi = inputs.gaussian_state(D, 6)
    d = to_dev(torch, psi)
    o = {"krylov_dim": 20}
    need = B.syk_krylov_workspace_bytes(h, B.SYK_C128, o)
    small = torch.empty(need - 16, dtype=torch.uint8, device="cuda")
    with pytest.raises(B.SykError) as e:
        B.syk_krylov_evolve(h, d, 1.0, 0.0, small, o)
    assert e.value.code == B.SYK_ENOMEM
    with pytest.raises(B.SykError):
        B.syk_krylov_evolve(h, d, float("nan"), 0.0, work(torch, need), o)
    with pytest.raises(B.SykError):
        B.syk_krylov_evolve(h, d, 1.0, 0.0, work(torch, need), {"krylov_dim": 1})
    # sub-step limit: result still written, soft error
    st = B.syk_krylov_evolve(h, d, 50.0, 0.0, work(torch, need), {"krylov_dim": 3, "max_substeps": 2, "tol": 1e-12},
                             allow_noconv=True)
    assert st["rc"] == B.SYK_ENOCONV and st["err_est"] > 1e-12
    # host entry point
    hp = psi.copy()
    B.syk_krylov_evolve_host(h, hp, 1.0, -0.5, work(torch, need + D * 16), o)
    assert relerr(hp, prop.apply(1.0 - 0.5j, psi)) <= 1e-10


# ------------------------------------------------------------------------------------------------------------
# a-5 OTOC
# ------------------------------------------------------------------------------------------------------------
def test_otoc_config0_vs_oracle(B, torch):
    """BASELINE configs[0]: N=16 dense, gamma_0 / gamma_1, beta = 5, t in [0,10] step 0.5, Krylov dim 20."""
    cfg = inputs.CONFIGS[0]
    N = cfg["N"]
    q, J = couplings(N, None, seed=cfg["seed"])
    D = 1 << (N // 2)
    psi = orng.random_state(N, cfg["seed"], 0)
    prop = oev.ExactPropagator(N, q, J)
    t_grid = np.array(cfg["t_grid"])
    ref = ootoc.otoc_same_psi(prop, N, cfg["i_W"], cfg["j_V"], cfg["beta"], t_grid, psi)
    h = B.syk_build_hamiltonian(N, 1.0, cfg["seed"], 0)
    o = {"krylov_dim": cfg["krylov_dim"]}
    wk = work(torch, B.syk_otoc_workspace_bytes(h, B.SYK_C128, o))
    scratch = work(torch, B.syk_reduce_scratch_bytes())
    d_psi = torch.empty(D, dtype=torch.complex128, device="cuda")
    B.syk_random_state(N, cfg["seed"], 0, d_psi, scratch)
    F, st = B.syk_otoc(h, cfg["i_W"], cfg["j_V"], cfg["beta"], t_grid, d_psi, wk, o)
    assert np.max(np.abs(F - ref)) / abs(ref[0]) <= 1e-10
    # (the same-psi F(0) is complex: conjugation exchanges W and V; only the exact trace is real -- pin P11)
    # two-pass and complex64 variants
    o2 = {"krylov_dim": cfg["krylov_dim"], "two_pass": 1}
    B.syk_random_state(N, cfg["seed"], 0, d_psi, scratch)
    F2, _ = B.syk_otoc(h, cfg["i_W"], cfg["j_V"], cfg["beta"], t_grid[:5], d_psi,
                       work(torch, B.syk_otoc_workspace_bytes(h, B.SYK_C128, o2)), o2)
    assert np.max(np.abs(F2 - ref[:5])) / abs(ref[0]) <= 1e-10
    psi32 = psi.astype(np.complex64)
    ref32 = ootoc.otoc_same_psi(prop, N, cfg["i_W"], cfg["j_V"], cfg["beta"], t_grid[:5], psi32.astype(np.complex128))
    F32, _ = B.syk_otoc(h, cfg["i_W"], cfg["j_V"], cfg["beta"], t_grid[:5], to_dev(torch, psi32),
                        work(torch, B.syk_otoc_workspace_bytes(h, B.SYK_C64, o)), o)
    assert np.max(np.abs(F32 - ref32)) / abs(ref32[0]) <= 1e-5


def test_otoc_closed_form_beta0_t0(B, torch):
    """Pin P11: beta = 0, t = 0 gives F = -s^4 for every psi, exactly (g_i g_j g_i g_j = -s^4)."""
    N = 20
    D = 1 << (N // 2)
    for gn, want in ((0, -1.0), (1, -0.25)):
        h = B.syk_build_hamiltonian(N, inputs.bernoulli_p(N, 4), 1, 0, gn)
        o = {"krylov_dim": 10}
        wk = work(torch, B.syk_otoc_workspace_bytes(h, B.SYK_C128, o))
        F, _ = B.syk_otoc(h, 19, 18, 0.0, [0.0], to_dev(torch, inputs.gaussian_state(D, 77)), wk, o)
        assert abs(F[0] - want) <= 1e-14


def test_otoc_batched_vs_oracle(B, torch):
    """Realizations batched on one GPU (configs[1] shape at reduced N): each against its own exact oracle."""
    N, nb = 16, 3
    D = 1 << (N // 2)
    p = inputs.bernoulli_p(N, 4)
    t_grid = np.array([0.0, 0.7, 2.0])
    hams = [B.syk_build_hamiltonian(N, p, 0, r) for r in range(nb)]
    psis = np.stack([orng.random_state(N, 0, r) for r in range(nb)])
    o = {"krylov_dim": 16}
    wk = work(torch, B.syk_otoc_workspace_bytes(hams[0], B.SYK_C128, o))
    F, st = B.syk_otoc_batched(hams, 15, 14, 5.0, t_grid, to_dev(torch, psis.reshape(-1)), D, wk, o)
    for r in range(nb):
        q, J, _ = orng.sample_couplings(N, p, 0, r)
        ref = ootoc.otoc_same_psi(oev.ExactPropagator(N, q, J), N, 15, 14, 5.0, t_grid, psis[r])
        assert np.max(np.abs(F[r] - ref)) / abs(ref[0]) <= 1e-10


def test_otoc_argument_errors(B, torch):
    h = B.syk_build_hamiltonian(16, 1.0, 0)
    o = {"krylov_dim": 8}
    wk = work(torch, B.syk_otoc_workspace_bytes(h, B.SYK_C128, o))
    psi = to_dev(torch, inputs.gaussian_state(256, 1))
    for args in ((3, 3, 1.0, [0.0]), (16, 0, 1.0, [0.0]), (0, 1, -1.0, [0.0]), (0, 1, 1.0, [1.0, 0.5])):
        with pytest.raises(B.SykError):
            B.syk_otoc(h, args[0], args[1], args[2], args[3], psi, wk, o)


# ------------------------------------------------------------------------------------------------------------
# NEXT-2 Green function
# ------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("dt", ["c128", "c64"])
def test_green_vs_oracle(B, torch, dt):
    """G(t) = <psi|e^{(it-b/2)H} g e^{-iHt} g e^{-bH/2}|psi> against the exact-diagonalisation oracle, N=16 dense
    (configs[0] Hamiltonian) and N=20 sparse; one-pass and two-pass."""
    for N, k, n, beta, o in ((16, None, 15, 5.0, {"krylov_dim": 20}), (20, 4, 3, 2.0, {"krylov_dim": 16, "two_pass": 1})):
        q, J = couplings(N, k, seed=0)
        D = 1 << (N // 2)
        psi = inputs.gaussian_state(D, 31, npdtype(dt))
        prop = oev.ExactPropagator(N, q, J)
        t_grid = np.array([0.0, 0.5, 1.0, 2.5, 2.5, 6.0])
        ref = ogreen.green_same_psi(prop, N, n, beta, t_grid, psi.astype(np.complex128))
        h = B.syk_build_from_terms(N, q, J)
        code = B.SYK_C128 if dt == "c128" else B.SYK_C64
        wk = work(torch, B.syk_otoc_workspace_bytes(h, code, o))
        G, st = B.syk_green(h, n, beta, t_grid, to_dev(torch, psi), wk, o)
        assert np.max(np.abs(G - ref)) / abs(ref[0]) <= TOL[dt], (N, dt)
        assert st["n_matvec"] > 0


def test_green_closed_form_and_errors(B, torch):
    """G(0) = s^2 <psi|e^{-bH}|psi>; beta = 0, t = 0 gives exactly s^2 for a normalised psi; argument errors."""
    N = 20
    D = 1 << (N // 2)
    psi = inputs.gaussian_state(D, 5)
    for gn, s2 in ((0, 1.0), (1, 0.5)):
        h = B.syk_build_hamiltonian(N, inputs.bernoulli_p(N, 4), 1, 0, gn)
        o = {"krylov_dim": 12}
        wk = work(torch, B.syk_otoc_workspace_bytes(h, B.SYK_C128, o))
        G, _ = B.syk_green(h, 7, 0.0, [0.0], to_dev(torch, psi), wk, o)
        assert abs(G[0] - s2) <= 1e-13
        d = to_dev(torch, psi)
        B.syk_krylov_evolve(h, d, 0.0, -0.75, wk, o)                        # e^{-bH/2} psi, b = 1.5
        n2 = float(torch.linalg.vector_norm(d).item()) ** 2
        G, _ = B.syk_green(h, 7, 1.5, [0.0], to_dev(torch, psi), wk, o)
        assert abs(G[0] - s2 * n2) <= 1e-12 * n2
    for bad in (dict(n=-1), dict(n=N), dict(beta=-1.0), dict(t=[1.0, 0.5])):
        with pytest.raises(B.SykError):
            B.syk_green(h, bad.get("n", 3), bad.get("beta", 1.0), bad.get("t", [0.0]), to_dev(torch, psi), wk, o)
    with pytest.raises(B.SykError):
        B.syk_green(h, 3, 1.0, [0.0], to_dev(torch, psi), work(torch, 1024), o)


# ------------------------------------------------------------------------------------------------------------
# NEXT-1 parity blocks (DESIGN.md R-BLOCK)
# ------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("dt", ["c128", "c64"])
def test_parity_block_apply_H_and_gamma(B, torch, dt):
    """apply_H on a block handle = oracle block matrix; gamma blocks (all n, both directions) = oracle blocks
    selected from the Kronecker matrices; large enough for the tile kernels (N=28 -> 2^13 amplitudes per block)."""
    from oracle import parity as opar
    for N, k in ((12, None), (28, 4)):
        L = N // 2
        q, J = couplings(N, k, seed=6)
        h = B.syk_build_from_terms(N, q, J)
        v = inputs.gaussian_state(1 << L, 55, npdtype(dt))
        for sector in (0, 1):
            hb = B.syk_build_parity_block(h, sector)
            vs = opar.restrict(v, L, sector)
            full = opar.embed(vs.astype(np.complex128), L, sector)
            ref = opar.restrict(ohm.matvec_sequential(N, q, J, full), L, sector)
            d_out = torch.empty(1 << (L - 1), dtype=tdtype(torch, dt), device="cuda")
            B.syk_apply_H(hb, to_dev(torch, vs), d_out)
            assert relerr(d_out.cpu().numpy(), ref) <= TOL[dt], (N, sector)
            for n in sorted({0, 1, 2, 7, N - 3, N - 2, N - 1}):
                gref = opar.restrict(ohm.apply_gamma(N, n, full), L, 1 - sector)
                d_g = torch.empty_like(d_out)
                B.syk_apply_gamma_block(N, n, 1 - sector, to_dev(torch, vs), d_g)
                assert relerr(d_g.cpu().numpy(), gref) <= (1e-15 if dt == "c128" else 1e-7), (N, n, sector)
                d_ip = to_dev(torch, vs)
                B.syk_apply_gamma_block(N, n, 1 - sector, d_ip, d_ip)           # in place
                assert torch.equal(torch.view_as_real(d_ip), torch.view_as_real(d_g))


@pytest.mark.parametrize("dt", ["c128", "c64"])
def test_parity_block_otoc_and_green(B, torch, dt):
    """Block OTOC / Green function against the oracle's block pipeline (dense block propagators and gamma blocks),
    and the sum over the two sectors against the full-space library calls ("+ swap UD")."""
    from oracle import parity as opar
    N, L = 16, 8
    q, J = couplings(N, None, seed=0)
    h = B.syk_build_from_terms(N, q, J)
    he, ho = B.syk_build_parity_block(h, 0), B.syk_build_parity_block(h, 1)
    props = [opar.BlockPropagator(N, q, J, s) for s in (0, 1)]
    psi = inputs.gaussian_state(1 << L, 8, npdtype(dt))
    t_grid = np.array([0.0, 0.5, 2.0, 4.5])
    o = {"krylov_dim": 20}
    code = B.SYK_C128 if dt == "c128" else B.SYK_C64
    wk = work(torch, B.syk_otoc_workspace_bytes(he, code, o))
    for (iW, jV) in ((N - 1, N - 2), (0, 1), (5, N - 1)):
        Fsum = 0
        for s in (0, 1):
            ps = opar.restrict(psi, L, s)
            ref = opar.otoc_block_same_psi(props, N, iW, jV, 5.0, t_grid, ps.astype(np.complex128), s)
            F, _ = B.syk_otoc_block(he, ho, s, iW, jV, 5.0, t_grid, to_dev(torch, ps), wk, o)
            assert np.max(np.abs(F - ref)) <= TOL[dt] * max(abs(ref[0]), 1e-3), (iW, jV, s)
            Fsum = Fsum + F
        wkf = work(torch, B.syk_otoc_workspace_bytes(h, code, o))
        Ffull, _ = B.syk_otoc(h, iW, jV, 5.0, t_grid, to_dev(torch, psi), wkf, o)
        assert np.max(np.abs(Fsum - Ffull)) <= 4 * TOL[dt] * abs(Ffull[0])
    Gsum = 0
    for s in (0, 1):
        ps = opar.restrict(psi, L, s)
        ref = opar.green_block_same_psi(props, N, N - 1, 2.0, t_grid, ps.astype(np.complex128), s)
        G, _ = B.syk_green_block(he, ho, s, N - 1, 2.0, t_grid, to_dev(torch, ps), wk, o)
        assert np.max(np.abs(G - ref)) <= TOL[dt] * abs(ref[0]), s
        Gsum = Gsum + G
    Gfull, _ = B.syk_green(h, N - 1, 2.0, t_grid, to_dev(torch, psi), work(torch, B.syk_otoc_workspace_bytes(h, code, o)), o)
    assert np.max(np.abs(Gsum - Gfull)) <= 4 * TOL[dt] * abs(Gfull[0])
    # argument errors: blocks swapped, full handle where a block is expected, block where a full handle is expected
    ps = to_dev(torch, opar.restrict(psi, L, 0))
    for bad in (lambda: B.syk_otoc_block(ho, he, 0, 1, 2, 1.0, [0.0], ps, wk, o),
                lambda: B.syk_otoc_block(h, h, 0, 1, 2, 1.0, [0.0], ps, wk, o),
                lambda: B.syk_otoc_block(he, ho, 2, 1, 2, 1.0, [0.0], ps, wk, o),
                lambda: B.syk_otoc_block(he, ho, 0, N, 2, 1.0, [0.0], ps, wk, o),
                lambda: B.syk_otoc(he, 1, 2, 1.0, [0.0], ps, wk, o),
                lambda: B.syk_green(he, 1, 1.0, [0.0], ps, wk, o)):
        with pytest.raises(B.SykError):
            bad()


# ------------------------------------------------------------------------------------------------------------
# NEXT-4 generic Pauli sums: spin chains through the same kernels
# ------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("dt", ["c128", "c64"])
def test_spin_chain_apply_and_evolve(B, torch, dt):
    """Heisenberg XYZ + transverse field on 14 spins: H.v with every kernel against the oracle's Kronecker-product
    matrix; exp(-i tau H) psi against dense diagonalisation (L = 10)."""
    from oracle import pauli as opauli
    L = 14
    terms = opauli.heisenberg_terms(L, 0.9, -0.6, 1.2, periodic=True) + opauli.transverse_ising_terms(L, 0.0, 0.45)
    h = B.syk_build_from_pauli_strings(L, terms)
    v = inputs.gaussian_state(1 << L, 77, npdtype(dt))
    # the oracle matrix is 2^14 x 2^14 dense = 4 GB: apply it string by string instead (same Kronecker definition,
    # one 2 x 2 factor at a time on the reshaped vector)
    ref = np.zeros(1 << L, dtype=np.complex128)
    for x, z, c in terms:
        w = v.astype(np.complex128).reshape([2] * L)              # axis 0 = top qubit
        for q in range(L):
            site = np.eye(2, dtype=np.complex128)
            if (z >> q) & 1:
                site = site @ opauli.SZ
            if (x >> q) & 1:
                site = site @ opauli.SX
            w = np.moveaxis(np.tensordot(site, w, axes=([1], [L - 1 - q])), 0, L - 1 - q)
        ref += c * w.reshape(-1)
    code = B.dtype_code(to_dev(torch, v))
    seen = set()
    for kind in (0, 1, 2, 3, 4):
        B.syk_set_apply_H_kernel(h, kind)
        got_kind = B.syk_apply_H_kernel_kind(h, code)
        seen.add(got_kind)
        d_out = torch.zeros(1 << L, dtype=tdtype(torch, dt), device="cuda")
        B.syk_apply_H(h, to_dev(torch, v), d_out)
        assert relerr(d_out.cpu().numpy(), ref) <= TOL[dt], kind
    assert seen == {0, 1, 2, 3, 4}
    L2 = 10
    terms2 = opauli.heisenberg_terms(L2, 0.9, -0.6, 1.2) + opauli.transverse_ising_terms(L2, 0.5, 0.45, periodic=False)
    H2 = opauli.sum_matrix(L2, terms2)
    assert np.allclose(H2, H2.conj().T, atol=0)
    w2, U2 = np.linalg.eigh(H2)
    h2 = B.syk_build_from_pauli_strings(L2, terms2)
    psi = inputs.gaussian_state(1 << L2, 78, npdtype(dt))
    o = {"krylov_dim": 24}
    wk = work(torch, B.syk_krylov_workspace_bytes(h2, code, o))
    for tau in (2.0 + 0j, -0.8j, 1.5 - 0.5j):
        d = to_dev(torch, psi)
        B.syk_krylov_evolve(h2, d, tau.real, tau.imag, wk, o)
        exact = U2 @ (np.exp(-1j * tau * w2) * (U2.conj().T @ psi.astype(np.complex128)))
        assert relerr(d.cpu().numpy(), exact) <= TOL[dt], tau
    with pytest.raises(B.SykError):
        B.syk_otoc(h2, 0, 1, 1.0, [0.0], to_dev(torch, psi), work(torch, B.syk_otoc_workspace_bytes(h2, code, o)), o)


# ------------------------------------------------------------------------------------------------------------
# lock-step batched realizations (BASELINE configs[1] shape)
# ------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("dt", ["c128", "c64"])
def test_krylov_evolve_batched_vs_exact(B, torch, dt):
    """grid.y = realization: five different sparse Hamiltonians (one of them a single term, which breaks down after
    two Lanczos steps while the others need sub-steps) evolved in lock step, padded batch stride, each against its
    own exact propagator; and against the one-by-one library call."""
    N, nb = 24, 5
    D = 1 << (N // 2)
    stride = D + 64
    code = B.SYK_C128 if dt == "c128" else B.SYK_C64
    qs, Js = [], []
    for r in range(nb):
        q, J = couplings(N, 4, seed=20 + r)
        if r == 2:
            q, J = q[:1], np.array([0.9])
        qs.append(q)
        Js.append(J)
    hams = [B.syk_build_from_terms(N, q, J) for q, J in zip(qs, Js)]
    psis = np.zeros((nb, stride), dtype=npdtype(dt))
    for r in range(nb):
        psis[r, :D] = (1.0 + 0.3 * r) * inputs.gaussian_state(D, 300 + r, npdtype(dt))
    psis[:, D:] = 7.0                                                    # padding must stay untouched
    o = {"krylov_dim": 10}
    wk = work(torch, B.syk_krylov_workspace_bytes_batched(hams[0], nb, code, o))
    for tau in ((6.0, 0.0), (1.5, -1.0)):
        d = to_dev(torch, psis.reshape(-1))
        st = B.syk_krylov_evolve_batched(hams, d, stride, tau[0], tau[1], wk, o)
        out = d.cpu().numpy().reshape(nb, stride)
        assert np.all(out[:, D:] == 7.0)
        assert st["n_substeps"] >= (2 if dt == "c128" else 1) and st["krylov_dim_used"] == 2   # single-term member: breakdown
        wk1 = work(torch, B.syk_krylov_workspace_bytes(hams[0], code, o))
        for r in range(nb):
            prop = oev.ExactPropagator(N, qs[r], Js[r])
            ref = prop.apply(complex(*tau), psis[r, :D].astype(np.complex128))
            assert relerr(out[r, :D], ref) <= TOL[dt], (r, tau)
            d1 = to_dev(torch, psis[r, :D].copy())
            B.syk_krylov_evolve(hams[r], d1, tau[0], tau[1], wk1, o)
            assert relerr(out[r, :D], d1.cpu().numpy()) <= TOL[dt]
    # conditions of the lock-step mode
    with pytest.raises(B.SykError):
        B.syk_krylov_evolve_batched(hams, d, stride, 1.0, 0.0, wk, {"krylov_dim": 10, "two_pass": 1})
    with pytest.raises(B.SykError):
        B.syk_krylov_evolve_batched(hams, d, D - 1, 1.0, 0.0, wk, o)
    with pytest.raises(B.SykError):
        B.syk_krylov_evolve_batched(hams, d, stride, 1.0, 0.0, work(torch, 4096), o)
    small = [B.syk_build_hamiltonian(12, 1.0, 0, r) for r in range(2)]       # vector smaller than a tile
    with pytest.raises(B.SykError):
        B.syk_krylov_evolve_batched(small, d, 64, 1.0, 0.0, wk, o)


@pytest.mark.parametrize("dt", ["c128", "c64"])
def test_otoc_batched_lockstep_vs_oracle(B, torch, dt):
    """syk_otoc_batched in lock-step mode (work space of syk_otoc_batched_workspace_bytes) at N=24: each realization
    against its own exact oracle, and against the back-to-back mode of the same call."""
    N, nb = 24, 4
    D = 1 << (N // 2)
    code = B.SYK_C128 if dt == "c128" else B.SYK_C64
    p = inputs.bernoulli_p(N, 4)
    t_grid = np.array([0.0, 0.6, 1.5, 1.5, 3.0])
    hams = [B.syk_build_hamiltonian(N, p, 0, r) for r in range(nb)]
    psis = np.stack([orng.random_state(N, 0, r) for r in range(nb)]).astype(npdtype(dt))
    o = {"krylov_dim": 14}
    wk = work(torch, B.syk_otoc_batched_workspace_bytes(hams[0], nb, code, o))
    n0 = B.syk_launch_count(reset=True)
    F, st = B.syk_otoc_batched(hams, N - 1, N - 2, 5.0, t_grid, to_dev(torch, psis.reshape(-1)), D, wk, o)
    n_lock = B.syk_launch_count(reset=True)
    wk1 = work(torch, B.syk_otoc_workspace_bytes(hams[0], code, o))
    F1, st1 = B.syk_otoc_batched(hams, N - 1, N - 2, 5.0, t_grid, to_dev(torch, psis.reshape(-1)), D, wk1, o)
    n_seq = B.syk_launch_count(reset=True)
    assert n_lock * 2 < n_seq                                             # the batch shares its launches
    for r in range(nb):
        q, J, _ = orng.sample_couplings(N, p, 0, r)
        ref = ootoc.otoc_same_psi(oev.ExactPropagator(N, q, J), N, N - 1, N - 2, 5.0, t_grid,
                                  psis[r].astype(np.complex128))
        assert np.max(np.abs(F[r] - ref)) / abs(ref[0]) <= TOL[dt], r
        assert np.max(np.abs(F[r] - F1[r])) / abs(ref[0]) <= 2 * TOL[dt], r


def test_otoc_run_and_sweep_scripts(B, torch):
    """The two user-facing drivers of the package run end to end (small sizes) and agree with direct library calls."""
    import json
    import os
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    out = subprocess.run([sys.executable, "-m", "paper_2311_00639_b200.otoc_run", "--N", "20", "--k", "4", "--tmax", "2",
                          "--nt", "3", "--krylov-dim", "12"], cwd=root, capture_output=True, text=True, check=True)
    d = json.loads(out.stdout.strip().splitlines()[-1])
    N = 20
    h = B.syk_build_hamiltonian(N, inputs.bernoulli_p(N, 4), 0, 0)
    scratch = work(torch, B.syk_reduce_scratch_bytes())
    psi = torch.empty(1 << (N // 2), dtype=torch.complex128, device="cuda")
    B.syk_random_state(N, 0, 0, psi, scratch)
    o = {"krylov_dim": 12}
    F, _ = B.syk_otoc(h, N - 1, N - 2, 5.0, np.linspace(0.0, 2.0, 3), psi, work(torch, B.syk_otoc_workspace_bytes(h, B.SYK_C128, o)), o)
    assert np.allclose(np.array(d["F_re"]) + 1j * np.array(d["F_im"]), F, atol=1e-12)
    assert abs(d["ratio_re"][0] - 1.0) < 1e-15 and d["n_matvec"] > 0
    outb = subprocess.run([sys.executable, "-m", "paper_2311_00639_b200.otoc_run", "--N", "20", "--k", "4", "--tmax", "1",
                           "--nt", "2", "--krylov-dim", "12", "--block", "--green"], cwd=root, capture_output=True,
                          text=True, check=True)
    db = json.loads(outb.stdout.strip().splitlines()[-1])
    assert db["parity_blocks"] and db["what"] == "green" and abs(db["ratio_re"][0] - 1.0) < 1e-15
    sw = subprocess.run([sys.executable, "-m", "paper_2311_00639_b200.sweep", "--quick"], cwd=root, capture_output=True,
                        text=True, check=True)
    assert "| (i) k=4 |" in sw.stdout and "Affine fit" in sw.stdout


# ------------------------------------------------------------------------------------------------------------
# NEXT-3 qubit relabelling (include/syk.h "Qubit layout of a handle")
# ------------------------------------------------------------------------------------------------------------
def _to_storage_index(idx, perm):
    """canonical basis index -> index in a vector stored in the layout perm (qubit q = index bit perm[q])"""
    idx = np.asarray(idx, dtype=np.uint64)
    out = np.zeros_like(idx)
    for q, b in enumerate(perm):
        out |= ((idx >> np.uint64(q)) & np.uint64(1)) << np.uint64(int(b))
    return out


@pytest.mark.parametrize("dt", ["c128", "c64"])
def test_qubit_layout_apply_gamma_state(B, torch, dt):
    """A relabelled handle computes the SAME operator on vectors stored in its layout: canonical vector -> device ->
    syk_permute_vector -> apply_H (every kernel kind) -> back = oracle H.v; likewise gamma_n (all n), the random state,
    the Lanczos coefficients and the host entry points.  Layouts: the optimiser's choice and a random permutation."""
    N = 28
    L = N // 2
    D = 1 << L
    q, J = couplings(N, 4, seed=11)
    v = inputs.gaussian_state(D, 61, npdtype(dt))
    ref = ohm.matvec_sequential(N, q, J, v.astype(np.complex128))
    code = B.SYK_C128 if dt == "c128" else B.SYK_C64
    h = B.syk_build_from_terms(N, q, J)
    canon = h.tables()
    wk = work(torch, B.syk_krylov_workspace_bytes(h, code, {"krylov_dim": 5}))
    a0, b0, _ = B.syk_lanczos_run(h, to_dev(torch, v), 5, wk)
    rng = np.random.default_rng(5)
    scratch = work(torch, B.syk_reduce_scratch_bytes())
    for which in ("optimised", "random", "random2"):
        if which == "optimised":                       # (at L = 14 the tile spans almost all qubits: may be the identity)
            perm = [int(x) for x in B.syk_ham_optimize_layout(h, code)["perm"]]
        else:
            perm = [int(x) for x in rng.permutation(L)]
            B.syk_ham_set_layout(h, perm)
            assert perm != list(range(L))
        assert all(np.array_equal(canon[k], h.tables()[k]) for k in ("x", "z", "group_off"))
        d_can = to_dev(torch, v)
        d_lay = torch.empty_like(d_can)
        B.syk_permute_vector(h, True, d_can, d_lay)
        # the permutation itself: stored[P(b)] = canonical[b]
        sidx = _to_storage_index(np.arange(D), perm).astype(np.int64)
        assert np.array_equal(d_lay.cpu().numpy()[sidx], v)
        for kind in (0, 1, 2, 3):
            B.syk_set_apply_H_kernel(h, kind)
            assert B.syk_apply_H_kernel_kind(h, code) == kind
            d_out = torch.full((D,), complex(float("nan"), float("nan")), dtype=tdtype(torch, dt), device="cuda")
            B.syk_apply_H(h, d_lay, d_out)
            d_back = torch.empty_like(d_out)
            B.syk_permute_vector(h, False, d_out, d_back)
            assert relerr(d_back.cpu().numpy(), ref) <= TOL[dt], (which, kind)
        B.syk_set_apply_H_kernel(h, -1)
        # gamma_n in the layout
        for n in (0, 1, 2, 9, N - 2, N - 1):
            d_g = torch.empty_like(d_lay)
            B.syk_apply_gamma_h(h, n, d_lay, d_g)
            d_back = torch.empty_like(d_g)
            B.syk_permute_vector(h, False, d_g, d_back)
            assert relerr(d_back.cpu().numpy(), ohm.apply_gamma(N, n, v.astype(np.complex128))) <= (1e-15 if dt == "c128" else 1e-7), n
        # the random state is the same physical state
        d_psi = torch.empty(D, dtype=tdtype(torch, dt), device="cuda")
        B.syk_random_state_h(h, 3, 1, d_psi, scratch)
        d_back = torch.empty_like(d_psi)
        B.syk_permute_vector(h, False, d_psi, d_back)
        assert relerr(d_back.cpu().numpy(), orng.random_state(N, 3, 1)) <= (1e-13 if dt == "c128" else 1e-7)
        # Lanczos coefficients do not depend on the basis
        a1, b1, _ = B.syk_lanczos_run(h, d_lay, 5, wk)
        tol = 1e-12 if dt == "c128" else 2e-5
        assert np.max(np.abs(a1 - a0)) <= tol and np.max(np.abs(b1 - b0)) <= tol
        # host entry points take canonical vectors
        out_h = np.zeros(D, dtype=npdtype(dt))
        B.syk_apply_H_host(h, v, out_h, work(torch, 2 * D * v.itemsize))
        assert relerr(out_h, ref) <= TOL[dt]
        o = {"krylov_dim": 8}
        hp = v.copy()
        B.syk_krylov_evolve_host(h, hp, 0.7, -0.2, work(torch, B.syk_krylov_workspace_bytes(h, code, o) + D * v.itemsize), o)
        ref_ev = oev.chebyshev_propagate(N, q, J, 0.7 - 0.2j, v.astype(np.complex128))
        assert relerr(hp, ref_ev) <= TOL[dt], which


@pytest.mark.parametrize("dt", ["c128", "c64"])
def test_qubit_layout_otoc_green_blocks(B, torch, dt):
    """OTOC and Green function through relabelled handles (full space and parity blocks that share one layout) against the
    oracle: F(t), G(t) do not depend on the basis when the state is the same physical state."""
    from oracle import parity as opar
    N, L = 20, 10
    p = inputs.bernoulli_p(N, 4)
    q, J, _ = orng.sample_couplings(N, p, 2, 0)
    prop = oev.ExactPropagator(N, q, J)
    psi = orng.random_state(N, 2, 0).astype(npdtype(dt))
    t_grid = np.array([0.0, 0.8, 2.0])
    code = B.SYK_C128 if dt == "c128" else B.SYK_C64
    o = {"krylov_dim": 16}
    scratch = work(torch, B.syk_reduce_scratch_bytes())
    h = B.syk_build_hamiltonian(N, p, 2, 0)
    perm = [3, 7, 0, 9, 1, 8, 2, 6, 5, 4]
    B.syk_ham_set_layout(h, perm)
    wk = work(torch, B.syk_otoc_workspace_bytes(h, code, o))
    d_psi = torch.empty(1 << L, dtype=tdtype(torch, dt), device="cuda")
    for (iW, jV) in ((N - 1, N - 2), (4, 13)):
        B.syk_random_state_h(h, 2, 0, d_psi, scratch)
        F, _ = B.syk_otoc(h, iW, jV, 5.0, t_grid, d_psi, wk, o)
        ref = ootoc.otoc_same_psi(prop, N, iW, jV, 5.0, t_grid, psi.astype(np.complex128))
        assert np.max(np.abs(F - ref)) / abs(ref[0]) <= TOL[dt], (iW, jV)
    B.syk_random_state_h(h, 2, 0, d_psi, scratch)
    G, _ = B.syk_green(h, 7, 2.0, t_grid, d_psi, wk, o)
    refG = ogreen.green_same_psi(prop, N, 7, 2.0, t_grid, psi.astype(np.complex128))
    assert np.max(np.abs(G - refG)) / abs(refG[0]) <= TOL[dt]
    # parity blocks: cut from the canonical Hamiltonian, then both blocks get the same layout on the L-1 kept qubits
    B.syk_ham_set_layout(h, None)
    he, ho = B.syk_build_parity_block(h, 0), B.syk_build_parity_block(h, 1)
    permb = [4, 0, 8, 2, 6, 1, 7, 3, 5]
    B.syk_ham_set_layout(he, permb)
    with pytest.raises(B.SykError):                      # blocks with different layouts are rejected
        B.syk_otoc_block(he, ho, 0, 1, 2, 1.0, [0.0], to_dev(torch, opar.restrict(psi, L, 0)), wk, o)
    B.syk_ham_set_layout(ho, permb)
    props = [opar.BlockPropagator(N, q, J, s) for s in (0, 1)]
    for s in (0, 1):
        ps = opar.restrict(psi, L, s)
        hb = he if s == 0 else ho
        d_can = to_dev(torch, ps)
        d_lay = torch.empty_like(d_can)
        B.syk_permute_vector(hb, True, d_can, d_lay)
        for (iW, jV) in ((N - 1, N - 2), (3, N - 1), (5, 8)):
            ref = opar.otoc_block_same_psi(props, N, iW, jV, 5.0, t_grid, ps.astype(np.complex128), s)
            F, _ = B.syk_otoc_block(he, ho, s, iW, jV, 5.0, t_grid, d_lay.clone(), wk, o)
            assert np.max(np.abs(F - ref)) <= TOL[dt] * max(abs(ref[0]), 1e-3), (s, iW, jV)
        refG = opar.green_block_same_psi(props, N, 6, 2.0, t_grid, ps.astype(np.complex128), s)
        G, _ = B.syk_green_block(he, ho, s, 6, 2.0, t_grid, d_lay.clone(), wk, o)
        assert np.max(np.abs(G - refG)) <= TOL[dt] * abs(refG[0])
        # gamma between blocks in the layout = oracle block of gamma
        full = opar.embed(ps.astype(np.complex128), L, s)
        for n in (0, 5, N - 3, N - 2, N - 1):
            gref = opar.restrict(ohm.apply_gamma(N, n, full), L, 1 - s)
            d_g = torch.empty_like(d_lay)
            B.syk_apply_gamma_block_h(hb, n, 1 - s, d_lay, d_g)
            d_back = torch.empty_like(d_g)
            B.syk_permute_vector(hb, False, d_g, d_back)
            assert relerr(d_back.cpu().numpy(), gref) <= (1e-15 if dt == "c128" else 1e-7), (s, n)


# ------------------------------------------------------------------------------------------------------------
# NEXT-4: non-Hermitian operators through Arnoldi (oracle/nonhermitian.py)
# ------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("dt", ["c128", "c64"])
def test_nonhermitian_syk_complex_couplings(B, torch, dt):
    """Non-Hermitian SYK (complex J) at N = 20: H.v with every kernel the handle can use against the dense matrix, and
    exp(-i tau H) psi by Arnoldi against the dense matrix exponential for real, imaginary and complex tau."""
    from oracle import nonhermitian as onh
    N = 20
    D = 1 << (N // 2)
    q, J = couplings(N, 4, seed=13)
    Jc = J * np.exp(1j * np.random.default_rng(2).uniform(0, 2 * np.pi, len(J)))
    H = onh.complex_syk_hamiltonian(N, q, Jc)
    assert np.linalg.norm(H - H.conj().T) > 0.1 * np.linalg.norm(H)
    h = B.syk_build_from_terms_complex(N, q, Jc)
    assert not B.syk_ham_is_hermitian(h)
    code = B.SYK_C128 if dt == "c128" else B.SYK_C64
    v = inputs.gaussian_state(D, 91, npdtype(dt))
    ref = H @ v.astype(np.complex128)
    seen = set()
    for kind in (0, 1, 2, 3, 4):
        B.syk_set_apply_H_kernel(h, kind)
        seen.add(B.syk_apply_H_kernel_kind(h, code))
        d_out = torch.full((D,), complex(float("nan"), float("nan")), dtype=tdtype(torch, dt), device="cuda")
        B.syk_apply_H(h, to_dev(torch, v), d_out)
        assert relerr(d_out.cpu().numpy(), ref) <= TOL[dt], kind
    # general complex coefficients: only the generic and the 16 KiB-tile kernels (the latter needs D >= one tile)
    assert seen == ({0, 1} if dt == "c128" else {0})
    B.syk_set_apply_H_kernel(h, -1)
    o = {"krylov_dim": 20}
    wk = work(torch, B.syk_krylov_workspace_bytes(h, code, o))
    for tau in (1.5 + 0j, -0.8j, 1.0 - 0.5j, -2.0 + 0.3j):
        d = to_dev(torch, v)
        st = B.syk_krylov_evolve(h, d, tau.real, tau.imag, wk, o)
        exact = onh.expm_propagate(H, tau, v)
        assert relerr(d.cpu().numpy(), exact) <= TOL[dt], (tau, st)
        assert st["n_matvec"] >= 2 and st["err_est"] <= TOL[dt]
    # norm carrying on the Arnoldi path: the vector keeps its norm, exp(log_norm) restores the result
    d = to_dev(torch, v)
    st = B.syk_krylov_evolve(h, d, 1.0, -2.5, wk, {"krylov_dim": 20, "renormalize": 1})
    got = d.cpu().numpy().astype(np.complex128)
    assert abs(np.linalg.norm(got) / np.linalg.norm(v) - 1.0) <= (1e-12 if dt == "c128" else 1e-5)
    assert relerr(got * math.exp(st["log_norm"]), onh.expm_propagate(H, 1.0 - 2.5j, v)) <= TOL[dt]
    # group law through the library itself
    a, b = to_dev(torch, v), to_dev(torch, v)
    B.syk_krylov_evolve(h, a, 0.4, -0.1, wk, o)
    B.syk_krylov_evolve(h, a, 0.6, 0.0, wk, o)
    B.syk_krylov_evolve(h, b, 1.0, -0.1, wk, o)
    assert relerr(a.cpu().numpy(), b.cpu().numpy()) <= 10 * TOL[dt]
    # what needs H = H^+ is refused
    with pytest.raises(B.SykError):
        B.syk_krylov_evolve(h, to_dev(torch, v), 1.0, 0.0, wk, {"krylov_dim": 20, "two_pass": 1})
    with pytest.raises(B.SykError):
        B.syk_lanczos_run(h, to_dev(torch, v), 4, wk)
    with pytest.raises(B.SykError):
        B.syk_otoc(h, 0, 1, 1.0, [0.0], to_dev(torch, v), work(torch, B.syk_otoc_workspace_bytes(h, code, o)), o)


@pytest.mark.parametrize("dt", ["c128", "c64"])
def test_nonhermitian_closed_form_and_spin_chain(B, torch, dt):
    """(i) one term with a complex coupling, H = J P, P^2 = 1: exp(-i tau H) = cos(tau J) - i sin(tau J) P with complex
    tau J; Arnoldi breaks down after two steps (exact).  (ii) a non-Hermitian spin chain (asymmetric hopping a la
    Hatano-Nelson + an imaginary field; every coefficient purely real or imaginary, so the tile kernels apply) on 10 and
    14 spins: H.v with every kernel against the string-by-string Kronecker action, exp(-i tau H) psi against expm."""
    import cmath
    from oracle import nonhermitian as onh
    from oracle import pauli as opauli
    code = B.SYK_C128 if dt == "c128" else B.SYK_C64
    N, D = 16, 256
    psi = inputs.gaussian_state(D, 5, npdtype(dt))
    qd, Jd = np.array([[1, 4, 6, 11]], dtype=np.int32), np.array([0.7 - 0.4j])
    h = B.syk_build_from_terms_complex(N, qd, Jd)
    P = ohm.matvec_sequential(N, qd, np.array([1.0]), psi.astype(np.complex128))
    o = {"krylov_dim": 8}
    wk = work(torch, B.syk_krylov_workspace_bytes(h, code, o))
    d = to_dev(torch, psi)
    st = B.syk_krylov_evolve(h, d, 2.5, -0.3, wk, o)
    zz = (2.5 - 0.3j) * Jd[0]
    ref = cmath.cos(zz) * psi.astype(np.complex128) - 1j * cmath.sin(zz) * P
    assert relerr(d.cpu().numpy(), ref) <= (1e-12 if dt == "c128" else 1e-5)
    assert st["krylov_dim_used"] == 2

    def chain(L, g):
        terms = []
        for i in range(L - 1):
            pair = (1 << i) | (1 << (i + 1))
            # (1+g) s+_i s-_{i+1} + (1-g) s-_i s+_{i+1} = (XX + YY)/2 + i g (YX - XY)/2 ... written as Z^z X^x strings:
            terms.append((pair, 0, 0.5))                     # X X / 2
            terms.append((pair, pair, -0.5))                 # Y Y / 2 = -(ZX)(ZX) / 2
            terms.append((pair, 1 << i, 0.5 * g))            # i g (Y_i X_j)/2 = i g (-i Z_i X_i) X_j / 2 = g/2 Z_i X_i X_j
            terms.append((pair, 1 << (i + 1), -0.5 * g))     # -i g (X_i Y_j)/2 = -g/2 X_i Z_j X_j
        for i in range(L):
            terms.append((0, 1 << i, 0.3j * (i % 3 - 1)))    # imaginary longitudinal field
        return terms

    L2 = 10
    t2 = chain(L2, 0.35)
    H2 = opauli.sum_matrix(L2, t2)
    assert np.linalg.norm(H2 - H2.conj().T) > 0.1
    h2 = B.syk_build_from_pauli_strings(L2, t2)
    assert not B.syk_ham_is_hermitian(h2)
    v2 = inputs.gaussian_state(1 << L2, 6, npdtype(dt))
    o2 = {"krylov_dim": 24}
    wk2 = work(torch, B.syk_krylov_workspace_bytes(h2, code, o2))
    for tau in (1.2 + 0j, 0.7 - 0.4j):
        d = to_dev(torch, v2)
        B.syk_krylov_evolve(h2, d, tau.real, tau.imag, wk2, o2)
        assert relerr(d.cpu().numpy(), onh.expm_propagate(H2, tau, v2)) <= TOL[dt], tau
    L3 = 14
    t3 = chain(L3, -0.6)
    h3 = B.syk_build_from_pauli_strings(L3, t3)
    v3 = inputs.gaussian_state(1 << L3, 7, npdtype(dt))
    ref3 = np.zeros(1 << L3, dtype=np.complex128)
    for x, z, c in t3:
        w = v3.astype(np.complex128).reshape([2] * L3)
        for qq in range(L3):
            site = np.eye(2, dtype=np.complex128)
            if (z >> qq) & 1:
                site = site @ opauli.SZ
            if (x >> qq) & 1:
                site = site @ opauli.SX
            w = np.moveaxis(np.tensordot(site, w, axes=([1], [L3 - 1 - qq])), 0, L3 - 1 - qq)
        ref3 += c * w.reshape(-1)
    seen = set()
    for kind in (0, 1, 2, 3, 4):
        B.syk_set_apply_H_kernel(h3, kind)
        seen.add(B.syk_apply_H_kernel_kind(h3, code))
        d_out = torch.zeros(1 << L3, dtype=tdtype(torch, dt), device="cuda")
        B.syk_apply_H(h3, to_dev(torch, v3), d_out)
        assert relerr(d_out.cpu().numpy(), ref3) <= TOL[dt], kind
    assert seen == {0, 1, 2, 3, 4}


# ------------------------------------------------------------------------------------------------------------
# norm carrying in imaginary time (syk_krylov_opts.renormalize / syk_stats.log_norm)
# ------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("dt", ["c128", "c64"])
def test_renormalize_evolve_and_otoc(B, torch, propagators, dt):
    """renormalize = 1: the returned vector keeps the norm of the input and exp(log_norm) x vector is the oracle's
    result (one-pass, two-pass, several sub-steps); OTOC and Green function are unchanged by it; and at a beta whose
    growth exp(beta |E_0|) leaves the fp32 range the complex64 pipeline still matches the oracle (PAPER.md:363 runs
    beta = 20 at N = 64 in single precision)."""
    N = 16
    q, J, prop = propagators(N, None)
    D = 1 << (N // 2)
    code = B.SYK_C128 if dt == "c128" else B.SYK_C64
    psi = (2.5 * inputs.gaussian_state(D, 17, npdtype(dt))).astype(npdtype(dt))
    h = B.syk_build_from_terms(N, q, J)
    for o in ({"krylov_dim": 20, "renormalize": 1}, {"krylov_dim": 6, "renormalize": 1, "two_pass": 1}):
        wk = work(torch, B.syk_krylov_workspace_bytes(h, code, o))
        for tau in ((0.0, -30.0), (2.0, -7.5), (3.0, 0.0)):
            d = to_dev(torch, psi)
            st = B.syk_krylov_evolve(h, d, tau[0], tau[1], wk, o)
            ref = prop.apply(complex(*tau), psi.astype(np.complex128))
            got = d.cpu().numpy().astype(np.complex128)
            assert abs(np.linalg.norm(got) / np.linalg.norm(psi) - 1.0) <= (1e-12 if dt == "c128" else 1e-5)
            assert relerr(got * math.exp(st["log_norm"]), ref) <= TOL[dt], (o, tau)
            assert abs(st["log_norm"] - math.log(np.linalg.norm(ref) / np.linalg.norm(psi))) <= (1e-10 if dt == "c128" else 1e-5)
    # OTOC / Green: same values with and without; large beta in complex64
    psi1 = orng.random_state(N, 0, 0).astype(npdtype(dt))
    t_grid = np.array([0.0, 1.0, 2.5])
    o0, o1 = {"krylov_dim": 20}, {"krylov_dim": 20, "renormalize": 1}
    wk = work(torch, B.syk_otoc_workspace_bytes(h, code, o1))
    ref = ootoc.otoc_same_psi(prop, N, 0, 1, 5.0, t_grid, psi1.astype(np.complex128))
    F1, st1 = B.syk_otoc(h, 0, 1, 5.0, t_grid, to_dev(torch, psi1), wk, o1)
    F0, _ = B.syk_otoc(h, 0, 1, 5.0, t_grid, to_dev(torch, psi1), wk, o0)
    assert np.max(np.abs(F1 - ref)) / abs(ref[0]) <= TOL[dt] and np.max(np.abs(F1 - F0)) / abs(ref[0]) <= 2 * TOL[dt]
    assert st1["log_norm"] != 0.0
    refG = ogreen.green_same_psi(prop, N, 3, 4.0, t_grid, psi1.astype(np.complex128))
    G1, _ = B.syk_green(h, 3, 4.0, t_grid, to_dev(torch, psi1), wk, o1)
    assert np.max(np.abs(G1 - refG)) / abs(refG[0]) <= TOL[dt]
    beta = 200.0                                             # exp(beta |E_0|) ~ 1e60 and more: beyond fp32
    E0 = prop.eigenvalues()[0]
    assert beta * abs(E0) > 130.0
    refB = ootoc.otoc_same_psi(prop, N, 0, 1, beta, t_grid, psi1.astype(np.complex128))
    FB, _ = B.syk_otoc(h, 0, 1, beta, t_grid, to_dev(torch, psi1), wk, o1)
    assert np.all(np.isfinite(FB))
    assert np.max(np.abs(FB - refB)) / abs(refB[0]) <= (1e-9 if dt == "c128" else 5e-5), np.abs(FB - refB) / abs(refB[0])
    if dt == "c64":                                          # without norm carrying the same call leaves the fp32 range
        Fplain, _ = B.syk_otoc(h, 0, 1, beta, t_grid, to_dev(torch, psi1), wk, o0)
        assert not np.all(np.isfinite(Fplain)) or np.max(np.abs(Fplain - refB)) / abs(refB[0]) > 1e-3


def test_cuda_graph_latency_path(B, torch):
    """The Krylov driver replays one captured CUDA graph per Lanczos round for small vectors (syk_set_cuda_graphs): bitwise
    the same results as direct launches (one-pass, two-pass, OTOC over several buffers and handles), same kernel count,
    and the graph survives a change of layout / kernel choice of the handle (new key)."""
    N = 16
    D = 256
    q, J = couplings(N, None)
    psi = inputs.gaussian_state(D, 4)
    t_grid = np.array([0.0, 0.5, 1.5, 3.0])
    outs = {}
    for on in (1, 0, 1):
        B.syk_set_cuda_graphs(on)
        try:
            h = B.syk_build_from_terms(N, q, J)
            res = []
            for o in ({"krylov_dim": 12}, {"krylov_dim": 7, "two_pass": 1}):
                wk = work(torch, B.syk_otoc_workspace_bytes(h, B.SYK_C128, o))
                d = to_dev(torch, psi)
                B.syk_launch_count(reset=True)
                st = B.syk_krylov_evolve(h, d, 3.0, -1.0, wk, o)
                n_k = B.syk_launch_count(reset=True)
                res.append((d.cpu().numpy().copy(), st["n_matvec"], st["n_substeps"], n_k))
                F, _ = B.syk_otoc(h, 0, 1, 5.0, t_grid, to_dev(torch, psi), wk, o)
                res.append(F.copy())
                B.syk_set_apply_H_kernel(h, 0)                       # another kernel for the same handle: a new graph
                d2 = to_dev(torch, psi)
                B.syk_krylov_evolve(h, d2, 3.0, -1.0, wk, o)
                B.syk_set_apply_H_kernel(h, -1)
                res.append(d2.cpu().numpy().copy())
            outs.setdefault(on, []).append(res)
        finally:
            B.syk_set_cuda_graphs(1)
    ref = outs[0][0]
    for res in outs[1]:
        for a, b in zip(res, ref):
            if isinstance(a, tuple):
                assert np.array_equal(a[0], b[0]) and a[1:] == b[1:]
            else:
                assert np.array_equal(a, b)
    prop = oev.ExactPropagator(N, q, J)
    assert relerr(ref[0][0], prop.apply(3.0 - 1.0j, psi)) <= 1e-10


def test_no_device_allocation_after_prepare(B, torch):
    """include/syk.h: after syk_ham_prepare no compute call on the handle allocates device memory (the
    memory discipline is part of the method).  cudaMemGetInfo (which sees the library's own cudaMalloc calls) must not move
    across apply_H / Lanczos / Krylov / OTOC calls, for a sparse handle (tile kernels), a dense handle in the split form of
    the dense-table kernel (scratch of partial sums) and a relabelled handle; an UNPREPARED dense handle does allocate in
    its first call, which is what the check is able to see.  (CUDA graphs of the latency path off: instantiating a graph
    is the driver's allocation.)"""
    B.syk_set_cuda_graphs(0)
    try:
        N = 28
        D = 1 << (N // 2)
        o = {"krylov_dim": 6}
        psi = inputs.gaussian_state(D, 3)
        cases = []
        q, J = couplings(N, 4, seed=3)
        cases.append(("sparse", B.syk_build_from_terms(N, q, J)))
        hr = B.syk_build_from_terms(N, q, J)
        B.syk_ham_set_layout(hr, list(range(N // 2 - 1, -1, -1)))
        cases.append(("relabelled", hr))
        qd, Jd = couplings(N, None, seed=3)
        cases.append(("dense", B.syk_build_from_terms(N, qd, Jd)))
        for name, h in cases:
            wk = work(torch, B.syk_otoc_workspace_bytes(h, B.SYK_C128, o))
            d_in, d_out = to_dev(torch, psi), torch.empty(D, dtype=torch.complex128, device="cuda")
            B.syk_ham_prepare(h, B.SYK_C128)
            if name == "dense":
                assert B.syk_apply_H_kernel_kind(h, B.SYK_C128) == 4 and B.syk_apply_H_dense_info(h, B.SYK_C128)["split"] > 1
            torch.cuda.synchronize()
            free0 = torch.cuda.mem_get_info()[0]
            B.syk_apply_H(h, d_in, d_out)
            B.syk_lanczos_run(h, d_in, 4, wk)
            B.syk_krylov_evolve(h, d_in, 0.3, -0.1, wk, o)
            B.syk_otoc(h, 0, 1, 1.0, [0.0, 0.2], d_in, wk, o)
            torch.cuda.synchronize()
            assert torch.cuda.mem_get_info()[0] == free0, name
        hd = B.syk_build_from_terms(N, qd, Jd)                      # not prepared: the first call creates the tables + scratch
        d_in, d_out = to_dev(torch, psi), torch.empty(D, dtype=torch.complex128, device="cuda")
        torch.cuda.synchronize()
        free0 = torch.cuda.mem_get_info()[0]
        B.syk_apply_H(hd, d_in, d_out)
        torch.cuda.synchronize()
        assert torch.cuda.mem_get_info()[0] < free0
    finally:
        B.syk_set_cuda_graphs(1)


@pytest.mark.parametrize("dt", ["c128", "c64"])
def test_green_batched_vs_oracle(B, torch, dt):
    """syk_green_batched in lock-step mode and back to back: each realization against its own oracle."""
    N, nb = 24, 3
    D = 1 << (N // 2)
    code = B.SYK_C128 if dt == "c128" else B.SYK_C64
    p = inputs.bernoulli_p(N, 4)
    t_grid = np.array([0.0, 0.7, 2.0])
    hams = [B.syk_build_hamiltonian(N, p, 3, r) for r in range(nb)]
    psis = np.stack([orng.random_state(N, 3, r) for r in range(nb)]).astype(npdtype(dt))
    o = {"krylov_dim": 14}
    wk = work(torch, B.syk_otoc_batched_workspace_bytes(hams[0], nb, code, o))
    B.syk_launch_count(reset=True)
    G, _ = B.syk_green_batched(hams, 5, 3.0, t_grid, to_dev(torch, psis.reshape(-1)), D, wk, o)
    n_lock = B.syk_launch_count(reset=True)
    wk1 = work(torch, B.syk_otoc_workspace_bytes(hams[0], code, o))
    G1, _ = B.syk_green_batched(hams, 5, 3.0, t_grid, to_dev(torch, psis.reshape(-1)), D, wk1, o)
    n_seq = B.syk_launch_count(reset=True)
    assert n_lock * 2 < n_seq
    for r in range(nb):
        q, J, _ = orng.sample_couplings(N, p, 3, r)
        ref = ogreen.green_same_psi(oev.ExactPropagator(N, q, J), N, 5, 3.0, t_grid, psis[r].astype(np.complex128))
        assert np.max(np.abs(G[r] - ref)) / abs(ref[0]) <= TOL[dt], r
        assert np.max(np.abs(G1[r] - ref)) / abs(ref[0]) <= TOL[dt], r
    with pytest.raises(B.SykError):
        B.syk_green_batched(hams, N, 3.0, t_grid, to_dev(torch, psis.reshape(-1)), D, wk, o)


# ------------------------------------------------------------------------------------------------------------
# diagnostic: syk_apply_H_trace (timeline of one persistent CTA of the scatter-tile kernel)
# ------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("dt", ["c128", "c64"])
def test_apply_H_trace_matches_apply_H(B, torch, dt):
    """The traced launch is the plain scatter-tile product (vs the oracle, and bitwise equal to syk_apply_H); its clock
    stamps are ordered (issue <= got, asked <= got, chunks in list order) and its load list is the layout's."""
    N = 30
    code = B.SYK_C128 if dt == "c128" else B.SYK_C64
    q, J = couplings(N, 4, seed=5)
    h = B.syk_build_from_terms(N, q, J)
    B.syk_set_apply_H_kernel(h, 3)
    assert B.syk_apply_H_kernel_kind(h, code) == 3
    rs = np.random.default_rng(11)
    v = (rs.standard_normal(1 << (N // 2)) + 1j * rs.standard_normal(1 << (N // 2))).astype(npdtype(dt))
    d_in = to_dev(torch, v)
    d_ref, d_out = torch.empty_like(d_in), torch.empty_like(d_in)
    B.syk_apply_H(h, d_in, d_ref)
    lay = B.syk_apply_H_layout(h, code)
    n_tiles = (1 << (N // 2)) >> bin(lay["tile_mask"]).count("1")
    for cta in (0, n_tiles - 1):
        d_out.fill_(float("nan"))
        tr = B.syk_apply_H_trace(h, d_in, d_out, cta=cta, round=0)
        assert torch.equal(d_out, d_ref)
        assert tr["n_loads"] == lay["n_loads"] and tr["rot"] == 0
        assert int(tr["load_terms"].sum()) == len(J) and (tr["load_terms"] >= 1).all()
        assert (tr["issue"] > 0).all() and (tr["after_wait"] >= tr["before_wait"]).all()
        assert (tr["after_wait"] >= tr["issue"]).all()
        assert (np.diff(tr["before_wait"]) > 0).all() and (np.diff(tr["issue"]) > 0).all()
        assert not tr["first_decoded"].any()                                  # three-stamp build
        tr7 = B.syk_apply_H_trace(h, d_in, d_out, cta=cta, round=0, detail=1)    # seven stamps, in order within a chunk
        assert torch.equal(d_out, d_ref)
        for a, b in (("after_wait", "first_decoded"), ("first_decoded", "first_issued"), ("first_issued", "all_issued"),
                     ("all_issued", "arrived")):
            assert (tr7[b] >= tr7[a]).all() and (tr7[a] > 0).all(), (a, b)
    ref = ohm.matvec_sequential(N, q, J, v.astype(np.complex128))
    assert relerr(d_out.cpu().numpy(), ref) <= TOL[dt]
    # a CTA / round that does not exist, a handle on another kernel
    with pytest.raises(B.SykError):
        B.syk_apply_H_trace(h, d_in, d_out, cta=n_tiles, round=0)
    with pytest.raises(B.SykError):
        B.syk_apply_H_trace(h, d_in, d_out, cta=0, round=1)
    B.syk_set_apply_H_kernel(h, 1)
    with pytest.raises(B.SykError):
        B.syk_apply_H_trace(h, d_in, d_out)


# ------------------------------------------------------------------------------------------------------------
# dense-table kernel: x-local groups (one table of 2^popcount(x) values per X-mask)
# ------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("dt", ["c128", "c64"])
def test_dense_local_groups_canonical_and_relabelled(B, torch, dt):
    """Dense p = 1 (Algorithm 1): every four-qubit X-mask is an x-local group (its 16 terms
    differ in Z only on the flipped qubits), C(L,4) of them; two-qubit and diagonal masks are not.  apply_H against the
    oracle in the canonical layout and with the qubits relabelled (the criterion is invariant under a permutation of bits);
    a mixed Hamiltonian (dense on 12 Majoranas + sparse rest) has local and term-by-term groups in one chunk."""
    from math import comb
    code = B.SYK_C128 if dt == "c128" else B.SYK_C64
    rs = np.random.default_rng(21)
    for N in (24, 26):
        L, D = N // 2, 1 << (N // 2)
        q, J, _ = orng.sample_couplings(N, 1.0, 2, 0)
        v = (rs.standard_normal(D) + 1j * rs.standard_normal(D)).astype(npdtype(dt))
        ref = ohm.matvec_sequential(N, q, J, v.astype(np.complex128))
        for perm in (None, rs.permutation(L)):
            h = B.syk_build_from_terms(N, q, J)
            if perm is not None:
                B.syk_ham_set_layout(h, perm)
            assert B.syk_apply_H_kernel_kind(h, code) == 4
            assert B.syk_apply_H_dense_info(h, code)["n_local_groups"] == comb(L, 4)
            d_can = to_dev(torch, v)
            d_in, d_out, d_back = torch.empty_like(d_can), torch.empty_like(d_can), torch.empty_like(d_can)
            B.syk_permute_vector(h, True, d_can, d_in)
            d_out.fill_(float("nan"))
            B.syk_apply_H(h, d_in, d_out)
            B.syk_permute_vector(h, False, d_out, d_back)
            assert relerr(d_back.cpu().numpy(), ref) <= TOL[dt], (N, perm)
    # mixed: all quartets on Majoranas 0..11 plus sparse quartets elsewhere; kind 4 forced
    N, D = 28, 1 << 14
    import itertools
    qd = np.array(list(itertools.combinations(range(12), 4)), dtype=np.int32)
    qs, Js = couplings(N, 4, seed=9)
    qs = np.array([t for t in qs if max(t) >= 12], dtype=np.int32)
    Js = Js[: len(qs)]
    q = np.concatenate([qd, qs])
    J = np.concatenate([rs.standard_normal(len(qd)) * 0.1, Js])
    h = B.syk_build_from_terms(N, q, J)
    B.syk_set_apply_H_kernel(h, 4)
    assert B.syk_apply_H_kernel_kind(h, code) == 4
    assert B.syk_apply_H_dense_info(h, code)["n_local_groups"] == comb(6, 4)
    v = (rs.standard_normal(D) + 1j * rs.standard_normal(D)).astype(npdtype(dt))
    d_in = to_dev(torch, v)
    d_out = torch.empty_like(d_in)
    B.syk_apply_H(h, d_in, d_out)
    assert relerr(d_out.cpu().numpy(), ohm.matvec_sequential(N, q, J, v.astype(np.complex128))) <= TOL[dt]


@pytest.mark.parametrize("dt", ["c128", "c64"])
def test_dense_local_groups_generic_pauli_strings(B, torch, dt):
    """x-local groups beyond what SYK produces (generic Pauli sums): X-masks of 1, 2, 3 and 4 qubits placed on
    thread bits, on the per-thread index bits 9..11 and above the 4096-amplitude tile, all or some of the 2^k Z-patterns on the
    flipped qubits, one common Z-pattern elsewhere, real and imaginary coefficients in one group.  Groups with >= 4 terms go
    through the table lookup, the others through the term-by-term walk; apply_H against the oracle's factor-by-factor
    application of every string (oracle.pauli.apply_sum)."""
    from oracle import pauli as opauli
    code = B.SYK_C128 if dt == "c128" else B.SYK_C64
    L, D = 14, 1 << 14
    rs = np.random.default_rng(33)
    masks = [0b1 << 3, 0b1 << 10, 0b1 << 13,                                            # one qubit (2 terms: walked)
             (1 << 2) | (1 << 7), (1 << 5) | (1 << 9), (1 << 11) | (1 << 12), (1 << 10) | (1 << 11),
             (1 << 0) | (1 << 4) | (1 << 8), (1 << 6) | (1 << 9) | (1 << 13), (1 << 9) | (1 << 10) | (1 << 11),
             (1 << 1) | (1 << 3) | (1 << 5) | (1 << 7), (1 << 8) | (1 << 9) | (1 << 12) | (1 << 13),
             (1 << 2) | (1 << 10) | (1 << 11) | (1 << 12), (1 << 9) | (1 << 10) | (1 << 11) | (1 << 13)]
    terms, n_local = [], 0
    for gi, x in enumerate(masks):
        bits = [q for q in range(L) if (x >> q) & 1]
        z_out = int(rs.integers(0, D)) & ~x
        pats = list(range(1 << len(bits)))
        if gi % 3 == 1 and len(pats) > 4:
            pats = sorted(rs.choice(pats, size=len(pats) - 3, replace=False).tolist())   # an incomplete set of Z-patterns
        if len(pats) >= 4:
            n_local += 1
        for pz in pats:
            z = z_out | sum(1 << bits[j] for j in range(len(bits)) if (pz >> j) & 1)
            a = float(rs.standard_normal())
            terms.append((x, z, a * (1j if rs.integers(0, 2) else 1.0)))
    # a second group on an X-mask of the list whose Z-patterns differ OUTSIDE x: not local, must be walked
    x = masks[4]
    for _ in range(6):
        terms.append((x | (1 << 1), int(rs.integers(0, D)), float(rs.standard_normal())))
    h = B.syk_build_from_pauli_strings(L, terms)
    B.syk_set_apply_H_kernel(h, 4)
    assert B.syk_apply_H_kernel_kind(h, code) == 4
    assert B.syk_apply_H_dense_info(h, code)["n_local_groups"] == n_local
    v = (rs.standard_normal(D) + 1j * rs.standard_normal(D)).astype(npdtype(dt))
    d_in = to_dev(torch, v)
    d_out = torch.full((D,), complex(float("nan"), float("nan")), dtype=d_in.dtype, device="cuda")
    B.syk_apply_H(h, d_in, d_out)
    ref = opauli.apply_sum(L, terms, v.astype(np.complex128))
    assert relerr(d_out.cpu().numpy(), ref) <= TOL[dt]
    # the same operator term by term (generic kernel): the two CUDA paths agree as well
    B.syk_set_apply_H_kernel(h, 0)
    d_gen = torch.empty_like(d_out)
    B.syk_apply_H(h, d_in, d_gen)
    assert relerr(d_gen.cpu().numpy(), ref) <= TOL[dt]
