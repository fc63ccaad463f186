"""Parity at BASELINE.json's full sizes (N=56 complex128, N=64 complex64), in the launch configuration bench.py
times.  No oracle can hold these vectors, so outputs are checked (i) on sampled indices b, each evaluated one by
one by the oracle from rows of the term matrices (pin P13: out[b] = sum_t H[b, col_t] in[col_t], the inputs
fetched from the device at the oracle's column indices), and (ii) through properties that hold at any size
(pins P2, P3): Hermiticity, exact parity-sector zeros, the second-moment sum rule.
"""
import numpy as np
import pytest

from oracle import hamiltonian as ohm
from oracle import rng as orng
from paper_2311_00639_b200 import inputs

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def B():
    import torch
    assert torch.cuda.is_available()
    from paper_2311_00639_b200 import binding
    return binding


def _free_gb():
    import torch
    free, _ = torch.cuda.mem_get_info()
    return free / 2 ** 30


def _storage_index(idx, perm):
    """canonical basis index -> index in a vector stored in the qubit layout perm (None = canonical)"""
    idx = np.asarray(idx, dtype=np.uint64)
    if perm is None:
        return idx
    out = np.zeros_like(idx)
    for q, b in enumerate(perm):
        out |= ((idx >> np.uint64(q)) & np.uint64(1)) << np.uint64(int(b))
    return out


def _oracle_samples(N, q, J, idx, d_in, perm=None):
    """out[b] for b in idx (canonical indices) by the oracle's monomial rows; in[col] is read back from the device
    (through the qubit layout `perm` of the handle, if any)."""
    import torch
    cols, vals = ohm.hamiltonian_rows(N, q, J, idx)                      # [T, n] each
    flat = torch.from_numpy(_storage_index(cols.reshape(-1), perm).astype(np.int64)).cuda()
    src = d_in[flat].cpu().numpy().astype(np.complex128).reshape(cols.shape)
    return (vals * src).sum(axis=0)


def _fullsize_case(B, N, k, tdt, tol, n_samples, relabel=False):
    import torch
    D = 1 << (N // 2)
    p = inputs.bernoulli_p(N, k)
    q, J, _ = orng.sample_couplings(N, p, 0, 0)
    h = B.syk_build_hamiltonian(N, p, 0, 0)
    assert h.info()["n_terms"] == len(J)
    code = B.SYK_C128 if tdt == torch.complex128 else B.SYK_C64
    perm = None
    if relabel:                                                           # the configuration bench.py times (NEXT-3)
        loads0 = B.syk_apply_H_layout(h, code)["n_loads"]
        perm = list(B.syk_ham_optimize_layout(h, code)["perm"])
        assert B.syk_apply_H_layout(h, code)["n_loads"] < loads0
    assert B.syk_apply_H_kernel_kind(h, code) == 3                        # the kernel bench.py times
    scratch = torch.empty(B.syk_reduce_scratch_bytes(), dtype=torch.uint8, device="cuda")
    d_in = torch.empty(D, dtype=tdt, device="cuda")
    d_out = torch.empty(D, dtype=tdt, device="cuda")
    B.syk_random_state_h(h, 0, 0, d_in, scratch)
    # (i) sampled outputs, including the first/last amplitude and the first/last tiles of the vector (16 KiB and
    #     64 / 128 KiB tiles), for all three TMA kernels; the default (scatter-tile) kernel runs last and feeds (ii)
    idx = inputs.sample_indices(D, n_samples, seed=17)
    edge = np.array([1, 1023, 1024, 4095, 4096, 8191, 8192, D // 2 - 1, D // 2, D - 8192, D - 4097, D - 1024, D - 2],
                    dtype=np.uint64)
    idx = np.unique(np.concatenate([idx, edge]))
    if relabel:                                                           # the same edges in the STORED vector as well
        inv = np.argsort(np.array(perm))                                  # index bit j holds qubit inv[j]
        idx = np.unique(np.concatenate([idx, _storage_index(edge, inv)]))
    ref = _oracle_samples(N, q, J, idx, d_in, perm)
    sidx = torch.from_numpy(_storage_index(idx, perm).astype(np.int64)).cuda()
    scale = np.sqrt(np.mean(np.abs(ref) ** 2))
    for kind in (1, 2, 3):
        B.syk_set_apply_H_kernel(h, kind)
        assert B.syk_apply_H_kernel_kind(h, code) == kind
        d_out.zero_()
        B.syk_apply_H(h, d_in, d_out)
        torch.cuda.synchronize()
        got = d_out[sidx].cpu().numpy().astype(np.complex128)
        assert np.max(np.abs(got - ref)) <= tol * scale * 10, (kind, float(np.max(np.abs(got - ref)) / scale))
        assert np.linalg.norm(got - ref) / np.linalg.norm(ref) <= tol, kind
    B.syk_set_apply_H_kernel(h, -1)
    # (ii) sum rule: |H psi|^2 = <psi|H^2|psi> ~ Tr H^2 / D = sum J^2 (s = 1), fluctuation O(D^-1/2)
    n2 = B.syk_dot(N, d_out, d_out, scratch).real
    assert abs(n2 / float(np.sum(J ** 2)) - 1.0) <= 5e-3
    alpha = B.syk_dot(N, d_in, d_out, scratch)
    assert abs(alpha.imag) <= (1e-12 if code == B.SYK_C128 else 1e-6)    # <psi|H|psi> real
    return h, d_in, d_out, scratch


def test_apply_H_N56_c128_sampled(B):
    """BASELINE configs[3]: N=56, k=4, complex128 (2 x 4.3 GB)."""
    import torch
    if _free_gb() < 12:
        pytest.skip("needs 12 GB of device memory")
    _fullsize_case(B, 56, 4, torch.complex128, 1e-10, 800, relabel=True)   # relabelled handle (what bench.py times)
    torch.cuda.empty_cache()
    h, d_in, d_out, scratch = _fullsize_case(B, 56, 4, torch.complex128, 1e-10, 1500)
    # parity sectors: zero the odd-popcount amplitudes of the input -> odd-popcount outputs are EXACTLY zero
    D = d_in.numel()
    step = 1 << 24
    for lo in range(0, D, step):
        b = torch.arange(lo, lo + step, device="cuda", dtype=torch.int64)
        par = b ^ (b >> 16)
        par = par ^ (par >> 8)
        par = par ^ (par >> 4)
        par = par ^ (par >> 2)
        par = (par ^ (par >> 1)) & 1
        d_in[lo:lo + step] = torch.where(par == 0, d_in[lo:lo + step], torch.zeros((), dtype=d_in.dtype, device="cuda"))
        del b
    B.syk_apply_H(h, d_in, d_out)
    worst = 0.0
    for lo in range(0, D, step):
        b = torch.arange(lo, lo + step, device="cuda", dtype=torch.int64)
        par = b ^ (b >> 16)
        par = par ^ (par >> 8)
        par = par ^ (par >> 4)
        par = par ^ (par >> 2)
        par = (par ^ (par >> 1)) & 1
        worst = max(worst, float((d_out[lo:lo + step].abs() * par).max()))
    assert worst == 0.0


def test_apply_H_N64_c64_sampled(B):
    """BASELINE configs[4]: N=64, k=2, complex64 (2 x 34.4 GB): 64-bit indexing end to end."""
    import torch
    if _free_gb() < 72:
        pytest.skip("needs 72 GB of device memory")
    _fullsize_case(B, 64, 2, torch.complex64, 1e-5, 1500)
    torch.cuda.empty_cache()
    _fullsize_case(B, 64, 2, torch.complex64, 1e-5, 800, relabel=True)


def test_lanczos_step_N56_hermiticity(B):
    """Fused Lanczos steps at N=56 (the configuration bench.py times): alpha_1 = <v|H|v> and
    beta_2^2 = <v|H^2|v> - alpha_1^2 with both right-hand sides from separate apply_H + dot calls."""
    import torch
    if _free_gb() < 24:
        pytest.skip("needs 24 GB of device memory")
    N = 56
    D = 1 << 28
    h = B.syk_build_hamiltonian(N, inputs.bernoulli_p(N, 4), 0, 0)
    m = 2
    wk = torch.empty(B.syk_krylov_workspace_bytes(h, B.SYK_C128, {"krylov_dim": m}), dtype=torch.uint8, device="cuda")
    scratch = torch.empty(B.syk_reduce_scratch_bytes(), dtype=torch.uint8, device="cuda")
    psi = torch.empty(D, dtype=torch.complex128, device="cuda")
    B.syk_random_state(N, 0, 1, psi, scratch)
    alpha, beta, st = B.syk_lanczos_run(h, psi, m, wk)
    Hpsi = torch.empty_like(psi)
    B.syk_apply_H(h, psi, Hpsi)
    a1 = B.syk_dot(N, psi, Hpsi, scratch).real
    h2 = B.syk_dot(N, Hpsi, Hpsi, scratch).real
    assert abs(beta[0] - 1.0) <= 1e-13
    assert abs(alpha[0] - a1) <= 1e-13
    assert abs(beta[1] ** 2 - (h2 - a1 * a1)) <= 1e-12


def test_lockstep_pacing_does_not_change_results(B):
    """syk_set_lockstep only paces the producers of the register-tile kernel: outputs are bitwise equal for free
    running CTAs, the default pacing and the tightest pacing (N=48: 268 MB vector > L2; both paced kernels)."""
    import torch
    N = 48
    D = 1 << 24
    h = B.syk_build_hamiltonian(N, inputs.bernoulli_p(N, 4), 0, 3)
    scratch = torch.empty(B.syk_reduce_scratch_bytes(), dtype=torch.uint8, device="cuda")
    d_in = torch.empty(D, dtype=torch.complex128, device="cuda")
    B.syk_random_state(N, 0, 3, d_in, scratch)
    for kind in (2, 3):
        B.syk_set_apply_H_kernel(h, kind)
        assert B.syk_apply_H_kernel_kind(h, B.SYK_C128) == kind
        outs = []
        try:
            for epoch_len, lag in ((0, 0), (8, 1), (1, 0), (3, 5)):
                B.syk_set_lockstep(epoch_len, lag)
                o = torch.zeros(D, dtype=torch.complex128, device="cuda")
                B.syk_apply_H(h, d_in, o)
                torch.cuda.synchronize()
                outs.append(o)
        finally:
            B.syk_set_lockstep(8, 1)
        for o in outs[1:]:
            assert torch.equal(torch.view_as_real(o), torch.view_as_real(outs[0]))
    with pytest.raises(B.SykError):
        B.syk_set_lockstep(-1, 0)
    with pytest.raises(B.SykError):
        B.syk_set_lockstep(4, 31)


def test_apply_H_N66_parity_block_sampled(B):
    """Beyond the paper's largest size (N = 64): N = 66 in one parity block (32 qubits, 2 x 34.4 GB in
    complex64).  Outputs sampled at random reduced indices b' against the oracle's monomial rows of the FULL 33-qubit
    term matrices (row b = b' | (parity(b') xor sector) << 32; the columns, all in the same sector, are read back
    through their low 32 bits), plus the second-moment sum rule."""
    import torch
    if _free_gb() < 72:
        pytest.skip("needs 72 GB of device memory")
    N, sector = 66, 1
    p = inputs.bernoulli_p(N, 2)
    q, J, _ = orng.sample_couplings(N, p, 0, 0)
    h = B.syk_build_hamiltonian(N, p, 0, 0)
    hb = B.syk_build_parity_block(h, sector)
    assert hb.info()["n_terms"] == len(J) and hb.info()["dim"] == 1 << 32
    assert B.syk_apply_H_kernel_kind(hb, B.SYK_C64) == 3
    Dr = 1 << 32
    scratch = torch.empty(B.syk_reduce_scratch_bytes(), dtype=torch.uint8, device="cuda")
    d_in = torch.empty(Dr, dtype=torch.complex64, device="cuda")
    d_out = torch.empty(Dr, dtype=torch.complex64, device="cuda")
    B.syk_random_state(N - 2, 0, 5, d_in, scratch)
    B.syk_apply_H(hb, d_in, d_out)
    torch.cuda.synchronize()
    bp = inputs.sample_indices(Dr, 800, seed=23)
    top = (ohm._popcount_parity(bp) ^ sector).astype(np.uint64)
    full = bp | (top << np.uint64(32))
    cols, vals = ohm.hamiltonian_rows(N, q, J, full)
    assert np.all((ohm._popcount_parity(cols.reshape(-1)) & 1) == sector)          # H conserves parity
    low = (cols & np.uint64(Dr - 1)).astype(np.int64).reshape(-1)
    src = d_in[torch.from_numpy(low).cuda()].cpu().numpy().astype(np.complex128).reshape(cols.shape)
    ref = (vals * src).sum(axis=0)
    got = d_out[torch.from_numpy(bp.astype(np.int64)).cuda()].cpu().numpy().astype(np.complex128)
    assert np.linalg.norm(got - ref) / np.linalg.norm(ref) <= 1e-5
    n2 = B.syk_dot(N - 2, d_out, d_out, scratch).real
    assert abs(n2 / float(np.sum(J ** 2)) - 1.0) <= 5e-3
    assert abs(B.syk_dot(N - 2, d_in, d_out, scratch).imag) <= 1e-6


@pytest.mark.parametrize("N,k,seed", [(46, 4, 0), (46, 1, 1), (48, 8, 2), (50, 2, 3), (50, 16, 4), (52, 4, 5)])
def test_scatter_kernel_many_layouts_sampled(B, N, k, seed):
    """The scatter-tile kernel picks its tile / window bits per Hamiltonian: different seeds and sparsities give
    different layouts (free r bits low, high, adjacent; few or many loads).  Sampled outputs of both precisions against
    the oracle's monomial rows, plain and through a forced register-tile run of the same product."""
    import torch
    D = 1 << (N // 2)
    p = inputs.bernoulli_p(N, k)
    q, J, _ = orng.sample_couplings(N, p, seed, 0)
    h = B.syk_build_hamiltonian(N, p, seed, 0)
    scratch = torch.empty(B.syk_reduce_scratch_bytes(), dtype=torch.uint8, device="cuda")
    idx = inputs.sample_indices(D, 300, seed=31 + seed)
    didx = torch.from_numpy(idx.astype(np.int64)).cuda()
    for tdt, tol in ((torch.complex128, 1e-10), (torch.complex64, 1e-5)):
        code = B.SYK_C128 if tdt == torch.complex128 else B.SYK_C64
        B.syk_set_apply_H_kernel(h, 3)
        if B.syk_apply_H_kernel_kind(h, code) != 3:
            pytest.skip("more than 1024 terms")
        lay = B.syk_apply_H_layout(h, code)
        assert 1 <= lay["n_passes"] <= lay["n_loads"] <= h.info()["n_xmasks"]
        assert lay["tile_mask"] & 0x7FF == 0x7FF and lay["window_mask"] & lay["tile_mask"] == lay["tile_mask"]
        d_in = torch.empty(D, dtype=tdt, device="cuda")
        d_out = torch.empty(D, dtype=tdt, device="cuda")
        B.syk_random_state(N, seed, 7, d_in, scratch)
        B.syk_apply_H(h, d_in, d_out)
        ref = _oracle_samples(N, q, J, idx, d_in)
        got = d_out[didx].cpu().numpy().astype(np.complex128)
        assert np.linalg.norm(got - ref) / np.linalg.norm(ref) <= tol, (N, k, seed, lay)
        B.syk_set_apply_H_kernel(h, 2)
        d_out2 = torch.empty(D, dtype=tdt, device="cuda")
        B.syk_apply_H(h, d_in, d_out2)
        diff = float(torch.linalg.vector_norm(d_out - d_out2) / torch.linalg.vector_norm(d_out2))
        assert diff <= tol
        del d_in, d_out, d_out2


@pytest.mark.parametrize("N,n_samples", [(40, 320), (44, 128)])
def test_dense_table_kernel_multichunk_sampled(B, N, n_samples):
    """Algorithm 1 on the dense p = 1 Hamiltonian (the dense rows of PAPER.md:342-354; BASELINE
    configs[2] "dense p=1") in the form the dense-table kernel takes for N >= 40: ONE persistent CTA per tile (no split),
    several table chunks per source tile streamed through the double buffer.  N = 40: 91 390 terms, 2^20 amplitudes,
    256 tiles; N = 44: 135 751 terms, 1024 tiles.  Sampled outputs (plus the edges of the first / last tiles) against the
    oracle's monomial rows, both precisions, plain and inside two fused Lanczos steps; sum rule; two-pass (out aliases
    prev) against one-pass."""
    import torch
    D = 1 << (N // 2)
    q, J, _ = orng.sample_couplings(N, 1.0, 3, 0)
    h = B.syk_build_from_terms(N, q, J)
    scratch = torch.empty(B.syk_reduce_scratch_bytes(), dtype=torch.uint8, device="cuda")
    idx = inputs.sample_indices(D, n_samples, seed=5)
    edge = np.array([1, 511, 512, 4095, 4096, 8191, D // 2 - 1, D // 2, D - 4097, D - 4096, D - 513, D - 2], dtype=np.uint64)
    idx = np.unique(np.concatenate([idx, edge]))
    didx = torch.from_numpy(idx.astype(np.int64)).cuda()
    cols, vals = ohm.hamiltonian_rows(N, q, J, idx)                      # [T, n] each: the oracle's rows, used for all checks
    flat = torch.from_numpy(cols.astype(np.int64).reshape(-1)).cuda()

    def rows_times(d_vec):
        src = d_vec[flat].cpu().numpy().astype(np.complex128).reshape(cols.shape)
        return (vals * src).sum(axis=0)

    for tdt, code, tol in ((torch.complex128, B.SYK_C128, 1e-10), (torch.complex64, B.SYK_C64, 1e-5)):
        assert B.syk_apply_H_kernel_kind(h, code) == 4                    # automatic choice for dense H
        B.syk_ham_prepare(h, code)
        info = B.syk_apply_H_dense_info(h, code)
        assert info["split"] == 1 and info["n_chunks"] >= info["n_loads"] + 100, info   # non-split; many multi-chunk loads
        d_in = torch.empty(D, dtype=tdt, device="cuda")
        B.syk_random_state(N, 3, 0, d_in, scratch)
        d_out = torch.full((D,), complex(float("nan"), float("nan")), dtype=tdt, device="cuda")
        B.syk_launch_count(reset=True)
        B.syk_apply_H(h, d_in, d_out)
        torch.cuda.synchronize()
        assert B.syk_launch_count(reset=True) == 1                        # one kernel: not split + reduce
        ref = rows_times(d_in)
        got = d_out[didx].cpu().numpy().astype(np.complex128)
        scale = np.sqrt(np.mean(np.abs(ref) ** 2))
        assert np.linalg.norm(got - ref) / np.linalg.norm(ref) <= tol, (N, tdt)
        assert np.max(np.abs(got - ref)) <= 10 * tol * scale
        assert not bool(torch.isnan(torch.view_as_real(d_out)).any())
        n2 = B.syk_dot(N, d_out, d_out, scratch).real                     # sum rule (pin P3): |H psi|^2 ~ sum J^2
        assert abs(n2 / float(np.sum(J ** 2)) - 1.0) <= 2e-2
        # two fused Lanczos steps (one-pass layout: u_2, u_3 are the first two work vectors):
        #   u_2 = H u_1/|u_1| - alpha_1 u_1/|u_1| ;  u_3 = H u_2/|u_2| - (|u_2|/|u_1|) u_1 - alpha_2 u_2/|u_2|
        m = 2
        wk = torch.empty(B.syk_krylov_workspace_bytes(h, code, {"krylov_dim": m}), dtype=torch.uint8, device="cuda")
        alpha, beta, _ = B.syk_lanczos_run(h, d_in, m, wk)
        hdr = (wk.numel() - m * D * d_in.element_size())
        vecs = wk[hdr:].view(tdt).view(m, D)
        u1 = d_in[didx].cpu().numpy().astype(np.complex128)
        u2 = vecs[0][didx].cpu().numpy().astype(np.complex128)
        u3 = vecs[1][didx].cpu().numpy().astype(np.complex128)
        ref2 = ref / beta[0] - alpha[0] * u1 / beta[0]
        assert np.linalg.norm(u2 - ref2) / np.linalg.norm(ref2) <= 2 * tol, (N, tdt)
        ref3 = rows_times(vecs[0]) / beta[1] - (beta[1] / beta[0]) * u1 - alpha[1] * u2 / beta[1]
        assert np.linalg.norm(u3 - ref3) / np.linalg.norm(ref3) <= 4 * tol, (N, tdt)
        a1 = B.syk_dot(N, d_in, d_out, scratch).real / beta[0] ** 2       # alpha_1 = <v|H|v> from the plain product
        assert abs(alpha[0] - a1) <= 10 * tol
        # two-pass (out aliases prev from step 3 on) = one-pass, same kernel
        if N == 40:
            o1, o2 = {"krylov_dim": 5}, {"krylov_dim": 5, "two_pass": 1}
            a, b = d_in.clone(), d_in.clone()
            B.syk_krylov_evolve(h, a, 0.2, -0.1, torch.empty(B.syk_krylov_workspace_bytes(h, code, o1), dtype=torch.uint8, device="cuda"), o1)
            B.syk_krylov_evolve(h, b, 0.2, -0.1, torch.empty(B.syk_krylov_workspace_bytes(h, code, o2), dtype=torch.uint8, device="cuda"), o2)
            rel = float(torch.linalg.vector_norm(a - b) / torch.linalg.vector_norm(a))
            assert rel <= (1e-13 if code == B.SYK_C128 else 2e-6), rel
        del d_in, d_out, wk


@pytest.mark.parametrize("N,k,dt,need_gb", [(56, 4, "c128", 20), (64, 2, "c64", 112)])
def test_fused_lanczos_fullsize_sampled_vs_oracle(B, N, k, dt, need_gb):
    """The FUSED launches bench.py times (scatter-tile kernel, relabelled handle, epilogue out = H u_j/|u_j| - (|u_j|/|u_{j-1}|)
    u_{j-1} with the operands staged through the ring) against the oracle's monomial rows at
    the headline sizes: two fused Lanczos steps in the one-pass layout (u_2, u_3 = the two work vectors), sampled outputs
    incl. the edges of the first / last tiles:
        u_2 = H u_1/|u_1| - alpha_1 u_1/|u_1| ;   u_3 = H u_2/|u_2| - (|u_2|/|u_1|) u_1 - alpha_2 u_2/|u_2| ."""
    import torch
    if _free_gb() < need_gb:
        pytest.skip(f"needs {need_gb} GB of device memory")
    tdt = torch.complex128 if dt == "c128" else torch.complex64
    code = B.SYK_C128 if dt == "c128" else B.SYK_C64
    tol = 1e-10 if dt == "c128" else 1e-5
    D = 1 << (N // 2)
    p = inputs.bernoulli_p(N, k)
    q, J, _ = orng.sample_couplings(N, p, 0, 0)
    h = B.syk_build_hamiltonian(N, p, 0, 0)
    perm = list(B.syk_ham_optimize_layout(h, code)["perm"])
    B.syk_ham_prepare(h, code)
    assert B.syk_apply_H_kernel_kind(h, code) == 3
    scratch = torch.empty(B.syk_reduce_scratch_bytes(), dtype=torch.uint8, device="cuda")
    m = 2
    wk = torch.empty(B.syk_krylov_workspace_bytes(h, code, {"krylov_dim": m}), dtype=torch.uint8, device="cuda")
    psi = torch.empty(D, dtype=tdt, device="cuda")
    B.syk_random_state_h(h, 0, 0, psi, scratch)
    alpha, beta, _ = B.syk_lanczos_run(h, psi, m, wk)
    hdr = wk.numel() - m * D * psi.element_size()
    vecs = wk[hdr:].view(tdt).view(m, D)
    idx = inputs.sample_indices(D, 600, seed=23)
    edge = np.array([0, 1, 8191, 8192, 16383, 16384, D // 2 - 1, D // 2, D - 16385, D - 16384, D - 8193, D - 1], dtype=np.uint64)
    inv = np.argsort(np.array(perm))
    idx = np.unique(np.concatenate([idx, edge, _storage_index(edge, inv)]))
    sidx = torch.from_numpy(_storage_index(idx, perm).astype(np.int64)).cuda()
    u1 = psi[sidx].cpu().numpy().astype(np.complex128)
    u2 = vecs[0][sidx].cpu().numpy().astype(np.complex128)
    u3 = vecs[1][sidx].cpu().numpy().astype(np.complex128)
    Hu1 = _oracle_samples(N, q, J, idx, psi, perm)
    ref2 = Hu1 / beta[0] - alpha[0] * u1 / beta[0]
    assert np.linalg.norm(u2 - ref2) / np.linalg.norm(ref2) <= 2 * tol, (N, dt)
    assert np.max(np.abs(u2 - ref2)) <= 20 * tol * np.sqrt(np.mean(np.abs(ref2) ** 2))
    Hu2 = _oracle_samples(N, q, J, idx, vecs[0], perm)
    ref3 = Hu2 / beta[1] - (beta[1] / beta[0]) * u1 - alpha[1] * u2 / beta[1]
    assert np.linalg.norm(u3 - ref3) / np.linalg.norm(ref3) <= 4 * tol, (N, dt)
    assert np.max(np.abs(u3 - ref3)) <= 40 * tol * np.sqrt(np.mean(np.abs(ref3) ** 2))
    # Lanczos identities with the oracle-checked vectors: beta_2 = |u_2|, alpha_1 real part of <u_1|H u_1> / |u_1|^2
    assert abs(beta[0] - 1.0) <= 1e-12 and beta[1] > 0.0
    n2 = B.syk_dot(N, vecs[0], vecs[0], scratch).real
    assert abs(np.sqrt(n2) / beta[1] - 1.0) <= (1e-12 if dt == "c128" else 1e-6)


def test_two_pass_equals_one_pass_N56(B):
    """Two-pass Lanczos (bounded memory; from step 3 on the fused epilogue's `out` aliases `prev`, both staged
    through the ring of the scatter-tile kernel) against the one-pass evolution of the same relabelled N=56 handle, whose fused
    launches are oracle-checked above: the recurrence is repeated bit-identically, so the results agree to rounding of the
    final combination; and the two-pass run is unitary for real tau."""
    import torch
    if _free_gb() < 48:
        pytest.skip("needs 48 GB of device memory")
    N, D = 56, 1 << 28
    h = B.syk_build_hamiltonian(N, inputs.bernoulli_p(N, 4), 0, 0)
    B.syk_ham_optimize_layout(h, B.SYK_C128)
    B.syk_ham_prepare(h, B.SYK_C128)
    scratch = torch.empty(B.syk_reduce_scratch_bytes(), dtype=torch.uint8, device="cuda")
    a = torch.empty(D, dtype=torch.complex128, device="cuda")
    B.syk_random_state_h(h, 0, 2, a, scratch)
    b = a.clone()
    o1, o2 = {"krylov_dim": 6}, {"krylov_dim": 6, "two_pass": 1}
    w1 = torch.empty(B.syk_krylov_workspace_bytes(h, B.SYK_C128, o1), dtype=torch.uint8, device="cuda")
    st1 = B.syk_krylov_evolve(h, a, 0.3, 0.0, w1, o1)
    del w1
    w2 = torch.empty(B.syk_krylov_workspace_bytes(h, B.SYK_C128, o2), dtype=torch.uint8, device="cuda")
    st2 = B.syk_krylov_evolve(h, b, 0.3, 0.0, w2, o2)
    assert st2["n_matvec"] > st1["n_matvec"]                              # the recurrence ran twice
    rel = float(torch.linalg.vector_norm(a - b) / torch.linalg.vector_norm(a))
    assert rel <= 1e-13, rel
    assert abs(B.syk_dot(N, b, b, scratch).real - 1.0) <= 1e-10           # unitary
