"""syk_dot_static: the allocation-free inner product (per-CTA partial sums in a file-scope __device__ array) against the
existing syk_dot (caller-supplied scratch).  Collected last on purpose (the suite runs with pytest -x): a failure here
hides nothing.  Passes alone in a fresh process and after the other GPU tests (the static array keeps whatever earlier
calls left in it; nothing in it has to start at zero)."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

TOL = {"c128": 1e-10, "c64": 1e-5}   # the parity tolerances of tests/test_gpu_parity.py (BASELINE.json north_star)


@pytest.fixture(scope="module")
def B():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2311_00639_b200 import binding   # raises if the library is not built: no CPU path
    return binding


def _vec(torch, rs, D, dt):
    v = rs.standard_normal(D) + 1j * rs.standard_normal(D)
    return torch.from_numpy(v.astype(np.complex128 if dt == "c128" else np.complex64)).cuda()


@pytest.mark.parametrize("dt", ["c128", "c64"])
def test_dot_static_matches_dot_two_calls_in_a_row(B, dt):
    import torch
    rs = np.random.default_rng(17)
    scratch = torch.empty(B.syk_reduce_scratch_bytes(), dtype=torch.uint8, device="cuda")
    B.syk_dot_static_prepare()
    # a long vector first (N = 46: 2^23 amplitudes, 1024 / 512 partial sums), then a short one (N = 30: 4 / 2 partials, the
    # rest of the array still holds the first call's), then a tiny one (N = 4: one partly filled CTA)
    cases = [(46, _vec(torch, rs, 1 << 23, dt), _vec(torch, rs, 1 << 23, dt)),
             (30, _vec(torch, rs, 1 << 15, dt), _vec(torch, rs, 1 << 15, dt)),
             (4, _vec(torch, rs, 4, dt), _vec(torch, rs, 4, dt))]
    res = torch.full((len(cases), 2), float("nan"), dtype=torch.float64, device="cuda")
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    for i, (N, a, b) in enumerate(cases):            # back to back on one stream, no synchronisation in between
        B.syk_dot_static(N, a, b, res[i])
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free0      # cudaMemGetInfo sees the library's own cudaMalloc calls: none
    got = res.cpu().numpy()
    for i, (N, a, b) in enumerate(cases):
        ref = B.syk_dot(N, a, b, scratch)
        scale = float(torch.linalg.vector_norm(a) * torch.linalg.vector_norm(b))
        assert abs(complex(got[i, 0], got[i, 1]) - ref) <= TOL[dt] * scale, (N, got[i], ref)
        # and against the plain definition in fp64 (numpy): sum conj(a) b
        plain = np.vdot(a.cpu().numpy().astype(np.complex128), b.cpu().numpy().astype(np.complex128))
        assert abs(complex(got[i, 0], got[i, 1]) - plain) <= TOL[dt] * scale
    # the same call again gives the same bits (fixed summation order, no dependence on what the array held)
    res2 = torch.empty(2, dtype=torch.float64, device="cuda")
    B.syk_dot_static(cases[0][0], cases[0][1], cases[0][2], res2)
    torch.cuda.synchronize()
    assert torch.equal(res2, res[0])


def test_dot_static_limits_and_errors(B):
    import torch
    assert B.syk_dot_static_max_N(B.SYK_C128) == 50 and B.syk_dot_static_max_N(B.SYK_C64) == 52
    a = torch.zeros(16, dtype=torch.complex128, device="cuda")
    out = torch.full((2,), 7.0, dtype=torch.float64, device="cuda")
    for N, code in ((52, B.SYK_ELIMIT), (64, B.SYK_ELIMIT), (5, B.SYK_EINVAL), (2, B.SYK_EINVAL)):
        with pytest.raises(B.SykError) as ei:         # rejected before anything is launched or read
            B.syk_dot_static(N, a, a, out)
        assert ei.value.code == code, (N, ei.value.code)
    c = torch.zeros(16, dtype=torch.complex64, device="cuda")
    with pytest.raises(B.SykError) as ei:
        B.syk_dot_static(54, c, c, out)
    assert ei.value.code == B.SYK_ELIMIT
    torch.cuda.synchronize()
    assert out.tolist() == [7.0, 7.0]
    assert b"syk_dot_static_max_N" in B._lib.syk_strerror(B.SYK_ELIMIT)
