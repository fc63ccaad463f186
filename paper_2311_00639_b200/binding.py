"""ctypes binding of libsyk_b200 (include/syk.h): the same names, argument marshalling only.

Every step of the hot path runs inside the CUDA library; this module turns torch tensors into
`data_ptr()` + `torch.cuda.current_stream().cuda_stream`, numpy arrays into host pointers, and error
codes into exceptions.  There is no CPU fallback: if the library has not been built, importing this
module raises; on a machine without a CUDA device every compute call raises `SykError(SYK_ECUDA)`.
"""
import ctypes
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libsyk_b200.so")

SYK_OK, SYK_EINVAL, SYK_ENOMEM, SYK_ECUDA, SYK_ENOCONV, SYK_ELIMIT = 0, -1, -2, -3, -4, -5
SYK_C64, SYK_C128 = 0, 1
SYK_GAMMA_PAULI, SYK_GAMMA_HALF = 0, 1

if not os.path.exists(LIB_PATH):
    raise ImportError(
        f"{LIB_PATH} is missing: build it with `python -m paper_2311_00639_b200.build` "
        "(nvcc, sm_100a).  There is no CPU fallback.")
_lib = ctypes.CDLL(LIB_PATH)


class syk_krylov_opts(ctypes.Structure):
    _fields_ = [("krylov_dim", ctypes.c_int), ("tol", ctypes.c_double), ("two_pass", ctypes.c_int),
                ("max_substeps", ctypes.c_int), ("renormalize", ctypes.c_int)]


class syk_stats(ctypes.Structure):
    _fields_ = [("n_matvec", ctypes.c_int64), ("n_substeps", ctypes.c_int), ("krylov_dim_used", ctypes.c_int),
                ("err_est", ctypes.c_double), ("model_bytes", ctypes.c_double), ("elapsed_ms", ctypes.c_double),
                ("log_norm", ctypes.c_double)]

    def as_dict(self):
        return {name: getattr(self, name) for name, _ in self._fields_}


class SykError(RuntimeError):
    def __init__(self, code, where):
        self.code = code
        text = _lib.syk_strerror(code).decode()
        cuda = _lib.syk_last_cuda_error().decode() if code == SYK_ECUDA else ""
        super().__init__(f"{where}: {text} ({code})" + (f" [{cuda}]" if cuda else ""))


_vp, _i, _i64, _u64, _u32, _d, _sz = (ctypes.c_void_p, ctypes.c_int, ctypes.c_int64, ctypes.c_uint64,
                                     ctypes.c_uint32, ctypes.c_double, ctypes.c_size_t)
_P = ctypes.POINTER
_SIGNATURES = {
    "syk_strerror": (ctypes.c_char_p, [_i]),
    "syk_last_cuda_error": (ctypes.c_char_p, []),
    "syk_version": (_i, []),
    "syk_build_hamiltonian": (_i, [_i, _d, _u64, _u32, _i, _P(_vp)]),
    "syk_build_from_terms": (_i, [_i, _i64, _vp, _vp, _i, _P(_vp)]),
    "syk_build_from_pauli_strings": (_i, [_i, _i64, _vp, _vp, _vp, _P(_vp)]),
    "syk_build_from_terms_complex": (_i, [_i, _i64, _vp, _vp, _i, _P(_vp)]),
    "syk_ham_is_hermitian": (_i, [_vp]),
    "syk_free_hamiltonian": (None, [_vp]),
    "syk_ham_info": (_i, [_vp, _P(_i), _P(_i64), _P(_i64), _P(_i64)]),
    "syk_ham_tables": (_i, [_vp, _vp, _vp, _vp, _vp, _vp, _vp]),
    "syk_ham_prepare": (_i, [_vp, _i]),
    "syk_ham_optimize_layout": (_i, [_vp, _i]),
    "syk_ham_set_layout": (_i, [_vp, _vp]),
    "syk_ham_layout": (_i, [_vp, _vp, _P(_i)]),
    "syk_permute_vector": (_i, [_vp, _i, _i, _vp, _vp, _vp]),
    "syk_random_state_h": (_i, [_vp, _u64, _u32, _i, _vp, _vp, _vp]),
    "syk_apply_gamma_h": (_i, [_vp, _i, _i, _vp, _vp, _vp]),
    "syk_apply_gamma_block_h": (_i, [_vp, _i, _i, _i, _vp, _vp, _vp]),
    "syk_apply_H_dense_info": (_i, [_vp, _i, _P(_i), _P(_i), _P(_i), _P(_i)]),
    "syk_apply_H": (_i, [_vp, _i, _vp, _vp, _vp]),
    "syk_apply_H_batched": (_i, [_P(_vp), _i, _i, _vp, _vp, _i64, _vp]),
    "syk_apply_H_host": (_i, [_vp, _i, _vp, _vp, _vp, _sz, _vp]),
    "syk_apply_gamma": (_i, [_i, _i, _i, _i, _vp, _vp, _vp]),
    "syk_reduce_scratch_bytes": (_sz, []),
    "syk_random_state": (_i, [_i, _u64, _u32, _i, _vp, _vp, _vp]),
    "syk_dot": (_i, [_i, _i, _vp, _vp, _vp, _P(_d), _vp]),
    "syk_dot_static_max_N": (_i, [_i]),
    "syk_dot_static_prepare": (_i, []),
    "syk_dot_static": (_i, [_i, _i, _vp, _vp, _vp, _vp]),
    "syk_krylov_workspace_bytes": (_i, [_vp, _i, _P(syk_krylov_opts), _P(_sz)]),
    "syk_lanczos_run": (_i, [_vp, _i, _vp, _i, _vp, _vp, _vp, _sz, _P(syk_stats), _vp]),
    "syk_krylov_evolve": (_i, [_vp, _i, _vp, _d, _d, _P(syk_krylov_opts), _vp, _sz, _P(syk_stats), _vp]),
    "syk_krylov_evolve_host": (_i, [_vp, _i, _vp, _d, _d, _P(syk_krylov_opts), _vp, _sz, _P(syk_stats), _vp]),
    "syk_otoc_workspace_bytes": (_i, [_vp, _i, _P(syk_krylov_opts), _P(_sz)]),
    "syk_otoc": (_i, [_vp, _i, _i, _i, _d, _vp, _i, _vp, _vp, _P(syk_krylov_opts), _vp, _sz, _P(syk_stats), _vp]),
    "syk_green": (_i, [_vp, _i, _i, _d, _vp, _i, _vp, _vp, _P(syk_krylov_opts), _vp, _sz, _P(syk_stats), _vp]),
    "syk_build_parity_block": (_i, [_vp, _i, _P(_vp)]),
    "syk_apply_gamma_block": (_i, [_i, _i, _i, _i, _i, _vp, _vp, _vp]),
    "syk_otoc_block": (_i, [_vp, _vp, _i, _i, _i, _i, _d, _vp, _i, _vp, _vp, _P(syk_krylov_opts), _vp, _sz, _P(syk_stats),
                            _vp]),
    "syk_green_block": (_i, [_vp, _vp, _i, _i, _i, _d, _vp, _i, _vp, _vp, _P(syk_krylov_opts), _vp, _sz, _P(syk_stats),
                             _vp]),
    "syk_krylov_workspace_bytes_batched": (_i, [_vp, _i, _i, _P(syk_krylov_opts), _P(_sz)]),
    "syk_krylov_evolve_batched": (_i, [_P(_vp), _i, _i, _vp, _i64, _d, _d, _P(syk_krylov_opts), _vp, _sz, _P(syk_stats),
                                       _vp]),
    "syk_otoc_batched_workspace_bytes": (_i, [_vp, _i, _i, _P(syk_krylov_opts), _P(_sz)]),
    "syk_otoc_batched": (_i, [_P(_vp), _i, _i, _i, _i, _d, _vp, _i, _vp, _i64, _vp, _P(syk_krylov_opts), _vp, _sz,
                              _P(syk_stats), _vp]),
    "syk_green_batched": (_i, [_P(_vp), _i, _i, _i, _d, _vp, _i, _vp, _i64, _vp, _P(syk_krylov_opts), _vp, _sz,
                               _P(syk_stats), _vp]),
    "syk_apply_H_kernel_kind": (_i, [_vp, _i]),
    "syk_set_apply_H_kernel": (_i, [_vp, _i]),
    "syk_set_lockstep": (_i, [_i, _i]),
    "syk_set_cuda_graphs": (_i, [_i]),
    "syk_apply_H_layout": (_i, [_vp, _i, _P(_i), _P(_i), _P(_u32), _P(_u32)]),
    "syk_apply_H_trace": (_i, [_vp, _i, _vp, _vp, _i, _i, _i, _vp, _i, _vp, _vp, _i, _P(_i), _P(_i), _vp]),
    "syk_launch_count": (_i64, [_i]),
    "syk_microbench_workspace_bytes": (_sz, []),
    "syk_microbench": (_i, [_i, _i, _i, _vp, _sz, _vp, _sz, _P(_d), _vp]),
    "syk_profile_enable": (_i, [_i]),
    "syk_profile_read": (_i, [_P(_d), _P(_i64), _i]),
}
for _name, (_res, _args) in _SIGNATURES.items():
    _fn = getattr(_lib, _name)
    _fn.restype, _fn.argtypes = _res, _args

EXPORTED = tuple(_SIGNATURES)


def _check(code, where, soft=(SYK_OK,)):
    if code not in soft:
        raise SykError(code, where)
    return code


def _dptr(t):
    """Device pointer of a torch tensor (must be contiguous and on a CUDA device) or a raw int."""
    if isinstance(t, int):
        return t
    if not t.is_cuda:
        raise SykError(SYK_ECUDA, "expected a CUDA tensor (there is no CPU path)")
    if not t.is_contiguous():
        raise SykError(SYK_EINVAL, "tensor must be contiguous")
    return t.data_ptr()


def _stream(stream=None):
    if stream is not None:
        return int(stream)
    import torch
    return torch.cuda.current_stream().cuda_stream if torch.cuda.is_available() else 0


def dtype_code(t):
    import torch
    if t.dtype == torch.complex128:
        return SYK_C128
    if t.dtype == torch.complex64:
        return SYK_C64
    raise SykError(SYK_EINVAL, f"unsupported dtype {t.dtype}")


def _opts(opts):
    if opts is None:
        return None
    if isinstance(opts, syk_krylov_opts):
        return ctypes.byref(opts)
    o = syk_krylov_opts(int(opts.get("krylov_dim", 0)), float(opts.get("tol", 0.0)), int(opts.get("two_pass", 0)),
                        int(opts.get("max_substeps", 0)), int(opts.get("renormalize", 0)))
    return ctypes.byref(o)


class Hamiltonian:
    """Owner of one `syk_ham*` handle."""

    def __init__(self, handle):
        self._h = ctypes.c_void_p(handle)

    @property
    def handle(self):
        return self._h

    def close(self):
        if self._h:
            _lib.syk_free_hamiltonian(self._h)
            self._h = ctypes.c_void_p(None)

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def info(self):
        return syk_ham_info(self)

    def tables(self):
        return syk_ham_tables(self)


def _h(h):
    return h.handle if isinstance(h, Hamiltonian) else h


# ---- a-1 ---------------------------------------------------------------------------------------------------
def syk_build_hamiltonian(N, p, seed, realization=0, gamma_norm=SYK_GAMMA_PAULI):
    out = ctypes.c_void_p()
    _check(_lib.syk_build_hamiltonian(int(N), float(p), int(seed), int(realization), int(gamma_norm),
                                      ctypes.byref(out)), "syk_build_hamiltonian")
    return Hamiltonian(out.value)


def syk_build_from_terms(N, quartets, J, gamma_norm=SYK_GAMMA_PAULI):
    q = np.ascontiguousarray(quartets, dtype=np.int32).reshape(-1, 4)
    Jc = np.ascontiguousarray(J, dtype=np.float64).reshape(-1)
    if len(q) != len(Jc):
        raise SykError(SYK_EINVAL, "syk_build_from_terms: quartets and J differ in length")
    out = ctypes.c_void_p()
    _check(_lib.syk_build_from_terms(int(N), len(Jc), q.ctypes.data, Jc.ctypes.data, int(gamma_norm),
                                     ctypes.byref(out)), "syk_build_from_terms")
    return Hamiltonian(out.value)


def syk_build_from_terms_complex(N, quartets, J, gamma_norm=SYK_GAMMA_PAULI):
    """Complex couplings: the non-Hermitian SYK model."""
    q = np.ascontiguousarray(quartets, dtype=np.int32).reshape(-1, 4)
    Jc = np.asarray(J, dtype=np.complex128).reshape(-1)
    if len(q) != len(Jc):
        raise SykError(SYK_EINVAL, "syk_build_from_terms_complex: quartets and J differ in length")
    Jri = np.ascontiguousarray(np.stack([Jc.real, Jc.imag], axis=1), dtype=np.float64)
    out = ctypes.c_void_p()
    _check(_lib.syk_build_from_terms_complex(int(N), len(Jc), q.ctypes.data, Jri.ctypes.data, int(gamma_norm),
                                             ctypes.byref(out)), "syk_build_from_terms_complex")
    return Hamiltonian(out.value)


def syk_ham_is_hermitian(h):
    return bool(_check(_lib.syk_ham_is_hermitian(_h(h)), "syk_ham_is_hermitian", soft=(0, 1)))


def syk_build_from_pauli_strings(L, terms):
    """terms: iterable of (x, z, c), c any complex number (see include/syk.h for when the sum is Hermitian)."""
    terms = list(terms)
    x = np.array([int(t[0]) for t in terms], dtype=np.uint64)
    z = np.array([int(t[1]) for t in terms], dtype=np.uint64)
    c = np.array([[complex(t[2]).real, complex(t[2]).imag] for t in terms], dtype=np.float64).reshape(-1, 2)
    out = ctypes.c_void_p()
    _check(_lib.syk_build_from_pauli_strings(int(L), len(terms), x.ctypes.data, z.ctypes.data, c.ctypes.data,
                                             ctypes.byref(out)), "syk_build_from_pauli_strings")
    return Hamiltonian(out.value)


def syk_ham_info(h):
    N, nt, nx, dim = ctypes.c_int(), ctypes.c_int64(), ctypes.c_int64(), ctypes.c_int64()
    _check(_lib.syk_ham_info(_h(h), ctypes.byref(N), ctypes.byref(nt), ctypes.byref(nx), ctypes.byref(dim)),
           "syk_ham_info")
    return {"N": N.value, "n_terms": nt.value, "n_xmasks": nx.value, "dim": dim.value}


def syk_ham_tables(h):
    info = syk_ham_info(h)
    nt, nx = info["n_terms"], info["n_xmasks"]
    x = np.zeros(nx, dtype=np.uint64)
    off = np.zeros(nx + 1, dtype=np.uint32)
    z = np.zeros(nt, dtype=np.uint64)
    c = np.zeros((nt, 2), dtype=np.float64)
    quart = np.zeros((nt, 4), dtype=np.int32)
    J = np.zeros(nt, dtype=np.float64)
    _check(_lib.syk_ham_tables(_h(h), x.ctypes.data, off.ctypes.data, z.ctypes.data, c.ctypes.data,
                               quart.ctypes.data, J.ctypes.data), "syk_ham_tables")
    return {"x": x, "group_off": off, "z": z, "c": c[:, 0] + 1j * c[:, 1], "quartet_of_term": quart, "J": J}


def syk_ham_optimize_layout(h, dtype):
    _check(_lib.syk_ham_optimize_layout(_h(h), int(dtype)), "syk_ham_optimize_layout")
    return syk_ham_layout(h)


def syk_ham_set_layout(h, perm):
    """perm[q] = index bit of qubit q (None = identity)."""
    if perm is None:
        _check(_lib.syk_ham_set_layout(_h(h), None), "syk_ham_set_layout")
        return
    p = np.ascontiguousarray(perm, dtype=np.int32)
    if len(p) != syk_ham_info(h)["N"] // 2:
        raise SykError(SYK_EINVAL, "syk_ham_set_layout: perm must have N/2 entries")
    _check(_lib.syk_ham_set_layout(_h(h), p.ctypes.data), "syk_ham_set_layout")


def syk_ham_layout(h):
    L = syk_ham_info(h)["N"] // 2
    p = np.zeros(L, dtype=np.int32)
    ident = _i()
    _check(_lib.syk_ham_layout(_h(h), p.ctypes.data, ctypes.byref(ident)), "syk_ham_layout")
    return {"perm": p, "identity": bool(ident.value)}


def syk_permute_vector(h, to_layout, d_in, d_out, stream=None):
    _check(_lib.syk_permute_vector(_h(h), dtype_code(d_in), 1 if to_layout else 0, _dptr(d_in), _dptr(d_out),
                                   _stream(stream)), "syk_permute_vector")
    return d_out


def syk_random_state_h(h, seed, realization, d_psi, d_scratch, stream=None):
    _check(_lib.syk_random_state_h(_h(h), int(seed), int(realization), dtype_code(d_psi), _dptr(d_psi), _dptr(d_scratch),
                                   _stream(stream)), "syk_random_state_h")
    return d_psi


def syk_apply_gamma_h(h, n, d_in, d_out, stream=None):
    _check(_lib.syk_apply_gamma_h(_h(h), int(n), dtype_code(d_in), _dptr(d_in), _dptr(d_out), _stream(stream)),
           "syk_apply_gamma_h")
    return d_out


def syk_apply_gamma_block_h(h_block, n, sector_out, d_in, d_out, stream=None):
    _check(_lib.syk_apply_gamma_block_h(_h(h_block), int(n), int(sector_out), dtype_code(d_in), _dptr(d_in), _dptr(d_out),
                                        _stream(stream)), "syk_apply_gamma_block_h")
    return d_out


def syk_ham_prepare(h, dtype):
    _check(_lib.syk_ham_prepare(_h(h), int(dtype)), "syk_ham_prepare")


def syk_apply_H_dense_info(h, dtype):
    nl, nc, sp, ng = _i(), _i(), _i(), _i()
    _check(_lib.syk_apply_H_dense_info(_h(h), int(dtype), ctypes.byref(nl), ctypes.byref(nc), ctypes.byref(sp),
                                       ctypes.byref(ng)), "syk_apply_H_dense_info")
    return {"n_loads": nl.value, "n_chunks": nc.value, "split": sp.value, "n_local_groups": ng.value}


# ---- a-2 ---------------------------------------------------------------------------------------------------
def syk_apply_H(h, d_in, d_out, stream=None):
    _check(_lib.syk_apply_H(_h(h), dtype_code(d_in), _dptr(d_in), _dptr(d_out), _stream(stream)), "syk_apply_H")
    return d_out


def syk_apply_H_batched(hams, d_in, d_out, batch_stride, stream=None):
    arr = (ctypes.c_void_p * len(hams))(*[_h(h).value for h in hams])
    _check(_lib.syk_apply_H_batched(arr, len(hams), dtype_code(d_in), _dptr(d_in), _dptr(d_out), int(batch_stride),
                                    _stream(stream)), "syk_apply_H_batched")
    return d_out


def syk_apply_H_host(h, h_in, h_out, d_work, stream=None):
    """h_in / h_out: numpy complex64/complex128 arrays or pinned CPU torch tensors; d_work: CUDA byte tensor."""
    code, pin, pout = _host_vec(h_in), _host_ptr(h_in), _host_ptr(h_out)
    _check(_lib.syk_apply_H_host(_h(h), code, pin, pout, _dptr(d_work), d_work.numel() * d_work.element_size(),
                                 _stream(stream)), "syk_apply_H_host")
    return h_out


def _host_vec(a):
    if isinstance(a, np.ndarray):
        if a.dtype == np.complex128:
            return SYK_C128
        if a.dtype == np.complex64:
            return SYK_C64
        raise SykError(SYK_EINVAL, f"unsupported dtype {a.dtype}")
    return dtype_code(a)


def _host_ptr(a):
    if isinstance(a, np.ndarray):
        if not a.flags["C_CONTIGUOUS"]:
            raise SykError(SYK_EINVAL, "host array must be contiguous")
        return a.ctypes.data
    if a.is_cuda:
        raise SykError(SYK_EINVAL, "expected a host tensor")
    return a.data_ptr()


def syk_apply_gamma(N, n, d_in, d_out, gamma_norm=SYK_GAMMA_PAULI, stream=None):
    _check(_lib.syk_apply_gamma(int(N), int(n), int(gamma_norm), dtype_code(d_in), _dptr(d_in), _dptr(d_out),
                                _stream(stream)), "syk_apply_gamma")
    return d_out


# ---- state, dot --------------------------------------------------------------------------------------------
def syk_reduce_scratch_bytes():
    return int(_lib.syk_reduce_scratch_bytes())


def syk_random_state(N, seed, realization, d_psi, d_scratch, stream=None):
    _check(_lib.syk_random_state(int(N), int(seed), int(realization), dtype_code(d_psi), _dptr(d_psi),
                                 _dptr(d_scratch), _stream(stream)), "syk_random_state")
    return d_psi


def syk_dot(N, d_a, d_b, d_scratch, stream=None):
    out = (ctypes.c_double * 2)()
    _check(_lib.syk_dot(int(N), dtype_code(d_a), _dptr(d_a), _dptr(d_b), _dptr(d_scratch), out, _stream(stream)),
           "syk_dot")
    return complex(out[0], out[1])


def syk_dot_static_max_N(dtype):
    return int(_lib.syk_dot_static_max_N(int(dtype)))


def syk_dot_static_prepare():
    _check(_lib.syk_dot_static_prepare(), "syk_dot_static_prepare")


def syk_dot_static(N, d_a, d_b, d_result, stream=None):
    """(Re, Im) <a|b> into the DEVICE tensor d_result (2 float64); allocation-free, asynchronous (include/syk.h)."""
    _check(_lib.syk_dot_static(int(N), dtype_code(d_a), _dptr(d_a), _dptr(d_b), _dptr(d_result), _stream(stream)),
           "syk_dot_static")
    return d_result


# ---- a-3 / a-4 ---------------------------------------------------------------------------------------------
def syk_krylov_workspace_bytes(h, dtype, opts=None):
    n = ctypes.c_size_t()
    _check(_lib.syk_krylov_workspace_bytes(_h(h), int(dtype), _opts(opts), ctypes.byref(n)),
           "syk_krylov_workspace_bytes")
    return n.value


def syk_lanczos_run(h, d_psi, m, d_work, stream=None):
    alpha = np.zeros(m, dtype=np.float64)
    beta = np.zeros(m + 1, dtype=np.float64)
    st = syk_stats()
    _check(_lib.syk_lanczos_run(_h(h), dtype_code(d_psi), _dptr(d_psi), int(m), alpha.ctypes.data, beta.ctypes.data,
                                _dptr(d_work), d_work.numel() * d_work.element_size(), ctypes.byref(st),
                                _stream(stream)), "syk_lanczos_run")
    return alpha, beta, st.as_dict()


def syk_krylov_evolve(h, d_psi, tau_re, tau_im, d_work, opts=None, stream=None, allow_noconv=False):
    st = syk_stats()
    rc = _check(_lib.syk_krylov_evolve(_h(h), dtype_code(d_psi), _dptr(d_psi), float(tau_re), float(tau_im),
                                       _opts(opts), _dptr(d_work), d_work.numel() * d_work.element_size(),
                                       ctypes.byref(st), _stream(stream)), "syk_krylov_evolve",
                soft=(SYK_OK, SYK_ENOCONV) if allow_noconv else (SYK_OK,))
    d = st.as_dict()
    d["rc"] = rc
    return d


def syk_krylov_evolve_host(h, h_psi, tau_re, tau_im, d_work, opts=None, stream=None):
    st = syk_stats()
    _check(_lib.syk_krylov_evolve_host(_h(h), _host_vec(h_psi), _host_ptr(h_psi), float(tau_re), float(tau_im),
                                       _opts(opts), _dptr(d_work), d_work.numel() * d_work.element_size(),
                                       ctypes.byref(st), _stream(stream)), "syk_krylov_evolve_host")
    return st.as_dict()


# ---- a-5 ---------------------------------------------------------------------------------------------------
def syk_otoc_workspace_bytes(h, dtype, opts=None):
    n = ctypes.c_size_t()
    _check(_lib.syk_otoc_workspace_bytes(_h(h), int(dtype), _opts(opts), ctypes.byref(n)), "syk_otoc_workspace_bytes")
    return n.value


def syk_otoc(h, i_W, j_V, beta, t_grid, d_psi, d_work, opts=None, stream=None):
    """Returns (F[n_t] complex128 un-normalised, stats).  d_psi is destroyed."""
    t = np.ascontiguousarray(t_grid, dtype=np.float64)
    F = np.zeros((len(t), 2), dtype=np.float64)
    st = syk_stats()
    _check(_lib.syk_otoc(_h(h), dtype_code(d_psi), int(i_W), int(j_V), float(beta), t.ctypes.data, len(t),
                         _dptr(d_psi), F.ctypes.data, _opts(opts), _dptr(d_work),
                         d_work.numel() * d_work.element_size(), ctypes.byref(st), _stream(stream)), "syk_otoc")
    return F[:, 0] + 1j * F[:, 1], st.as_dict()


def syk_green(h, n, beta, t_grid, d_psi, d_work, opts=None, stream=None):
    """Returns (G[n_t] complex128 un-normalised, stats).  d_psi is destroyed."""
    t = np.ascontiguousarray(t_grid, dtype=np.float64)
    G = np.zeros((len(t), 2), dtype=np.float64)
    st = syk_stats()
    _check(_lib.syk_green(_h(h), dtype_code(d_psi), int(n), float(beta), t.ctypes.data, len(t), _dptr(d_psi),
                          G.ctypes.data, _opts(opts), _dptr(d_work), d_work.numel() * d_work.element_size(),
                          ctypes.byref(st), _stream(stream)), "syk_green")
    return G[:, 0] + 1j * G[:, 1], st.as_dict()


def syk_build_parity_block(h, sector):
    out = ctypes.c_void_p()
    _check(_lib.syk_build_parity_block(_h(h), int(sector), ctypes.byref(out)), "syk_build_parity_block")
    return Hamiltonian(out.value)


def syk_apply_gamma_block(N, n, sector_out, d_in, d_out, gamma_norm=SYK_GAMMA_PAULI, stream=None):
    _check(_lib.syk_apply_gamma_block(int(N), int(n), int(gamma_norm), int(sector_out), dtype_code(d_in), _dptr(d_in),
                                      _dptr(d_out), _stream(stream)), "syk_apply_gamma_block")
    return d_out


def syk_otoc_block(h_even, h_odd, sector, i_W, j_V, beta, t_grid, d_psi, d_work, opts=None, stream=None):
    """One parity sector's term of F(t); d_psi is the reduced state (destroyed)."""
    t = np.ascontiguousarray(t_grid, dtype=np.float64)
    F = np.zeros((len(t), 2), dtype=np.float64)
    st = syk_stats()
    _check(_lib.syk_otoc_block(_h(h_even), _h(h_odd), int(sector), dtype_code(d_psi), int(i_W), int(j_V), float(beta),
                               t.ctypes.data, len(t), _dptr(d_psi), F.ctypes.data, _opts(opts), _dptr(d_work),
                               d_work.numel() * d_work.element_size(), ctypes.byref(st), _stream(stream)),
           "syk_otoc_block")
    return F[:, 0] + 1j * F[:, 1], st.as_dict()


def syk_green_block(h_even, h_odd, sector, n, beta, t_grid, d_psi, d_work, opts=None, stream=None):
    """One parity sector's term of G(t); d_psi is the reduced state (destroyed)."""
    t = np.ascontiguousarray(t_grid, dtype=np.float64)
    G = np.zeros((len(t), 2), dtype=np.float64)
    st = syk_stats()
    _check(_lib.syk_green_block(_h(h_even), _h(h_odd), int(sector), dtype_code(d_psi), int(n), float(beta),
                                t.ctypes.data, len(t), _dptr(d_psi), G.ctypes.data, _opts(opts), _dptr(d_work),
                                d_work.numel() * d_work.element_size(), ctypes.byref(st), _stream(stream)),
           "syk_green_block")
    return G[:, 0] + 1j * G[:, 1], st.as_dict()


def syk_krylov_workspace_bytes_batched(h, n_batch, dtype, opts=None):
    n = ctypes.c_size_t()
    _check(_lib.syk_krylov_workspace_bytes_batched(_h(h), int(n_batch), int(dtype), _opts(opts), ctypes.byref(n)),
           "syk_krylov_workspace_bytes_batched")
    return n.value


def syk_krylov_evolve_batched(hams, d_psi, batch_stride, tau_re, tau_im, d_work, opts=None, stream=None):
    arr = (ctypes.c_void_p * len(hams))(*[_h(h).value for h in hams])
    st = syk_stats()
    _check(_lib.syk_krylov_evolve_batched(arr, len(hams), dtype_code(d_psi), _dptr(d_psi), int(batch_stride),
                                          float(tau_re), float(tau_im), _opts(opts), _dptr(d_work),
                                          d_work.numel() * d_work.element_size(), ctypes.byref(st), _stream(stream)),
           "syk_krylov_evolve_batched")
    return st.as_dict()


def syk_otoc_batched_workspace_bytes(h, n_batch, dtype, opts=None):
    n = ctypes.c_size_t()
    _check(_lib.syk_otoc_batched_workspace_bytes(_h(h), int(n_batch), int(dtype), _opts(opts), ctypes.byref(n)),
           "syk_otoc_batched_workspace_bytes")
    return n.value


def syk_otoc_batched(hams, i_W, j_V, beta, t_grid, d_psi, batch_stride, d_work, opts=None, stream=None):
    t = np.ascontiguousarray(t_grid, dtype=np.float64)
    F = np.zeros((len(hams), len(t), 2), dtype=np.float64)
    arr = (ctypes.c_void_p * len(hams))(*[_h(h).value for h in hams])
    st = syk_stats()
    _check(_lib.syk_otoc_batched(arr, len(hams), dtype_code(d_psi), int(i_W), int(j_V), float(beta), t.ctypes.data,
                                 len(t), _dptr(d_psi), int(batch_stride), F.ctypes.data, _opts(opts), _dptr(d_work),
                                 d_work.numel() * d_work.element_size(), ctypes.byref(st), _stream(stream)),
           "syk_otoc_batched")
    return F[..., 0] + 1j * F[..., 1], st.as_dict()


def syk_green_batched(hams, n, beta, t_grid, d_psi, batch_stride, d_work, opts=None, stream=None):
    t = np.ascontiguousarray(t_grid, dtype=np.float64)
    G = np.zeros((len(hams), len(t), 2), dtype=np.float64)
    arr = (ctypes.c_void_p * len(hams))(*[_h(h).value for h in hams])
    st = syk_stats()
    _check(_lib.syk_green_batched(arr, len(hams), dtype_code(d_psi), int(n), float(beta), t.ctypes.data, len(t),
                                  _dptr(d_psi), int(batch_stride), G.ctypes.data, _opts(opts), _dptr(d_work),
                                  d_work.numel() * d_work.element_size(), ctypes.byref(st), _stream(stream)),
           "syk_green_batched")
    return G[..., 0] + 1j * G[..., 1], st.as_dict()


# ---- introspection -------------------------------------------------------------------------------------------
def syk_apply_H_kernel_kind(h, dtype):
    return int(_lib.syk_apply_H_kernel_kind(_h(h), int(dtype)))


def syk_set_apply_H_kernel(h, kind):
    _check(_lib.syk_set_apply_H_kernel(_h(h), int(kind)), "syk_set_apply_H_kernel")


def syk_apply_H_layout(h, dtype):
    nl, npass, tm, wm = _i(), _i(), _u32(), _u32()
    _check(_lib.syk_apply_H_layout(_h(h), int(dtype), ctypes.byref(nl), ctypes.byref(npass), ctypes.byref(tm),
                                   ctypes.byref(wm)), "syk_apply_H_layout")
    return {"n_loads": nl.value, "n_passes": npass.value, "tile_mask": tm.value, "window_mask": wm.value}


def syk_apply_H_trace(h, d_in, d_out, cta=0, round=2, detail=0, stream=None):
    """One plain scatter-tile product with the timeline of one persistent CTA (include/syk.h).  Returns a dict with the
    clock stamps per ring chunk (issue, before_wait, after_wait, first_decoded, first_issued, all_issued, arrived), the load list (terms, xo per load) and the CTA's rotation."""
    n_loads_max = 1024
    clk = np.zeros(7 * 2 * n_loads_max, dtype=np.uint64)
    terms = np.zeros(n_loads_max, dtype=np.int32)
    xo = np.zeros(n_loads_max, dtype=np.uint32)
    nl, rot = _i(), _i()
    _check(_lib.syk_apply_H_trace(_h(h), dtype_code(d_in), _dptr(d_in), _dptr(d_out), int(cta), int(round), int(detail),
                                  clk.ctypes.data, len(clk), terms.ctypes.data, xo.ctypes.data, n_loads_max,
                                  ctypes.byref(nl), ctypes.byref(rot), _stream(stream)), "syk_apply_H_trace")
    n = 2 * nl.value
    c = clk.astype(np.int64)
    return {"n_loads": nl.value, "rot": rot.value, "issue": c[:n], "before_wait": c[n:2 * n], "after_wait": c[2 * n:3 * n], "first_decoded": c[3 * n:4 * n], "first_issued": c[4 * n:5 * n], "all_issued": c[5 * n:6 * n],
            "arrived": c[6 * n:7 * n],
            "load_terms": terms[:nl.value].copy(), "load_xo": xo[:nl.value].copy()}


def syk_set_lockstep(epoch_len, lag):
    _check(_lib.syk_set_lockstep(int(epoch_len), int(lag)), "syk_set_lockstep")


def syk_set_cuda_graphs(on):
    _check(_lib.syk_set_cuda_graphs(1 if on else 0), "syk_set_cuda_graphs")


def syk_launch_count(reset=False):
    return int(_lib.syk_launch_count(1 if reset else 0))


def syk_profile_enable(on):
    _check(_lib.syk_profile_enable(1 if on else 0), "syk_profile_enable")


def syk_profile_read(reset=True):
    """(summed apply_H device time in ms, number of timed apply_H launches)."""
    ms, n = ctypes.c_double(), ctypes.c_int64()
    _check(_lib.syk_profile_read(ctypes.byref(ms), ctypes.byref(n), 1 if reset else 0), "syk_profile_read")
    return ms.value, n.value


def syk_microbench_workspace_bytes():
    return int(_lib.syk_microbench_workspace_bytes())


def syk_microbench(kind, arg0, arg1, d_buf, d_work, stream=None):
    """One on-chip peak measurement (include/syk.h); returns {"ms", "cycles", "units", "lds_bytes"}."""
    res = (ctypes.c_double * 6)()
    nb = 0 if d_buf is None else d_buf.numel() * d_buf.element_size()
    _check(_lib.syk_microbench(int(kind), int(arg0), int(arg1), 0 if d_buf is None else _dptr(d_buf), nb, _dptr(d_work),
                               d_work.numel() * d_work.element_size(), res, _stream(stream)), "syk_microbench")
    return {"ms": res[0], "cycles": res[1], "units": res[2], "lds_bytes": res[3], "cycles_even": res[4],
            "cycles_odd": res[5]}


def syk_version():
    return int(_lib.syk_version())
