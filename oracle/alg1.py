"""Oracle, pin P6: the paper's own data structure and Algorithm 1, transcribed literally.

Test infrastructure only (see oracle/__init__.py).

* Pauli-letter algebra ("operator product"): an operator is a list of
  (letters, lambda) with letters[q] in {0,1,2,3} = {1, sigma_x, sigma_y, sigma_z} on site q; products use
  the single-site table sigma_a sigma_b = delta_ab 1 + i eps_abc sigma_c with the textbook sigma_y
  (DESIGN.md R-Y).  This is a third construction of H, independent of oracle/hamiltonian.py.
* <bits, coeff> encoding: bits = s_{i_{L-1}} ... s_{i_0}, s_0=00, s_1=01, s_2=11, s_3=10,
  coeff = lambda * i^{#sigma_y}.
* Algorithm 1 in Python for tiny L (`apply_python`) and in C (oracle/alg1.c, built by
  oracle/build.py) for anything larger (`apply_c`), the latter being the timed CPU baseline.
"""
import ctypes
import os

import numpy as np

from . import majorana

# single-site products: _MUL[a][b] = (phase, c) with sigma_a sigma_b = phase * sigma_c
_MUL = {
    0: {0: (1, 0), 1: (1, 1), 2: (1, 2), 3: (1, 3)},
    1: {0: (1, 1), 1: (1, 0), 2: (1j, 3), 3: (-1j, 2)},       # XY = iZ, XZ = -iY
    2: {0: (1, 2), 1: (-1j, 3), 2: (1, 0), 3: (1j, 1)},       # YX = -iZ, YZ = iX
    3: {0: (1, 3), 1: (1j, 2), 2: (-1j, 1), 3: (1, 0)},       # ZX = iY, ZY = -iX
}
_CODE = {0: 0b00, 1: 0b01, 2: 0b11, 3: 0b10}


def jw_gamma_letters(N, n, gamma_norm=majorana.GAMMA_PAULI):
    """gamma_n = s Z_0..Z_{q-1} (X|Y)_q as (letters, lambda)  (DESIGN.md R-JW)."""
    L = N // 2
    q = n // 2
    letters = [3] * q + [1 if n % 2 == 0 else 2] + [0] * (L - q - 1)
    return letters, complex(majorana.gamma_scale(gamma_norm))


def multiply(a, b):
    """(letters_a, lam_a) * (letters_b, lam_b), site by site."""
    la, ca = a
    lb, cb = b
    out, lam = [], ca * cb
    for sa, sb in zip(la, lb):
        ph, sc = _MUL[sa][sb]
        lam *= ph
        out.append(sc)
    return out, lam


def encode(letters, lam):
    """<bits, coeff> of one Pauli string; site 0 occupies the two lowest bits."""
    bits = 0
    for q, s in enumerate(letters):
        bits |= _CODE[s] << (2 * q)
    ny = sum(1 for s in letters if s == 2)
    return bits, lam * (1j ** ny)


def hamiltonian_tuples(N, quartets, J, gamma_norm=majorana.GAMMA_PAULI):
    """Eq. (1) as the paper's list of <bits, coeff> tuples, one per kept quartet."""
    bits = np.zeros(len(J), dtype=np.uint64)
    coeff = np.zeros(len(J), dtype=np.complex128)
    for t, (q, Jt) in enumerate(zip(np.asarray(quartets).reshape(-1, 4), J)):
        op = jw_gamma_letters(N, int(q[0]), gamma_norm)
        for n in q[1:]:
            op = multiply(op, jw_gamma_letters(N, int(n), gamma_norm))
        bt, ct = encode(op[0], op[1] * float(Jt))
        bits[t], coeff[t] = bt, ct
    return bits, coeff


def apply_python(L, bits, coeff, psi):
    """Algorithm 1, line by line.  Pure Python: tiny L only."""
    D = 1 << L
    phi = np.zeros(D, dtype=np.complex128)
    for m in range(D):
        for bt, cf in zip(bits, coeff):
            n = m
            minus = False
            bt = int(bt)
            for i in range(2 * L):                     # "each i-th non-zero bit", from the LSB
                if (bt >> i) & 1:
                    if i % 2 == 0:
                        n ^= 1 << (i // 2)
                    elif (n >> (i // 2)) & 1:
                        minus = not minus
            if not minus:
                phi[m] += cf * psi[n]
            else:
                phi[m] -= cf * psi[n]
    return phi


_LIB = None


def _lib():
    global _LIB
    if _LIB is None:
        from . import build
        path = build.build_alg1()
        lib = ctypes.CDLL(path)
        lib.alg1_apply.argtypes = [ctypes.c_int, ctypes.c_int64, ctypes.c_void_p, ctypes.c_void_p,
                                   ctypes.c_void_p, ctypes.c_void_p, ctypes.c_uint64, ctypes.c_uint64]
        lib.alg1_apply.restype = None
        lib.alg1_num_threads.restype = ctypes.c_int
        _LIB = lib
    return _LIB


def num_threads():
    return int(_lib().alg1_num_threads())


def apply_c(L, bits, coeff, psi, m_begin=0, m_end=None):
    """Algorithm 1 in C (oracle/alg1.c); returns rows [m_begin, m_end) of Phi = S Psi."""
    D = 1 << L
    m_end = D if m_end is None else m_end
    bits = np.ascontiguousarray(bits, dtype=np.uint64)
    coeff = np.ascontiguousarray(coeff, dtype=np.complex128)
    psi = np.ascontiguousarray(psi, dtype=np.complex128)
    assert psi.shape == (D,)
    phi = np.empty(m_end - m_begin, dtype=np.complex128)
    _lib().alg1_apply(L, len(bits), bits.ctypes.data, coeff.ctypes.data, psi.ctypes.data,
                      phi.ctypes.data, m_begin, m_end)
    return phi
