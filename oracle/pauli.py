"""Oracle for generic sums of Pauli strings on a spin chain (the operator algebra of
PAPER.md:257-299 is not specific to SYK).

Test infrastructure only (see oracle/__init__.py).

A spin operator is a sum of strings  lambda sigma_{i_{L-1}} (x) ... (x) sigma_{i_0}.  The library's
tuple (x, z, c) means  c * prod_q (Z^{z_q} X^{x_q})  on qubit q (Z to the left of X on every site), qubit 0 the
least significant bit of the basis index (R-ENDIAN).  Here that product is written out with Kronecker products of
2 x 2 matrices -- no bit masks act on vectors.
"""
import numpy as np

from . import majorana

I2, SX, SZ = majorana.I2, majorana.SX, majorana.SZ


def string_matrix(L, x, z, c=1.0):
    """Dense 2^L x 2^L matrix of c * (x)_q Z^{z_q} X^{x_q}; the left-most Kronecker factor is the top qubit."""
    m = np.ones((1, 1), dtype=np.complex128)
    for q in range(L - 1, -1, -1):
        site = I2
        if (z >> q) & 1:
            site = site @ SZ
        if (x >> q) & 1:
            site = site @ SX
        m = np.kron(m, site)
    return complex(c) * m


def apply_string(L, x, z, c, v):
    """c * (x)_q Z^{z_q} X^{x_q} applied to the vector v of 2^L amplitudes WITHOUT forming the 2^L x 2^L matrix: the vector is
    viewed as an L-index tensor (index q = qubit q) and the 2 x 2 factor of every site is contracted with its own index --
    the Kronecker product of PAPER.md:259 applied factor by factor (for vectors too long for `string_matrix`; pinned against
    it in tests/test_oracle_pins.py)."""
    t = np.asarray(v, dtype=np.complex128).reshape((2,) * L)      # C order: axis a = qubit L - 1 - a
    for q in range(L):
        site = I2
        if (z >> q) & 1:
            site = site @ SZ
        if (x >> q) & 1:
            site = site @ SX
        if site is not I2:
            t = np.moveaxis(np.tensordot(site, t, axes=([1], [L - 1 - q])), 0, L - 1 - q)
    return complex(c) * t.reshape(-1)


def apply_sum(L, terms, v):
    """sum of apply_string over terms (x, z, c)."""
    out = np.zeros(1 << L, dtype=np.complex128)
    for x, z, c in terms:
        out += apply_string(L, int(x), int(z), c, v)
    return out


def sum_matrix(L, terms):
    """terms: iterable of (x, z, c)."""
    H = np.zeros((1 << L, 1 << L), dtype=np.complex128)
    for x, z, c in terms:
        H += string_matrix(L, int(x), int(z), c)
    return H


def transverse_ising_terms(L, J, h, periodic=True):
    """H = -J sum_i Z_i Z_{i+1} - h sum_i X_i  as (x, z, c) strings."""
    terms = []
    for i in range(L if periodic else L - 1):
        terms.append((0, (1 << i) | (1 << ((i + 1) % L)), -J))
    for i in range(L):
        terms.append((1 << i, 0, -h))
    return terms


def heisenberg_terms(L, Jx, Jy, Jz, periodic=False):
    """H = sum_i Jx X_i X_{i+1} + Jy Y_i Y_{i+1} + Jz Z_i Z_{i+1};  Y = i X Z = -i Z X, so Y_i Y_j = -(Z_i X_i)(Z_j X_j)."""
    terms = []
    for i in range(L if periodic else L - 1):
        j = (i + 1) % L
        pair = (1 << i) | (1 << j)
        terms.append((pair, 0, Jx))
        terms.append((pair, pair, -Jy))
        terms.append((0, pair, Jz))
    return terms
