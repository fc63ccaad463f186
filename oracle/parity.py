"""Oracle for the parity-block form of the calculation.

Test infrastructure only (see oracle/__init__.py).

H is a sum of products of four gammas, every gamma flips the fermion parity, so H = H_UU (+) H_DD
 and a single gamma maps one block to the other.  The paper uses this to halve the vectors:

    F(t) = <psi_U| e^{(it-b/8)H_UU} g^{UD}_W e^{-(it+b/4)H_DD} g^{DU}_V e^{(it-b/4)H_UU} g^{UD}_W e^{-(it+b/4)H_DD}
                   g^{DU}_V e^{-bH_UU/8} |psi_U>  +  {swap U,D}
    G(t) = <psi_U| e^{(it-b/2)H_UU} g^{UD} e^{-iH_DD t} g^{DU} e^{-bH_UU/2} |psi_U> + {swap U,D}

In the Jordan-Wigner representation of this build (DESIGN.md R-JW) the parity operator is Z^{(x)L}: the blocks are
the index sets of even (sector 0) and odd (sector 1) popcount.  A block is stored on L-1 qubits (DESIGN.md R-BLOCK):
reduced index b' = the low L-1 bits of b, the dropped top bit being  parity(b') xor sector.

Everything here is the plain definition: rows and columns of the full-space matrices (built elsewhere in this
oracle from Kronecker products / monomial rows) are SELECTED; nothing is re-derived with bit masks on the operator.
"""
import numpy as np

from . import hamiltonian, majorana


def sector_indices(L, sector):
    """Full-space index b(b') for b' = 0 .. 2^(L-1)-1 in the given parity sector."""
    bp = np.arange(1 << (L - 1), dtype=np.uint64)
    top = (hamiltonian._popcount_parity(bp) ^ int(sector)).astype(np.uint64)
    return bp | (top << np.uint64(L - 1))


def restrict(v, L, sector):
    """Reduced vector v_s[b'] = v[b(b')]."""
    return np.asarray(v)[sector_indices(L, sector).astype(np.int64)]


def embed(v_s, L, sector):
    """Full-space vector that equals v_s on the sector and zero on the other one."""
    out = np.zeros(1 << L, dtype=np.complex128)
    out[sector_indices(L, sector).astype(np.int64)] = v_s
    return out


def block_hamiltonian(N, quartets, J, sector, gamma_norm=majorana.GAMMA_PAULI):
    """Dense H_ss on the reduced basis, selected from the sparse-by-rows full H (O5).  Also checks that H has no
    matrix element between the sectors."""
    L = N // 2
    H = hamiltonian.sparse_hamiltonian(N, quartets, J, gamma_norm)
    idx = sector_indices(L, sector).astype(np.int64)
    other = sector_indices(L, 1 - sector).astype(np.int64)
    assert abs(H[idx][:, other]).sum() == 0.0, "H does not conserve parity"
    return H[idx][:, idx].toarray()


def block_gamma(N, n, sector_out, gamma_norm=majorana.GAMMA_PAULI):
    """Dense block of gamma_n that maps sector 1 - sector_out to sector_out, on the reduced bases, selected from the
    Kronecker-product matrix (O2)."""
    L = N // 2
    g = majorana.jw_gammas(N, gamma_norm)[n]
    rows = sector_indices(L, sector_out).astype(np.int64)
    cols = sector_indices(L, 1 - sector_out).astype(np.int64)
    assert abs(g[np.ix_(rows, rows)]).sum() == 0.0, "gamma does not flip parity"
    return g[np.ix_(rows, cols)]


class BlockPropagator:
    """exp(-i tau H_ss) on the reduced basis of one sector by full diagonalisation of the block."""

    def __init__(self, N, quartets, J, sector, gamma_norm=majorana.GAMMA_PAULI):
        self.w, self.U = np.linalg.eigh(block_hamiltonian(N, quartets, J, sector, gamma_norm))

    def apply(self, tau, v):
        return self.U @ (np.exp(-1j * complex(tau) * self.w) * (self.U.conj().T @ np.asarray(v, dtype=np.complex128)))


def otoc_block_same_psi(props, N, i_W, j_V, beta, t_grid, psi_s, sector, gamma_norm=majorana.GAMMA_PAULI):
    """One of the two terms of PAPER.md:232 for a reduced state psi_s in `sector`; props[s] = BlockPropagator of
    sector s.  Factor by factor, right to left; the gammas are dense blocks."""
    s, o = int(sector), 1 - int(sector)
    gV_os = block_gamma(N, j_V, o, gamma_norm)      # sector s -> o
    gW_so = block_gamma(N, i_W, s, gamma_norm)      # sector o -> s
    psi_s = np.asarray(psi_s, dtype=np.complex128)
    out = np.empty(len(t_grid), dtype=np.complex128)
    for k, t in enumerate(t_grid):
        r = props[s].apply(-1j * beta / 8.0, psi_s)
        r = gV_os @ r
        r = props[o].apply(t - 1j * beta / 4.0, r)
        r = gW_so @ r
        r = props[s].apply(-t - 1j * beta / 4.0, r)
        r = gV_os @ r
        r = props[o].apply(t - 1j * beta / 4.0, r)
        r = gW_so @ r
        r = props[s].apply(-t - 1j * beta / 8.0, r)
        out[k] = np.vdot(psi_s, r)
    return out


def green_block_same_psi(props, N, n, beta, t_grid, psi_s, sector, gamma_norm=majorana.GAMMA_PAULI):
    """One of the two terms of PAPER.md:220 for a reduced state psi_s in `sector`."""
    s, o = int(sector), 1 - int(sector)
    g_os = block_gamma(N, n, o, gamma_norm)
    g_so = block_gamma(N, n, s, gamma_norm)
    psi_s = np.asarray(psi_s, dtype=np.complex128)
    out = np.empty(len(t_grid), dtype=np.complex128)
    for k, t in enumerate(t_grid):
        r = props[s].apply(-1j * beta / 2.0, psi_s)
        r = g_os @ r
        r = props[o].apply(t, r)
        r = g_so @ r
        r = props[s].apply(-t - 1j * beta / 2.0, r)
        out[k] = np.vdot(psi_s, r)
    return out
