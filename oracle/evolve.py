"""Oracle O6 / O8: the exact propagator E(tau) = exp(-i tau H) for complex tau.

Test infrastructure only (see oracle/__init__.py).

PAPER.md:301 computes exp(-iHt)|Psi> by a (restarted) Krylov method -- an approximation with a
controllable error.  Its oracle is therefore the exact exponential:

* `ExactPropagator` : full diagonalisation, E(tau) = U diag(exp(-i tau w)) U^dagger  (O6).  H commutes
  with the parity operator Z^{(x)L} (every term is a product of four gammas and each gamma flips
  parity; PAPER.md:220 uses the same block structure), so the even- and odd-popcount index sets are
  diagonalised separately -- the same matrix, just permuted into two blocks.
* `chebyshev_propagate` : textbook Chebyshev series exp(z x) = I_0(z) + 2 sum_n I_n(z) T_n(x) on the
  sequential-gamma matvec (O8) -- shares nothing with Lanczos; used where eigh would take minutes.

Complex "time" (DESIGN.md R-TAU):  real time t: tau = t;  exp(-beta H/4): tau = -i beta/4;
exp(-(it+beta/4)H): tau = t - i beta/4;  exp((it-beta/4)H): tau = -t - i beta/4.
"""
import numpy as np

from . import hamiltonian, majorana


def dense_propagator(H, tau):
    """exp(-i tau H) as a dense matrix for Hermitian H (any complex tau)."""
    w, U = np.linalg.eigh(H)
    return (U * np.exp(-1j * complex(tau) * w)) @ U.conj().T


class ExactPropagator:
    """exp(-i tau H) v by diagonalising the two parity blocks of H (N <= ~28)."""

    def __init__(self, N, quartets, J, gamma_norm=majorana.GAMMA_PAULI):
        self.N = N
        D = 1 << (N // 2)
        H = hamiltonian.sparse_hamiltonian(N, quartets, J, gamma_norm)
        idx = np.arange(D, dtype=np.uint64)
        par = hamiltonian._popcount_parity(idx)
        self.blocks = []
        for p in (0, 1):
            sel = np.nonzero(par == p)[0]
            Hb = H[sel][:, sel].toarray()
            assert abs(H[sel][:, np.nonzero(par != p)[0]]).sum() == 0.0, "H does not conserve parity"
            w, U = np.linalg.eigh(Hb)
            self.blocks.append((sel, w, U))

    def eigenvalues(self):
        return np.sort(np.concatenate([w for _, w, _ in self.blocks]))

    def apply(self, tau, v):
        v = np.asarray(v, dtype=np.complex128)
        out = np.empty_like(v)
        for sel, w, U in self.blocks:
            out[sel] = U @ (np.exp(-1j * complex(tau) * w) * (U.conj().T @ v[sel]))
        return out


def spectral_bound(J, gamma_norm=majorana.GAMMA_PAULI):
    """||H|| <= sum_t |J_t| s^4, since each product of four gammas has norm s^4."""
    return float(np.sum(np.abs(J))) * majorana.gamma_scale(gamma_norm) ** 4


def chebyshev_propagate(N, quartets, J, tau, v, gamma_norm=majorana.GAMMA_PAULI, rtol=1e-15):
    """exp(-i tau H) v = sum_n (2 - delta_n0) I_n(z) T_n(H/a) v,  z = -i tau a,  a >= ||H||."""
    from scipy.special import ive
    a = spectral_bound(J, gamma_norm) * 1.0000001
    if a == 0.0:
        return np.asarray(v, dtype=np.complex128).copy()
    z = -1j * complex(tau) * a
    matvec = lambda u: hamiltonian.matvec_sequential(N, quartets, J, u, gamma_norm) / a
    nmax = int(abs(z) * 1.5 + 60)
    # ive(n, z) = iv(n, z) exp(-|Re z|): scaled to avoid overflow; undo the scaling at the end
    coef = np.array([ive(n, z) for n in range(nmax + 1)], dtype=np.complex128)
    t_prev = np.asarray(v, dtype=np.complex128)
    t_cur = matvec(t_prev)
    acc = coef[0] * t_prev + 2.0 * coef[1] * t_cur
    peak = np.max(np.abs(coef))
    for n in range(2, nmax + 1):
        t_prev, t_cur = t_cur, 2.0 * matvec(t_cur) - t_prev
        acc += 2.0 * coef[n] * t_cur
        if n > abs(z) and abs(coef[n]) < rtol * peak and abs(coef[n - 1]) < rtol * peak:
            break
    else:
        raise RuntimeError("Chebyshev series did not converge")
    return acc * np.exp(abs(z.real))
