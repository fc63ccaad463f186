"""Oracle for NON-HERMITIAN operators (the library's extensions include the non-Hermitian SYK model;
SURVEY 8(f) NEXT-4).

Test infrastructure only (see oracle/__init__.py).

* `complex_syk_hamiltonian` : Eq. (1) with complex couplings J = J' + i J''.  Eq. (1) is linear in J, so
  H = H[J'] + i H[J''] with both parts the (pinned) Hermitian matrices of oracle/hamiltonian.py.
* `expm_propagate`          : exp(-i tau H) v for ANY square H and complex tau by the dense matrix exponential
  (scipy.linalg.expm, Pade + scaling and squaring).  No diagonalisation: a non-normal H may have no well-conditioned
  eigenbasis (or none at all, see the nilpotent pin).

Pins (tests/test_oracle_pins.py): nilpotent 2 x 2 (exp(-i tau H) = 1 - i tau H exactly), diagonal complex H
(element-wise exponentials), a Hermitian H (equals the eigh propagator of oracle/evolve.py), the group law
E(a) E(b) = E(a + b) for a non-normal H, and the anti-Hermitian case H = i K (K Hermitian): exp(-i t H) = exp(t K).
"""
import numpy as np

from . import hamiltonian, majorana


def complex_syk_hamiltonian(N, quartets, J, gamma_norm=majorana.GAMMA_PAULI):
    """Dense H = sum_t J_t gamma_i gamma_j gamma_k gamma_l with complex J_t (N <= ~22)."""
    J = np.asarray(J, dtype=np.complex128)
    Hre = hamiltonian.sparse_hamiltonian(N, quartets, J.real.copy(), gamma_norm)
    Him = hamiltonian.sparse_hamiltonian(N, quartets, J.imag.copy(), gamma_norm)
    return (Hre + 1j * Him).toarray()


def expm_propagate(H, tau, v):
    """exp(-i tau H) v by the dense matrix exponential."""
    from scipy.linalg import expm
    H = np.asarray(H, dtype=np.complex128)
    return expm(-1j * complex(tau) * H) @ np.asarray(v, dtype=np.complex128)
