"""Oracle for the retarded Green function of PAPER.md:214-218.

Test infrastructure only (see oracle/__init__.py).

    G_R(t) = Re G(t)/G(0),
    G(t)   = <psi| e^{(it - b/2)H} g_n e^{-iHt} g_n e^{-bH/2} |psi>            (n = N-1 there)

In terms of E(tau) = exp(-i tau H)  (DESIGN.md R-TAU):

    G(t) = psi^dagger E(-t - i b/2) g_n E(t) g_n E(-i b/2) psi

`green_same_psi` evaluates the sandwich for one given psi, factor by factor in the order printed (what the CUDA
pipeline is compared with); `green_exact_trace` replaces <psi|.|psi> by Tr(.)/D with dense matrices.
"""
import numpy as np

from . import hamiltonian, majorana


def green_same_psi(prop, N, n, beta, t_grid, psi, gamma_norm=majorana.GAMMA_PAULI):
    """Un-normalised complex G(t_k) for the given psi.  prop: object with .apply(tau, v)."""
    g = lambda v: hamiltonian.apply_gamma(N, n, v, gamma_norm)
    psi = np.asarray(psi, dtype=np.complex128)
    out = np.empty(len(t_grid), dtype=np.complex128)
    for k, t in enumerate(t_grid):
        r = prop.apply(-1j * beta / 2.0, psi)          # e^{-bH/2} psi
        r = g(r)
        r = prop.apply(t, r)                           # e^{-iHt}
        r = g(r)
        r = prop.apply(-t - 1j * beta / 2.0, r)        # e^{(it - b/2)H}
        out[k] = np.vdot(psi, r)
    return out


def green_exact_trace(H, g, beta, t_grid):
    """Tr[e^{(it-b/2)H} g e^{-iHt} g e^{-bH/2}]/D with dense matrices (tiny N only)."""
    w, U = np.linalg.eigh(H)
    E = lambda tau: (U * np.exp(-1j * complex(tau) * w)) @ U.conj().T
    D = H.shape[0]
    return np.array([np.trace(E(-t - 1j * beta / 2.0) @ g @ E(t) @ g @ E(-1j * beta / 2.0)) / D for t in t_grid])
