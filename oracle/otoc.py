"""Oracle O7: the regularised OTOC of PAPER.md:230 (authoritative form; DESIGN.md R-EQ2).

Test infrastructure only (see oracle/__init__.py).

    F(t) = <psi| e^{(it-b/8)H} g_W e^{-(it+b/4)H} g_V e^{(it-b/4)H} g_W e^{-(it+b/4)H} g_V e^{-bH/8} |psi>

with W = gamma_{N-1} and V = gamma_{N-2} in the paper and b = beta.  In terms of
E(tau) = exp(-i tau H):

    F(t) = psi^dagger E(-t - i b/8) g_W E(t - i b/4) g_V E(-t - i b/4) g_W E(t - i b/4) g_V E(-i b/8) psi

OTOC(t) = F(t)/F(0).  `otoc_same_psi` evaluates the sandwich for one given psi (what
the CUDA pipeline is compared with); `otoc_exact_trace` replaces <psi|.|psi> by Tr(.)/D
(the quantity the random state estimates).
"""
import numpy as np

from . import evolve, hamiltonian, majorana


def otoc_same_psi(prop, N, i_W, j_V, beta, t_grid, psi, gamma_norm=majorana.GAMMA_PAULI):
    """Un-normalised complex F(t_k) for the given psi.  prop: object with .apply(tau, v)."""
    gW = lambda v: hamiltonian.apply_gamma(N, i_W, v, gamma_norm)
    gV = lambda v: hamiltonian.apply_gamma(N, j_V, v, gamma_norm)
    out = np.empty(len(t_grid), dtype=np.complex128)
    psi = np.asarray(psi, dtype=np.complex128)
    for n, t in enumerate(t_grid):
        r = prop.apply(-1j * beta / 8.0, psi)
        r = gV(r)
        r = prop.apply(t - 1j * beta / 4.0, r)
        r = gW(r)
        r = prop.apply(-t - 1j * beta / 4.0, r)
        r = gV(r)
        r = prop.apply(t - 1j * beta / 4.0, r)
        r = gW(r)
        r = prop.apply(-t - 1j * beta / 8.0, r)
        out[n] = np.vdot(psi, r)
    return out


def otoc_exact_trace(H, gW, gV, beta, t_grid):
    """Tr[...]/D with dense matrices (tiny N only): the same operator product as `otoc_same_psi`."""
    w, U = np.linalg.eigh(H)
    E = lambda tau: (U * np.exp(-1j * complex(tau) * w)) @ U.conj().T
    D = H.shape[0]
    out = np.empty(len(t_grid), dtype=np.complex128)
    for n, t in enumerate(t_grid):
        M = (E(-t - 1j * beta / 8.0) @ gW @ E(t - 1j * beta / 4.0) @ gV @ E(-t - 1j * beta / 4.0)
             @ gW @ E(t - 1j * beta / 4.0) @ gV @ E(-1j * beta / 8.0))
        out[n] = np.trace(M) / D
    return out


def main_text_trace(H, gW, gV, beta, t):
    """Tr[y W(t) y V y W(t) y V]/D with y = exp(-beta H/4), W(t) = e^{iHt} W e^{-iHt}: the quantity
    Eq. (2) regularises; used to pin the reading R-EQ2 of the garbled third factor."""
    w, U = np.linalg.eigh(H)
    f = lambda c: (U * np.exp(c * w)) @ U.conj().T
    y = f(-beta / 4.0)
    Wt = f(1j * t) @ gW @ f(-1j * t)
    return np.trace(y @ Wt @ y @ gV @ y @ Wt @ y @ gV) / H.shape[0]
