"""Oracle O2: Majorana operators as dense matrices built from Kronecker products.

Test infrastructure only (see oracle/__init__.py).

PAPER.md:30 -- "The Majorana operators satisfy the Clifford algebra ... and can be expressed as a
tensor product of Pauli matrices."  Two representations are built here:

* `jw_gammas`   : Jordan-Wigner on L = N/2 qubits (the representation BASELINE.json's north_star
                  names; reading R-JW):
                      gamma_{2q}   = s * Z_0 ... Z_{q-1} X_q
                      gamma_{2q+1} = s * Z_0 ... Z_{q-1} Y_q        Y = [[0,-i],[i,0]]  (R-Y)
* `paper_gammas`: the chiral representation of Eq. (S1) in its compact form (PAPER.md:206-210,
                  DESIGN.md reading R-S1), used only as a cross-check (pin P5).

Basis convention ("most significant bit left-most"; DESIGN.md R-ENDIAN): the basis
index is b = sum_q bit_q 2^q, qubit 0 is the least significant bit, i.e. the RIGHT-most Kronecker
factor.  s = 1 gives {g_m, g_n} = 2 delta_mn; s = 1/sqrt(2) gives delta_mn.
"""
import numpy as np

I2 = np.eye(2, dtype=np.complex128)
SX = np.array([[0, 1], [1, 0]], dtype=np.complex128)
SZ = np.array([[1, 0], [0, -1]], dtype=np.complex128)
SY = np.array([[0, -1j], [1j, 0]], dtype=np.complex128)              # textbook; DESIGN.md R-Y
SY_PRINTED = np.array([[0, 1j], [-1j, 0]], dtype=np.complex128)      # as printed at PAPER.md:198

GAMMA_PAULI = 0   # s = 1
GAMMA_HALF = 1    # s = 1/sqrt(2)


def gamma_scale(gamma_norm):
    if gamma_norm == GAMMA_PAULI:
        return 1.0
    if gamma_norm == GAMMA_HALF:
        return float(np.sqrt(0.5))
    raise ValueError("gamma_norm must be 0 or 1")


def site_operator(op, q, L):
    """op acting on qubit q of an L-qubit chain: 1 (x) ... (x) op (x) ... (x) 1."""
    m = np.ones((1, 1), dtype=np.complex128)
    for site in range(L - 1, -1, -1):          # left-most factor = most significant qubit
        m = np.kron(m, op if site == q else I2)
    return m


def jw_gammas(N, gamma_norm=GAMMA_PAULI):
    """List of the N dense Jordan-Wigner Majorana matrices, each 2^(N/2) x 2^(N/2)."""
    L = N // 2
    s = gamma_scale(gamma_norm)
    out = []
    for n in range(N):
        q = n // 2
        m = np.eye(1 << L, dtype=np.complex128)
        for j in range(q):
            m = m @ site_operator(SZ, j, L)
        m = m @ site_operator(SX if n % 2 == 0 else SY, q, L)
        out.append(s * m)
    return out


def paper_gammas(N, sigma_y=SY_PRINTED):
    """Eq. (S1), compact form, s = 1.  Dimension 2^(N/2); the parity qubit is the
    most significant one, so each gamma is [[0, P],[P, 0]] and gamma_{N-1} = [[0,-i],[i,0]] (x) 1."""
    Lp = N // 2 - 1
    Dp = 1 << Lp
    zero = np.zeros((Dp, Dp), dtype=np.complex128)
    out = []
    for n in range(N - 1):
        P = np.eye(Dp, dtype=np.complex128)
        if n > 0:
            P = P @ site_operator(sigma_y if n % 2 == 1 else SZ, (n - 1) // 2, Lp)
        for i in range((n + 1) // 2, Lp):       # product over i = floor((n+1)/2) .. N/2-2
            P = P @ site_operator(SX, i, Lp)
        out.append(np.block([[zero, P], [P, zero]]))
    one = np.eye(Dp, dtype=np.complex128)
    out.append(np.block([[zero, -1j * one], [1j * one, zero]]))
    return out
