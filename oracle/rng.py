"""Oracle O1: sampling the sparse SYK couplings of Eq. (1).

Test infrastructure only (see oracle/__init__.py).

PAPER.md:32 fixes the distribution -- p_ijkl ~ Bernoulli(p), J_ijkl ~ N(0, 3/(8 p N^3)),
k = (p/N) C(N,4) -- but not the generator.  DESIGN.md "R-RNG" fixes a counter-based one so
that the CUDA library and this oracle can each implement it independently:

    GOLD      = 0x9E3779B97F4A7C15
    fmix(z)   : z ^= z>>30; z *= 0xBF58476D1CE4E5B9; z ^= z>>27; z *= 0x94D049BB133111EB; z ^= z>>31
    absorb(h,w) = fmix((h ^ w) + GOLD)                      (all arithmetic mod 2^64)
    key(seed, realization, stream) = absorb(absorb(absorb(0, seed), realization), stream)
    draw(key, index, d) = absorb(absorb(key, index), d) >> 11        (a 53-bit integer)

Hamiltonian stream = 1.  Quartets i<j<k<l are ranked r = 0,1,... in lexicographic order.
  keep quartet r   iff  draw(key, r, 0) < floor(p * 2^53)            (integer compare; p=1 keeps all)
  J_r = sigma * sqrt(-2 ln u1) * cos(2 pi u2),  u1 = (draw(key,r,1)+1)/2^53,  u2 = draw(key,r,2)/2^53,
  sigma = sqrt(3 / (8 p N^3)).
State stream = 2 (the "Haar-random state" of PAPER.md:212): amplitude b gets
  rho = sqrt(-2 ln u1), psi[b] = rho*cos(2 pi u2) + i*rho*sin(2 pi u2),  u1,u2 from draw(key,b,0), draw(key,b,1),
  then psi is divided by its 2-norm.
"""
import itertools
import math

import numpy as np

MASK64 = (1 << 64) - 1
GOLD = 0x9E3779B97F4A7C15
STREAM_HAMILTONIAN = 1
STREAM_STATE = 2


def fmix(z):
    z &= MASK64
    z ^= z >> 30
    z = (z * 0xBF58476D1CE4E5B9) & MASK64
    z ^= z >> 27
    z = (z * 0x94D049BB133111EB) & MASK64
    z ^= z >> 31
    return z


def absorb(h, w):
    return fmix(((h ^ w) + GOLD) & MASK64)


def make_key(seed, realization, stream):
    return absorb(absorb(absorb(0, seed), realization), stream)


def draw(key, index, d):
    return absorb(absorb(key, index), d) >> 11


# ---- vectorised twin of the scalar functions above (numpy uint64 wraps mod 2^64) ----------------
def _fmix_np(z):
    z = z.copy()
    z ^= z >> np.uint64(30)
    z *= np.uint64(0xBF58476D1CE4E5B9)
    z ^= z >> np.uint64(27)
    z *= np.uint64(0x94D049BB133111EB)
    z ^= z >> np.uint64(31)
    return z


def _absorb_np(h, w):
    with np.errstate(over="ignore"):
        return _fmix_np((h ^ w) + np.uint64(GOLD))


def draw_np(key, index, d):
    """draw() for an array of indices; returns uint64 53-bit integers."""
    index = np.asarray(index, dtype=np.uint64)
    with np.errstate(over="ignore"):
        h = _absorb_np(np.full(index.shape, key, dtype=np.uint64), index)
        h = _absorb_np(h, np.full(index.shape, d, dtype=np.uint64))
    return h >> np.uint64(11)


def sparsity_p(N, k):
    """p = k N / C(N,4)  (k = (p/N) C(N,4)); None/inf-like k<=0 is not allowed."""
    return float(k) * float(N) / float(math.comb(N, 4))


def sample_couplings(N, p, seed, realization):
    """Eq. (1) sampling.  Returns (quartets[int32, T x 4], J[float64, T], ranks[int64, T]) in rank order."""
    if N % 2 or N < 4:
        raise ValueError("N must be even and >= 4")
    if not (0.0 < p <= 1.0):
        raise ValueError("p must be in (0, 1]")
    key = make_key(seed, realization, STREAM_HAMILTONIAN)
    threshold = int(math.floor(p * 2.0 ** 53))
    sigma = math.sqrt(3.0 / (8.0 * p * float(N) ** 3))
    quartets, Js, ranks = [], [], []
    for r, q in enumerate(itertools.combinations(range(N), 4)):   # lexicographic i<j<k<l
        if draw(key, r, 0) < threshold:
            u1 = (draw(key, r, 1) + 1) * 2.0 ** -53
            u2 = draw(key, r, 2) * 2.0 ** -53
            Js.append(sigma * math.sqrt(-2.0 * math.log(u1)) * math.cos(2.0 * math.pi * u2))
            quartets.append(q)
            ranks.append(r)
    return (np.array(quartets, dtype=np.int32).reshape(-1, 4),
            np.array(Js, dtype=np.float64),
            np.array(ranks, dtype=np.int64))


def random_state(N, seed, realization, chunk=1 << 20):
    """Normalised complex Gaussian ("Haar-random") state of dimension 2^(N/2), complex128."""
    D = 1 << (N // 2)
    key = make_key(seed, realization, STREAM_STATE)
    psi = np.empty(D, dtype=np.complex128)
    for lo in range(0, D, chunk):
        idx = np.arange(lo, min(D, lo + chunk), dtype=np.uint64)
        u1 = (draw_np(key, idx, 0).astype(np.float64) + 1.0) * 2.0 ** -53
        u2 = draw_np(key, idx, 1).astype(np.float64) * 2.0 ** -53
        rho = np.sqrt(-2.0 * np.log(u1))
        ang = 2.0 * np.pi * u2
        psi[lo:lo + len(idx)] = rho * np.cos(ang) + 1j * (rho * np.sin(ang))
    return psi / math.sqrt(float(np.vdot(psi, psi).real))
