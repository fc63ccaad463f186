"""Seeded synthetic inputs shared by the tests, the benchmark and the smoke check.

This module holds NONE of the method's arithmetic: no Majorana algebra, no masks, no evolution.  It only
names the BASELINE.json workloads (N, sparsity k, dtype) and draws seeded random vectors / quartet lists with
numpy.  The Hamiltonian sampling of Eq. (1) is part of the method and is implemented twice,
independently (oracle/rng.py and csrc/term_compiler.cpp), not here.

The paper's workloads are themselves synthetic ensembles (Gaussian couplings, Bernoulli sparsity, Haar-random
states), so these configurations are the paper's input distribution, not stand-ins.
"""
import math

import numpy as np

# BASELINE.json `configs`, in order.  k = None means dense (p = 1).
CONFIGS = (
    {"name": "N16_dense_c128", "N": 16, "k": None, "dtype": "c128", "seed": 0, "beta": 5.0,
     "t_grid": tuple(0.5 * i for i in range(21)), "krylov_dim": 20, "i_W": 0, "j_V": 1},
    {"name": "N32_k4_c128_x100", "N": 32, "k": 4, "dtype": "c128", "seed": 0, "beta": 5.0, "realizations": 100,
     "dt": 0.1, "t_max": 10.0},
    {"name": "N48_sweep_c128", "N": 48, "k": (1, 2, 4, 8, None), "dtype": "c128", "seed": 0, "beta": (2.0, 5.0, 10.0),
     "realizations": 20, "krylov_dim": 30},
    {"name": "N56_k4_c128", "N": 56, "k": 4, "dtype": "c128", "seed": 0, "beta": 5.0, "t_max": 8.0},
    {"name": "N64_k2_c64", "N": 64, "k": 2, "dtype": "c64", "seed": 0, "beta": 5.0, "two_pass": True},
)


def bernoulli_p(N, k):
    """Keep-probability of a workload: p = k N / C(N,4) for sparsity k, 1 for dense (k None)."""
    return 1.0 if k is None else float(k) * N / math.comb(N, 4)


def gaussian_state(D, seed, dtype=np.complex128):
    """Normalised iid complex Gaussian vector of length D from numpy's PCG64 (seeded); rounded ONCE to `dtype`
    (DESIGN.md R-C64) and renormalised in that dtype's values."""
    r = np.random.default_rng(seed)
    v = r.standard_normal(D) + 1j * r.standard_normal(D)
    v /= np.linalg.norm(v)
    return v.astype(dtype)


def random_quartets(N, T, seed, sigma=None):
    """T distinct sorted quartets of {0..N-1} chosen uniformly (numpy PCG64) with Gaussian couplings of standard
    deviation sigma (default sqrt(3/(8 p N^3)) with p = T/C(N,4)): a fixed-size stand-in used only by edge-case
    tests (the Bernoulli ensemble itself comes from the method's own sampler)."""
    r = np.random.default_rng(seed)
    total = math.comb(N, 4)
    T = min(T, total)
    seen = set()
    while len(seen) < T:
        q = tuple(sorted(int(a) for a in r.choice(N, size=4, replace=False)))
        seen.add(q)
    quartets = np.array(sorted(seen), dtype=np.int32).reshape(-1, 4)
    if sigma is None:
        sigma = math.sqrt(3.0 / (8.0 * (T / total) * N ** 3))
    return quartets, sigma * r.standard_normal(len(quartets))


def quartets_on_qubits(qubits, T, seed, sigma=1.0):
    """T distinct quartets whose Majoranas live on the given qubits (Majoranas 2q, 2q+1): the structured mask
    sets of the bandwidth sweep (all X-mask bits inside `qubits`)."""
    r = np.random.default_rng(seed)
    maj = sorted(m for q in qubits for m in (2 * q, 2 * q + 1))
    total = math.comb(len(maj), 4)
    T = min(T, total)
    seen = set()
    while len(seen) < T:
        seen.add(tuple(sorted(int(a) for a in r.choice(maj, size=4, replace=False))))
    quartets = np.array(sorted(seen), dtype=np.int32).reshape(-1, 4)
    return quartets, sigma * r.standard_normal(len(quartets))


def sample_indices(D, n, seed):
    """n distinct basis indices in [0, D) (uint64), always including 0 and D-1."""
    r = np.random.default_rng(seed)
    idx = r.integers(0, D, size=n, dtype=np.uint64)
    idx[0], idx[-1] = 0, D - 1
    return np.unique(idx)
