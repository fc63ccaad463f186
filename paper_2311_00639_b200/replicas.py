"""Disorder realizations over ranks ("... and then performing the disorder average").

Realizations are independent, so the only thing that shards without a data-path exchange is the realization
index ("replicas only").  This module holds the host logic: which rank runs which
realization, and the collection of the per-realization F(t) arrays at the end (`all_gather_object`: result
collection, not a data-path collective).  The compute itself is `binding.syk_otoc` on each rank's own GPU; the
`compute` callable is a parameter so the sharding and gathering can be exercised with the gloo backend on CPU
(tests/test_replicas_gloo.py) -- there is still no CPU implementation of the path.
"""
import numpy as np


def realizations_of_rank(n_realizations, rank, world_size):
    """Round-robin assignment: rank r runs realizations r, r + W, r + 2W, ...  (balanced to within one)."""
    if n_realizations < 0 or world_size < 1 or not (0 <= rank < world_size):
        raise ValueError("bad (n_realizations, rank, world_size)")
    return list(range(rank, n_realizations, world_size))


def gather_curves(local, n_realizations, n_t, group=None):
    """local: {realization: complex array [n_t]} computed by this rank.  Returns on every rank the full
    [n_realizations, n_t] complex128 array.  Uses torch.distributed when it is initialised with more than one
    rank; otherwise `local` must already be complete."""
    import torch.distributed as dist
    parts = [local]
    if dist.is_available() and dist.is_initialized() and dist.get_world_size(group) > 1:
        parts = [None] * dist.get_world_size(group)
        dist.all_gather_object(parts, local, group=group)
    out = np.full((n_realizations, n_t), np.nan + 1j * np.nan, dtype=np.complex128)
    seen = set()
    for part in parts:
        for r, curve in part.items():
            if r in seen:
                raise RuntimeError(f"realization {r} computed twice")
            seen.add(r)
            out[r] = np.asarray(curve, dtype=np.complex128).reshape(n_t)
    if len(seen) != n_realizations:
        raise RuntimeError(f"{n_realizations - len(seen)} realizations missing after the gather")
    return out


def run_replicas(compute, n_realizations, n_t, rank=None, world_size=None, group=None):
    """Runs compute(realization) -> complex array [n_t] for this rank's realizations and gathers all curves."""
    import torch.distributed as dist
    if rank is None or world_size is None:
        if dist.is_available() and dist.is_initialized():
            rank, world_size = dist.get_rank(group), dist.get_world_size(group)
        else:
            rank, world_size = 0, 1
    local = {r: np.asarray(compute(r)) for r in realizations_of_rank(n_realizations, rank, world_size)}
    return gather_curves(local, n_realizations, n_t, group)


def normalised_average(F):
    """OTOC(t) from un-normalised F[r, k] (t_grid[0] must be 0): the per-realization ratio averaged over
    realizations, and the ratio of the averages (DESIGN.md R-F).  Real parts."""
    F = np.asarray(F)
    per = (F / F[:, :1]).real.mean(axis=0)
    ratio = (F.mean(axis=0) / F[:, 0].mean()).real
    return per, ratio


def otoc_disorder_average(N, p, seed, n_realizations, i_W, j_V, beta, t_grid, dtype="c128", opts=None,
                          gamma_norm=0, group=None):
    """The OTOC of PAPER.md:230 for `n_realizations` disorder realizations (seed, r), one Haar-random state each
    (R-PSI), this rank's share on the current CUDA device.  Returns (F[n_realizations, n_t], per-realization-ratio
    average, ratio of averages).  Requires a GPU on every rank."""
    import torch
    from . import binding as B
    tdt = torch.complex128 if dtype == "c128" else torch.complex64
    code = B.SYK_C128 if dtype == "c128" else B.SYK_C64
    D = 1 << (N // 2)
    t_grid = np.ascontiguousarray(t_grid, dtype=np.float64)
    state = {}

    def compute(r):
        h = B.syk_build_hamiltonian(N, p, seed, r, gamma_norm)
        if "wk" not in state:
            state["wk"] = torch.empty(B.syk_otoc_workspace_bytes(h, code, opts), dtype=torch.uint8, device="cuda")
            state["psi"] = torch.empty(D, dtype=tdt, device="cuda")
            state["scratch"] = torch.empty(B.syk_reduce_scratch_bytes(), dtype=torch.uint8, device="cuda")
        B.syk_random_state(N, seed, r, state["psi"], state["scratch"])
        F, _ = B.syk_otoc(h, i_W, j_V, beta, t_grid, state["psi"], state["wk"], opts)
        h.close()
        return F

    F = run_replicas(compute, n_realizations, len(t_grid), group=group)
    per, ratio = normalised_average(F)
    return F, per, ratio
