"""N > 1 path on CPU: world_size-2 `gloo` run of the replica sharding (realizations are
independent, no data-path collective).  The per-realization compute is replaced by the ORACLE's
same-psi OTOC so that the gathered array can be checked value by value; the product compute (binding.syk_otoc)
needs a GPU and is covered by tests/test_gpu_parity.py."""
import os
import socket

import numpy as np
import pytest

from paper_2311_00639_b200 import replicas


def test_round_robin_assignment_is_a_partition():
    for n in (0, 1, 5, 100):
        for w in (1, 2, 3, 8):
            parts = [replicas.realizations_of_rank(n, r, w) for r in range(w)]
            assert sorted(x for p in parts for x in p) == list(range(n))
            assert max(len(p) for p in parts) - min(len(p) for p in parts) <= 1
    with pytest.raises(ValueError):
        replicas.realizations_of_rank(4, 2, 2)


def test_gather_single_process_and_missing():
    F = replicas.run_replicas(lambda r: np.array([r, 2 * r + 1j]), 3, 2, rank=0, world_size=1)
    assert np.array_equal(F, np.array([[0, 1j], [1, 2 + 1j], [2, 4 + 1j]]))
    with pytest.raises(RuntimeError):
        replicas.gather_curves({0: np.zeros(2)}, 2, 2)


def test_normalised_average():
    F = np.array([[2.0, 1.0], [4.0, 1.0]], dtype=complex)
    per, ratio = replicas.normalised_average(F)
    assert np.allclose(per, [1.0, 0.375]) and np.allclose(ratio, [1.0, 1.0 / 3.0])


def _oracle_curve(N, k, seed, r, t_grid, beta):
    from oracle import evolve as oev, otoc as ootoc, rng as orng
    from paper_2311_00639_b200 import inputs
    q, J, _ = orng.sample_couplings(N, inputs.bernoulli_p(N, k), seed, r)
    prop = oev.ExactPropagator(N, q, J)
    return ootoc.otoc_same_psi(prop, N, N - 1, N - 2, beta, t_grid, orng.random_state(N, seed, r))


def _worker(rank, world, port, out_dir):
    import torch.distributed as dist
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    t_grid = np.array([0.0, 1.0, 2.0])
    F = replicas.run_replicas(lambda r: _oracle_curve(8, 4, 3, r, t_grid, 2.0), 5, len(t_grid))
    np.save(os.path.join(out_dir, f"F_{rank}.npy"), F)
    dist.barrier()
    dist.destroy_process_group()


def test_world_size_2_gloo(tmp_path):
    import torch.multiprocessing as mp
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    mp.spawn(_worker, args=(2, port, str(tmp_path)), nprocs=2, join=True)
    F0, F1 = np.load(tmp_path / "F_0.npy"), np.load(tmp_path / "F_1.npy")
    assert np.array_equal(F0, F1)                      # every rank holds the full result
    t_grid = np.array([0.0, 1.0, 2.0])
    ref = np.stack([_oracle_curve(8, 4, 3, r, t_grid, 2.0) for r in range(5)])
    assert np.array_equal(F0, ref)                     # same code on the same inputs: bitwise
    per, ratio = replicas.normalised_average(F0)
    assert abs(per[0] - 1.0) < 1e-14 and abs(ratio[0] - 1.0) < 1e-14
