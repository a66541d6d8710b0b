"""N > 1 path on CPU: world-size-2 (and 3, ragged) `gloo` runs of the energy sharding that bench.py --gpus N uses.

The data path has no collective (energy points are independent, PAPER.md L204/L210/L262); what is tested is the
rank -> energy partition, the gather of T(E) back into global energy order, and the max-over-ranks timing reduce.
The per-rank "solve" is replaced by the oracle on a tiny problem so that the gathered T(E) can be compared with the
single-process result element by element.
"""
import os
import socket

import numpy as np
import pytest

torch = pytest.importorskip("torch")
import torch.distributed as dist  # noqa: E402
import torch.multiprocessing as mp  # noqa: E402

from paper_1812_01396_b200 import inputs, sharding  # noqa: E402


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, n_total, out_dir):
    from oracle import dense
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        p = inputs.random_problem(4, 3, n_total, 2, seed=7)
        idx = sharding.energy_indices(n_total, rank, world)
        T_local = []
        for e in idx:
            r = dense.solve_energy(p.E[e], p.H_diag, p.H_upper, p.S_diag, p.S_upper, p.Sigma_L[e], p.Sigma_R[e],
                                   p.Inj_first[e], None)
            T_local.append(r["T_LR"])
        T = sharding.gather_transmission(np.array(T_local), n_total, rank, world)
        tmax = sharding.max_over_ranks(10.0 + rank, world)
        np.save(os.path.join(out_dir, f"T_{rank}.npy"), T)
        np.save(os.path.join(out_dir, f"t_{rank}.npy"), np.array([tmax]))
    finally:
        dist.destroy_process_group()


def _bcast_worker(rank, world, port, out_dir):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        p = inputs.random_problem(3, 4, 1, 1, seed=9)
        names = ("H_diag", "H_upper", "S_diag", "S_upper")
        if rank == 0:
            ts = [torch.from_numpy(getattr(p, k).copy()) for k in names]
        else:
            ts = [torch.zeros(getattr(p, k).shape, dtype=torch.complex128) for k in names]
        sharding.broadcast_hamiltonian(ts, 0, world)
        ok = all(np.array_equal(t.numpy(), getattr(p, k)) for t, k in zip(ts, names))
        np.save(os.path.join(out_dir, f"ok_{rank}.npy"), np.array([ok]))
    finally:
        dist.destroy_process_group()


def test_hamiltonian_broadcast_replicates_rank0_data(tmp_path):
    port = _free_port()
    mp.spawn(_bcast_worker, args=(2, port, str(tmp_path)), nprocs=2, join=True)
    for r in range(2):
        assert bool(np.load(tmp_path / f"ok_{r}.npy")[0])


@pytest.mark.parametrize("world,n_total", [(2, 6), (2, 5), (3, 7)])
def test_energy_sharding_gather_matches_single_process(tmp_path, world, n_total):
    from oracle import dense
    port = _free_port()
    mp.spawn(_worker, args=(world, port, n_total, str(tmp_path)), nprocs=world, join=True)
    p = inputs.random_problem(4, 3, n_total, 2, seed=7)
    _, T_ref = dense.solve_all(p)
    for r in range(world):
        T = np.load(tmp_path / f"T_{r}.npy")
        assert np.array_equal(T, T_ref)                   # same arithmetic on every rank: bit-identical
        assert float(np.load(tmp_path / f"t_{r}.npy")[0]) == 10.0 + world - 1


def test_partition_is_exact_cover():
    for world in (1, 2, 3, 4, 8):
        for n in (0, 1, 7, 8, 64):
            got = np.sort(np.concatenate([sharding.energy_indices(n, r, world) for r in range(world)]))
            assert np.array_equal(got, np.arange(n))
            assert sum(sharding.local_count(n, r, world) for r in range(world)) == n
    with pytest.raises(ValueError):
        sharding.energy_indices(4, 2, 2)
