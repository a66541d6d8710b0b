"""Energy-level sharding over ranks (one process per GPU): the only multi-GPU structure the path has.

Energy points are independent (Fig. 9 caption, L210, L262 "embarrassingly parallel"), so the
energy grid is dealt round-robin over ranks, every rank holds a full replica of H and S, and the data path needs
no collective.  The only exchange is the gather of the per-energy scalars T(E) (8 bytes each) at the end, plus
the max-over-ranks of the step time for bench.py.  Host-side logic only: no method arithmetic here.
"""
from __future__ import annotations

import numpy as np


def energy_indices(n_total: int, rank: int, world: int) -> np.ndarray:
    """Global energy indices owned by `rank`: rank, rank + world, rank + 2*world, ..."""
    if not (0 <= rank < world) or n_total < 0:
        raise ValueError("bad rank/world/n_total")
    return np.arange(rank, n_total, world, dtype=np.int64)


def local_count(n_total: int, rank: int, world: int) -> int:
    return int(len(energy_indices(n_total, rank, world)))


def gather_transmission(T_local, n_total: int, rank: int, world: int, device=None):
    """All-gathers the ranks' T(E) shards and returns them in GLOBAL energy order (numpy float64 [n_total]).
    Shards may be ragged (n_total not a multiple of world): they are padded to the largest shard.
    Uses torch.distributed (nccl on GPUs, gloo on CPU); world == 1 needs no process group."""
    T_local = np.asarray(T_local, dtype=np.float64)
    if len(T_local) != local_count(n_total, rank, world):
        raise ValueError("shard length does not match energy_indices")
    if world == 1:
        return T_local.copy()
    import torch
    import torch.distributed as dist
    width = local_count(n_total, 0, world)               # rank 0 owns the largest shard
    buf = torch.zeros(width, dtype=torch.float64, device=device)
    buf[:len(T_local)] = torch.from_numpy(T_local).to(buf.device)
    out = [torch.empty_like(buf) for _ in range(world)]
    dist.all_gather(out, buf)
    T = np.empty(n_total, dtype=np.float64)
    for r in range(world):
        idx = energy_indices(n_total, r, world)
        T[idx] = out[r][:len(idx)].cpu().numpy()
    return T


def max_over_ranks(value: float, world: int, device=None) -> float:
    """Max of a per-rank scalar (bench.py: step time)."""
    if world == 1:
        return float(value)
    import torch
    import torch.distributed as dist
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def broadcast_hamiltonian(tensors, src: int, world: int):
    """Replicates H and S on every rank ("one ncclBroadcast of H,S at ss_set_hamiltonian"): the analogue of
    the paper's MPI_Bcast of the Hamiltonian and overlap matrices to all nodes before they are copied to the GPUs
    (PAPER.md L212).  `tensors`: the same list of equally shaped torch tensors on every rank (device tensors with nccl, CPU
    tensors with gloo); rank `src` holds the data, the others receive in place.  complex128 is sent as its float64 view.
    One collective per array (4 for H_diag, H_upper, S_diag, S_upper); world == 1 is a no-op."""
    if world == 1:
        return tensors
    import torch
    import torch.distributed as dist
    for t in tensors:
        v = torch.view_as_real(t) if t.is_complex() else t
        dist.broadcast(v, src=src)
    return tensors
