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


# ---------------------------------------------------------------------------------------------------------
# ONE energy batch on TWO GPUs, one block column of A^-1 per GPU
# ---------------------------------------------------------------------------------------------------------
# computing the first and the last block column of A^-1 "naturally scale[s] to two accelerators"; L175:
# R and Cy are built on the accelerators holding the first / last partition, z is solved for and distributed.
#
# Partition (world = 2, or pairs of ranks of a larger job):  rank 0 of the pair runs the first-column sweep (Q_i), rank 1
# the last-column sweep (P_i), both with a full replica of H and S.  Exchange: the corner blocks (blocks 1 and nb of each
# column, [n_energy][2][bs][bs] per rank) by one all-gather inside the pair; the 2bs x 2bs corner system is then built and
# solved REDUNDANTLY on both ranks (it needs all four corner blocks and costs ~1/nb of a sweep), so no broadcast of its
# solution is needed; each rank forms its share of X = Q w_top + P w_bot and one sum-all-reduce inside the pair completes
# X on both.  Bytes crossing the link per energy: 4 bs^2 * 16 (corners) + nb * bs * nrhs * 16 (X shares).
#
# `engine` supplies the per-rank work, so that the same orchestration runs over the CUDA library on GPUs (nccl) and over
# a CPU stand-in in the world-size-2 gloo test:
#     engine.sweep(column)                           a0-a4 for that block column
#     engine.corners(column)        -> tensor [n_energy, 2, bs, bs]
#     engine.post(column, peer_corners) -> (X_part tensor [n_energy, n, nrhs], T numpy [n_energy])

def column_of_rank(rank: int) -> int:
    """Which block column a rank of a pair owns: even ranks the first (Q), odd ranks the last (P)."""
    return rank & 1


def column_split_solve(engine, rank: int, group=None):
    """Runs the two-GPU split of one energy batch on this rank and returns (X, T) complete on both ranks of the pair.
    `group`: the process group of the pair (None = the default group, which must then have exactly 2 ranks)."""
    import torch
    import torch.distributed as dist
    col = column_of_rank(rank)
    engine.sweep(col)
    mine = engine.corners(col).contiguous()
    both = [torch.empty_like(mine), torch.empty_like(mine)]
    dist.all_gather([torch.view_as_real(t) for t in both], torch.view_as_real(mine), group=group)
    X_part, T = engine.post(col, both[1 - col])
    if X_part is not None:
        dist.all_reduce(torch.view_as_real(X_part), op=dist.ReduceOp.SUM, group=group)
    return X_part, T


class LibraryColumnEngine:
    """The CUDA library behind column_split_solve: one SplitSolve handle per rank, device tensors, the current stream."""

    def __init__(self, ss, E, Sigma_L, Sigma_R, Inj_first, Inj_last=None):
        self.ss, self.E = ss, E
        self.args = (Sigma_L, Sigma_R, Inj_first, Inj_last)

    def sweep(self, column):
        self.ss.sweep_column(self.E, column)

    def corners(self, column):
        return self.ss.corner_blocks(column)

    def post(self, column, peer):
        X = self.ss.post_column(column, peer.contiguous(), *self.args)
        return X, self.ss.transmission()


# ---------------------------------------------------------------------------------------------------------
# SURVEY.md 8(f2), second half: ONE energy batch on 2^k GPUs, the device split along the transport axis
# ---------------------------------------------------------------------------------------------------------
# PAPER.md L167 ("horizontal split into two halves"), L169 (SPIKE: "power of 2" partitions, merged recursively): every rank
# of a team owns a contiguous run of blocks and only ITS slices of H and S.  Per rank: sweep of the sub-device (first / last
# block column of its own inverse); then log2(world) merge levels: at level l teams of 2^(l+1) ranks join their top and
# bottom halves through the two bs x bs interface systems of include/splitsolve.h (ss_merge_partition) -- every rank of the
# team needs the LAST block of both columns held by the last rank of the top half and the FIRST block held by the first rank of
# the bottom half, solves the interface systems redundantly and updates its own rows; finally the corner blocks (first
# rank's first, last rank's last) go to everybody, the corner system and T(E) are computed redundantly and every rank forms
# X for its own rows.  X ends up distributed by rows (no reduction).  What crosses the link: per level and rank 4 blocks per
# energy in an all-gather (every rank contributes its two edge block pairs), i.e. world * 4 bs^2 * 16 B received.
#
# `engine` (per rank): sweep(); edges() -> tensor [2, n_energy, 2, bs, bs] (first / last block of the first and last
# column); merge(part, iface [n_energy, 2, 2, bs, bs], boundary) with boundary = global index h of the first block of the
# bottom half (the coupling blocks are S_upper[h-1], H_upper[h-1]); post(corners [n_energy, 2, 2, bs, bs]) -> (X_rows, T).

def split_blocks(nb: int):
    """Blocks of the top half: h = ceil(nb / 2); the bottom half gets the rest (both >= 1 for nb >= 2)."""
    return (nb + 1) // 2


def partition_bounds(nb: int, world: int, lo: int = 0):
    """[(lo, hi)) block ranges of `world` = 2^k partitions by recursive halving (the merge tree splits the same way)."""
    if world < 1 or world & (world - 1):
        raise ValueError("the number of partitions must be a power of 2 (PAPER.md L169)")
    if world == 1:
        return [(lo, lo + nb)]
    h = split_blocks(nb)
    return partition_bounds(h, world // 2, lo) + partition_bounds(nb - h, world // 2, lo + h)


def merge_plan(nb: int, world: int, rank: int):
    """The merge levels of `rank`: list of (part, rank of the top half's last partition, rank of the bottom half's first
    partition, boundary block index)."""
    bounds = partition_bounds(nb, world)
    plan = []
    size = 2
    while size <= world:
        r0 = (rank // size) * size
        mid = r0 + size // 2
        plan.append((0 if rank < mid else 1, mid - 1, mid, bounds[mid][0]))
        size *= 2
    return plan


def _all_gather(t, group):
    import torch
    import torch.distributed as dist
    t = t.contiguous()
    out = [torch.empty_like(t) for _ in range(dist.get_world_size(group))]
    dist.all_gather([torch.view_as_real(x) for x in out], torch.view_as_real(t), group=group)
    return out


def spatial_split_solve(engine, nb: int, rank: int, world: int = 2, group=None):
    """Runs the spatial split on this rank of a team of `world` = 2^k ranks (rank = index inside the team) and returns
    (X_rows of this rank's blocks, T)."""
    import torch
    engine.sweep()
    for part, top_last, bottom_first, boundary in merge_plan(nb, world, rank):
        edges = _all_gather(engine.edges(), group)                       # [world] x [2, nE, 2, bs, bs]
        iface = torch.stack([edges[top_last][1], edges[bottom_first][0]], dim=1)      # [nE, 2, 2, bs, bs]
        engine.merge(part, iface, boundary)
    edges = _all_gather(engine.edges(), group)
    corners = torch.stack([edges[0][0], edges[world - 1][1]], dim=1)
    return engine.post(corners)


class LibraryPartitionEngine:
    """The CUDA library behind spatial_split_solve: a SplitSolve handle created for THIS rank's sub-device (with its
    slices of H and S registered), `couple(h)` returning the device tensors (S_upper[h-1], H_upper[h-1]) of a boundary,
    and the (replicated) boundary inputs."""

    def __init__(self, ss, E, couple, Sigma_L, Sigma_R, Inj_first, Inj_last=None):
        self.ss, self.E, self.couple = ss, E, couple
        self.args = (Sigma_L, Sigma_R, Inj_first, Inj_last)

    def sweep(self):
        self.ss.sweep_partition(self.E)

    def edges(self):
        import torch
        return torch.stack([self.ss.edge_blocks(0), self.ss.edge_blocks(1)])

    def merge(self, part, iface, boundary):
        S_c, H_c = self.couple(boundary)
        self.ss.merge_partition(part, iface.contiguous(), S_c, H_c)

    def post(self, corners):
        X = self.ss.post_partition(corners.contiguous(), *self.args)
        return X, self.ss.transmission()
