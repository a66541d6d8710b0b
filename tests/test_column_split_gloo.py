"""SURVEY.md 8(f2) on CPU: world-size-2 `gloo` run of the two-GPU split of one energy batch (first block column of A^-1 on
rank 0, last on rank 1: PAPER.md L167, L175).  What is tested is the partition and the exchange logic of
`sharding.column_split_solve` -- which rank sweeps which column, the all-gather of the corner blocks, the redundant corner
solve from own + peer corners, the sum-all-reduce of the X shares -- with the per-rank work done by the oracle's step-by-step
restatement of Algorithm 1 (`oracle/stepwise.py`), and the result compared element by element with the dense oracle."""
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


class OracleColumnEngine:
    """CPU stand-in for the library's column calls: Algorithm 1 / its mirror from oracle/stepwise.py per energy; the corner
    system R = 1 - C [Q P] from the four corner blocks only; X share = own column times its half of w."""

    def __init__(self, p):
        self.p = p
        self.col = {}

    def sweep(self, column):
        from oracle import stepwise
        p = self.p
        fn = stepwise.algorithm1_first_column if column == 0 else stepwise.algorithm1_last_column
        self.col[column] = np.stack([fn(p.E[e], p.H_diag, p.H_upper, p.S_diag, p.S_upper)[0] for e in range(p.n_energy)])

    def corners(self, column):
        c = self.col[column]                                   # [nE, nb, bs, bs]
        return torch.from_numpy(np.ascontiguousarray(np.stack([c[:, 0], c[:, -1]], axis=1)))

    def post(self, column, peer):
        from oracle import dense
        p, bs = self.p, self.p.bs
        own = self.col[column]
        peer = peer.numpy()
        Xs, Ts = [], []
        for e in range(p.n_energy):
            q1, qn = (own[e, 0], own[e, -1]) if column == 0 else (peer[e, 0], peer[e, 1])
            p1, pn = (peer[e, 0], peer[e, 1]) if column == 0 else (own[e, 0], own[e, -1])
            R = np.eye(2 * bs, dtype=np.complex128)
            R[:bs, :bs] -= p.Sigma_L[e] @ q1
            R[:bs, bs:] -= p.Sigma_L[e] @ p1
            R[bs:, :bs] -= p.Sigma_R[e] @ qn
            R[bs:, bs:] -= p.Sigma_R[e] @ pn
            b = np.concatenate([p.Inj_first[e], np.zeros_like(p.Inj_first[e]) if p.Inj_last is None else p.Inj_last[e]])
            Rinv = np.linalg.inv(R)
            w = Rinv @ b
            half = w[:bs] if column == 0 else w[bs:]
            Xs.append((own[e] @ half).reshape(p.nb * bs, -1))
            G1N = q1 @ Rinv[:bs, bs:] + p1 @ Rinv[bs:, bs:]
            Ts.append(dense.transmission_from_G(p.Sigma_L[e], p.Sigma_R[e], G1N).real)
        return torch.from_numpy(np.stack(Xs)), np.array(Ts)


def _worker(rank, world, port, out_dir):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        p = inputs.random_problem(5, 6, 3, 4, seed=41, inj_last=True)
        X, T = sharding.column_split_solve(OracleColumnEngine(p), rank)
        np.save(os.path.join(out_dir, f"X_{rank}.npy"), X.numpy())
        np.save(os.path.join(out_dir, f"T_{rank}.npy"), T)
    finally:
        dist.destroy_process_group()


def test_column_split_world2_matches_dense_oracle(tmp_path):
    from oracle import dense
    port = _free_port()
    mp.spawn(_worker, args=(2, port, str(tmp_path)), nprocs=2, join=True)
    p = inputs.random_problem(5, 6, 3, 4, seed=41, inj_last=True)
    Xo, To = dense.solve_all(p)
    for rank in range(2):
        X = np.load(tmp_path / f"X_{rank}.npy")
        T = np.load(tmp_path / f"T_{rank}.npy")
        assert np.abs(X - Xo).max() <= 1e-10 * np.abs(Xo).max(), rank
        assert np.abs(T - To).max() <= 1e-10 * np.abs(To).max(), rank
    assert sharding.column_of_rank(0) == 0 and sharding.column_of_rank(1) == 1 and sharding.column_of_rank(2) == 0


# ------------------------------------------------------------------------------------------------------
# spatial split (2^k partitions of the device, SPIKE-style merges): sharding.spatial_split_solve on gloo
# ------------------------------------------------------------------------------------------------------
class OraclePartitionEngine:
    """CPU stand-in for the library's partition calls.  Sub-device columns from oracle/stepwise.py on the rank's slices of H, S;
    the merge written out in numpy from the interface equations (include/splitsolve.h, ss_merge_partition); the corner system
    from the four corner blocks."""

    def __init__(self, p, lo, hi):
        self.p = p
        self.Hd, self.Sd = p.H_diag[lo:hi], p.S_diag[lo:hi]
        self.Hu, self.Su = p.H_upper[lo:hi - 1], p.S_upper[lo:hi - 1]

    def sweep(self):
        from oracle import stepwise
        p = self.p
        self.Q = np.stack([stepwise.algorithm1_first_column(p.E[e], self.Hd, self.Hu, self.Sd, self.Su)[0] for e in range(p.n_energy)])
        self.P = np.stack([stepwise.algorithm1_last_column(p.E[e], self.Hd, self.Hu, self.Sd, self.Su)[0] for e in range(p.n_energy)])

    def edges(self):
        e = [np.stack([self.Q[:, i], self.P[:, i]], axis=1) for i in (0, -1)]
        return torch.from_numpy(np.ascontiguousarray(np.stack(e)))

    def merge(self, part, iface, boundary):
        p, iface = self.p, iface.numpy()
        Hc, Sc = p.H_upper[boundary - 1], p.S_upper[boundary - 1]
        for e in range(p.n_energy):
            U = p.E[e] * Sc - Hc
            L = p.E[e] * Sc.conj().T - Hc.conj().T
            one = np.eye(p.bs)
            QTh, PTh, QB1, PB1 = iface[e, 0, 0], iface[e, 0, 1], iface[e, 1, 0], iface[e, 1, 1]
            a = np.linalg.solve(one - PTh @ U @ QB1 @ L, QTh)
            b = -QB1 @ L @ a
            b2 = np.linalg.solve(one - QB1 @ L @ PTh @ U, PB1)
            a2 = -PTh @ U @ b2
            if part == 0:
                Qn = self.Q[e] - self.P[e] @ (U @ b)
                Pn = -self.P[e] @ (U @ b2)
            else:
                Pn = self.P[e] - self.Q[e] @ (L @ a2)
                Qn = -self.Q[e] @ (L @ a)
            self.Q[e], self.P[e] = Qn, Pn

    def post(self, corners):
        from oracle import dense
        p, bs, c = self.p, self.p.bs, corners.numpy()
        Xs, Ts = [], []
        for e in range(p.n_energy):
            q1, p1, qn, pn = c[e, 0, 0], c[e, 0, 1], c[e, 1, 0], c[e, 1, 1]
            R = np.eye(2 * bs, dtype=np.complex128)
            R[:bs, :bs] -= p.Sigma_L[e] @ q1
            R[:bs, bs:] -= p.Sigma_L[e] @ p1
            R[bs:, :bs] -= p.Sigma_R[e] @ qn
            R[bs:, bs:] -= p.Sigma_R[e] @ pn
            b = np.concatenate([p.Inj_first[e], np.zeros_like(p.Inj_first[e]) if p.Inj_last is None else p.Inj_last[e]])
            Rinv = np.linalg.inv(R)
            w = Rinv @ b
            Xs.append((self.Q[e] @ w[:bs] + self.P[e] @ w[bs:]).reshape(-1, b.shape[1]))
            Ts.append(dense.transmission_from_G(p.Sigma_L[e], p.Sigma_R[e], q1 @ Rinv[:bs, bs:] + p1 @ Rinv[bs:, bs:]).real)
        return torch.from_numpy(np.stack(Xs)), np.array(Ts)


def _spatial_worker(rank, world, port, out_dir, nb):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        p = inputs.random_problem(4, nb, 2, 3, seed=43, inj_last=True)
        lo, hi = sharding.partition_bounds(nb, world)[rank]
        X, T = sharding.spatial_split_solve(OraclePartitionEngine(p, lo, hi), nb, rank, world)
        np.save(os.path.join(out_dir, f"X_{rank}.npy"), X.numpy())
        np.save(os.path.join(out_dir, f"T_{rank}.npy"), T)
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("nb,world", [(2, 2), (5, 2), (6, 2), (4, 4), (9, 4)])
def test_spatial_split_matches_dense_oracle(tmp_path, nb, world):
    """The partitions' X rows stacked equal the dense oracle's X; T(E) is complete on every rank.  Two partitions (one merge)
    and four (two merge levels), uneven partitions, and the smallest devices (one block per partition)."""
    from oracle import dense
    port = _free_port()
    mp.spawn(_spatial_worker, args=(world, port, str(tmp_path), nb), nprocs=world, join=True)
    p = inputs.random_problem(4, nb, 2, 3, seed=43, inj_last=True)
    Xo, To = dense.solve_all(p)
    X = np.concatenate([np.load(tmp_path / f"X_{r}.npy") for r in range(world)], axis=1)
    assert X.shape == Xo.shape
    assert np.abs(X - Xo).max() <= 1e-10 * np.abs(Xo).max()
    for rank in range(world):
        assert np.abs(np.load(tmp_path / f"T_{rank}.npy") - To).max() <= 1e-10 * np.abs(To).max()
    assert sharding.partition_bounds(9, 4) == [(0, 3), (3, 5), (5, 7), (7, 9)]
    with pytest.raises(ValueError):
        sharding.partition_bounds(9, 3)
