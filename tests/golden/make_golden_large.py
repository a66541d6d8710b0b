"""Writes tests/golden/c3_fingerprint.txt / c4_fingerprint.txt: Tier B (oracle/banded.py, LU with partial pivoting of
the FULL matrix T of Eq. 5 in band storage -- the plain definition) results for ONE energy point of
BASELINE.json config 3 (bs=2048, nb=32) resp. config 4 (bs=4096, nb=24).  Calls ONLY oracle/ and the seeded input
generators, never the CUDA path.  Run from the repo root (host RAM: C3 ~ 20 GB, C4 ~ 50 GB; hours of CPU time):

    python tests/golden/make_golden_large.py C3 [--energy 5] [--threads 4]
    python tests/golden/make_golden_large.py C4 [--energy 2] [--threads 4]

What is stored (a compact fingerprint; the full X of one energy is 0.27 / 0.81 GB):
  * T_LR = Re Tr(Gamma_L G_1N Gamma_R G_1N^H) from the banded solve of the whole last block column (bs right-hand sides);
  * for N_XCOLS fixed columns of Inj: ||X[:, c]||_2, the projection r^H X[:, c] on a seeded random vector r (depends on
    every row), and X on N_ROWS seeded rows spread over all blocks plus the first and last 4 rows of the device;
  * ||G_1N||_F and G_1N on a seeded sample of positions.
Every value is written with repr() (round-trips exactly).
"""
import argparse
import os
import sys
import time

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, os.path.dirname(os.path.dirname(HERE)))

from oracle import banded  # noqa: E402
from paper_1812_01396_b200 import inputs  # noqa: E402

N_XCOLS, N_ROWS, N_GPOS = 16, 256, 2048
DEFAULT_ENERGY = {"C3": 5, "C4": 2}


def sample_plan(cfg):
    """The seeded sample (shared with the test through this function's arguments only: the test re-derives it from the
    header of the file)."""
    rng = np.random.default_rng([cfg.seed, 9001, cfg.bs])
    n = cfg.nb * cfg.bs
    x_cols = np.sort(rng.choice(cfg.nrhs, size=N_XCOLS, replace=False))
    rows = np.unique(np.concatenate([rng.integers(0, n, size=N_ROWS), np.arange(4), np.arange(n - 4, n)]))
    r = rng.standard_normal(n) + 1j * rng.standard_normal(n)
    gpos = np.stack([rng.integers(0, cfg.bs, size=N_GPOS), rng.integers(0, cfg.bs, size=N_GPOS)], axis=1)
    return x_cols, rows, r, gpos


class LazyBlocks:
    """A block stack that generates block i on access (input plumbing only: config 4's H and S are 25 GB)."""

    def __init__(self, fn, count):
        self.fn, self.count = fn, count

    def __len__(self):
        return self.count

    def __getitem__(self, i):
        if not 0 <= i < self.count:
            raise IndexError(i)
        return self.fn(i)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("config", choices=["C3", "C4", "C2"])
    ap.add_argument("--energy", type=int, default=None)
    ap.add_argument("--threads", type=int, default=4)
    ap.add_argument("--out", default=None)
    a = ap.parse_args()
    cfg = inputs.CONFIGS[a.config]
    e = DEFAULT_ENERGY.get(a.config, 0) if a.energy is None else a.energy
    t0 = time.perf_counter()
    Hd = LazyBlocks(lambda i: inputs.h_diag_block(cfg.seed, i, cfg.bs), cfg.nb)
    Hu = LazyBlocks(lambda i: inputs.h_upper_block(cfg.seed, i, cfg.bs), cfg.nb - 1)
    Sd = LazyBlocks(lambda i: inputs.s_diag_block(cfg.seed, i, cfg.bs), cfg.nb)
    Su = LazyBlocks(lambda i: inputs.s_upper_block(cfg.seed, i, cfg.bs), cfg.nb - 1)
    E = inputs.energy_grid(cfg.n_energy, cfg.e_lo, cfg.e_hi, cfg.eta)[e]
    sl, sr = inputs.sigma_block(cfg.seed, e, cfg.bs, "L"), inputs.sigma_block(cfg.seed, e, cfg.bs, "R")
    inj = inputs.inj_block(cfg.seed, e, cfg.bs, cfg.nrhs)
    x_cols, rows, r, gpos = sample_plan(cfg)
    print(f"inputs {time.perf_counter() - t0:.1f} s", flush=True)
    res = banded.solve_energy_columns(E, Hd, Hu, Sd, Su, sl, sr, inj, None,
                                      x_cols=x_cols, chunk=16, threads=a.threads)
    dt = time.perf_counter() - t0
    print(f"banded solve done {dt:.1f} s, T_LR = {res['T_LR']!r}", flush=True)
    X, G = res["X_cols"], res["G_1N"]
    out = a.out or os.path.join(HERE, f"{a.config.lower()}_fingerprint.txt")
    with open(out, "w") as f:
        f.write(f"# Tier B fingerprint of BASELINE.json config {a.config} (bs={cfg.bs} nb={cfg.nb} nrhs={cfg.nrhs} seed {cfg.seed}), "
                f"energy index {e}; oracle/banded.py solve_energy_columns (zgbtrf/zgbtrs on the full matrix T, Eq. 5 PAPER.md L82);\n"
                f"# written by tests/golden/make_golden_large.py in {dt:.0f} s on {os.cpu_count()} host cores\n")
        f.write(f"config {a.config}\nenergy_index {e}\nE {float(E.real)!r} {float(E.imag)!r}\n")
        f.write(f"T_LR {float(res['T_LR'])!r}\nT_LR_imag {float(res['T_LR_complex'].imag)!r}\n")
        f.write(f"G1N_fro {float(np.linalg.norm(G))!r}\n")
        for j, c in enumerate(x_cols):
            pr = np.vdot(r, X[:, j])
            f.write(f"xcol {int(c)} {float(np.linalg.norm(X[:, j]))!r} {float(pr.real)!r} {float(pr.imag)!r}\n")
        for j, c in enumerate(x_cols):
            for i in rows:
                v = X[i, j]
                f.write(f"x {int(i)} {int(c)} {float(v.real)!r} {float(v.imag)!r}\n")
        for (i, j) in gpos:
            v = G[i, j]
            f.write(f"g {int(i)} {int(j)} {float(v.real)!r} {float(v.imag)!r}\n")
    print("wrote", out, flush=True)


if __name__ == "__main__":
    main()
