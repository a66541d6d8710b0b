"""Seeded synthetic inputs for the SplitSolve hot path (BASELINE.json `configs`).

This module is the ONE piece of code shared by the CPU oracle's tests and the CUDA path's tests /
bench: it draws random matrices and writes down the perfect-chain recipe, and holds none of the
method's arithmetic (no block sweep, no LU, no Woodbury, no transmission).  It imports neither
`oracle/` nor the CUDA binding.

The matrices stand in for the paper's CP2K Hamiltonians of the Si nanowire / UTB devices
(Fig. 8 caption), which are not available; block shapes follow the paper's
"dense or treated as such" bs x bs blocks.

Recipe:
  * every array comes from its own counter-keyed stream
        rng = numpy.random.default_rng([seed, tag, index])
        g   = rng.standard_normal(shape + (2,));  Z = (g[...,0] + 1j*g[...,1]) * sigma/sqrt(2)
    so that E|z|^2 = sigma^2 and any block can be regenerated alone;
  * tags: 0 H_diag[i], 1 H_upper[i], 2 S_diag[i], 3 S_upper[i], 4/5 Sigma_L Hermitian part / Y [e],
    6/7 Sigma_R [e], 8 Inj[e];
  * "Hermitian Gaussian" = (R + R^H)/2 with R complex Gaussian sigma = 1/sqrt(bs);
  * "energies uniform in [a,b]" = the deterministic midpoint grid E_j = a + (b-a)(j+1/2)/n_E.
"""
from __future__ import annotations

from concurrent.futures import ThreadPoolExecutor
from dataclasses import dataclass
from typing import Optional

import numpy as np

TAG_H_DIAG, TAG_H_UPPER, TAG_S_DIAG, TAG_S_UPPER = 0, 1, 2, 3
TAG_SIGL_HERM, TAG_SIGL_Y, TAG_SIGR_HERM, TAG_SIGR_Y, TAG_INJ = 4, 5, 6, 7, 8


@dataclass(frozen=True)
class Config:
    """One BASELINE.json config: sizes + which generator."""
    name: str
    bs: int
    nb: int
    n_energy: int
    nrhs: int
    kind: str = "random"          # "random" (config-0 generator) or "chain" (perfect chain)
    seed: int = 0
    e_lo: float = -1.0
    e_hi: float = 1.0
    eta: float = 1e-3             # imaginary part of E


# BASELINE.json configs[0..4]
CONFIGS = {
    "C0": Config("C0", bs=16, nb=8, n_energy=4, nrhs=4),
    "C1": Config("C1", bs=64, nb=256, n_energy=64, nrhs=64, kind="chain", e_lo=-1.9, e_hi=1.9, eta=0.0),
    "C2": Config("C2", bs=512, nb=64, n_energy=32, nrhs=128),
    "C3": Config("C3", bs=2048, nb=32, n_energy=8, nrhs=256),
    "C4": Config("C4", bs=4096, nb=24, n_energy=4, nrhs=512),
}


def complex_gaussian(seed: int, tag: int, index: int, shape, sigma: float) -> np.ndarray:
    """Complex Gaussian with E|z|^2 = sigma^2 from the stream keyed (seed, tag, index)."""
    rng = np.random.default_rng([seed, tag, index])
    g = rng.standard_normal(tuple(shape) + (2,))
    z = np.empty(tuple(shape), dtype=np.complex128)
    z.real = g[..., 0]
    z.imag = g[..., 1]
    z *= sigma / np.sqrt(2.0)
    return z


def hermitian_gaussian(seed: int, tag: int, index: int, bs: int) -> np.ndarray:
    r = complex_gaussian(seed, tag, index, (bs, bs), 1.0 / np.sqrt(bs))
    return 0.5 * (r + r.conj().T)


def h_diag_block(seed: int, i: int, bs: int) -> np.ndarray:
    return hermitian_gaussian(seed, TAG_H_DIAG, i, bs)


def h_upper_block(seed: int, i: int, bs: int) -> np.ndarray:
    return complex_gaussian(seed, TAG_H_UPPER, i, (bs, bs), 0.5 / np.sqrt(bs))


def s_diag_block(seed: int, i: int, bs: int) -> np.ndarray:
    s = 0.05 * hermitian_gaussian(seed, TAG_S_DIAG, i, bs)
    s[np.arange(bs), np.arange(bs)] += 1.0
    return s


def s_upper_block(seed: int, i: int, bs: int) -> np.ndarray:
    return 0.02 * complex_gaussian(seed, TAG_S_UPPER, i, (bs, bs), 1.0 / np.sqrt(bs))


def sigma_block(seed: int, e: int, bs: int, side: str) -> np.ndarray:
    """0.3*(Hermitian Gaussian) - i*Y*Y^H/bs : anti-Hermitian part negative semidefinite (retarded)."""
    th, ty = (TAG_SIGL_HERM, TAG_SIGL_Y) if side == "L" else (TAG_SIGR_HERM, TAG_SIGR_Y)
    herm = hermitian_gaussian(seed, th, e, bs)
    y = complex_gaussian(seed, ty, e, (bs, bs), 1.0)
    return 0.3 * herm - 1j * (y @ y.conj().T) / bs


def inj_block(seed: int, e: int, bs: int, nrhs: int) -> np.ndarray:
    return complex_gaussian(seed, TAG_INJ, e, (bs, nrhs), 1.0)


def energy_grid(n_energy: int, lo: float, hi: float, eta: float) -> np.ndarray:
    j = np.arange(n_energy, dtype=np.float64)
    return (lo + (hi - lo) * (j + 0.5) / n_energy) + 1j * eta


@dataclass
class Problem:
    """All inputs of one ss_set_hamiltonian + ss_solve call (host arrays, C-contiguous complex128)."""
    bs: int
    nb: int
    H_diag: np.ndarray      # [nb, bs, bs]
    H_upper: np.ndarray     # [nb-1, bs, bs]   H_{i,i+1}
    S_diag: np.ndarray      # [nb, bs, bs]
    S_upper: np.ndarray     # [nb-1, bs, bs]   S_{i,i+1}
    E: np.ndarray           # [n_energy]
    Sigma_L: np.ndarray     # [n_energy, bs, bs]
    Sigma_R: np.ndarray     # [n_energy, bs, bs]
    Inj_first: np.ndarray   # [n_energy, bs, nrhs]
    Inj_last: Optional[np.ndarray] = None  # [n_energy, bs, nrhs] or None (= zeros)

    @property
    def n_energy(self) -> int:
        return int(self.E.shape[0])

    @property
    def nrhs(self) -> int:
        return int(self.Inj_first.shape[2])


def _stack(fn, count, bs, threads):
    out = np.empty((count, bs, bs), dtype=np.complex128)
    if count == 0:
        return out

    def work(i):
        out[i] = fn(i)
    if threads > 1 and count > 1:
        with ThreadPoolExecutor(max_workers=threads) as ex:
            list(ex.map(work, range(count)))
    else:
        for i in range(count):
            work(i)
    return out


def random_problem(bs: int, nb: int, n_energy: int, nrhs: int, seed: int = 0, e_lo: float = -1.0,
                   e_hi: float = 1.0, eta: float = 1e-3, inj_last: bool = False,
                   threads: int = 1) -> Problem:
    """BASELINE.json config-0 generator at any size."""
    H_diag = _stack(lambda i: h_diag_block(seed, i, bs), nb, bs, threads)
    H_upper = _stack(lambda i: h_upper_block(seed, i, bs), nb - 1, bs, threads)
    S_diag = _stack(lambda i: s_diag_block(seed, i, bs), nb, bs, threads)
    S_upper = _stack(lambda i: s_upper_block(seed, i, bs), nb - 1, bs, threads)
    E = energy_grid(n_energy, e_lo, e_hi, eta)
    Sigma_L = _stack(lambda e: sigma_block(seed, e, bs, "L"), n_energy, bs, threads)
    Sigma_R = _stack(lambda e: sigma_block(seed, e, bs, "R"), n_energy, bs, threads)
    Inj = np.empty((n_energy, bs, nrhs), dtype=np.complex128)
    for e in range(n_energy):
        Inj[e] = inj_block(seed, e, bs, nrhs)
    Inj_last = None
    if inj_last:
        Inj_last = np.empty((n_energy, bs, nrhs), dtype=np.complex128)
        for e in range(n_energy):
            Inj_last[e] = inj_block(seed + 1000003, e, bs, nrhs)
    return Problem(bs, nb, H_diag, H_upper, S_diag, S_upper, E, Sigma_L, Sigma_R, Inj, Inj_last)


def chain_wavevector(E: np.ndarray, t: float) -> np.ndarray:
    """k in (0, pi) with cos k = E/(2t)."""
    return np.arccos(np.real(E) / (2.0 * t))


def perfect_chain_problem(bs: int, nb: int, n_energy: int, t: float = -1.0, e_lo: float = -1.9,
                          e_hi: float = 1.9) -> Problem:
    """BASELINE.json config 1: H_ii = 0, H_{i,i+1} = t*1, S = 1, Sigma_L = Sigma_R = t e^{ik} 1,
    Inj = injected plane wave t (1 - e^{2ik}) 1 in the first block (one column per channel, nrhs = bs).
    Expected (closed form): X_j = e^{ikj} 1 (j = 1..nb) and T(E) = bs."""
    eye = np.eye(bs, dtype=np.complex128)
    H_diag = np.zeros((nb, bs, bs), dtype=np.complex128)
    H_upper = np.broadcast_to(t * eye, (nb - 1, bs, bs)).copy()
    S_diag = np.broadcast_to(eye, (nb, bs, bs)).copy()
    S_upper = np.zeros((nb - 1, bs, bs), dtype=np.complex128)
    E = energy_grid(n_energy, e_lo, e_hi, 0.0)
    k = chain_wavevector(E, t)
    Sigma = (t * np.exp(1j * k))[:, None, None] * eye[None]
    Inj = (t * (1.0 - np.exp(2j * k)))[:, None, None] * eye[None]
    return Problem(bs, nb, H_diag, H_upper, S_diag, S_upper, E, Sigma.copy(), Sigma.copy(),
                   np.ascontiguousarray(Inj), None)


def make_problem(cfg: Config, threads: int = 1) -> Problem:
    if cfg.kind == "chain":
        assert cfg.nrhs == cfg.bs
        return perfect_chain_problem(cfg.bs, cfg.nb, cfg.n_energy, t=-1.0, e_lo=cfg.e_lo, e_hi=cfg.e_hi)
    return random_problem(cfg.bs, cfg.nb, cfg.n_energy, cfg.nrhs, seed=cfg.seed, e_lo=cfg.e_lo,
                          e_hi=cfg.e_hi, eta=cfg.eta, threads=threads)
