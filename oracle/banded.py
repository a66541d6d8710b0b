"""Tier B oracle: the SAME full matrix T, held in LAPACK band storage, LU with partial pivoting.
TEST INFRASTRUCTURE.

Still "LU of the whole matrix" (Eq. 5) -- it only skips the structural zeros outside
the band kl = ku = 2*bs - 1 of the block-tridiagonal pattern (Fig. 4 caption, L74), which is what lets
the oracle reach sizes whose dense form (16 n^2 bytes) does not fit on the host.  No block recursion,
no Woodbury.  Uses LAPACK zgbsv (scipy.linalg.lapack).  Pinned to dense.py in tests/test_oracle_pins.py.
"""
from __future__ import annotations

import numpy as np
from scipy.linalg import lapack

from . import dense


def assemble_T_band(E, H_diag, H_upper, S_diag, S_upper, Sigma_L, Sigma_R):
    """T = E*S - H - Sigma^RB (Eq. 5; Sigma blocks per L148) in zgbsv layout:
    ab[kl + ku + i - j, j] = T[i, j], shape (2*kl + ku + 1, n), kl = ku = 2*bs - 1."""
    H_diag = np.asarray(H_diag, dtype=np.complex128)
    nb, bs, _ = H_diag.shape
    n = nb * bs
    kl = ku = 2 * bs - 1
    E = complex(E)
    ab = np.zeros((2 * kl + ku + 1, n), dtype=np.complex128)
    ii, jj = np.meshgrid(np.arange(bs), np.arange(bs), indexing="ij")

    def put(block, r0, c0):
        ab[kl + ku + (r0 - c0) + ii - jj, c0 + jj] = block

    for i in range(nb):
        blk = E * np.asarray(S_diag[i], dtype=np.complex128) - H_diag[i]
        if i == 0:
            blk = blk - np.asarray(Sigma_L, dtype=np.complex128)
        if i == nb - 1:
            blk = blk - np.asarray(Sigma_R, dtype=np.complex128)
        put(blk, i * bs, i * bs)
    for i in range(nb - 1):
        su = np.asarray(S_upper[i], dtype=np.complex128)
        hu = np.asarray(H_upper[i], dtype=np.complex128)
        put(E * su - hu, i * bs, (i + 1) * bs)
        put(E * su.conj().T - hu.conj().T, (i + 1) * bs, i * bs)   # E not conjugated (reading c8)
    return ab, kl, ku


def solve_energy(E, H_diag, H_upper, S_diag, S_upper, Sigma_L, Sigma_R, Inj_first, Inj_last=None,
                 want_G=True):
    """Same contract as dense.solve_energy (X, G_1N, G_N1, T_LR, T_RL), via banded LU (zgbsv)."""
    H_diag = np.asarray(H_diag)
    nb, bs, _ = H_diag.shape
    n = nb * bs
    ab, kl, ku = assemble_T_band(E, H_diag, H_upper, S_diag, S_upper, Sigma_L, Sigma_R)
    b = dense.pad_injection(Inj_first, Inj_last, nb)
    m = b.shape[1]
    extra = 2 * bs if want_G else 0
    rhs = np.zeros((n, m + extra), dtype=np.complex128, order="F")
    rhs[:, :m] = b
    if want_G:
        rhs[n - bs:, m:m + bs] = np.eye(bs)
        rhs[:bs, m + bs:] = np.eye(bs)
    _lub, _piv, sol, info = lapack.zgbsv(kl, ku, ab, rhs, overwrite_ab=True, overwrite_b=True)
    if info != 0:
        raise np.linalg.LinAlgError(f"zgbsv info={info}")
    out = dict(X=np.ascontiguousarray(sol[:, :m]))
    if want_G:
        G_1N = np.ascontiguousarray(sol[:bs, m:m + bs])
        G_N1 = np.ascontiguousarray(sol[n - bs:, m + bs:])
        t_lr = dense.transmission_from_G(Sigma_L, Sigma_R, G_1N)
        t_rl = dense.transmission_from_G(Sigma_R, Sigma_L, G_N1)
        out.update(G_1N=G_1N, G_N1=G_N1, T_LR=t_lr.real, T_RL=t_rl.real, T_LR_complex=t_lr)
    return out


def solve_all(problem, energies=None):
    """Energies `energies` (default all) of a Problem-like object.  Returns X [k, n, m], T_LR [k]."""
    idx = range(len(problem.E)) if energies is None else energies
    Xs, Ts = [], []
    for e in idx:
        il = None if problem.Inj_last is None else problem.Inj_last[e]
        r = solve_energy(problem.E[e], problem.H_diag, problem.H_upper, problem.S_diag, problem.S_upper,
                         problem.Sigma_L[e], problem.Sigma_R[e], problem.Inj_first[e], il)
        Xs.append(r["X"])
        Ts.append(r["T_LR"])
    return np.stack(Xs), np.array(Ts)
