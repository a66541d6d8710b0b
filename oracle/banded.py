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
    ab[kl + ku + i - j, j] = T[i, j], shape (2*kl + ku + 1, n), kl = ku = 2*bs - 1.
    The block stacks are only indexed block by block (H_diag[i], ...), so lazy sequences that generate a block on
    access work too (BASELINE.json config 4: H and S are 25 GB, the band 39 GB).  Column-major, as LAPACK wants it."""
    nb = len(H_diag)
    bs = np.asarray(H_diag[0]).shape[0]
    n = nb * bs
    kl = ku = 2 * bs - 1
    E = complex(E)
    ab = np.zeros((2 * kl + ku + 1, n), dtype=np.complex128, order="F")
    ii, jj = np.meshgrid(np.arange(bs), np.arange(bs), indexing="ij")

    def put(block, r0, c0):
        ab[kl + ku + (r0 - c0) + ii - jj, c0 + jj] = block

    for i in range(nb):
        blk = E * np.asarray(S_diag[i], dtype=np.complex128) - np.asarray(H_diag[i], dtype=np.complex128)
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
    nb = len(H_diag)
    bs = np.asarray(H_diag[0]).shape[0]
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


def factor(E, H_diag, H_upper, S_diag, S_upper, Sigma_L, Sigma_R):
    """LU with partial pivoting (LAPACK zgbtrf) of the full matrix T of Eq. 5 (L82) in band storage.
    Returns (lub, piv, kl, ku) for `solve_factored`."""
    ab, kl, ku = assemble_T_band(E, H_diag, H_upper, S_diag, S_upper, Sigma_L, Sigma_R)
    lub, piv, info = lapack.zgbtrf(ab, kl, ku, overwrite_ab=True)
    if info != 0:
        raise np.linalg.LinAlgError(f"zgbtrf info={info}")
    return lub, piv, kl, ku


def solve_factored(fac, rhs, chunk: int = 0, threads: int = 1):
    """T^-1 rhs (LAPACK zgbtrs on the factors of `factor`) for rhs [n, k].  The columns of a solve are independent, so
    with chunk > 0 they are handed to zgbtrs `chunk` columns at a time, on `threads` host threads (LAPACK releases the
    GIL): the same arithmetic per column as one call, only wall-clock time changes.  This is what lets Tier B reach
    BASELINE.json configs 3 and 4 ("Oracle outputs for C3-C4 may be cached on disk")."""
    from concurrent.futures import ThreadPoolExecutor
    lub, piv, kl, ku = fac
    rhs = np.asarray(rhs, dtype=np.complex128)
    k = rhs.shape[1]
    if chunk <= 0 or chunk >= k:
        sol, info = lapack.zgbtrs(lub, kl, ku, np.asfortranarray(rhs), piv)
        if info != 0:
            raise np.linalg.LinAlgError(f"zgbtrs info={info}")
        return np.ascontiguousarray(sol)
    out = np.empty(rhs.shape, dtype=np.complex128)

    def work(c0):
        sol, info = lapack.zgbtrs(lub, kl, ku, np.asfortranarray(rhs[:, c0:c0 + chunk]), piv)
        if info != 0:
            raise np.linalg.LinAlgError(f"zgbtrs info={info}")
        out[:, c0:c0 + chunk] = sol

    starts = list(range(0, k, chunk))
    if threads > 1:
        with ThreadPoolExecutor(max_workers=threads) as ex:
            list(ex.map(work, starts))
    else:
        for c0 in starts:
            work(c0)
    return out


def solve_energy_columns(E, H_diag, H_upper, S_diag, S_upper, Sigma_L, Sigma_R, Inj_first, Inj_last=None,
                         x_cols=None, chunk: int = 64, threads: int = 1):
    """Large-size form of `solve_energy`: one banded LU of T, then X only for the columns `x_cols` of Inj (every
    column of X = T^-1 Inj is its own solve, Eq. 5) and the whole last block column of T^-1 (Eq. 4), whose top block
    is G_1N.  Returns dict(X_cols [n, len(x_cols)], x_cols, G_last [n, bs], G_1N, T_LR, T_LR_complex)."""
    nb = len(H_diag)
    bs = np.asarray(H_diag[0]).shape[0]
    n = nb * bs
    b = dense.pad_injection(Inj_first, Inj_last, nb)
    x_cols = list(range(b.shape[1])) if x_cols is None else [int(c) for c in x_cols]
    fac = factor(E, H_diag, H_upper, S_diag, S_upper, Sigma_L, Sigma_R)
    rhs = np.zeros((n, len(x_cols) + bs), dtype=np.complex128)
    rhs[:, :len(x_cols)] = b[:, x_cols]
    rhs[n - bs:, len(x_cols):] = np.eye(bs)                  # e_nb (x) 1
    sol = solve_factored(fac, rhs, chunk=chunk, threads=threads)
    G_last = sol[:, len(x_cols):]
    G_1N = np.ascontiguousarray(G_last[:bs])
    t_lr = dense.transmission_from_G(Sigma_L, Sigma_R, G_1N)
    return dict(X_cols=np.ascontiguousarray(sol[:, :len(x_cols)]), x_cols=x_cols, G_last=np.ascontiguousarray(G_last),
                G_1N=G_1N, T_LR=t_lr.real, T_LR_complex=t_lr)
