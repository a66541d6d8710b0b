"""Tier C: oracle-free residual and the error metrics of BASELINE.json's tolerances.  TEST INFRASTRUCTURE.

`backward_error` evaluates  ||T X - Inj||_F / (||T||_F ||X||_F + ||Inj||_F)  (north_star "normwise
backward error <= 1e-12"; reading c18) by a block-tridiagonal mat-mul, block row by block
row, directly from the definition of T (Eq. 5; Sigma placement L148).  T is never
assembled, so it works at any size (used for the full-size configs C3, C4 where no solve-oracle fits).
"""
from __future__ import annotations

import numpy as np


def _A_diag(E, H_diag, S_diag, i):
    return complex(E) * np.asarray(S_diag[i]) - np.asarray(H_diag[i])


def _A_up(E, H_upper, S_upper, i):
    return complex(E) * np.asarray(S_upper[i]) - np.asarray(H_upper[i])


def _A_lo(E, H_upper, S_upper, i):
    """Block (i+1, i): E*S_up^H - H_up^H, E not conjugated (reading c8)."""
    return complex(E) * np.asarray(S_upper[i]).conj().T - np.asarray(H_upper[i]).conj().T


def apply_T(E, H_diag, H_upper, S_diag, S_upper, Sigma_L, Sigma_R, X):
    """Y = T X for X [n, m], block row by block row.  Also returns ||T||_F^2."""
    H_diag = np.asarray(H_diag)
    nb, bs, _ = H_diag.shape
    X = np.asarray(X, dtype=np.complex128)
    Xb = X.reshape(nb, bs, -1)
    Y = np.empty_like(Xb)
    t2 = 0.0
    for i in range(nb):
        D = _A_diag(E, H_diag, S_diag, i)
        if i == 0:
            D = D - np.asarray(Sigma_L)
        if i == nb - 1:
            D = D - np.asarray(Sigma_R)
        t2 += float(np.sum(np.abs(D) ** 2))
        acc = D @ Xb[i]
        if i + 1 < nb:
            U = _A_up(E, H_upper, S_upper, i)
            t2 += float(np.sum(np.abs(U) ** 2))
            acc += U @ Xb[i + 1]
        if i > 0:
            L = _A_lo(E, H_upper, S_upper, i - 1)
            t2 += float(np.sum(np.abs(L) ** 2))
            acc += L @ Xb[i - 1]
        Y[i] = acc
    return Y.reshape(X.shape), t2


def backward_error(E, H_diag, H_upper, S_diag, S_upper, Sigma_L, Sigma_R, Inj_first, Inj_last, X) -> float:
    nb, bs, _ = np.asarray(H_diag).shape
    Y, t2 = apply_T(E, H_diag, H_upper, S_diag, S_upper, Sigma_L, Sigma_R, X)
    Yb = Y.reshape(nb, bs, -1).copy()
    Yb[0] -= np.asarray(Inj_first)
    inj2 = float(np.sum(np.abs(Inj_first) ** 2))
    if Inj_last is not None:
        Yb[nb - 1] -= np.asarray(Inj_last)
        inj2 += float(np.sum(np.abs(Inj_last) ** 2))
    num = float(np.sqrt(np.sum(np.abs(Yb) ** 2)))
    den = np.sqrt(t2) * float(np.linalg.norm(X)) + np.sqrt(inj2)
    return num / den if den > 0 else num


def rel_frobenius(X, X_ref) -> float:
    """||X - X_ref||_F / ||X_ref||_F  (north_star "relative Frobenius error of X <= 1e-8")."""
    d = float(np.linalg.norm(np.asarray(X) - np.asarray(X_ref)))
    r = float(np.linalg.norm(X_ref))
    return d / r if r > 0 else d


def rel_T(T, T_ref) -> float:
    """|T - T_ref| / max(|T_ref|, 1e-300)  (north_star "relative T(E) error <= 1e-9")."""
    return abs(float(T) - float(T_ref)) / max(abs(float(T_ref)), 1e-300)


def inverse_column_residual(E, H_diag, H_upper, S_diag, S_upper, Q, P) -> float:
    """|| A [Q|P] - [e_1|e_nb] ||_F / (||A||_F ||[Q|P]||_F), Sigma = 0."""
    nb, bs, _ = np.asarray(H_diag).shape
    QP = np.concatenate([np.asarray(Q).reshape(nb * bs, bs), np.asarray(P).reshape(nb * bs, bs)], axis=1)
    Z = np.zeros((bs, bs), dtype=np.complex128)
    Y, t2 = apply_T(E, H_diag, H_upper, S_diag, S_upper, Z, Z, QP)
    Y = Y.copy()
    Y[:bs, :bs] -= np.eye(bs)
    Y[-bs:, bs:] -= np.eye(bs)
    return float(np.linalg.norm(Y)) / (np.sqrt(t2) * float(np.linalg.norm(QP)))
