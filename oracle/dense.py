"""Tier A oracle: assemble the full matrix, dense LU with partial pivoting, T(E).  TEST INFRASTRUCTURE.

Plain definition of what the SplitSolve path computes (see oracle/__init__.py).  Every function
cites the passage it follows.  complex128 everywhere.  Shapes / notation follow SURVEY.md §8:
bs = block size (s in the paper), nb = n_B, n = nb*bs = N_SS, blocks 1-indexed in the comments.
"""
from __future__ import annotations

import numpy as np


def assemble_A(E, H_diag, H_upper, S_diag, S_upper) -> np.ndarray:
    """A = E*S - H as a dense n x n matrix ("A", L184 "A = (E.S - H)").

    H, S are block tridiagonal (L127, Fig. 4 caption L74) and given by their diagonal blocks
    [nb,bs,bs] and upper blocks [nb-1,bs,bs] = (i,i+1); the lower blocks are the conjugate transposes
    of the upper ones (H, S Hermitian: L154).  E multiplies S as a plain complex scalar and is NOT
    conjugated in the lower blocks: A_{i+1,i} = E*S_{i,i+1}^H - H_{i,i+1}^H (reading c8).
    """
    H_diag = np.asarray(H_diag, dtype=np.complex128)
    S_diag = np.asarray(S_diag, dtype=np.complex128)
    H_upper = np.asarray(H_upper, dtype=np.complex128)
    S_upper = np.asarray(S_upper, dtype=np.complex128)
    nb, bs, _ = H_diag.shape
    n = nb * bs
    E = complex(E)
    A = np.zeros((n, n), dtype=np.complex128)
    for i in range(nb):
        r = slice(i * bs, (i + 1) * bs)
        A[r, r] = E * S_diag[i] - H_diag[i]
    for i in range(nb - 1):
        r = slice(i * bs, (i + 1) * bs)
        c = slice((i + 1) * bs, (i + 2) * bs)
        A[r, c] = E * S_upper[i] - H_upper[i]
        A[c, r] = E * S_upper[i].conj().T - H_upper[i].conj().T
    return A


def assemble_T(E, H_diag, H_upper, S_diag, S_upper, Sigma_L, Sigma_R) -> np.ndarray:
    """T = E*S - H - Sigma^RB (Eq. 5; Fig. 4 caption L74).

    Sigma^RB = B*C is non-zero only in the top-left (Sigma^{RB,L}) and bottom-right (Sigma^{RB,R})
    s x s blocks, and it is SUBTRACTED (L78, L135: T = A - BC).
    """
    A = assemble_A(E, H_diag, H_upper, S_diag, S_upper)
    bs = np.asarray(H_diag).shape[1]
    A[:bs, :bs] -= np.asarray(Sigma_L, dtype=np.complex128)
    A[-bs:, -bs:] -= np.asarray(Sigma_R, dtype=np.complex128)
    return A


def pad_injection(Inj_first, Inj_last, nb: int) -> np.ndarray:
    """b = Inj as an n x m matrix: non-zero only in the top and bottom block rows."""
    Inj_first = np.asarray(Inj_first, dtype=np.complex128)
    bs, m = Inj_first.shape
    b = np.zeros((nb * bs, m), dtype=np.complex128)
    b[:bs] = Inj_first
    if Inj_last is not None:
        b[-bs:] += np.asarray(Inj_last, dtype=np.complex128)
    return b


def gamma(Sigma) -> np.ndarray:
    """Broadening Gamma = i (Sigma - Sigma^H) (north_star; Datta [21])."""
    Sigma = np.asarray(Sigma, dtype=np.complex128)
    return 1j * (Sigma - Sigma.conj().T)


def transmission_from_G(Sigma_L, Sigma_R, G_1N) -> complex:
    """Tr(Gamma_L G_1N Gamma_R G_1N^H) as a complex number; T(E) is its real part (north_star)."""
    GL, GR = gamma(Sigma_L), gamma(Sigma_R)
    return complex(np.trace(GL @ G_1N @ GR @ G_1N.conj().T))


def solve_energy(E, H_diag, H_upper, S_diag, S_upper, Sigma_L, Sigma_R, Inj_first, Inj_last=None):
    """One energy point, by the plain definition.

    1. assemble dense T (Eq. 5);
    2. one LU with partial pivoting (LAPACK zgesv through numpy.linalg.solve) of T against
       [Inj | e_nb (x) 1 | e_1 (x) 1]  ->  X (Eq. 5), last and first block columns of G^R = T^-1 (Eq. 4);
    3. G_1N = top block of the last block column, G_N1 = bottom block of the first block column;
       T_LR = Re Tr(Gamma_L G_1N Gamma_R G_1N^H), T_RL = Re Tr(Gamma_R G_N1 Gamma_L G_N1^H).

    Returns dict(X [n,m], G_1N, G_N1, T_LR, T_RL, T_LR_complex).
    """
    H_diag = np.asarray(H_diag)
    nb, bs, _ = H_diag.shape
    n = nb * bs
    T = assemble_T(E, H_diag, H_upper, S_diag, S_upper, Sigma_L, Sigma_R)
    b = pad_injection(Inj_first, Inj_last, nb)
    m = b.shape[1]
    rhs = np.zeros((n, m + 2 * bs), dtype=np.complex128)
    rhs[:, :m] = b
    rhs[n - bs:, m:m + bs] = np.eye(bs)          # e_nb (x) 1
    rhs[:bs, m + bs:] = np.eye(bs)               # e_1 (x) 1
    sol = np.linalg.solve(T, rhs)
    X = sol[:, :m]
    G_1N = sol[:bs, m:m + bs]
    G_N1 = sol[n - bs:, m + bs:]
    t_lr = transmission_from_G(Sigma_L, Sigma_R, G_1N)
    t_rl = transmission_from_G(Sigma_R, Sigma_L, G_N1)
    return dict(X=X, G_1N=G_1N, G_N1=G_N1, T_LR=t_lr.real, T_RL=t_rl.real, T_LR_complex=t_lr)


def solve_all(problem):
    """All energies of a `Problem`-like object (attributes H_diag, ..., E, Sigma_L, Sigma_R, Inj_first,
    Inj_last).  Returns X [n_E, n, m] and T_LR [n_E]."""
    Xs, Ts = [], []
    for e in range(len(problem.E)):
        il = None if problem.Inj_last is None else problem.Inj_last[e]
        r = solve_energy(problem.E[e], problem.H_diag, problem.H_upper, problem.S_diag, problem.S_upper,
                         problem.Sigma_L[e], problem.Sigma_R[e], problem.Inj_first[e], il)
        Xs.append(r["X"])
        Ts.append(r["T_LR"])
    return np.stack(Xs), np.array(Ts)


def inverse_columns(E, H_diag, H_upper, S_diag, S_upper):
    """First and last block columns of A^-1, A = E*S - H WITHOUT the boundary self-energy
    ("Q consists of the first and last s columns of A^-1"; L167).
    Dense LU of A against [e_1 (x) 1 | e_nb (x) 1].  Returns Q [nb,bs,bs] with Q[i] = (A^-1)_{i+1,1}
    and P [nb,bs,bs] with P[i] = (A^-1)_{i+1,nb}."""
    H_diag = np.asarray(H_diag)
    nb, bs, _ = H_diag.shape
    n = nb * bs
    A = assemble_A(E, H_diag, H_upper, S_diag, S_upper)
    rhs = np.zeros((n, 2 * bs), dtype=np.complex128)
    rhs[:bs, :bs] = np.eye(bs)
    rhs[n - bs:, bs:] = np.eye(bs)
    sol = np.linalg.solve(A, rhs)
    Q = sol[:, :bs].reshape(nb, bs, bs).copy()
    P = sol[:, bs:].reshape(nb, bs, bs).copy()
    return Q, P
