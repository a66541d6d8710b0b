"""Step-by-step restatement of the paper's algebra, in its order and notation.  TEST INFRASTRUCTURE.

NOT the reference for parity (that is dense.py / banded.py, the plain definition).  It exists so the
tests can pin, against the plain definition, (a) Algorithm 1 with our readings of
its undefined / garbled spots, (b) the mirrored sweep for the last block column (L167), (c) the four
steps of Eq. 11-13 (L135-146) with the choice of B and C of L148, and (d) the one-step form
x = Q (b' + z) = Q R^-1 b' (L155).  "Solve" steps use numpy.linalg.solve on the bs x bs block, as the
paper uses a library solver there (L186).  Small inputs only (python loop over blocks).

Readings: c1  A_{1,0} := 1 and, in the mirror, A_{nb,nb+1} := 1;
                      c2  mirror sweep: Y_0 := 0; (A_ii - A_{i,i-1} Y_{i-1}) Y_i = A_{i,i+1}; P_{nb+1} := -1; P_i = -Y_i P_{i+1};
                      c3  Eq. 12 signs as printed: x = y + Q (1 - CQ)^-1 C y  (T = A - BC);
                      c4  Step 3 is (1 - CQ) z = C y.
"""
from __future__ import annotations

import numpy as np


def _blocks(E, H_diag, H_upper, S_diag, S_upper):
    E = complex(E)
    nb = len(H_diag)
    Ad = [E * np.asarray(S_diag[i]) - np.asarray(H_diag[i]) for i in range(nb)]
    Au = [E * np.asarray(S_upper[i]) - np.asarray(H_upper[i]) for i in range(nb - 1)]          # A_{i,i+1}
    Al = [E * np.asarray(S_upper[i]).conj().T - np.asarray(H_upper[i]).conj().T for i in range(nb - 1)]  # A_{i+1,i}
    return Ad, Au, Al


def algorithm1_first_column(E, H_diag, H_upper, S_diag, S_upper):
    """Algorithm 1 (L159-165): X_{nB+1} <- 0; Q_0 <- -1;
    for i = nB -> 1: Solve (A_ii - A_{i,i+1} X_{i+1}) X_i = A_{i,i-1};   for i = 1 -> nB: Q_i <- -X_i Q_{i-1}.
    Returns Q [nb,bs,bs], Q[i-1] = (A^-1)_{i,1}, and the list of X_i."""
    Ad, Au, Al = _blocks(E, H_diag, H_upper, S_diag, S_upper)
    nb = len(Ad)
    bs = Ad[0].shape[0]
    one = np.eye(bs, dtype=np.complex128)
    X = [None] * (nb + 2)
    X[nb + 1] = np.zeros((bs, bs), dtype=np.complex128)
    for i in range(nb, 0, -1):
        D = Ad[i - 1] - (Au[i - 1] @ X[i + 1] if i < nb else 0.0)
        rhs = Al[i - 2] if i > 1 else one            # A_{i,i-1}; A_{1,0} := 1 (reading c1)
        X[i] = np.linalg.solve(D, rhs)
    Q = [None] * (nb + 1)
    Q[0] = -one
    for i in range(1, nb + 1):
        Q[i] = -X[i] @ Q[i - 1]
    return np.stack(Q[1:]), X[1:nb + 1]


def schur_complements_first_column(E, H_diag, H_upper, S_diag, S_upper):
    """The matrices D_i = A_ii - A_{i,i+1} X_{i+1} that Algorithm 1's "Solve" step (L164) factors, i = 1..nb
    (D[i-1] = D_i).  PAPER.md L154: "A is usually real symmetric in 3-D structures and complex Hermitian in 1-D and
    2-D" -- at real E every D_i is then Hermitian, which is what L266's zhesv_nopiv_gpu exploits."""
    Ad, Au, Al = _blocks(E, H_diag, H_upper, S_diag, S_upper)
    nb = len(Ad)
    D = [None] * (nb + 1)
    Xn = None
    for i in range(nb, 0, -1):
        D[i] = Ad[i - 1] - (Au[i - 1] @ Xn if i < nb else 0.0)
        if i > 1:
            Xn = np.linalg.solve(D[i], Al[i - 2])
    return D[1:]


def algorithm1_last_column(E, H_diag, H_upper, S_diag, S_upper):
    """Mirror of Algorithm 1 for the last block column (L167 "derived similarly"; reading c2).
    Returns P [nb,bs,bs], P[i-1] = (A^-1)_{i,nb}, and the list of Y_i."""
    Ad, Au, Al = _blocks(E, H_diag, H_upper, S_diag, S_upper)
    nb = len(Ad)
    bs = Ad[0].shape[0]
    one = np.eye(bs, dtype=np.complex128)
    Y = [None] * (nb + 2)
    Y[0] = np.zeros((bs, bs), dtype=np.complex128)
    for i in range(1, nb + 1):
        D = Ad[i - 1] - (Al[i - 2] @ Y[i - 1] if i > 1 else 0.0)
        rhs = Au[i - 1] if i < nb else one           # A_{i,i+1}; A_{nb,nb+1} := 1
        Y[i] = np.linalg.solve(D, rhs)
    P = [None] * (nb + 2)
    P[nb + 1] = -one
    for i in range(nb, 0, -1):
        P[i] = -Y[i] @ P[i + 1]
    return np.stack(P[1:nb + 1]), Y[1:nb + 1]


def four_steps(Q, P, Sigma_L, Sigma_R, Inj_first, Inj_last=None):
    """Steps 1-4 of L141-146 given Step 1's result Q = A^-1 B = [first | last block column of A^-1]
    (B, C as in L148).  y = A^-1 b = Q b' (L155);  R = 1 - C Q;  z = R^-1 C y;  x = y + Q z (Eq. 13).
    Returns x [n, m], R [2bs,2bs], and x_onestep = Q (b' + z) = Q R^-1 b' (L155)."""
    nb, bs, _ = Q.shape
    n = nb * bs
    Qfull = np.concatenate([Q.reshape(n, bs), P.reshape(n, bs)], axis=1)        # N_SS x 2s
    m = Inj_first.shape[1]
    bprime = np.zeros((2 * bs, m), dtype=np.complex128)
    bprime[:bs] = Inj_first
    if Inj_last is not None:
        bprime[bs:] = Inj_last
    C = np.zeros((2 * bs, n), dtype=np.complex128)                               # L148
    C[:bs, :bs] = Sigma_L
    C[bs:, n - bs:] = Sigma_R
    y = Qfull @ bprime                                                           # Step 2 (L155)
    R = np.eye(2 * bs) - C @ Qfull                                               # L141
    z = np.linalg.solve(R, C @ y)                                                # Step 3 (reading c4)
    x = y + Qfull @ z                                                            # Step 4, Eq. 13
    x_onestep = Qfull @ np.linalg.solve(R, bprime)                               # x = Q (b' + z)
    return x, R, x_onestep
