"""Observables derived from the wave functions c(E) = X.  TEST INFRASTRUCTURE.

PAPER.md L85: "charge and current densities can be directly derived from G^R(E) or c(E)".  In the wave-function
formalism the carrier density on orbital i is the occupation-weighted sum over energies and injected modes of the
squared modulus of the wave-function coefficient (Datta [21]); occupations and integration weights are
inputs here (they come from the contacts' Fermi functions and the energy grid, which OMEN builds: L250).

Pin status: density -- pinned (tests/test_oracle_pins.py: perfect chain X_j = e^{ikj} 1 gives rho_i = sum_e w_e exactly;
brute-force python loop on tiny inputs).
"""
from __future__ import annotations

import numpy as np


def density(X, w=None) -> np.ndarray:
    """rho[i] = sum_e w[e] * sum_c |X[e, i, c]|^2 ;  X [n_energy, n, nrhs] complex, w [n_energy] real (default ones)."""
    X = np.asarray(X, dtype=np.complex128)
    p = (X.real ** 2 + X.imag ** 2).sum(axis=2)              # [n_energy, n]
    if w is None:
        return p.sum(axis=0)
    return np.tensordot(np.asarray(w, dtype=np.float64), p, axes=(0, 0))


def bond_current(E, H_upper, S_upper, X) -> np.ndarray:
    """J[i] = 2 Im Tr( X_i^H A_{i,i+1} X_{i+1} ), A_{i,i+1} = E*S_{i,i+1} - H_{i,i+1} (Eq. 5), for one energy;
    X [n, m] with n = nb*bs.  Interior block rows of T x = b read A_{i,i-1} x_{i-1} + A_ii x_i + A_{i,i+1} x_{i+1} = 0; with
    x_i^H from the left and Im E = 0 (A_ii Hermitian, A_{i,i-1} = A_{i-1,i}^H) the imaginary part gives J[i-1] = J[i]:
    the current is conserved along the device (pinned in tests/test_oracle_pins.py)."""
    H_upper = np.asarray(H_upper)
    nbm1, bs, _ = H_upper.shape
    Xb = np.asarray(X, dtype=np.complex128).reshape(nbm1 + 1, bs, -1)
    J = np.empty(nbm1)
    for i in range(nbm1):
        A = complex(E) * np.asarray(S_upper[i]) - H_upper[i]
        J[i] = 2.0 * np.imag(np.trace(Xb[i].conj().T @ (A @ Xb[i + 1])))
    return J
