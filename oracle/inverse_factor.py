"""O4 - inverse factorisation of the overlap matrix, PAPER.md:693-703 (A17-A21).  Test infrastructure only.

    X_n = Z_n^T S Z_n                         (A19)
    Z_{n+1} = Z_n sum_{k=0}^{2} a_k X_n^k     (A20)
    a_k = {1.875, -1.25, 0.375}               (A21)

with Z_0 such that ||Z_0^T S Z_0 - I|| < 1; the error decays cubically.  Plain numpy, fp64,
one line per line of the recursion.  Reading (the paper leaves Z_0 open): Z_0 = I / sqrt(eps_max) with
eps_max the Gershgorin upper bound of S, which puts the spectrum of X_0 into (0, 1] for a positive definite S;
every Z_n is then a polynomial in S and the limit is the Loewdin factor S^(-1/2).
"""
from __future__ import annotations

import numpy as np

A_K = (1.875, -1.25, 0.375)      # PAPER.md:701 (A21)


def gershgorin_max(s):
    s = np.asarray(s, dtype=np.float64)
    d = np.diag(s)
    return float((d + np.abs(s).sum(axis=1) - np.abs(d)).max())


def inverse_factor(s, max_iter=30, tol=1e-12):
    """Return (Z, errors) with errors[n] = ||X_n - I||_F; stops when the error is below tol."""
    s = np.asarray(s, dtype=np.float64)
    n = s.shape[0]
    eye = np.eye(n)
    z = eye / np.sqrt(gershgorin_max(s))
    errors = []
    for _ in range(max_iter):
        x = z.T @ s @ z                                            # A19
        errors.append(float(np.linalg.norm(x - eye)))
        if errors[-1] <= tol:
            break
        z = z @ (A_K[0] * eye + A_K[1] * x + A_K[2] * (x @ x))     # A20
    return z, errors
