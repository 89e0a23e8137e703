"""O1 - the definition of the result, by eigendecomposition (fp64).  Test infrastructure only.

D0 = theta(mu I - H0) with Tr D0 = N_occ                      PAPER.md:72 (Eq. 5), 81
D^(k) = (1/k!) d^k theta(mu I - H(lambda)) / d lambda^k       PAPER.md:164 (Eq. 20), 352 (Eq. 49)
Directional derivative of a matrix function in the eigenbasis (Daleckii-Krein):
    V (G o (V^T H1 V)) V^T,  G_ij = divided difference         PAPER.md:369-376 (Eqs. 53-54)
For the step function the divided differences are (f_i - f_j)/(eps_i - eps_j) with
f = 1 (occupied) / 0 (virtual), and 0 inside the occ-occ and virt-virt blocks - the 0/1
pattern of PAPER.md:384-393 (Eqs. 56-58) divided by the level spacing.

D2 has no printed formula; it follows from the order-2 blocks of D^2 = D and HD - DH = 0
 with H^(2) = 0.  `density_matrices_to_order` carries the same
two block identities to any order k (the (m+1)N x (m+1)N upper-triangular block
matrices of D and H are idempotent and commute, order by order).
"""
from __future__ import annotations

import numpy as np


def eigensystem(h0):
    """Ascending eigenvalues and eigenvectors of the symmetric matrix h0 (fp64)."""
    h0 = np.asarray(h0, dtype=np.float64)
    return np.linalg.eigh(0.5 * (h0 + h0.T))


def density_matrices(h0, h1, n_occ, order=1, eig=None):
    """Return (D0, D1[, D2]) of theta(mu I - (H0 + lambda H1)) at lambda = 0.

    h0, h1: symmetric (n, n); n_occ lowest eigenstates are occupied; the gap between level
    n_occ-1 and n_occ must be open (non-degenerate perturbation theory).
    """
    eps, v = eigensystem(h0) if eig is None else eig
    h1 = np.asarray(h1, dtype=np.float64)
    n = eps.shape[0]
    if not 0 < n_occ < n:
        raise ValueError("need 0 < n_occ < n")
    f = np.zeros(n)
    f[:n_occ] = 1.0
    vo = v[:, :n_occ]
    d0 = vo @ vo.T                                   # PAPER.md:72, A11

    a = v.T @ h1 @ v                                 # H1 in the eigenbasis of H0
    de = eps[:, None] - eps[None, :]
    df = f[:, None] - f[None, :]
    g = np.zeros((n, n))
    mask = df != 0.0
    g[mask] = df[mask] / de[mask]                    # PAPER.md:375 (Eq. 54) for the step function
    y = g * a                                        # PAPER.md:371 (Eq. 53)
    d1 = v @ y @ v.T
    if order == 1:
        return d0, d1

    o = slice(0, n_occ)
    u = slice(n_occ, n)
    z = np.zeros((n, n))
    z[o, o] = -y[o, u] @ y[u, o]                     # oo block of D0 D2 + D1 D1 + D2 D0 = D2
    z[u, u] = y[u, o] @ y[o, u]                      # vv block of the same
    num = y[o, u] @ a[u, u] - a[o, o] @ y[o, u]      # ov block of [H0, D2] + [H1, D1] = 0
    z[o, u] = num / de[o, u]
    z[u, o] = z[o, u].T
    d2 = v @ z @ v.T
    return d0, d1, d2


def density_matrices_to_order(h0, h1, n_occ, order, eig=None):
    """[D0, D1, ..., D_order] with D_k = (1/k!) d^k theta(mu I - H0 - lambda H1)/d lambda^k at 0.

    In the eigenbasis of H0 (Z_k = V^T D_k V, A = V^T H1 V, Z_0 = diag(f)) the order-k blocks of
    D(lambda)^2 = D(lambda) and [H(lambda), D(lambda)] = 0, with H^(k) = 0 for k >= 2, read
        sum_{j=0..k} Z_j Z_{k-j} = Z_k          and          [diag(eps), Z_k] + [A, Z_{k-1}] = 0,
    which give, with C_k = sum_{0<j<k} Z_j Z_{k-j},
        (Z_k)_oo = -(C_k)_oo,   (Z_k)_vv = (C_k)_vv,   (Z_k)_ia = (Z_{k-1} A - A Z_{k-1})_ia / (eps_i - eps_a).
    Orders 1 and 2 reduce to `density_matrices`.
    """
    eps, v = eigensystem(h0) if eig is None else eig
    a = v.T @ np.asarray(h1, dtype=np.float64) @ v
    n = eps.shape[0]
    if not 0 < n_occ < n:
        raise ValueError("need 0 < n_occ < n")
    o = slice(0, n_occ)
    u = slice(n_occ, n)
    de = eps[:, None] - eps[None, :]
    f = np.zeros(n)
    f[:n_occ] = 1.0
    z = [np.diag(f)]
    for k in range(1, order + 1):
        c = np.zeros((n, n))
        for j in range(1, k):
            c += z[j] @ z[k - j]
        zk = np.zeros((n, n))
        zk[o, o] = -c[o, o]
        zk[u, u] = c[u, u]
        num = z[k - 1] @ a - a @ z[k - 1]
        zk[o, u] = num[o, u] / de[o, u]
        zk[u, o] = zk[o, u].T
        z.append(zk)
    return [v @ zk @ v.T for zk in z]


def invariants(h0, h1, d0, d1, d2=None):
    """Max-abs residuals of the blocks of D^2 = D and HD - DH = 0."""
    h0 = np.asarray(h0, dtype=np.float64)
    h1 = np.asarray(h1, dtype=np.float64)
    d0 = np.asarray(d0, dtype=np.float64)
    d1 = np.asarray(d1, dtype=np.float64)
    out = {
        "idem0": np.abs(d0 @ d0 - d0).max(),
        "idem1": np.abs(d0 @ d1 + d1 @ d0 - d1).max(),
        "comm0": np.abs(h0 @ d0 - d0 @ h0).max(),
        "comm1": np.abs(h0 @ d1 - d1 @ h0 + h1 @ d0 - d0 @ h1).max(),
        "sym0": np.abs(d0 - d0.T).max(),
        "sym1": np.abs(d1 - d1.T).max(),
        "tr0": float(np.trace(d0)),
        "tr1": float(np.trace(d1)),
    }
    if d2 is not None:
        d2 = np.asarray(d2, dtype=np.float64)
        out["idem2"] = np.abs(d0 @ d2 + d1 @ d1 + d2 @ d0 - d2).max()
        out["comm2"] = np.abs(h0 @ d2 - d2 @ h0 + h1 @ d1 - d1 @ h1).max()
        out["sym2"] = np.abs(d2 - d2.T).max()
        out["tr2"] = float(np.trace(d2))
    return out
