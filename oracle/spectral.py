"""O3 - Algorithms 1-3 in the eigenbasis of H0 (fp64).  Test infrastructure only.

In the eigenbasis of H0 every iterate S0_n is diagonal, so the recursion acts elementwise:
    lambda <- sigma lambda^2 + (1 - sigma) lambda                    PAPER.md:182 (Eq. 23)
    Y_ij   <- sigma (lambda_i + lambda_j) Y_ij + (1 - sigma) Y_ij    PAPER.md:193 (Eq. 25)
with Y = V^T S1 V; (lambda_i + lambda_j) is the divided difference of x^2 (PAPER.md:369-376,
Eqs. 53-54).  Traces and Frobenius norms are basis independent, so sigma_n, N_S, N_X, IdErr
and both stopping tests follow without a single matrix product.  Uses: an independent pin of
O2's control flow, and layer-count prediction at sizes where O2 is out of reach.
"""
from __future__ import annotations

import numpy as np

C_D0 = 4.5
C_PT = 9.0


def spectral_recursion(eps, n_occ, eps_min, eps_max, a=None, max_layers=200):
    """eps: eigenvalues of H0; a: V^T H1 V (or None to follow D0 only, stopping at n_c).

    Returns dict(layers, layers_d0, sigma, tr_s, tr_x, id_err, fro_err0, fro_err1, lam, y).
    """
    eps = np.asarray(eps, dtype=np.float64)
    w = eps_max - eps_min
    lam = (eps_max - eps) / w                                  # PAPER.md:249 (Eq. 34)
    y = None if a is None else -np.asarray(a, dtype=np.float64) / w
    n_s = float(lam.sum())
    sig, tr_s, tr_x, id_err, fro1 = [], [], [], [], []
    conv0 = conv1 = False
    n_c = 0
    fro0 = float("nan")
    nl = 1
    while nl <= max_layers and not conv1:
        tr_s.append(n_s)
        if not conv0:
            x = lam * lam
            n_x = float(x.sum())
            ide = n_s - n_x
            s = 1 if abs(2.0 * n_s - n_x - n_occ) >= abs(n_x - n_occ) else -1
            tr_x.append(n_x)
            id_err.append(ide)
            sig.append(s)
            stop = not (ide > 0.0)
            if not stop and nl > 2 and sig[nl - 2] != sig[nl - 3]:
                stop = not (ide <= C_D0 * id_err[nl - 3] ** 2)
            if stop:
                conv0 = True
                n_c = nl
                fro0 = float(np.sqrt(np.sum((lam - x) ** 2)))
                if y is None:
                    break
        else:
            tr_x.append(float("nan"))
            id_err.append(float("nan"))
            sig.append(-sig[nl - 2])
        s = sig[nl - 1]
        if y is not None:
            # X1 uses S0_{n-1}: the eigenvalues BEFORE this layer's update of S0
            lam_prev = lam
            x1 = (lam_prev[:, None] + lam_prev[None, :]) * y
            if conv0:
                fro1.append(float(np.sqrt(np.sum((y - x1) ** 2))))
                if nl - 2 >= n_c and not (fro1[nl - 1] < C_PT * fro0 * fro1[nl - 3]):
                    conv1 = True
            else:
                fro1.append(float("nan"))
            if not conv1:
                y = s * x1 + (1 - s) * y
        if not conv0:
            lam = s * x + (1 - s) * lam
            n_s = s * n_x + (1 - s) * n_s
        nl += 1
    layers = nl if (y is None and conv0) else nl - 1
    return dict(layers=layers, layers_d0=n_c, sigma=sig, tr_s=tr_s, tr_x=tr_x, id_err=id_err,
                fro_err0=fro0, fro_err1=fro1, lam=lam, y=y)
