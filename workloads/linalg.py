"""Construction-only dense linear algebra for sizes the device eigensolver refuses.

cuSOLVER's `syevd` (behind `torch.linalg.eigh`) fails with CUSOLVER_STATUS_INVALID_VALUE for
n >= ~28k on this image (measured: 24576 works, 28672 and 32768 do not), and a host LAPACK
`dsyevd` at N = 32768 needs the better part of an hour.  `eigh_sdc` gets the full
eigendecomposition of a symmetric fp64 matrix from pieces that do work at that size: a spectral
divide and conquer around a shift `mu` -

    X   = sign(H - mu I)                 Newton-Schulz iteration X <- X (3 I - X^2) / 2 (matmuls only)
    P<  = (I - X)/2,  P> = (I + X)/2     spectral projectors below / above mu
    Q<  = orth(P< G),  Q> = orth(P> G')  Householder QR of projected Gaussian blocks
    H<  = Q<^T H Q<,  H> = Q>^T H Q>     two half-size symmetric problems -> torch.linalg.eigh
    V   = [Q< U<, Q> U>],  w = [w<, w>]

Used to BUILD inputs with a known gap (workloads/hamiltonians.py, scissor shift) and by the GPU
tests' fp64 cross-reference; it is generic linear algebra, not the method under test, and nothing
in the product imports it.
"""
from __future__ import annotations

import math

EIGH_DIRECT_MAX = 24576        # largest n torch.linalg.eigh (cuSOLVER) was seen to accept on this image


def _spectral_radius_estimate(a, iters=40):
    import torch

    g = torch.Generator(device=a.device)
    g.manual_seed(12345)
    v = torch.randn(a.shape[0], 4, dtype=a.dtype, device=a.device, generator=g)
    r = 0.0
    for _ in range(iters):
        v = a @ v
        nrm = torch.linalg.vector_norm(v, dim=0)
        r = float(nrm.max())
        v = v / nrm
    return r


def sign_newton_schulz(a, tol=1e-12, max_iter=150):
    """Matrix sign of a symmetric fp64 torch matrix with no eigenvalue at 0.  Consumes `a`."""
    import torch

    n = a.shape[0]
    inf_norm = float(a.abs().sum(dim=1).max())                   # Gershgorin: ||a||_2 <= ||a||_inf
    r = min(inf_norm, 1.25 * _spectral_radius_estimate(a))       # power iteration never overshoots
    x = a.div_(r)                                                # ||x||_2 <= 1.25 < sqrt(3)
    for it in range(max_iter):
        x2 = x @ x
        # ||x^2 - I||_F^2 without forming I
        err = math.sqrt(max(0.0, float((x2 * x2).sum()) - 2.0 * float(torch.diagonal(x2).sum()) + n))
        if err <= tol * math.sqrt(n):
            break
        x = torch.addmm(x, x, x2, beta=1.5, alpha=-0.5)
        del x2
    else:
        raise RuntimeError(f"sign iteration did not converge (residual {err:.3e}): eigenvalue too close to the shift")
    return 0.5 * (x + x.T), it


def eigh_sdc(h, mu):
    """(w ascending, v) of the symmetric fp64 device matrix `h` by one spectral split at `mu`.

    Both sides of the split must hold at most EIGH_DIRECT_MAX eigenvalues."""
    import torch

    n = h.shape[0]
    a = h.clone()
    a.diagonal().sub_(mu)
    x, _ = sign_newton_schulz(a)
    del a
    k = int(round(0.5 * (n - float(torch.diagonal(x).sum()))))   # eigenvalues below mu
    if not (0 < k < n) or max(k, n - k) > EIGH_DIRECT_MAX:
        raise RuntimeError(f"split at mu={mu} leaves {k} / {n - k} eigenvalues: outside the direct solver's range")
    g = torch.Generator(device=h.device)
    g.manual_seed(20220309)
    ws, vs = [], []
    for sgn, m in ((-1.0, k), (1.0, n - k)):
        gm = torch.randn(n, m, dtype=h.dtype, device=h.device, generator=g)
        b = torch.addmm(gm, x, gm, beta=0.5, alpha=0.5 * sgn)     # (I + sgn X)/2 G
        del gm
        q, _ = torch.linalg.qr(b)
        del b
        hq = q.T @ (h @ q)
        w, u = torch.linalg.eigh(0.5 * (hq + hq.T))
        del hq
        ws.append(w)
        vs.append(q @ u)
        del q, u
    del x
    if not float(ws[0][-1]) < mu < float(ws[1][0]):
        raise RuntimeError("spectral split is not clean")
    return torch.cat(ws), torch.cat(vs, dim=1)


def eigh_any(h, mu_hint=None):
    """torch.linalg.eigh where it works, eigh_sdc(h, mu_hint) above that size."""
    import torch

    if h.shape[0] <= EIGH_DIRECT_MAX:
        return torch.linalg.eigh(h)
    if mu_hint is None:
        raise ValueError("n above the direct solver's range: a shift inside the spectrum is needed")
    return eigh_sdc(h, float(mu_hint))
