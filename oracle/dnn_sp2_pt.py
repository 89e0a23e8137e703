"""O2 - the DNN-SP2-PT method, Algorithms 1-3, step by step.  Test infrastructure only.

Follows PAPER.md:485-525 in the paper's order and notation, with the readings of
SURVEY.md 8(c) (R1-R20) where the extracted pseudocode is silent or garbled; every
reading is listed in DESIGN.md.  Dense numpy matrices, fp64 scalars.  No blocking,
no fusion: each line below is one line of the algorithms.

Two product back-ends:
  Fp64Product      exact-arithmetic reference (the oracle proper, "O2").
  DualHalfProduct  CPU emulation of the paper's dual half-precision product
                   (Eqs. 12-16, 291-323 Eqs. 41-46): numpy float16
                   rounding (round-to-nearest-even), three fp32 GEMMs, fp32 sum, fp32
                   storage ("O2-dh").  It predicts the layer count and the accuracy
                   floor of ANY implementation of the method at that precision; it is
                   not the GPU code and shares nothing with it.
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

C_D0 = 4.5   # PAPER.md:518 (Alg. 2)
C_PT = 9.0   # PAPER.md:465, 524 (Alg. 3)


# ----------------------------------------------------------------------------
# spectral bounds
# ----------------------------------------------------------------------------
def gershgorin(h0):
    """Gershgorin row discs of a symmetric matrix: (eps_min, eps_max), fp64 (reading R1)."""
    h0 = np.asarray(h0, dtype=np.float64)
    d = np.diag(h0)
    r = np.abs(h0).sum(axis=1) - np.abs(d)
    return float((d - r).min()), float((d + r).max())


# ----------------------------------------------------------------------------
# products
# ----------------------------------------------------------------------------
class Fp64Product:
    """S^(j) S^(k-j) in exact (fp64) arithmetic."""
    store = np.float64
    name = "fp64"

    def square(self, s):
        return s @ s

    def cross(self, a, b, order_a=0, order_b=1):
        return a @ b


class DualHalfProduct:
    """Dual half-precision representation and product.

    split:   X_hi = FP16[X],  X_lo = FP16[X - X_hi]                  PAPER.md:120 (Eq. 13), 304-307
    square:  FP32[A + B + B^T], A = hi x hi, B = hi x lo             PAPER.md:124-136 (Eqs. 14-16)
    cross:   FP32[A + B + C], A = hi x hi, B = hi x lo, C = lo x hi  PAPER.md:316-323 (Eqs. 45-46)
    lo x lo is discarded.  fp16 operands, fp32 accumulation (numpy sgemm), fp32 sum.

    `shift0` / `shift1`: exact power-of-two pre-scale 2^shift applied to an iterate before it
    is split and removed (exactly) from the product afterwards - readings R12/R17 of
    SURVEY.md 8(c).  shift = 0 is the paper's Eq. 13 verbatim.  shift1 = "auto" picks, for every
    split of a response iterate, the power of two that brings max|X| into [8, 16).
    """
    store = np.float32
    name = "dual-half"

    def __init__(self, shift0=0, shift1=0):
        self.shift0 = shift0
        self.shift1 = shift1

    @staticmethod
    def _auto(x):
        m = float(np.abs(x).max())
        if not np.isfinite(m) or m == 0.0:
            return 0
        return 3 - int(np.floor(np.log2(m)))

    def split(self, x, shift):
        e = self._auto(x) if shift == "auto" else int(shift)
        xs = np.ldexp(np.asarray(x, dtype=np.float32), e)           # exact
        hi = xs.astype(np.float16)                                   # Eq. 13, first line
        lo = (xs - hi.astype(np.float32)).astype(np.float16)         # Eq. 13, second line
        return hi.astype(np.float32), lo.astype(np.float32), e

    def square(self, s):
        hi, lo, e = self.split(s, self.shift0)
        a = hi @ hi                                                  # Eq. 15
        b = hi @ lo                                                  # Eq. 16
        return np.ldexp(a + b + b.T, -2 * e)                         # Eq. 14

    def cross(self, x, y, order_x=0, order_y=1):
        xh, xl, ex = self.split(x, self.shift0 if order_x == 0 else self.shift1)
        yh, yl, ey = self.split(y, self.shift0 if order_y == 0 else self.shift1)
        a = xh @ yh                                                  # Eq. 46
        b = xh @ yl
        c = xl @ yh
        return np.ldexp(a + b + c, -(ex + ey))                       # Eq. 45


# ----------------------------------------------------------------------------
# result record
# ----------------------------------------------------------------------------
@dataclass
class Sp2PtResult:
    d0: np.ndarray
    d1: np.ndarray
    d2: np.ndarray | None
    layers: int                 # passes of the while loop of Algorithm 1
    layers_d0: int              # n_c: layer at which D0 converged (0 if never)
    layers_d1: int              # layer at which D1 converged (0 if never)
    status: str                 # "ok" | "noconv"
    eps_min: float
    eps_max: float
    fro_err0: float
    sigma: list = field(default_factory=list)      # sigma[n-1] for layer n
    tr_s: list = field(default_factory=list)       # N_S = Tr S0_{n-1} entering layer n
    tr_x: list = field(default_factory=list)       # N_X = Tr X0_n (nan once S0 froze)
    id_err: list = field(default_factory=list)     # IdErr_n (nan once S0 froze)
    fro_err1: list = field(default_factory=list)   # FroErr1_n (nan before D0 converged)
    fro_err2: list = field(default_factory=list)   # FroErr2_n (order 2; nan before D1 converged)
    dk: list = field(default_factory=list)         # [D0, D1, ..., D_order]
    layers_dk: list = field(default_factory=list)  # layer at which the test of each order fired
    fro_errk: list = field(default_factory=list)   # fro_errk[k][n-1] = FroErr^(k)_n, k >= 1


def _fro(x):
    return float(np.sqrt(np.sum(np.asarray(x, dtype=np.float64) ** 2)))


# ----------------------------------------------------------------------------
# Algorithms 1-3
# ----------------------------------------------------------------------------
def dnn_sp2_pt(h0, h1, n_occ, order=1, max_layers=200, product=None, bounds=None,
               nx_mode="trace"):
    """DNN-SP2-PT to response order `order` >= 1 (Algorithms 1-3 are printed for order 1; orders >= 2 follow
    Eq. 26, "a straightforward generalization", with the cascaded stop of reading R15).

    h0, h1: symmetric (n, n) (already orthogonalised); n_occ: occupied count.
    bounds: (eps_min, eps_max) or None for Gershgorin (R1, R18).
    nx_mode: "trace" takes N_X = Tr[X_n] as the paper prints it;
             "fro" takes the mathematically identical ||S0_{n-1}||_F^2 (reading R9).
    """
    P = product if product is not None else Fp64Product()
    st = P.store
    h0 = np.asarray(h0, dtype=np.float64)
    h1 = np.asarray(h1, dtype=np.float64)
    n = h0.shape[0]
    m = int(order)
    if m < 1:
        raise ValueError("order >= 1 (dnn_sp2 is the ground-state recursion)")
    eps_min, eps_max = gershgorin(h0) if bounds is None else bounds
    w = eps_max - eps_min
    if not (np.isfinite(w) and w > 0.0):
        raise ValueError("degenerate spectral bounds")

    # initial normalisation layer                        PAPER.md:209-215, 249 (Eq. 34), 493
    s0 = ((eps_max * np.eye(n) - h0) / w).astype(st)
    sk = [None, (-h1 / w).astype(st)] + [np.zeros((n, n), dtype=st) for _ in range(2, m + 1)]   # H^(k) = 0, k >= 2
    n_s = float(np.trace(s0.astype(np.float64)))                  # N_S = Tr[S0_0]

    res = Sp2PtResult(d0=None, d1=None, d2=None, layers=0, layers_d0=0, layers_d1=0,
                      status="noconv", eps_min=eps_min, eps_max=eps_max, fro_err0=float("nan"))
    sig, id_err = res.sigma, res.id_err
    fro = [None, res.fro_err1, res.fro_err2] + [[] for _ in range(3, m + 1)]     # fro[k][n-1] = FroErr^(k)_n
    conv = [False] * (m + 1)          # conv[0]: Algorithm 2; conv[k]: Algorithm 3 for order k
    n_cv = [0] * (m + 1)              # layer at which each fired
    fro0 = float("nan")
    nan = float("nan")
    nl = 1
    while nl <= max_layers and not conv[m]:                              # R2
        # activation functions f^(k) = sum_j S^(j) S^(k-j)   PAPER.md:201 (Eq. 26), 285 (Eq. 40); the products
        # with j > k/2 are the transposes of those with j < k/2
        xk = [None] * (m + 1)
        for k in range(1, m + 1):
            acc = None
            for j in range(0, (k + 1) // 2):
                p = P.cross(s0 if j == 0 else sk[j], sk[k - j], j, k - j)
                t = p + p.T
                acc = t if acc is None else acc + t
            if k % 2 == 0:
                acc = acc + P.cross(sk[k // 2], sk[k // 2], k // 2, k // 2)
            xk[k] = acc
        res.tr_s.append(n_s)
        if not conv[0]:
            x0 = P.square(s0)
            if nx_mode == "trace":
                n_x = float(np.trace(x0.astype(np.float64)))
            else:
                n_x = float(np.sum(s0.astype(np.float64) ** 2))           # R9
            ide = n_s - n_x
            s = 1 if abs(2.0 * n_s - n_x - n_occ) >= abs(n_x - n_occ) else -1   # PAPER.md:501, R3
            res.tr_x.append(n_x)
            id_err.append(ide)
            sig.append(s)
            # Algorithm 2                                 PAPER.md:515-519 (R4, R6)
            stop = not (ide > 0.0)
            if not stop and nl > 2 and sig[nl - 2] != sig[nl - 3]:
                stop = not (ide <= C_D0 * id_err[nl - 3] ** 2)
            if stop:
                conv[0] = True
                n_cv[0] = nl
                fro0 = _fro(s0.astype(np.float64) - x0.astype(np.float64))
            else:
                s0 = (s * x0 + (1 - s) * s0).astype(st)                   # PAPER.md:182 (Eq. 23)
                n_s = s * n_x + (1 - s) * n_s
        else:
            res.tr_x.append(nan)
            id_err.append(nan)
            sig.append(-sig[nl - 2])
        s = sig[nl - 1]

        # Algorithm 3 (R5, R6, R7) for order 1; the same test cascaded for every further order
        # (reading R15): order k is measured once order k-1 has converged, first test two layers later
        for k in range(1, m + 1):
            if conv[k]:
                fro[k].append(nan)
                continue
            if conv[k - 1]:
                fro[k].append(_fro(sk[k].astype(np.float64) - xk[k].astype(np.float64)))
                if nl - 2 >= n_cv[k - 1] and not (fro[k][nl - 1] < C_PT * fro0 * fro[k][nl - 3]):
                    conv[k] = True
                    n_cv[k] = nl
            else:
                fro[k].append(nan)
            if not conv[k]:
                sk[k] = (s * xk[k] + (1 - s) * sk[k]).astype(st)          # PAPER.md:193-201 (Eqs. 25, 26)
        nl += 1

    res.layers = nl - 1
    res.layers_d0 = n_cv[0]
    res.layers_d1 = n_cv[1]
    res.layers_dk = list(n_cv)
    res.fro_err0 = fro0
    res.fro_errk = fro
    res.status = "ok" if conv[m] else "noconv"
    res.d0 = np.asarray(s0, dtype=np.float64)
    res.d1 = np.asarray(sk[1], dtype=np.float64)
    res.d2 = None if m < 2 else np.asarray(sk[2], dtype=np.float64)
    res.dk = [res.d0] + [np.asarray(x, dtype=np.float64) for x in sk[1:]]
    return res


# ----------------------------------------------------------------------------
# ground-state SP2 only (used by the finite-difference pin)
# ----------------------------------------------------------------------------
def dnn_sp2(h0, n_occ, max_layers=200, bounds=None):
    """D0 alone: Algorithm 1 with the response lines removed, Algorithm 2 unchanged (fp64)."""
    h0 = np.asarray(h0, dtype=np.float64)
    n = h0.shape[0]
    eps_min, eps_max = gershgorin(h0) if bounds is None else bounds
    s0 = (eps_max * np.eye(n) - h0) / (eps_max - eps_min)
    n_s = float(np.trace(s0))
    sig, id_err = [], []
    for nl in range(1, max_layers + 1):
        x0 = s0 @ s0
        n_x = float(np.trace(x0))
        ide = n_s - n_x
        s = 1 if abs(2.0 * n_s - n_x - n_occ) >= abs(n_x - n_occ) else -1
        sig.append(s)
        id_err.append(ide)
        stop = not (ide > 0.0)
        if not stop and nl > 2 and sig[nl - 2] != sig[nl - 3]:
            stop = not (ide <= C_D0 * id_err[nl - 3] ** 2)
        if stop:
            return s0, nl
        s0 = s * x0 + (1 - s) * s0
        n_s = s * n_x + (1 - s) * n_s
    return s0, max_layers
