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


def _fro(x):
    return float(np.sqrt(np.sum(np.asarray(x, dtype=np.float64) ** 2)))


# ----------------------------------------------------------------------------
# Algorithms 1-3
# ----------------------------------------------------------------------------
def dnn_sp2_pt(h0, h1, n_occ, order=1, max_layers=200, product=None, bounds=None,
               nx_mode="trace"):
    """First- (or second-) order DNN-SP2-PT.

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
    eps_min, eps_max = gershgorin(h0) if bounds is None else bounds
    w = eps_max - eps_min
    if not (np.isfinite(w) and w > 0.0):
        raise ValueError("degenerate spectral bounds")

    # initial normalisation layer                        PAPER.md:209-215, 249 (Eq. 34), 493
    s0 = ((eps_max * np.eye(n) - h0) / w).astype(st)
    s1 = (-h1 / w).astype(st)
    s2 = np.zeros((n, n), dtype=st) if order == 2 else None      # H^(2) = 0
    n_s = float(np.trace(s0.astype(np.float64)))                  # N_S = Tr[S0_0]

    res = Sp2PtResult(d0=None, d1=None, d2=None, layers=0, layers_d0=0, layers_d1=0,
                      status="noconv", eps_min=eps_min, eps_max=eps_max, fro_err0=float("nan"))
    sig, id_err, fro1, fro2 = res.sigma, res.id_err, res.fro_err1, res.fro_err2
    conv0 = conv1 = conv2 = False
    n_c = n_c1 = 0
    fro0 = float("nan")
    nan = float("nan")
    nl = 1
    while nl <= max_layers and not (conv2 if order == 2 else conv1):      # R2
        # activation functions f^(1), f^(2)              PAPER.md:497, 195 (Eq. 25), 325-329
        p1 = P.cross(s0, s1, 0, 1)
        x1 = p1 + p1.T
        if order == 2:
            p2 = P.cross(s0, s2, 0, 1)
            q2 = P.cross(s1, s1, 1, 1)
            x2 = p2 + p2.T + q2
        res.tr_s.append(n_s)
        if not conv0:
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
                conv0 = True
                n_c = nl
                fro0 = _fro(s0.astype(np.float64) - x0.astype(np.float64))
            else:
                s0 = (s * x0 + (1 - s) * s0).astype(st)                   # PAPER.md:182 (Eq. 23)
                n_s = s * n_x + (1 - s) * n_s
        else:
            res.tr_x.append(nan)
            id_err.append(nan)
            sig.append(-sig[nl - 2])
        s = sig[nl - 1]

        # Algorithm 3                                     PAPER.md:521-525 (R5, R6, R7)
        if not conv1:
            if conv0:
                fro1.append(_fro(s1.astype(np.float64) - x1.astype(np.float64)))
                if nl - 2 >= n_c and not (fro1[nl - 1] < C_PT * fro0 * fro1[nl - 3]):
                    conv1 = True
                    n_c1 = nl
            else:
                fro1.append(nan)
            if not conv1:
                s1 = (s * x1 + (1 - s) * s1).astype(st)                   # PAPER.md:193 (Eq. 25)
        else:
            fro1.append(nan)

        # second order: the same test cascaded (reading R15)
        if order == 2:
            if conv1:
                fro2.append(_fro(s2.astype(np.float64) - x2.astype(np.float64)))
                if nl - 2 >= n_c1 and not (fro2[nl - 1] < C_PT * fro0 * fro2[nl - 3]):
                    conv2 = True
            else:
                fro2.append(nan)
            if not conv2:
                s2 = (s * x2 + (1 - s) * s2).astype(st)                   # PAPER.md:195 (Eq. 25)
        nl += 1

    res.layers = nl - 1
    res.layers_d0 = n_c
    res.layers_d1 = n_c1
    res.fro_err0 = fro0
    res.status = "ok" if (conv2 if order == 2 else conv1) else "noconv"
    res.d0 = np.asarray(s0, dtype=np.float64)
    res.d1 = np.asarray(s1, dtype=np.float64)
    res.d2 = None if s2 is None else np.asarray(s2, dtype=np.float64)
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
