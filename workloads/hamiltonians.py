"""Synthetic gapped Hamiltonians shaped like the paper's workloads.

Five configurations follow BASELINE.json `configs` (sizes, fill fractions,
value distributions); SURVEY.md section 8(d) fixes the details the config text
leaves open.  Everything is seeded (numpy PCG64, seed = 20220309 + index),
generated in fp64, rounded ONCE to fp32 and handed as the same fp32 values to
the CUDA path and to the oracle.

No method arithmetic lives here: dense linear algebra (QR, eigh, matmul) is
only used to *construct* inputs with a known spectrum or to open a gap
("scissor shift").  Heavy linear algebra may run through torch on
a CUDA device when `device="cuda"` is asked for (N >= 8192); the random numbers
always come from numpy on the host so a config is the same matrix family on
any machine.
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

BASE_SEED = 20220309


def seed_for(config_index: int) -> int:
    return BASE_SEED + int(config_index)


@dataclass
class Workload:
    name: str
    n: int
    n_occ: int
    order: int
    h0: np.ndarray  # (n, n) float32, exactly symmetric
    h1: np.ndarray  # (n, n) float32, exactly symmetric
    meta: dict = field(default_factory=dict)


# ----------------------------------------------------------------------------
# linear-algebra backends (construction only)
# ----------------------------------------------------------------------------
def _use_torch(device) -> bool:
    return device is not None and str(device).startswith("cuda")


def _qr_q(g: np.ndarray, device) -> np.ndarray:
    """Orthogonal factor of a square matrix, columns signed so diag(R) > 0."""
    if _use_torch(device):
        import torch

        gt = torch.from_numpy(g).to(device)
        q, r = torch.linalg.qr(gt)
        s = torch.sign(torch.diagonal(r))
        s[s == 0] = 1.0
        q = q * s[None, :]
        return q.cpu().numpy()
    q, r = np.linalg.qr(g)
    s = np.sign(np.diag(r))
    s[s == 0] = 1.0
    return q * s[None, :]


def _q_diag_qt(q: np.ndarray, eps: np.ndarray, device) -> np.ndarray:
    if _use_torch(device):
        import torch

        qt = torch.from_numpy(q).to(device)
        e = torch.from_numpy(eps).to(device)
        h = (qt * e[None, :]) @ qt.T
        return h.cpu().numpy()
    return (q * eps[None, :]) @ q.T


def _eigh(h: np.ndarray, device):
    if _use_torch(device):
        import torch

        w, v = torch.linalg.eigh(torch.from_numpy(h).to(device))
        return w.cpu().numpy(), v.cpu().numpy()
    return np.linalg.eigh(h)


def _mirror_upper(h: np.ndarray, blk: int = 2048) -> None:
    """Copy the strict upper triangle onto the lower one, in place, block by block."""
    n = h.shape[0]
    for r0 in range(0, n, blk):
        r1 = min(n, r0 + blk)
        h[r0:r1, :r0] = h[:r0, r0:r1].T
        d = h[r0:r1, r0:r1]
        iu = np.triu_indices(r1 - r0, 1)
        d.T[iu] = d[iu]


def _sym_round32(h: np.ndarray, blk: int = 2048) -> np.ndarray:
    """Symmetrise in fp64, round once to fp32; result is exactly symmetric.

    Row blocks keep the temporaries small (N = 32768: 8 GiB per fp64 matrix)."""
    n = h.shape[0]
    h32 = np.empty((n, n), dtype=np.float32)
    for r0 in range(0, n, blk):
        r1 = min(n, r0 + blk)
        h32[r0:r1] = (0.5 * (h[r0:r1] + h[:, r0:r1].T)).astype(np.float32)
    # (a+b)/2 is commutative in IEEE arithmetic, so h32 is already bit-symmetric;
    # keep the upper triangle anyway so that symmetry never depends on that.
    _mirror_upper(h32, blk)
    return h32


# ----------------------------------------------------------------------------
# building blocks
# ----------------------------------------------------------------------------
def symmetric_gaussian(rng: np.random.Generator, n: int, scale: float) -> np.ndarray:
    """Symmetric matrix whose every entry is scale * N(0,1)."""
    a = rng.standard_normal((n, n))
    h1 = np.triu(a) + np.triu(a, 1).T
    return scale * h1


def gapped_random_orthogonal(rng, n, n_occ, occ_range, virt_range, device=None):
    """H0 = Q diag(eps) Q^T, Q the orthogonal factor of a Gaussian matrix.

    Returns (H0 fp64, eps ascending, Q with columns in the same order).
    """
    g = rng.standard_normal((n, n))
    q = _qr_q(g, device)
    del g
    e_occ = rng.uniform(occ_range[0], occ_range[1], size=n_occ)
    e_virt = rng.uniform(virt_range[0], virt_range[1], size=n - n_occ)
    eps = np.concatenate([np.sort(e_occ), np.sort(e_virt)])
    h0 = _q_diag_qt(q, eps, device)
    return h0, eps, q


def tight_binding_cube(rng, n_atoms, density=0.1, decay=1.5, onsite_sigma=0.3, orbitals=4):
    """Config-2 style tight-binding matrix on atoms at uniform random positions.

    Open boundaries.  Off-diagonal H0_ij = -exp(-r_ij/decay)*u_ij with
    u_ij = u_ji ~ U(0.5, 1) and r_ij the distance between the orbitals' atoms (0 on the
    same atom); diagonal ~ N(0, onsite_sigma).
    Returns (H0 fp64 symmetric, positions (n_atoms, 3), atom index of each orbital).
    """
    n = n_atoms * orbitals
    box = (n_atoms / density) ** (1.0 / 3.0)
    pos = rng.uniform(0.0, box, size=(n_atoms, 3))
    onsite = rng.normal(0.0, onsite_sigma, size=n)
    atom = np.repeat(np.arange(n_atoms), orbitals)
    h0 = np.empty((n, n), dtype=np.float64)
    # row blocks keep the temporaries small; u is drawn row block by row block in a
    # fixed order, and only its strict upper triangle is used.
    blk = 1024
    for r0 in range(0, n, blk):
        r1 = min(n, r0 + blk)
        u = rng.uniform(0.5, 1.0, size=(r1 - r0, n))
        d = pos[atom[r0:r1], None, :] - pos[None, atom, :]
        r = np.sqrt(np.einsum("ijk,ijk->ij", d, d))
        h0[r0:r1, :] = -np.exp(-r / decay) * u
    _mirror_upper(h0)
    h0[np.arange(n), np.arange(n)] = onsite
    return h0, pos, atom


def _scissor(h0: np.ndarray, n_occ: int, target_gap: float, device, mu_hint=None):
    """Open the HOMO-LUMO gap to `target_gap`.

    H0 <- H0 + delta * (I - 2 V_occ V_occ^T): occupied levels move down by delta and
    virtual levels up by delta, eigenvectors unchanged.  Returns (H0', eps', gap before).
    """
    if _use_torch(device):
        # everything on the device; only the shifted matrix comes back (N = 32768: 8 GiB per matrix)
        import torch

        from .linalg import eigh_any

        ht = torch.from_numpy(h0).to(device)
        wt, v = eigh_any(ht, mu_hint)
        w = wt.cpu().numpy()
        gap0 = float(w[n_occ] - w[n_occ - 1])
        delta = max(0.0, 0.5 * (target_gap - gap0))
        if delta > 0.0:
            vo = v[:, :n_occ]
            del v
            ht.addmm_(vo, vo.T, beta=1.0, alpha=-2.0 * delta)
            ht.diagonal().add_(delta)
            h0 = ht.cpu().numpy()
            w[:n_occ] -= delta
            w[n_occ:] += delta
        del ht
        torch.cuda.empty_cache()
        return h0, w, gap0
    w, v = _eigh(h0, device)
    gap0 = float(w[n_occ] - w[n_occ - 1])
    delta = max(0.0, 0.5 * (target_gap - gap0))
    if delta > 0.0:
        vo = v[:, :n_occ]
        p = vo @ vo.T
        h0 = h0 + delta * (np.eye(h0.shape[0]) - 2.0 * p)
        w = w.copy()
        w[:n_occ] -= delta
        w[n_occ:] += delta
    return h0, w, gap0


# ----------------------------------------------------------------------------
# the five configurations
# ----------------------------------------------------------------------------
CONFIGS = {
    1: dict(kind="orth", n=256, fill=0.5, occ=(-1.0, -0.1), virt=(0.1, 1.0),
            h1="gauss", h1_scale=0.01, order=1, name="N=256 fp64-oracle ref"),
    2: dict(kind="tb", n=2048, fill=0.5, h1="dipole_x", order=1, gap=1.0,
            name="N=2048 SCC-DFTB-like"),
    3: dict(kind="tb", n=8192, fill=0.375, h1="gauss", h1_scale=1e-3, order=1, gap=1.0,
            name="N=8192 CPHF-like"),
    4: dict(kind="orth", n=16384, fill=0.5, occ=(-1.0, -0.05), virt=(0.05, 1.0),
            h1="gauss", h1_scale=0.01, order=1, name="N=16384 peak-throughput"),
    5: dict(kind="tb", n=32768, fill=0.5, h1="dipole_z", order=2, gap=1.0,
            name="N=32768 large/second-order"),
}


def make_config(index: int, n: int | None = None, device=None, seed: int | None = None,
                scissor: bool = True) -> Workload:
    """Build configuration `index` (1..5) of BASELINE.json, optionally at a reduced size `n`.

    `n` keeps the construction and the fill fraction and only shrinks the matrix (tests use
    this to get cases the oracle finishes in seconds).  `scissor=False` keeps the literal,
    nearly gapless tight-binding spectrum of configs 2, 3, 5.
    """
    cfg = CONFIGS[index]
    n = int(cfg["n"] if n is None else n)
    rng = np.random.default_rng(seed_for(index) if seed is None else seed)
    n_occ = int(round(cfg["fill"] * n))
    meta: dict = {"config": index, "seed": seed_for(index) if seed is None else seed}

    if cfg["kind"] == "orth":
        h0, eps, _q = gapped_random_orthogonal(rng, n, n_occ, cfg["occ"], cfg["virt"], device)
        del _q
        meta["gap"] = float(eps[n_occ] - eps[n_occ - 1])
        meta["mu"] = float(0.5 * (eps[n_occ] + eps[n_occ - 1]))
        meta["spectrum"] = (float(eps[0]), float(eps[-1]))
        meta["eps"] = np.asarray(eps, dtype=np.float64)      # the constructed spectrum (before the fp32 rounding of H0)
        pos = atom = None
    else:
        if n % 4:
            raise ValueError("tight-binding configs need n divisible by 4")
        h0, pos, atom = tight_binding_cube(rng, n // 4)
        if scissor:
            mu_hint = None
            from .linalg import EIGH_DIRECT_MAX

            if _use_torch(device) and n > EIGH_DIRECT_MAX:
                # the device eigensolver refuses this size (workloads/linalg.py): split the spectrum near
                # the Fermi level, located on a small sibling of the same generator (same density of states)
                sib, _, _ = tight_binding_cube(np.random.default_rng(meta["seed"] + 7919), 1024)
                ws = np.linalg.eigvalsh(sib)
                k = int(round(cfg["fill"] * ws.shape[0]))
                mu_hint = 0.5 * (ws[k - 1] + ws[k])
                del sib
            h0, eps, gap0 = _scissor(h0, n_occ, cfg["gap"], device, mu_hint)
            meta["gap_literal"] = gap0
            meta["gap"] = float(eps[n_occ] - eps[n_occ - 1])
            meta["mu"] = float(0.5 * (eps[n_occ] + eps[n_occ - 1]))
            meta["spectrum"] = (float(eps[0]), float(eps[-1]))
            meta["eps"] = np.asarray(eps, dtype=np.float64)  # spectrum after the scissor shift (before fp32 rounding)
        else:
            meta["gap"] = None

    if cfg["h1"] == "gauss":
        h1 = symmetric_gaussian(rng, n, cfg["h1_scale"])
    else:
        axis = {"dipole_x": 0, "dipole_y": 1, "dipole_z": 2}[cfg["h1"]]
        h1 = None

    h0_32 = _sym_round32(h0)
    del h0
    if h1 is None:      # dipole field: diagonal, already symmetric; rounded once like everything else
        h1_32 = np.zeros((n, n), dtype=np.float32)
        h1_32[np.arange(n), np.arange(n)] = pos[atom, axis].astype(np.float32)
    else:
        h1_32 = _sym_round32(h1)
        del h1
    return Workload(name=cfg["name"] if n == cfg["n"] else f'{cfg["name"]} @ n={n}',
                    n=n, n_occ=n_occ, order=cfg["order"], h0=h0_32, h1=h1_32, meta=meta)
