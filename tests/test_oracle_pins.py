"""Pins for the CPU oracle (no GPU).  Each test checks the oracle against something OTHER than
itself: a textbook closed form, a finite difference, brute force on tiny inputs, an invariant
the paper states, a special case, or a number the paper prints (tests/golden/)."""
import os

import numpy as np
import pytest

from oracle import closed_form as O1
from oracle import dnn_sp2_pt as O2
from oracle import spectral as O3
from workloads import make_config, symmetric_gaussian

GOLD = {}
with open(os.path.join(os.path.dirname(__file__), "golden", "paper_constants.txt")) as fh:
    for line in fh:
        if line.strip() and not line.startswith("#"):
            k, v = line.split()[:2]
            GOLD[k] = float(v)


def small_problem(n=48, n_occ=20, seed=7, gap=0.4, h1_scale=0.05):
    rng = np.random.default_rng(seed)
    q, _ = np.linalg.qr(rng.standard_normal((n, n)))
    eps = np.concatenate([np.sort(rng.uniform(-1.0, -gap / 2, n_occ)),
                          np.sort(rng.uniform(gap / 2, 1.0, n - n_occ))])
    h0 = (q * eps) @ q.T
    h0 = 0.5 * (h0 + h0.T)
    h1 = symmetric_gaussian(rng, n, h1_scale)
    return h0, h1, n_occ, eps, q


# ------------------------------------------------------------------ O1: the definition
def test_o1_diagonal_h0_textbook():
    """Diagonal H0: D0 is the 0/1 occupation matrix and D1_ij = H1_ij/(eps_i - eps_j) on
    occupied/virtual pairs (first-order perturbation theory, BASELINE.json north_star)."""
    rng = np.random.default_rng(1)
    n, n_occ = 12, 5
    eps = np.sort(rng.uniform(-1, 1, n))
    perm = rng.permutation(n)
    e = eps[perm]                       # unsorted diagonal
    h0 = np.diag(e)
    h1 = symmetric_gaussian(rng, n, 1.0)
    d0, d1 = O1.density_matrices(h0, h1, n_occ)
    occ = np.argsort(e)[:n_occ]
    f = np.zeros(n)
    f[occ] = 1
    assert np.allclose(d0, np.diag(f), atol=1e-14)
    ref = np.zeros((n, n))
    for i in range(n):
        for j in range(n):
            if f[i] != f[j]:
                # occupied i / virtual j: H1_ij/(eps_i - eps_j); and its transpose
                ref[i, j] = h1[i, j] / (e[i] - e[j]) if f[i] == 1 else h1[i, j] / (e[j] - e[i])
    assert np.allclose(d1, ref, atol=1e-13)


def _theta(h, n_occ):
    w, v = np.linalg.eigh(h)
    return v[:, :n_occ] @ v[:, :n_occ].T


def test_o1_d1_finite_difference():
    """PAPER.md:352 (Eq. 49), 564 (Eq. 83): D1 is the directional derivative of theta."""
    h0, h1, n_occ, _, _ = small_problem()
    d0, d1 = O1.density_matrices(h0, h1, n_occ)
    h = 1e-4
    fd = (_theta(h0 + h * h1, n_occ) - _theta(h0 - h * h1, n_occ)) / (2 * h)
    assert np.abs(fd - d1).max() < 1e-6 * max(1.0, np.abs(d1).max())
    # 4-point stencil, PAPER.md:573 (Eq. 84)
    fd4 = (-_theta(h0 + 2 * h * h1, n_occ) + 8 * _theta(h0 + h * h1, n_occ)
           - 8 * _theta(h0 - h * h1, n_occ) + _theta(h0 - 2 * h * h1, n_occ)) / (12 * h)
    assert np.abs(fd4 - d1).max() < 1e-8 * max(1.0, np.abs(d1).max())
    assert np.abs(d0 - _theta(h0, n_occ)).max() < 1e-13


def test_o1_d2_second_difference():
    """PAPER.md:164 (Eq. 20): D2 = (1/2) d^2 theta / d lambda^2."""
    h0, h1, n_occ, _, _ = small_problem(n=40, n_occ=17, seed=3)
    d0, d1, d2 = O1.density_matrices(h0, h1, n_occ, order=2)
    h = 2e-3
    fd = (_theta(h0 + h * h1, n_occ) + _theta(h0 - h * h1, n_occ) - 2 * _theta(h0, n_occ)) / (2 * h * h)
    assert np.abs(fd - d2).max() < 2e-4 * max(1.0, np.abs(d2).max())


def test_o1_general_order_matches_finite_differences_and_block_identities():
    """Orders 3 and 4 of the definition (closed_form.density_matrices_to_order): D_k = (1/k!) d^k theta / d lambda^k
    (Eq. 20) against central difference stencils of eigh projectors, the order-k blocks of D^2 = D and
    [H, D] = 0 through the (m+1)N x (m+1)N block upper-triangular matrices, and orders <= 2
    against the separately written order-2 closed form."""
    h0, h1, n_occ, _, _ = small_problem(n=40, n_occ=17, seed=3)
    n = h0.shape[0]
    d = O1.density_matrices_to_order(h0, h1, n_occ, 4)
    for a, b in zip(d, O1.density_matrices(h0, h1, n_occ, order=2)):
        assert np.abs(a - b).max() < 1e-14
    T = lambda x: _theta(h0 + x * h1, n_occ)
    h = 5e-3
    fd3 = (T(2 * h) - 2 * T(h) + 2 * T(-h) - T(-2 * h)) / (2 * h ** 3) / 6.0
    fd4 = (T(2 * h) - 4 * T(h) + 6 * T(0.0) - 4 * T(-h) + T(-2 * h)) / h ** 4 / 24.0
    assert np.abs(fd3 - d[3]).max() < 3e-4 * np.abs(d[3]).max()
    assert np.abs(fd4 - d[4]).max() < 3e-4 * np.abs(d[4]).max()
    # halving h divides the stencil error by four: the mismatch is the stencil's, not the closed form's
    h = 1e-2
    fd3b = (T(2 * h) - 2 * T(h) + 2 * T(-h) - T(-2 * h)) / (2 * h ** 3) / 6.0
    assert 3.0 < np.abs(fd3b - d[3]).max() / np.abs(fd3 - d[3]).max() < 5.0
    z = np.zeros((n, n))
    m = 4
    bd = np.block([[d[c - r] if c >= r else z for c in range(m + 1)] for r in range(m + 1)])
    hs = [h0, h1, z, z, z]
    bh = np.block([[hs[c - r] if c >= r else z for c in range(m + 1)] for r in range(m + 1)])
    assert np.abs(bd @ bd - bd).max() < 1e-11
    assert np.abs(bh @ bd - bd @ bh).max() < 1e-11
    for k in (3, 4):
        assert abs(np.trace(d[k])) < 1e-10 and np.abs(d[k] - d[k].T).max() < 1e-12


def test_o1_invariants_and_block_identities():
    """Blocks of D^2 = D and HD - DH = 0 up to order 2; Tr D0 = N_occ;
    Idemp^(1) = 0."""
    h0, h1, n_occ, _, _ = small_problem()
    d0, d1, d2 = O1.density_matrices(h0, h1, n_occ, order=2)
    inv = O1.invariants(h0, h1, d0, d1, d2)
    for k in ("idem0", "idem1", "idem2", "comm0", "comm1", "comm2", "sym0", "sym1", "sym2"):
        assert inv[k] < 1e-11, (k, inv[k])
    assert abs(inv["tr0"] - n_occ) < 1e-11
    assert abs(inv["tr1"]) < 1e-11 and abs(inv["tr2"]) < 1e-10
    # the same through the 3N x 3N block upper-triangular matrices of PAPER.md:239-243
    n = h0.shape[0]
    z = np.zeros((n, n))
    bd = np.block([[d0, d1, d2], [z, d0, d1], [z, z, d0]])
    bh = np.block([[h0, h1, z], [z, h0, h1], [z, z, h0]])
    assert np.abs(bd @ bd - bd).max() < 1e-11
    assert np.abs(bh @ bd - bd @ bh).max() < 1e-11


def test_o1_special_cases():
    h0, h1, n_occ, _, _ = small_problem(n=64, n_occ=30, seed=11)
    n = h0.shape[0]
    d0, d1 = O1.density_matrices(h0, h1, n_occ)
    assert np.abs(O1.density_matrices(h0, 0 * h1, n_occ)[1]).max() == 0.0
    assert np.abs(O1.density_matrices(h0, h0, n_occ)[1]).max() < 1e-13          # [H0, D0] = 0
    assert np.abs(O1.density_matrices(h0, 3.0 * np.eye(n), n_occ)[1]).max() < 1e-13
    assert np.allclose(O1.density_matrices(h0, 2.5 * h1, n_occ)[1], 2.5 * d1, atol=1e-12)
    e0, e1 = O1.density_matrices(h0 + 0.7 * np.eye(n), h1, n_occ)
    assert np.allclose(e0, d0, atol=1e-12) and np.allclose(e1, d1, atol=1e-11)
    p0, p1 = O1.density_matrices(-h0, -h1, n - n_occ)                           # particle-hole
    assert np.allclose(p0, np.eye(n) - d0, atol=1e-12) and np.allclose(p1, -d1, atol=1e-11)


# ------------------------------------------------------------------ O2: the method
def test_gershgorin_brute_force_and_enclosure():
    rng = np.random.default_rng(5)
    h = symmetric_gaussian(rng, 9, 1.0)
    lo, hi = O2.gershgorin(h)
    los, his = [], []
    for i in range(9):
        r = sum(abs(h[i, j]) for j in range(9) if j != i)
        los.append(h[i, i] - r)
        his.append(h[i, i] + r)
    assert lo == pytest.approx(min(los), abs=1e-14) and hi == pytest.approx(max(his), abs=1e-14)
    w = np.linalg.eigvalsh(h)
    assert lo <= w[0] and w[-1] <= hi


def test_matmul_triple_loop():
    """The library matmul the oracle uses as a step, against three nested loops."""
    rng = np.random.default_rng(2)
    a, b = rng.standard_normal((7, 5)), rng.standard_normal((5, 6))
    c = np.zeros((7, 6))
    for i in range(7):
        for j in range(6):
            for k in range(5):
                c[i, j] += a[i, k] * b[k, j]
    assert np.allclose(O2.Fp64Product().cross(a, b), c, atol=1e-14)


def test_o2_matches_definition_config1(config1):
    """Brute force: the recursion reaches the eigendecomposition result."""
    w = config1
    d0, d1 = O1.density_matrices(w.h0, w.h1, w.n_occ)
    r = O2.dnn_sp2_pt(w.h0, w.h1, w.n_occ)
    assert r.status == "ok"
    assert np.abs(r.d0 - d0).max() < 1e-11
    assert np.abs(r.d1 - d1).max() < 1e-10 * np.abs(d1).max() + 1e-13
    assert abs(np.trace(r.d0) - w.n_occ) < 1e-9
    extra = r.layers - r.layers_d0
    assert 2 <= extra <= 6                      # "around three or four"
    assert 25 <= r.layers <= 45


def test_o2_second_order_matches_definition():
    h0, h1, n_occ, _, _ = small_problem(n=96, n_occ=40, seed=21, gap=0.5, h1_scale=0.02)
    d0, d1, d2 = O1.density_matrices(h0, h1, n_occ, order=2)
    r = O2.dnn_sp2_pt(h0, h1, n_occ, order=2)
    assert r.status == "ok"
    assert np.abs(r.d0 - d0).max() < 1e-11
    assert np.abs(r.d1 - d1).max() < 1e-10 * max(1.0, np.abs(d1).max())
    assert np.abs(r.d2 - d2).max() < 1e-9 * max(1.0, np.abs(d2).max())
    assert r.layers_d0 < r.layers_d1 < r.layers


def test_o2_general_order_matches_definition_and_block_matrix_squaring():
    """Order m of the method (Eq. 26 with the symmetry saving of PAPER.md:325-329): limits against the
    definition at every order; the iterates against squaring the (m+1)N upper-triangular block matrix
    (Eqs. 35-37, 285 Eq. 40) with the logged sigma; the cascaded stops two layers apart (R15)."""
    h0, h1, n_occ, _, _ = small_problem(n=48, n_occ=20, seed=21, gap=0.5, h1_scale=0.02)
    n = h0.shape[0]
    for m in (3, 4):
        d = O1.density_matrices_to_order(h0, h1, n_occ, m)
        r = O2.dnn_sp2_pt(h0, h1, n_occ, order=m)
        assert r.status == "ok" and len(r.dk) == m + 1
        for k in range(m + 1):
            assert np.abs(r.dk[k] - d[k]).max() < 1e-9 * max(1.0, np.abs(d[k]).max()), (m, k)
        assert all(b - a >= 2 for a, b in zip(r.layers_dk, r.layers_dk[1:])) and r.layers == r.layers_dk[m]
        # block-matrix squaring while every order is still being updated (layers 1 .. n_c - 1)
        z = np.zeros((n, n))
        hs = [h0, h1] + [z] * (m - 1)
        bh = np.block([[hs[c - q] if c >= q else z for c in range(m + 1)] for q in range(m + 1)])
        bs = (r.eps_max * np.eye((m + 1) * n) - bh) / (r.eps_max - r.eps_min)
        for k in range(r.layers_d0 - 1):
            bs = r.sigma[k] * (bs @ bs) + (1 - r.sigma[k]) * bs
        assert np.abs(bs[:n, :n] - r.d0).max() < 1e-12
        # from there on S0 is frozen; carry the first block row forward by Eq. 26 with the logged sigma, freezing
        # order k at the layer its test fired
        sk = [bs[:n, k * n:(k + 1) * n].copy() for k in range(m + 1)]
        for layer in range(r.layers_d0, r.layers + 1):
            s = r.sigma[layer - 1]
            xs = [None] + [sum(sk[j] @ sk[k - j] for j in range(k + 1)) for k in range(1, m + 1)]
            for k in range(1, m + 1):
                if layer < r.layers_dk[k]:
                    sk[k] = s * xs[k] + (1 - s) * sk[k]
        for k in range(1, m + 1):
            assert np.abs(sk[k] - r.dk[k]).max() < 1e-10 * max(1.0, np.abs(r.dk[k]).max()), (m, k)


def test_o2_dual_half_general_order_accuracy():
    """O2-dh at order 3: every order within a few 1e-6 of the definition on a well-gapped problem (the same
    floor as the paper's 5e-5 relative 2-norm figure at order 1)."""
    h0, h1, n_occ, _, _ = small_problem(n=96, n_occ=40, seed=21, gap=0.5, h1_scale=0.02)
    d = O1.density_matrices_to_order(h0, h1, n_occ, 3)
    r = O2.dnn_sp2_pt(h0.astype(np.float32), h1.astype(np.float32), n_occ, order=3,
                      product=O2.DualHalfProduct(shift0=14, shift1="auto"), nx_mode="fro")
    assert r.status == "ok"
    for k in range(4):
        assert np.abs(r.dk[k] - d[k]).max() < 5e-5 * max(1.0, np.abs(d[k]).max()), k


def test_o2_h1_equal_h0_gives_zero_response():
    h0, _, n_occ, _, _ = small_problem(n=64, n_occ=30, seed=13)
    r = O2.dnn_sp2_pt(h0, h0, n_occ)
    assert np.abs(r.d1).max() < 1e-12


def test_o2_control_flow_matches_spectral_recursion():
    """O3 is an independent route (eigenvalues only) to sigma_n, N_S, N_X, IdErr, FroErr."""
    for seed in (0, 1, 2):
        h0, h1, n_occ, _, _ = small_problem(n=80, n_occ=33, seed=seed)
        r = O2.dnn_sp2_pt(h0, h1, n_occ)
        eps, v = np.linalg.eigh(h0)
        a = v.T @ h1 @ v
        s = O3.spectral_recursion(eps, n_occ, r.eps_min, r.eps_max, a=a)
        # identical decisions while IdErr is above the fp64 noise floor; at the floor the two
        # routes round differently and may stop a layer or two apart (by design)
        k = max(i for i, e in enumerate(r.id_err[:r.layers_d0]) if e > 1e-9) + 1
        assert k >= r.layers_d0 - 3
        assert s["sigma"][:k] == r.sigma[:k]
        assert abs(s["layers_d0"] - r.layers_d0) <= 2
        assert np.allclose(s["tr_s"][:k], r.tr_s[:k], rtol=0, atol=1e-10)
        assert np.allclose(s["tr_x"][:k], r.tr_x[:k], rtol=0, atol=1e-10)
        assert np.allclose(s["id_err"][:k], r.id_err[:k], rtol=0, atol=1e-10)
        # the first-order norms too, on a run where S0 is frozen by hand at the same layer
    h0, h1, n_occ, _, _ = small_problem(n=40, n_occ=17, seed=5)
    r = O2.dnn_sp2_pt(h0, h1, n_occ)
    eps, v = np.linalg.eigh(h0)
    lam = (r.eps_max - eps) / (r.eps_max - r.eps_min)
    y = -(v.T @ h1 @ v) / (r.eps_max - r.eps_min)
    for k in range(r.layers_d0 - 1):
        sg = r.sigma[k]
        y = sg * (lam[:, None] + lam[None, :]) * y + (1 - sg) * y
        lam = sg * lam * lam + (1 - sg) * lam
    fro1 = np.sqrt(np.sum((y - (lam[:, None] + lam[None, :]) * y) ** 2))
    assert fro1 == pytest.approx(r.fro_err1[r.layers_d0 - 1], rel=1e-6)
    assert np.sqrt(np.sum((lam - lam * lam) ** 2)) == pytest.approx(r.fro_err0, rel=1e-3, abs=1e-14)


def test_o2_block_matrix_equivalence():
    """squaring [[S0,S1],[0,S0]] gives the order-0/1 updates."""
    h0, h1, n_occ, _, _ = small_problem(n=24, n_occ=10, seed=4)
    r = O2.dnn_sp2_pt(h0, h1, n_occ)
    n = h0.shape[0]
    w = r.eps_max - r.eps_min
    z = np.zeros((n, n))
    bh = np.block([[h0, h1], [z, h0]])
    bs = (r.eps_max * np.eye(2 * n) - bh) / w                       # PAPER.md:249 (Eq. 34)
    # layers 1 .. n_c - 1 update both orders with sigma_n (Eqs. 35-37)
    for k in range(r.layers_d0 - 1):
        s = r.sigma[k]
        bs = s * (bs @ bs) + (1 - s) * bs
    assert np.abs(bs[:n, :n] - r.d0).max() < 1e-12                  # S0 froze at n_c - 1
    s1 = bs[:n, n:]
    s0 = bs[:n, :n]
    for k in range(r.layers_d0 - 1, r.layers - 1):                  # S0 frozen, sigma as logged
        s = r.sigma[k]
        x1 = s0 @ s1 + s1 @ s0
        s1 = s * x1 + (1 - s) * s1
    assert np.abs(s1 - r.d1).max() < 1e-12 * max(1.0, np.abs(r.d1).max())


def test_o2_sigma_tie_and_idempotent_input():
    """sign(0) -> +1 (R3); an exactly idempotent S0 stops at layer 1 by IdErr <= 0."""
    n, n_occ = 8, 3
    h0 = np.diag([-1.0] * n_occ + [1.0] * (n - n_occ))
    h1 = np.zeros((n, n))
    r = O2.dnn_sp2_pt(h0, h1, n_occ, bounds=(-1.0, 1.0))
    assert r.layers_d0 == 1 and r.sigma[0] == 1
    assert np.allclose(r.d0, np.diag([1.0] * n_occ + [0.0] * (n - n_occ)))


def test_o2_finite_difference_of_ground_state_sp2():
    """PAPER.md:562-566 (Eq. 83): differencing ground-state DNN-SP2 runs gives the same D1."""
    h0, h1, n_occ, _, _ = small_problem(n=32, n_occ=14, seed=8)
    r = O2.dnn_sp2_pt(h0, h1, n_occ)
    h = 1e-4
    b = (r.eps_min - 0.1, r.eps_max + 0.1)
    dp, _ = O2.dnn_sp2(h0 + h * h1, n_occ, bounds=b)
    dm, _ = O2.dnn_sp2(h0 - h * h1, n_occ, bounds=b)
    fd = (dp - dm) / (2 * h)
    assert np.abs(fd - r.d1).max() < 1e-5 * max(1.0, np.abs(r.d1).max())


def test_cpt_constant_bound():
    """|h'(x)| <= C_pt |x - x^2| on [-0.25, 1.25] with C_pt = 9, for both
    sigma-flip polynomials; and the printed inflection points."""
    x = np.linspace(GOLD["c_pt_interval_lo"], GOLD["c_pt_interval_hi"], 20001)
    for hp in (lambda t: 4 * t - 4 * t ** 3, lambda t: 2 * (2 * t - t * t) * (2 - 2 * t)):
        assert np.all(np.abs(hp(x)) <= GOLD["c_pt"] * np.abs(x - x * x) + 1e-12)
    assert O2.C_PT == GOLD["c_pt"] and O2.C_D0 == GOLD["c_d0"]
    assert O3.C_PT == GOLD["c_pt"] and O3.C_D0 == GOLD["c_d0"]
    assert 1 - 1 / np.sqrt(3) == pytest.approx(GOLD["inflection_2x_minus_x2_squared"], abs=5e-3)
    assert 1 / np.sqrt(3) == pytest.approx(GOLD["inflection_2x2_minus_x4"], abs=5e-3)


# ------------------------------------------------------------------ O2-dh: dual half precision
def test_dual_half_split_accuracy():
    """X ~ X_high + X_low to about 1e-6; FP16 epsilon about 1e-3."""
    rng = np.random.default_rng(9)
    x = rng.uniform(0.25, 1.0, 4096).astype(np.float32)
    hi, lo, _ = O2.DualHalfProduct().split(x, 0)
    assert np.abs(x - hi).max() / 0.25 < 2 * GOLD["fp16_epsilon"]
    rel = np.abs(x - (hi + lo)) / np.abs(x)
    assert rel.max() < GOLD["split_accuracy"]
    assert rel.max() > GOLD["split_accuracy"] / 100          # ... and it is not exact either


def test_dual_half_product_terms():
    """Eqs. 14-16 / 44-46: the product is hi.hi + hi.lo + lo.hi, lo.lo dropped."""
    rng = np.random.default_rng(10)
    n = 64
    a = symmetric_gaussian(rng, n, 0.1).astype(np.float32)
    b = symmetric_gaussian(rng, n, 0.1).astype(np.float32)
    P = O2.DualHalfProduct()
    ah, al, _ = P.split(a, 0)
    bh, bl, _ = P.split(b, 0)
    ref = (ah.astype(np.float64) @ bh + ah.astype(np.float64) @ bl + al.astype(np.float64) @ bh)
    assert np.abs(P.cross(a, b, 0, 0) - ref).max() < 1e-6
    full = (ah + al).astype(np.float64) @ (bh + bl).astype(np.float64)
    dropped = al.astype(np.float64) @ bl
    assert np.allclose(full - ref, dropped, atol=1e-12)
    sq = P.square(a)
    ref2 = ah.astype(np.float64) @ ah + ah.astype(np.float64) @ al + al.astype(np.float64) @ ah
    assert np.abs(sq - ref2).max() < 1e-6
    # exact power-of-two pre-scale leaves the value of the product unchanged (R12/R17)
    P2 = O2.DualHalfProduct(shift0=6, shift1="auto")
    assert np.abs(P2.cross(a, b, 0, 1) - a.astype(np.float64) @ b).max() < 2e-6


def test_dual_half_accuracy_matches_paper_figure():
    """relative 2-norm error of D1 vs the fp64 run 'hovers around 5e-5', on the
    SCC-DFTB-like workload (config 2 construction at a size the oracle finishes in a second),
    with Eq. 13 verbatim (no pre-scale)."""
    w = make_config(2, n=512)
    ref = O2.dnn_sp2_pt(w.h0, w.h1, w.n_occ)
    dh = O2.dnn_sp2_pt(w.h0, w.h1, w.n_occ, product=O2.DualHalfProduct())
    assert dh.status == "ok"
    rel = np.linalg.norm(dh.d1 - ref.d1, 2) / np.linalg.norm(ref.d1, 2)
    assert GOLD["d1_rel_2norm_error"] / 3 < rel < GOLD["d1_rel_2norm_error"] * 3
    assert np.abs(dh.d0 - ref.d0).max() < 5e-5
    assert ref.layers - 5 <= dh.layers <= ref.layers + 1                         # R14
    extra = dh.layers - dh.layers_d0
    assert 2 <= extra <= 6


def test_dual_half_prescale_is_a_refinement(config1):
    """Readings R12/R17: an exact power-of-two pre-scale before the split changes nothing in
    exact arithmetic and only removes fp16 underflow - accuracy must not get worse."""
    w = config1
    ref = O2.dnn_sp2_pt(w.h0, w.h1, w.n_occ)
    plain = O2.dnn_sp2_pt(w.h0, w.h1, w.n_occ, product=O2.DualHalfProduct())
    scaled = O2.dnn_sp2_pt(w.h0, w.h1, w.n_occ, product=O2.DualHalfProduct(shift0=14, shift1="auto"))
    e = lambda r: np.abs(r.d1 - ref.d1).max() / np.abs(ref.d1).max()
    assert e(scaled) < e(plain) and e(scaled) < 5e-4
    assert np.abs(scaled.d0 - ref.d0).max() < 5e-5
    assert abs(scaled.layers - ref.layers) <= 5


# ------------------------------------------------------------------ inputs
def test_workloads_are_seeded_symmetric_and_gapped():
    a = make_config(1)
    b = make_config(1)
    assert np.array_equal(a.h0, b.h0) and np.array_equal(a.h1, b.h1)
    assert a.h0.dtype == np.float32 and np.array_equal(a.h0, a.h0.T) and np.array_equal(a.h1, a.h1.T)
    w = np.linalg.eigvalsh(a.h0.astype(np.float64))
    assert w[a.n_occ] - w[a.n_occ - 1] == pytest.approx(a.meta["gap"], abs=1e-5)
    assert a.meta["gap"] >= 0.2
    t = make_config(2, n=256)
    assert np.array_equal(t.h0, t.h0.T) and t.n_occ == 128
    w = np.linalg.eigvalsh(t.h0.astype(np.float64))
    assert w[t.n_occ] - w[t.n_occ - 1] == pytest.approx(1.0, abs=1e-4)
    assert np.count_nonzero(t.h1 - np.diag(np.diag(t.h1))) == 0                # dipole: diagonal
    lit = make_config(2, n=256, scissor=False)
    w = np.linalg.eigvalsh(lit.h0.astype(np.float64))
    assert w[lit.n_occ] - w[lit.n_occ - 1] < 0.2                                # W2: nearly gapless


def test_ground_state_sp2_matches_the_definition():
    """O2 with the response lines removed (oracle.dnn_sp2, the reference of the order-0 mode): D0 is the
    projector onto the N_occ lowest eigenstates (Eq. 5), and its layer count is the D0 stop
    layer of the full recursion (the ground-state part of Algorithm 1 does not depend on H1)."""
    from workloads import make_config

    for cfg, n in ((1, 96), (2, 128), (4, 160)):
        wl = make_config(cfg, n=n)
        d0, layers = O2.dnn_sp2(wl.h0, wl.n_occ)
        ref0, _ = O1.density_matrices(wl.h0, wl.h1, wl.n_occ)
        assert np.abs(d0 - ref0).max() < 1e-10
        assert abs(np.trace(d0) - wl.n_occ) < 1e-9
        assert layers == O2.dnn_sp2_pt(wl.h0, wl.h1, wl.n_occ).layers_d0


def test_inverse_factor_recursion():
    """PAPER.md:686-703 (A17-A21): Z^T S Z = I, the limit from Z_0 ~ I is the Loewdin factor S^(-1/2), the
    error decays cubically, and the polynomial is the third-order expansion of x^(-1/2) around 1."""
    from oracle.inverse_factor import A_K, inverse_factor

    rng = np.random.default_rng(11)
    n = 60
    g = rng.standard_normal((n, n)) / np.sqrt(n)
    s = np.eye(n) + 0.35 * (g + g.T)
    w, v = np.linalg.eigh(s)
    assert w.min() > 0.05
    z, err = inverse_factor(s)
    assert np.abs(z.T @ s @ z - np.eye(n)).max() < 1e-12                     # A17
    assert np.abs(z - (v / np.sqrt(w)) @ v.T).max() < 1e-11                   # Loewdin factor
    # cubic decay once inside the convergence region: e_{n+1} <= C e_n^3 with a modest C
    tail = [e for e in err if e < 0.3]
    assert len(tail) >= 2 and all(b <= 2.0 * a ** 3 + 1e-13 for a, b in zip(tail, tail[1:]))
    # A21: (1 + d)^(-1/2) = 1 - d/2 + 3 d^2/8 + O(d^3), rewritten in x = 1 + d
    d = 1e-3
    x = 1.0 + d
    assert abs((A_K[0] + A_K[1] * x + A_K[2] * x * x) - x ** -0.5) < 1.0 * d ** 3
    assert abs(sum(A_K) - 1.0) < 1e-15
