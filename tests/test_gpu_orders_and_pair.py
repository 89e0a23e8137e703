"""GPU tests of the SURVEY.md 8(f) rows added or finished in round 2:

  f1  the order-parallel pair: order-0 side and order-1 side as two contexts with a one-way
      per-layer hand-off; on ONE device (two streams, device-local copies) it must reproduce dmpt_run bit for bit;
  f2  general response order: order 3 (Eq. 26, symmetry saving of PAPER.md:325-329) against the oracle
      (O2 at order 3, pinned to the definition at orders 3 and 4 in tests/test_oracle_pins.py);
  f4  the finite-difference stencils of ground-state runs (Eqs. 83-84, Fig. 5) against the
      first-order recursion; f3's congruence transform behind the C ABI.
"""
import numpy as np
import pytest

torch = pytest.importorskip("torch")

pytestmark = pytest.mark.gpu

TOL_D0, TOL_D1, TOL_DK, TOL_TR = 5e-5, 5e-4, 5e-4, 1e-3      # TOL_DK: the D1 tolerance carried to orders 2, 3
C_PROD = 4e-6                                                  # one dual-half product (tests/test_gpu_parity.py)


@pytest.fixture(scope="module")
def dev():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    return torch.device("cuda:0")


def _run1(wl, dev, **kw):
    from paper_2203_09621_b200 import Dmpt
    s = Dmpt(wl.n, device=dev, **kw)
    s.set_hamiltonian(torch.from_numpy(wl.h0).to(dev), torch.from_numpy(wl.h1).to(dev), wl.n_occ)
    r = s.run()
    out = (r, r.d0.cpu().numpy(), r.d1.cpu().numpy())
    s.close()
    return out


def _run_pair(wl, dev, **kw):
    from paper_2203_09621_b200.binding import DmptPair
    p = DmptPair(wl.n, device0=dev, device1=dev, **kw)
    p.set_hamiltonian(torch.from_numpy(wl.h0).to(dev), torch.from_numpy(wl.h1).to(dev), wl.n_occ)
    r = p.run()
    out = (r, r.d0.cpu().numpy(), r.d1.cpu().numpy())
    p.close()
    return out


# ------------------------------------------------------------------------------------------ f1
@pytest.mark.parametrize("cfg,n", [(1, 256), (2, 512), (3, 768), (4, 1024), (2, 1284), (1, 37)])
def test_pair_on_one_device_is_bit_identical_to_run(dev, cfg, n):
    """Both sides on one GPU: D0, D1, the layer counts and every per-layer record equal dmpt_run's exactly."""
    from workloads import make_config

    wl = make_config(cfg, n=n)
    a, a0, a1 = _run1(wl, dev)
    b, b0, b1 = _run_pair(wl, dev)
    assert a.status == 0 and b.status == 0
    assert (a.layers, a.layers_d0, a.layers_d1) == (b.layers, b.layers_d0, b.layers_d1)
    assert np.array_equal(a0, b0) and np.array_equal(a1, b1)
    assert a.sigma == b.sigma
    assert a.eps_min == b.eps_min and a.eps_max == b.eps_max and a.fro_err0 == b.fro_err0
    nc = a.layers_d0
    assert a.tr_s[:nc] == b.tr_s[:nc] and a.tr_x[:nc] == b.tr_x[:nc] and a.id_err[:nc] == b.id_err[:nc]
    fa, fb = np.array(a.fro_err1), np.array(b.fro_err1)
    assert np.array_equal(np.isnan(fa), np.isnan(fb)) and np.array_equal(fa[~np.isnan(fa)], fb[~np.isnan(fb)])


def test_pair_matches_oracle_and_multi_wave(dev):
    """The pair against the oracle proper (O2, fp64) on config 2 at n = 2048, and bit-identity with dmpt_run at
    n = 4096 (272 pair tiles = 3.7 waves: the two sides' cooperative launches take turns on the device)."""
    from oracle.dnn_sp2_pt import dnn_sp2_pt
    from workloads import make_config

    wl = make_config(2)
    ref = dnn_sp2_pt(wl.h0, wl.h1, wl.n_occ)
    r, d0, d1 = _run_pair(wl, dev)
    assert r.status == 0
    assert np.abs(d0 - ref.d0).max() <= TOL_D0
    assert np.abs(d1 - ref.d1).max() <= TOL_D1 * np.abs(ref.d1).max()
    assert abs(np.trace(d0.astype(np.float64)) - wl.n_occ) <= TOL_TR
    assert ref.layers - 8 <= r.layers <= ref.layers + 2
    wl = make_config(4, n=4096)
    a, a0, a1 = _run1(wl, dev)
    b, b0, b1 = _run_pair(wl, dev)
    assert (a.layers, a.layers_d0) == (b.layers, b.layers_d0)
    assert np.array_equal(a0, b0) and np.array_equal(a1, b1)


def test_pair_options_and_errors(dev):
    """Caller-supplied bounds and the plain Eq. 13 / Eq. 43 split go through the pair unchanged; max_layers and bad
    arguments are reported as dmpt_run reports them."""
    from paper_2203_09621_b200 import binding as B
    from workloads import make_config

    wl = make_config(1, n=200)
    ev = np.linalg.eigvalsh(wl.h0.astype(np.float64))
    kw = dict(bounds=(ev[0] - 1e-3, ev[-1] + 1e-3))
    a, a0, a1 = _run1(wl, dev, **kw)
    b, b0, b1 = _run_pair(wl, dev, **kw)
    assert a.layers == b.layers and np.array_equal(a0, b0) and np.array_equal(a1, b1)
    kw = dict(s0_shift=0, s1_autoscale=False)
    a, a0, a1 = _run1(wl, dev, **kw)
    b, b0, b1 = _run_pair(wl, dev, **kw)
    assert a.layers == b.layers and np.array_equal(a0, b0) and np.array_equal(a1, b1)
    # max_layers: both report DMPT_ENOCONV and the same last iterate
    from paper_2203_09621_b200 import Dmpt
    s = Dmpt(wl.n, device=dev, max_layers=7)
    s.set_hamiltonian(torch.from_numpy(wl.h0).to(dev), torch.from_numpy(wl.h1).to(dev), wl.n_occ)
    ra = s.run(check=False)
    p = B.DmptPair(wl.n, device0=dev, device1=dev, max_layers=7)
    p.set_hamiltonian(torch.from_numpy(wl.h0).to(dev), torch.from_numpy(wl.h1).to(dev), wl.n_occ)
    rb = p.run(check=False)
    assert ra.status == B.DMPT_ENOCONV and rb.status == B.DMPT_ENOCONV and ra.layers == rb.layers == 7
    assert torch.equal(ra.d0, rb.d0) and torch.equal(ra.d1, rb.d1)
    p.close()
    s.close()
    # argument errors
    assert B.dmpt_pair_workspace_bytes(0, 0) == 0 and B.dmpt_pair_workspace_bytes(64, 2) == 0
    ws = torch.empty(B.dmpt_pair_workspace_bytes(64, 1), dtype=torch.uint8, device=dev)
    opt = B.dmpt_default_options()
    opt.order = 2
    with pytest.raises(B.DmptError):
        B.dmpt_pair_create(64, opt, 0, ws.data_ptr(), ws.numel(), 0, ws.data_ptr(), ws.numel())
    with pytest.raises(B.DmptError):
        B.dmpt_pair_create(64, None, 0, ws.data_ptr(), ws.numel(), 99, ws.data_ptr(), ws.numel())
    with pytest.raises(B.DmptError):          # side-0 workspace too small
        B.dmpt_pair_create(64, None, 0, ws.data_ptr(), 1024, 0, ws.data_ptr(), ws.numel())


# ------------------------------------------------------------------------------------------ f2: order 3
@pytest.mark.parametrize("n", [40, 128, 333, 640])
def test_layer_products3_match_fp64(dev, n):
    """X3 = S0 S3 + S3 S0 + S1 S2 + S2 S1 (Eq. 26 at k = 3) through the order-3 pass, element by element
    within the bound of its four dual-half products."""
    from paper_2203_09621_b200 import Dmpt

    rng = np.random.default_rng(17 * n)
    a = rng.uniform(-1, 1, size=(n, n)) / np.sqrt(n)
    s0 = ((a + a.T) / 2 + np.diag(rng.uniform(0, 1, size=n))).astype(np.float32)
    sym = lambda sc: (lambda b: (sc * (b + b.T)).astype(np.float32))(rng.standard_normal((n, n)))
    s1, s2, s3 = sym(0.37), sym(2.1e-3), sym(5.0e-5)
    s = Dmpt(n, device=dev, order=3)
    x3 = s.layer_products3(*(torch.from_numpy(m).to(dev) for m in (s0, s1, s2, s3))).double().cpu().numpy()
    s.close()
    s0d, s1d, s2d, s3d = (m.astype(np.float64) for m in (s0, s1, s2, s3))
    p3, q3 = s0d @ s3d, s1d @ s2d
    ref = p3 + p3.T + q3 + q3.T
    m = np.abs(s0d - 0.5 * np.eye(n))
    a1, a2, a3 = np.abs(s1d), np.abs(s2d), np.abs(s3d)
    bound = (C_PROD * (m @ a3 + a3 @ m + a1 @ a2 + a2 @ a1) + 3e-7 * np.abs(ref) + 1e-7 * a3.max())
    assert np.all(np.abs(x3 - ref) <= bound), f"X3: worst ratio {np.max(np.abs(x3 - ref) / bound):.2f}"
    assert np.array_equal(x3, x3.T)


def _run3(wl, dev, h1=None, **kw):
    from paper_2203_09621_b200 import Dmpt
    s = Dmpt(wl.n, device=dev, order=3, **kw)
    s.set_hamiltonian(torch.from_numpy(wl.h0).to(dev), torch.from_numpy(wl.h1 if h1 is None else h1).to(dev), wl.n_occ)
    r = s.run_orders()
    out = tuple(m.double().cpu().numpy() for m in (r.d0, r.d1, r.d2, r.d3))
    s.close()
    return r, out


@pytest.mark.parametrize("cfg,n", [(1, 256), (5, 512), (2, 1284), (4, 1024)])
def test_third_order_matches_oracle(dev, cfg, n):
    """Order 3 at sizes the oracle finishes in seconds: every order against O2 (fp64) run to order 3, the layer
    counts against O2-dh, the cascade of stops, and orders 0-2 bit-identical to the order-2 run."""
    from oracle.dnn_sp2_pt import DualHalfProduct, dnn_sp2_pt
    from paper_2203_09621_b200 import Dmpt
    from workloads import make_config

    wl = make_config(cfg, n=n)
    ref = dnn_sp2_pt(wl.h0, wl.h1, wl.n_occ, order=3)
    assert ref.status == "ok"
    r, d = _run3(wl, dev)
    assert r.status == 0
    assert np.abs(d[0] - ref.dk[0]).max() <= TOL_D0
    assert abs(np.trace(d[0]) - wl.n_occ) <= TOL_TR
    for k, tol in ((1, TOL_D1), (2, TOL_DK), (3, TOL_DK)):
        e = np.abs(d[k] - ref.dk[k]).max() / np.abs(ref.dk[k]).max()
        assert e <= tol, f"order {k}: max|D - ref|/max|ref| = {e:.3e}"
        assert np.array_equal(d[k], d[k].T)
        assert abs(np.trace(d[k])) <= 1e-3 * np.abs(ref.dk[k]).max() * np.sqrt(n)
    # layer counts: within 2 of the interval the two O2-dh variants span, for every stop of the cascade
    dh = [dnn_sp2_pt(wl.h0, wl.h1, wl.n_occ, order=3, product=DualHalfProduct(shift0=14, shift1="auto"), nx_mode=m)
          for m in ("trace", "fro")]
    got = [r.layers_d0, r.layers_d1, r.layers_d2, r.layers_d3]
    for k in range(4):
        want = [x.layers_dk[k] for x in dh]
        assert min(want) - 2 <= got[k] <= max(want) + 2, (k, got, [x.layers_dk for x in dh], ref.layers_dk)
    assert r.layers == r.layers_d3
    assert all(b - a >= 2 for a, b in zip(got, got[1:]))                  # cascade, reading R15
    assert len(r.fro_err3) == r.layers and np.isfinite(r.fro_err3[r.layers_d2 - 1]) and np.isnan(r.fro_err3[0])
    # FroErr3 of the last layer against its definition on the returned iterates
    am = np.abs(d[0] - 0.5 * np.eye(n))
    f3 = np.linalg.norm(d[3] - (d[0] @ d[3] + d[3] @ d[0] + d[1] @ d[2] + d[2] @ d[1]))
    b3 = (C_PROD * np.linalg.norm(am @ np.abs(d[3]) + np.abs(d[3]) @ am + 2 * np.abs(d[1]) @ np.abs(d[2]))
          + 1e-7 * np.abs(d[3]).max())
    assert abs(r.fro_err3[r.layers - 1] - f3) <= b3, (r.fro_err3[r.layers - 1], f3, b3)
    # orders 0-2 of an order-3 run are the order-2 run (same kernels, same decisions)
    s = Dmpt(wl.n, device=dev, order=2)
    s.set_hamiltonian(torch.from_numpy(wl.h0).to(dev), torch.from_numpy(wl.h1).to(dev), wl.n_occ)
    r2 = s.run()
    assert r2.layers == r.layers_d2
    for k, m in enumerate((r2.d0, r2.d1, r2.d2)):
        assert np.array_equal(m.double().cpu().numpy(), d[k]), k
    s.close()


def test_third_order_special_cases_and_scaling(dev):
    """H1 = 0 -> D1 = D2 = D3 = 0 exactly; D_k(c H1) = c^k D_k(H1) for a power of two c bit for bit (every scale in
    the path is a power of two); determinism."""
    from workloads import make_config

    wl = make_config(1, n=200)
    r, d = _run3(wl, dev, h1=np.zeros_like(wl.h1))
    assert r.status == 0 and all(np.abs(d[k]).max() == 0.0 for k in (1, 2, 3))
    ra, da = _run3(wl, dev)
    rb, db = _run3(wl, dev, wave_sync=False)
    assert ra.layers == rb.layers and all(np.array_equal(x, y) for x, y in zip(da, db))
    c = 2.0 ** -6
    rc, dc = _run3(wl, dev, h1=(wl.h1 * np.float32(c)))
    assert rc.status == 0 and rc.layers == ra.layers
    for k in (1, 2, 3):
        assert np.array_equal(dc[k], da[k] * c ** k), k


def test_order3_argument_checks(dev):
    from paper_2203_09621_b200 import binding as B

    assert B.dmpt_workspace_bytes(64, 3) > B.dmpt_workspace_bytes(64, 2) > 0 and B.dmpt_workspace_bytes(64, 4) == 0
    s = B.Dmpt(64, device=dev, order=3)
    z = torch.zeros((64, 64), device=dev)
    assert B.dmpt_run(s.ctx, z.data_ptr(), z.data_ptr(), z.data_ptr(), 64, None) == B.DMPT_EINVAL     # needs dmpt_run_orders
    assert B.dmpt_run_orders(s.ctx, [z.data_ptr()] * 4, 64, None) == B.DMPT_ESTATE                    # no Hamiltonian yet
    s2 = B.Dmpt(64, device=dev, order=2)
    assert B.dmpt_layer_products3(s2.ctx, *([z.data_ptr()] * 4), 64, z.data_ptr(), 64) == B.DMPT_EINVAL
    s.close()
    s2.close()


# ------------------------------------------------------------------------------------------ f4
def test_finite_difference_stencils_against_the_first_order_recursion(dev):
    """Fig. 5 on a config-2-like input: D1 from 2 and 4 ground-state runs (dmpt_fd_response) over a
    sweep of h, against the definition O1, next to the first-order run.
      * both stencils converge at their order while truncation dominates (error ratio between two h a factor 2
        apart: ~4 for Eq. 83, ~16 for Eq. 84) - this pins the stencil weights;
      * the error turns up again for small h (rounding noise / h): an optimal h exists and has to be searched;
      * at its best h the 2-point stencil is several times less accurate than DNN-SP2-PT, the 4-point stencil
        comes closer but does not beat it, at 8 instead of 5 products per layer."""
    from oracle.closed_form import density_matrices
    from paper_2203_09621_b200 import Dmpt
    from workloads import make_config

    wl = make_config(2, n=768)
    n = wl.n
    _, ref = density_matrices(wl.h0, wl.h1, wl.n_occ)
    nref = np.linalg.norm(ref, 2)
    h0, h1 = torch.from_numpy(wl.h0).to(dev), torch.from_numpy(wl.h1).to(dev)
    r, _, d1 = _run1(wl, dev)
    e_pt = np.linalg.norm(d1.astype(np.float64) - ref, 2) / nref
    assert e_pt <= 1e-4                                  # the paper's ~5e-5 relative 2-norm
    gs = Dmpt(n, order=0, device=dev)
    scale = float(np.abs(wl.h1).max())
    steps = [2.0 ** -k for k in range(1, 13)]            # h max|H1| from 0.5 down to 2.4e-4
    err = {2: [], 4: []}
    for points in (2, 4):
        for hs in steps:
            d, layers, ms = gs.fd_response(h0, h1, wl.n_occ, hs / scale, points)
            assert len(layers) == points and all(x > 5 for x in layers) and ms > 0
            assert torch.equal(d, d.t())
            err[points].append(np.linalg.norm(d.double().cpu().numpy() - ref, 2) / nref)
    gs.close()
    print("DMPT", e_pt, "2-point", err[2], "4-point", err[4])
    for points, rate in ((2, 4.0), (4, 16.0)):
        e = err[points]
        # the truncation-dominated part: the largest steps, while the error is still well above the stencil's own
        # noise floor (measured at n = 768: 2-point 0.038, 0.0093, 0.0023, 5.7e-4, 2.0e-4, then up again;
        # 4-point 0.0146, 6.8e-4, 1.4e-4, 1.0e-4, then up again; DNN-SP2-PT 7.5e-6)
        ratios = []
        for i in range(len(e) - 1):
            if e[i + 1] < 5 * min(e):
                break
            ratios.append(e[i] / e[i + 1])
        assert ratios and all(0.6 * rate <= q <= 2.0 * rate for q in ratios), (points, ratios, e)
        assert e[-1] > 2 * min(e)                          # too small a step: noise / h
    assert min(err[2]) >= 3 * e_pt
    assert min(err[4]) >= 1.0 * e_pt and min(err[4]) <= min(err[2])


def test_fd_response_argument_checks(dev):
    from paper_2203_09621_b200 import binding as B

    z = torch.zeros((64, 64), device=dev)
    s1 = B.Dmpt(64, device=dev, order=1)
    assert B.dmpt_fd_response(s1.ctx, z.data_ptr(), z.data_ptr(), 64, 20, 1e-2, 2, z.data_ptr(), 64)[0] == B.DMPT_EINVAL
    s1.close()
    s0 = B.Dmpt(64, device=dev, order=0)
    for kw in (dict(h=0.0), dict(points=3), dict(n_occ=0), dict(ld=32)):
        a = dict(h=1e-2, points=2, n_occ=20, ld=64)
        a.update(kw)
        rc = B.dmpt_fd_response(s0.ctx, z.data_ptr(), z.data_ptr(), a["ld"], a["n_occ"], a["h"], a["points"],
                                z.data_ptr(), 64)[0]
        assert rc == B.DMPT_EINVAL, kw
    s0.close()


def test_congruence_both_directions(dev):
    """dmpt_congruence (Eq. 81, A17-A18): Z^T X Z and Z X Z^T for a NON-symmetric Z, against fp64, and
    identical to the two chained dmpt_product_nt calls with a host-side transpose."""
    from paper_2203_09621_b200 import Dmpt

    for n in (96, 333, 640):
        rng = np.random.default_rng(n)
        z = (rng.standard_normal((n, n)) / np.sqrt(n) + np.eye(n)).astype(np.float32)
        b = rng.standard_normal((n, n))
        x = ((b + b.T) / 2).astype(np.float32)
        s = Dmpt(n, device=dev)
        zt, xt = torch.from_numpy(z).to(dev), torch.from_numpy(x).to(dev)
        c1 = s.congruence(zt, xt, transpose_z=True)
        c2 = s.congruence(zt, xt, transpose_z=False)
        zT = zt.t().contiguous()
        assert torch.equal(c1, s.product_nt(s.product_nt(zT, xt), zT))
        assert torch.equal(c2, s.product_nt(s.product_nt(zt, xt), zt))
        s.close()
        zd, xd = z.astype(np.float64), x.astype(np.float64)
        for c, ref in ((c1, zd.T @ xd @ zd), (c2, zd @ xd @ zd.T)):
            assert np.abs(c.double().cpu().numpy() - ref).max() <= 1e-5 * np.abs(ref).max()


# ------------------------------------------------------------------------------------------ bounds = 2 (reading R18)
@pytest.mark.parametrize("cfg,n", [(1, 256), (2, 512), (3, 768), (4, 1024), (5, 640), (1, 37)])
def test_lanczos_bounds_enclose_the_spectrum_and_save_layers(dev, cfg, n):
    """dmpt_options::bounds = 2: the Gershgorin discs tightened by Lanczos steps on the device.  The pair of numbers
    the run reports (a) encloses the spectrum of H0 (numpy eigvalsh), (b) is much tighter than the discs, and - handed
    to the oracle unchanged (R18) - (c) the run matches O2 (fp64) within the four tolerances and O2-dh's layer count,
    in fewer layers than the Gershgorin run."""
    from oracle.dnn_sp2_pt import DualHalfProduct, dnn_sp2_pt, gershgorin
    from paper_2203_09621_b200 import Dmpt
    from workloads import make_config

    wl = make_config(cfg, n=n)
    ev = np.linalg.eigvalsh(wl.h0.astype(np.float64))
    g_lo, g_hi = gershgorin(wl.h0)
    s = Dmpt(wl.n, device=dev, bounds="lanczos", order=1)
    h0, h1 = torch.from_numpy(wl.h0).to(dev), torch.from_numpy(wl.h1).to(dev)
    s.set_hamiltonian(h0, h1, wl.n_occ)
    r = s.run()
    d0, d1 = r.d0.double().cpu().numpy(), r.d1.double().cpu().numpy()
    s.close()
    assert r.status == 0
    assert r.eps_min <= ev[0] and r.eps_max >= ev[-1], (r.eps_min, ev[0], ev[-1], r.eps_max)
    assert g_lo - 1e-9 <= r.eps_min and r.eps_max <= g_hi + 1e-9
    width, true = r.eps_max - r.eps_min, ev[-1] - ev[0]
    assert width <= 2.0 * true, (width, true, g_hi - g_lo)
    ref = dnn_sp2_pt(wl.h0, wl.h1, wl.n_occ, bounds=(r.eps_min, r.eps_max))
    assert ref.status == "ok"
    assert np.abs(d0 - ref.d0).max() <= TOL_D0
    assert np.abs(d1 - ref.d1).max() <= TOL_D1 * np.abs(ref.d1).max()
    assert abs(np.trace(d0) - wl.n_occ) <= TOL_TR
    dh = [dnn_sp2_pt(wl.h0, wl.h1, wl.n_occ, bounds=(r.eps_min, r.eps_max),
                     product=DualHalfProduct(shift0=14, shift1="auto"), nx_mode=m) for m in ("trace", "fro")]
    want = [x.layers for x in dh]
    assert min(want) - 2 <= r.layers <= max(want) + 2, (r.layers, want, ref.layers)
    g, _, _ = _run1(wl, dev)
    assert r.layers <= g.layers and (g_hi - g_lo < 3 * true or r.layers <= g.layers - 2), (r.layers, g.layers)


def test_lanczos_bounds_degenerate_and_options(dev):
    """A diagonal H0 with two distinct levels: the Krylov space is invariant after two steps - the discs are kept
    (they are exact for a diagonal matrix).  More steps never loosen the bounds beyond the discs; the pair carries the
    option to its order-0 side; bad option values are refused."""
    from paper_2203_09621_b200 import Dmpt
    from paper_2203_09621_b200 import binding as B
    from workloads import make_config

    n, n_occ = 64, 24
    h0 = np.diag(np.array([-1.0] * n_occ + [1.0] * (n - n_occ), dtype=np.float32))
    rng = np.random.default_rng(5)
    b = rng.standard_normal((n, n)).astype(np.float32)
    h1 = ((b + b.T) / 2).astype(np.float32)
    s = Dmpt(n, device=dev, bounds="lanczos")
    s.set_hamiltonian(torch.from_numpy(h0).to(dev), torch.from_numpy(h1).to(dev), n_occ)
    r = s.run()
    s.close()
    assert r.status == 0 and (r.eps_min, r.eps_max) == (-1.0, 1.0)
    # extreme eigenvectors (e_1 -+ e_2)/sqrt(2), which a start vector of equal-magnitude entries can miss by symmetry
    n2 = 96
    hs = np.diag(rng.uniform(-1.0, 1.0, n2)).astype(np.float32)
    hs[0, 0] = hs[1, 1] = 0.0
    hs[0, 1] = hs[1, 0] = -3.0
    evs = np.linalg.eigvalsh(hs.astype(np.float64))
    b2 = rng.standard_normal((n2, n2)).astype(np.float32)
    s = Dmpt(n2, device=dev, bounds="lanczos", lanczos_steps=30)
    s.set_hamiltonian(torch.from_numpy(hs).to(dev), torch.from_numpy(((b2 + b2.T) / 2).astype(np.float32)).to(dev), 40)
    r = s.run(check=False)
    s.close()
    assert r.eps_min <= evs[0] and r.eps_max >= evs[-1], (r.eps_min, evs[0], evs[-1], r.eps_max)
    wl = make_config(1, n=200)
    ev = np.linalg.eigvalsh(wl.h0.astype(np.float64))
    widths = []
    for steps in (4, 20, 64):
        s = Dmpt(wl.n, device=dev, bounds="lanczos", lanczos_steps=steps)
        s.set_hamiltonian(torch.from_numpy(wl.h0).to(dev), torch.from_numpy(wl.h1).to(dev), wl.n_occ)
        r = s.run()
        s.close()
        assert r.status == 0 and r.eps_min <= ev[0] and r.eps_max >= ev[-1], steps
        widths.append(r.eps_max - r.eps_min)
    a, a0, a1 = _run1(wl, dev, bounds="lanczos")
    b_, b0, b1 = _run_pair(wl, dev, bounds="lanczos")
    assert (a.eps_min, a.eps_max, a.layers) == (b_.eps_min, b_.eps_max, b_.layers)
    assert np.array_equal(a0, b0) and np.array_equal(a1, b1)
    opt = B.dmpt_default_options()
    ws = torch.empty(B.dmpt_workspace_bytes(64, 1), dtype=torch.uint8, device=dev)
    for field, val in (("bounds", 3), ("bounds", -1), ("lanczos_steps", -2)):
        o = B.dmpt_default_options()
        setattr(o, field, val)
        with pytest.raises(B.DmptError):
            B.dmpt_create(64, o, ws.data_ptr(), ws.numel())


# ------------------------------------------------------------------------------------------ the two final epilogues
@pytest.mark.parametrize("cfg,n", [(1, 256), (2, 640), (4, 1284), (3, 200)])
def test_epilogue_paths_are_bit_identical(dev, cfg, n):
    """The final epilogue through shared memory and TMA (off-diagonal blocks: box stores; blocks the diagonal crosses:
    masked coalesced stores from the same staging) and round 1's row-per-thread epilogue (epilogue_direct = 1) do the
    same arithmetic: D0, D1 and the layer counts are equal bit for bit, the iterates stay exactly symmetric, and the
    per-layer scalars (summed in a different order) agree to rounding."""
    from workloads import make_config

    wl = make_config(cfg, n=n)
    a, a0, a1 = _run1(wl, dev)
    b, b0, b1 = _run1(wl, dev, epilogue_direct=True)
    assert a.status == 0 and b.status == 0
    assert (a.layers, a.layers_d0, a.layers_d1, a.sigma) == (b.layers, b.layers_d0, b.layers_d1, b.sigma)
    assert np.array_equal(a0, b0) and np.array_equal(a1, b1)
    assert np.array_equal(a0, a0.T) and np.array_equal(a1, a1.T)
    assert np.allclose(a.tr_s, b.tr_s, rtol=1e-12, atol=1e-9)
    assert np.allclose(a.id_err[:a.layers_d0], b.id_err[:a.layers_d0], rtol=1e-6, atol=1e-7 * n)
    assert abs(a.fro_err0 - b.fro_err0) <= 1e-5 * a.fro_err0


def test_bench_side_modes_print_one_json_line(dev):
    """bench.py --fd and --order-parallel on the small configuration: one JSON line each, exit code 0 (the pair's line
    also asserts bit-identity with the single-context run)."""
    import json
    import os
    import subprocess
    import sys

    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    for flags in (["--fd", "--config", "1", "--fd-steps", "0.01", "0.05", "0.2"],
                  ["--order-parallel", "--config", "1", "--steps", "2", "--warmup", "2"]):
        r = subprocess.run([sys.executable, os.path.join(root, "bench.py")] + flags, capture_output=True, text=True,
                           timeout=600)
        assert r.returncode == 0, r.stderr[-2000:]
        lines = [ln for ln in r.stdout.splitlines() if ln.startswith("{")]
        assert len(lines) == 1
        d = json.loads(lines[0])
        assert d["mode"] in ("fd", "order-parallel") and d["gpu_launches"] > 0 and d["data"] == "synthetic"
        if d["mode"] == "fd":
            assert len(d["fd_sweep"]) == 6 and d["best"]["two_point_over_dmpt"] > 1.0 and d["cpu_baseline"]["kind"] == "oracle"
        else:
            assert d["config"]["bit_identical_to_single_context"] is True and d["value"] > 0


# ------------------------------------------------------------------------------------------ device-side layer loop
@pytest.mark.parametrize("cfg,n,order,nf", [(1, 256, 1, 1), (1, 256, 0, 1), (1, 200, 2, 1), (2, 512, 1, 2), (4, 1284, 1, 1)])
def test_loop_graph_is_bit_identical_to_chunked_launches(dev, cfg, n, order, nf):
    """dmpt_options::loop_graph: the layer loop as ONE launch of a CUDA graph whose WHILE node is driven by the control
    step on the device (no flag for the host).  Same kernels: D0, D1 (D2, every field), layer counts and sigma equal
    the chunked-launch run bit for bit; the launch count is reported from the layers."""
    from paper_2203_09621_b200 import Dmpt
    from workloads import make_config

    wl = make_config(cfg, n=n)
    h0, h1 = torch.from_numpy(wl.h0).to(dev), torch.from_numpy(wl.h1).to(dev)
    got = {}
    for lg in (False, True):
        s = Dmpt(n, device=dev, order=order, num_fields=nf, loop_graph=lg)
        if nf > 1:
            s.set_hamiltonian_fields(h0, [h1, (h1 * 0.5).contiguous()], wl.n_occ)
            r = s.run_fields()
            r = s.run_fields()                      # a second run re-uses the instantiated graph
            mats = [r.d0] + list(r.d1)
        else:
            s.set_hamiltonian(h0, h1 if order else None, wl.n_occ)
            r = s.run_orders()
            r = s.run_orders()
            mats = [m for m in (r.d0, r.d1, r.d2) if m is not None]
        assert r.status == 0
        got[lg] = (r, [m.clone() for m in mats])
        s.close()
    (a, ma), (b, mb) = got[False], got[True]
    assert (a.layers, a.layers_d0, a.layers_d1, a.layers_d2, a.sigma) == (b.layers, b.layers_d0, b.layers_d1, b.layers_d2, b.sigma)
    assert all(torch.equal(x, y) for x, y in zip(ma, mb))
    passes = order if order >= 2 else (2 if nf > 1 else 1)
    assert b.launches >= b.layers * passes and b.launches <= b.layers * passes + 12


def test_loop_graph_ends_on_errors_and_follows_n_occ(dev):
    """The WHILE loop must also end when the run is over before its first layer (degenerate bounds) and at max_layers;
    the graph holds a copy of the problem description and is rebuilt when n_occ changes."""
    from paper_2203_09621_b200 import Dmpt
    from paper_2203_09621_b200 import binding as B
    from workloads import make_config

    s = Dmpt(128, device=dev, loop_graph=True)
    z = torch.zeros((128, 128), device=dev)
    s.set_hamiltonian(z, z, 64)
    r = s.run(check=False)
    assert r.status == B.DMPT_EDEGENERATE and r.layers == 0
    s.close()
    wl = make_config(1)
    h0, h1 = torch.from_numpy(wl.h0).to(dev), torch.from_numpy(wl.h1).to(dev)
    s = Dmpt(256, device=dev, loop_graph=True, max_layers=5)
    s.set_hamiltonian(h0, h1, wl.n_occ)
    r = s.run(check=False)
    assert r.status == B.DMPT_ENOCONV and r.layers == 5
    s.close()
    s = Dmpt(256, device=dev, loop_graph=True)
    t = Dmpt(256, device=dev)
    for n_occ in (wl.n_occ, 100, wl.n_occ):
        s.set_hamiltonian(h0, h1, n_occ)
        t.set_hamiltonian(h0, h1, n_occ)
        a, b = s.run(check=False), t.run(check=False)
        assert a.status == b.status and a.layers == b.layers and torch.equal(a.d0, b.d0) and torch.equal(a.d1, b.d1)
    s.close()
    t.close()
