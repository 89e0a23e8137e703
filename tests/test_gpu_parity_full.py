"""Multi-wave parity of the CUDA path (through the C ABI) against the oracle itself.  Needs a B200; `slow`.

What each full size is compared with (north_star tolerances):
    n = 4096  (configs 2, 4; 272 pair tiles = 3.7 waves of 74 CTA pairs)   oracle O2 itself (fp64, ~25 s): this file
    N = 8192  (config 3)   the definition O1 on the CPU (numpy eigh) and O3 with the full response for the layer count
    N = 16384 (config 4), N = 32768 (config 5)   values: device fp64 cross-reference, pinned to O1 at N = 256, 2048 and
              8192; layer count: O3 on the spectrum the generator constructed      (those three: tests/test_gpu_parity.py)
"""
import numpy as np
import pytest

torch = pytest.importorskip("torch")

from test_gpu_parity import _check_against, _o3_d0, _run  # noqa: E402

pytestmark = [pytest.mark.gpu, pytest.mark.slow]


@pytest.fixture(scope="module")
def dev():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    return torch.device("cuda:0")


@pytest.mark.parametrize("cfg", [2, 4])
def test_multi_wave_launch_matches_the_oracle_itself(dev, cfg):
    """n = 4096: 272 pair tiles on 74 CTA pairs = 3.7 waves - the persistent tile loop, the wave barrier and the
    multi-wave tile order - compared element by element with oracle.dnn_sp2_pt (O2, fp64), not a cross-reference."""
    from oracle.dnn_sp2_pt import dnn_sp2_pt
    from workloads import make_config

    wl = make_config(cfg, n=4096, device="cuda")
    ref = dnn_sp2_pt(wl.h0, wl.h1, wl.n_occ)
    assert ref.status == "ok"
    res, d0, d1 = _run(wl, dev)
    assert res.status == 0
    e0, e1, tr = _check_against(ref.d0, ref.d1, wl.n_occ, d0, d1)
    assert np.array_equal(d0, d0.T) and np.array_equal(d1, d1.T)
    assert ref.layers - 5 <= res.layers <= ref.layers + 2, (res.layers, ref.layers)
    assert ref.layers_d0 - 5 <= res.layers_d0 <= ref.layers_d0 + 2, (res.layers_d0, ref.layers_d0)
    o3 = _o3_d0(wl)
    assert o3["layers_d0"] == ref.layers_d0            # O3 on the constructed spectrum predicts O2's D0 stop layer
    # per-layer IdErr over the common sigma prefix (a6); fp32 storage of S0 at n = 4096: 2e-4 per trace
    k = 0
    while k < min(res.layers_d0, ref.layers_d0) - 1 and res.sigma[k] == ref.sigma[k]:
        k += 1
    assert k >= min(res.layers_d0, ref.layers_d0) - 3
    for i in range(k):
        assert abs(res.id_err[i] - ref.id_err[i]) <= 1e-3, (i, res.id_err[i], ref.id_err[i])
    print(f"config {cfg} @ n=4096: layers gpu {res.layers} (D0 {res.layers_d0}) O2 fp64 {ref.layers} (D0 {ref.layers_d0}) "
          f"max|D0 err| {e0:.2e} D1 {e1:.2e} tr {tr:.2e}")


def test_pair_full_size_is_bit_identical_to_run(dev):
    """SURVEY.md 8(f) f1 at N = 8192 (config 3; 1056 pair tiles, 14.3 waves, cooperative launches of the two sides
    taking turns on one device): D0, D1 and the layer counts of the order-parallel pair equal dmpt_run's exactly."""
    from paper_2203_09621_b200 import DmptPair
    from workloads import make_config

    wl = make_config(3, device="cuda")
    a, a0, a1 = _run(wl, dev)
    p = DmptPair(wl.n, device0=dev, device1=dev)
    p.set_hamiltonian(torch.from_numpy(wl.h0).to(dev), torch.from_numpy(wl.h1).to(dev), wl.n_occ)
    b = p.run()
    assert a.status == 0 and b.status == 0
    assert (a.layers, a.layers_d0, a.layers_d1, a.sigma) == (b.layers, b.layers_d0, b.layers_d1, b.sigma)
    assert np.array_equal(a0, b.d0.double().cpu().numpy()) and np.array_equal(a1, b.d1.double().cpu().numpy())
    p.close()


def test_third_order_multi_wave_matches_the_oracle(dev):
    """SURVEY.md 8(f) f2 at n = 2048 (config 2's size: 72 pair tiles, three launches per layer): D0 .. D3 against
    oracle.dnn_sp2_pt run to order 3 (fp64, ~1 min on the host)."""
    from oracle.dnn_sp2_pt import dnn_sp2_pt
    from paper_2203_09621_b200 import Dmpt
    from workloads import make_config

    wl = make_config(2)
    ref = dnn_sp2_pt(wl.h0, wl.h1, wl.n_occ, order=3)
    assert ref.status == "ok"
    s = Dmpt(wl.n, device=dev, order=3)
    s.set_hamiltonian(torch.from_numpy(wl.h0).to(dev), torch.from_numpy(wl.h1).to(dev), wl.n_occ)
    r = s.run_orders()
    d = [m.double().cpu().numpy() for m in (r.d0, r.d1, r.d2, r.d3)]
    s.close()
    assert r.status == 0
    assert np.abs(d[0] - ref.dk[0]).max() <= 5e-5 and abs(np.trace(d[0]) - wl.n_occ) <= 1e-3
    errs = [np.abs(d[k] - ref.dk[k]).max() / np.abs(ref.dk[k]).max() for k in (1, 2, 3)]
    assert all(e <= 5e-4 for e in errs), errs
    got = [r.layers_d0, r.layers_d1, r.layers_d2, r.layers_d3]
    assert all(w - 8 <= g <= w + 2 for g, w in zip(got, ref.layers_dk)), (got, ref.layers_dk)
    print(f"order 3 @ n=2048: layers gpu {got} O2 fp64 {ref.layers_dk} errors D1..D3 {errs}")
