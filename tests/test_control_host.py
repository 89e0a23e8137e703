"""The device-side control flow (csrc/control.cuh: sigma choice, Algorithm 2, Algorithm 3, the order-2
cascade and the per-field stops) compiled for the host and driven with scripted reductions.

The scripts come from the oracle's own per-layer records (so the decisions must reproduce the oracle's
sigma sequence and stop layers exactly) and from hand-made norm sequences that make the response slots
stop on different layers - a case the GPU workloads do not produce (their tests all fire at n_c + 2)."""
import math
import os
import subprocess
import tempfile

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
RED = dict(TR_S0=0, FRO_S0=1, FRO0=2, FRO1=3, MAX1=4, FRO2=5, MAX2=6, FRO3=7, MAX3=8, COUNT=10)


@pytest.fixture(scope="module")
def driver():
    d = tempfile.mkdtemp()
    exe = os.path.join(d, "control_host")
    subprocess.run(["g++", "-std=c++17", "-O1", "-x", "c++", "-I", os.path.join(ROOT, "paper_2203_09621_b200", "csrc"),
                    os.path.join(ROOT, "tests", "support", "control_host_driver.cpp"), "-o", exe], check=True)
    return exe


def _drive(exe, order, nfields, n_occ, n_s, n_x, layers, max_layers=200):
    txt = f"{order} {nfields} {n_occ} {max_layers} 1\n{n_s!r} {n_x!r}\n"
    for red in layers:
        txt += " ".join(repr(float(x)) for x in red) + "\n"
    out = subprocess.run([exe], input=txt, capture_output=True, text=True, check=True).stdout.strip().split("\n")
    dec = [tuple(int(x) for x in ln.split()) for ln in out if not ln.startswith("end")]
    end = [ln for ln in out if ln.startswith("end")]
    return dec, (end[0].split()[1:] if end else None)


def _script_from_oracle(ref, order):
    """Reductions the epilogues would report, from the oracle's per-layer records (exact arithmetic:
    N_X of layer n+1 = ||S0_n||_F^2 = Tr X0_{n+1}, reading R9)."""
    layers = []
    for n in range(1, ref.layers + 1):
        red = [0.0] * RED["COUNT"]
        if n < ref.layers_d0:                            # S0 updated on layer n
            red[RED["TR_S0"]] = ref.tr_s[n]              # N_S entering layer n + 1
            red[RED["FRO_S0"]] = ref.tr_x[n]             # N_X of layer n + 1
        if n == ref.layers_d0:
            red[RED["FRO0"]] = ref.fro_err0 ** 2
        if n >= ref.layers_d0 and not math.isnan(ref.fro_err1[n - 1]):
            red[RED["FRO1"]] = ref.fro_err1[n - 1] ** 2
        red[RED["MAX1"]] = 1.0
        if order == 2:
            f2 = ref.fro_err2[n - 1]
            red[RED["FRO2"]] = 0.0 if math.isnan(f2) else f2 ** 2
            red[RED["MAX2"]] = 1.0
        layers.append(red)
    return layers


@pytest.mark.parametrize("cfg,n,order", [(1, 96, 1), (2, 128, 1), (4, 160, 1), (1, 96, 2), (2, 128, 2)])
def test_control_reproduces_the_oracles_decisions(driver, cfg, n, order):
    from oracle.dnn_sp2_pt import dnn_sp2_pt
    from workloads import make_config

    wl = make_config(cfg, n=n)
    ref = dnn_sp2_pt(wl.h0, wl.h1, wl.n_occ, order=order)
    assert ref.status == "ok"
    dec, end = _drive(driver, order, 1, wl.n_occ, ref.tr_s[0], ref.tr_x[0], _script_from_oracle(ref, order))
    assert end is not None, "the device control did not stop where the oracle did"
    layers, n_c, n_c1 = int(end[0]), int(end[1]), int(end[2])
    assert (layers, n_c, n_c1) == (ref.layers, ref.layers_d0, ref.layers_d1)
    assert [d[1] for d in dec[:ref.layers]] == ref.sigma            # sigma_n of every layer
    assert abs(float(end[5]) - ref.fro_err0) <= 1e-12 * ref.fro_err0
    assert dec[-1][7] == 1 and dec[-1][8] == 0                      # done, status ok


def test_ground_state_mode_stops_on_the_decision(driver):
    from oracle.dnn_sp2_pt import dnn_sp2, dnn_sp2_pt
    from workloads import make_config

    wl = make_config(1, n=96)
    ref = dnn_sp2_pt(wl.h0, wl.h1, wl.n_occ)
    _, layers0 = dnn_sp2(wl.h0, wl.n_occ)
    dec, end = _drive(driver, 0, 1, wl.n_occ, ref.tr_s[0], ref.tr_x[0], _script_from_oracle(ref, 1))
    assert int(end[0]) == layers0 == ref.layers_d0 and len(dec) == layers0       # no launch for the stop layer


def _expected_stop(fro, n_c, fro0, c_pt=9.0):
    """Algorithm 3 on a FroErr sequence indexed by layer, first test at n_c + 2."""
    n = n_c + 2
    while fro[n] < c_pt * fro0 * fro[n - 2]:
        n += 1
    return n


def test_fields_stop_on_their_own_layers(driver):
    """Three first-order fields whose FroErr1 sequences stop the test on different layers; the run ends with
    the last one, and a stopped field's iterate is no longer accepted (its buffer stops flipping)."""
    from oracle.dnn_sp2_pt import dnn_sp2_pt
    from workloads import make_config

    wl = make_config(1, n=96)
    ref = dnn_sp2_pt(wl.h0, wl.h1, wl.n_occ)
    n_c, fro0 = ref.layers_d0, ref.fro_err0
    base = _script_from_oracle(ref, 1)
    # FroErr sequences from layer n_c on: r^k with r^2 = 4.5 fro0 (inside the inequality by a factor 2) down
    # to a floor r^m, where the test then fires on layer n_c + m + 1
    r = math.sqrt(0.5 * 9.0 * fro0)

    def seq(m):
        return {n_c + k: max(r ** k, r ** m) for k in range(0, 40)}
    f1, f2, f3 = seq(3), seq(5), seq(7)
    stops = [_expected_stop(f, n_c, fro0) for f in (f1, f2, f3)]
    assert len(set(stops)) == 3 and stops[0] < stops[1] < stops[2]
    layers = []
    for n in range(1, stops[2] + 1):
        red = list(base[n - 1]) if n <= len(base) else [0.0] * RED["COUNT"]
        if n >= n_c:
            red[RED["FRO1"]], red[RED["FRO2"]], red[RED["FRO3"]] = f1[n] ** 2, f2[n] ** 2, f3[n] ** 2
        red[RED["MAX1"]] = red[RED["MAX2"]] = red[RED["MAX3"]] = 1.0
        layers.append(red)
    dec, end = _drive(driver, 1, 3, wl.n_occ, ref.tr_s[0], ref.tr_x[0], layers)
    assert end is not None
    assert [int(end[0]), int(end[2]), int(end[3]), int(end[4])] == [stops[2]] + stops
    # conv flags switch on exactly after each field's stop layer, in order
    for d in dec:
        layer = d[0]
        assert d[4] == int(layer > stops[0]) and d[5] == int(layer > stops[1])


def test_max_layers_and_non_finite_state(driver):
    from oracle.dnn_sp2_pt import dnn_sp2_pt
    from workloads import make_config

    wl = make_config(1, n=96)
    ref = dnn_sp2_pt(wl.h0, wl.h1, wl.n_occ)
    script = _script_from_oracle(ref, 1)
    dec, end = _drive(driver, 1, 1, wl.n_occ, ref.tr_s[0], ref.tr_x[0], script, max_layers=7)
    assert dec[-1][7] == 1 and dec[-1][8] == -5 and int(end[0]) == 7           # DMPT_ENOCONV after 7 layers
    script[3][RED["FRO_S0"]] = float("nan")
    dec, end = _drive(driver, 1, 1, wl.n_occ, ref.tr_s[0], ref.tr_x[0], script)
    assert dec[-1][7] == 1 and dec[-1][8] == -6                                # DMPT_ENUMERIC


@pytest.mark.parametrize("cfg,n", [(1, 96), (2, 128), (4, 160)])
def test_order_parallel_pair_takes_the_same_decisions(driver, cfg, n):
    """the control flow split over the two sides of an order-parallel pair (order-0 side: sigma_n
    and Algorithm 2, published per layer as DmptHandoff records; order-1 side: Algorithm 3, sigma flips after the
    freeze) reproduces the single-context decisions and the oracle's sigma sequence and stop layers."""
    from oracle.dnn_sp2_pt import dnn_sp2_pt
    from workloads import make_config

    wl = make_config(cfg, n=n)
    ref = dnn_sp2_pt(wl.h0, wl.h1, wl.n_occ)
    script = _script_from_oracle(ref, 1)
    one, end1 = _drive(driver, 1, 1, wl.n_occ, ref.tr_s[0], ref.tr_x[0], script)
    two, end2 = _drive(driver, 11, 1, wl.n_occ, ref.tr_s[0], ref.tr_x[0], script)
    assert end2 is not None and end1[:3] == end2[:3] and float(end1[5]) == float(end2[5])
    assert (int(end2[0]), int(end2[1]), int(end2[2])) == (ref.layers, ref.layers_d0, ref.layers_d1)
    assert [d[1] for d in two[:ref.layers]] == ref.sigma
    assert [(d[0], d[1], d[3]) for d in two[:ref.layers]] == [(d[0], d[1], d[3]) for d in one[:ref.layers]]
    assert all(d[2] == 2 for d in two[:ref.layers])             # the order-1 side never forms S0^2 (MODE_FROZEN)
    assert two[-1][7] == 1 and two[-1][8] == 0
    # max_layers on the pair: DMPT_ENOCONV after 7 layers, like a single context
    two, end2 = _drive(driver, 11, 1, wl.n_occ, ref.tr_s[0], ref.tr_x[0], script, max_layers=7)
    assert two[-1][7] == 1 and two[-1][8] == -5 and int(end2[0]) == 7


def test_third_order_cascade(driver):
    """Order 3: the stop of every order opens the gate of the next, two layers apart at least
    (reading R15); the oracle's order-3 records drive the device control to the same stop layers."""
    from oracle.dnn_sp2_pt import dnn_sp2_pt
    from workloads import make_config

    wl = make_config(1, n=96)
    ref = dnn_sp2_pt(wl.h0, wl.h1, wl.n_occ, order=3)
    assert ref.status == "ok"
    layers = _script_from_oracle(ref, 2)
    for n in range(1, ref.layers + 1):
        f3 = ref.fro_errk[3][n - 1]
        layers[n - 1][RED["FRO3"]] = 0.0 if math.isnan(f3) else f3 ** 2
        layers[n - 1][RED["MAX3"]] = 1.0
    dec, end = _drive(driver, 3, 1, wl.n_occ, ref.tr_s[0], ref.tr_x[0], layers)
    assert end is not None
    assert [int(end[1]), int(end[2]), int(end[3]), int(end[4])] == ref.layers_dk and int(end[0]) == ref.layers
    assert [d[1] for d in dec[:ref.layers]] == ref.sigma
