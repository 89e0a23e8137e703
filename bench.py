#!/usr/bin/env python
"""bench.py - throughput of the DNN-SP2-PT hot path (arXiv 2203.09621) on B200.

A "step" is one pass of the whole hot path: dmpt_run = Gershgorin bounds -> initial transform ->
split -> every deep layer until both parameter-free stopping tests fire -> D0, D1.  The workload
is BASELINE.json configs[3] (N = 16384, the size the metric is quoted on; synthetic, seeded, see
DESIGN.md "Input recipe").  Matrices are 1 GiB each: every timed pass streams inputs far larger
than the 126 MB L2, so no explicit L2 flush is needed (stated in `config`).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 4] [--n 16384]
    python bench.py --impl reference      # the fp64 CPU oracle, bounded sample, same JSON line
    python bench.py --fd [--config 2]     # finite-difference stencils vs the first-order recursion (Fig. 5)
    python bench.py --order-parallel      # the two-device variant of PAPER.md:287 (one device: both sides on it)

value      paper-convention Tflops (one FMA = one flop, Eq. 82):
           (5 N^3 L_active + 3 N^3 L_frozen) / time of the whole dmpt_run, inputs resident in HBM.
e2e        the same through dmpt_run_host: H0, H1 in pinned host memory, D0, D1 read back.
roofline   the layer kernel (tcgen05 GEMM + fused epilogue): EXECUTED tensor flops (2 per FMA, as
           the measured peak counts them) per launch / its average launch duration (CUDA events on
           the launching stream around the layer loop), against MEASURED_PEAKS.json.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "dmpt_layer_tflops_fma1"
UNIT = "Tflops (FMA=1)"
NOMINAL_FP16_TFMA = 1125.0     # 2250 Tflops dense fp16 at 2 flops/FMA (B200_PROFILING.md)
FALLBACK_PEAKS = {"hbm_gbs": 6650.0, "bf16_tflops": 1590.0, "bf16_tflops_sustained": 1400.0}


def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            return json.load(f), "measured"
    return dict(FALLBACK_PEAKS), "fallback"


def library_gemm_sustained(dev, dtype, seconds=3.0, m=8192):
    """Context for the roofline line, not its denominator: the library GEMM (torch.matmul = cuBLAS) of the layer
    kernel's OPERAND dtype, m^3, back to back for `seconds` under the same power cap, TFLOP/s at 2 flops per FMA.
    MEASURED_PEAKS.json holds the bf16 figure; fp16 operands cost more energy per product than bf16's."""
    import torch

    a = torch.randn((m, m), device=dev, dtype=torch.float32).to(dtype)
    b = torch.randn((m, m), device=dev, dtype=torch.float32).to(dtype)
    c = torch.empty((m, m), device=dev, dtype=dtype)
    for _ in range(20):
        torch.matmul(a, b, out=c)
    torch.cuda.synchronize(dev)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    reps, batch = 0, 50
    t0 = time.perf_counter()
    e0.record()
    while time.perf_counter() - t0 < seconds:
        for _ in range(batch):
            torch.matmul(a, b, out=c)
        torch.cuda.synchronize(dev)
        reps += batch
    e1.record()
    torch.cuda.synchronize(dev)
    return 2.0 * m ** 3 * reps / (e0.elapsed_time(e1) * 1e-3) / 1e12


class ClockSampler:
    """nvidia-smi clocks/throttle reasons sampled every 200 ms while the timed region runs."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index=0):
        self.index = index
        self.proc = None
        self.lines = []

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                 "-lms", "200"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._pump, daemon=True)
            self.t.start()
        except OSError:
            self.proc = None

    def _pump(self):
        for line in self.proc.stdout:
            self.lines.append(line.strip())

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        sm, mx, pw, reasons = [], None, [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for ln in self.lines:
            f = [x.strip() for x in ln.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0]))
                mx = float(f[1])
                pw.append(float(f[2]))
            except ValueError:
                continue
            for name, val in zip(names, f[3:7]):
                if val.lower().startswith("active"):
                    reasons.add(name)
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": mx,
                "power_w_max": max(pw) if pw else None, "samples": len(sm), "reasons": sorted(reasons)}


def _layer_split(layers, layers_d0, layers_d1, order):
    """(layers with S0 active, layers with S0 frozen and S1 active, layers with only S2 active)."""
    la = layers_d0 if layers_d0 > 0 else layers
    l1 = (layers_d1 if (order == 2 and layers_d1 > 0) else layers) - la
    return la, l1, layers - la - l1


def flops_paper(n, layers, layers_d0, order=1, layers_d1=0):
    """Eq. 82 with the layers after S0 froze counted as 3 N^3 (SURVEY.md 8(d) accounting rules); order 2 adds
    3 N^3 (S0.S2) + 2 N^3 (S1.S1) per layer, and after the D1 stop only those remain."""
    la, l1, l2 = _layer_split(layers, layers_d0, layers_d1, order)
    per = (5.0 * la + 3.0 * l1) + (5.0 * layers if order == 2 else 0.0)
    return per * float(n) ** 3


def fma_executed(n_pad, layers, layers_d0, order=1, layers_d1=0):
    """Tensor FMAs the layer kernel needs: the 128x128 output blocks on or above the diagonal, 9 (6 once
    S0 froze) 128x128xK products each.  The CTA-pair kernel also issues the nb/2
    sub-diagonal blocks of its 256x128 diagonal pair tiles (+0.8 % at N = 16384); they are not counted."""
    nb = n_pad // 128
    tiles = nb * (nb + 1) // 2
    la, l1, l2 = _layer_split(layers, layers_d0, layers_d1, order)
    per_mma = 128.0 * 128.0 * n_pad
    return tiles * per_mma * (9.0 * la + 6.0 * l1 + (9.0 * layers if order == 2 else 0.0))


# ---------------------------------------------------------------------------------------------
# CPU oracle legs (cpu_baseline and --impl reference): the only places that touch oracle/
# ---------------------------------------------------------------------------------------------
ORACLE_FP64_TFLOPS_GUESS = 0.4      # dgemm rate of the host BLAS on 16 threads (round 1: 0.5 Tflops FMA=1 ... /1.25), sizing only


def oracle_sample(config, n_sample, layers, wl=None):
    """Time oracle.dnn_sp2_pt (fp64, numpy/host BLAS, as it stands) for `layers` layers of the
    bench workload's generator at size n_sample (the bench workload itself when `wl` is given).
    Returns (Tflops FMA=1, seconds, threads, layers run)."""
    from oracle.dnn_sp2_pt import dnn_sp2_pt
    from workloads import make_config

    if wl is None or wl.n != n_sample:
        import torch
        wl = make_config(config, n=n_sample, device="cuda" if (n_sample >= 8192 and torch.cuda.is_available()) else None)
    t0 = time.perf_counter()
    res = dnn_sp2_pt(wl.h0, wl.h1, wl.n_occ, order=wl.order, max_layers=layers)
    dt = time.perf_counter() - t0
    fl = flops_paper(n_sample, res.layers, res.layers_d0, wl.order, res.layers_d1)
    return fl / dt / 1e12, dt, len(os.sched_getaffinity(0)), res.layers


def oracle_o3_d0(wl):
    """Layer at which Algorithm 2 fires in fp64, from O3 (oracle/spectral.py) on the spectrum the generator
    constructed and the oracle's own Gershgorin bounds of the rounded H0: O(N) per layer."""
    from oracle.dnn_sp2_pt import gershgorin
    from oracle.spectral import spectral_recursion

    if "eps" not in wl.meta:
        return None
    lo, hi = gershgorin(wl.h0)
    return int(spectral_recursion(wl.meta["eps"], wl.n_occ, lo, hi)["layers_d0"])


def reference_sample_size(n, order, steps, budget_s=300.0):
    """Bounded sample of the reference arm: the bench workload's own N with 3 layers per step when K steps of it
    fit `budget_s`, else the generator at N/2, N/4, ... with as many layers (<= 20) as fit.  Cost model: 2 (order
    2: 4) dgemm of 2 n^3 flop per layer at ORACLE_FP64_TFLOPS_GUESS, + 30 % for the elementwise passes."""
    per_step = budget_s / max(1, steps)
    dgemms = 4 if order == 2 else 2
    n_s = n
    while True:
        per_layer = 1.3 * dgemms * 2.0 * float(n_s) ** 3 / (ORACLE_FP64_TFLOPS_GUESS * 1e12)
        if 3 * per_layer <= per_step or n_s <= 512:
            return n_s, (3 if (n_s == n and n > 4096) else int(max(3, min(20, per_step // per_layer))))
        n_s //= 2


def run_reference(args):
    from paper_2203_09621_b200 import replicas
    from workloads import CONFIGS

    if replicas.env_ranks()[0] != 0:          # under torchrun rank 0 alone runs and prints the oracle's line
        return 0
    order = CONFIGS[args.config]["order"]
    n_s, layers = reference_sample_size(args.n, order, args.steps)
    if args.ref_n is not None:
        n_s = args.ref_n
    if args.ref_layers is not None:
        layers = args.ref_layers
    for _ in range(args.warmup and 1):          # one untimed pass pages numpy/BLAS in
        oracle_sample(args.config, min(n_s, 512), 1)
    from workloads import make_config
    import torch
    wl = make_config(args.config, n=n_s, device="cuda" if (n_s >= 8192 and torch.cuda.is_available()) else None)
    vals, secs = [], []
    cores = len(os.sched_getaffinity(0))
    for _ in range(args.steps):
        v, dt, cores, _ = oracle_sample(args.config, n_s, layers, wl)
        vals.append(v)
        secs.append(dt)
    value = sum(vals) / len(vals)
    sample = (f"oracle.dnn_sp2_pt (fp64) on the config-{args.config} generator at n={n_s}, first {layers} layers, per step"
              + ("" if n_s == args.n else f" (the workload's N={args.n} does not fit {args.steps} steps in a few minutes)"))
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": replicas.env_ranks()[2],
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * sum(secs) / len(secs),
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic", "gpu_launches": 0,
        "config": {"workload": workload_name(args), "sample": sample},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }
    print(json.dumps(line), flush=True)
    return 0


def workload_name(args):
    from workloads import CONFIGS
    order = {1: "first", 2: "second"}[CONFIGS[args.config]["order"]]
    return (f"BASELINE.json configs[{args.config - 1}] (config {args.config}): N={args.n}, {order}-order response, "
            "seeded synthetic gapped Hamiltonian")


# ---------------------------------------------------------------------------------------------
# the CUDA arm
# ---------------------------------------------------------------------------------------------
def run_ours(args):
    import numpy as np
    import torch
    import torch.distributed as dist

    from paper_2203_09621_b200 import Dmpt
    from workloads import make_config

    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: the product has no CPU path")
    from paper_2203_09621_b200 import replicas

    rank, local, world = replicas.env_ranks()
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)

    # Replicas only: every rank solves its own seeded problem of the same
    # configuration; there is no data-path collective.
    wl = make_config(args.config, n=args.n, device=str(dev), seed=replicas.replica_seed(args.config, rank))
    n = wl.n
    h0_host = torch.from_numpy(wl.h0).pin_memory()
    h1_host = torch.from_numpy(wl.h1).pin_memory()
    h0 = h0_host.to(dev)
    h1 = h1_host.to(dev)
    order = wl.order
    nf = args.fields
    if nf > 1:
        # several perturbations sharing H0 (DESIGN.md f2): the config's H1 plus seeded symmetric Gaussians
        if order != 1:
            raise SystemExit("--fields needs a first-order config")
        from workloads.hamiltonians import symmetric_gaussian
        h1s = [h1] + [torch.from_numpy(symmetric_gaussian(np.random.default_rng(wl.meta["seed"] + 100 * f), n, 0.01)
                                       .astype(np.float32)).to(dev) for f in range(1, nf)]
        solver = Dmpt(n, order=1, device=dev, num_fields=nf)
        solver.set_hamiltonian_fields(h0, h1s, wl.n_occ)
    else:
        solver = Dmpt(n, order=order, device=dev, bounds="lanczos" if args.bounds == "lanczos" else None)
        solver.set_hamiltonian(h0, h1, wl.n_occ)
    d0 = torch.empty((n, n), dtype=torch.float32, device=dev)
    d1 = torch.empty((n, n), dtype=torch.float32, device=dev)
    d0_host = torch.empty((n, n), dtype=torch.float32).pin_memory()
    d1_host = torch.empty((n, n), dtype=torch.float32).pin_memory()
    n_out = 2 + (order == 2)
    outs = (d0, d1) + ((torch.empty((n, n), dtype=torch.float32, device=dev),) if order == 2 else ())
    outs_host = (d0_host, d1_host) + ((torch.empty((n, n), dtype=torch.float32).pin_memory(),) if order == 2 else ())

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize(dev)

    def max_over_ranks(x):
        return replicas.max_over_ranks(x, dev)

    def sum_over_ranks(x):
        return replicas.sum_over_ranks(x, dev)

    def one_run():
        """(result, paper-convention FMA, tensor FMA needed) of one step."""
        if nf == 1:
            r = solver.run(out=outs)
            return (r, flops_paper(n, r.layers, r.layers_d0, order, r.layers_d1),
                    fma_executed(solver_n_pad(n), r.layers, r.layers_d0, order, r.layers_d1))
        r = solver.run_fields()
        stops = [r.layers_d1, r.layers_d2, r.layers_d3][:nf]
        # paper convention: every field as a run of its own (S0^2 counted per field)
        fl = sum(flops_paper(n, st, r.layers_d0) for st in stops)
        fx = sum(fma_executed(solver_n_pad(n), st, r.layers_d0) for st in stops)
        la = r.layers_d0 if r.layers_d0 > 0 else r.layers
        nb = solver_n_pad(n) // 128
        fx -= (nf - 1) * (nb * (nb + 1) // 2) * 128.0 * 128.0 * solver_n_pad(n) * 3.0 * la     # S0^2 is formed once
        return r, fl, fx

    for _ in range(args.warmup):
        res = one_run()[0]
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    # ---- device-resident arm: K steps between two barriers, CUDA events on the launching stream
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    ev0.record()
    flops = fma = ms_loop = 0.0
    launches = layers_total = 0
    dev_mhz = []
    for _ in range(args.steps):
        res, fl, fx = one_run()
        flops += fl
        fma += fx
        ms_loop += res.ms_loop
        dev_mhz.append(getattr(res, "sm_clock_mhz", 0.0))
        launches += res.launches
        layers_total += res.layers
    ev1.record()
    barrier()
    ms = max_over_ranks(ev0.elapsed_time(ev1))
    clocks = sampler.stop() if rank == 0 else None
    total_flops = sum_over_ranks(flops)
    value = total_flops / (ms * 1e-3) / 1e12

    # ---- end-to-end arm: host buffers through dmpt_run_host / dmpt_run_fields_host, copies inside the timed region
    if nf > 1:
        h1s_host = [h1_host] + [m.cpu().pin_memory() for m in h1s[1:]]
        d1s_host = [d1_host] + [torch.empty((n, n), dtype=torch.float32).pin_memory() for _ in range(nf - 1)]

    def one_run_host():
        if nf == 1:
            r2 = solver.run_host(h0_host, h1_host, wl.n_occ, out=outs_host)
            return flops_paper(n, r2.layers, r2.layers_d0, order, r2.layers_d1)
        r2 = solver.run_fields_host(h0_host, h1s_host, wl.n_occ, out=(d0_host, d1s_host))
        return sum(flops_paper(n, st, r2.layers_d0) for st in [r2.layers_d1, r2.layers_d2, r2.layers_d3][:nf])

    one_run_host()
    barrier()
    ev0.record()
    e2e_flops = 0.0
    for _ in range(args.steps):
        e2e_flops += one_run_host()
    ev1.record()
    barrier()
    ms_e2e = max_over_ranks(ev0.elapsed_time(ev1))
    e2e_value = sum_over_ranks(e2e_flops) / (ms_e2e * 1e-3) / 1e12

    # ---- time-to-D1 with the optional tighter bounds (bounds = 2, R18), reported next to the headline
    lanczos = None
    if rank == 0 and nf == 1 and order == 1 and args.bounds == "gershgorin":
        solver.close()
        solver = Dmpt(n, order=order, device=dev, bounds="lanczos")
        solver.set_hamiltonian(h0, h1, wl.n_occ)
        solver.run(out=outs)
        rl = [solver.run(out=outs) for _ in range(2)][-1]
        lanczos = {"time_to_d1_ms": rl.ms_total, "layers": rl.layers, "layers_d0": rl.layers_d0, "ms_bounds": rl.ms_bounds,
                   "eps_min": rl.eps_min, "eps_max": rl.eps_max,
                   "note": "dmpt_options.bounds = 2: Gershgorin discs tightened by 20 Lanczos steps on the device; same "
                           "D0, D1 in fewer layers; not the headline (the paper's example bounds are Gershgorin's)"}

    if rank == 0:
        traffic, traffic_src = ncu_traffic(n, order, nf, args.traffic)
        peaks, peaks_kind = load_peaks()
        peak_tf = float(peaks.get("bf16_tflops_sustained", peaks["bf16_tflops"]))
        layer_ms = ms_loop / max(1, layers_total)
        achieved_tf = 2.0 * fma / (ms_loop * 1e-3) / 1e12
        # the SM clock of the layer loop from the device's own counters (dmpt_result.sm_clock_mhz): under the power cap
        # it lies below what nvidia-smi samples show; the tensor peak AT that clock is what the kernel can be held to
        dev_mhz = [m for m in dev_mhz if m > 0.0]
        sm_mhz_device = sum(dev_mhz) / len(dev_mhz) if dev_mhz else None
        if clocks is not None:
            clocks["sm_mhz_device"] = sm_mhz_device
            clocks["sm_mhz_device_note"] = ("SM cycle counters over the device nanosecond timer across the layer loop, "
                                            "all SMs (dmpt_result.sm_clock_mhz); sm_mhz is nvidia-smi's sample")
        lib_tf = None
        if n >= 8192 and nf == 1 and order == 1:            # the sizes the power cap governs
            lib_tf = library_gemm_sustained(dev, torch.float16)
        n_sm = torch.cuda.get_device_properties(dev).multi_processor_count
        peak_at_clock = n_sm * 4096 * sm_mhz_device * 1e6 / 1e12 if sm_mhz_device else None      # T-FMA/s, fp16 dense
        # the oracle as it stands on THIS workload: 3 layers at the bench N when that is about
        # 1-3 min of host time, the whole run when it is shorter; per-layer seconds and the time-to-D1 extrapolated
        # with O3's layer count.  A second, smaller sample (n = 4096 generator, 20 layers) keeps round 1's key.
        ref_n = args.ref_n if args.ref_n is not None else n
        ref_layers = args.ref_layers if args.ref_layers is not None else (3 if n > 4096 else 200)
        cpu_v, cpu_dt, cores, cpu_layers = oracle_sample(args.config, ref_n, ref_layers, wl)
        o3_d0 = oracle_o3_d0(wl) if ref_n == n else None
        cpu_extra = {}
        if ref_n == n and n > 4096 and args.ref_n is None:
            v2, dt2, _, l2 = oracle_sample(args.config, 4096, 20)
            cpu_extra = {"secondary": {"value": v2, "seconds": dt2, "sample": f"config-{args.config} generator at n=4096, first {l2} layers"}}
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms / args.steps, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f16 x f16 -> f32 (dual-half), f64 scalars",
            "data": "synthetic", "gpu_launches": launches,
            "config": {"workload": workload_name(args), "n": n, "n_occ": wl.n_occ, "order": order, "fields": nf,
                       "layers": res.layers, "layers_d0": res.layers_d0, "layers_d0_oracle_o3": o3_d0,
                       "layers_note": "O3 = the fp64 recursion on the constructed spectrum; it runs 1-5 layers past "
                                      "any dual-half run (stop at the noise floor, R14)",
                       "gap": wl.meta.get("gap"),
                       "parallelism": "replicas only" if world > 1 else "1 GPU",
                       "l2": f"inputs larger than L2 ({n * n * 4 / 2**30:.2f} GiB per matrix); no flush needed",
                       "time_to_d1_ms": ms / args.steps, "loop_ms": ms_loop / args.steps,
                       "bounds": args.bounds, "eps_min": res.eps_min, "eps_max": res.eps_max,
                       "with_lanczos_bounds": lanczos,
                       "tflops_fma1_loop_only": flops / (ms_loop * 1e-3) / 1e12,
                       "frac_nominal_fp16_peak_fma1": value / NOMINAL_FP16_TFMA,
                       "paper_context": "~120 Tflops (FMA=1) on one A100, N=19008 (PAPER.md:546); another machine"},
            "clocks": clocks,
            "e2e": {"value": e2e_value, "unit": UNIT, "ms_per_step": ms_e2e / args.steps,
                    "h2d_bytes_per_step": (1 + nf) * n * n * 4,
                    "d2h_bytes_per_step": (n_out if nf == 1 else 1 + nf) * n * n * 4},
            "roofline": {"bound": "tensor", "kernel": "dmpt_layer_kernel", "achieved": achieved_tf, "peak": peak_tf,
                         "unit": "TFLOP/s", "frac": achieved_tf / peak_tf, "traffic": traffic,
                         "traffic_source": traffic_src,
                         "peak_kind": f"bf16_tflops_sustained, {peaks_kind} (fp16 = bf16 rate), 2 flops per FMA",
                         "avg_launch_ms": layer_ms, "executed_tfma_per_s": achieved_tf / 2.0,
                         "frac_nominal_1125_tfma": achieved_tf / 2.0 / NOMINAL_FP16_TFMA,
                         "library_fp16_gemm_sustained": ({"tflops": lib_tf, "frac": achieved_tf / lib_tf,
                                                          "what": "torch.matmul fp16 8192^3 (cuBLAS) back to back for "
                                                                  "3 s on this GPU, after the timed region: the "
                                                                  "library GEMM of the kernel's operand dtype under "
                                                                  "the same cap; context, not the denominator"}
                                                         if lib_tf else None),
                         "tfma_peak_at_device_clock": peak_at_clock,
                         "frac_of_peak_at_device_clock": (achieved_tf / 2.0 / peak_at_clock) if peak_at_clock else None,
                         "device_clock_note": "4096 dense fp16 FMA per SM and clock x SMs x clocks.sm_mhz_device: "
                                              "what is left of the nominal peak at the clock the 1 kW cap allows"},
            "cpu_baseline": dict({"value": cpu_v, "unit": UNIT, "cores": cores, "kind": "oracle", "seconds": cpu_dt,
                                  "sample": f"oracle.dnn_sp2_pt (fp64) on the bench workload itself (config {args.config}, "
                                            f"n={ref_n}), first {cpu_layers} layers incl. bounds and transform",
                                  "seconds_per_layer": cpu_dt / max(1, cpu_layers),
                                  "time_to_d1_s_extrapolated": (cpu_dt / max(1, cpu_layers) * (o3_d0 + 3)
                                                                if o3_d0 and cpu_layers < o3_d0 else None),
                                  "extrapolation": "seconds_per_layer x (O3 fp64 D0 stop layer + 3 further layers, "
                                                   "PAPER.md:483); extrapolated, not run"}, **cpu_extra),
        }
        print(json.dumps(line), flush=True)
    solver.close()
    if world > 1:
        dist.destroy_process_group()
    return 0


# ---------------------------------------------------------------------------------------------
# --order-parallel: the two-device variant of PAPER.md:287, 548-550
# ---------------------------------------------------------------------------------------------
def run_pair(args):
    """The order-parallel pair (dmpt_pair_*) on the bench workload: the order-0 side on cuda:0, the order-1 side on
    cuda:1 when the box has a second GPU, else on cuda:0 too (two streams, device-local hand-off: the two sides' launches
    then take turns on the SMs and the line only shows that the path runs at full size).  Same metric as the default
    line; the single-context run of the same input is timed beside it and the results are compared bit for bit."""
    import torch

    from paper_2203_09621_b200 import Dmpt, DmptPair
    from workloads import make_config

    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: the product has no CPU path")
    two = torch.cuda.device_count() > 1
    dev0, dev1 = torch.device("cuda", 0), torch.device("cuda", 1 if two else 0)
    wl = make_config(args.config, n=args.n, device="cuda:0" if args.n >= 8192 else None)
    if wl.order != 1:
        raise SystemExit("--order-parallel needs a first-order config")
    n = wl.n
    h0 = torch.from_numpy(wl.h0).to(dev0)
    h1 = torch.from_numpy(wl.h1).to(dev1)
    pair = DmptPair(n, device0=dev0, device1=dev1)
    pair.set_hamiltonian(h0, h1, wl.n_occ)
    for _ in range(max(1, args.warmup - 1)):
        rp = pair.run()
    sampler = ClockSampler(0)
    sampler.start()
    t0 = time.perf_counter()
    ms = flops = 0.0
    launches = 0
    for _ in range(args.steps):
        rp = pair.run()
        ms += rp.ms_total
        flops += flops_paper(n, rp.layers, rp.layers_d0)
        launches += rp.launches
    wall = time.perf_counter() - t0
    clocks = sampler.stop()
    d0p, d1p = rp.d0.clone(), rp.d1.to(dev0)
    pair.close()
    one = Dmpt(n, order=1, device=dev0)
    one.set_hamiltonian(h0, h1.to(dev0), wl.n_occ)
    one.run()
    r1 = one.run()
    same = bool(torch.equal(r1.d0, d0p) and torch.equal(r1.d1, d1p) and r1.layers == rp.layers)
    one.close()
    line = {"mode": "order-parallel", "metric": METRIC, "value": flops / (ms * 1e-3) / 1e12, "unit": UNIT,
            "n_gpus": 2 if two else 1, "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms / args.steps,
            "higher_is_better": True, "scaling": "strong", "vs_baseline": None,
            "dtype": "f16 x f16 -> f32 (dual-half), f64 scalars", "data": "synthetic", "gpu_launches": launches,
            "config": {"workload": workload_name(args), "n": n, "layers": rp.layers, "layers_d0": rp.layers_d0,
                       "parallelism": ("order-parallel pair: S0^2 on cuda:0, S0.S1 + S1.S0 on cuda:1, one hand-off of "
                                       "4 N^2 bytes per layer (cudaMemcpyPeerAsync)") if two else
                                      ("order-parallel pair with BOTH sides on cuda:0 (this box has one GPU): the two "
                                       "sides' launches take turns on the SMs; not a scaling number"),
                       "single_context_ms": r1.ms_total, "bit_identical_to_single_context": same,
                       "wall_s": wall,
                       "paper_context": "2 x A100: ~195 vs ~120 Tflops, +63 % (PAPER.md:550)"},
            "clocks": clocks, "e2e": None}
    print(json.dumps(line), flush=True)
    return 0 if same else 1


# ---------------------------------------------------------------------------------------------
# --fd: the finite-difference comparison of PAPER.md:562-582 (Eqs. 83-84, Fig. 5) as a workload
# ---------------------------------------------------------------------------------------------
def run_fd(args):
    """D1 by the 2- and 4-point stencils (dmpt_fd_response: 2 / 4 ground-state runs) over a sweep of step sizes h,
    next to the first-order DNN-SP2-PT run on the same input.  Errors are relative to the definition (oracle O1,
    evaluated and timed on the host: this mode's cpu_baseline) in the paper's measure - the relative 2-norm - and as
    max|.|/max|ref|.  Cost per layer in the paper's count: 4 / 8 products against 5."""
    import numpy as np
    import torch

    from paper_2203_09621_b200 import Dmpt
    from workloads import make_config

    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: the product has no CPU path")
    dev = torch.device("cuda", 0)
    wl = make_config(args.config, n=args.n, device=str(dev) if args.n >= 8192 else None)
    if wl.order != 1:
        raise SystemExit("--fd needs a first-order config")
    n = wl.n
    h0, h1 = torch.from_numpy(wl.h0).to(dev), torch.from_numpy(wl.h1).to(dev)
    # the definition (O1) on the host, timed: the reference of every error below
    from oracle.closed_form import density_matrices
    t0 = time.perf_counter()
    _, d1_ref = density_matrices(wl.h0, wl.h1, wl.n_occ)
    cpu_s = time.perf_counter() - t0
    ref = torch.from_numpy(d1_ref).to(dev)
    ref2 = float(torch.linalg.matrix_norm(ref, ord=2))
    refmax = float(ref.abs().max())

    def errors(d1):
        e = d1.double() - ref
        return {"rel_2norm": float(torch.linalg.matrix_norm(e, ord=2)) / ref2, "max_rel": float(e.abs().max()) / refmax}

    pt = Dmpt(n, order=1, device=dev)
    pt.set_hamiltonian(h0, h1, wl.n_occ)
    for _ in range(2):
        r = pt.run()
    dmpt = dict(errors(r.d1), layers=r.layers, layers_d0=r.layers_d0, ms=r.ms_total, products_per_layer=5,
                products=5 * r.layers_d0 + 3 * (r.layers - r.layers_d0))
    pt.close()
    h1_scale = float(h1.abs().max())
    gs = Dmpt(n, order=0, device=dev)
    sweep = []
    launches = 0
    for points in (2, 4):
        for hs in args.fd_steps:
            # h is quoted relative to the perturbation's size: h max|H1| is the largest change of a matrix element
            h = hs / h1_scale
            d1, layers, ms = gs.fd_response(h0, h1, wl.n_occ, h, points)
            d1, layers, ms = gs.fd_response(h0, h1, wl.n_occ, h, points)          # second call: warm
            sweep.append(dict(errors(d1), points=points, h=h, h_times_max_h1=hs, layers=layers, ms=ms,
                              products_per_layer=2 * points, products=2 * sum(layers)))
            launches += sum(layers)
    gs.close()
    best = {p: min((x for x in sweep if x["points"] == p), key=lambda x: x["rel_2norm"]) for p in (2, 4)}
    line = {"mode": "fd", "metric": "d1_relative_2norm_error", "unit": "relative 2-norm error", "higher_is_better": False,
            "value": dmpt["rel_2norm"], "n_gpus": 1, "data": "synthetic", "gpu_launches": launches,
            "config": {"workload": workload_name(args) + "; finite-difference stencils of ground-state runs against "
                                   "the first-order recursion (PAPER.md:562-582, Fig. 5)", "n": n, "n_occ": wl.n_occ,
                       "gap": wl.meta.get("gap")},
            "dmpt": dmpt, "fd_sweep": sweep,
            "best": {"two_point": best[2], "four_point": best[4],
                     "two_point_over_dmpt": best[2]["rel_2norm"] / dmpt["rel_2norm"],
                     "four_point_over_dmpt": best[4]["rel_2norm"] / dmpt["rel_2norm"],
                     "paper": "best 2-point: almost an order of magnitude less accurate than DNN-SP2-PT; best 4-point: "
                              "a factor 2 less accurate, at 8 instead of 5 products per layer (PAPER.md:578-582)"},
            "cpu_baseline": {"value": cpu_s, "unit": "s", "cores": len(os.sched_getaffinity(0)), "kind": "oracle",
                             "sample": f"oracle.closed_form.density_matrices (fp64 eigendecomposition) at n={n}: the "
                                       "reference of every error in this line"}}
    print(json.dumps(line), flush=True)
    return 0


def solver_n_pad(n):
    return (n + 255) // 256 * 256      # CTA-pair tiles: 256 rows


def kernel_source_sha():
    """sha256 (first 16 hex digits) of the layer kernel's sources: an ncu capture is only quoted for the code it saw."""
    import hashlib
    h = hashlib.sha256()
    for f in ("layer_kernel.cuh", "ptx.cuh"):
        with open(os.path.join(ROOT, "paper_2203_09621_b200", "csrc", f), "rb") as fh:
            h.update(fh.read())
    return h.hexdigest()[:16]


def ncu_traffic(n, order, nf, override):
    """dram__bytes_read.sum + dram__bytes_write.sum of ONE dmpt_layer_kernel launch from the `ncu --set full` capture
    recorded in profiles/layer_kernel_traffic.json (written from the capture named there); null when that capture
    saw other kernel sources than the ones being timed, or another workload."""
    if override is not None:
        return override, "--traffic"
    p = os.path.join(ROOT, "profiles", "layer_kernel_traffic.json")
    if not os.path.exists(p):
        return None, "no capture recorded"
    with open(p) as f:
        rec = json.load(f)
    if rec.get("n") != n or rec.get("order") != order or nf != 1:
        return None, "capture is of another workload"
    if rec.get("kernel_source_sha") != kernel_source_sha():
        return None, f"stale: {rec.get('capture')} saw kernel sources {rec.get('kernel_source_sha')}"
    return rec["dram_bytes_per_launch"], rec.get("capture")


def respawn_under_torchrun(args):
    """`python bench.py --gpus N` with N > 1 outside torchrun: launch the N ranks ourselves (one per GPU)."""
    import socket
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
           "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
    return subprocess.call(cmd)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=4)
    ap.add_argument("--n", type=int, default=None, help="override the matrix size (default: the config's)")
    ap.add_argument("--ref-n", type=int, default=None, help="size of the oracle's bounded sample (default: the workload's)")
    ap.add_argument("--ref-layers", type=int, default=None)
    ap.add_argument("--fields", type=int, default=1,
                    help="perturbations sharing H0 in one run (1..3); value then counts every field as a run of its own")
    ap.add_argument("--traffic", type=float, default=None, help="dram bytes per layer launch from ncu (profiles/)")
    ap.add_argument("--bounds", default="gershgorin", choices=["gershgorin", "lanczos"],
                    help="spectral bounds of the timed runs (default: Gershgorin discs, the paper's example)")
    ap.add_argument("--order-parallel", action="store_true",
                    help="the order-parallel pair (PAPER.md:287): order 0 on cuda:0, order 1 on cuda:1 if present")
    ap.add_argument("--fd", action="store_true",
                    help="finite-difference stencils (Eqs. 83-84) against the first-order recursion; default config 2")
    ap.add_argument("--fd-steps", type=float, nargs="+", default=[1e-3, 3e-3, 1e-2, 3e-2, 6e-2, 1e-1, 2e-1, 4e-1],
                    help="step sizes h of the sweep, as h x max|H1|")
    args = ap.parse_args()
    if args.fd and "--config" not in " ".join(sys.argv):
        args.config = 2
    if args.n is None:
        from workloads import CONFIGS
        args.n = CONFIGS[args.config]["n"]
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if args.gpus != world:
        if world == 1 and args.gpus > 1:
            return respawn_under_torchrun(args)
        raise SystemExit(f"bench.py: --gpus {args.gpus} but WORLD_SIZE={world}")
    if args.fd:
        return run_fd(args)
    if args.order_parallel:
        return run_pair(args)
    if args.warmup < 3 and args.impl == "ours":
        print("bench.py: warmup raised to 3 (timing rules)", file=sys.stderr)
        args.warmup = 3
    return run_reference(args) if args.impl == "reference" else run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
