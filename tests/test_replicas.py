"""Host-side logic of the N > 1 bench path (replicas only), on CPU with gloo."""
import json
import os
import subprocess
import sys

import pytest

torch = pytest.importorskip("torch")

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, out):
    import torch.distributed as dist

    sys.path.insert(0, ROOT)
    from paper_2203_09621_b200 import replicas

    os.environ.update(RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", init_method=f"tcp://127.0.0.1:{port}", rank=rank, world_size=world)
    try:
        assert replicas.env_ranks() == (rank, rank, world)
        units = 100.0 * (rank + 1)          # rank 0: 100 units, rank 1: 200 units
        ms = 1000.0 if rank == 0 else 2000.0
        dist.barrier()
        rate = replicas.whole_job_rate(units, ms)
        mx = replicas.max_over_ranks(ms)
        sm = replicas.sum_over_ranks(units)
        out.put((rank, rate, mx, sm, replicas.replica_seed(4, rank)))
    finally:
        dist.destroy_process_group()


def test_whole_job_rate_is_sum_of_units_over_slowest_rank_gloo_world2():
    import socket

    import torch.multiprocessing as mp

    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    got = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, rate, mx, sm, seed in got:
        assert mx == 2000.0 and sm == 300.0
        assert rate == pytest.approx(300.0 / 2.0)          # all units / slowest rank's seconds
    assert got[0][4] is None and got[1][4] == 20220309 + 4 + 1000      # distinct problems per replica


def test_single_process_needs_no_process_group():
    sys.path.insert(0, ROOT)
    from paper_2203_09621_b200 import replicas

    assert replicas.max_over_ranks(3.5) == 3.5 and replicas.sum_over_ranks(2.0) == 2.0
    assert replicas.whole_job_rate(10.0, 500.0) == pytest.approx(20.0)


def test_reference_arm_prints_one_json_line_on_rank0_only():
    """`bench.py --impl reference`: the fp64 oracle on a bounded sample; other ranks exit 0 without work."""
    env = dict(os.environ, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2"],
                       env=env, capture_output=True, text=True, timeout=300)
    assert r.returncode == 0 and r.stdout.strip() == ""
    env = dict(os.environ, RANK="0", WORLD_SIZE="1", LOCAL_RANK="0")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--steps", "1",
                        "--warmup", "0", "--ref-n", "128", "--ref-layers", "3"],
                       env=env, capture_output=True, text=True, timeout=300)
    assert r.returncode == 0, r.stderr
    lines = [ln for ln in r.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["metric"] == "dmpt_layer_tflops_fma1" and d["higher_is_better"] is True
    assert d["value"] > 0 and d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["value"] == d["value"]
    assert d["e2e"] == {"value": d["value"], "unit": d["unit"], "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}
