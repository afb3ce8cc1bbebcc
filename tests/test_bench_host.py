"""Host-side logic of bench.py on CPU: multi-rank aggregation over gloo (world size 2), the reference arm's JSON line."""
import json
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, q):
    import torch.distributed as dist
    sys.path.insert(0, ROOT)
    import bench
    dist.init_process_group("gloo", init_method="tcp://127.0.0.1:%d" % port, rank=rank, world_size=world)
    ms = bench.max_over_ranks(10.0 + 5.0 * rank, world)          # rank 1 is the slow one
    q.put((rank, ms, bench.aggregate_value(1000, 4, world, ms)))
    dist.barrier()
    dist.destroy_process_group()


def test_max_over_ranks_gloo_world2():
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29500 + os.getpid() % 2000
    ps = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in ps:
        p.start()
    res = sorted(q.get(timeout=120) for _ in ps)
    for p in ps:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, ms, val in res:
        assert ms == 15.0                                         # time = max over ranks
        assert val == pytest.approx(1000 * 4 * 2 / 15e-3)         # whole-job aggregate over both ranks


def test_reference_arm_line_and_silent_nonzero_ranks():
    env = dict(os.environ, OMP_NUM_THREADS="4")
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--config", "1",
                          "--steps", "1", "--warmup", "0"], capture_output=True, text=True, env=env, timeout=300)
    assert out.returncode == 0, out.stderr
    line = json.loads(out.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["value"] > 0 and line["unit"] == "cell-direction updates/s"
    assert line["cpu_baseline"]["kind"] == "oracle" and line["cpu_baseline"]["cores"] == 4
    assert line["e2e"]["h2d_bytes_per_step"] == 0 and line["e2e"]["d2h_bytes_per_step"] == 0
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--config", "1"],
                         capture_output=True, text=True, env=dict(env, RANK="1", WORLD_SIZE="2"), timeout=60)
    assert out.returncode == 0 and out.stdout.strip() == ""


def test_measured_peak_and_clock_parser():
    sys.path.insert(0, ROOT)
    import bench
    gbs, which = bench.measured_peak()
    assert gbs > 1000 and ("measured" in which or "fallback" in which)
    c = bench.ClockSampler()
    c.proc = object()
    c.rows = [["1965", "1965", "300.1", "Not Active", "Not Active", "Not Active", "Active"],
              ["1800", "1965", "310.0", "Not Active", "Not Active", "Not Active", "Not Active"]]
    c.proc = type("P", (), {"terminate": lambda self: None, "wait": lambda self, timeout=None: None})()
    r = c.stop()
    assert r["sm_max_mhz"] == 1965 and r["reasons"] == ["sw_power_cap"] and r["samples"] == 2
