"""Host-side logic of bench.py that needs no GPU, including the N > 1 path under gloo
(world_size 2): row-shard assignment, barrier + max-over-ranks aggregation, JSON contract of
the reference arm."""
import json
import os
import subprocess
import sys
from pathlib import Path

import pytest

ROOT = Path(__file__).resolve().parents[1]
sys.path.insert(0, str(ROOT))
import bench  # noqa: E402


def test_shard_rows_partition_the_global_db():
    world, rows = 4, 131072
    spans = [bench.shard_rows(r, world, rows) for r in range(world)]
    assert spans[0][0] == 0 and spans[-1][1] == world * rows
    for a, b in zip(spans, spans[1:]):
        assert a[1] == b[0]
    assert all(hi - lo == rows for lo, hi in spans)  # weak scaling: fixed work per GPU


def test_aggregate_uses_slowest_rank():
    value, ms = bench.aggregate([100.0, 125.0], units_per_rank=16.0, steps=50)
    assert ms == pytest.approx(2.5)
    assert value == pytest.approx(2 * 16.0 * 50 / 0.125)


def _worker(rank, world, port, q):
    import torch
    import torch.distributed as dist
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    lo, hi = bench.shard_rows(rank, world, 1024)
    dist.barrier()
    my_ms = 10.0 * (rank + 1)  # pretend device time of this rank's timed region
    t = torch.tensor([my_ms, float(lo), float(hi)], dtype=torch.float64)
    gathered = [torch.zeros_like(t) for _ in range(world)]
    dist.all_gather(gathered, t)
    dist.barrier()
    if rank == 0:
        times = [float(g[0]) for g in gathered]
        spans = [(int(g[1]), int(g[2])) for g in gathered]
        value, ms = bench.aggregate(times, units_per_rank=1.0, steps=10)
        q.put((times, spans, value, ms))
    dist.destroy_process_group()


def test_two_rank_gloo_aggregation():
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29500 + os.getpid() % 2000
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    times, spans, value, ms = q.get(timeout=120)
    for p in procs:
        p.join(60)
        assert p.exitcode == 0
    assert times == [10.0, 20.0] and spans == [(0, 1024), (1024, 2048)]
    assert ms == pytest.approx(2.0) and value == pytest.approx(2 * 10 / 0.020)


def test_reference_arm_json_contract():
    out = subprocess.run([sys.executable, str(ROOT / "bench.py"), "--impl", "reference", "--steps", "1", "--warmup", "1",
                          "--ref-sample-rows", "64"], capture_output=True, text=True, timeout=300, cwd=ROOT)
    assert out.returncode == 0, out.stderr
    line = json.loads(out.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["metric"] == bench.METRIC and line["unit"] == bench.UNIT
    assert line["higher_is_better"] is True and line["value"] > 0
    assert line["cpu_baseline"]["kind"] == "oracle" and line["cpu_baseline"]["cores"] >= 1
    assert line["e2e"] == {"value": line["value"], "unit": bench.UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}


def test_reference_arm_nonzero_rank_exits_quietly():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2")
    out = subprocess.run([sys.executable, str(ROOT / "bench.py"), "--impl", "reference", "--steps", "1"],
                         capture_output=True, text=True, timeout=120, cwd=ROOT, env=env)
    assert out.returncode == 0 and out.stdout.strip() == ""
