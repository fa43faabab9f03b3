"""Host logic of bench.py that needs no GPU: the stratified oracle sample and the N > 1 aggregation
(MAX of the per-rank times, SUM of the per-rank units) over a world_size-2 gloo group on CPU."""
import os
import socket
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
import bench  # noqa: E402


def test_sample_regions_are_distinct_aligned_and_in_range():
    regs = bench.sample_regions(256, 300)
    assert len(regs) == 300 and len(set(regs)) == 300
    assert regs[0] == ((0, 0, 0), (16, 16, 16))            # a domain corner is always in the sample
    for lo, hi in regs:
        assert all(l % 16 == 0 and h == l + 16 and 0 <= l and h <= 256 for l, h in zip(lo, hi))
    faces = sum(1 for lo, hi in regs if min(lo) == 0 or max(hi) == 256)
    assert 0 < faces < len(regs)                             # boundary and interior regions both occur
    assert bench.sample_regions(256, 300)[:10] == regs[:10]  # deterministic


def test_single_rank_aggregate_is_identity():
    assert bench.aggregate_over_ranks(12.5, 1000) == (12.5, 1000)


def _worker(rank, world, port, out):
    import torch
    import torch.distributed as dist
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    ms, units = bench.aggregate_over_ranks(10.0 + 5.0 * rank, 1000 * (rank + 1), dist, torch.device("cpu"))
    out[rank] = (ms, units)
    dist.destroy_process_group()


def test_aggregate_over_two_gloo_ranks():
    import torch.multiprocessing as mp
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    mgr = mp.Manager()
    out = mgr.dict()
    mp.spawn(_worker, args=(2, port, out), nprocs=2, join=True)
    assert out[0] == out[1] == (15.0, 3000)                 # max of the times, sum of the units


def test_reference_arm_line():
    """`bench.py --impl reference` needs no GPU: the oracle on the host cores, one JSON line with the contract's keys."""
    import json
    import subprocess
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--workload", "cfg2", "--steps", "1",
                        "--warmup", "1", "--ref-seconds", "0.2"], capture_output=True, text=True, cwd=ROOT, timeout=600)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [l for l in r.stdout.splitlines() if l.strip()]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["metric"] == "fmm_cell_interactions_per_s" and d["value"] > 0
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["value"] == d["value"]
    assert d["e2e"] == {"value": d["value"], "unit": d["unit"], "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}
