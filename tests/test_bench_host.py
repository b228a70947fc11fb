"""Host logic of bench.py for N > 1 (replicas only): the max-over-ranks timing and the
whole-job value, exercised with world_size 2 on the gloo backend (no GPU), and the reference arm's JSON line."""
from __future__ import annotations

import json
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank: int, world: int, port: int, out_dir: str):
    import torch.distributed as dist
    sys.path.insert(0, ROOT)
    import bench
    dist.init_process_group("gloo", init_method=f"tcp://127.0.0.1:{port}", rank=rank, world_size=world)
    ms = 10.0 + 5.0 * rank                      # rank 1 is the slow replica
    ms_max = bench.max_over_ranks(ms, world, "cpu")
    value = bench.job_value(world, 1000, 4, ms_max)
    with open(os.path.join(out_dir, f"r{rank}.json"), "w") as f:
        json.dump({"ms_max": ms_max, "value": value}, f)
    dist.destroy_process_group()


def test_max_over_ranks_and_job_value_world2(tmp_path):
    import torch.multiprocessing as mp
    port = 29500 + os.getpid() % 2000
    mp.spawn(_worker, args=(2, port, str(tmp_path)), nprocs=2, join=True)
    for r in range(2):
        rec = json.load(open(tmp_path / f"r{r}.json"))
        assert rec["ms_max"] == 15.0                                # the slowest rank on every rank
        assert rec["value"] == pytest.approx(2 * 1000 * 4 / 15.0e-3)  # both replicas' cells over that time


def test_single_rank_passthrough():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.max_over_ranks(3.5, 1, "cpu") == 3.5
    assert bench.job_value(1, 100, 2, 10.0) == pytest.approx(100 * 2 / 10.0e-3)
    names3, names2, names2odd = bench.kernel_names(3, 1024), bench.kernel_names(2, 16384), bench.kernel_names(2, 29)
    assert names3["Lz+"].startswith("k_march3") and names3["Lx-"].startswith("k_lane3")
    assert names2["Lz+"].startswith("k_march ") and names2["Lx-"].startswith("k_lane2 ")
    assert names2odd["Lx+"].startswith("k_lane ")


def test_reference_arm_prints_one_json_line():
    """--impl reference runs the oracle on a bounded sample and prints the contract's keys (C1 is small)."""
    res = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--workload", "C1",
                          "--steps", "2", "--warmup", "1"], capture_output=True, text=True, timeout=600, cwd=ROOT)
    assert res.returncode == 0, res.stderr
    lines = [l for l in res.stdout.splitlines() if l.strip()]
    assert len(lines) == 1
    rec = json.loads(lines[0])
    assert rec["impl"] == "reference" and rec["unit"] == "cell-updates/s" and rec["value"] > 0
    assert rec["cpu_baseline"]["kind"] == "oracle" and rec["cpu_baseline"]["cores"] == 1
    assert rec["e2e"]["h2d_bytes_per_step"] == 0 and rec["e2e"]["d2h_bytes_per_step"] == 0
