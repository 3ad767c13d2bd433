"""world_size-2 gloo test (CPU) of bench.py's multi-rank host logic (replicas only):
the max-over-ranks reduction of the step time, the whole-job rate, and the reference arm's rank rule."""
import json
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r"""
import os, sys, json
sys.path.insert(0, {root!r})
import torch, torch.distributed as dist
import bench
dist.init_process_group(backend="gloo")
rank, world = dist.get_rank(), dist.get_world_size()
ms = bench.max_over_ranks(10.0 * (rank + 1), dist)          # ranks report 10 ms and 20 ms
rate = bench.aggregate_rate(1_000_000_000, world, ms)       # 1e9 pairs per rank
# line sharding: 7 rings over 2 ranks (4 + 3); every rank holds "I(q)" of its own rings, value = 100 * map + ring
n0 = 7
i0, i1 = bench.shard_lines(n0, world, rank)
local = torch.stack([100.0 * k + torch.arange(i0, i1, dtype=torch.float32) for k in range(3)])
full = bench.gather_lines(local, n0, world, rank, dist)
dist.barrier()
if rank == 0:
    print(json.dumps({{"ms": ms, "rate": rate, "world": world, "full": full.tolist(), "share": [i0, i1]}}))
dist.destroy_process_group()
"""


def test_max_over_ranks_and_aggregate_rate_gloo(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(WORKER.format(root=ROOT))
    env = dict(os.environ, MASTER_ADDR="127.0.0.1")
    out = subprocess.run([sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2",
                          "--master-addr", "127.0.0.1", "--master-port", "29533", str(script)],
                         capture_output=True, text=True, timeout=300, env=env, cwd=ROOT)
    assert out.returncode == 0, out.stderr[-2000:]
    line = [l for l in out.stdout.splitlines() if l.startswith("{")][-1]
    d = json.loads(line)
    assert d["world"] == 2
    assert d["ms"] == pytest.approx(20.0)                      # the slower rank decides
    assert d["rate"] == pytest.approx(2 * 1e9 / 20e-3 / 1e9)   # both ranks' pairs over the max time
    assert d["share"] == [0, 4]
    assert d["full"] == [[100.0 * k + i for i in range(7)] for k in range(3)]   # rings back in detector order


def test_line_sharding_partitions_the_detector():
    """--shard lines: the ranks' shares are contiguous, balanced, disjoint and cover every detector line; a rank's
    workload is the same sample on the sub-grid with the very same float32 abscissae."""
    sys.path.insert(0, ROOT)
    import numpy as np
    import bench
    import nms_inputs as ni
    for n0 in (1, 7, 64, 512):
        for world in (1, 2, 3, 8):
            shares = [bench.shard_lines(n0, world, r) for r in range(world)]
            assert shares[0][0] == 0 and shares[-1][1] == n0
            assert all(shares[r][1] == shares[r + 1][0] for r in range(world - 1))
            sizes = [b - a for a, b in shares]
            assert max(sizes) - min(sizes) <= 1
    wl = ni.make_config("C5", small=True)
    parts = [bench.shard_workload(wl, 3, r) for r in range(3)]
    assert np.array_equal(np.concatenate([p.grid.u0 for p, _, _ in parts]), wl.grid.u0)
    for p, i0, i1 in parts:
        assert p.grid.n0 == i1 - i0 and p.n_bins == i1 - i0 and np.array_equal(p.grid.u1, wl.grid.u1)
        assert p.pos is wl.pos and p.m is wl.m                      # cells replicated, not copied
    with pytest.raises(SystemExit):
        bench.shard_workload(ni.make_config("C2"), 2, 0)            # |q| histogram on a Cartesian detector


def test_single_process_helpers():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.max_over_ranks(3.5) == 3.5
    assert bench.aggregate_rate(4_000_000_000, 1, 2000.0) == pytest.approx(2.0)


def test_reference_arm_other_ranks_exit_without_work():
    """Under torchrun only rank 0 runs the oracle arm; the other ranks exit 0 and print nothing."""
    env = dict(os.environ, RANK="1", LOCAL_RANK="1", WORLD_SIZE="2")
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2"],
                         capture_output=True, text=True, timeout=120, env=env, cwd=ROOT)
    assert out.returncode == 0, out.stderr[-2000:]
    assert out.stdout.strip() == ""


def test_gpus_n_without_torchrun_starts_its_own_ranks():
    """`python bench.py --gpus 2` outside torchrun re-executes itself under torch.distributed.run with 2 ranks on
    127.0.0.1 (driven here through the oracle arm, which needs no GPU): exactly one JSON line, n_gpus = 2."""
    env = {k: v for k, v in os.environ.items() if k not in ("RANK", "LOCAL_RANK", "WORLD_SIZE", "MASTER_ADDR", "MASTER_PORT")}
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--workload", "C1",
                          "--oracle-seconds", "0.5", "--steps", "1", "--warmup", "0"],
                         capture_output=True, text=True, timeout=300, env=env, cwd=ROOT)
    assert out.returncode == 0, out.stderr[-2000:]
    lines = [l for l in out.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["n_gpus"] == 2 and d["cpu_baseline"]["cores"] >= 1


def test_auto_sharding_rule():
    sys.path.insert(0, ROOT)
    import bench
    import nms_inputs as ni
    assert bench.can_shard_lines(ni.make_config("C5", small=True), 8)         # polar rings
    assert bench.can_shard_lines(ni.make_config("C4", small=True), 2)         # Cartesian rows, no histogram
    assert not bench.can_shard_lines(ni.make_config("C2"), 2)                 # |q| histogram on a Cartesian detector
    assert not bench.can_shard_lines(ni.make_config("C5", small=True), 64)    # more ranks than rings
