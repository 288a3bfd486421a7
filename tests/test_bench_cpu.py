"""Host-side logic of bench.py for N > 1, on CPU with the gloo backend (world_size 2): the
max-over-ranks reduction, the whole-job aggregate, and the reference arm under torchrun (rank 0
alone prints one JSON line, the other rank exits 0 without work)."""
import json
import os
import socket
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


WORKER = r"""
import os, sys, json
sys.path.insert(0, {root!r})
import torch.distributed as dist
import bench
dist.init_process_group("gloo")
rank, world = dist.get_rank(), dist.get_world_size()
ms = 10.0 if rank == 0 else 25.0            # rank 1 is the slow one
slow = bench.max_over_ranks(ms, world, "cpu")
with open(os.path.join({out!r}, "rank%d.json" % rank), "w") as f:       # one file per rank: stdout of two ranks can interleave
    json.dump({{"rank": rank, "world": world, "slow": slow,
               "value": bench.aggregate_value(5.0e9, world, slow)}}, f)
dist.destroy_process_group()
"""


def test_max_over_ranks_and_aggregate_world2(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(WORKER.format(root=ROOT, out=str(tmp_path)))
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2",
           "--master-addr", "127.0.0.1", "--master-port", str(free_port()), str(script)]
    out = subprocess.run(cmd, capture_output=True, text=True, timeout=300, cwd=ROOT)
    assert out.returncode == 0, out.stderr[-2000:]
    lines = [json.loads((tmp_path / f"rank{r}.json").read_text()) for r in (0, 1)]
    assert sorted(l["rank"] for l in lines) == [0, 1]
    for l in lines:
        assert l["world"] == 2 and l["slow"] == 25.0                    # every rank sees the slowest time
        assert l["value"] == pytest.approx(2 * 5.0e9 / 25.0e-3 / 1e9)   # all ranks' units / that time


def test_single_rank_needs_no_process_group():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.max_over_ranks(7.5, 1, "cpu") == 7.5
    assert bench.aggregate_value(1.0e9, 1, 1000.0) == pytest.approx(1.0)


def test_reference_arm_under_torchrun_world2():
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2",
           "--master-addr", "127.0.0.1", "--master-port", str(free_port()),
           os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "1",
           "--warmup", "0", "--workload", "cfg0_100x100x67_n10"]
    out = subprocess.run(cmd, capture_output=True, text=True, timeout=600, cwd=ROOT)
    assert out.returncode == 0, out.stderr[-2000:]
    lines = [json.loads(l) for l in out.stdout.splitlines() if l.startswith('{"')]
    assert len(lines) == 1                                               # rank 0 alone prints
    r = lines[0]
    assert r["impl"] == "reference" and r["n_gpus"] == 2 and r["unit"] == "Gvoxel-iter/s"
    assert r["cpu_baseline"]["kind"] == "oracle" and r["cpu_baseline"]["value"] == r["value"] > 0
    assert r["e2e"] == {"value": r["value"], "unit": r["unit"], "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}


def test_ncu_counter_table_lookup():
    """bench.py's `roofline.traffic`, its ALU figures and L2 bytes come from profiles/ncu_per_launch.txt, keyed by
    (plan, workload); every entry names the note and commit it was measured at, and a plan that was never captured
    on a workload gets nothing (the line then withholds the figures instead of borrowing another plan's)."""
    sys.path.insert(0, ROOT)
    import bench
    e = bench.ncu_counters("idg_tma_kernel fuse=4 tile=0", "cfg3_1024x1024x512_n20")
    assert 4.2e9 < e["dram_bytes"] < 4.6e9 and e["warp_instructions"] > 9e8 and "source" in e and "commit" in e
    assert bench.ncu_counters("no such kernel", "cfg3_1024x1024x512_n20") == {}
    assert bench.ncu_counters("idg_tma_kernel fuse=4 tile=0", "cfg0_100x100x67_n10") == {}
    table = json.load(open(os.path.join(ROOT, "profiles", "ncu_per_launch.txt")))["entries"]
    for entry in table:
        assert os.path.exists(os.path.join(ROOT, entry["source"].split(" ")[0])), entry["source"]
        assert entry["workload"] in bench.WORKLOADS
