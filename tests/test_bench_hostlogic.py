"""Host logic of bench.py that needs no GPU: the N > 1 aggregation (replicas only) over a
world_size-2 gloo group, the algorithmic-byte count, and the reference arm's JSON line."""
import json
import os
import socket
import subprocess
import sys

import pytest
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
import bench  # noqa: E402


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _rank_main(rank, world, port, out_dir):
    import torch.distributed as dist
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    # rank r: its own chain flipped 1000*(r+1) spins in 10*(r+1) updates and took 2*(r+1) ms on its device
    agg = bench.aggregate_replicas(1000 * (rank + 1), 10 * (rank + 1), 2.0 * (rank + 1), world)
    with open(os.path.join(out_dir, "rank%d.json" % rank), "w") as f:
        json.dump(agg, f)
    dist.barrier()
    dist.destroy_process_group()


def test_replica_aggregation_world_size_2_gloo(tmp_path):
    world = 2
    mp.spawn(_rank_main, args=(world, _free_port(), str(tmp_path)), nprocs=world, join=True)
    for rank in range(world):
        agg = json.load(open(tmp_path / ("rank%d.json" % rank)))
        assert agg["flipped"] == 3000 and agg["updates"] == 30      # sum over ranks
        assert agg["total_ms"] == 4.0                               # max over ranks
        assert agg["value"] == pytest.approx(3000 / 4e-3)           # whole-job units / slowest rank
        assert agg["updates_per_s"] == pytest.approx(30 / 4e-3)


def test_single_rank_is_a_no_op():
    agg = bench.aggregate_replicas(500, 5, 2.5, 1)
    assert agg == {"total_ms": 2.5, "flipped": 500, "updates": 5, "value": 500 / 2.5e-3, "updates_per_s": 5 / 2.5e-3}


def test_algorithmic_bytes_per_added_spin():
    # 2*dim neighbour bytes + 4 (list write) + 4 (list read) per spin, 4 per claim attempt
    assert bench.algorithmic_bytes(2, 100, 117) == 100 * 12 + 4 * 117
    assert bench.algorithmic_bytes(3, 100, 107) == 100 * 14 + 4 * 107


def test_reference_arm_prints_one_json_line():
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--workload", "C1",
                          "--steps", "2", "--warmup", "1", "--reference-updates", "50"],
                         capture_output=True, text=True, timeout=300, cwd=ROOT)
    assert out.returncode == 0, out.stderr
    lines = [l for l in out.stdout.splitlines() if l.strip()]
    assert len(lines) == 1
    rec = json.loads(lines[0])
    assert rec["impl"] == "reference" and rec["gpu_launches"] == 0
    assert rec["cpu_baseline"]["kind"] == "oracle" and rec["cpu_baseline"]["value"] == rec["value"]
    assert rec["e2e"] == {"value": rec["value"], "unit": rec["unit"], "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}
    assert rec["value"] > 0 and rec["higher_is_better"] is True


def test_reference_arm_other_ranks_exit_quietly():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2")
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2"],
                         capture_output=True, text=True, timeout=120, cwd=ROOT, env=env)
    assert out.returncode == 0 and out.stdout.strip() == ""
