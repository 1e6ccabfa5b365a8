"""N > 1 path of bench.py on CPU: two gloo ranks (world_size 2, 127.0.0.1).  The hot path does not shard
(replicas only), so the only multi-rank logic is the reduction of the timing (MAX) and of
the particle updates (SUM) and the rule that only rank 0 runs the reference arm."""
import json
import os
import socket
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

_WORKER = r"""
import os, sys
sys.path.insert(0, os.environ["GRPIC_ROOT"])
import torch.distributed as dist
import bench
dist.init_process_group("gloo")
rank = dist.get_rank()
ms, units = bench.reduce_over_ranks(10.0 + 5.0 * rank, 1000 * (rank + 1), dist.get_world_size(), device="cpu")
assert ms == 15.0 and units == 3000.0, (ms, units)
dist.barrier()
dist.destroy_process_group()
open(os.path.join(os.environ["GRPIC_OUT"], f"rank{rank}.ok"), "w").write("ok")
"""


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def test_reduce_over_ranks_gloo_world2(tmp_path):
    w = tmp_path / "worker.py"
    w.write_text(_WORKER)
    env = dict(os.environ, GRPIC_ROOT=ROOT, GRPIC_OUT=str(tmp_path), MASTER_ADDR="127.0.0.1")
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node=2", "--master-addr", "127.0.0.1",
           "--master-port", str(_free_port()), str(w)]
    r = subprocess.run(cmd, env=env, capture_output=True, text=True, timeout=300)
    assert r.returncode == 0, r.stdout + r.stderr
    assert (tmp_path / "rank0.ok").exists() and (tmp_path / "rank1.ok").exists()   # both ranks passed their asserts


def test_reference_arm_runs_on_rank0_only():
    """--impl reference under torchrun: rank != 0 exits 0 without work or output."""
    env = dict(os.environ, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "1",
                        "--warmup", "0"], env=env, capture_output=True, text=True, timeout=120)
    assert r.returncode == 0 and r.stdout.strip() == ""


def test_reference_arm_line_small():
    """The reference arm prints one JSON line with the contract's keys (tiny workload so that the CPU suite stays short)."""
    env = dict(os.environ)
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--workload", "tiny", "--steps", "1",
                        "--warmup", "0"], env=env, capture_output=True, text=True, timeout=600)
    assert r.returncode == 0, r.stderr
    d = json.loads(r.stdout.strip().splitlines()[-1])
    assert d["impl"] == "reference" and d["unit"] == "updates/s" and d["value"] > 0
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["cores"] >= 1
    assert d["e2e"]["h2d_bytes_per_step"] == 0 and d["e2e"]["d2h_bytes_per_step"] == 0
