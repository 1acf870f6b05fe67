"""The N > 1 host logic of bench.py on CPU (gloo, world_size 2): the path is single-GPU by BASELINE.json
north_star, so N ranks are N independent replicas and the only cross-rank logic is the
barrier around the timed region, the max-over-ranks of the time, and "rank 0 alone prints".  No GPU needed."""
import json
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r'''
import os, sys
sys.path.insert(0, {root!r})
import torch, torch.distributed as dist
import bench
rank, local_rank, world = bench.dist_env()
assert world == 2 and rank in (0, 1) and local_rank == rank
dist.init_process_group("gloo")
bench.barrier()
t = bench.max_over_ranks(10.0 + 5.0 * rank)          # every rank must see the slowest replica's time
assert t == 15.0, t
assert bench.max_over_ranks(3.0 - rank) == 3.0
bench.barrier()
if rank == 0:
    print("RESULT", t)
dist.destroy_process_group()
'''


def test_max_over_ranks_and_barrier_world_size_2(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(WORKER.format(root=ROOT))
    env = dict(os.environ, MASTER_ADDR="127.0.0.1", MASTER_PORT="29533")
    out = subprocess.run([sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2",
                          "--master-addr", "127.0.0.1", "--master-port", "29533", str(script)],
                         capture_output=True, text=True, env=env, timeout=300)
    assert out.returncode == 0, out.stderr[-2000:]
    assert out.stdout.count("RESULT 15.0") == 1


def test_reference_arm_prints_on_rank_0_only(tmp_path):
    """bench.py --impl reference under two ranks: rank 1 exits 0 without work, rank 0 prints ONE JSON line."""
    env1 = dict(os.environ, RANK="1", LOCAL_RANK="1", WORLD_SIZE="2")
    r1 = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2"],
                        capture_output=True, text=True, env=env1, timeout=120)
    assert r1.returncode == 0 and r1.stdout.strip() == ""
    env0 = dict(os.environ, RANK="0", LOCAL_RANK="0", WORLD_SIZE="2")
    r0 = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
                         "--workload", "C1", "--steps", "1", "--warmup", "1", "--oracle-rows", "20000"],
                        capture_output=True, text=True, env=env0, timeout=300)
    assert r0.returncode == 0, r0.stderr[-2000:]
    lines = [ln for ln in r0.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["cpu_baseline"]["kind"] == "oracle" and d["gpu_launches"] == 0
    assert d["e2e"]["h2d_bytes_per_step"] == 0 and d["metric"] == "ms_per_lsqr_iteration"
