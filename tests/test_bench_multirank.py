"""The N > 1 path of bench.py on CPU: two gloo ranks (the path does not shard, `--gpus N` runs N
independent replicas; only the timing is reduced across ranks: max over ranks, value = all ranks' rounds / that time)."""

import os
import subprocess
import sys
import textwrap

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = textwrap.dedent("""
    import os, sys, json
    sys.path.insert(0, %r)
    import torch.distributed as dist
    import bench
    dist.init_process_group("gloo")
    rank, world = dist.get_rank(), dist.get_world_size()
    ms_local = [40.0, 55.0][rank]                       # rank 1 is the slow replica
    ms = bench.barrier_max(ms_local, world, device="cpu")
    if rank == 0:
        print(json.dumps({"ms": ms, "value": bench.whole_job_value(10, world, ms)}))
    dist.barrier()
    dist.destroy_process_group()
""") % ROOT


def test_two_rank_replicas_report_max_time_and_aggregate_value(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(WORKER)
    env = dict(os.environ, MASTER_ADDR="127.0.0.1")
    out = subprocess.run([sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2",
                          "--master-addr", "127.0.0.1", "--master-port", "29731", str(script)],
                         capture_output=True, text=True, timeout=240, env=env, cwd=ROOT)
    assert out.returncode == 0, out.stderr[-2000:]
    import json
    line = [l for l in out.stdout.splitlines() if l.startswith("{")][-1]
    res = json.loads(line)
    assert res["ms"] == 55.0                                   # the slowest rank's time
    assert abs(res["value"] - 2 * 10 / 0.055) < 1e-9           # whole-job rounds/s over both replicas


def test_reference_arm_runs_on_rank0_only():
    """--impl reference under a multi-rank launch: rank 0 alone works and prints, other ranks exit 0 without output."""
    env = dict(os.environ, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1")
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "1",
                          "--warmup", "0", "--workload", "cfg1"], capture_output=True, text=True, timeout=240, env=env, cwd=ROOT)
    assert out.returncode == 0 and out.stdout.strip() == ""
