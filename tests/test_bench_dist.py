"""CPU, world_size 2, gloo: the host-side multi-process logic of bench.py (replicas only -- no data-path
collective; ranks only agree on the time of the slowest one and rank 0 reports the sum of the work)."""
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r'''
import json, os, sys
sys.path.insert(0, %r)
import torch
import torch.distributed as dist
import bench
rank, world, local = bench.dist_env()
dist.init_process_group("gloo")
ms_local = 10.0 + 5.0 * rank                      # rank 1 is the slow replica
ms = bench.max_over_ranks(torch, dist, ms_local, torch.device("cpu"))
dist.barrier()
if rank == 0:
    print(json.dumps({"world": world, "ms": ms, "value": bench.whole_job_gflops(world, 1000, ms)}))
dist.destroy_process_group()
'''


def test_replica_timing_is_max_over_ranks_and_value_is_whole_job(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(WORKER % ROOT)
    env = dict(os.environ, MASTER_ADDR="127.0.0.1")
    out = subprocess.run([sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2",
                          "--master-addr", "127.0.0.1", "--master-port", "29541", str(script)],
                         capture_output=True, text=True, timeout=300, env=env)
    assert out.returncode == 0, out.stderr[-2000:]
    import json
    line = [l for l in out.stdout.splitlines() if l.startswith("{")][-1]
    d = json.loads(line)
    assert d["world"] == 2
    assert abs(d["ms"] - 15.0) < 1e-9                       # the slowest rank's time
    import bench
    assert abs(d["value"] - 2 * bench.whole_job_gflops(1, 1000, 15.0)) < 1e-9   # sum of both replicas' work


def test_reference_arm_runs_on_rank0_only():
    """Under torchrun the oracle arm runs on rank 0 alone; other ranks exit 0 without output."""
    env = dict(os.environ, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1")
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "1",
                          "--warmup", "1"], capture_output=True, text=True, timeout=300, env=env)
    assert out.returncode == 0 and out.stdout.strip() == ""
