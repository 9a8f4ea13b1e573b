"""The N>1 path of bench.py is 'replicas only': each rank steps its own
replica; the only cross-rank traffic is the max-over-ranks of the elapsed time and the sum of the
units.  Exercised here with world_size 2 on the gloo backend."""
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r"""
import os, sys
sys.path.insert(0, %r)
import torch, torch.distributed as dist
import bench
dist.init_process_group("gloo")
r = dist.get_rank()
t, u = bench.reduce_max_and_sum(1.0 + r, 100.0 * (r + 1), torch.device("cpu"))
assert t == 2.0 and u == 300.0, (t, u)
dist.barrier()
if r == 0:
    print("OK", t, u)
dist.destroy_process_group()
"""


def test_replica_aggregation_world_size_2(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(WORKER % ROOT)
    env = dict(os.environ, MASTER_ADDR="127.0.0.1")
    out = subprocess.run([sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2",
                          "--master-addr", "127.0.0.1", "--master-port", "29617", str(script)],
                         capture_output=True, text=True, env=env, timeout=300)
    assert out.returncode == 0, out.stderr[-2000:]
    assert "OK 2.0 300.0" in out.stdout


def test_single_process_aggregation_is_identity():
    import torch
    import bench
    assert bench.reduce_max_and_sum(1.5, 10, torch.device("cpu")) == (1.5, 10)
    w, name = bench.workload(1)
    per, evals = bench.interactions_per_step(w)
    assert evals == 2 and per == 2 * 2048 * 2047
