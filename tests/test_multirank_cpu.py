"""The N>1 path of bench.py: massive mode = replicas only; the particle and
multi-system modes shard their particles / systems (workloads.shard) with no data-path
collective.  The only cross-rank traffic is the max-over-ranks of the elapsed time and the sum of the
units.  Exercised here with world_size 2 on the gloo backend, the shards stepped by the oracle."""
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
    # under N ranks the multi-system config is N times as large and each rank holds its 4096 systems
    w0, _ = bench.workload(3, 0, 2)
    w1, _ = bench.workload(3, 1, 2)
    assert w0["n_systems"] == w1["n_systems"] == 4096 and w1["shard"] == (1, 2, 4096, 8192)
    full, _ = bench.workload(3)
    assert (w0["x"] == full["x"]).all() and not (w1["x"] == full["x"]).all()
    assert bench.workload(1, 1, 2)[0]["x"].shape == (3, 2048)          # massive mode: replicas


SHARD_WORKER = r"""
import os, sys
sys.path.insert(0, %r)
import numpy as np, torch, torch.distributed as dist
import workloads, oracle, bench
dist.init_process_group("gloo")
r, W = dist.get_rank(), dist.get_world_size()
for full in (workloads.config2(n_massive=3, n_test=41), workloads.config3(n_systems=5, n_per=6)):
    w = workloads.shard(full, r, W)
    o = oracle.Sim(w)
    o.step(3, w["dt"], w["order"])
    x, v = o.state()
    per, _ = bench.interactions_per_step(w)
    perf, _ = bench.interactions_per_step(full)
    _, u = bench.reduce_max_and_sum(1.0, per, torch.device("cpu"))
    assert u == perf, (u, perf)                       # the shards' units add up to the global job's
    # rank 0 checks every shard against the unsharded oracle run, bit for bit
    parts = [None] * W
    dist.all_gather_object(parts, (w["shard"], x, v))
    if r == 0:
        of = oracle.Sim(full); of.step(3, full["dt"], full["order"]); xf, vf = of.state()
        nm = full["n_massive"]
        for (rk, _, lo, hi), xs, vs in parts:
            if full["mode"] == 1:
                assert np.array_equal(xs[:, :nm], xf[:, :nm]) and np.array_equal(vs[:, :nm], vf[:, :nm])
                assert np.array_equal(xs[:, nm:], xf[:, nm + lo:nm + hi]) and np.array_equal(vs[:, nm:], vf[:, nm + lo:nm + hi])
            else:
                assert np.array_equal(xs, xf[:, lo * nm:hi * nm]) and np.array_equal(vs, vf[:, lo * nm:hi * nm])
dist.barrier()
if r == 0:
    print("SHARDS OK")
dist.destroy_process_group()
"""


def test_sharded_modes_world_size_2(tmp_path):
    script = tmp_path / "shard_worker.py"
    script.write_text(SHARD_WORKER % ROOT)
    env = dict(os.environ, MASTER_ADDR="127.0.0.1")
    out = subprocess.run([sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2",
                          "--master-addr", "127.0.0.1", "--master-port", "29618", str(script)],
                         capture_output=True, text=True, env=env, timeout=300)
    assert out.returncode == 0, out.stderr[-2000:]
    assert "SHARDS OK" in out.stdout


def test_shard_partitions_cover_every_unit_once():
    import numpy as np
    import pytest
    import workloads
    full = workloads.config2(n_massive=4, n_test=103)
    seen = []
    for r in range(5):
        w = workloads.shard(full, r, 5)
        assert w["n_massive"] == 4 and w["x"].shape == (3, 4 + w["n_test"])
        assert np.array_equal(w["x"][:, :4], full["x"][:, :4])
        seen.append(w["x"][:, 4:])
    assert np.array_equal(np.concatenate(seen, axis=1), full["x"][:, 4:])
    full = workloads.config3(n_systems=7, n_per=5)
    parts = [workloads.shard(full, r, 3) for r in range(3)]
    assert sum(p["n_systems"] for p in parts) == 7
    assert np.array_equal(np.concatenate([p["v"] for p in parts], axis=1), full["v"])
    assert np.array_equal(np.concatenate([p["m0"] for p in parts]), full["m0"])
    with pytest.raises(ValueError):
        workloads.shard(workloads.config0(), 0, 2)
    with pytest.raises(ValueError):
        workloads.shard(full, 3, 3)
