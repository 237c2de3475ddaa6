"""-m "not gpu": the N>1 plumbing of bench.py on CPU with the gloo backend, world_size 2.  The path itself does not shard
(replicas only, no collective on the data path); what runs across ranks is the timing reduction (max over
ranks), the whole-job aggregate and the per-rank seeding, plus the reference arm's "rank 0 only" rule."""
import json
import os
import subprocess
import sys
import textwrap

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = textwrap.dedent("""
    import json, os, sys
    sys.path.insert(0, {root!r})
    import numpy as np
    import torch, torch.distributed as dist
    import bench
    from paper_2604_06575_b200 import workloads as W
    dist.init_process_group("gloo")
    rank, world = dist.get_rank(), dist.get_world_size()
    ms = bench.max_over_ranks(dist, 10.0 + 5.0 * rank, "cpu")          # rank 1 is the slow one
    p, _ = W.config1(1000, bench.replica_seed_offset(rank))
    digest = float(np.abs(p.coef).sum())
    out = [None] * world
    dist.all_gather_object(out, digest)
    if rank == 0:
        print(json.dumps({{"ms": ms, "value": bench.aggregate_value(1000, world, ms), "digests": out}}))
    dist.destroy_process_group()
""")


def test_two_rank_gloo_timing_and_replicas(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(WORKER.format(root=ROOT))
    env = dict(os.environ, MASTER_ADDR="127.0.0.1")
    r = subprocess.run([sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node=2", "--master-addr", "127.0.0.1",
                        "--master-port", "29731", str(script)], capture_output=True, text=True, timeout=300, env=env, cwd=ROOT)
    assert r.returncode == 0, r.stderr[-2000:]
    line = [l for l in r.stdout.splitlines() if l.startswith("{")][-1]
    d = json.loads(line)
    assert d["ms"] == 15.0                                     # the slowest rank's time
    assert abs(d["value"] - 2 * 1000 / 15e-3) < 1e-6           # terms of BOTH ranks over that time
    assert d["digests"][0] != d["digests"][1]                  # each rank has its own polynomial


def test_reference_arm_runs_on_rank_zero_only():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "1",
                        "--warmup", "0", "--config", "1"], capture_output=True, text=True, timeout=300, env=env, cwd=ROOT)
    assert r.returncode == 0 and r.stdout.strip() == ""        # ranks other than 0 exit without work
    env["RANK"] = "0"
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "1",
                        "--warmup", "0", "--config", "1"], capture_output=True, text=True, timeout=300, env=env, cwd=ROOT)
    assert r.returncode == 0, r.stderr[-2000:]
    d = json.loads(r.stdout.strip().splitlines()[-1])
    assert d["impl"] == "reference" and d["cpu_baseline"]["kind"] == "oracle" and d["value"] > 0
    assert d["e2e"]["h2d_bytes_per_step"] == 0 and d["e2e"]["d2h_bytes_per_step"] == 0
