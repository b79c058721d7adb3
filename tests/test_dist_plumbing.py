"""-m "not gpu": the N > 1 plumbing of bench.py (replicas only) with world_size 2 on gloo:
rendezvous from the torchrun environment variables, barrier, max-over-ranks timing, and the reference arm's
rule that only rank 0 runs and prints."""
import json
import os
import socket
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r"""
import os, sys, json
sys.path.insert(0, os.environ["SANGAM_ROOT"])
import bench
rank, world, dist = bench.dist_setup()
assert world == 2 and dist is not None and dist.get_backend() == "gloo"
bench.barrier(dist)
t = bench.max_over_ranks(1.0 + rank, dist)          # rank 1 is the slow one
bench.barrier(dist)
print(json.dumps({"rank": rank, "max": t}))
dist.destroy_process_group()
"""


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _env(rank, port):
    e = dict(os.environ)
    e.update({"RANK": str(rank), "LOCAL_RANK": str(rank), "WORLD_SIZE": "2", "MASTER_ADDR": "127.0.0.1",
              "MASTER_PORT": str(port), "SANGAM_ROOT": ROOT, "CUDA_VISIBLE_DEVICES": ""})
    return e


def test_max_over_ranks_world2_gloo():
    port = _free_port()
    procs = [subprocess.Popen([sys.executable, "-c", WORKER], env=_env(r, port), stdout=subprocess.PIPE,
                              stderr=subprocess.PIPE, text=True) for r in range(2)]
    outs = [p.communicate(timeout=120) for p in procs]
    for p, (o, e) in zip(procs, outs):
        assert p.returncode == 0, e[-2000:]
    vals = [json.loads(o.strip().splitlines()[-1]) for o, _ in outs]
    assert sorted(v["rank"] for v in vals) == [0, 1]
    assert all(v["max"] == 2.0 for v in vals)       # every rank sees the slowest rank's time


def test_reference_arm_only_rank0_prints():
    port = _free_port()
    cmd = [sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "1",
           "--warmup", "0", "--workload", "1"]
    procs = [subprocess.Popen(cmd, env=_env(r, port), stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True)
             for r in range(2)]
    outs = [p.communicate(timeout=300) for p in procs]
    for p, (o, e) in zip(procs, outs):
        assert p.returncode == 0, e[-2000:]
    assert outs[1][0].strip() == ""                 # rank 1 exits 0 without work or output
    line = json.loads(outs[0][0].strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["cpu_baseline"]["kind"] == "oracle" and line["value"] > 0
    assert line["e2e"]["h2d_bytes_per_step"] == 0 and line["e2e"]["d2h_bytes_per_step"] == 0
