"""N > 1 path on CPU: world_size-2 gloo.  The path is 'replicas only': the only
collective is the bench's timing reduction (barrier, max over ranks, sum of units)."""
import json
import os
import socket
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r"""
import json, os, sys
sys.path.insert(0, os.environ["KV_ROOT"])
from paper_2606_31093_b200.replicas import Replicas
rep = Replicas("gloo")
assert rep.world == 2
rep.barrier()
t = [0.25, 0.40][rep.rank]          # this rank's device-timed seconds
units = [100.0, 120.0][rep.rank]    # GB this rank moved
out = {"rank": rep.rank, "tmax": rep.max_over_ranks(t), "usum": rep.sum_over_ranks(units),
       "rate": rep.whole_job_rate(units, t)}
rep.close()
print(json.dumps(out))
"""


def free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def test_two_rank_timing_reduction():
    port = free_port()
    procs = []
    for r in range(2):
        env = dict(os.environ, RANK=str(r), LOCAL_RANK=str(r), WORLD_SIZE="2", MASTER_ADDR="127.0.0.1",
                   MASTER_PORT=str(port), KV_ROOT=ROOT)
        procs.append(subprocess.Popen([sys.executable, "-c", WORKER], env=env, stdout=subprocess.PIPE,
                                      stderr=subprocess.PIPE, text=True))
    outs = []
    for p in procs:
        o, e = p.communicate(timeout=120)
        assert p.returncode == 0, e
        outs.append(json.loads(o.strip().splitlines()[-1]))
    for o in outs:
        assert o["tmax"] == 0.40 and o["usum"] == 220.0
        assert abs(o["rate"] - 220.0 / 0.40) < 1e-9


def test_reference_arm_runs_on_rank0_only():
    """bench.py --impl reference under torchrun: rank 0 prints the line, other ranks exit 0 silently."""
    env = dict(os.environ, RANK="1", LOCAL_RANK="1", WORLD_SIZE="2")
    p = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
                        "--steps", "1", "--warmup", "1"], env=env, capture_output=True, text=True, timeout=120)
    assert p.returncode == 0 and p.stdout.strip() == ""
    env["RANK"] = "0"
    p = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
                        "--steps", "1", "--warmup", "1"], env=env, capture_output=True, text=True, timeout=300)
    assert p.returncode == 0
    line = json.loads(p.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["cpu_baseline"]["kind"] == "oracle" and line["value"] > 0
    assert line["e2e"]["h2d_bytes_per_step"] == 0 and line["unit"] == "GB/s"
