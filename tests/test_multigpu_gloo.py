"""The N>1 path of bench.py is "replicas only" (the north_star forbids sharding and
collectives on the data path).  Its host-side logic — torchrun-style rendezvous on 127.0.0.1,
barrier, MAX-over-ranks of the device time, SUM-over-ranks of the processed units — is covered
here with world_size 2 on the gloo backend (no GPU needed)."""
import json
import os
import socket
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r"""
import json, os, sys
sys.path.insert(0, %(root)r)
import bench
rank, world = bench.init_dist("gloo")
assert world == 2
bench.barrier(world)
# rank 0 pretends to take 100 ms for 1000 units, rank 1 takes 250 ms for 1000 units
ms = 100.0 if rank == 0 else 250.0
rate, max_ms = bench.aggregate_rate(1000.0, ms, world)
mx = bench.max_over_ranks(float(rank + 1), world)
sm = bench.sum_over_ranks(float(rank + 1), world)
bench.barrier(world)
if rank == 0:
    print(json.dumps({"rate": rate, "max_ms": max_ms, "mx": mx, "sm": sm}))
"""


def free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def test_world_size_2_aggregation_on_gloo(tmp_path):
    port = free_port()
    script = tmp_path / "worker.py"
    script.write_text(WORKER % {"root": ROOT})
    procs = []
    for rank in range(2):
        env = dict(os.environ, RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE="2",
                   MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), CUDA_VISIBLE_DEVICES="")
        procs.append(subprocess.Popen([sys.executable, str(script)], env=env, stdout=subprocess.PIPE,
                                      stderr=subprocess.PIPE, text=True))
    outs = [p.communicate(timeout=240) for p in procs]
    for p, (o, e) in zip(procs, outs):
        assert p.returncode == 0, e[-2000:]
    res = json.loads(outs[0][0].strip().splitlines()[-1])
    assert res["max_ms"] == 250.0                     # the job is as slow as its slowest replica
    assert abs(res["rate"] - 2000.0 / 0.25) < 1e-9    # units of ALL ranks / max time
    assert res["mx"] == 2.0 and res["sm"] == 3.0


def test_reference_arm_prints_one_json_line_and_other_ranks_stay_silent():
    """bench.py --impl reference: rank 0 times the oracle; other ranks exit 0 without work."""
    env = dict(os.environ, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1", CUDA_VISIBLE_DEVICES="")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
                        "--steps", "1", "--warmup", "0"], env=env, capture_output=True, text=True, timeout=240)
    assert r.returncode == 0 and r.stdout.strip() == ""
    env = dict(os.environ, CUDA_VISIBLE_DEVICES="")
    for k in ("RANK", "WORLD_SIZE", "LOCAL_RANK"):
        env.pop(k, None)
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--workload", "k0",
                        "--steps", "2", "--warmup", "1"], env=env, capture_output=True, text=True, timeout=240)
    assert r.returncode == 0, r.stderr[-2000:]
    line = json.loads(r.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["unit"] == "site-updates/s" and line["value"] > 0
    assert line["cpu_baseline"]["kind"] == "oracle" and line["e2e"]["h2d_bytes_per_step"] == 0
