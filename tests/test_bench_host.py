"""Host-side logic of bench.py that needs no GPU: workload construction, the instruction accounting of the
ALU roofline and the JSON description of a workload."""
import numpy as np

import bench
from paper_1003_3779_b200 import inputs as qi


def test_coin_cost_matches_the_kernels_instruction_counts():
    k1 = qi.k1(sites=64, steps=1)
    assert bench.coin_cost(k1, "fused") == (6, 10)                       # 2 mul + 4 fma
    i, f = bench.coin_cost(k1, "blocked")                                # 15 bare butterflies + 1 scaled step per 16
    assert abs(i - (15 * 4 + 6) / 16) < 1e-12 and abs(f - (15 * 4 + 10) / 16) < 1e-12
    k4 = qi.k4(batch=2, half=4, steps=1)
    assert bench.coin_cost(k4, "resident") == (24, 40)                   # general 2x2 (16) + site phase (8)
    for coin, bare in (("hxh", 16), ("dft", 16)):
        k3 = qi.k3(extents=(8, 8), steps=1, coin=coin)
        assert bench.coin_cost(k3, "fused") == (20, 24)
        i, _ = bench.coin_cost(k3, "tiled")
        assert abs(i - (7 * bare + 20) / 8) < 1e-12                      # K = 8 for complex64
    i, _ = bench.coin_cost(qi.k2(half=4), "tiled")
    assert abs(i - (5 * 14 + 16) / 6) < 1e-12                            # K = 6 for complex128, Grover
    rng = np.random.default_rng(0)
    w = qi.Workload("x", 2, (4, 4), 1, qi.PERIODIC, np.dtype(np.complex128), 1, qi.COIN_UNIFORM, qi.random_unitary(rng, 4))
    assert bench.coin_cost(w, "fused") == (64, 120)


def test_alu_peak_is_lanes_times_clock():
    assert bench.alu_peak(qi.k1(sites=64, steps=1), 1965.0) == 148 * 64 * 1.965e9
    assert bench.alu_peak(qi.k1(sites=64, steps=1, dtype=np.complex64), 1965.0) == 148 * 128 * 1.965e9


def test_paper_table_context_workloads():
    t1 = bench.make_workload("t1")
    assert t1.extents == (10001,) and t1.steps == 10000 and t1.boundary == qi.OPEN and t1.delta_site == (5000,)
    t2 = bench.make_workload("t2")
    assert t2.extents == (1001, 1001) and t2.lattice == qi.DIAGONAL and t2.steps == 500
    assert np.array_equal(t2.coin, qi.dft4(np.complex128))
    cfg = bench.workload_config("t2", t2)
    assert "DIAGONAL" in cfg["workload"] and cfg["baseline_config"] is None
    assert bench.workload_config("k1", qi.k1(sites=64, steps=3))["baseline_config"] == 1


def test_gpus_n_outside_torchrun_starts_its_own_ranks():
    """`python bench.py --gpus 2` with no WORLD_SIZE in the environment re-executes itself under torch.distributed.run with
    two ranks (it used to time one replica and print n_gpus 1).  Checked with the reference arm, which needs
    no GPU: rank 0 prints the one JSON line, rank 1 exits 0 without work."""
    import json
    import os
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    env = {k: v for k, v in os.environ.items() if k not in ("WORLD_SIZE", "RANK", "LOCAL_RANK")}
    r = subprocess.run([sys.executable, os.path.join(root, "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "1",
                        "--warmup", "0", "--workload", "k0"], capture_output=True, text=True, timeout=600, env=env, cwd=root)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [ln for ln in r.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["n_gpus"] == 2 and d["value"] > 0
