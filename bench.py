#!/usr/bin/env python
"""bench.py — site-updates/s of the quantum-walk hot path on B200 (BASELINE.json:metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload k1|k1c64|k2|k3hxh|k3dft|k4]
    python -m torch.distributed.run --nproc-per-node N ... bench.py --gpus N ...
    python bench.py --impl reference ...          # the CPU oracle, as it stands, on the host cores

One bench "step" is one pass of the whole hot path over the resident workload: qw_step(walk_steps)
(coin + conditional shift, eq. 2) followed by the workload's outputs (qw_moments and/or
qw_probabilities).  The default workload is BASELINE.json:configs[1] (K1: 1D Hadamard
ring of 2^26 sites, complex128, 1000 walk steps, norm/mean/variance) — the configuration the
metric is quoted on; the other configs are reachable with --workload (parity-tested in tests/).
The state (2 x 2 GiB ping-pong) is far larger than the 126 MB L2, so no explicit L2 flush is needed.

Multi-GPU: the north_star forbids sharding ("no sharding across GPUs, no collectives"), so
--gpus N runs N independent replicas; value is the
aggregate over replicas and the time is the max over ranks.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_1003_3779_b200 import inputs as qi  # noqa: E402

METRIC = "site-updates/s"
FALLBACK_HBM_GBS = 6650.0    # /opt/skills/guides/B200_PROFILING.md fallback


# ----------------------------------------------------------------------------------------------
def make_workload(name: str, walk_steps=None):
    if name == "k1":
        return qi.k1(steps=walk_steps or 1000)
    if name == "k1c64":
        return qi.k1(steps=walk_steps or 1000, dtype=np.complex64)
    if name == "k2":
        return qi.k2(steps=walk_steps)
    if name == "k3hxh":
        return qi.k3(steps=walk_steps or 500, coin="hxh")
    if name == "k3dft":
        return qi.k3(steps=walk_steps or 500, coin="dft")
    if name == "k4":
        return qi.k4(steps=walk_steps)
    if name == "k0":
        return qi.k0(steps=walk_steps or 100)
    if name == "dis":
        # coin families on a long lattice (SURVEY.md 8(a) A8 beyond the resident kernel; eq. 1): 4 rings of
        # 2^24 sites, each with its own SU(2) coin and per-site phase disorder (BASELINE.json:configs[4]'s family)
        n, batch = 1 << 24, 4
        rng = np.random.default_rng(qi.SEED_K4)
        ang = rng.uniform(0.0, 2 * np.pi, (batch, 3))
        phi = rng.uniform(0.0, 2 * np.pi, (batch, n))
        return qi.Workload("DIS", 1, (n,), batch, qi.PERIODIC, np.dtype(np.complex128), walk_steps or 192, qi.COIN_PER_WALK,
                           qi.su2(ang[:, 0], ang[:, 1], ang[:, 2]), phases=np.exp(1j * phi),
                           state=qi.random_state(qi.SEED_K4 + 1, batch, n, 2, np.complex128, normalise_per_walk=True),
                           outputs=("moments",))
    if name == "seg":
        # NEXT-3: the paper's Fig. 3-left "segment": an open 1D Hadamard segment with
        # the delta start of K0, run for five times its length so that the front reflects off the walls (A3, PAPER.md:94-101
        # with RBL = 0) about ten times.  Parity-tested at full length (tests/test_parity_gpu.py::test_segment_workload).
        w = qi.k0(steps=walk_steps or 10000, half_width=1000)
        w.name = "SEG"
        return w
    if name == "t1":
        # context only: the largest row of the paper's Table 1 (1D segment of size 10000).  The paper
        # does not state the number of iterations; iterations = size is SURVEY.md section 6's conjecture.
        w = qi.k0(steps=walk_steps or 10000)
        w.name, w.extents, w.delta_site = "T1", (10001,), (5000,)
        return w
    if name == "t2":
        # context only: the largest row of the paper's Table 2 (2D DIAGONAL lattice, size 500), Fourier
        # coin ("Fourier walker"); iterations = size is a conjecture, the precision is not stated
        w = qi.k2(half=500, steps=walk_steps or 500)
        w.name, w.lattice, w.coin = "T2", qi.DIAGONAL, qi.dft4(np.complex128)
        return w
    raise SystemExit("unknown workload %r" % name)


def workload_config(name, w, extra=None):
    cfg = {
        "workload": "%s: %dD %s lattice %s, batch %d, %s, coin %s, %d walk steps per bench step, outputs %s"
                    % (w.name, w.dim, ("periodic" if w.boundary == qi.PERIODIC else "open") + (" DIAGONAL" if w.lattice == qi.DIAGONAL else ""),
                       "x".join(str(e) for e in w.extents), w.batch, np.dtype(w.dtype).name,
                       {0: "uniform", 1: "per-walk", 2: "per-site"}[w.coin_mode] + ("+site-phases" if w.phases is not None else ""),
                       w.steps, "+".join(w.outputs)),
        "baseline_config": {"k0": 0, "k1": 1, "k1c64": 1, "k2": 2, "k3hxh": 3, "k3dft": 3, "k4": 4}.get(name),
        "sites": w.sites, "batch": w.batch, "walk_steps": w.steps,
        "l2": "working set (2 ping-pong state buffers) exceeds the 126 MB L2; no flush needed"
              if 2 * w.sites * w.batch * w.coin_dim * np.dtype(w.dtype).itemsize > 2 * 126e6 else
              "state fits in L2/SM: resident workload, HBM is touched only at the ends",
        "parallelism": "replicas",
    }
    if extra:
        cfg.update(extra)
    return cfg


def coin_cost(w, sched_name="fused", kdepth=0):
    """(instructions, flops) per site-step of the coin arithmetic the named schedule executes for this workload
    (csrc/qw_coin.cuh::apply_coin): mul = 1 flop, fma = 2 flops, add = 1 flop.
    The temporally blocked 1D kernel defers the Hadamard scale: 15 bare butterflies (4 add) + 1 scaled step
    (2 mul + 4 fma) per 16 steps = 4.125 instructions, 4.375 flops per site-step."""
    c = np.asarray(w.coin)
    if w.dim == 1:
        had = w.coin_mode == qi.COIN_UNIFORM and np.all(c.imag == 0) and c[0, 0] == c[0, 1] == c[1, 0] == -c[1, 1]
        if had and sched_name == "blocked":
            return (15 * 4 + 6) / 16.0, (15 * 4 + 10) / 16.0
        instr, flops = (6, 10) if had else (16, 28)
        if w.phases is not None:
            instr, flops = instr + 8, flops + 12
        return instr, flops
    # 2D named coins: scaled evaluation 20 / 16 / 20 instructions; the tiled kernel defers the power-of-two scale:
    # K-1 bare steps (H(x)H, DFT: 16 add; Grover: 6 add + 8 fma) + 1 scaled step per K steps
    K = kdepth if kdepth in (2, 4, 6, 8, 10, 12) else (8 if w.dtype == np.complex64 else 6)
    def tiled(bare_i, bare_f, full_i, full_f):
        if sched_name == "tiled":
            return ((K - 1) * bare_i + full_i) / K, ((K - 1) * bare_f + full_f) / K
        return full_i, full_f
    if w.coin_mode == qi.COIN_UNIFORM and np.all(c.imag == 0) and np.all(np.abs(c) == abs(c[0, 0])):
        if np.array_equal(np.sign(c.real), np.sign(qi.hadamard_x_hadamard().real)):
            return tiled(16, 16, 20, 24)      # scaled: 2 mul + 4 fma + 4 add per real component
    if w.coin_mode == qi.COIN_UNIFORM and np.array_equal(c, qi.grover4(c.dtype)):
        return tiled(14, 22, 16, 24)
    if w.coin_mode == qi.COIN_UNIFORM and np.array_equal(c, qi.dft4(c.dtype)):
        return tiled(16, 16, 20, 24)
    return 64, 120


def alu_peak(w, sm_max_mhz):
    """Plain-ALU peak: 148 SMs x 64 FP64 (128 FP32) FMA lanes x SM clock (B200)."""
    lanes = 64 if w.dtype == np.complex128 else 128
    ghz = (sm_max_mhz or 1965.0) / 1e3
    return 148 * lanes * ghz * 1e9      # instructions/s; x2 for FMA flops


def measured_peak():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(p) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md 6.65 TB/s)"


def stored_traffic(name):
    """DRAM bytes per launch of the dominant kernel from the committed ncu capture, if any."""
    try:
        with open(os.path.join(ROOT, "profiles", "traffic.json")) as f:
            return json.load(f).get(name)
    except Exception:
        return None


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled DURING the timed region."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index = index
        self.proc = None
        self.lines = []

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q, "--format=csv,noheader,nounits", "-lms", "100"],
                stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._pump, daemon=True)
            self.thread.start()
        except Exception:
            self.proc = None

    def _pump(self):
        for line in self.proc.stdout:
            self.lines.append(line.strip())

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        sm, mx, reasons = [], None, set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for ln in self.lines:
            f = [x.strip() for x in ln.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx = float(f[1])
            except ValueError:
                continue
            for nm, val in zip(names, f[3:7]):
                if val.lower().startswith("active"):
                    reasons.add(nm)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": mx, "reasons": sorted(reasons),
                "samples": len(sm)}


# ----------------------------------------------------------------------------------------------
def dist_env():
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    return rank, world, local


def init_dist(backend: str):
    """Initialise torch.distributed from the torchrun environment (127.0.0.1 rendezvous)."""
    import torch.distributed as dist
    rank, world, _ = dist_env()
    if world > 1 and not dist.is_initialized():
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        os.environ.setdefault("MASTER_PORT", "29511")
        dist.init_process_group(backend=backend, rank=rank, world_size=world)
    return rank, world


def barrier(world):
    if world > 1:
        import torch.distributed as dist
        dist.barrier()


def max_over_ranks(value: float, world: int, device=None) -> float:
    """MAX of a per-rank scalar (device time in ms): the job is as slow as its slowest replica."""
    if world <= 1:
        return float(value)
    import torch
    import torch.distributed as dist
    t = torch.tensor([float(value)], dtype=torch.float64, device=device if device is not None else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def sum_over_ranks(value: float, world: int, device=None) -> float:
    if world <= 1:
        return float(value)
    import torch
    import torch.distributed as dist
    t = torch.tensor([float(value)], dtype=torch.float64, device=device if device is not None else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return float(t.item())


def aggregate_rate(units_per_rank: float, ms_per_rank: float, world: int, device=None):
    """Whole-job rate: units all ranks processed / max-over-ranks time."""
    ms = max_over_ranks(ms_per_rank, world, device)
    units = sum_over_ranks(units_per_rank, world, device)
    return units / (ms * 1e-3), ms


# ----------------------------------------------------------------------------------------------
def dataclasses_replace_ring(w, n):
    """The first walk of a ring workload, cut to its first n sites (inputs for the oracle's bounded sample)."""
    import dataclasses
    return dataclasses.replace(w, extents=(n,), batch=1, coin=np.ascontiguousarray(w.coin[:1]),
                               phases=np.ascontiguousarray(w.phases[:1, :n]), state=np.ascontiguousarray(w.state[:1, :n]))


def cpu_model():
    try:
        with open("/proc/cpuinfo") as f:
            for line in f:
                if line.startswith("model name"):
                    return line.split(":", 1)[1].strip()
    except OSError:
        pass
    return "unknown"


class pinned_to_one_core:
    """the oracle is timed on ONE host core (what `taskset -c <core>` does)."""
    def __enter__(self):
        self.old = None
        try:
            self.old = os.sched_getaffinity(0)
            self.core = min(self.old)
            os.sched_setaffinity(0, {self.core})
        except (AttributeError, OSError):
            self.core = None
        return self

    def __exit__(self, *exc):
        if self.old is not None:
            try:
                os.sched_setaffinity(0, self.old)
            except OSError:
                pass


def oracle_sample(name: str, w, seconds_target: float = 15.0):
    """Time the CPU oracle, as it stands, on a bounded sample of workload `name`: the FULL lattice of the config
     for a few walk steps (about `seconds_target` seconds), one thread pinned to one core."""
    import oracle
    oracle.build()
    sw = w
    if name == "k4":
        sw = qi.k4(batch=256, half=1024, steps=1)        # the per-site matrices of all 4096 walks would be 537 MB x 2
        desc = "256 of the 4096 walks, full length of each, %d walk steps"
    elif name == "dis":
        sw = dataclasses_replace_ring(w, 1 << 22)             # per-site matrices of the full workload would be 4 GiB
        desc = "one of the 4 rings cut to 2^22 sites, %d walk steps"
    elif name in ("k0", "seg", "t1"):
        desc = "the whole lattice, %d walk steps"
    else:
        desc = "the FULL lattice of the config, %d walk steps"
    mode, coin = sw.general_coin_f64()
    psi = np.ascontiguousarray(sw.initial_state().astype(np.complex128))
    if sw.state is None:                                     # delta start: spread the walker first (cost is per site anyway)
        psi[:] = 1.0 / np.sqrt(psi.size)
    kw = dict(boundary=sw.boundary, coin_mode=mode, batch=sw.batch, lattice=sw.lattice)
    with pinned_to_one_core() as pin:
        # calibrate: one step, then scale the step count to ~seconds_target
        t0 = time.perf_counter(); oracle.step(sw.extents, coin, psi, 1, **kw); t1 = time.perf_counter() - t0
        steps = int(max(1, min(100000, seconds_target / max(t1, 1e-7))))
        t0 = time.perf_counter(); oracle.step(sw.extents, coin, psi, steps, **kw); dt = time.perf_counter() - t0
        if "probabilities" in sw.outputs:
            oracle.probabilities(sw.extents, psi, batch=sw.batch)
        if "moments" in sw.outputs:
            oracle.moments(sw.extents, psi, batch=sw.batch)
    rate = sw.sites * sw.batch * steps / dt
    return {"value": rate, "unit": METRIC, "cores": 1, "kind": "oracle",
            "sample": (desc % steps) + ", single thread pinned to core %s (sched_setaffinity = taskset -c), g++ -O2 "
                      "-ffp-contract=off (oracle/qw_oracle.cpp)" % pin.core,
            "seconds": dt, "cpu_model": cpu_model(), "host_cores_available": os.cpu_count()}


def run_reference(args):
    """--impl reference: the oracle on the host cores, same metric/config keys (rank 0 only)."""
    rank, world, _ = dist_env()
    if rank != 0:
        return 0
    import oracle
    oracle.build()
    if args.workload in ("k1", "k1c64"):
        dtype = np.complex128 if args.workload == "k1" else np.complex64
        sw = qi.k1(log2_sites=22, steps=4, dtype=dtype)
        sample = "ring cut to 2^22 sites, 4 walk steps per bench step (oracle: double precision, 1 thread)"
        full_sites, full_batch, full_steps = 1 << 26, 1, args.walk_steps or 1000
        wl_name = "K1"
    else:
        sw = {"k2": lambda: qi.k2(half=512, steps=2), "k3hxh": lambda: qi.k3(extent=1024, steps=2, coin="hxh"),
              "k3dft": lambda: qi.k3(extent=1024, steps=2, coin="dft"), "k4": lambda: qi.k4(batch=64, steps=16),
              "k0": lambda: qi.k0(), "seg": lambda: make_workload("seg", 1000), "dis": lambda: qi.k4(batch=64, steps=16),
              "t1": lambda: make_workload("t1", 8), "t2": lambda: make_workload("t2", 8)}[args.workload]()
        sample = "%s cut to %d sites x batch %d, %d walk steps per bench step" % (sw.name, sw.sites, sw.batch, sw.steps)
        full_sites, full_batch, full_steps = sw.sites, sw.batch, sw.steps
        wl_name = sw.name
    mode, coin = sw.general_coin_f64()
    psi = np.ascontiguousarray(sw.initial_state().astype(np.complex128))
    kw = dict(boundary=sw.boundary, coin_mode=mode, batch=sw.batch, lattice=sw.lattice)

    def one():
        oracle.step(sw.extents, coin, psi, sw.steps, **kw)
        if "moments" in sw.outputs:
            oracle.moments(sw.extents, psi, batch=sw.batch)
        if "probabilities" in sw.outputs:
            oracle.probabilities(sw.extents, psi, batch=sw.batch)

    if args.steps is None:
        args.steps = 3
    with pinned_to_one_core() as pin:
        for _ in range(args.warmup):
            one()
        t0 = time.perf_counter()
        for _ in range(args.steps):
            one()
        dt = time.perf_counter() - t0
    rate = sw.sites * sw.batch * sw.steps * args.steps / dt
    line = {
        "impl": "reference", "metric": METRIC, "value": rate, "unit": METRIC, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": dt * 1e3 / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": "%s (BASELINE.json configs[%d]); reference arm = CPU oracle on a bounded sample: %s"
                               % (wl_name, {"k0": 0, "k1": 1, "k1c64": 1, "k2": 2, "k3hxh": 3, "k3dft": 3, "k4": 4}.get(args.workload, -1), sample),
                   "sites": full_sites, "batch": full_batch, "walk_steps": full_steps, "parallelism": "replicas"},
        "cpu_baseline": {"value": rate, "unit": METRIC, "cores": 1, "kind": "oracle", "cpu_model": cpu_model(),
                         "sample": sample + "; one thread pinned to core %s" % pin.core},
        "e2e": {"value": rate, "unit": METRIC, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))
    return 0


# ----------------------------------------------------------------------------------------------
def run_gpu(args):
    import torch
    from paper_1003_3779_b200 import binding as qw

    rank, world, local = dist_env()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: libqw has no CPU fallback (use --impl reference for the oracle)")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    init_dist("nccl")
    qw.load()

    w = make_workload(args.workload, args.walk_steps)
    if args.coin == "su2":
        if w.dim != 1 or w.coin_mode != qi.COIN_UNIFORM:
            raise SystemExit("--coin su2 needs a 1D workload with a uniform coin")
        w.coin = qi.su2(0.7, 1.1, 2.3).astype(w.dtype)      # a general 2x2 coin: 16 FP instructions per site-step
        w.name += "-su2"
    if args.lattice == "diagonal":
        if w.dim != 2:
            raise SystemExit("--lattice diagonal needs a 2D workload")
        w.lattice = qi.DIAGONAL                       # PAPER.md:106 Fig. 1c: the lattice of the paper's Tables 2-3
    real = np.float64 if w.dtype == np.complex128 else np.float32
    ebytes = np.dtype(w.dtype).itemsize
    site_updates_per_step = float(w.sites) * w.batch * w.steps
    # read + write every amplitude once (+ the site's phase where the coin family has one)
    alg_bytes_per_site = 2 * w.coin_dim * ebytes + (ebytes if w.phases is not None else 0)

    h = qw.create_for(w)
    if args.schedule is not None:
        qw.qw_set_schedule(h, {"auto": 0, "generic": 1, "fused": 2, "blocked": 3, "resident": 4, "tiled": 5}[args.schedule], args.k)
    for kv in args.opt:
        key, value = kv.split("=")
        qw.qw_set_option(h, int(key), int(value))
    if args.no_window:
        qw.qw_set_window(h, 0)
    if args.rbl is not None:
        # NEXT-2: every link redrawn broken with probability p at every step (eqs. 9-10)
        qw.qw_set_random_broken_links(h, 1, args.rbl, qi.SEED_RBL)
    stream = torch.cuda.current_stream()
    qw.qw_set_stream(h, stream.cuda_stream)

    # outputs on the device; host-pinned copies for the end-to-end leg
    mom_d = torch.empty((w.batch, 3 if w.dim == 1 else 6), dtype=torch.float64, device=dev)
    P_d = torch.empty((w.batch, w.sites), dtype=torch.float64 if real == np.float64 else torch.float32, device=dev) \
        if "probabilities" in w.outputs else None

    def outputs_device():
        if "moments" in w.outputs:
            qw.qw_moments(h, mom_d)
        if P_d is not None:
            qw.qw_probabilities(h, P_d)

    # ---- device-resident leg ------------------------------------------------------------------
    # Random-state workloads (K1, K3) keep evolving the resident state; delta-start workloads (K0, K2,
    # K4) restart from the delta every bench step (a device-side memset + one tiny kernel) so that
    # every bench step IS the config: the walker starts at the centre and never reaches the boundary.
    delta = w.state is None
    delta_coin = np.ascontiguousarray(w.delta_coin, dtype=w.dtype) if delta else None

    def hot_path():
        if delta:
            qw.qw_set_state_delta(h, w.delta_site, delta_coin)
        qw.qw_step(h, w.steps)

    # measured plain-ALU peak of this device (register-only DADD / DFMA / FADD2 / FFMA2 chains on every SM,
    # csrc/qw_peak.cu): the denominator of the roofline of the schedules that are not HBM-bound
    dcode = qw.dtype_code(w.dtype)
    alu_measured = {"add": qw.qw_measure_alu_peak(dcode, qw.QW_PEAK_ADD), "fma": qw.qw_measure_alu_peak(dcode, qw.QW_PEAK_FMA)}

    qw.load_state(h, w)
    for _ in range(max(args.warmup, 3)):
        hot_path()
        outputs_device()
    torch.cuda.synchronize()
    if args.steps is None:
        # as many bench steps as make the timed region last about 2 s (>= 10 clock samples at 100 ms), at least 3
        ca = torch.cuda.Event(enable_timing=True); cb = torch.cuda.Event(enable_timing=True)
        ca.record(stream); hot_path(); outputs_device(); cb.record(stream)
        torch.cuda.synchronize()
        one_ms = max_over_ranks(ca.elapsed_time(cb), world, dev)
        args.steps = int(max(3, min(100000, np.ceil(2000.0 / max(one_ms, 1e-3)))))
    barrier(world)
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    ev = [[torch.cuda.Event(enable_timing=True) for _ in range(3)] for _ in range(args.steps)]
    l0 = qw.qw_get_info(h, qw.QW_INFO_LAUNCHES)
    touched0 = qw.qw_get_info(h, qw.QW_INFO_SITES_TOUCHED)
    torch.cuda.synchronize()
    for i in range(args.steps):
        ev[i][0].record(stream)
        hot_path()
        ev[i][1].record(stream)
        outputs_device()
        ev[i][2].record(stream)
    torch.cuda.synchronize()
    barrier(world)
    clocks = sampler.stop() if rank == 0 else None
    launches = qw.qw_get_info(h, qw.QW_INFO_LAUNCHES) - l0
    touched_per_step = (qw.qw_get_info(h, qw.QW_INFO_SITES_TOUCHED) - touched0) / float(args.steps)
    total_ms = ev[0][0].elapsed_time(ev[-1][2])
    step_ms = sum(e[0].elapsed_time(e[1]) for e in ev)
    out_ms = sum(e[1].elapsed_time(e[2]) for e in ev)
    sched = qw.qw_get_info(h, qw.QW_INFO_LAST_SCHEDULE)
    kdepth = qw.qw_get_info(h, qw.QW_INFO_LAST_K)
    windowed = qw.qw_get_info(h, qw.QW_INFO_WINDOW)
    value, ms = aggregate_rate(site_updates_per_step * args.steps, total_ms, world, dev)
    qw.qw_moments(h, mom_d)
    mom_host = mom_d.cpu().numpy()

    # ---- end-to-end leg: host buffers, H2D + D2H inside the timed region -----------------------
    e2e = None
    if not args.no_e2e:
        init = w.initial_state()
        st_pin = torch.from_numpy(init).pin_memory()
        mom_pin = torch.empty((w.batch, mom_d.shape[1]), dtype=torch.float64).pin_memory()
        P_pin = torch.empty((w.batch, w.sites), dtype=P_d.dtype).pin_memory() if P_d is not None else None
        h2d = st_pin.numel() * st_pin.element_size()
        d2h = (mom_pin.numel() * 8 if "moments" in w.outputs else 0) + (P_pin.numel() * P_pin.element_size() if P_pin is not None else 0)

        def e2e_step():
            qw.qw_set_state(h, st_pin)                    # H2D copy + layout kernel (general state: no window)
            qw.qw_step(h, w.steps)
            if "moments" in w.outputs:
                qw.qw_moments(h, mom_pin)                 # D2H, synchronises
            if P_pin is not None:
                qw.qw_probabilities(h, P_pin)

        e2e_step()
        torch.cuda.synchronize(); barrier(world)
        n_e2e = max(1, min(args.steps, 3 if h2d > (1 << 28) else 50))
        t0 = time.perf_counter()
        a = torch.cuda.Event(enable_timing=True); b = torch.cuda.Event(enable_timing=True)
        a.record(stream)
        for _ in range(n_e2e):
            e2e_step()
        b.record(stream)
        torch.cuda.synchronize()
        wall_ms = (time.perf_counter() - t0) * 1e3
        e2e_ms = max(a.elapsed_time(b), wall_ms)          # host-synchronous pieces count too
        barrier(world)
        e_val, e_ms = aggregate_rate(site_updates_per_step * n_e2e, e2e_ms, world, dev)
        e2e = {"value": e_val, "unit": METRIC, "h2d_bytes_per_step": int(h2d), "d2h_bytes_per_step": int(d2h),
               "ms_per_step": e_ms / n_e2e, "steps": n_e2e, "api": "qw_set_state(host) + qw_step + qw_moments/qw_probabilities(host)"}
    # ---- single-step leg: the fused coin+shift kernel alone (HBM roofline evidence) -----------
    fused = None
    if sched != qw.QW_SCHED_FUSED and not args.no_fused_leg:
        nf = min(w.steps, 100)
        qw.qw_set_schedule(h, qw.QW_SCHED_FUSED, 0)
        qw.qw_set_window(h, 0)
        if delta:   # leave the delta neighbourhood: a spread-out state, full-lattice launches
            qw.qw_set_state_delta(h, w.delta_site, delta_coin)
        qw.qw_step(h, 3)
        torch.cuda.synchronize(); barrier(world)
        fa = torch.cuda.Event(enable_timing=True); fb = torch.cuda.Event(enable_timing=True)
        fa.record(stream)
        qw.qw_step(h, nf)
        fb.record(stream)
        torch.cuda.synchronize()
        fms = max_over_ranks(fa.elapsed_time(fb), world, dev)
        fused = {"walk_steps": nf, "avg_launch_ms": fms / nf,
                 "site_updates_per_s": float(w.sites) * w.batch * nf / (fms * 1e-3)}
    qw.qw_destroy(h)

    if rank != 0:
        return 0
    peak, peak_src = measured_peak()
    kernel_ms = step_ms / args.steps            # device time of the hot path per bench step, gaps included
    eff_gbs = site_updates_per_step * alg_bytes_per_site / (kernel_ms * 1e-3) / 1e9
    sched_name = {0: "auto", 1: "generic", 2: "fused", 3: "blocked", 4: "resident", 5: "tiled"}.get(sched, str(sched))
    kname = {1: "step_scatter_kernel (generic)", 2: "step_scatter_kernel (fused coin+shift)",
             3: "step_blocked1d_kernel" if w.dim == 1 else "step_blocked2d_kernel", 4: "step_resident1d_kernel",
             5: "step_stream2d_kernel" if (w.lattice == qi.NATURAL and "2=1" not in args.opt) else "step_tiled2d_kernel"}.get(sched, "?")
    touched_frac = touched_per_step / site_updates_per_step          # < 1 when the light-cone window skipped work
    if sched in (1, 2):
        touched_gbs = eff_gbs * touched_frac
        roofline = {
            "bound": "hbm", "kernel": kname, "achieved": touched_gbs, "peak": peak, "unit": "GB/s", "frac": touched_gbs / peak,
            "peak_source": "of " + peak_src, "frac_of_nominal_8000": touched_gbs / 8000.0,
            "effective_achieved": eff_gbs, "effective_frac": eff_gbs / peak,
            "algorithmic_bytes_per_site_step": alg_bytes_per_site,
            "avg_launch_ms": step_ms / (w.steps * args.steps),
            "traffic": stored_traffic(args.workload),
            "note": "achieved = 2*coin_dim*sizeof(complex) B x site-updates the kernels produced (QW_INFO_SITES_TOUCHED) / CUDA-event "
                    "time of qw_step (launch gaps included); effective_* counts the FULL lattice (BASELINE.json:metric)",
        }
    else:
        instr, flops = coin_cost(w, sched_name, kdepth)
        ipeak_derived = alu_peak(w, clocks["sm_max_mhz"] if clocks else None)
        ipeak = alu_measured["add"] if alu_measured["add"] > 0 else ipeak_derived
        rate = site_updates_per_step / (kernel_ms * 1e-3)         # full lattice (the metric)
        rate_touched = rate * touched_frac                        # what the kernels computed
        fpi = flops / instr                      # flops per instruction of this kernel's op mix (add/mul 1, fma 2)
        roofline = {
            "bound": "alu", "kernel": kname, "achieved": rate_touched * flops / 1e12, "peak": ipeak * fpi / 1e12, "unit": "TFLOP/s",
            "frac": rate_touched * instr / ipeak,
            "effective_frac": rate * instr / ipeak,
            "peak_source": "measured: qw_measure_alu_peak (csrc/qw_peak.cu), independent %s chains on all SMs = %.4g thread-level "
                           "instructions/s (%s: %.4g), x %.3f flops per instruction of this kernel's arithmetic (add/mul = 1, fma = 2)"
                           % ("DADD" if w.dtype == np.complex128 else "FADD2", alu_measured["add"],
                              "DFMA" if w.dtype == np.complex128 else "FFMA2", alu_measured["fma"], fpi),
            "peak_derived": ipeak_derived * fpi / 1e12, "frac_of_derived_peak": rate_touched * instr / ipeak_derived,
            "peak_derived_source": "148 SMs x %d %s lanes x sm_max_mhz (B200_PROFILING.md / B300_MICROARCH.md unit counts)"
                                   % (64 if w.dtype == np.complex128 else 128, "FP64" if w.dtype == np.complex128 else "FP32"),
            "frac_of_fma_peak": rate_touched * flops / (2 * alu_measured["fma"]) if alu_measured["fma"] > 0 else None,
            "fma_peak": 2 * alu_measured["fma"] / 1e12,
            "algorithmic_flops_per_site_step": flops, "algorithmic_instr_per_site_step": instr,
            "touched_site_updates_per_bench_step": touched_per_step, "touched_fraction_of_full_lattice": touched_frac,
            "traffic": stored_traffic(args.workload + "_" + sched_name),
            "effective_hbm_gbs_vs_single_step": eff_gbs, "single_step_hbm_roofline_x": eff_gbs / peak,
            "note": "temporal blocking / SM residency removes the HBM bound; frac counts the FP instructions of the site-updates the "
                    "kernels produced (halo / starter recomputation excluded; with the light-cone window only the tiles and warps "
                    "that were not skipped), effective_frac counts the full lattice (BASELINE.json:metric)",
        }
        if kname == "step_stream2d_kernel" and args.rbl is None and kdepth >= 2:
            # The streaming 2D kernel reads and writes every amplitude once per launch of k steps, and at its default depth that
            # is what binds it (ncu: DRAM 83 % of the measured copy peak, FP pipe 52 %; profiles/r02_stream2d.md).  So the
            # roofline of this kernel is HBM: algorithmic bytes per launch = 2*coin_dim*sizeof(complex) B x the sites it
            # produced, per launch duration; the instruction-slot figures stay beside it.
            alu = roofline
            launch_bytes_per_site = alg_bytes_per_site            # one read + one write of the lattice per launch
            gbs = rate_touched * launch_bytes_per_site / kdepth / 1e9
            roofline = {
                "bound": "hbm", "kernel": kname, "achieved": gbs, "peak": peak, "unit": "GB/s", "frac": gbs / peak,
                "peak_source": "of " + peak_src, "frac_of_nominal_8000": gbs / 8000.0,
                "effective_frac": rate * launch_bytes_per_site / kdepth / 1e9 / peak,
                "algorithmic_bytes_per_site_per_launch": launch_bytes_per_site, "steps_per_launch": kdepth,
                "algorithmic_bytes_per_site_step": launch_bytes_per_site / kdepth,
                "touched_site_updates_per_bench_step": touched_per_step, "touched_fraction_of_full_lattice": touched_frac,
                "traffic": stored_traffic(args.workload + "_" + sched_name),
                "alu_frac": alu["frac"], "alu_effective_frac": alu["effective_frac"], "alu_peak_tflops": alu["peak"],
                "alu_peak_source": alu["peak_source"], "algorithmic_instr_per_site_step": instr,
                "algorithmic_flops_per_site_step": flops,
                "effective_hbm_gbs_vs_single_step": eff_gbs, "single_step_hbm_roofline_x": eff_gbs / peak,
                "note": "k walk steps per HBM round trip: achieved = algorithmic bytes per launch (2*coin_dim*sizeof(complex) B per "
                        "site the kernel produced) / launch duration (CUDA events over qw_step, remainder launches and gaps "
                        "included); alu_frac = FP instructions of the produced site-updates / measured instruction-slot peak; "
                        "effective_* count the full lattice (BASELINE.json:metric)",
            }
    if args.rbl is not None and roofline.get("bound") == "alu":
        roofline["note"] += ("; with --rbl the temporally blocked kernels are bound by the INTEGER instructions of the in-kernel link "
                             "draws (one Philox4x32-10 call per four links, ~64 integer instructions), which frac does not count: "
                             "profiles/r02_stream2d.md section 3, r02_chain1d.md")
    if fused is not None:
        fg = fused["site_updates_per_s"] * alg_bytes_per_site / 1e9
        fused.update({"bound": "hbm", "kernel": "step_scatter_kernel (fused coin+shift)", "achieved": fg, "peak": peak,
                      "unit": "GB/s", "frac": fg / peak, "frac_of_nominal_8000": fg / 8000.0,
                      "traffic": stored_traffic(args.workload)})
    line = {
        "metric": METRIC, "value": value, "unit": METRIC, "n_gpus": world, "steps": args.steps,
        "warmup": max(args.warmup, 3), "ms_per_step": ms / args.steps, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64" if w.dtype == np.complex128 else "f32",
        "data": "synthetic",
        "config": workload_config(args.workload, w, {"schedule": sched_name, "k": kdepth, "window": bool(windowed),
                                                     "step_ms": step_ms / args.steps, "outputs_ms": out_ms / args.steps,
                                                     **({"random_broken_links_p": args.rbl} if args.rbl is not None else {})}),
        "effective_hbm_gbs": eff_gbs,
        "roofline": roofline,
        "fused_single_step": fused,
        "clocks": clocks,
        "alu_peak_measured": {"add_ops_per_s": alu_measured["add"], "fma_ops_per_s": alu_measured["fma"],
                              "how": "qw_measure_alu_peak: register-only chains, 8 CTAs x 256 threads per SM, best of 4"},
        "gpu_launches": int(launches),
        "e2e": e2e,
        "result": {"norm": float(mom_host[0, 0]), "mean": float(mom_host[0, 1]), "var": float(mom_host[0, -1] if w.dim == 1 else mom_host[0, 3])},
    }
    if clocks is not None and (clocks.get("samples") or 0) < 3:
        # a timed region shorter than a few sampler periods has no clock record: not a result (use more --steps)
        line["invalid"] = "only %d clock samples during the timed region (%.0f ms): rerun with more --steps" % (
            clocks.get("samples") or 0, ms)
    if not args.no_cpu_baseline and world == 1:
        line["cpu_baseline"] = oracle_sample(args.workload, w)
    elif world > 1:
        line["cpu_baseline"] = None
    print(json.dumps(line))
    return 0


def spawn_ranks(args):
    """`python bench.py --gpus N` outside torchrun: start the N ranks ourselves (one process per GPU) with the very
    command line the driver uses, and hand its exit code back.  Rank 0 of the child job prints the JSON line."""
    port = 29500 + os.getpid() % 2000
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(args.gpus),
           "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
    return subprocess.call(cmd)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=None,
                    help="timed bench steps (default: as many as make the timed region last about 2 s, at least 3)")
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="k1", choices=["k0", "k1", "k1c64", "k2", "k3hxh", "k3dft", "k4", "seg", "dis", "t1", "t2"])
    ap.add_argument("--walk-steps", type=int, default=None, help="walk steps per bench step (default: the config's)")
    ap.add_argument("--schedule", default=None, choices=["auto", "generic", "fused", "blocked", "resident", "tiled"])
    ap.add_argument("--k", type=int, default=0)
    ap.add_argument("--no-window", action="store_true")
    ap.add_argument("--lattice", default=None, choices=["natural", "diagonal"], help="override the 2D lattice kind")
    ap.add_argument("--coin", default=None, choices=["su2"], help="k1 / k1c64 only: a general SU(2) coin instead of Hadamard")
    ap.add_argument("--rbl", type=float, default=None, help="random broken links redrawn every step with this probability")
    ap.add_argument("--opt", action="append", default=[], metavar="KEY=VALUE",
                    help="qw_set_option(key, value) by number, e.g. --opt 1=1 forces the halo kernel of the blocked 1D schedule")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-fused-leg", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    args = ap.parse_args()
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        return spawn_ranks(args)
    if args.gpus != int(os.environ.get("WORLD_SIZE", "1")):
        raise SystemExit("--gpus %d does not match WORLD_SIZE=%s" % (args.gpus, os.environ.get("WORLD_SIZE")))
    if args.impl == "reference":
        return run_reference(args)
    return run_gpu(args)


if __name__ == "__main__":
    sys.exit(main())
