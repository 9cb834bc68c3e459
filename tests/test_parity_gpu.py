"""GPU parity: libqw (through the C ABI, via the ctypes binding) against the CPU oracle, element by
element on the same seeded inputs.  Gates (BASELINE.json:north_star):
    complex128   max |d amplitude| <= 1e-12, |d probability| <= 1e-12 per site
    complex64    max |d amplitude| <= 2e-5, |1 - norm| <= 1e-4 after the full step count
    moments      complex128 relative 1e-10; complex64 relative 1e-4          (R24)
The oracle always runs in double on exactly the bytes the library received (for complex64: the
float-rounded state and coin promoted to double, R21).
"""
import numpy as np
import pytest

from paper_1003_3779_b200 import inputs as qi

pytestmark = pytest.mark.gpu

AMP_TOL = {np.dtype(np.complex128): 1e-12, np.dtype(np.complex64): 2e-5}
MOM_RTOL = {np.dtype(np.complex128): 1e-10, np.dtype(np.complex64): 1e-4}


@pytest.fixture(scope="module")
def dev(qw):
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    torch.cuda.init()
    return torch.device("cuda:0")


def real_dtype(w):
    return np.float64 if w.dtype == np.complex128 else np.float32


def gpu_run(qw, w, steps=None, schedule=None, k=0, window=True, inverse=0, broken=None, get_state=True, options=None):
    """Run workload w on the GPU; returns (amps AoS in w.dtype, P, moments, info)."""
    steps = w.steps if steps is None else steps
    h = qw.create_for(w)
    try:
        for key, value in (options or {}).items():
            qw.qw_set_option(h, key, value)
        if broken is not None:
            qw.qw_set_broken_links(h, broken)
        if schedule is not None:
            qw.qw_set_schedule(h, schedule, k)
        qw.qw_set_window(h, window)
        qw.load_state(h, w)
        qw.qw_step(h, steps)
        if inverse:
            qw.qw_step_inverse(h, inverse)
        amps = None
        if get_state:
            amps = np.empty((w.batch, w.sites, w.coin_dim), dtype=w.dtype)
            qw.qw_get_state(h, amps)
        P = np.empty((w.batch, w.sites), dtype=real_dtype(w))
        qw.qw_probabilities(h, P)
        mom = np.empty((w.batch, 3 if w.dim == 1 else 6), dtype=np.float64)
        qw.qw_moments(h, mom)
        info = {"launches": qw.qw_get_info(h, qw.QW_INFO_LAUNCHES), "sched": qw.qw_get_info(h, qw.QW_INFO_LAST_SCHEDULE),
                "k": qw.qw_get_info(h, qw.QW_INFO_LAST_K), "t": qw.qw_get_info(h, qw.QW_INFO_TIME)}
        return amps, P, mom, info
    finally:
        qw.qw_destroy(h)


def oracle_run(oracle, w, steps=None, inverse=0, broken=None):
    steps = w.steps if steps is None else steps
    mode, coin = w.general_coin_f64()
    psi = np.ascontiguousarray(w.initial_state().astype(np.complex128))
    kw = dict(boundary=w.boundary, coin_mode=mode, batch=w.batch, lattice=w.lattice, broken=broken)
    oracle.step(w.extents, coin, psi, steps, **kw)
    if inverse:
        oracle.step_inverse(w.extents, coin, psi, inverse, **kw)
    return psi, oracle.probabilities(w.extents, psi, batch=w.batch), oracle.moments(w.extents, psi, batch=w.batch)


def check_parity(w, gpu, ora, mom_abs_mean=None):
    amps, P, mom, _ = gpu
    psi, Po, momo = ora
    tol = AMP_TOL[np.dtype(w.dtype)]
    if amps is not None:
        d = np.max(np.abs(amps.astype(np.complex128) - psi)) if psi.size else 0.0
        assert d <= tol, "max |d amplitude| = %.3e > %.1e" % (d, tol)
    ptol = 1e-12 if w.dtype == np.complex128 else 4 * w.coin_dim * tol
    dP = np.max(np.abs(P.astype(np.float64) - Po)) if Po.size else 0.0
    assert dP <= ptol, "max |d probability| = %.3e" % dP
    rt = MOM_RTOL[np.dtype(w.dtype)]
    ext = max(w.extents)
    nm = 1 if w.dim == 1 else 2
    for b in range(w.batch):
        assert abs(mom[b, 0] - momo[b, 0]) <= rt * abs(momo[b, 0]), ("norm", mom[b, 0], momo[b, 0])
        for j in range(1, 1 + nm):                                   # means: absolute rt*extent where mean ~ 0
            assert abs(mom[b, j] - momo[b, j]) <= rt * (abs(momo[b, j]) + ext), ("mean", mom[b], momo[b])
        second = 1.0 + max(abs(momo[b, j]) for j in range(1 + nm, mom.shape[1])) + max(momo[b, j] ** 2 for j in range(1, 1 + nm))
        for j in range(1 + nm, mom.shape[1]):                        # variances / covariance: relative to E[x^2]
            assert abs(mom[b, j] - momo[b, j]) <= rt * second, ("second moment", j, mom[b], momo[b])
    if w.dtype == np.complex64:
        assert np.max(np.abs(1 - mom[:, 0])) <= 1e-4


# ------------------------------------------------------------------ the five configs, scaled twins
def test_k0_exact_config(qw, oracle, dev):
    w = qi.k0()
    gpu = gpu_run(qw, w)
    check_parity(w, gpu, oracle_run(oracle, w))
    P = gpu[1][0]
    assert np.max(np.abs(P - P[::-1])) <= 1e-15                      # P5 symmetry on the GPU too
    assert np.all(P[(np.arange(-100, 101) + 100) % 2 == 1] == 0.0)   # P4 exact zeros


@pytest.mark.parametrize("dtype", [np.complex128, np.complex64])
@pytest.mark.parametrize("sites,steps", [(1 << 16, 200), (100003, 64), (1024 * 4 * 3 + 1, 33)])
def test_k1_ring_twins(qw, oracle, dev, dtype, sites, steps):
    w = qi.k1(sites=sites, steps=steps, dtype=dtype)
    check_parity(w, gpu_run(qw, w), oracle_run(oracle, w))


@pytest.mark.parametrize("sites,coin,k", [((1 << 20) + 3, "hadamard", 48), ((1 << 20) + 3, "su2", 16)])
@pytest.mark.parametrize("dtype", [np.complex128, np.complex64])
def test_k1_prime_twin_every_site(qw, oracle, dev, dtype, sites, coin, k):
    """SURVEY.md 8(d) K1' at its stated size: a ring of 2^20 + 3 sites x 200 steps, EVERY site against the oracle,
    through the temporally blocked schedule at an explicit depth and as AUTO picks it.  2^20 sites are more tiles
    than the grid has warps, so the persistent multi-tile loop with its prefetch runs under an element-wise check
    (Hadamard: 512-site tiles, deferred scale; SU(2): 256-site tiles, M = 8)."""
    w = qi.k1(sites=sites, steps=200, dtype=dtype)
    if coin == "su2":
        w.coin = qi.su2(0.7, 1.1, 2.3).astype(dtype)
    ora = oracle_run(oracle, w)
    for schedule, kk in ((qw.QW_SCHED_BLOCKED, k), (qw.QW_SCHED_AUTO, 0)):
        gpu = gpu_run(qw, w, schedule=schedule, k=kk)
        assert gpu[3]["sched"] == qw.QW_SCHED_BLOCKED and gpu[3]["launches"] <= 200 // 8
        check_parity(w, gpu, ora)


@pytest.mark.parametrize("half,steps", [(64, 64), (40, 100)])
def test_k2_grover_twins(qw, oracle, dev, half, steps):
    w = qi.k2(half=half, steps=steps)                                # steps > half: the wall reflects
    gpu = gpu_run(qw, w)
    check_parity(w, gpu, oracle_run(oracle, w))
    if steps <= half:
        # GPU-side mirror symmetry (m -> -m, m <-> n), NOT an oracle gate.  The bound is 1e-15 rather than bit equality
        # because the Grover evaluation g*((v0+v1)+(v2+v3)) + (d-g)*v_a (qw_coin.cuh, DESIGN.md section 2 "Arithmetic
        # choice") adds the four components in a fixed order: mirroring the lattice permutes v0..v3 (c0 <-> c3, c1 <-> c2),
        # so the mirrored site rounds its sum differently by <= 1 ulp per step.  Probabilities here are <= 0.25.
        P = gpu[1][0].reshape(w.extents)
        assert np.max(np.abs(P - P[::-1, :])) < 1e-15 and np.max(np.abs(P - P.T)) < 1e-15


@pytest.mark.parametrize("coin", ["hxh", "dft", "grover"])
@pytest.mark.parametrize("extents,steps", [((256, 256), 50), ((61, 35), 40), ((8, 1030), 25)])
def test_k3_torus_twins(qw, oracle, dev, coin, extents, steps):
    w = qi.k3(extents=extents, steps=steps, coin=coin)
    check_parity(w, gpu_run(qw, w), oracle_run(oracle, w))


@pytest.mark.parametrize("batch,half,steps", [(16, 64, 64), (5, 21, 100), (3, 1024, 40)])
def test_k4_batch_twins(qw, oracle, dev, batch, half, steps):
    w = qi.k4(batch=batch, half=half, steps=steps)
    check_parity(w, gpu_run(qw, w), oracle_run(oracle, w))


# ------------------------------------------------------------------ feature matrix on small lattices
def small_workload(dim, boundary, dtype, coin_mode, rng, lattice=qi.NATURAL, phases=False, batch=2, extents=None):
    ext = extents if extents is not None else ((37,) if dim == 1 else (11, 14))
    sites = int(np.prod(ext))
    cd = 2 * dim
    if coin_mode == qi.COIN_UNIFORM:
        coin = qi.random_unitary(rng, cd)
    elif coin_mode == qi.COIN_PER_WALK:
        coin = np.stack([qi.random_unitary(rng, cd) for _ in range(batch)])
    else:
        coin = np.stack([qi.random_unitary(rng, cd) for _ in range(batch * sites)]).reshape(batch, sites, cd, cd)
    ph = np.exp(1j * rng.uniform(0, 2 * np.pi, (batch, sites))).astype(dtype) if phases else None
    return qi.Workload("small", dim, tuple(ext), batch, boundary, np.dtype(dtype), 30, coin_mode,
                       coin.astype(dtype), phases=ph,
                       state=qi.random_state(77, batch, sites, cd, dtype, normalise_per_walk=True), lattice=lattice)


@pytest.mark.parametrize("dtype", [np.complex128, np.complex64])
@pytest.mark.parametrize("boundary", [qi.OPEN, qi.PERIODIC])
@pytest.mark.parametrize("dim", [1, 2])
@pytest.mark.parametrize("coin_mode,phases", [(qi.COIN_UNIFORM, False), (qi.COIN_UNIFORM, True),
                                              (qi.COIN_PER_WALK, True), (qi.COIN_PER_SITE, False)])
def test_feature_matrix(qw, oracle, dev, dtype, boundary, dim, coin_mode, phases):
    rng = np.random.default_rng(100 + 10 * dim + boundary)
    w = small_workload(dim, boundary, dtype, coin_mode, rng, phases=phases)
    check_parity(w, gpu_run(qw, w), oracle_run(oracle, w))


@pytest.mark.parametrize("boundary", [qi.OPEN, qi.PERIODIC])
@pytest.mark.parametrize("dtype", [np.complex128, np.complex64])
def test_diagonal_lattice(qw, oracle, dev, boundary, dtype):
    rng = np.random.default_rng(5)
    w = small_workload(2, boundary, dtype, qi.COIN_UNIFORM, rng, lattice=qi.DIAGONAL)
    check_parity(w, gpu_run(qw, w), oracle_run(oracle, w))


@pytest.mark.parametrize("boundary", [qi.OPEN, qi.PERIODIC])
@pytest.mark.parametrize("dtype", [np.complex128, np.complex64])
@pytest.mark.parametrize("coin", ["hxh", "dft", "grover"])
def test_diagonal_lattice_fused_path_multi_tile(qw, oracle, dev, boundary, dtype, coin):
    """The lattice of the paper's Tables 2-3 (Fig. 1c :106) through the vectorised fused kernel:
    several CTAs per row with ragged tails, named coins, random state and a delta start whose light-cone window
    reaches the walls; fused == generic bit for bit."""
    w = qi.k3(extents=(37, 1100), steps=21, coin=coin, dtype=dtype)
    w.lattice, w.boundary = qi.DIAGONAL, boundary
    a = gpu_run(qw, w, schedule=qw.QW_SCHED_FUSED)
    g = gpu_run(qw, w, schedule=qw.QW_SCHED_GENERIC)
    assert a[3]["sched"] == qw.QW_SCHED_FUSED and np.array_equal(a[0], g[0])
    assert np.array_equal(a[0], gpu_run(qw, w)[0])                      # AUTO picks a kernel that knows the lattice
    check_parity(w, a, oracle_run(oracle, w))
    d = qi.k2(half=30, steps=45)
    d.lattice, d.boundary = qi.DIAGONAL, boundary
    d.dtype = np.dtype(dtype); d.coin = {"hxh": qi.hadamard_x_hadamard, "dft": qi.dft4, "grover": qi.grover4}[coin](dtype)
    d.delta_coin = d.delta_coin.astype(dtype)
    on = gpu_run(qw, d, window=True)
    off = gpu_run(qw, d, window=False)
    assert np.array_equal(on[0], off[0])
    check_parity(d, on, oracle_run(oracle, d))


@pytest.mark.parametrize("dim,lattice", [(1, qi.NATURAL), (2, qi.NATURAL), (2, qi.DIAGONAL)])
@pytest.mark.parametrize("boundary", [qi.OPEN, qi.PERIODIC])
def test_static_broken_links(qw, oracle, dev, dim, lattice, boundary):
    rng = np.random.default_rng(6)
    w = small_workload(dim, boundary, np.complex128, qi.COIN_UNIFORM, rng, lattice=lattice)
    mask = qi.symmetric_broken_links(qi.SEED_RBL, dim, w.extents, w.batch, 0.25, boundary, lattice)
    gpu = gpu_run(qw, w, broken=mask)
    check_parity(w, gpu, oracle_run(oracle, w, broken=mask))
    assert np.max(np.abs(gpu[2][:, 0] - 1)) < 1e-13                  # still unitary


@pytest.mark.parametrize("extents", [(1,), (2,), (3,), (1, 1), (1, 5), (5, 1), (2, 2), (2, 3)])
@pytest.mark.parametrize("boundary", [qi.OPEN, qi.PERIODIC])
def test_degenerate_extents(qw, oracle, dev, extents, boundary):
    rng = np.random.default_rng(8)
    for dtype in (np.complex128, np.complex64):
        w = small_workload(len(extents), boundary, dtype, qi.COIN_UNIFORM, rng, batch=3, extents=extents)
        check_parity(w, gpu_run(qw, w), oracle_run(oracle, w))


# ------------------------------------------------------------------ inverse step / reversibility (P6)
@pytest.mark.parametrize("dim", [1, 2])
@pytest.mark.parametrize("boundary", [qi.OPEN, qi.PERIODIC])
def test_inverse_step(qw, oracle, dev, dim, boundary):
    rng = np.random.default_rng(9)
    w = small_workload(dim, boundary, np.complex128, qi.COIN_PER_WALK, rng, phases=True)
    check_parity(w, gpu_run(qw, w, steps=7, inverse=3), oracle_run(oracle, w, steps=7, inverse=3))
    amps, _, _, info = gpu_run(qw, w, steps=100, inverse=100)
    assert info["t"] == 0
    assert np.max(np.abs(amps - w.initial_state())) <= 1e-13


# ------------------------------------------------------------------ schedule / window invariance (P13), P12
def test_generic_and_fused_schedules_agree_bit_for_bit(qw, dev):
    for w in (qi.k1(sites=50021, steps=40), qi.k1(sites=50021, steps=40, dtype=np.complex64),
              qi.k3(extents=(97, 130), steps=20, coin="dft"), qi.k3(extents=(97, 130), steps=20, coin="hxh"),
              qi.k2(half=33, steps=50)):
        a = gpu_run(qw, w, schedule=qw.QW_SCHED_GENERIC)
        b = gpu_run(qw, w, schedule=qw.QW_SCHED_FUSED)
        assert a[3]["sched"] == qw.QW_SCHED_GENERIC and b[3]["sched"] == qw.QW_SCHED_FUSED
        assert np.array_equal(a[0], b[0]), w.name


@pytest.mark.parametrize("dtype", [np.complex128, np.complex64])
@pytest.mark.parametrize("boundary", [qi.PERIODIC, qi.OPEN])
@pytest.mark.parametrize("coin", ["hadamard", "su2"])
def test_blocked_1d_schedule_is_bit_identical_to_single_steps(qw, oracle, dev, dtype, boundary, coin, ):
    """P13: k steps per HBM round trip (warp-private register tiles) == k fused single steps, bit for bit
    (general coin) or to <= 4 ulp per step (Hadamard coin, whose scale is applied once per 16 steps);
    sizes span several tiles, a ragged last tile and the periodic seam / the reflecting walls."""
    rng = np.random.default_rng(3)
    for sites, steps, k, batch in ((5000, 96, 32, 1), (1031, 100, 16, 3), (70001, 131, 0, 1), (512, 48, 48, 2)):
        c = qi.hadamard(dtype) if coin == "hadamard" else qi.su2(*rng.uniform(0, 2 * np.pi, 3)).astype(dtype)
        w = qi.Workload("blk", 1, (sites,), batch, boundary, np.dtype(dtype), steps, qi.COIN_UNIFORM, c,
                        state=qi.random_state(9, batch, sites, 2, dtype, normalise_per_walk=True))
        a = gpu_run(qw, w, schedule=qw.QW_SCHED_FUSED)
        b = gpu_run(qw, w, schedule=qw.QW_SCHED_BLOCKED, k=k)
        assert b[3]["sched"] == qw.QW_SCHED_BLOCKED and b[3]["launches"] < a[3]["launches"]
        auto = gpu_run(qw, w)
        if coin == "hadamard":
            # deferred scale: 16 bare butterflies, then one multiplication by s^16 (qw_step_blocked1d.cu) -- equal to
            # 16 scaled single steps up to rounding: <= 4 ulp per step; a wrong halo, seam or
            # wall moves O(|amp|), ten orders above this bound
            eps = np.finfo(np.float64 if dtype == np.complex128 else np.float32).eps
            bound = 4 * eps * steps * float(np.max(np.abs(a[0])))
            assert np.max(np.abs(a[0].astype(np.complex128) - b[0].astype(np.complex128))) <= bound, (sites, steps, k)
            b16 = gpu_run(qw, w, schedule=qw.QW_SCHED_BLOCKED, k=16)
            assert np.array_equal(b[0], b16[0]), "the launch depth k must not change the result"
            assert np.array_equal(b16[0], auto[0]) or auto[3]["sched"] != qw.QW_SCHED_BLOCKED
        else:
            assert np.array_equal(a[0], b[0]), (sites, steps, k)
            assert np.array_equal(a[0], auto[0])
        check_parity(w, b, oracle_run(oracle, w))                     # every configuration, not only the last


@pytest.mark.parametrize("dtype", [np.complex128, np.complex64])
@pytest.mark.parametrize("coin", ["hadamard", "su2"])
def test_chained_blocked_1d_kernel(qw, oracle, dev, dtype, coin):
    """The chained ring kernel (qw_step_chain1d.cu: tiles in the frame moving with the R plane, the L outflow of a tile
    fed to its left neighbour through a FIFO, one redundant starter tile per chain) against the halo kernel (bit for
    bit: same arithmetic per site), the fused single steps and the oracle.  QW_OPT_MAX_CTAS shrinks the persistent
    grid so that small rings give chains of many tiles; sizes: ragged last chain / last tile, a batch, the minimal
    ring of two tiles, chains of one tile, every depth, several launches with a remainder."""
    rng = np.random.default_rng(23)
    M = 16 if coin == "hadamard" else 8
    cases = ((20000, 112, 48, 1, 1), (3001, 64, 16, 3, 2), (70001, 131, 0, 1, 0), (64 * M, 64, 64, 2, 1),
             (100003, 200, 64, 1, 3), (9973, 40, 32, 2, 1), (2048, 48, 16, 20, 1))     # last: 20 chains over 4 warps
    for sites, steps, k, batch, max_ctas in cases:
        c = qi.hadamard(dtype) if coin == "hadamard" else qi.su2(*rng.uniform(0, 2 * np.pi, 3)).astype(dtype)
        w = qi.Workload("chain", 1, (sites,), batch, qi.PERIODIC, np.dtype(dtype), steps, qi.COIN_UNIFORM, c,
                        state=qi.random_state(11, batch, sites, 2, dtype, normalise_per_walk=True))
        opt = {qw.QW_OPT_MAX_CTAS: max_ctas}
        chain = gpu_run(qw, w, schedule=qw.QW_SCHED_BLOCKED, k=k, options={**opt, qw.QW_OPT_BLOCKED1D_KERNEL: 2})
        halo = gpu_run(qw, w, schedule=qw.QW_SCHED_BLOCKED, k=k if k <= 48 else 48, options={**opt, qw.QW_OPT_BLOCKED1D_KERNEL: 1})
        assert chain[3]["sched"] == qw.QW_SCHED_BLOCKED
        assert np.array_equal(chain[0], halo[0]), (sites, steps, k, batch)
        fused = gpu_run(qw, w, schedule=qw.QW_SCHED_FUSED)
        if coin == "hadamard":      # deferred scale: <= 4 ulp per step from the scaled single steps
            eps = np.finfo(np.float64 if dtype == np.complex128 else np.float32).eps
            bound = 4 * eps * steps * float(np.max(np.abs(fused[0])))
            assert np.max(np.abs(fused[0].astype(np.complex128) - chain[0].astype(np.complex128))) <= bound
        else:
            assert np.array_equal(chain[0], fused[0]), (sites, steps, k, batch)
        check_parity(w, chain, oracle_run(oracle, w))


@pytest.mark.parametrize("dtype", [np.complex128, np.complex64])
@pytest.mark.parametrize("boundary", [qi.PERIODIC, qi.OPEN])
def test_resident_1d_schedule_is_bit_identical_to_single_steps(qw, oracle, dev, dtype, boundary):
    """P13: one CTA per walk with the state in registers for all n steps == n fused single steps."""
    rng = np.random.default_rng(4)
    for sites, steps, batch, kind in ((1, 5, 2, "su2"), (2, 7, 2, "had"), (3, 9, 1, "su2"), (37, 100, 3, "had"),
                                      (201, 131, 2, "su2+ph"), (256, 64, 1, "had"), (257, 33, 2, "perwalk+ph"),
                                      (2049, 75, 3, "perwalk+ph"), (4096, 41, 2, "had"), (4095, 18, 1, "perwalk")):
        if kind.startswith("perwalk"):
            a3 = rng.uniform(0, 2 * np.pi, (batch, 3))
            mode, c = qi.COIN_PER_WALK, qi.su2(a3[:, 0], a3[:, 1], a3[:, 2]).astype(dtype)
        elif kind.startswith("su2"):
            mode, c = qi.COIN_UNIFORM, qi.su2(*rng.uniform(0, 2 * np.pi, 3)).astype(dtype)
        else:
            mode, c = qi.COIN_UNIFORM, qi.hadamard(dtype)
        ph = np.exp(1j * rng.uniform(0, 2 * np.pi, (batch, sites))).astype(dtype) if kind.endswith("+ph") else None
        w = qi.Workload("res", 1, (sites,), batch, boundary, np.dtype(dtype), steps, mode, c, phases=ph,
                        state=qi.random_state(19, batch, sites, 2, dtype, normalise_per_walk=True))
        a = gpu_run(qw, w, schedule=qw.QW_SCHED_FUSED)
        b = gpu_run(qw, w, schedule=qw.QW_SCHED_RESIDENT)
        assert b[3]["sched"] == qw.QW_SCHED_RESIDENT and b[3]["launches"] < a[3]["launches"]
        assert np.array_equal(a[0], b[0]), (sites, steps, kind)
        auto = gpu_run(qw, w)
        assert auto[3]["sched"] == qw.QW_SCHED_RESIDENT and np.array_equal(a[0], auto[0])
        check_parity(w, b, oracle_run(oracle, w))


@pytest.mark.parametrize("window", [True, False])
def test_resident_delta_start_with_light_cone(qw, oracle, dev, window):
    for w in (qi.k0(steps=130), qi.k4(batch=6, half=300, steps=450), qi.k4(batch=2, half=1024, steps=1024)):
        a = gpu_run(qw, w, schedule=qw.QW_SCHED_FUSED, window=False)
        b = gpu_run(qw, w, schedule=qw.QW_SCHED_RESIDENT, window=window)
        assert np.array_equal(a[0], b[0]), w.name
        if w.batch <= 2:
            check_parity(w, b, oracle_run(oracle, w))
    # split stepping: two resident launches continue the same cone
    w = qi.k4(batch=3, half=200, steps=150)
    h = qw.create_for(w)
    try:
        qw.qw_set_window(h, window)
        qw.load_state(h, w)
        qw.qw_step(h, 70); qw.qw_step(h, 80)
        got = np.empty((w.batch, w.sites, 2), dtype=w.dtype)
        qw.qw_get_state(h, got)
    finally:
        qw.qw_destroy(h)
    assert np.array_equal(got, gpu_run(qw, w, schedule=qw.QW_SCHED_FUSED, window=False)[0])


@pytest.mark.parametrize("dtype", [np.complex128, np.complex64])
@pytest.mark.parametrize("boundary", [qi.PERIODIC, qi.OPEN])
@pytest.mark.parametrize("coin", ["grover", "hxh", "dft", "random"])
def test_blocked_2d_schedule_is_bit_identical_to_single_steps(qw, oracle, dev, dtype, boundary, coin):
    """P13 in 2D: TMA-staged shared-memory tiles advanced k steps in place == k fused single steps."""
    rng = np.random.default_rng(12)
    for extents, steps, k, batch in (((97, 130), 20, 0, 1), ((64, 64), 9, 3, 2), ((33, 200), 17, 1, 1), ((150, 41), 24, 7, 1)):
        c = {"grover": qi.grover4, "hxh": qi.hadamard_x_hadamard, "dft": qi.dft4}[coin](dtype) if coin != "random" \
            else qi.random_unitary(rng, 4).astype(dtype)
        sites = extents[0] * extents[1]
        w = qi.Workload("blk2d", 2, extents, batch, boundary, np.dtype(dtype), steps, qi.COIN_UNIFORM, c,
                        state=qi.random_state(29, batch, sites, 4, dtype, normalise_per_walk=True))
        a = gpu_run(qw, w, schedule=qw.QW_SCHED_FUSED)
        b = gpu_run(qw, w, schedule=qw.QW_SCHED_BLOCKED, k=k)
        assert b[3]["sched"] == qw.QW_SCHED_BLOCKED
        assert np.array_equal(a[0], b[0]), (extents, steps, k)
    check_parity(w, b, oracle_run(oracle, w))


def test_blocked_2d_delta_start_reaches_the_walls(qw, dev):
    w = qi.k2(half=40, steps=100)
    a = gpu_run(qw, w, schedule=qw.QW_SCHED_FUSED, window=False)
    b = gpu_run(qw, w, schedule=qw.QW_SCHED_BLOCKED, k=4, window=False)
    assert np.array_equal(a[0], b[0])


@pytest.mark.parametrize("kernel", [2, 1], ids=["stream", "tiles"])
@pytest.mark.parametrize("dtype", [np.complex128, np.complex64])
@pytest.mark.parametrize("boundary", [qi.PERIODIC, qi.OPEN])
@pytest.mark.parametrize("coin", ["grover", "hxh", "dft", "random"])
def test_tiled_2d_schedule_is_bit_identical_to_single_steps(qw, oracle, dev, dtype, boundary, coin, kernel):
    """P13 in 2D, state held in registers for k steps == k fused single steps, for both kernels of QW_SCHED_TILED:
    the streaming kernel (warps streaming down strips of columns with a k-level pipeline of rows, shuffles along n, no
    exchange along m) and the CTA tiles (TMA-prefetched tiles, renamed shifts, shuffles along n, shared-memory slots along m).
    Extents span several tiles / strips with ragged tails, fewer units than SMs, more units than SMs, odd widths."""
    rng = np.random.default_rng(13)
    for extents, steps, k, batch in (((97, 130), 21, 0, 1), ((64, 64), 9, 2, 3), ((33, 200), 17, 4, 1),
                                     ((150, 41), 26, 6, 1), ((500, 700), 16, 8, 1), ((35, 32), 8, 8, 2)):
        c = {"grover": qi.grover4, "hxh": qi.hadamard_x_hadamard, "dft": qi.dft4}[coin](dtype) if coin != "random" \
            else qi.random_unitary(rng, 4).astype(dtype)
        sites = extents[0] * extents[1]
        w = qi.Workload("til2d", 2, extents, batch, boundary, np.dtype(dtype), steps, qi.COIN_UNIFORM, c,
                        state=qi.random_state(31, batch, sites, 4, dtype, normalise_per_walk=True))
        a = gpu_run(qw, w, schedule=qw.QW_SCHED_FUSED)
        b = gpu_run(qw, w, schedule=qw.QW_SCHED_TILED, k=k, options={qw.QW_OPT_TILED2D_KERNEL: kernel})
        assert b[3]["sched"] == qw.QW_SCHED_TILED
        assert np.array_equal(a[0], b[0]), (extents, steps, k)
        if sites < 20000:
            check_parity(w, b, oracle_run(oracle, w))


@pytest.mark.parametrize("dtype", [np.complex128, np.complex64])
@pytest.mark.parametrize("boundary", [qi.PERIODIC, qi.OPEN])
def test_streaming_2d_kernel_depths_chains_and_edges(qw, oracle, dev, dtype, boundary):
    """The streaming kernel beyond the shapes of the test above: its deepest pipelines (k = 10 for complex64, 8 for
    complex128), few warps (QW_OPT_MAX_CTAS) so that every warp runs many units one after the other and segments are cut
    at many rows, lattices whose last strip holds one or two columns, a row count that is not a multiple of anything, odd
    widths (a lane segment cut by the end of the row), batches; streaming == CTA tiles == fused steps bit for bit, and
    parity with the oracle."""
    rng = np.random.default_rng(17)
    deep = (10, 8) if dtype == np.complex64 else (8, 6)
    cases = [((211, 97), 27, deep[0], 1, 0), ((64, 49), 24, deep[1], 2, 1), ((301, 145), 20, 8, 1, 2),
             ((73, 200), 31, 4, 3, 3), ((1000, 129), 16, 0, 1, 0),
             # one unit over all rows: on the torus its input crosses the seam twice (rows -k .. em+k-1)
             ((40, 64), 24, 10 if dtype == np.complex64 else 8, 2, 1)]
    for extents, steps, k, batch, ctas in cases:
        for coin in ("dft", "grover", "random"):
            c = {"grover": qi.grover4, "dft": qi.dft4}[coin](dtype) if coin != "random" else qi.random_unitary(rng, 4).astype(dtype)
            sites = extents[0] * extents[1]
            w = qi.Workload("str2d", 2, extents, batch, boundary, np.dtype(dtype), steps, qi.COIN_UNIFORM, c,
                            state=qi.random_state(37, batch, sites, 4, dtype, normalise_per_walk=True))
            a = gpu_run(qw, w, schedule=qw.QW_SCHED_FUSED)
            b = gpu_run(qw, w, schedule=qw.QW_SCHED_TILED, k=k, options={qw.QW_OPT_TILED2D_KERNEL: 2, qw.QW_OPT_MAX_CTAS: ctas})
            assert b[3]["sched"] == qw.QW_SCHED_TILED
            assert np.array_equal(a[0], b[0]), (extents, steps, k, coin)
            if k in (0, 2, 4, 6, 8):
                t = gpu_run(qw, w, schedule=qw.QW_SCHED_TILED, k=k, options={qw.QW_OPT_TILED2D_KERNEL: 1})
                assert np.array_equal(t[0], b[0]), (extents, steps, k, coin)
            if sites < 25000 and coin != "grover":
                check_parity(w, b, oracle_run(oracle, w))
    # a depth the kernel has no instance for
    w = qi.k3(extents=(96, 80), steps=14, coin="dft", dtype=dtype)
    h = qw.create_for(w)
    try:
        qw.load_state(h, w)
        qw.qw_set_schedule(h, qw.QW_SCHED_TILED, 14)
        with pytest.raises(qw.QwError) as ei:
            qw.qw_step(h, 14)
        assert ei.value.code == qw.QW_EINVAL
    finally:
        qw.qw_destroy(h)


@pytest.mark.parametrize("kernel", [2, 1], ids=["stream", "tiles"])
@pytest.mark.parametrize("window", [True, False])
@pytest.mark.parametrize("dtype", [np.complex128, np.complex64])
def test_tiled_2d_delta_start_reaches_the_walls(qw, dev, window, dtype, kernel):
    """Light-cone window on the tiled schedule (only tiles meeting the cone are launched) and the
    reflecting walls inside register tiles: the walker hits all four walls and comes back."""
    w = qi.k2(half=40, steps=131)
    w.dtype = np.dtype(dtype)
    w.coin = w.coin.astype(dtype)
    w.delta_coin = w.delta_coin.astype(dtype)
    a = gpu_run(qw, w, schedule=qw.QW_SCHED_FUSED, window=False)
    opt = {qw.QW_OPT_TILED2D_KERNEL: kernel}
    for k in (0, 4):
        b = gpu_run(qw, w, schedule=qw.QW_SCHED_TILED, k=k, window=window, options=opt)
        assert b[3]["sched"] == qw.QW_SCHED_TILED
        assert np.array_equal(a[0], b[0])
        assert np.array_equal(a[1], b[1])
    # off-centre start near a corner, walls met at different times
    w.delta_site = (3, 70)
    a = gpu_run(qw, w, schedule=qw.QW_SCHED_FUSED, window=False)
    b = gpu_run(qw, w, schedule=qw.QW_SCHED_TILED, window=window, options=opt)
    assert np.array_equal(a[0], b[0])


def test_tiled_2d_is_the_auto_schedule_and_rejects_bad_depths(qw, dev):
    w = qi.k3(extents=(96, 80), steps=11, coin="dft")
    a = gpu_run(qw, w)
    assert a[3]["sched"] == qw.QW_SCHED_TILED and a[3]["k"] == 8
    assert np.array_equal(a[0], gpu_run(qw, w, schedule=qw.QW_SCHED_FUSED)[0])
    h = qw.create_for(w)
    try:
        qw.load_state(h, w)
        qw.qw_set_schedule(h, qw.QW_SCHED_TILED, 3)
        with pytest.raises(qw.QwError) as ei:
            qw.qw_step(h, 4)
        assert ei.value.code == qw.QW_EINVAL
    finally:
        qw.qw_destroy(h)


def test_blocked_schedule_rejected_where_it_does_not_apply(qw, dev):
    w = qi.k3(extents=(64, 64), steps=4, coin="dft")
    w.lattice = qi.DIAGONAL
    h = qw.create_for(w)
    try:
        qw.load_state(h, w)
        qw.qw_set_schedule(h, qw.QW_SCHED_BLOCKED, 0)
        with pytest.raises(qw.QwError) as ei:
            qw.qw_step(h, 4)
        assert ei.value.code == qw.QW_EUNSUPPORTED
    finally:
        qw.qw_destroy(h)


@pytest.mark.parametrize("wl", ["k0", "k2", "k4", "k2-periodic-corner"])
def test_light_cone_window_is_exact(qw, dev, wl):
    """the 'line' variant updates only the sites the walker can have reached."""
    if wl == "k0":
        w = qi.k0(steps=130, half_width=100)          # front reaches the wall at step 100, then reflects
    elif wl == "k2":
        w = qi.k2(half=30, steps=45)
    elif wl == "k4":
        w = qi.k4(batch=4, half=40, steps=60)
    else:
        w = qi.k2(half=20, steps=30)
        w.boundary = qi.PERIODIC
        w.delta_site = (1, 39)                        # window wraps at once in both directions
    on = gpu_run(qw, w, window=True)
    off = gpu_run(qw, w, window=False)
    assert np.array_equal(on[0], off[0])
    assert np.array_equal(on[1], off[1])


@pytest.mark.parametrize("dtype", [np.complex128, np.complex64])
@pytest.mark.parametrize("coin", ["grover", "hxh", "dft", "random"])
def test_tiled_2d_diagonal_lattice_is_bit_identical_to_single_steps(qw, oracle, dev, dtype, coin):
    """The lattice of the paper's Tables 2-3 (Fig. 1c) in the register-tiled kernel: every plane crosses
    lanes AND warps each step (corner elements travel with their row).  Torus, random state: several tiles with ragged
    tails, fewer and more tiles than SMs, every depth K; tiled == fused bit for bit, and parity with the oracle."""
    rng = np.random.default_rng(14)
    for extents, steps, k, batch in (((97, 130), 21, 0, 1), ((64, 64), 9, 2, 3), ((33, 200), 17, 4, 1),
                                     ((150, 41), 26, 6, 1), ((500, 700), 16, 8, 1), ((35, 32), 8, 8, 2)):
        c = {"grover": qi.grover4, "hxh": qi.hadamard_x_hadamard, "dft": qi.dft4}[coin](dtype) if coin != "random" \
            else qi.random_unitary(rng, 4).astype(dtype)
        sites = extents[0] * extents[1]
        w = qi.Workload("dgt2d", 2, extents, batch, qi.PERIODIC, np.dtype(dtype), steps, qi.COIN_UNIFORM, c,
                        state=qi.random_state(33, batch, sites, 4, dtype, normalise_per_walk=True), lattice=qi.DIAGONAL)
        a = gpu_run(qw, w, schedule=qw.QW_SCHED_FUSED)
        b = gpu_run(qw, w, schedule=qw.QW_SCHED_TILED, k=k)
        assert b[3]["sched"] == qw.QW_SCHED_TILED
        assert np.array_equal(a[0], b[0]), (extents, steps, k)
        if sites < 20000:
            check_parity(w, b, oracle_run(oracle, w))
    assert gpu_run(qw, w)[3]["sched"] == qw.QW_SCHED_TILED                     # the AUTO schedule on a diagonal torus


@pytest.mark.parametrize("dtype", [np.complex128, np.complex64])
@pytest.mark.parametrize("boundary", [qi.OPEN, qi.PERIODIC])
def test_tiled_2d_diagonal_lattice_delta_start(qw, oracle, dev, dtype, boundary):
    """Delta start on the diagonal lattice (the paper's Table 2 workload in small): the tiled kernel has no wall code, so
    on an open lattice the dispatcher hands over to the fused kernel when the light cone reaches a wall, and on a torus
    the window is dropped when the cone wraps.  Off-centre start, more steps than the distance to the nearest wall."""
    c = qi.dft4(dtype)
    dc = np.array([0.5, -0.5, -0.5, 0.5], dtype=dtype)
    w = qi.Workload("dgd", 2, (140, 170), 1, boundary, np.dtype(dtype), 90, qi.COIN_UNIFORM, c, delta_site=(40, 100),
                    delta_coin=dc, lattice=qi.DIAGONAL)
    ref = gpu_run(qw, w, schedule=qw.QW_SCHED_FUSED, window=False)
    for window in (True, False) if boundary == qi.PERIODIC else (True,):
        t = gpu_run(qw, w, schedule=qw.QW_SCHED_TILED, window=window)
        assert np.array_equal(ref[0], t[0]), window
    auto = gpu_run(qw, w)
    assert np.array_equal(ref[0], auto[0])
    check_parity(w, auto, oracle_run(oracle, w))
    if boundary == qi.OPEN:                       # launch count: the first 40 - 8 steps at least were blocked
        assert auto[3]["launches"] < ref[3]["launches"] - 20
        h = qw.create_for(w)
        try:
            qw.qw_set_schedule(h, qw.QW_SCHED_TILED, 0)
            qw.qw_set_state(h, w.initial_state())                               # general state on an open diagonal lattice
            with pytest.raises(qw.QwError) as ei:
                qw.qw_step(h, 8)
            assert ei.value.code == qw.QW_EUNSUPPORTED
        finally:
            qw.qw_destroy(h)


@pytest.mark.parametrize("kernel", [2, 1], ids=["stream", "tiles"])
@pytest.mark.parametrize("dtype", [np.complex128, np.complex64])
@pytest.mark.parametrize("coin", ["grover", "dft"])
def test_light_cone_diamond_of_the_tiled_kernel(qw, oracle, dev, dtype, coin, kernel):
    """Both kernels of the tiled 2D schedule skip every tile / unit outside the cone's diamond |dm| + |dn| <= t (natural lattice).  Multi-tile
    lattices, off-centre starts: (a) open, the diamond is cut by two walls and reflects; (b) torus, the diamond is used
    until the cone's box wraps around, then switched off; (c) split stepping continues the same cone.  Window on ==
    window off bit for bit, and parity with the oracle."""
    c = {"grover": qi.grover4, "dft": qi.dft4}[coin](dtype)
    dc = np.array([0.5, -0.5, -0.5, 0.5], dtype=dtype)
    for boundary, ext, site, steps in ((qi.OPEN, (150, 210), (20, 170), 120), (qi.PERIODIC, (97, 130), (48, 65), 70)):
        w = qi.Workload("dia", 2, ext, 1, boundary, np.dtype(dtype), steps, qi.COIN_UNIFORM, c, delta_site=site, delta_coin=dc)
        on = gpu_run(qw, w, schedule=qw.QW_SCHED_TILED, window=True, options={qw.QW_OPT_TILED2D_KERNEL: kernel})
        off = gpu_run(qw, w, schedule=qw.QW_SCHED_FUSED, window=False)
        assert on[3]["sched"] == qw.QW_SCHED_TILED
        assert np.array_equal(on[0], off[0]), (boundary, ext)
        check_parity(w, on, oracle_run(oracle, w))
        h = qw.create_for(w)
        try:
            qw.qw_set_option(h, qw.QW_OPT_TILED2D_KERNEL, kernel)
            qw.qw_set_schedule(h, qw.QW_SCHED_TILED, 0)
            qw.load_state(h, w)
            qw.qw_step(h, 13); qw.qw_step(h, steps - 13)
            got = np.empty((1, w.sites, 4), dtype=w.dtype)
            qw.qw_get_state(h, got)
        finally:
            qw.qw_destroy(h)
        assert np.array_equal(got, off[0])


@pytest.mark.parametrize("dtype", [np.complex128, np.complex64])
@pytest.mark.parametrize("boundary", [qi.OPEN, qi.PERIODIC])
def test_streaming_2d_kernel_enumerates_the_active_units_of_the_diamond(qw, oracle, dev, dtype, boundary):
    """With the light-cone diamond the streaming kernel deals only the ACTIVE units (per segment row the strips that meet the
    diamond: one interval in closed form) to its warps.  A batch (the scan runs over walks x segments), off-centre starts cut
    by the walls / close to the seams, many and few warps (QW_OPT_MAX_CTAS: every warp takes many units / every warp at most
    one), steps split over calls so that cones of many radii are launched: window on == window off (fused) bit for bit, and
    parity with the oracle."""
    c = qi.grover4(dtype)
    dc = np.array([0.5, -0.5, -0.5, 0.5], dtype=dtype)
    for ext, site, steps, batch, ctas in (((230, 310), (100, 150), 96, 3, 0), ((230, 310), (12, 290), 70, 2, 1),
                                          ((401, 130), (200, 64), 120, 1, 2)):
        w = qi.Workload("dia-batch", 2, ext, batch, boundary, np.dtype(dtype), steps, qi.COIN_UNIFORM, c, delta_site=site, delta_coin=dc)
        off = gpu_run(qw, w, schedule=qw.QW_SCHED_FUSED, window=False)
        h = qw.create_for(w)
        try:
            qw.qw_set_option(h, qw.QW_OPT_TILED2D_KERNEL, 2)
            qw.qw_set_option(h, qw.QW_OPT_MAX_CTAS, ctas)
            qw.qw_set_schedule(h, qw.QW_SCHED_TILED, 0)
            qw.load_state(h, w)
            done = 0
            for n in (6, 20, 2, steps - 28):
                qw.qw_step(h, n); done += n
            assert done == steps and qw.qw_get_info(h, qw.QW_INFO_WINDOW) in (0, 1)
            got = np.empty((batch, w.sites, 4), dtype=w.dtype)
            qw.qw_get_state(h, got)
        finally:
            qw.qw_destroy(h)
        assert np.array_equal(got, off[0]), (ext, site, boundary)
        if batch == 1:
            check_parity(w, gpu_run(qw, w, schedule=qw.QW_SCHED_TILED, options={qw.QW_OPT_TILED2D_KERNEL: 2}), oracle_run(oracle, w))


@pytest.mark.parametrize("dtype", [np.complex128, np.complex64])
def test_coin_family_fast_paths(qw, oracle, dev, dtype):
    """PAPER.md:35-38 eq. 1 "collections C = (C_v)": per-walk matrices and / or per-site phases on lattices too long for
    the resident kernel.  The vectorised fused kernel (FAM instance) and, on rings, the chained blocked kernel (phases
    renamed like a plane that moves one site per step, the entering phase read a step ahead) must give the generic
    kernel's state bit for bit, and the oracle's within the gates."""
    rng = np.random.default_rng(51)
    cases = []
    for sites, batch, steps, kind in ((40000, 3, 72, "perwalk+ph"), (9001, 2, 40, "perwalk"), (20011, 1, 56, "uniform+ph")):
        if kind.startswith("perwalk"):
            a3 = rng.uniform(0, 2 * np.pi, (batch, 3))
            mode, c = qi.COIN_PER_WALK, qi.su2(a3[:, 0], a3[:, 1], a3[:, 2]).astype(dtype)
        else:
            mode, c = qi.COIN_UNIFORM, qi.su2(*rng.uniform(0, 2 * np.pi, 3)).astype(dtype)
        ph = np.exp(1j * rng.uniform(0, 2 * np.pi, (batch, sites))).astype(dtype) if kind.endswith("+ph") else None
        cases.append(qi.Workload("fam1d", 1, (sites,), batch, qi.PERIODIC, np.dtype(dtype), steps, mode, c, phases=ph,
                                 state=qi.random_state(21, batch, sites, 2, dtype, normalise_per_walk=True)))
    for w in cases:
        g = gpu_run(qw, w, schedule=qw.QW_SCHED_GENERIC)
        f = gpu_run(qw, w, schedule=qw.QW_SCHED_FUSED)
        assert np.array_equal(g[0], f[0]), w.name
        for k, max_ctas in ((16, 1), (0, 0)):
            b = gpu_run(qw, w, schedule=qw.QW_SCHED_BLOCKED, k=k, options={qw.QW_OPT_MAX_CTAS: max_ctas})
            assert b[3]["sched"] == qw.QW_SCHED_BLOCKED and b[3]["launches"] < g[3]["launches"]
            assert np.array_equal(g[0], b[0]), (w.sites, k)
        auto = gpu_run(qw, w)
        assert auto[3]["sched"] == qw.QW_SCHED_BLOCKED and np.array_equal(auto[0], g[0])
        check_parity(w, f, oracle_run(oracle, w))
    # 2D, open and periodic: fused family kernel == generic kernel
    for boundary in (qi.OPEN, qi.PERIODIC):
        batch, ext = 2, (97, 130)
        c = np.stack([qi.random_unitary(rng, 4) for _ in range(batch)]).astype(dtype)
        ph = np.exp(1j * rng.uniform(0, 2 * np.pi, (batch, ext[0] * ext[1]))).astype(dtype)
        w = qi.Workload("fam2d", 2, ext, batch, boundary, np.dtype(dtype), 12, qi.COIN_PER_WALK, c, phases=ph,
                        state=qi.random_state(22, batch, ext[0] * ext[1], 4, dtype, normalise_per_walk=True))
        g = gpu_run(qw, w, schedule=qw.QW_SCHED_GENERIC)
        f = gpu_run(qw, w, schedule=qw.QW_SCHED_FUSED)
        assert np.array_equal(g[0], f[0])
        check_parity(w, f, oracle_run(oracle, w))


def test_moments_of_a_narrow_distribution_far_from_the_centre(qw, oracle, dev):
    """qw_moments shifts every block partial to the mean before it forms the second moments: a walker that sits 2^21
    sites from the lattice centre (x^2 ~ 4e12) keeps a variance accurate to 1e-8, where E[x^2] - E[x]^2 in double loses
    every digit below 1e-3.  Reference: the central moments of the ORACLE's state, about its own mean."""
    N = 1 << 22
    w = qi.k0(steps=40)
    w.extents, w.delta_site = (N,), (7,)
    gpu = gpu_run(qw, w, get_state=False)
    psi = np.zeros((1, 101, 2), dtype=np.complex128)                 # the walker stays within 41 sites of site 7
    psi[0, 7] = w.delta_coin
    oracle.step((101,), w.coin, psi, 40, boundary=qi.OPEN)
    P = oracle.probabilities((101,), psi)[0]
    x = np.arange(101) - N // 2
    mean = float(np.sum((x - x[7]) * P) / P.sum()) + float(x[7])
    var = float(np.sum((x - mean) ** 2 * P) / P.sum())
    assert abs(gpu[2][0, 0] - P.sum()) <= 1e-14
    assert abs(gpu[2][0, 1] - mean) <= 1e-9
    assert abs(gpu[2][0, 2] - var) <= 1e-8, (gpu[2][0, 2], var)
    assert np.array_equal(gpu[1][0, :101] > 0, P > 0)


def test_moments_of_more_than_65535_walks_and_of_an_empty_walk(qw, dev):
    batch = 70001
    st = qi.random_state(3, batch, 8, 2, np.complex64, normalise_per_walk=True)
    st[5] = 0                                                        # a walk with norm 0 reports zeros, not NaN
    h = qw.qw_create_batch(batch, 1, (8,), 2, qw.QW_C64, qw.QW_PERIODIC)
    try:
        qw.qw_set_state(h, st)
        mom = np.empty((batch, 3))
        qw.qw_moments(h, mom)
    finally:
        qw.qw_destroy(h)
    assert np.all(mom[5] == 0) and np.all(np.isfinite(mom))
    keep = np.arange(batch) != 5
    assert np.max(np.abs(mom[keep, 0] - 1)) < 1e-5
    P = np.sum(np.abs(st.astype(np.complex128)) ** 2, axis=2)
    x = np.arange(8) - 4
    assert np.max(np.abs(mom[keep, 1] - (P[keep] @ x) / P[keep].sum(axis=1))) < 1e-5


def test_segment_workload_full_length_and_segment_vs_line(qw, oracle, dev):
    """NEXT-3 (Fig. 3: "segment (left plot) ... line (right plot)"): the `seg` workload of
    bench.py — an open Hadamard segment of 2001 sites, K0's delta start, 10 000 steps, so the front reflects off the
    walls (PAPER.md:94-101 with RBL = 0) ten times — element by element against the oracle at its FULL length; and the
    qualitative statement of Fig. 3: segment and line give the same distribution until the front reaches the wall and
    different ones afterwards."""
    import bench
    w = bench.make_workload("seg")
    assert w.boundary == qi.OPEN and w.sites == 2001 and w.steps == 10000
    gpu = gpu_run(qw, w)
    check_parity(w, gpu, oracle_run(oracle, w))
    assert abs(gpu[2][0, 0] - 1) <= 1e-14 + 2e-16 * w.steps          # still unitary after ~10 reflections (R23 drift)
    # the probability front of the Hadamard walk travels at 1/sqrt(2) sites per step: it meets the walls at t ~ 1414
    for steps, same in ((900, True), (1800, False)):
        seg = qi.k0(steps=steps, half_width=1000)                    # walls at +-1000
        line = qi.k0(steps=steps, half_width=2000)                   # walls out of reach: the paper's "line"
        Ps = gpu_run(qw, seg)[1][0]
        Pl = gpu_run(qw, line)[1][0][1000:-1000]
        if same:
            assert np.array_equal(Ps, Pl)
        else:
            assert np.max(np.abs(Ps - Pl)) > 1e-3                    # the reflected front is O(0.01) of probability
            assert abs(Ps.sum() - 1) < 1e-12 and Pl.sum() < 1 - 1e-2  # the line has lost weight beyond +-1000


def test_lattice_switch_in_mid_walk_drops_the_light_cone_window(qw, oracle, dev):
    """After steps on the DIAGONAL lattice the support is a square of L1 radius 2t, larger than the diamond the tiled
    kernel of the NATURAL lattice derives from the step count: qw_set_lattice in mid-walk must drop the window
    (ADVICE round 1).  Delta start, 20 diagonal steps, then 24 natural steps under AUTO / TILED vs GENERIC, vs oracle."""
    c = qi.dft4(np.complex128)
    dc = np.array([0.5, -0.5, -0.5, 0.5], dtype=np.complex128)
    w = qi.Workload("sw", 2, (200, 200), 1, qi.OPEN, np.dtype(np.complex128), 44, qi.COIN_UNIFORM, c, delta_site=(100, 100),
                    delta_coin=dc, lattice=qi.DIAGONAL)
    out = {}
    for sched in (qw.QW_SCHED_AUTO, qw.QW_SCHED_TILED, qw.QW_SCHED_GENERIC):
        h = qw.create_for(w)
        try:
            qw.load_state(h, w)
            qw.qw_step(h, 20)
            qw.qw_set_lattice(h, qw.QW_NATURAL)
            assert qw.qw_get_info(h, qw.QW_INFO_WINDOW) == 0
            qw.qw_set_schedule(h, sched, 0)
            qw.qw_step(h, 24)
            got = np.empty((1, w.sites, 4), dtype=w.dtype)
            qw.qw_get_state(h, got)
            out[sched] = got
        finally:
            qw.qw_destroy(h)
    assert np.array_equal(out[qw.QW_SCHED_AUTO], out[qw.QW_SCHED_GENERIC])
    assert np.array_equal(out[qw.QW_SCHED_TILED], out[qw.QW_SCHED_GENERIC])
    psi = np.ascontiguousarray(w.initial_state())
    oracle.step(w.extents, c, psi, 20, boundary=qi.OPEN, lattice=qi.DIAGONAL)
    oracle.step(w.extents, c, psi, 24, boundary=qi.OPEN, lattice=qi.NATURAL)
    assert np.max(np.abs(out[qw.QW_SCHED_AUTO] - psi)) <= 1e-12


@pytest.mark.parametrize("dtype", [np.complex128, np.complex64])
def test_translation_covariance_bit_exact(qw, dev, dtype):
    """P12: on a periodic lattice with a uniform coin, shifting psi0 by s sites shifts psi(t) by s."""
    w = qi.k1(sites=40000, steps=50, dtype=dtype)
    a = gpu_run(qw, w)[0]
    w2 = qi.k1(sites=40000, steps=50, dtype=dtype)
    w2.state = np.ascontiguousarray(np.roll(w.state, 12345, axis=1))
    b = gpu_run(qw, w2)[0]
    assert np.array_equal(np.roll(a, 12345, axis=1), b)
    w = qi.k3(extents=(96, 200), steps=30, coin="dft", dtype=dtype)
    a = gpu_run(qw, w)[0].reshape(96, 200, 4)
    w2 = qi.k3(extents=(96, 200), steps=30, coin="dft", dtype=dtype)
    w2.state = np.ascontiguousarray(np.roll(w.state.reshape(96, 200, 4), (37, 101), axis=(0, 1)).reshape(1, -1, 4))
    b = gpu_run(qw, w2)[0].reshape(96, 200, 4)
    assert np.array_equal(np.roll(a, (37, 101), axis=(0, 1)), b)


# ------------------------------------------------------------------ boundary behaviour: pointers, streams, errors
def test_device_pointers_and_user_stream(qw, oracle, dev):
    import torch
    w = qi.k3(extents=(64, 96), steps=12, coin="dft")
    stream = torch.cuda.Stream()
    h = qw.create_for(w)
    try:
        qw.qw_set_stream(h, stream.cuda_stream)
        with torch.cuda.stream(stream):
            st = torch.from_numpy(w.state).to(dev, non_blocking=False)
            qw.qw_set_state(h, st)
            qw.qw_step(h, w.steps)
            out = torch.empty((w.batch, w.sites, 4), dtype=torch.complex64, device=dev)
            P = torch.empty((w.batch, w.sites), dtype=torch.float32, device=dev)
            mom = torch.empty((w.batch, 6), dtype=torch.float64, device=dev)
            qw.qw_get_state(h, out); qw.qw_probabilities(h, P); qw.qw_moments(h, mom)
        qw.qw_synchronize(h)
        stream.synchronize()
        gpu = (out.cpu().numpy(), P.cpu().numpy(), mom.cpu().numpy(), None)
    finally:
        qw.qw_destroy(h)
    check_parity(w, gpu, oracle_run(oracle, w))


def test_error_codes_on_device(qw, dev):
    h = qw.qw_create(1, [64], 2, qw.QW_C128, qw.QW_OPEN)
    try:
        with pytest.raises(qw.QwError) as ei:
            qw.qw_step(h, 1)
        assert ei.value.code == qw.QW_ESTATE                        # no coin yet
        qw.qw_set_coin(h, qw.QW_COIN_UNIFORM, qi.hadamard())
        with pytest.raises(qw.QwError) as ei:
            qw.qw_step(h, 1)
        assert ei.value.code == qw.QW_ESTATE                        # no state yet
        with pytest.raises(qw.QwError) as ei:
            qw.qw_set_state_delta(h, [64], np.array([1, 0], dtype=np.complex128))
        assert ei.value.code == qw.QW_EINVAL
        qw.qw_set_state_delta(h, [32], np.array([1, 0], dtype=np.complex128))
        with pytest.raises(qw.QwError) as ei:
            qw.qw_step(h, -1)
        assert ei.value.code == qw.QW_EINVAL
        qw.qw_step(h, 0)
        assert qw.qw_get_info(h, qw.QW_INFO_TIME) == 0
        with pytest.raises(qw.QwError) as ei:
            qw.qw_set_lattice(h, qw.QW_DIAGONAL)
        assert ei.value.code == qw.QW_EINVAL
        with pytest.raises(qw.QwError):
            qw.qw_set_coin(h, 9, qi.hadamard())
    finally:
        qw.qw_destroy(h)


def test_set_state_round_trip_is_exact(qw, dev):
    """Host buffers stream through two 64 MiB staging buffers (copy of chunk i+1 under the layout kernel of chunk i):
    the last two cases span several chunks with a ragged last one, and chunk borders inside a walk and inside a row."""
    for dtype in (np.complex128, np.complex64):
        for ext, batch in (((1001,), 3), ((33, 47), 2), ((3000001,), 2), ((1500, 1401), 1)):
            sites = int(np.prod(ext))
            st = qi.random_state(5, batch, sites, 2 * len(ext), dtype)
            h = qw.qw_create_batch(batch, len(ext), ext, 2 * len(ext), qw.dtype_code(dtype), qw.QW_PERIODIC)
            try:
                qw.qw_set_state(h, st)
                back = np.empty_like(st)
                qw.qw_get_state(h, back)
                assert np.array_equal(back, st)
            finally:
                qw.qw_destroy(h)
