"""GPU parity for random broken links redrawn at every step (eqs. 9-10; R27):
libqw evaluates the Philox4x32-10 link function inside its step kernels, the oracle evaluates its own copy
of the published generator on the CPU; both must break exactly the same links at every step, so the states
agree to the usual gates (complex128 1e-12, complex64 2e-5).  A single wrongly broken link moves O(|amp|)
of amplitude, far above either gate.
"""
import numpy as np
import pytest

from paper_1003_3779_b200 import inputs as qi
from test_parity_gpu import AMP_TOL, dev, small_workload  # noqa: F401  (dev is a fixture)

pytestmark = pytest.mark.gpu

SEED = qi.SEED_RBL


def gpu_rbl(qw, w, p, seed, steps, schedule=None, inverse=0, window=True, split=None, k=0, options=None):
    h = qw.create_for(w)
    try:
        qw.qw_set_random_broken_links(h, 1, p, seed)
        for key, value in (options or {}).items():
            qw.qw_set_option(h, key, value)
        if schedule is not None:
            qw.qw_set_schedule(h, schedule, k)
        qw.qw_set_window(h, window)
        qw.load_state(h, w)
        if split:
            qw.qw_step(h, split)
            qw.qw_step(h, steps - split)
        else:
            qw.qw_step(h, steps)
        if inverse:
            qw.qw_step_inverse(h, inverse)
        amps = np.empty((w.batch, w.sites, w.coin_dim), dtype=w.dtype)
        qw.qw_get_state(h, amps)
        mom = np.empty((w.batch, 3 if w.dim == 1 else 6))
        qw.qw_moments(h, mom)
        return amps, mom, qw.qw_get_info(h, qw.QW_INFO_LAST_SCHEDULE), qw.qw_get_info(h, qw.QW_INFO_TIME)
    finally:
        qw.qw_destroy(h)


def oracle_rbl(oracle, w, p, seed, steps, inverse=0):
    mode, coin = w.general_coin_f64()
    psi = np.ascontiguousarray(w.initial_state().astype(np.complex128))
    kw = dict(boundary=w.boundary, coin_mode=mode, batch=w.batch, lattice=w.lattice)
    oracle.step_rbl(w.extents, coin, psi, steps, p, seed, **kw)
    if inverse:
        oracle.step_inverse_rbl(w.extents, coin, psi, inverse, p, seed, t0=steps, **kw)
    return psi


def close(w, amps, psi):
    d = float(np.max(np.abs(amps.astype(np.complex128) - psi)))
    assert d <= AMP_TOL[np.dtype(w.dtype)], "max |d amplitude| = %.3e" % d


@pytest.mark.parametrize("dtype", [np.complex128, np.complex64])
@pytest.mark.parametrize("dim,lattice", [(1, qi.NATURAL), (2, qi.NATURAL), (2, qi.DIAGONAL)])
@pytest.mark.parametrize("boundary", [qi.OPEN, qi.PERIODIC])
@pytest.mark.parametrize("p", [0.1, 0.5])
def test_rbl_small_lattices_every_kernel(qw, oracle, dev, dtype, dim, lattice, boundary, p):
    """Uniform random coin, batch of 2 (the walk index enters the counter): fused-RBL kernel where eligible
    (natural lattice), generic kernel forced and for the diagonal lattice; same links => same state."""
    rng = np.random.default_rng(41)
    w = small_workload(dim, boundary, dtype, qi.COIN_UNIFORM, rng, lattice=lattice)
    psi = oracle_rbl(oracle, w, p, SEED, 30)
    a, mom, _, t = gpu_rbl(qw, w, p, SEED, 30)
    close(w, a, psi)
    assert t == 30
    g, _, sched, _ = gpu_rbl(qw, w, p, SEED, 30, schedule=qw.QW_SCHED_GENERIC)
    assert sched == qw.QW_SCHED_GENERIC
    assert np.array_equal(a, g)                               # fused-RBL and generic kernels agree bit for bit
    s, _, _, _ = gpu_rbl(qw, w, p, SEED, 30, split=11)        # the step index carries over between calls
    assert np.array_equal(a, s)
    if dtype == np.complex128:
        assert np.max(np.abs(mom[:, 0] - 1)) < 1e-13          # every U(t) is unitary


@pytest.mark.parametrize("coin_mode,phases", [(qi.COIN_PER_WALK, True), (qi.COIN_PER_SITE, False)])
@pytest.mark.parametrize("dim", [1, 2])
def test_rbl_with_coin_families(qw, oracle, dev, coin_mode, phases, dim):
    rng = np.random.default_rng(42)
    w = small_workload(dim, qi.OPEN, np.complex128, coin_mode, rng, phases=phases, batch=3)
    close(w, gpu_rbl(qw, w, 0.3, 12345678901234567, 25)[0], oracle_rbl(oracle, w, 0.3, 12345678901234567, 25))


@pytest.mark.parametrize("dim", [1, 2])
def test_rbl_p0_and_p1_closed_forms(qw, oracle, dev, dim):
    """p = 0: no link breaks => the plain walk, bit for bit.  p = 1: every link breaks => no amplitude ever
    leaves its site (P(x) is conserved site by site)."""
    rng = np.random.default_rng(43)
    w = small_workload(dim, qi.PERIODIC, np.complex128, qi.COIN_UNIFORM, rng)
    plain = np.ascontiguousarray(w.initial_state().astype(np.complex128))
    oracle.step(w.extents, w.general_coin_f64()[1], plain, 12, boundary=w.boundary, batch=w.batch)
    a0 = gpu_rbl(qw, w, 0.0, 7, 12)[0]
    close(w, a0, plain)
    a1 = gpu_rbl(qw, w, 1.0, 7, 12)[0]
    P0 = np.sum(np.abs(w.initial_state()) ** 2, axis=-1)
    assert np.max(np.abs(np.sum(np.abs(a1) ** 2, axis=-1) - P0)) < 1e-14
    close(w, a1, oracle_rbl(oracle, w, 1.0, 7, 12))


@pytest.mark.parametrize("dim,lattice", [(1, qi.NATURAL), (2, qi.NATURAL), (2, qi.DIAGONAL)])
def test_rbl_inverse_undoes_the_same_link_sequence(qw, oracle, dev, dim, lattice):
    rng = np.random.default_rng(44)
    w = small_workload(dim, qi.OPEN, np.complex128, qi.COIN_UNIFORM, rng, lattice=lattice)
    close(w, gpu_rbl(qw, w, 0.4, SEED, 20, inverse=7)[0], oracle_rbl(oracle, w, 0.4, SEED, 20, inverse=7))
    back, _, _, t = gpu_rbl(qw, w, 0.4, SEED, 20, inverse=20)
    assert t == 0
    assert np.max(np.abs(back - w.initial_state())) <= 1e-13
    h = qw.create_for(w)
    try:
        qw.qw_set_random_broken_links(h, 1, 0.4, SEED)
        qw.load_state(h, w)
        qw.qw_step(h, 3)
        with pytest.raises(qw.QwError) as e:
            qw.qw_step_inverse(h, 4)                             # would pass t = 0
        assert e.value.code == qw.QW_ESTATE
        with pytest.raises(qw.QwError) as e:
            qw.qw_set_random_broken_links(h, 1, 1.5, 0)
        assert e.value.code == qw.QW_EINVAL
    finally:
        qw.qw_destroy(h)


@pytest.mark.parametrize("dtype", [np.complex128, np.complex64])
def test_rbl_multi_tile_lattices(qw, oracle, dev, dtype):
    """Sizes that span several CTAs with ragged tails (owner indices cross block and row boundaries), the
    named coins of PAPER.md:82, delta starts with the light-cone window (broken links only shrink the cone)."""
    for w, p in ((qi.k1(sites=100003, steps=40, dtype=dtype), 0.05),
                 (qi.k3(extents=(61, 1030), steps=24, coin="dft") if dtype == np.complex64
                  else qi.k2(half=40, steps=60), 0.2),
                 (qi.k4(batch=5, half=300, steps=200) if dtype == np.complex128
                  else qi.k3(extents=(130, 97), steps=20, coin="hxh"), 0.1)):
        psi = oracle_rbl(oracle, w, p, SEED, w.steps)
        a, mom, _, _ = gpu_rbl(qw, w, p, SEED, w.steps)
        close(w, a, psi)
        if w.state is None:                                       # delta start: the window must not change anything
            b = gpu_rbl(qw, w, p, SEED, w.steps, window=False)[0]
            assert np.array_equal(a, b)


@pytest.mark.parametrize("dtype", [np.complex128, np.complex64])
@pytest.mark.parametrize("coin", ["hadamard", "su2"])
def test_rbl_inside_the_temporally_blocked_ring_kernel(qw, oracle, dev, dtype, coin):
    """Random broken links inside the chained blocked 1D kernel (qw_step_chain1d.cu): one Philox call per (site, step)
    in registers, a broken link = a predicated swap of two registers of the lane.  Rings of several chains / tiles with
    ragged ends and a batch, every depth, split stepping (the step index carries over), p = 0.1 and 0.5: the same links as
    the oracle, and the same state as the fused-RBL kernel (bit for bit for a general coin; <= 4 ulp per step for the
    Hadamard coin, whose scale the blocked kernel applies once per 16 steps)."""
    rng = np.random.default_rng(45)
    for sites, steps, k, batch, max_ctas, p in ((20000, 112, 48, 1, 1, 0.1), (3001, 64, 16, 3, 2, 0.5), (70001, 80, 0, 1, 0, 0.1)):
        c = qi.hadamard(dtype) if coin == "hadamard" else qi.su2(*rng.uniform(0, 2 * np.pi, 3)).astype(dtype)
        w = qi.Workload("rblchain", 1, (sites,), batch, qi.PERIODIC, np.dtype(dtype), steps, qi.COIN_UNIFORM, c,
                        state=qi.random_state(12, batch, sites, 2, dtype, normalise_per_walk=True))
        opt = {qw.QW_OPT_MAX_CTAS: max_ctas, qw.QW_OPT_BLOCKED1D_KERNEL: 2}
        b, mom, sched, t = gpu_rbl(qw, w, p, SEED, steps, schedule=qw.QW_SCHED_BLOCKED, k=k, options=opt)
        assert sched == qw.QW_SCHED_BLOCKED and t == steps
        f = gpu_rbl(qw, w, p, SEED, steps, schedule=qw.QW_SCHED_FUSED)[0]
        if coin == "su2":
            assert np.array_equal(b, f), (sites, steps, k)
        else:
            eps = np.finfo(np.float64 if dtype == np.complex128 else np.float32).eps
            assert np.max(np.abs(b.astype(np.complex128) - f.astype(np.complex128))) <= 4 * eps * steps * float(np.max(np.abs(f)))
        close(w, b, oracle_rbl(oracle, w, p, SEED, steps))
        s2 = gpu_rbl(qw, w, p, SEED, steps, schedule=qw.QW_SCHED_BLOCKED, k=k, options=opt, split=steps // 2 // 16 * 16)[0]
        assert np.array_equal(b, s2)
        if dtype == np.complex128:
            assert np.max(np.abs(mom[:, 0] - 1)) < 1e-12
    low = gpu_rbl(qw, w, p, SEED, steps, schedule=qw.QW_SCHED_BLOCKED, k=4)   # depth below the tile granule: fused steps
    assert np.array_equal(low[0], f)
    auto = gpu_rbl(qw, w, p, SEED, steps)                             # AUTO takes the blocked kernel on a long ring
    assert auto[2] == qw.QW_SCHED_BLOCKED and np.array_equal(auto[0], b)


@pytest.mark.parametrize("dtype", [np.complex128, np.complex64])
@pytest.mark.parametrize("boundary", [qi.OPEN, qi.PERIODIC])
def test_rbl_2d_even_rows_share_generator_calls_between_lane_pairs(qw, oracle, dev, dtype, boundary):
    """2D natural lattice with an even row length: the fused-RBL kernel lets lane pairs share one generator call for the
    pair's own links and one for its upper-row links.  Delta start with the light-cone window at odd and even first
    columns (the launcher extends the box to an even column), several CTAs per row, rows that wrap to the last row."""
    c = qi.dft4(dtype)
    dc = np.array([0.5, -0.5, -0.5, 0.5], dtype=dtype)
    for ext, site, steps in (((60, 64), (30, 31), 25), ((9, 1200), (0, 600), 40), ((34, 530), (33, 2), 30)):
        w = qi.Workload("rbl2d", 2, ext, 2, boundary, np.dtype(dtype), steps, qi.COIN_UNIFORM, c, delta_site=site, delta_coin=dc)
        psi = oracle_rbl(oracle, w, 0.2, SEED, steps)
        on = gpu_rbl(qw, w, 0.2, SEED, steps, schedule=qw.QW_SCHED_FUSED, window=True)
        off = gpu_rbl(qw, w, 0.2, SEED, steps, schedule=qw.QW_SCHED_FUSED, window=False)
        gen = gpu_rbl(qw, w, 0.2, SEED, steps, schedule=qw.QW_SCHED_GENERIC, window=False)
        assert np.array_equal(on[0], off[0]) and np.array_equal(off[0], gen[0]), (ext, site)
        close(w, on[0], psi)


@pytest.mark.parametrize("dtype", [np.complex128, np.complex64])
@pytest.mark.parametrize("dim", [1, 2])
def test_ensemble_average_over_the_batch(qw, oracle, dev, dtype, dim):
    """qw_probabilities_mean (SURVEY.md 8(f) NEXT-2 "ensemble averages over the batch axis"): a batch of walks from ONE initial
    state, every walk with its own random broken links, averaged per site — against the oracle's
    average of the oracle's walks; host and device output buffers; odd row lengths; p = 0 gives the single walk back."""
    import torch
    batch = 24
    ext = (4099,) if dim == 1 else (37, 75)
    sites = int(np.prod(ext))
    one = qi.random_state(41, 1, sites, 2 * dim, dtype)
    state = np.ascontiguousarray(np.repeat(one, batch, axis=0))
    coin = qi.hadamard(dtype) if dim == 1 else qi.grover4(dtype)
    w = qi.Workload("ens", dim, ext, batch, qi.PERIODIC, np.dtype(dtype), 12, qi.COIN_UNIFORM, coin, state=state)
    rt = np.float64 if dtype == np.complex128 else np.float32
    tol = 1e-12 if dtype == np.complex128 else 1e-7
    for p in (0.25, 0.0):
        h = qw.create_for(w)
        try:
            qw.qw_set_random_broken_links(h, 1, p, SEED)
            qw.load_state(h, w)
            qw.qw_step(h, w.steps)
            host = np.empty((sites,), dtype=rt)
            qw.qw_probabilities_mean(h, host)
            devbuf = torch.empty((sites,), dtype=torch.float64 if rt == np.float64 else torch.float32, device=dev)
            qw.qw_probabilities_mean(h, devbuf)
            P = np.empty((batch, sites), dtype=rt)
            qw.qw_probabilities(h, P)
        finally:
            qw.qw_destroy(h)
        assert np.array_equal(host, devbuf.cpu().numpy())
        psi = oracle_rbl(oracle, w, p, SEED, w.steps)
        want = oracle.probabilities_mean(ext, psi, batch=batch)
        assert float(np.max(np.abs(host.astype(np.float64) - want))) <= tol
        assert abs(float(np.sum(host.astype(np.float64))) - 1.0) <= (1e-12 if dtype == np.complex128 else 1e-4)
        if p == 0.0:          # no broken links: all walks are the same walk
            assert float(np.max(np.abs(host.astype(np.float64) - P[0].astype(np.float64)))) <= tol
        else:                 # the realisations differ, the average is none of them
            assert float(np.max(np.abs(P[0].astype(np.float64) - P[1].astype(np.float64)))) > 1e-6


@pytest.mark.parametrize("dtype", [np.complex128, np.complex64])
@pytest.mark.parametrize("boundary", [qi.PERIODIC, qi.OPEN])
def test_rbl_inside_the_streaming_2d_kernel(qw, oracle, dev, dtype, boundary):
    """Random broken links drawn INSIDE the temporally blocked 2D kernel (eqs. 9-10; reading R27): level l of
    the row pipeline is step t + l, one generator call per lane, level and row for the four links its two sites own, the
    bit of the link to the next lane travels by shuffle, a broken link along m swaps phi_2 with the parked phi_1 one
    cascade later.  Streaming == fused-RBL bit for bit (same link function, same coin arithmetic) and parity with the
    oracle: several strips and segments, walls, batches (the walk index is part of the counter), every depth, split
    stepping (the step index carries over), p = 1 (every link broken: nothing moves)."""
    rng = np.random.default_rng(23)
    cases = [((70, 96), 13, 0, 1, 0.1), ((64, 64), 12, 2, 3, 0.5), ((201, 130), 16, 4, 1, 0.1), ((97, 200), 18, 6, 2, 0.25),
             ((130, 72), 16, 6, 1, 0.1), ((48, 40), 8, 4, 1, 1.0)]
    for extents, steps, k, batch, p in cases:
        for coin in ("dft", "grover", "random"):
            c = {"grover": qi.grover4, "dft": qi.dft4}[coin](dtype) if coin != "random" else qi.random_unitary(rng, 4).astype(dtype)
            sites = extents[0] * extents[1]
            w = qi.Workload("rbl2d", 2, extents, batch, boundary, np.dtype(dtype), steps, qi.COIN_UNIFORM, c,
                            state=qi.random_state(43, batch, sites, 4, dtype, normalise_per_walk=True))
            a = gpu_rbl(qw, w, p, SEED, steps, schedule=qw.QW_SCHED_FUSED)
            b = gpu_rbl(qw, w, p, SEED, steps, schedule=qw.QW_SCHED_TILED, k=k, split=5 if k else None)
            assert b[2] == qw.QW_SCHED_TILED
            assert np.array_equal(a[0], b[0]), (extents, steps, k, coin, p)
            if sites < 20000 and coin != "grover":
                close(w, b[0], oracle_rbl(oracle, w, p, SEED, steps))
    # AUTO takes the streaming kernel; a delta start with the light-cone window; few warps (many units per warp)
    w = qi.Workload("rbl2d-delta", 2, (121, 122), 1, boundary, np.dtype(dtype), 50, qi.COIN_UNIFORM, qi.grover4(dtype),
                    delta_site=(60, 61), delta_coin=np.array([0.5, -0.5, -0.5, 0.5], dtype=dtype))
    a = gpu_rbl(qw, w, 0.2, SEED, w.steps, schedule=qw.QW_SCHED_FUSED, window=False)
    b = gpu_rbl(qw, w, 0.2, SEED, w.steps, options={qw.QW_OPT_MAX_CTAS: 1})
    assert b[2] == qw.QW_SCHED_TILED and np.array_equal(a[0], b[0])
    close(w, b[0], oracle_rbl(oracle, w, 0.2, SEED, w.steps))
    # rows of odd length: two sites of a lane do not share a generator call -> no streaming instance, AUTO runs fused
    w = qi.k3(extents=(64, 65), steps=6, coin="dft", dtype=dtype)
    assert gpu_rbl(qw, w, 0.1, SEED, 6)[2] == qw.QW_SCHED_FUSED
    h = qw.create_for(w)
    try:
        qw.qw_set_random_broken_links(h, 1, 0.1, SEED)
        qw.qw_set_schedule(h, qw.QW_SCHED_TILED, 0)
        qw.load_state(h, w)
        with pytest.raises(qw.QwError) as ei:
            qw.qw_step(h, 4)
        assert ei.value.code == qw.QW_EUNSUPPORTED
    finally:
        qw.qw_destroy(h)
