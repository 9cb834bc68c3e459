"""Full-size parity: the five BASELINE.json configs at their real sizes, in the launch configuration
bench.py times (schedule AUTO, light-cone window on), checked against the oracle on SAMPLED outputs it
can compute one by one:

  * an amplitude at site x after t steps depends only on the initial state inside the light cone
    [x - t, x + t] (eq. 15 :160, eq. 18 :210), so the oracle evolves just that window
    (open ends, far enough away) and the centre sites must agree to the usual gates;
  * the reductions (qw_moments / qw_probabilities) are checked against the oracle's reductions applied to
    the state the GPU produced (same input bytes), plus the invariants that hold at any size.
"""
import numpy as np
import pytest

from paper_1003_3779_b200 import inputs as qi

pytestmark = pytest.mark.gpu

AMP_TOL = {np.dtype(np.complex128): 1e-12, np.dtype(np.complex64): 2e-5}


@pytest.fixture(scope="module")
def dev(qw):
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    return torch.device("cuda:0")


def run_full(qw, w, steps=None):
    """-> (AoS final state on the host, moments, info)"""
    h = qw.create_for(w)
    try:
        qw.load_state(h, w)
        qw.qw_step(h, w.steps if steps is None else steps)
        out = np.empty((w.batch, w.sites, w.coin_dim), dtype=w.dtype)
        qw.qw_get_state(h, out)
        mom = np.empty((w.batch, 3 if w.dim == 1 else 6))
        qw.qw_moments(h, mom)
        P = np.empty((w.batch, w.sites), dtype=np.float64 if w.dtype == np.complex128 else np.float32)
        qw.qw_probabilities(h, P)
        info = {"sched": qw.qw_get_info(h, qw.QW_INFO_LAST_SCHEDULE), "k": qw.qw_get_info(h, qw.QW_INFO_LAST_K),
                "launches": qw.qw_get_info(h, qw.QW_INFO_LAUNCHES)}
    finally:
        qw.qw_destroy(h)
    return out, mom, P, info


def check_reductions(oracle, w, final, mom, P, rtol):
    """Oracle reductions on the very state the GPU holds (promoted to double)."""
    st = np.ascontiguousarray(final.astype(np.complex128))
    momo = oracle.moments(w.extents, st, batch=w.batch)
    Po = oracle.probabilities(w.extents, st, batch=w.batch)
    ptol = 1e-12 if w.dtype == np.complex128 else 1e-6 * float(Po.max()) + 1e-12
    assert np.max(np.abs(P.astype(np.float64) - Po)) <= ptol
    nm = 1 if w.dim == 1 else 2
    ext = max(w.extents)
    for b in range(0, w.batch, max(1, w.batch // 64)):
        assert abs(mom[b, 0] - momo[b, 0]) <= rtol * momo[b, 0]
        for j in range(1, 1 + nm):
            assert abs(mom[b, j] - momo[b, j]) <= rtol * (abs(momo[b, j]) + ext)
        second = 1.0 + max(abs(momo[b, j]) for j in range(1 + nm, mom.shape[1])) + max(momo[b, j] ** 2 for j in range(1, 1 + nm))
        for j in range(1 + nm, mom.shape[1]):
            assert abs(mom[b, j] - momo[b, j]) <= rtol * second


# ------------------------------------------------------------------ K1: ring of 2^26 sites, 1000 steps
@pytest.mark.parametrize("dtype", [np.complex128, np.complex64])
def test_k1_full_size_sampled_light_cones(qw, oracle, dev, dtype):
    w = qi.k1(dtype=dtype)
    N, t = w.sites, w.steps
    final, mom, P, info = run_full(qw, w)
    assert info["sched"] == qw.QW_SCHED_BLOCKED            # the configuration bench.py times
    init = w.state[0]
    rng = np.random.default_rng(1)
    # seam, tile edges of the blocked kernel (valid = 512 - 2k sites per warp tile), random sites
    valid = 512 - 2 * info["k"]
    centres = [0, 5, N - 3, N // 2, valid, valid - 1, 7 * valid + 1, 4 * valid * 1000, N - valid] + \
        [int(x) for x in rng.integers(0, N, 23)]
    pad = 8
    half = t + pad
    worst = 0.0
    coin = w.coin.astype(np.complex128)
    for c in centres:
        idx = (np.arange(c - half, c + half + 1) % N)
        win = np.ascontiguousarray(init[idx].astype(np.complex128))[None]
        oracle.step((2 * half + 1,), coin, win, t, boundary=qi.OPEN)
        got = final[0, idx[half - pad:half + pad + 1]].astype(np.complex128)
        want = win[0, half - pad:half + pad + 1]
        worst = max(worst, float(np.max(np.abs(got - want))))
    assert worst <= AMP_TOL[np.dtype(dtype)], worst
    # invariants + reductions at full size
    if dtype == np.complex128:
        assert abs(mom[0, 0] - 1) <= 1e-14 + 2e-16 * t + 1e-12        # R23 drift (+ summation slack)
    else:
        assert abs(mom[0, 0] - 1) <= 1e-4
    check_reductions(oracle, w, final, mom, P, 1e-10 if dtype == np.complex128 else 1e-4)


# ------------------------------------------------------------------ K3: torus 8192^2, complex64
def oracle_patch_2d(oracle, init, E, coin, centre, steps, pad, stage=100):
    """Amplitudes of the (2*pad+1)^2 patch around `centre` after `steps` steps, from the oracle alone.

    The patch depends only on the initial state within `steps` + pad sites of it (eq. 18 :210).  The
    oracle evolves that window with open ends; what the (wrong) ends emit travels inwards one site per step, so after
    every `stage` steps the outer `stage` sites are dropped and the rest is still exact.  This is scheduling of calls
    to oracle.step, not a change of its arithmetic."""
    cm, cn = centre
    half = steps + pad
    im = np.arange(cm - half, cm + half + 1) % E
    inn = np.arange(cn - half, cn + half + 1) % E
    win = np.ascontiguousarray(init[np.ix_(im, inn)].astype(np.complex128))
    done = 0
    while done < steps:
        d = min(stage, steps - done)
        side = win.shape[0]
        flat = np.ascontiguousarray(win.reshape(1, side * side, 4))
        oracle.step((side, side), coin, flat, d, boundary=qi.OPEN)
        win = np.ascontiguousarray(flat.reshape(side, side, 4)[d:side - d, d:side - d])
        done += d
    assert win.shape[0] == 2 * pad + 1
    return win, (im[half - pad:half + pad + 1], inn[half - pad:half + pad + 1])


@pytest.mark.parametrize("coin,steps,nsamples", [("hxh", 96, 6), ("dft", 96, 6), ("hxh", 500, 4), ("dft", 500, 4)])
def test_k3_full_size_sampled_light_cones(qw, oracle, dev, coin, steps, nsamples):
    """BASELINE.json:configs[3] at its full size and (500) its full step count, both coins: >= 4 light-cone patches
    each (the torus seam in both directions, a tile corner of the 64 x 64 register tiles, the lattice centre)."""
    w = qi.k3(coin=coin, steps=steps)
    E = w.extents[0]
    final, mom, P, info = run_full(qw, w)
    assert info["sched"] == qw.QW_SCHED_TILED                 # the configuration bench.py times
    init = w.state[0].reshape(E, E, 4)
    fin = final[0].reshape(E, E, 4)
    rng = np.random.default_rng(2)
    centres = [(0, 0), (E - 1, 17), (E // 2, E - 1), (4095, 4096)][:nsamples] + \
        [tuple(int(v) for v in rng.integers(0, E, 2)) for _ in range(max(0, nsamples - 4))]
    pad = 2
    c128 = w.coin.astype(np.complex128)
    worst = 0.0
    for centre in centres:
        want, (rm, rn) = oracle_patch_2d(oracle, init, E, c128, centre, steps, pad)
        got = fin[np.ix_(rm, rn)].astype(np.complex128)
        worst = max(worst, float(np.max(np.abs(got - want))))
    assert worst <= 2e-5, worst
    assert abs(mom[0, 0] - 1) <= 1e-4
    if steps == 96 and coin == "dft":
        check_reductions(oracle, w, final, mom, P, 1e-4)


# ------------------------------------------------------------------ K2: open 4097^2 Grover walk
def oracle_delta_cone_2d(oracle, w_of_half, steps, stage=128):
    """The oracle's state of a delta-start walk after `steps` steps on the lattice of half-width steps + 1.

    A delta start is supported within t sites of its origin after t steps (eq. 18 :210) and everything
    outside is exactly zero, so the oracle may run the first t steps on any open lattice whose half-width exceeds t:
    the state is embedded in a larger lattice of zeros every `stage` steps.  Scheduling of oracle calls only."""
    done, psi, half = 0, None, 0
    while done < steps:
        d = min(stage, steps - done)
        nh = done + d + 1
        wo = w_of_half(nh)
        side = 2 * nh + 1
        if psi is None:
            big = wo.initial_state().reshape(side, side, 4)
        else:
            big = np.zeros((side, side, 4), dtype=np.complex128)
            o = nh - half
            big[o:o + 2 * half + 1, o:o + 2 * half + 1] = psi
        flat = np.ascontiguousarray(big.reshape(1, side * side, 4))
        oracle.step(wo.extents, wo.coin, flat, d, boundary=qi.OPEN)
        psi, half, done = flat.reshape(side, side, 4), nh, done + d
    return psi, half


def k2_against_the_whole_cone(qw, oracle, steps):
    w = qi.k2(steps=steps)
    final, mom, P, info = run_full(qw, w)
    assert info["sched"] == qw.QW_SCHED_TILED                 # the configuration bench.py times (diamond tile skip on)
    psi, half = oracle_delta_cone_2d(oracle, lambda h: qi.k2(half=h, steps=1), steps)
    side = 2 * half + 1
    fin = final[0].reshape(4097, 4097, 4)
    c = 2048
    lo, hi = max(0, c - half), min(4097, c + half + 1)        # 2048 steps: the cone's pad row lies outside the lattice
    o = lo - (c - half)
    want = psi[o:o + hi - lo, o:o + hi - lo]
    assert not psi[:o].any() and not psi[:, :o].any()         # ... and holds zeros only
    got = fin[lo:hi, lo:hi]
    err = float(np.max(np.abs(got - want)))
    assert err <= 1e-12, err
    outside = fin.copy()
    outside[lo:hi, lo:hi] = 0
    assert not outside.any()                                   # exact zeros outside the cone
    Po = oracle.probabilities((side, side), np.ascontiguousarray(psi.reshape(1, side * side, 4)))[0].reshape(side, side)
    perr = float(np.max(np.abs(P[0].reshape(4097, 4097)[lo:hi, lo:hi] - Po[o:o + hi - lo, o:o + hi - lo])))
    assert perr <= 1e-12, perr
    return err, perr, info


def test_k2_full_lattice_1024_steps_against_the_whole_light_cone(qw, oracle, dev):
    """Full 4097^2 lattice, 1024 of the config's 2048 steps, element by element over the WHOLE cone (2051^2 sites):
    the diamond tile-skip logic of the tiled kernel runs 1024 steps under an element-wise check."""
    k2_against_the_whole_cone(qw, oracle, 1024)


@pytest.mark.slow
def test_k2_full_config_2048_steps_against_the_whole_light_cone(qw, oracle, dev):
    """BASELINE.json:configs[2] exactly: 2048 steps, every amplitude and probability of the 4097^2 lattice against the
    oracle (about 15 min of oracle time: run with QW_RUN_SLOW=1; the builder's log line is kept in profiles/)."""
    err, perr, info = k2_against_the_whole_cone(qw, oracle, 2048)
    print("K2 full config, 2048 steps, element-wise over 4097^2 sites: max|d amp| = %.3e, max|d P| = %.3e, launches = %d"
          % (err, perr, info["launches"]))


def test_k2_full_config_invariants(qw, oracle, dev):
    """The real config (2048 steps): properties that hold at any size + the oracle's reductions."""
    w = qi.k2()
    final, mom, P, info = run_full(qw, w)
    Pg = P[0].reshape(4097, 4097)
    assert abs(Pg.sum() - 1) <= 1e-12 and abs(mom[0, 0] - 1) <= 1e-12       # Grover entries are exact: no drift
    m, n = np.meshgrid(np.arange(-2048, 2049), np.arange(-2048, 2049), indexing="ij", sparse=True)
    outside = (np.abs(m) + np.abs(n) > 2048) | (((m + n) % 2) == 1)          # diamond, parity of t = 2048
    assert not Pg[outside].any()
    assert np.max(np.abs(Pg - Pg[::-1, :])) < 1e-15 and np.max(np.abs(Pg - Pg.T)) < 1e-15
    assert abs(mom[0, 1]) < 1e-9 and abs(mom[0, 2]) < 1e-9 and abs(mom[0, 5]) < 1e-6
    check_reductions(oracle, w, final, mom, P, 1e-10)


# ------------------------------------------------------------------ K4: 4096 disordered walks
def test_k4_full_config_sampled_walks(qw, oracle, dev):
    w = qi.k4()
    final, mom, P, info = run_full(qw, w)
    # ~11 stages of the resident kernel that follow the light cone + the layout / output kernels: a handful, not 1024
    assert info["sched"] == qw.QW_SCHED_RESIDENT and info["launches"] <= 40
    mode, coin = w.general_coin_f64()
    pick = [0, 1, 147, 148, 2047, 4095] + [int(x) for x in np.random.default_rng(3).integers(0, 4096, 10)]
    init = w.initial_state()
    worst = 0.0
    for b in pick:
        psi = np.ascontiguousarray(init[b:b + 1].astype(np.complex128))
        oracle.step(w.extents, coin[b:b + 1], psi, w.steps, boundary=qi.OPEN, coin_mode=mode)
        worst = max(worst, float(np.max(np.abs(final[b] - psi[0]))))
        mo = oracle.moments(w.extents, psi)[0]
        assert abs(mom[b, 0] - mo[0]) <= 1e-10 and abs(mom[b, 1] - mo[1]) <= 1e-10 * 2049 + 1e-10 * abs(mo[1])
        assert abs(mom[b, 2] - mo[2]) <= 1e-10 * (1 + abs(mo[2]) + mo[1] ** 2)
        Po = oracle.probabilities(w.extents, psi)[0]
        assert np.max(np.abs(P[b] - Po)) <= 1e-12
    assert worst <= 1e-12, worst
    assert np.max(np.abs(mom[:, 0] - 1)) <= 1e-12


def test_k0_is_the_full_config(qw, oracle, dev):
    w = qi.k0()
    final, mom, P, info = run_full(qw, w)
    psi = w.initial_state()
    oracle.step(w.extents, w.coin, psi, w.steps, boundary=qi.OPEN)
    assert np.max(np.abs(final - psi)) <= 1e-12
    assert np.max(np.abs(P - oracle.probabilities(w.extents, psi))) <= 1e-12
    assert info["sched"] == qw.QW_SCHED_RESIDENT


# ------------------------------------------------------------------ a long disordered ring (K4's coin family, 2^24 sites)
def test_disordered_ring_2_24_sites_through_the_blocked_schedule(qw, oracle, dev):
    """BASELINE.json:configs[4]'s coin family (an SU(2) coin times per-site phase disorder, eq. 1) on a
    ring of 2^24 sites, far too long for the resident kernel: AUTO takes the chained blocked kernel; 24 sampled light
    cones (the seam, chain and tile borders, random sites) against the oracle, which evolves the window with the per-site
    matrices ph_x * C (R14)."""
    N, steps = 1 << 24, 96
    rng = np.random.default_rng(61)
    c = qi.su2(*rng.uniform(0, 2 * np.pi, 3))
    ph = np.exp(1j * rng.uniform(0, 2 * np.pi, (1, N)))
    w = qi.Workload("ring24", 1, (N,), 1, qi.PERIODIC, np.dtype(np.complex128), steps, qi.COIN_UNIFORM, c, phases=ph,
                    state=qi.random_state(62, 1, N, 2, np.complex128), outputs=("moments",))
    final, mom, P, info = run_full(qw, w)
    assert info["sched"] == qw.QW_SCHED_BLOCKED and info["launches"] < steps      # 2 step launches + the output kernels
    assert abs(mom[0, 0] - 1) <= 1e-12
    pad = 8
    half = steps + pad
    centres = [0, 3, N - 2, N // 2, 256, 255, 14176, 14175, 14176 * 700 + 1] + [int(x) for x in rng.integers(0, N, 15)]
    worst = 0.0
    for cx in centres:
        idx = np.arange(cx - half, cx + half + 1) % N
        win = np.ascontiguousarray(w.state[0, idx])[None]
        mats = qi.site_coin_matrices(c[None], ph[:, idx])
        oracle.step((2 * half + 1,), mats, win, steps, boundary=qi.OPEN, coin_mode=qi.COIN_PER_SITE)
        worst = max(worst, float(np.max(np.abs(final[0, idx[half - pad:half + pad + 1]] - win[0, half - pad:half + pad + 1]))))
    assert worst <= 1e-12, worst
