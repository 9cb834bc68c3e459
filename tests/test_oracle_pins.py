"""Pins for the CPU oracle (oracle/qw_oracle.cpp): everything it computes is checked here against
something OTHER than itself — exact path sums in integer arithmetic, hand-derived fixtures,
the Kronecker-product form of U = S(I (x) C) built with numpy, the spectral (FFT) closed form
on periodic lattices, exactly solvable degenerate coins, textbook moments of simple
distributions, and the invariants the paper states (normalisation PAPER.md:56 eq. 4,
light cone PAPER.md:116 / :160 eq. 15).  Pin numbers P1..P15 follow SURVEY.md §8(c).
"""
import itertools
import os
from fractions import Fraction

import numpy as np
import pytest

from paper_1003_3779_b200 import inputs as qi

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")
OPEN, PERIODIC = qi.OPEN, qi.PERIODIC

DIR1 = {0: (+1,), 1: (-1,)}
DIR2_NAT = {0: (0, +1), 1: (+1, 0), 2: (-1, 0), 3: (0, -1)}      # PAPER.md:88 eq. 8 with c = 2j+k
DIR2_DIAG = {0: (+1, +1), 1: (+1, -1), 2: (-1, +1), 3: (-1, -1)}  # PAPER.md:106 Fig. 1c


def eq8_direction(j, k):
    """PAPER.md:88 eq. 8 literally: (dm, dn) = ((-1)^j (1 - delta_jk), (-1)^j delta_jk)."""
    d = 1 if j == k else 0
    return ((-1) ** j * (1 - d), (-1) ** j * d)


def test_direction_table_is_eq8():
    for j in (0, 1):
        for k in (0, 1):
            assert DIR2_NAT[2 * j + k] == eq8_direction(j, k)


# ------------------------------------------------------------------ helpers (independent of oracle)
def delta_state(extents, site, coin_vec, batch=1):
    sites = int(np.prod(extents))
    psi = np.zeros((batch, sites, len(coin_vec)), dtype=np.complex128)
    psi[:, int(np.ravel_multi_index(site, extents)), :] = coin_vec
    return psi


def path_sum_amplitudes(int_coin, start_vec, dirs, t):
    """Exact sum over all coin sequences a_1..a_t of prod C[a_i][a_{i-1}] * psi0[a_0].

    int_coin / start_vec hold Gaussian integers as Python complex with integer parts (exact in
    floating point for these sizes).  Returns {(site..., coin): Gaussian integer}.
    """
    cd = len(start_vec)
    out = {}
    for a0 in range(cd):
        if start_vec[a0] == 0:
            continue
        for seq in itertools.product(range(cd), repeat=t):
            amp = start_vec[a0]
            prev = a0
            pos = [0] * len(dirs[0])
            for a in seq:
                amp = amp * int_coin[a][prev]
                if amp == 0:
                    break
                for d in range(len(pos)):
                    pos[d] += dirs[a][d]
                prev = a
            if amp != 0:
                key = tuple(pos) + (prev,)
                out[key] = out.get(key, 0) + amp
    return out


def kron_unitary(extents, coins, dirs, boundary, broken=None):
    """U = S (I (x) C) as explicit Kronecker products (eq. 2 with eq. 8 for S).

    Basis order |site> (x) |coin>, site = m*en + n.  coins: (cd,cd) or (sites,cd,cd).
    Periodic: S = sum_a P_a (x) |a><a| with P_a the cyclic site shift by d_a.
    Open / broken links: S = sum_a [T_a (x) |a><a| + B_a (x) |opp(a)><a|] where T_a moves the
    sites whose a-link is intact and B_a projects on those whose a-link is broken/outward
    (eqs. 9-10).
    """
    dim = len(extents)
    cd = 2 * dim
    sites = int(np.prod(extents))

    def shift1(n, d):
        if boundary == PERIODIC:
            return np.roll(np.eye(n), d, axis=0)          # P[y,x] = 1 iff y = x + d mod n
        return np.eye(n, k=-d)                            # T[y,x] = 1 iff y = x + d inside

    coins = np.asarray(coins, dtype=np.complex128)
    if coins.ndim == 2:
        IC = np.kron(np.eye(sites), coins)
    else:
        IC = np.zeros((sites * cd, sites * cd), dtype=np.complex128)
        for x in range(sites):
            IC[x * cd:(x + 1) * cd, x * cd:(x + 1) * cd] = coins[x]
    S = np.zeros((sites * cd, sites * cd))
    for a in range(cd):
        if dim == 1:
            T = shift1(extents[0], dirs[a][0])
        else:
            T = np.kron(shift1(extents[0], dirs[a][0]), shift1(extents[1], dirs[a][1]))
        if broken is not None:
            T = T @ np.diag(1.0 - broken[:, a].astype(np.float64))
        B = np.eye(sites) - T.T @ T                      # sites whose a-component has nowhere to go
        Ea = np.zeros((cd, cd)); Ea[a, a] = 1.0
        Eo = np.zeros((cd, cd)); Eo[cd - 1 - a, a] = 1.0
        S += np.kron(T, Ea) + np.kron(B, Eo)
    return S @ IC


def spectral_evolve(extents, coin, dirs, psi0, t):
    """Periodic lattice + uniform coin: psi^(k,t) = (D(k) C)^t psi^(k,0), D = diag(e^{-2 pi i k.d_a/N})."""
    dim = len(extents)
    cd = 2 * dim
    psi = psi0.reshape(tuple(extents) + (cd,))
    axes = tuple(range(dim))
    hat = np.fft.fftn(psi, axes=axes)
    ks = np.meshgrid(*[np.arange(e) for e in extents], indexing="ij")
    M = np.empty(tuple(extents) + (cd, cd), dtype=np.complex128)
    for a in range(cd):
        phase = sum(ks[d] * dirs[a][d] / extents[d] for d in range(dim))
        M[..., a, :] = np.exp(-2j * np.pi * phase)[..., None] * coin[a, :]
    Mt = np.linalg.matrix_power(M, t)
    hat = np.einsum("...ab,...b->...a", Mt, hat)
    return np.fft.ifftn(hat, axes=axes).reshape(-1, cd)


def read_golden(name):
    rows = []
    with open(os.path.join(GOLDEN, name)) as f:
        for line in f:
            line = line.strip()
            if line and not line.startswith("#"):
                rows.append(line.split())
    return rows


# ------------------------------------------------------------------ P1 / P2 Hadamard first steps
INT_H = [[1, 1], [1, -1]]


@pytest.mark.parametrize("start,vec,int_vec,pre", [
    ("sym", None, [1j, 1], 1),       # (i,1)/sqrt2: one extra factor 1/sqrt2
    ("R", [1.0, 0.0], [1, 0], 0),
])
def test_p1_p2_hadamard_golden_and_path_sums(oracle, start, vec, int_vec, pre):
    s = qi.SQRT_HALF_F64
    if vec is None:
        vec = [1j * s, s]
    half = 8
    ext = (2 * half + 1,)
    golden = {}
    for row in read_golden("hadamard_first_steps.txt"):
        if row[0] == start:
            golden.setdefault(int(row[1]), {})[int(row[2])] = Fraction(int(row[3]), int(row[4]))
    for t in range(0, 8):
        psi = delta_state(ext, (half,), vec)
        oracle.step(ext, qi.hadamard(), psi, t, boundary=OPEN)
        P = oracle.probabilities(ext, psi)[0]
        # exact path sum: amplitude * sqrt2^(t+pre) is a Gaussian integer
        amps = path_sum_amplitudes(INT_H, int_vec, DIR1, t)
        exact = {}
        for (x, a), g in amps.items():
            exact[x] = exact.get(x, 0) + Fraction(int(round(abs(g) ** 2)), 2 ** (t + pre))
        assert sum(exact.values()) == 1
        for x in range(-half, half + 1):
            want = float(exact.get(x, Fraction(0)))
            assert abs(P[x + half] - want) <= 4e-16 * max(1, t), (t, x)
            if want == 0.0:
                assert P[x + half] == 0.0                      # P4: exact zeros
        if t in golden:
            assert {x: p for x, p in exact.items() if p != 0} == golden[t]
        # amplitudes too, not only probabilities
        for (x, a), g in amps.items():
            want = g * s ** (t + pre)
            assert abs(psi[0, x + half, a] - want) <= 1e-15


def test_p1_first_amplitudes(oracle):
    """t=1: R component at x=+1 is (1+i)/2, L component at x=-1 is (-1+i)/2 (hand derivation)."""
    s = qi.SQRT_HALF_F64
    psi = delta_state((5,), (2,), [1j * s, s])
    oracle.step((5,), qi.hadamard(), psi, 1, boundary=OPEN)
    assert abs(psi[0, 3, 0] - (1 + 1j) / 2) < 1e-15 and abs(psi[0, 1, 1] - (-1 + 1j) / 2) < 1e-15
    assert np.count_nonzero(psi) == 2


def test_p2_mirror_start(oracle):
    ext = (41,)
    a = delta_state(ext, (20,), [1.0, 0.0]); oracle.step(ext, qi.hadamard(), a, 15, boundary=OPEN)
    b = delta_state(ext, (20,), [0.0, 1.0]); oracle.step(ext, qi.hadamard(), b, 15, boundary=OPEN)
    Pa, Pb = oracle.probabilities(ext, a)[0], oracle.probabilities(ext, b)[0]
    assert np.max(np.abs(Pa - Pb[::-1])) < 1e-15
    assert oracle.moments(ext, a)[0, 1] > 0 > oracle.moments(ext, b)[0, 1]   # R start drifts right


# ------------------------------------------------------------------ P3/P4/P5/P8 on config 0
def test_p3_p4_p5_p8_k0(oracle):
    w = qi.k0()
    psi = w.initial_state()
    oracle.step(w.extents, w.coin, psi, w.steps, boundary=w.boundary)
    P = oracle.probabilities(w.extents, psi)[0]
    norm, mean, var = oracle.moments(w.extents, psi)[0]
    t = w.steps
    # P3: coin entries are fl(1/sqrt2), so U is unitary only to ~1.4e-16 per step (R23)
    assert abs(norm - 1.0) <= 1e-14 + 2e-16 * t
    assert abs(P.sum() - norm) < 1e-15
    # P4: support on parity-t sites within [-t, t]; outermost probability 2^-t exactly
    x = np.arange(-100, 101)
    assert np.all(P[(x + t) % 2 == 1] == 0.0)
    assert abs(P[0] / 2.0 ** -t - 1) < 1e-12 and abs(P[-1] / 2.0 ** -t - 1) < 1e-12
    # P5: left/right symmetry of the (i|R>+|L>)/sqrt2 start
    assert np.max(np.abs(P - P[::-1])) <= 1e-15
    assert abs(mean) <= 1e-13
    # P8: ballistic spreading, var/t^2 -> 1 - 1/sqrt2 (Nayak & Vishwanath, ref. [9] of the paper)
    assert abs(var / t ** 2 - (1 - 1 / np.sqrt(2))) < 1e-3
    assert abs(var - 2929.422331) < 1e-5       # SURVEY.md 8(c) P8 [scratch], re-derived by spectral test below


def test_p4_light_cone_2d(oracle):
    """PAPER.md:210 eq. 18: after i steps the walker is inside the (2i+1)^2 square; in fact inside
    the diamond |m|+|n| <= i on sites with (m+n+i) even, and those zeros are exact."""
    w = qi.k2(half=12, steps=9)
    psi = w.initial_state()
    oracle.step(w.extents, w.coin, psi, w.steps, boundary=w.boundary)
    P = oracle.probabilities(w.extents, psi)[0].reshape(w.extents)
    m, n = np.meshgrid(np.arange(-12, 13), np.arange(-12, 13), indexing="ij")
    outside = (np.abs(m) + np.abs(n) > 9) | ((m + n + 9) % 2 == 1)
    assert np.all(P[outside] == 0.0) and np.all(P[~outside] >= 0)
    assert abs(P.sum() - 1) < 1e-14


# ------------------------------------------------------------------ P6 reversibility
@pytest.mark.parametrize("boundary", [OPEN, PERIODIC])
@pytest.mark.parametrize("dim", [1, 2])
def test_p6_reversibility(oracle, boundary, dim):
    rng = np.random.default_rng(5)
    ext = (23,) if dim == 1 else (7, 6)
    sites = int(np.prod(ext))
    coin = qi.random_unitary(rng, 2 * dim)
    psi0 = qi.random_state(11, 1, sites, 2 * dim)
    psi = psi0.copy()
    oracle.step(ext, coin, psi, 100, boundary=boundary)
    assert np.max(np.abs(psi - psi0)) > 1e-3
    oracle.step_inverse(ext, coin, psi, 100, boundary=boundary)
    assert np.max(np.abs(psi - psi0)) <= 1e-13


# ------------------------------------------------------------------ P7 dense brute force
@pytest.mark.parametrize("boundary", [OPEN, PERIODIC])
@pytest.mark.parametrize("case", ["1d-hadamard", "1d-su2-per-site", "2d-grover", "2d-hxh", "2d-dft",
                                  "2d-random", "2d-diag-dft", "1d-n1", "1d-n2", "2d-1x5", "2d-2x2"])
def test_p7_dense_kronecker(oracle, boundary, case):
    rng = np.random.default_rng(7)
    lattice, dirs, coin_mode = qi.NATURAL, None, qi.COIN_UNIFORM
    if case == "1d-hadamard":
        ext, coin = (64,), qi.hadamard()
    elif case == "1d-su2-per-site":
        ext = (17,)
        ang = rng.uniform(0, 2 * np.pi, (1, 3)); phi = rng.uniform(0, 2 * np.pi, (1, 17))
        coin = qi.site_coin_matrices(qi.su2(ang[:, 0], ang[:, 1], ang[:, 2]), np.exp(1j * phi))[0]
        coin_mode = qi.COIN_PER_SITE
    elif case == "1d-n1":
        ext, coin = (1,), qi.random_unitary(rng, 2)
    elif case == "1d-n2":
        ext, coin = (2,), qi.random_unitary(rng, 2)
    elif case == "2d-1x5":
        ext, coin = (1, 5), qi.random_unitary(rng, 4)
    elif case == "2d-2x2":
        ext, coin = (2, 2), qi.random_unitary(rng, 4)
    elif case == "2d-diag-dft":
        ext, coin, lattice = (6, 5), qi.dft4(), qi.DIAGONAL
    else:
        ext = (8, 8) if case != "2d-random" else (5, 7)
        coin = {"2d-grover": qi.grover4, "2d-hxh": qi.hadamard_x_hadamard, "2d-dft": qi.dft4,
                "2d-random": lambda: qi.random_unitary(rng, 4)}[case]()
    dim = len(ext)
    if dirs is None:
        dirs = DIR1 if dim == 1 else (DIR2_DIAG if lattice == qi.DIAGONAL else DIR2_NAT)
    U_ref = kron_unitary(ext, coin, dirs, boundary)
    D = U_ref.shape[0]
    assert np.max(np.abs(U_ref.conj().T @ U_ref - np.eye(D))) <= 1e-14       # U is unitary
    U = oracle.dense_unitary(ext, coin, boundary=boundary, coin_mode=coin_mode, lattice=lattice)
    assert np.max(np.abs(U - U_ref)) <= 1e-15
    # stepper vs U^t psi0
    psi0 = qi.random_state(3, 1, D // (2 * dim), 2 * dim)
    psi = psi0.copy()
    oracle.step(ext, coin, psi, 25, boundary=boundary, coin_mode=coin_mode, lattice=lattice)
    want = np.linalg.matrix_power(U_ref, 25) @ psi0.reshape(-1)
    assert np.max(np.abs(psi.reshape(-1) - want)) <= 1e-13
    # inverse step vs U^dagger
    back = psi0.copy()
    oracle.step_inverse(ext, coin, back, 3, boundary=boundary, coin_mode=coin_mode, lattice=lattice)
    want = np.linalg.matrix_power(U_ref.conj().T, 3) @ psi0.reshape(-1)
    assert np.max(np.abs(back.reshape(-1) - want)) <= 1e-13


@pytest.mark.parametrize("dim,lattice", [(1, qi.NATURAL), (2, qi.NATURAL), (2, qi.DIAGONAL)])
@pytest.mark.parametrize("boundary", [OPEN, PERIODIC])
def test_p7_dense_broken_links(oracle, dim, lattice, boundary):
    """Static random broken links (eqs. 9-10) against the Kronecker form."""
    rng = np.random.default_rng(9)
    ext = (19,) if dim == 1 else (5, 6)
    dirs = DIR1 if dim == 1 else (DIR2_DIAG if lattice == qi.DIAGONAL else DIR2_NAT)
    coin = qi.random_unitary(rng, 2 * dim)
    mask = qi.symmetric_broken_links(qi.SEED_RBL, dim, ext, 1, 0.3, boundary, lattice)
    assert mask.any()
    U_ref = kron_unitary(ext, coin, dirs, boundary, broken=mask[0])
    D = U_ref.shape[0]
    assert np.max(np.abs(U_ref.conj().T @ U_ref - np.eye(D))) <= 1e-14
    U = oracle.dense_unitary(ext, coin, boundary=boundary, lattice=lattice, broken=mask)
    assert np.max(np.abs(U - U_ref)) <= 1e-15
    psi0 = qi.random_state(4, 1, int(np.prod(ext)), 2 * dim)
    psi = psi0.copy()
    oracle.step(ext, coin, psi, 9, boundary=boundary, lattice=lattice, broken=mask)
    assert np.max(np.abs(psi.reshape(-1) - np.linalg.matrix_power(U_ref, 9) @ psi0.reshape(-1))) <= 1e-13
    oracle.step_inverse(ext, coin, psi, 9, boundary=boundary, lattice=lattice, broken=mask)
    assert np.max(np.abs(psi - psi0)) <= 1e-13


# ------------------------------------------------------------------ P9 spectral closed form (FFT)
@pytest.mark.parametrize("case", ["1d-su2", "1d-hadamard", "2d-dft", "2d-grover", "2d-hxh-rect",
                                  "2d-diag-grover"])
def test_p9_spectral(oracle, case):
    rng = np.random.default_rng(13)
    lattice = qi.NATURAL
    if case == "1d-su2":
        ext, t = (256,), 300
        a = rng.uniform(0, 2 * np.pi, 3); coin = qi.su2(a[0], a[1], a[2])
    elif case == "1d-hadamard":
        ext, t, coin = (250,), 400, qi.hadamard()
    elif case == "2d-dft":
        ext, t, coin = (16, 16), 40, qi.dft4()
    elif case == "2d-grover":
        ext, t, coin = (12, 20), 33, qi.grover4()
    elif case == "2d-hxh-rect":
        ext, t, coin = (9, 14), 21, qi.hadamard_x_hadamard()
    else:
        ext, t, coin, lattice = (10, 15), 17, qi.grover4(), qi.DIAGONAL
    dim = len(ext)
    dirs = DIR1 if dim == 1 else (DIR2_DIAG if lattice == qi.DIAGONAL else DIR2_NAT)
    psi0 = qi.random_state(17, 1, int(np.prod(ext)), 2 * dim)
    psi = psi0.copy()
    oracle.step(ext, coin, psi, t, boundary=PERIODIC, lattice=lattice)
    want = spectral_evolve(ext, coin, dirs, psi0[0], t)
    assert np.max(np.abs(psi[0] - want)) <= 1e-13


def test_p8_p11_long_time_values_by_spectral(oracle):
    """Long-time numbers quoted in SURVEY.md 8(c) (P2, P8, P11) re-derived with the FFT closed form
    on a ring/torus large enough that nothing wraps, then compared with the oracle."""
    s = qi.SQRT_HALF_F64
    # 1D, t=100, 256-ring (no wrap: support |x| <= 100)
    ext = (256,)
    for vec, mean_want, var_want in [([1j * s, s], 0.0, 2929.422331), ([1.0, 0.0], 28.9755601564, 2089.8392444184)]:
        psi0 = delta_state(ext, (128,), vec)
        want = spectral_evolve(ext, qi.hadamard(), DIR1, psi0[0], 100)
        psi = psi0.copy(); oracle.step(ext, qi.hadamard(), psi, 100, boundary=PERIODIC)
        assert np.max(np.abs(psi[0] - want)) < 1e-13
        Pw = (np.abs(want) ** 2).sum(axis=1); x = np.arange(256) - 128
        mean = (x * Pw).sum() / Pw.sum(); var = (x * x * Pw).sum() / Pw.sum() - mean ** 2
        assert abs(mean - mean_want) < 1e-8 and abs(var - var_want) < 1e-5
        nrm, m_o, v_o = oracle.moments(ext, psi)[0]
        assert abs(m_o - mean) < 1e-10 and abs(v_o - var) < 1e-8
    # 2D Grover, t=20, 48x48 torus
    ext = (48, 48)
    psi0 = delta_state(ext, (24, 24), [0.5, -0.5, -0.5, 0.5])
    want = spectral_evolve(ext, qi.grover4(), DIR2_NAT, psi0[0], 20)
    psi = psi0.copy(); oracle.step(ext, qi.grover4(), psi, 20, boundary=PERIODIC)
    assert np.max(np.abs(psi[0] - want)) < 1e-13
    P = (np.abs(want) ** 2).sum(axis=1).reshape(ext)
    assert abs(P[24, 24] - 9.169430122711e-4) < 1e-14          # spreading (non-localised) walk
    m = np.arange(48) - 24
    assert abs((m[:, None] ** 2 * P).sum() - 73.16169133526) < 1e-9
    mo = oracle.moments(ext, psi)[0]
    assert abs(mo[3] - 73.16169133526) < 1e-9 and abs(mo[4] - 73.16169133526) < 1e-9 and abs(mo[5]) < 1e-12


# ------------------------------------------------------------------ P10 degenerate coins
def test_p10_degenerate_coins(oracle):
    ext = (41,)
    # beta = 0: diagonal coin, |L> keeps moving left with unit probability; then bounces off the wall
    coin = qi.su2(0.3, 0.0, 1.1)
    for t, site, comp in [(5, 15, 1), (20, 0, 1), (21, 0, 0), (25, 4, 0)]:
        psi = delta_state(ext, (20,), [0.0, 1.0])
        oracle.step(ext, coin, psi, t, boundary=OPEN)
        P = oracle.probabilities(ext, psi)[0]
        assert abs(P[site] - 1.0) < 1e-14 and abs(abs(psi[0, site, comp]) - 1.0) < 1e-14, (t, site)
    # beta = pi: anti-diagonal coin, walker alternates between x=+1 (odd t) and x=0 (even t)
    coin = qi.su2(0.7, np.pi, 0.2)
    for t in range(1, 8):
        psi = delta_state(ext, (20,), [0.0, 1.0])
        oracle.step(ext, coin, psi, t, boundary=OPEN)
        P = oracle.probabilities(ext, psi)[0]
        assert abs(P[20 + (t % 2)] - 1.0) < 1e-14


# ------------------------------------------------------------------ P11 Grover first steps
def test_p11_grover_golden_and_path_sums(oracle):
    int_G = [[-1, 1, 1, 1], [1, -1, 1, 1], [1, 1, -1, 1], [1, 1, 1, -1]]      # 2*G
    golden = {}
    for row in read_golden("grover_first_steps.txt"):
        golden.setdefault(int(row[0]), {})[(int(row[1]), int(row[2]))] = Fraction(int(row[3]), int(row[4]))
    half = 6
    ext = (2 * half + 1, 2 * half + 1)
    for t in range(0, 6):
        psi = delta_state(ext, (half, half), [0.5, -0.5, -0.5, 0.5])
        oracle.step(ext, qi.grover4(), psi, t, boundary=OPEN)
        P = oracle.probabilities(ext, psi)[0].reshape(ext)
        amps = path_sum_amplitudes(int_G, [1, -1, -1, 1], DIR2_NAT, t)   # amplitude * 2^(t+1)
        exact = {}
        for (m, n, a), g in amps.items():
            exact[(m, n)] = exact.get((m, n), 0) + Fraction(int(round(abs(g) ** 2)), 4 ** (t + 1))
            assert abs(psi[0, (m + half) * ext[1] + n + half, a] - g / 2.0 ** (t + 1)) <= 1e-16
        exact = {k: v for k, v in exact.items() if v != 0}
        assert sum(exact.values()) == 1
        for m in range(-half, half + 1):
            for n in range(-half, half + 1):
                assert abs(P[m + half, n + half] - float(exact.get((m, n), 0))) <= 1e-16
        if t in golden:
            assert exact == golden[t]
        # symmetric under m->-m, n->-n, m<->n
        assert np.array_equal(P, P[::-1, :]) and np.array_equal(P, P[:, ::-1]) and np.array_equal(P, P.T)


# ------------------------------------------------------------------ P12 translation covariance
@pytest.mark.parametrize("dim", [1, 2])
def test_p12_translation_covariance_bit_exact(oracle, dim):
    rng = np.random.default_rng(21)
    ext = (50,) if dim == 1 else (9, 11)
    coin = qi.random_unitary(rng, 2 * dim)
    psi0 = qi.random_state(23, 1, int(np.prod(ext)), 2 * dim)
    a = psi0.copy(); oracle.step(ext, coin, a, 30, boundary=PERIODIC)
    shift = (7,) if dim == 1 else (4, 3)
    b = np.roll(psi0.reshape(ext + (2 * dim,)), shift, axis=tuple(range(dim))).reshape(psi0.shape).copy()
    oracle.step(ext, coin, b, 30, boundary=PERIODIC)
    a_shift = np.roll(a.reshape(ext + (2 * dim,)), shift, axis=tuple(range(dim))).reshape(psi0.shape)
    assert np.array_equal(a_shift, b)


# ------------------------------------------------------------------ P15 coin modes reduce to one another
def test_p15_per_walk_and_per_site_reduce_to_uniform(oracle):
    w = qi.k0()
    base = w.initial_state(); oracle.step(w.extents, w.coin, base, w.steps, boundary=OPEN)
    B = 3
    psi = np.repeat(w.initial_state(), B, axis=0).copy()
    oracle.step(w.extents, np.broadcast_to(w.coin, (B, 2, 2)).copy(), psi, w.steps, boundary=OPEN,
                coin_mode=qi.COIN_PER_WALK, batch=B)
    for b in range(B):
        assert np.array_equal(psi[b], base[0])
    psi = np.repeat(w.initial_state(), B, axis=0).copy()
    oracle.step(w.extents, np.broadcast_to(w.coin, (B, w.sites, 2, 2)).copy(), psi, w.steps,
                boundary=OPEN, coin_mode=qi.COIN_PER_SITE, batch=B)
    for b in range(B):
        assert np.array_equal(psi[b], base[0])


def test_batch_walks_are_independent(oracle):
    w = qi.k4(batch=4, half=16)
    mode, coin = w.general_coin_f64()
    psi = w.initial_state(); oracle.step(w.extents, coin, psi, w.steps, boundary=OPEN, coin_mode=mode, batch=4)
    for b in range(4):
        one = w.initial_state()[b:b + 1].copy()
        oracle.step(w.extents, coin[b:b + 1], one, w.steps, boundary=OPEN, coin_mode=mode, batch=1)
        assert np.array_equal(one[0], psi[b])
    nrm = oracle.moments(w.extents, psi, batch=4)[:, 0]
    assert np.max(np.abs(nrm - 1)) < 1e-13


# ------------------------------------------------------------------ moments / probabilities vs textbook closed forms
def test_moments_closed_forms(oracle):
    # point mass: mean = coordinate, variance 0 (coordinates x = index - floor(N/2))
    ext = (201,)
    psi = delta_state(ext, (130,), [0.6, 0.8j])
    assert np.allclose(oracle.moments(ext, psi)[0], [1.0, 30.0, 0.0], atol=1e-12)
    # two point masses with weights 1/4, 3/4 at x=-10, +30: mean 20, var = E[x^2]-400 = 25+675-400
    psi = np.zeros((1, 201, 2), dtype=np.complex128)
    psi[0, 90, 0] = 0.5; psi[0, 130, 1] = np.sqrt(0.75) * 1j
    assert np.allclose(oracle.moments(ext, psi)[0], [1.0, 20.0, 300.0], atol=1e-10)
    # un-normalised input: moments are divided by the norm
    assert np.allclose(oracle.moments(ext, 3.0 * psi)[0], [9.0, 20.0, 300.0], atol=1e-9)
    # uniform distribution on N sites: variance (N^2-1)/12; mean -1/2 for even N, 0 for odd N
    for N in (64, 65):
        psi = np.full((1, N, 2), 1 / np.sqrt(2 * N), dtype=np.complex128)
        nrm, mean, var = oracle.moments((N,), psi)[0]
        assert abs(nrm - 1) < 1e-14 and abs(mean - (-0.5 if N % 2 == 0 else 0.0)) < 1e-12
        assert abs(var - (N * N - 1) / 12.0) < 1e-9
    # 2D: product of independent uniform (rows) and two-point (columns) marginals; covariance of a
    # perfectly correlated pair
    ext = (4, 6)
    psi = np.zeros((1, 24, 4), dtype=np.complex128)
    psi[0, 0 * 6 + 1, 2] = np.sqrt(0.5); psi[0, 3 * 6 + 5, 0] = np.sqrt(0.5)   # (m,n) = (-2,-2), (1,2)
    mo = oracle.moments(ext, psi)[0]
    assert np.allclose(mo, [1.0, -0.5, 0.0, 2.25, 4.0, 3.0], atol=1e-12)
    P = oracle.probabilities(ext, psi)[0]
    assert P[1] == 0.5000000000000001 or abs(P[1] - 0.5) < 1e-15
    assert P.sum() == pytest.approx(1.0, abs=1e-15)


def test_probabilities_marginalise_over_coin(oracle):
    psi = qi.random_state(31, 2, 10, 4)
    P = oracle.probabilities((2, 5), psi, batch=2)
    for w in range(2):
        for x in range(10):
            want = sum(psi[w, x, a].real ** 2 + psi[w, x, a].imag ** 2 for a in range(4))
            assert abs(P[w, x] - want) <= 1e-17


def test_probabilities_mean_is_the_batch_average(oracle):
    """Pin of qwo_probabilities_mean (the ensemble average of the broken-links model): numpy's mean over
    the walks of |psi|^2 summed over the coin (another routine, another order); closed forms: identical walks average to
    the single walk, B delta states on B different sites give 1/B on each of them; the mean of normalised walks sums to 1."""
    psi = qi.random_state(33, 5, 12, 4, normalise_per_walk=True)
    got = oracle.probabilities_mean((3, 4), psi, batch=5)
    want = np.mean(np.sum(psi.real ** 2 + psi.imag ** 2, axis=2), axis=0)
    assert got.shape == (12,) and np.max(np.abs(got - want)) <= 1e-17
    assert abs(np.sum(got) - 1.0) <= 1e-15
    one = qi.random_state(34, 1, 9, 2)
    rep = np.ascontiguousarray(np.repeat(one, 4, axis=0))
    assert np.array_equal(oracle.probabilities_mean((9,), rep, batch=4), oracle.probabilities((9,), one)[0])
    d = np.zeros((3, 7, 2), dtype=np.complex128)
    for w, x in enumerate((1, 4, 6)):
        d[w, x, w % 2] = 1j
    got = oracle.probabilities_mean((7,), d, batch=3)
    want = np.zeros(7); want[[1, 4, 6]] = 1.0 / 3.0
    assert np.array_equal(got, want)
    # a dropped walk, a transposed axis or a missing division fails one of the above; so does the wrong normalisation:
    assert not np.allclose(got, np.sum(np.abs(d) ** 2, axis=(0, 2)))


def test_sqrt_half_bit_patterns():
    import struct
    assert struct.pack("<d", qi.SQRT_HALF_F64) == struct.pack("<Q", 0x3FE6A09E667F3BCD)
    assert qi.SQRT_HALF_F64 == np.sqrt(0.5)
    assert np.float32(qi.SQRT_HALF_F32) == np.float32(np.sqrt(np.float32(0.5)))
    for c in (qi.hadamard(), qi.grover4(), qi.hadamard_x_hadamard(), qi.dft4(), qi.su2(0.1, 0.2, 0.3)):
        assert np.max(np.abs(c.conj().T @ c - np.eye(len(c)))) < 3e-16
