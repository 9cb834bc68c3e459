"""Pins for the oracle's random-broken-links walk ("random broken links (termed RBL)",
PAPER.md:92-102 eqs. 9-10; reading R27): links redrawn at every step from the
counter-based generator Philox4x32-10.  Nothing here runs on a GPU.

What fixes the oracle, other than itself:
  * the generator: the known-answer vectors distributed with the Random123 library
    (Salmon, Moraes, Dror, Shaw, SC'11) for philox4x32, 10 rounds;
  * the link function: both ends of every link must see the same state -> checked with numpy
    rolls that know nothing of the oracle's `target`, and through U(t)^dagger U(t) = I of the dense
    matrix built with the (already pinned, tests/test_oracle_pins.py::test_p7_dense_broken_links)
    static-mask path; broken fraction = p within binomial bounds; independence over steps / walks / seeds;
  * the walk: p = 0 is the plain walk, p = 1 freezes the walker (closed form), any p is the
    step-by-step composition of static-mask steps, and U^dagger undoes it.
"""
import numpy as np
import pytest

from paper_1003_3779_b200 import inputs as qi

OPEN, PERIODIC = qi.OPEN, qi.PERIODIC
DIR1 = {0: (0, +1), 1: (0, -1)}
DIR2_NAT = {0: (0, +1), 1: (+1, 0), 2: (-1, 0), 3: (0, -1)}       # PAPER.md:88 eq. 8, c = 2j+k
DIR2_DIAG = {0: (+1, +1), 1: (+1, -1), 2: (-1, +1), 3: (-1, -1)}   # PAPER.md:106 Fig. 1c

# Random123 known-answer vectors, philox4x32 with 10 rounds: (counter, key, expected)
PHILOX_KAT = [
    ((0x00000000, 0x00000000, 0x00000000, 0x00000000), (0x00000000, 0x00000000),
     (0x6627e8d5, 0xe169c58d, 0xbc57ac4c, 0x9b00dbd8)),
    ((0xffffffff, 0xffffffff, 0xffffffff, 0xffffffff), (0xffffffff, 0xffffffff),
     (0x408f276d, 0x41c83b0e, 0xa20bc7c6, 0x6d5451fd)),
    ((0x243f6a88, 0x85a308d3, 0x13198a2e, 0x03707344), (0xa4093822, 0x299f31d0),     # digits of pi
     (0xd16cfe09, 0x94fdcceb, 0x5001e420, 0x24126ea1)),
]


def dirs_of(dim, lattice):
    return DIR1 if dim == 1 else (DIR2_DIAG if lattice == qi.DIAGONAL else DIR2_NAT)


def grid(ext):
    return (1, ext[0]) if len(ext) == 1 else tuple(ext)


@pytest.mark.parametrize("ctr,key,want", PHILOX_KAT)
def test_philox4x32_10_known_answers(oracle, ctr, key, want):
    assert tuple(int(x) for x in oracle.philox4x32_10(ctr, key)) == want


@pytest.mark.parametrize("dim,lattice", [(1, qi.NATURAL), (2, qi.NATURAL), (2, qi.DIAGONAL)])
@pytest.mark.parametrize("boundary", [OPEN, PERIODIC])
@pytest.mark.parametrize("ext1,ext2", [((23,), (6, 9)), ((2,), (2, 3)), ((1,), (1, 4))])
def test_both_ends_of_a_link_agree(oracle, dim, lattice, boundary, ext1, ext2):
    """mask[x][a] == mask[x + d_a][opposite(a)] wherever the link stays inside the lattice."""
    ext = ext1 if dim == 1 else ext2
    em, en = grid(ext)
    dirs = dirs_of(dim, lattice)
    cd = 2 * dim
    for t in (0, 1, 7):
        mask = oracle.rbl_mask(ext, 0.5, 99, t, boundary=boundary, batch=2, lattice=lattice).reshape(2, em, en, cd)
        for a, (dm, dn) in dirs.items():
            # the far end's view of the same link, brought back to the near end
            far = np.roll(mask[..., cd - 1 - a], shift=(-dm, -dn), axis=(1, 2))
            inside = np.ones((em, en), dtype=bool)
            if boundary == OPEN:
                mm, nn = np.meshgrid(np.arange(em), np.arange(en), indexing="ij")
                inside = (mm + dm >= 0) & (mm + dm < em) & (nn + dn >= 0) & (nn + dn < en)
                assert not mask[:, ~inside, a].any()          # outward links are not marked (always broken)
            assert np.array_equal(mask[:, inside, a], far[:, inside]), (a, t)


@pytest.mark.parametrize("p", [0.0, 0.1, 0.5, 0.93, 1.0])
def test_broken_fraction_and_independence(oracle, p):
    ext = (64, 64)
    masks = [oracle.rbl_mask(ext, p, 2024, t, boundary=PERIODIC, batch=3) for t in range(4)]
    m = np.stack(masks).astype(np.float64)                     # [t][w][site][coin]
    n_links = m[..., :2].size                                  # coins 0 and 1 enumerate every link once
    frac = m[..., :2].mean()
    assert abs(frac - p) <= 5 * np.sqrt(max(p * (1 - p), 1e-12) / n_links) + (0 if 0 < p < 1 else 0)
    if 0 < p < 1:
        a = m[..., :2] - p
        var = p * (1 - p)
        tol = 6 / np.sqrt(a[0, 0].size)
        assert abs((a[0, 0] * a[1, 0]).mean() / var) <= tol    # step t vs step t+1
        assert abs((a[0, 0] * a[0, 1]).mean() / var) <= tol    # walk 0 vs walk 1
        assert abs((a[0, 0, :, 0] * a[0, 0, :, 1]).mean() / var) <= 6 / np.sqrt(a[0, 0, :, 0].size)   # the two axes
        other = oracle.rbl_mask(ext, p, 2025, 0, boundary=PERIODIC, batch=1).astype(np.float64)[0, :, :2] - p
        assert abs((a[0, 0] * other).mean() / var) <= tol      # another seed


@pytest.mark.parametrize("dim,lattice", [(1, qi.NATURAL), (2, qi.NATURAL), (2, qi.DIAGONAL)])
@pytest.mark.parametrize("boundary", [OPEN, PERIODIC])
def test_every_step_is_unitary_and_composes(oracle, dim, lattice, boundary):
    """U(t) built with the step-t mask is unitary; the RBL walk is the product U(t0+n-1) ... U(t0)."""
    rng = np.random.default_rng(21)
    ext = (17,) if dim == 1 else (4, 5)
    coin = qi.random_unitary(rng, 2 * dim)
    sites = int(np.prod(ext))
    psi0 = qi.random_state(8, 1, sites, 2 * dim)
    p, seed, t0, n = 0.35, 77, 3, 6
    want = psi0.reshape(-1).copy()
    step_by_step = psi0.copy()
    some_broken = False
    for t in range(t0, t0 + n):
        mask = oracle.rbl_mask(ext, p, seed, t, boundary=boundary, lattice=lattice)
        some_broken |= bool(mask.any())
        U = oracle.dense_unitary(ext, coin, boundary=boundary, lattice=lattice, broken=mask)
        assert np.max(np.abs(U.conj().T @ U - np.eye(U.shape[0]))) <= 1e-14, t
        want = U @ want
        oracle.step(ext, coin, step_by_step, 1, boundary=boundary, lattice=lattice, broken=mask)
    assert some_broken
    psi = psi0.copy()
    oracle.step_rbl(ext, coin, psi, n, p, seed, t0=t0, boundary=boundary, lattice=lattice)
    assert np.array_equal(psi, step_by_step)
    assert np.max(np.abs(psi.reshape(-1) - want)) <= 1e-13
    assert abs(np.sum(np.abs(psi) ** 2) - 1) <= 1e-14
    oracle.step_inverse_rbl(ext, coin, psi, n, p, seed, t0=t0 + n, boundary=boundary, lattice=lattice)
    assert np.max(np.abs(psi - psi0)) <= 1e-13


@pytest.mark.parametrize("dim", [1, 2])
def test_p0_is_the_plain_walk_and_p1_freezes_the_walker(oracle, dim):
    rng = np.random.default_rng(5)
    ext = (31,) if dim == 1 else (7, 8)
    cd = 2 * dim
    coin = qi.random_unitary(rng, cd)
    sites = int(np.prod(ext))
    psi0 = qi.random_state(3, 2, sites, cd, normalise_per_walk=True)
    a, b = psi0.copy(), psi0.copy()
    oracle.step(ext, coin, a, 12, boundary=PERIODIC, batch=2)
    oracle.step_rbl(ext, coin, b, 12, 0.0, 1234, boundary=PERIODIC, batch=2)
    assert np.array_equal(a, b)
    # p = 1: every link broken -> psi'[x][opposite(a)] = (C psi[x])[a]: the walker never leaves its site
    # and one step is the site-local unitary R C (R = coin reversal); t steps = (R C)^t, a closed form.
    c = psi0.copy()
    oracle.step_rbl(ext, coin, c, 5, 1.0, 1234, boundary=PERIODIC, batch=2)
    RC = coin[::-1, :]
    want = np.einsum("ab,wxb->wxa", np.linalg.matrix_power(RC, 5), psi0)
    assert np.max(np.abs(c - want)) <= 1e-14
    assert np.allclose(np.sum(np.abs(c) ** 2, axis=2), np.sum(np.abs(psi0) ** 2, axis=2), rtol=0, atol=1e-15)


@pytest.mark.parametrize("dim,lattice", [(1, 0), (2, 0), (2, 1)])
def test_link_states_are_the_documented_function_of_the_generator(oracle, dim, lattice):
    """Reading R27, written out: link number = owner * dim + axis, counter = (number // 4, 0, t, walk), key = seed,
    broken iff word[number % 4] < floor(p 2^32).  The mask the oracle's stepper uses must be exactly that function of
    the generator (which the known-answer vectors pin): a wrong word index, owner or axis fails here."""
    ext = (23,) if dim == 1 else (5, 7)
    em, en = (1, ext[0]) if dim == 1 else ext
    p, seed, t, batch = 0.37, 0x0123456789ABCDEF, 5, 2
    thr = int(p * 2 ** 32)
    key = [seed & 0xffffffff, seed >> 32]
    mask = oracle.rbl_mask(ext, p, seed, t, boundary=0, batch=batch, lattice=lattice).reshape(batch, em, en, 2 * dim)
    if dim == 1:
        dirs = [(0, 1), (0, -1)]
    elif lattice == 0:
        dirs = [(0, 1), (1, 0), (-1, 0), (0, -1)]            # PAPER.md:88 eq. 8, c = 2j + k
    else:
        dirs = [(1, 1), (1, -1), (-1, 1), (-1, -1)]          # PAPER.md:106 Fig. 1c
    for w in range(batch):
        for m in range(em):
            for n in range(en):
                for a, (dm, dn) in enumerate(dirs):
                    tm, tn = (m + dm) % em, (n + dn) % en
                    positive = dm > 0 or (dm == 0 and dn > 0)
                    owner = (m * en + n) if positive else (tm * en + tn)
                    axis = (0 if dm * dn > 0 else 1) if (dm != 0 and dn != 0) else (1 if dm != 0 else 0)
                    number = owner * dim + axis
                    word = oracle.philox4x32_10([number // 4, 0, t, w], key)[number % 4]
                    assert mask[w, m, n, a] == (1 if int(word) < thr else 0), (w, m, n, a)


def test_batch_members_and_start_times_are_addressed_by_the_counter(oracle):
    """Walk w of a batch sees the links of counter word 3 = w; starting at t0 sees those of steps t0, t0+1, ..."""
    rng = np.random.default_rng(6)
    ext = (40,)
    coin = qi.random_unitary(rng, 2)
    psi0 = qi.random_state(2, 1, 40, 2)
    both = np.concatenate([psi0, psi0]).copy()
    oracle.step_rbl(ext, coin, both, 9, 0.4, 5, boundary=OPEN, batch=2)
    assert not np.array_equal(both[0], both[1])                # different links per walk
    one = psi0.copy()
    oracle.step_rbl(ext, coin, one, 9, 0.4, 5, boundary=OPEN, batch=1)
    assert np.array_equal(one[0], both[0])
    split = psi0.copy()
    oracle.step_rbl(ext, coin, split, 4, 0.4, 5, t0=0, boundary=OPEN)
    oracle.step_rbl(ext, coin, split, 5, 0.4, 5, t0=4, boundary=OPEN)
    assert np.array_equal(split, one)


def test_rbl_decoherence_slows_the_hadamard_walk(oracle):
    """Ref. [12] of the paper (the source of the RBL technique): broken links turn the ballistic
    spreading (variance ~ t^2) into diffusive spreading.  Qualitative pin on the physics: at t = 100 the variance
    with p = 0.3 is far below the unbroken walk's 2929.4 (tests/test_oracle_pins.py P8) and the norm is conserved."""
    w = qi.k0()
    psi = w.initial_state().astype(np.complex128)
    oracle.step_rbl(w.extents, w.coin, psi, 100, 0.3, 11, boundary=OPEN)
    norm, mean, var = oracle.moments(w.extents, psi)[0]
    assert abs(norm - 1) <= 1e-13
    assert 20 < var < 1200
