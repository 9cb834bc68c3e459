"""Seeded synthetic inputs for the quantum-walk hot path.

This module holds NONE of the method's arithmetic: it only produces the bytes (coin
matrices, initial states, phase tables, link masks) that are handed, identically, to the
CUDA library and — in tests / bench baselines — to the independent oracle.  It imports
neither of them.

The paper uses no dataset: its workloads are lattices with closed-form or random initial
states, so every workload here is fully synthetic and the
five ``K*`` builders mirror BASELINE.json:configs[0..4] (recipe: DESIGN.md "Inputs").
"""
from __future__ import annotations

import dataclasses
import struct
from typing import Optional, Tuple

import numpy as np

# --- constants the paper names but never prints (readings R10-R13) -----
# double nearest to 1/sqrt(2) (what sqrt(0.5) returns) and its float counterpart, fixed as bits
SQRT_HALF_F64 = struct.unpack("<d", struct.pack("<Q", 0x3FE6A09E667F3BCD))[0]
SQRT_HALF_F32 = struct.unpack("<f", struct.pack("<I", 0x3F3504F3))[0]

PERIODIC, OPEN = 0, 1
NATURAL, DIAGONAL = 0, 1
COIN_UNIFORM, COIN_PER_WALK, COIN_PER_SITE = 0, 1, 2

SEED_K1 = 1003377901
SEED_K3 = 1003377903
SEED_K4 = 1003377904
SEED_RBL = 1003377905


def _sqrt_half(dtype) -> float:
    return SQRT_HALF_F32 if np.dtype(dtype) == np.complex64 else SQRT_HALF_F64


def hadamard(dtype=np.complex128) -> np.ndarray:
    """1D Hadamard coin s*[[1,1],[1,-1]] with the fixed bit pattern for s."""
    s = _sqrt_half(dtype)
    return (np.array([[1, 1], [1, -1]], dtype=np.float64) * s).astype(dtype)


def grover4(dtype=np.complex128) -> np.ndarray:
    """2D Grover coin 2/4*J - I (BASELINE.json:configs[2]); entries +-1/2 are exact."""
    return (0.5 * np.ones((4, 4)) - np.eye(4)).astype(dtype)


def hadamard_x_hadamard(dtype=np.complex128) -> np.ndarray:
    """H (x) H with c = 2j+k: C[(j,k)][(j',k')] = H[j][j'] H[k][k']; entries +-1/2 exact."""
    h = np.array([[1, 1], [1, -1]], dtype=np.float64)
    return (0.5 * np.kron(h, h)).astype(dtype)


def dft4(dtype=np.complex128) -> np.ndarray:
    """4x4 Fourier coin F[a][b] = 1/2 * i^(a*b) (omega = e^{+2 pi i/4}); entries exact."""
    tab = [1, 1j, -1, -1j]
    return np.array([[0.5 * tab[(a * b) % 4] for b in range(4)] for a in range(4)]).astype(dtype)


def su2(alpha, beta, gamma) -> np.ndarray:
    """R_z(alpha) R_y(beta) R_z(gamma); broadcasts over leading axes -> (..., 2, 2) complex128."""
    alpha, beta, gamma = (np.asarray(v, dtype=np.float64) for v in (alpha, beta, gamma))
    c, s = np.cos(beta / 2), np.sin(beta / 2)
    out = np.empty(alpha.shape + (2, 2), dtype=np.complex128)
    out[..., 0, 0] = np.exp(-0.5j * (alpha + gamma)) * c
    out[..., 0, 1] = -np.exp(-0.5j * (alpha - gamma)) * s
    out[..., 1, 0] = np.exp(+0.5j * (alpha - gamma)) * s
    out[..., 1, 1] = np.exp(+0.5j * (alpha + gamma)) * c
    return out


def random_unitary(rng: np.random.Generator, n: int) -> np.ndarray:
    """Haar-ish random n x n unitary (QR of a complex Gaussian) for tests of the general coin."""
    z = rng.standard_normal((n, n)) + 1j * rng.standard_normal((n, n))
    q, r = np.linalg.qr(z)
    return q * (np.diag(r) / np.abs(np.diag(r)))


def random_state(seed: int, batch: int, sites: int, coin_dim: int, dtype=np.complex128,
                 normalise_per_walk: bool = False) -> np.ndarray:
    """re/im i.i.d. N(0,1), normalised in double (long-double accumulation), then cast.

    Draw order ``standard_normal((batch*sites, coin_dim, 2))`` (last axis re, im).
    Returns AoS [batch][site][coin].
    """
    rng = np.random.default_rng(seed)
    raw = rng.standard_normal((batch * sites, coin_dim, 2))
    z = raw.view(np.complex128).reshape(batch, sites, coin_dim)
    if normalise_per_walk:
        nrm = np.sqrt(np.sum(np.abs(z.reshape(batch, -1)) ** 2, axis=1, dtype=np.longdouble))
        z = z / nrm.astype(np.float64)[:, None, None]
    else:
        nrm = np.sqrt(np.sum(raw * raw, dtype=np.longdouble))
        z = z / np.float64(nrm)
    return np.ascontiguousarray(z.astype(dtype))


def site_coin_matrices(coins: np.ndarray, phases: np.ndarray) -> np.ndarray:
    """Per-site matrices M[w][x] = phases[w][x] * coins[w] as plain complex128 products.

    This is input preparation for the consumer that takes fully general per-site coins
    (reading R14); the walk arithmetic itself lives elsewhere.
    """
    return np.ascontiguousarray(phases[:, :, None, None] * coins[:, None, :, :])


def symmetric_broken_links(seed: int, dim: int, extents, batch: int, p: float, boundary: int,
                           lattice: int = NATURAL) -> np.ndarray:
    """Static random broken links: Bernoulli(p) per undirected link.

    Returns a [batch][site][coin] uint8 mask in which both ends of a link carry the same bit.
    Only the natural 2D lattice and 1D are supported (a diagonal link is shared by the two
    diagonal neighbours in the same way).
    """
    rng = np.random.default_rng(seed)
    if dim == 1:
        n = int(extents[0])
        # link i joins site i and i+1 (mod n); coin 0 (R) of site i and coin 1 (L) of site i+1
        link = (rng.random((batch, n)) < p).astype(np.uint8)
        if boundary == OPEN:
            link[:, n - 1] = 0  # handled by the wall anyway
        mask = np.zeros((batch, n, 2), dtype=np.uint8)
        mask[:, :, 0] = link
        mask[:, :, 1] = np.roll(link, 1, axis=1)
        return mask
    em, en = int(extents[0]), int(extents[1])
    mask = np.zeros((batch, em, en, 4), dtype=np.uint8)
    if lattice == NATURAL:
        ln = (rng.random((batch, em, en)) < p).astype(np.uint8)  # link (m,n)-(m,n+1)
        lm = (rng.random((batch, em, en)) < p).astype(np.uint8)  # link (m,n)-(m+1,n)
        mask[..., 0] = ln
        mask[..., 3] = np.roll(ln, 1, axis=2)
        mask[..., 1] = lm
        mask[..., 2] = np.roll(lm, 1, axis=1)
    else:
        la = (rng.random((batch, em, en)) < p).astype(np.uint8)  # link (m,n)-(m+1,n+1)
        lb = (rng.random((batch, em, en)) < p).astype(np.uint8)  # link (m,n)-(m+1,n-1)
        mask[..., 0] = la
        mask[..., 3] = np.roll(la, (1, 1), axis=(1, 2))
        mask[..., 1] = lb
        mask[..., 2] = np.roll(lb, (1, -1), axis=(1, 2))
    return mask.reshape(batch, em * en, 4)


@dataclasses.dataclass
class Workload:
    """One synthetic configuration: everything both sides need, as plain arrays."""
    name: str
    dim: int
    extents: Tuple[int, ...]
    batch: int
    boundary: int
    dtype: np.dtype
    steps: int
    coin_mode: int
    coin: np.ndarray                       # (2d,2d) | (batch,2d,2d) | (batch,sites,2d,2d), in `dtype`
    phases: Optional[np.ndarray] = None    # (batch, sites) unit-modulus, in `dtype`
    delta_site: Optional[Tuple[int, ...]] = None
    delta_coin: Optional[np.ndarray] = None
    state: Optional[np.ndarray] = None     # AoS [batch][site][coin] in `dtype`
    lattice: int = NATURAL
    outputs: Tuple[str, ...] = ("probabilities",)

    @property
    def sites(self) -> int:
        return int(np.prod(self.extents))

    @property
    def coin_dim(self) -> int:
        return 2 * self.dim

    def initial_state(self) -> np.ndarray:
        """AoS initial state in the workload dtype (materialises the delta start)."""
        if self.state is not None:
            return self.state
        psi = np.zeros((self.batch, self.sites, self.coin_dim), dtype=self.dtype)
        idx = int(np.ravel_multi_index(self.delta_site, self.extents))
        psi[:, idx, :] = self.delta_coin
        return psi

    def general_coin_f64(self) -> Tuple[int, np.ndarray]:
        """(coin_mode, complex128 matrices) for a consumer without a phase table."""
        coin = np.asarray(self.coin).astype(np.complex128)
        if self.phases is None:
            return self.coin_mode, coin
        ph = np.asarray(self.phases).astype(np.complex128)
        if self.coin_mode == COIN_UNIFORM:
            coin = np.broadcast_to(coin, (self.batch, self.coin_dim, self.coin_dim))
        return COIN_PER_SITE, site_coin_matrices(coin, ph)


def k0(steps: int = 100, half_width: int = 100) -> Workload:
    """configs[0]: 1D Hadamard, open, sites -hw..hw, start |0>(x)(i|R>+|L>)/sqrt2."""
    s = SQRT_HALF_F64
    return Workload("K0", 1, (2 * half_width + 1,), 1, OPEN, np.dtype(np.complex128), steps,
                    COIN_UNIFORM, hadamard(), delta_site=(half_width,),
                    delta_coin=np.array([1j * s, s], dtype=np.complex128))


def k1(log2_sites: int = 26, steps: int = 1000, dtype=np.complex128, seed: int = SEED_K1,
       sites: Optional[int] = None) -> Workload:
    """configs[1]: 1D Hadamard ring, random normalised state; outputs norm/mean/variance."""
    n = sites if sites is not None else 1 << log2_sites
    return Workload("K1", 1, (n,), 1, PERIODIC, np.dtype(dtype), steps, COIN_UNIFORM,
                    hadamard(dtype), state=random_state(seed, 1, n, 2, dtype),
                    outputs=("moments",))


def k2(half: int = 2048, steps: Optional[int] = None) -> Workload:
    """configs[2]: 2D Grover, open (2*half+1)^2, delta at the centre, coin (1,-1,-1,1)/2."""
    e = 2 * half + 1
    return Workload("K2", 2, (e, e), 1, OPEN, np.dtype(np.complex128),
                    half if steps is None else steps, COIN_UNIFORM, grover4(),
                    delta_site=(half, half),
                    delta_coin=np.array([0.5, -0.5, -0.5, 0.5], dtype=np.complex128))


def k3(extent: int = 8192, steps: int = 500, coin: str = "hxh", seed: int = SEED_K3,
       extents: Optional[Tuple[int, int]] = None, dtype=np.complex64) -> Workload:
    """configs[3]: 2D torus, complex64, H(x)H or DFT coin, random normalised state."""
    ext = extents if extents is not None else (extent, extent)
    c = {"hxh": hadamard_x_hadamard, "dft": dft4, "grover": grover4}[coin](dtype)
    return Workload("K3-" + coin, 2, tuple(ext), 1, PERIODIC, np.dtype(dtype), steps,
                    COIN_UNIFORM, c, state=random_state(seed, 1, ext[0] * ext[1], 4, dtype),
                    outputs=("moments",))


def k4(batch: int = 4096, half: int = 1024, steps: Optional[int] = None, seed: int = SEED_K4) -> Workload:
    """configs[4]: batch of open 1D walks, per-walk SU(2) coin x per-site phase disorder."""
    n = 2 * half + 1
    rng = np.random.default_rng(seed)
    ang = rng.uniform(0.0, 2 * np.pi, (batch, 3))
    phi = rng.uniform(0.0, 2 * np.pi, (batch, n))
    return Workload("K4", 1, (n,), batch, OPEN, np.dtype(np.complex128),
                    half if steps is None else steps, COIN_PER_WALK,
                    su2(ang[:, 0], ang[:, 1], ang[:, 2]), phases=np.exp(1j * phi),
                    delta_site=(half,), delta_coin=np.array([0.0, 1.0], dtype=np.complex128),
                    outputs=("probabilities", "moments"))
