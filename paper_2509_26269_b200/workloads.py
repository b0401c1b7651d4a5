"""Seeded synthetic inputs for the five BASELINE.json configs.

This module holds NONE of the method's arithmetic (no energy, gradient, Hessian,
eigen-solver or MMF formulas): it only builds lattices, initial spin textures and
atom positions as plain numpy arrays.  Those arrays are handed, unchanged, to both
the CUDA library and the CPU oracle (which share data, never code).  numpy/scipy
only -- it imports neither the CUDA binding nor ``oracle/``.

Recipes follow DESIGN.md "Input recipe" (SURVEY.md 8(c) readings A12-A15, A22):
  * triangular lattice, site i = iy*Lx + ix at r_i = ix*a1 + iy*a2,
    a1 = (1, 0), a2 = (1/2, sqrt(3)/2)
  * Neel skyrmion, helicity pi: m = (-sin(th) cos(ph), -sin(th) sin(ph), cos(th)),
    th(r) = 2 atan(R/r) exp(-r/(2R)), th(0) = pi   (BASELINE.json configs[1])
  * noise: m <- normalize(m + sigma*xi), xi ~ N(0, I3) iid, default_rng(seed), site order
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

A1 = np.array([1.0, 0.0])
A2 = np.array([0.5, np.sqrt(3.0) / 2.0])


@dataclass
class SpinWorkload:
    name: str
    Lx: int
    Ly: int
    pbc_x: int
    pbc_y: int
    J: float
    D: float
    K: float
    B: tuple  # (Bx, By, Bz)
    mu: float
    k: int
    seed: int
    spins: np.ndarray  # [N][3] float64, unit rows
    tol: float = 1e-8
    mmf_steps: int = 0
    dt: float = 0.05
    centres: np.ndarray | None = None

    @property
    def N(self) -> int:
        return self.Lx * self.Ly


@dataclass
class CartWorkload:
    name: str
    positions: np.ndarray  # [Na][3] float64, Angstrom
    fixed: np.ndarray  # [Na] uint8, 1 = frozen
    cell: np.ndarray  # [2][2] in-plane periodic cell vectors (rows), Angstrom
    De: float
    alpha: float
    r0: float
    rc: float
    k: int
    seed: int
    tol: float = 1e-8
    mmf_steps: int = 100
    dt: float = 0.05
    meta: dict = field(default_factory=dict)

    @property
    def Na(self) -> int:
        return self.positions.shape[0]


# --------------------------------------------------------------------------- lattice helpers
def site_positions(Lx: int, Ly: int) -> np.ndarray:
    """[N][2] Cartesian positions of the rhombic Lx x Ly triangular lattice."""
    ix = np.arange(Lx)[None, :]
    iy = np.arange(Ly)[:, None]
    x = ix * A1[0] + iy * A2[0]
    y = ix * A1[1] + iy * A2[1]
    return np.stack([np.broadcast_to(x, (Ly, Lx)), np.broadcast_to(y, (Ly, Lx))], axis=-1).reshape(-1, 2).astype(np.float64)


def _image_shifts(Lx: int, Ly: int, pbc_x: int, pbc_y: int) -> np.ndarray:
    sx = (-1, 0, 1) if pbc_x else (0,)
    sy = (-1, 0, 1) if pbc_y else (0,)
    return np.array([a * Lx * A1 + b * Ly * A2 for a in sx for b in sy])


def _normalize_rows(a: np.ndarray) -> np.ndarray:
    return a / np.linalg.norm(a, axis=1, keepdims=True)


def add_noise(spins: np.ndarray, sigma: float, rng: np.random.Generator) -> np.ndarray:
    if sigma == 0.0:
        return _normalize_rows(spins)
    xi = rng.standard_normal(spins.shape)
    return _normalize_rows(spins + sigma * xi)


def skyrmion_texture(Lx, Ly, pbc_x, pbc_y, centres_xy: np.ndarray, R: float) -> np.ndarray:
    """Nearest-centre rule (A14): every site takes (theta, phi) from its nearest centre
    (minimum image over the periodic directions)."""
    from scipy.spatial import cKDTree

    pos = site_positions(Lx, Ly)
    shifts = _image_shifts(Lx, Ly, pbc_x, pbc_y)
    imgs = (centres_xy[:, None, :] + shifts[None, :, :]).reshape(-1, 2)
    _, idx = cKDTree(imgs).query(pos, k=1)
    d = pos - imgs[idx]
    r = np.hypot(d[:, 0], d[:, 1])
    phi = np.arctan2(d[:, 1], d[:, 0])
    with np.errstate(divide="ignore"):
        theta = np.where(r > 0, 2.0 * np.arctan(R / np.where(r > 0, r, 1.0)) * np.exp(-r / (2.0 * R)), np.pi)
    st = np.sin(theta)
    m = np.stack([-st * np.cos(phi), -st * np.sin(phi), np.cos(theta)], axis=1)
    return _normalize_rows(m)


def _site_xy(ix: float, iy: float) -> np.ndarray:
    return ix * A1 + iy * A2


def _min_image_dist(p: np.ndarray, q: np.ndarray, shifts: np.ndarray) -> float:
    d = (p - q)[None, :] + shifts
    return float(np.min(np.hypot(d[:, 0], d[:, 1])))


# --------------------------------------------------------------------------- the five configs
_PARAMS = dict(J=1.0, D=0.3, K=0.05, mu=1.0)


def config0(seed: int = 1000, sigma: float = 0.1) -> SpinWorkload:
    """8x8 periodic, +z tilted by Gaussian noise sigma=0.1 (BASELINE.json configs[0])."""
    Lx = Ly = 8
    rng = np.random.default_rng(seed)
    m = np.zeros((Lx * Ly, 3))
    m[:, 2] = 1.0
    m = add_noise(m, sigma, rng)
    return SpinWorkload("cfg0_8x8_pbc", Lx, Ly, 1, 1, B=(0.0, 0.0, 0.02), k=2, seed=seed, spins=m, tol=1e-9, **_PARAMS)


def config1(seed: int = 1001, L: int = 70, R: float = 5.0, sigma: float = 0.02) -> SpinWorkload:
    """70x70 periodic, one Neel skyrmion R=5 at the lattice centre + noise (configs[1])."""
    rng = np.random.default_rng(seed)
    c = _site_xy(L // 2, L // 2)[None, :]
    m = skyrmion_texture(L, L, 1, 1, c, R)
    m = add_noise(m, sigma, rng)
    return SpinWorkload(f"cfg1_{L}x{L}_pbc_skyrmion", L, L, 1, 1, B=(0.0, 0.0, 0.02), k=2, seed=seed, spins=m,
                        tol=1e-9, centres=c, **_PARAMS)


def config2(seed: int = 1002, L: int = 256, R: float = 6.0, sep: float = 20.0) -> SpinWorkload:
    """256x256 open, two Neel skyrmions R=6, 20 sites apart at seeded positions (configs[2])."""
    rng = np.random.default_rng(seed)
    lo, hi = L // 4, 3 * L // 4
    c0 = _site_xy(rng.uniform(lo, hi), rng.uniform(lo, hi))
    psi = rng.uniform(0.0, 2.0 * np.pi)
    c1 = c0 + sep * np.array([np.cos(psi), np.sin(psi)])
    c = np.stack([c0, c1])
    m = skyrmion_texture(L, L, 0, 0, c, R)
    return SpinWorkload(f"cfg2_{L}x{L}_open_biskyrmion", L, L, 0, 0, B=(0.0, 0.0, 0.03), k=6, seed=seed, spins=m,
                        tol=1e-8, mmf_steps=100, dt=0.05, centres=c, **_PARAMS)


def config3(seed: int = 1003, L: int = 1000, n_sk: int = 200, R: float = 4.0, min_sep: float = 40.0,
            sigma: float = 0.01) -> SpinWorkload:
    """1000x1000 periodic, ~200 Neel skyrmions R=4 at seeded Poisson-disk positions + noise (configs[3]).
    Sequential dart throwing: uniform candidates in the cell, accepted when the minimum-image
    distance to every accepted centre is >= min_sep, until n_sk are placed (A15).
    Scaled-down instances keep the same density: n_sk ~ 200 * (L/1000)^2."""
    rng = np.random.default_rng(seed)
    shifts = _image_shifts(L, L, 1, 1)
    centres: list[np.ndarray] = []
    tries = 0
    while len(centres) < n_sk:
        tries += 1
        if tries > 200000:
            raise RuntimeError("dart throwing did not place all skyrmions")
        p = _site_xy(rng.uniform(0, L), rng.uniform(0, L))
        if all(_min_image_dist(p, q, shifts) >= min_sep for q in centres):
            centres.append(p)
    c = np.array(centres)
    m = skyrmion_texture(L, L, 1, 1, c, R)
    m = add_noise(m, sigma, rng)
    return SpinWorkload(f"cfg3_{L}x{L}_pbc_{n_sk}skyrmions", L, L, 1, 1, B=(0.0, 0.0, 0.02), k=2, seed=seed, spins=m,
                        tol=1e-6, mmf_steps=200, dt=0.05, centres=c, **_PARAMS)


def config3_scaled(L: int, seed: int = 1003) -> SpinWorkload:
    """Same-density scaled-down cfg 3 (L must be even), for oracle-sized parity cases."""
    n = max(1, int(round(200 * (L / 1000.0) ** 2)))
    return config3(seed=seed, L=L, n_sk=n)


def random_spins(Lx: int, Ly: int, seed: int) -> np.ndarray:
    """iid uniform directions on the sphere -- the paper's 'random spin configurations'."""
    rng = np.random.default_rng(seed)
    return _normalize_rows(rng.standard_normal((Lx * Ly, 3)))


def random_block(N: int, k: int, seed: int) -> np.ndarray:
    """[k][N][3] iid N(0,1) block of directions (not tangent, not orthonormal)."""
    rng = np.random.default_rng(seed)
    return rng.standard_normal((k, N, 3))


def config4(seed: int = 1004, nx: int = 20, ny: int = 20, layers: int = 4, a: float = 3.52,
            sigma: float = 0.05) -> CartWorkload:
    """fcc Ni(111) slab, 4 layers x 20x20 (bottom 2 fixed) + 7-atom heptamer on fcc hollows (configs[4], A22)."""
    rng = np.random.default_rng(seed)
    d = a / np.sqrt(2.0)
    dz = a / np.sqrt(3.0)
    a1 = d * np.array([1.0, 0.0])
    a2 = d * np.array([0.5, np.sqrt(3.0) / 2.0])
    shift = (a1 + a2) / 3.0
    pos = []
    fixed = []
    for l in range(layers):
        for iy in range(ny):
            for ix in range(nx):
                xy = ix * a1 + iy * a2 + l * shift
                pos.append([xy[0], xy[1], l * dz])
                fixed.append(1 if l < 2 else 0)
    # heptamer on the next stacking layer: centre site + its six in-plane neighbours
    cx, cy = nx // 2, ny // 2
    for (ox, oy) in [(0, 0), (1, 0), (-1, 0), (0, 1), (0, -1), (-1, 1), (1, -1)]:
        xy = (cx + ox) * a1 + (cy + oy) * a2 + layers * shift
        pos.append([xy[0], xy[1], layers * dz])
        fixed.append(0)
    pos = np.array(pos, dtype=np.float64)
    fixed = np.array(fixed, dtype=np.uint8)
    disp = sigma * rng.standard_normal(pos.shape)
    pos = pos + disp * (fixed[:, None] == 0)
    cell = np.stack([nx * a1, ny * a2])
    return CartWorkload("cfg4_Ni111_heptamer", pos, fixed, cell, De=0.4205, alpha=1.4199, r0=2.780, rc=6.0,
                        k=2, seed=seed, tol=1e-8, mmf_steps=100, dt=0.05,
                        meta=dict(nx=nx, ny=ny, layers=layers, a=a))


def small_cluster(n: int, seed: int, box: float = 9.0) -> CartWorkload:
    """Tiny random Morse cluster in a large periodic cell (edge cases / brute-force sized tests)."""
    rng = np.random.default_rng(seed)
    pts = []
    while len(pts) < n:
        p = rng.uniform(0.0, box, size=3)
        if all(np.linalg.norm(p - q) > 2.0 for q in pts):
            pts.append(p)
    pos = np.array(pts) + 20.0
    cell = np.array([[60.0, 0.0], [0.0, 60.0]])
    return CartWorkload(f"cluster{n}", pos, np.zeros(n, dtype=np.uint8), cell, De=0.4205, alpha=1.4199, r0=2.780,
                        rc=6.0, k=2, seed=seed)


# ---- general neighbour shells: stand-in for the paper's tabulated Pd/Fe/Ir(111) couplings
def shell_table(rcut: float, J1: float = 1.0, D1: float = 0.3, Dz1: float = 0.05, kF: float = 1.7):
    """All lattice offsets (dx, dy) != 0 with |dx a1 + dy a2| <= rcut, with synthetic, inversion-symmetric couplings that
    have the structure of a tabulated metallic film (the DFT tables of PAPER.md:328-616 are garbled and the UppASD inputs
    are not in the container): oscillating, decaying exchange J(r) = J1 cos(kF (r - 1)) / r^3, an in-plane Neel-type DMI
    D1 / r^3 (z x rhat) and an out-of-plane component Dz1 / r^3 with the sign of the bond's half-plane (so D(-d) = -D(d)).
    rcut = 1 gives the six nearest neighbours with J1, D1 (z x rhat) + sign * Dz1 z.  rcut = 10 gives 366 neighbours.
    Returns offsets [n][2] int32, J [n], D [n][3]."""
    R = int(np.ceil(rcut * 2 / np.sqrt(3.0))) + 1
    offs, Js, Ds = [], [], []
    for dy in range(-R, R + 1):
        for dx in range(-2 * R, 2 * R + 1):
            if dx == 0 and dy == 0:
                continue
            x, y = dx + 0.5 * dy, dy * np.sqrt(3.0) / 2.0
            r = float(np.hypot(x, y))
            if r > rcut + 1e-9:
                continue
            sgn = 1.0 if (dy > 0 or (dy == 0 and dx > 0)) else -1.0
            offs.append((dx, dy))
            Js.append(J1 * np.cos(kF * (r - 1.0)) / r ** 3)
            Ds.append((D1 / r ** 3 * (-y / r), D1 / r ** 3 * (x / r), sgn * Dz1 / r ** 3))
    return np.array(offs, dtype=np.int32), np.array(Js), np.array(Ds)


@dataclass
class ShellWorkload:
    name: str
    Lx: int
    Ly: int
    pbc_x: int
    pbc_y: int
    offsets: np.ndarray   # [n][2] int32
    Jd: np.ndarray        # [n]
    Dd: np.ndarray        # [n][3]
    K: float
    B: tuple
    mu: float
    k: int
    seed: int
    spins: np.ndarray
    tol: float = 1e-8

    @property
    def N(self) -> int:
        return self.Lx * self.Ly


def config_shells(L: int = 100, rcut: float = 10.0, seed: int = 1005, R: float = 5.0, sigma: float = 0.02, pbc: int = 1) -> ShellWorkload:
    """The paper's real workload class: L x L periodic lattice, couplings over every shell within rcut
    (366 neighbours per site at rcut = 10), one Neel skyrmion of radius R at the centre plus seeded noise (configs[1] recipe)."""
    rng = np.random.default_rng(seed)
    centre = np.array([_site_xy(L // 2, L // 2)])
    spins = add_noise(skyrmion_texture(L, L, pbc, pbc, centre, R), sigma, rng)
    offs, Js, Ds = shell_table(rcut)
    return ShellWorkload(f"shells{L}_rc{rcut:g}", L, L, pbc, pbc, offs, Js, Ds, K=0.05, B=(0.0, 0.0, 0.02), mu=1.0, k=2, seed=seed,
                         spins=spins)
