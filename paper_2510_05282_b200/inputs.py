"""Seeded synthetic workloads (the five BASELINE.json configs).

This module holds NO spherical-harmonic arithmetic: it only draws random numbers and lays
out points.  It is the single piece shared by the CUDA path's tests/bench and the oracle's
tests; neither `oracle/` nor `csrc/` is imported from here.

The paper measures on no public dataset (its inputs are 100 perturbed random points, PAPER.md
line 140, and 5180 random points in a sphere, line 130), so every input here is synthetic and
shaped like the use case the paper names: harmonics on 3-D grid points around atoms
("projectors ... in a 3-dimensional grid").
"""
from __future__ import annotations

import numpy as np

#: the 8 special points appended to config 1: origin (r = 0 convention),
#: the two poles and the four equatorial axis points.
SPECIAL_POINTS = np.array(
    [
        [0.0, 0.0, 0.0],
        [0.0, 0.0, 1.0],
        [0.0, 0.0, -1.0],
        [1.0, 0.0, 0.0],
        [-1.0, 0.0, 0.0],
        [0.0, 1.0, 0.0],
        [0.0, -1.0, 0.0],
    ],
    dtype=np.float64,
)
# origin is listed once; "plus 8 special points: origin, +-z poles, +-x, +-y axes" counts the
# origin together with a second r = 0 representation (signed zeros) to reach 8.
SPECIAL_POINTS = np.concatenate([SPECIAL_POINTS, np.array([[-0.0, -0.0, -0.0]])], axis=0)


def config1_cube(n_random: int = 10_000, seed: int = 0) -> np.ndarray:
    """Config 1: `n_random` points uniform in [-1,1]^3 (seed 0) plus the 8 special points."""
    rng = np.random.default_rng(seed)
    pts = rng.uniform(-1.0, 1.0, size=(n_random, 3))
    return np.ascontiguousarray(np.concatenate([pts, SPECIAL_POINTS], axis=0))


def config2_projector_grid(spacing: float = 0.1, radius: float = 3.0, seed: int = 2) -> np.ndarray:
    """Config 2: all nodes of a cubic grid (spacing 0.1 bohr) within `radius` of an atom that
    sits at a random sub-grid offset; returns positions relative to the atom, AoS [N][3]."""
    rng = np.random.default_rng(seed)
    offset = rng.uniform(0.0, spacing, size=3)
    m = int(np.ceil(radius / spacing)) + 1
    idx = np.arange(-m, m + 1, dtype=np.float64) * spacing
    gx, gy, gz = np.meshgrid(idx, idx, idx, indexing="ij")
    rel = np.stack([gx.ravel() - offset[0], gy.ravel() - offset[1], gz.ravel() - offset[2]], axis=1)
    keep = np.einsum("ij,ij->i", rel, rel) <= radius * radius
    return np.ascontiguousarray(rel[keep])


def config3_full_grid(points_per_side: int = 128, half_box: float = 6.0) -> np.ndarray:
    """Config 3 (headline): full `points_per_side`^3 grid over [-half_box, half_box)^3,
    x_i = -L + 2L*i/n (periodic-cell convention); z is the fastest index.  Contains the origin
    once and exact axis points (r = 0 and pole handling are exercised)."""
    n = points_per_side
    ax = -half_box + (2.0 * half_box) * np.arange(n, dtype=np.float64) / n
    gx, gy, gz = np.meshgrid(ax, ax, ax, indexing="ij")
    return np.ascontiguousarray(np.stack([gx.ravel(), gy.ravel(), gz.ravel()], axis=1))


def _directions(rng: np.random.Generator, n: int) -> np.ndarray:
    g = rng.standard_normal((n, 3))
    return g / np.sqrt(np.einsum("ij,ij->i", g, g))[:, None]


def config4_sphere_directions(n: int = 1 << 24, seed: int = 1) -> np.ndarray:
    """Config 4: `n` directions uniform on the unit sphere (normalized Gaussian vectors,
    seed 1) times radii log-uniform in [1e-3, 1e2]."""
    rng = np.random.default_rng(seed)
    d = _directions(rng, n)
    radius = 10.0 ** rng.uniform(-3.0, 2.0, size=n)
    return np.ascontiguousarray(d * radius[:, None])


def config5_ball(n: int = 1 << 22, radius: float = 5.0, seed: int = 5) -> np.ndarray:
    """Config 5: `n` points uniform in a ball of radius 5."""
    rng = np.random.default_rng(seed)
    d = _directions(rng, n)
    r = radius * np.cbrt(rng.uniform(0.0, 1.0, size=n))
    return np.ascontiguousarray(d * r[:, None])


def shard_range(n: int, rank: int, world_size: int) -> tuple[int, int]:
    """Contiguous point range [begin, end) owned by `rank`: points are independent
    (SURVEY.md section 8e), so multi-GPU runs shard N with no data-path collective."""
    if world_size < 1 or not (0 <= rank < world_size):
        raise ValueError("bad rank/world_size")
    base, rem = divmod(int(n), world_size)
    begin = rank * base + min(rank, rem)
    return begin, begin + base + (1 if rank < rem else 0)


def projector_channels(lmax: int = 3, per_l: int = 2, cutoff: float = 3.0, dr: float = 0.01):
    """Radial channels of a synthetic norm-conserving-pseudopotential-like projector set ("the atomic
    problem is solved in a radial grid ... angular-momentum dependent projectors"): `per_l` channels for every l <= lmax,
    l ascending; channel c of angular momentum l has f(r) = r^l exp(-a_c r^2) (1 - (r/cutoff)^2)^2 for r < cutoff, 0
    beyond, a_c = 0.8 (c + 1), tabulated at r_j = j dr up to and including the cutoff (last entry exactly 0).
    Returns (proj_l int32 [nproj], radial float64 [nproj][nr], dr).  No spherical-harmonic arithmetic here."""
    nr = int(round(cutoff / dr)) + 1
    r = np.arange(nr, dtype=np.float64) * dr
    proj_l, rows = [], []
    for l in range(lmax + 1):
        for c in range(per_l):
            f = r**l * np.exp(-0.8 * (c + 1) * r * r) * (1.0 - np.minimum(r / cutoff, 1.0) ** 2) ** 2
            f[-1] = 0.0
            proj_l.append(l)
            rows.append(f)
    return np.asarray(proj_l, dtype=np.int32), np.ascontiguousarray(np.stack(rows)), float(dr)


def wave_weights(n: int, nvec: int = 1, seed: int = 7, volume_element: float = 1.0e-3) -> np.ndarray:
    """Synthetic projection weights w[v][i] = psi_v(r_i) dV: standard-normal values times the grid's volume element
    (0.1^3 for the config-2 grid).  Random signs are the hard case for the summation (no smoothness to help)."""
    rng = np.random.default_rng(seed)
    return np.ascontiguousarray(rng.standard_normal((nvec, n)) * volume_element)
