"""Seeded synthetic inputs shared by the oracle tests, the GPU parity tests and bench.py.

This module holds NONE of the method's arithmetic (no tensor, no sum, no integrator): only
particle clouds, forces and row subsets.  The same arrays are handed to the CPU oracle and
to the CUDA path; no random number is drawn on the device.

The recipes follow BASELINE.json `configs` / SURVEY.md section 8(d); they stand in for the
paper's own workloads (fcc lattice at n = 0.1 a^-3 under uniform gravity, and
the four-sphere cluster of PAPER.md:247-253).  Units: a = 1, eta = 1/(6 pi) => mu0 = 1.
"""
from __future__ import annotations

import math

import numpy as np

SEED_BASE = 12056333
A = 1.0
ETA = 1.0 / (6.0 * math.pi)


def _rng(seed: int) -> np.random.Generator:
    return np.random.Generator(np.random.PCG64(seed))


def cube_side(n: int, phi: float, a: float = A) -> float:
    """Side L of the cube in which n spheres of radius a have volume fraction phi."""
    return (n * 4.0 / 3.0 * math.pi * a ** 3 / phi) ** (1.0 / 3.0)


def ball_radius(n: int, phi: float, a: float = A) -> float:
    """Radius R of the ball in which n spheres of radius a have volume fraction phi."""
    return a * (n / phi) ** (1.0 / 3.0)


def four_sphere(jitter_seed: int | None = None, jitter: float = 1e-3, a: float = A):
    """Four-sphere periodic sedimentation cluster (reading A1 in DESIGN.md).

    Couple {1,3} along x at z = +5a, couple {2,4} along y at z = -5a; F = (0, 0, -1) each.
    With jitter_seed, seeded uniform offsets in [-jitter, jitter]^3 break the exact symmetry.
    Returns (pos[4,3], force[4,3]) in fp64.
    """
    pos = a * np.array([[5.0, 0.0, 5.0], [0.0, 5.0, -5.0], [-5.0, 0.0, 5.0], [0.0, -5.0, -5.0]])
    if jitter_seed is not None:
        pos = pos + _rng(jitter_seed).uniform(-jitter, jitter, size=pos.shape)
    force = np.tile(np.array([0.0, 0.0, -1.0]), (4, 1))
    return pos, force


def uniform_cube(n: int, phi: float, seed: int, a: float = A) -> np.ndarray:
    """n i.i.d. uniform points in a cube centred on the origin (overlaps allowed)."""
    L = cube_side(n, phi, a)
    return _rng(seed).uniform(-0.5 * L, 0.5 * L, size=(n, 3))


def uniform_ball(n: int, phi: float, seed: int, a: float = A) -> np.ndarray:
    """n i.i.d. uniform points in a ball centred on the origin (overlaps allowed)."""
    R = ball_radius(n, phi, a)
    rng = _rng(seed)
    u = rng.normal(size=(n, 3))
    u /= np.linalg.norm(u, axis=1, keepdims=True)
    rad = R * rng.uniform(0.0, 1.0, size=(n, 1)) ** (1.0 / 3.0)
    return u * rad


def rsa_cube(n: int, phi: float, seed: int, a: float = A,
             shell: tuple[float, float] | None = None) -> np.ndarray:
    """Random sequential addition of n non-overlapping spheres (centre distance >= 2a) in a
    cube centred on the origin.  Cell grid with cell side >= 2a.
    shell = (lo, hi): a candidate is also rejected when its distance to an accepted centre lies in
    [lo, hi] -- clouds in which no pair sits near a cut-off radius (trajectory parity runs must not
    straddle the discontinuity of the lubrication correction at r = 3a, reading C3)."""
    L = cube_side(n, phi, a)
    rng = _rng(seed)
    reach = 2.0 * a if shell is None else max(2.0 * a, float(shell[1]))
    ncell = max(1, int(L // reach))
    cs = L / ncell
    cells: dict[tuple[int, int, int], list[int]] = {}
    pts = np.empty((n, 3))
    count = 0
    min2 = (2.0 * a) ** 2
    lo2, hi2 = (shell[0] ** 2, shell[1] ** 2) if shell is not None else (1.0, 0.0)
    while count < n:
        p = rng.uniform(0.0, L, size=3)
        c = tuple(int(v) for v in np.minimum(p // cs, ncell - 1))
        ok = True
        for dx in (-1, 0, 1):
            for dy in (-1, 0, 1):
                for dz in (-1, 0, 1):
                    key = (c[0] + dx, c[1] + dy, c[2] + dz)
                    for k in cells.get(key, ()):
                        q = pts[k]
                        d2 = (p[0] - q[0]) ** 2 + (p[1] - q[1]) ** 2 + (p[2] - q[2]) ** 2
                        if d2 < min2 or lo2 <= d2 <= hi2:
                            ok = False
                            break
                    if not ok:
                        break
                if not ok:
                    break
            if not ok:
                break
        if ok:
            pts[count] = p
            cells.setdefault(c, []).append(count)
            count += 1
    return pts - 0.5 * L


def fcc_lattice(n_cells: int, number_density: float = 0.1, a: float = A,
                jitter_seed: int | None = None, jitter: float = 1e-2) -> np.ndarray:
    """fcc lattice of 4 n_cells^3 sites at the given number density, centred.
    With jitter_seed every site is moved by a seeded uniform offset in [-jitter, jitter]^3 (units
    of a): the exact lattice has pairs at exactly half a box, where the nearest image of
    PAPER.md:115 is ambiguous."""
    cell = (4.0 / number_density) ** (1.0 / 3.0) * a
    base = np.array([[0.0, 0.0, 0.0], [0.5, 0.5, 0.0], [0.5, 0.0, 0.5], [0.0, 0.5, 0.5]])
    g = np.arange(n_cells)
    ijk = np.stack(np.meshgrid(g, g, g, indexing="ij"), axis=-1).reshape(-1, 1, 3)
    pts = (ijk + base[None, :, :]).reshape(-1, 3) * cell
    pts = pts - pts.mean(axis=0)
    if jitter_seed is not None:
        pts = pts + a * _rng(jitter_seed).uniform(-jitter, jitter, size=pts.shape)
    return pts


def sc_lattice(n_edge: int, number_density: float = 0.1, a: float = A,
               jitter_seed: int | None = None, jitter: float = 1e-2) -> np.ndarray:
    """Simple-cubic lattice of n_edge^3 sites at the given number density, centred, with the same
    seeded jitter as fcc_lattice.  With an ODD number of sites per edge half a box (sc_box) falls
    midway between two lattice planes, so no pair component lies within half a lattice spacing of
    the discontinuity of the nearest-image rule: the cloud for long trajectory
    comparisons in the periodic box (reading B3)."""
    sp = (1.0 / number_density) ** (1.0 / 3.0) * a
    g = np.arange(n_edge)
    pts = np.stack(np.meshgrid(g, g, g, indexing="ij"), axis=-1).reshape(-1, 3) * sp
    pts = pts - pts.mean(axis=0)
    if jitter_seed is not None:
        pts = pts + a * _rng(jitter_seed).uniform(-jitter, jitter, size=pts.shape)
    return pts


def sc_box(n_edge: int, number_density: float = 0.1, a: float = A) -> float:
    """Side L of the periodic cube commensurate with sc_lattice(n_edge)."""
    return n_edge * (1.0 / number_density) ** (1.0 / 3.0) * a


def fcc_box(n_cells: int, number_density: float = 0.1, a: float = A) -> float:
    """Side L of the periodic cube commensurate with fcc_lattice(n_cells): N / L^3 = density."""
    return n_cells * (4.0 / number_density) ** (1.0 / 3.0) * a


def normal_forces(n: int, seed: int) -> np.ndarray:
    """Forces with i.i.d. N(0,1) components."""
    return _rng(seed).normal(size=(n, 3))


def gravity_forces(n: int, g=(0.0, 0.0, -1.0)) -> np.ndarray:
    """The paper's uniform drag F = (0, 0, -F) on every particle."""
    return np.tile(np.asarray(g, dtype=np.float64), (n, 1))


def row_subset(n: int, nrows: int, seed: int) -> np.ndarray:
    """Sorted seeded subset of row indices (all rows when n <= nrows)."""
    if n <= nrows:
        return np.arange(n, dtype=np.int64)
    return np.sort(_rng(seed).choice(n, size=nrows, replace=False)).astype(np.int64)


def min_pair_distance(pos: np.ndarray, cutoff: float) -> float:
    """Smallest centre distance below `cutoff` (cell-grid search), or inf if none."""
    pos = np.asarray(pos, dtype=np.float64)
    lo = pos.min(axis=0)
    idx = np.floor((pos - lo) / cutoff).astype(np.int64)
    dims = idx.max(axis=0) + 1
    key = (idx[:, 0] * dims[1] + idx[:, 1]) * dims[2] + idx[:, 2]
    order = np.argsort(key, kind="stable")
    skey = key[order]
    best = math.inf
    for dx in (-1, 0, 1):
        for dy in (-1, 0, 1):
            for dz in (-1, 0, 1):
                nb = idx + np.array([dx, dy, dz])
                valid = np.all((nb >= 0) & (nb < dims), axis=1)
                nkey = (nb[:, 0] * dims[1] + nb[:, 1]) * dims[2] + nb[:, 2]
                lo_i = np.searchsorted(skey, nkey, side="left")
                hi_i = np.searchsorted(skey, nkey, side="right")
                maxlen = int((hi_i - lo_i)[valid].max(initial=0))
                for s in range(maxlen):
                    sel = valid & (lo_i + s < hi_i)
                    if not sel.any():
                        break
                    other = order[(lo_i + s)[sel]]
                    me = np.nonzero(sel)[0]
                    keep = other != me
                    if keep.any():
                        d = np.linalg.norm(pos[me[keep]] - pos[other[keep]], axis=1)
                        best = min(best, float(d.min()))
    return best


def to_xyzw(x: np.ndarray, dtype) -> np.ndarray:
    """[N,3] -> contiguous [N,4] records (xyz + zero pad lane) of `dtype`, rounded once: the
    paper's float4 record.  Pure marshalling."""
    x = np.asarray(x)
    out = np.zeros((x.shape[0], 4), dtype=dtype)
    out[:, :3] = x
    return out


# ---- the named configurations of BASELINE.json ------------------------------------------

def config2():
    """N=4096 non-overlapping spheres, cube at phi=0.05, N(0,1) forces."""
    n = 4096
    return rsa_cube(n, 0.05, SEED_BASE + 2), normal_forces(n, SEED_BASE + 102)


def config3():
    """N=65536 uniform points, cube at phi=0.01 (overlaps allowed), N(0,1) forces."""
    n = 65536
    return uniform_cube(n, 0.01, SEED_BASE + 3), normal_forces(n, SEED_BASE + 103)


def config4():
    """N=262144 uniform points in a ball at phi=0.02, gravity."""
    n = 262144
    return uniform_ball(n, 0.02, SEED_BASE + 4), gravity_forces(n)


def sweep(n: int):
    """Throughput sweep point: uniform cube at phi=0.01, N(0,1) forces."""
    return uniform_cube(n, 0.01, SEED_BASE + 5 + n), normal_forces(n, SEED_BASE + 105 + n)
