"""Pins of the oracle's periodic-box / nearest-image variant (CPU only).

PAPER.md:115, footnote 1: "a simulation box with periodic boundaries and include only
hydrodynamic interactions from the nearest image of each particle".  Nothing here touches the
CUDA path; the free-space oracle these pins lean on is itself pinned in test_oracle_pins.py.
"""
import itertools
import json
import math
import os

import numpy as np
import pytest

from oracle import sd_oracle as orc
from paper_1205_6333_b200 import workloads as wl

GOLD = os.path.join(os.path.dirname(__file__), "golden")
ETA1 = 1.0 / (6.0 * math.pi)
TENSORS = [orc.TENSOR_RPY, orc.TENSOR_OSEEN]


def _cloud(n, L, seed, spread=1.0):
    rng = np.random.Generator(np.random.PCG64(seed))
    return rng.uniform(-0.5 * spread * L, 0.5 * spread * L, size=(n, 3)), rng.normal(size=(n, 3))


def _brute_force_nearest_image(pos, force, a, eta, tensor, L):
    """v_i = mu0 F_i + sum_j block(d_ij) F_j with d_ij the SHORTEST of the 27 displacements
    r_i - r_j - L n, n in {-1,0,1}^3, of the positions wrapped into the box; the 3x3 block is
    read off the (separately pinned) free-space two-particle matrix."""
    n = pos.shape[0]
    w = pos - L * np.floor(pos / L + 0.5)
    shifts = np.array(list(itertools.product((-1.0, 0.0, 1.0), repeat=3))) * L
    mu0 = 1.0 / (6.0 * math.pi * eta * a)
    v = mu0 * force.copy()
    for i in range(n):
        for j in range(n):
            if i == j:
                continue
            cand = (w[i] - w[j])[None, :] - shifts
            d = cand[np.argmin(np.einsum("ij,ij->i", cand, cand))]
            blk = orc.assemble(np.array([d, [0.0, 0.0, 0.0]]), a, eta, tensor)[0:3, 3:6]
            v[i] += blk @ force[j]
    return v


@pytest.mark.parametrize("tensor", TENSORS)
def test_nearest_image_equals_brute_force_over_27_images(tensor):
    L = 11.0
    pos, F = _cloud(24, L, 7001, spread=3.0)  # positions up to 1.5 L outside: wrapping matters
    want = _brute_force_nearest_image(pos, F, 1.0, ETA1, tensor, L)
    got = orc.apply(pos, F, 1.0, ETA1, tensor, box=L)
    np.testing.assert_allclose(got, want, rtol=0, atol=1e-12)
    # and it is NOT the free-space result (the test would be vacuous otherwise)
    assert np.abs(got - orc.apply(pos, F, 1.0, ETA1, tensor)).max() > 1e-2


@pytest.mark.parametrize("tensor", TENSORS)
def test_large_box_reduces_to_free_space(tensor):
    pos, F = _cloud(40, 30.0, 7002)
    free = orc.apply(pos, F, 1.0, ETA1, tensor)
    # every |d_alpha| < 30 < L/2: remainder() returns d itself, results are bit-identical
    boxed = orc.apply(pos, F, 1.0, ETA1, tensor, box=61.0)
    assert np.array_equal(free, boxed)
    assert np.array_equal(free, orc.apply(pos, F, 1.0, ETA1, tensor, box=0.0))


def test_two_spheres_interact_through_the_boundary():
    """Spheres at x = +-(L/2 - 1): 2a apart through the face, L - 2 apart inside the box.
    Closed forms of Eq. (7b) at r = 2 (tests/golden/two_sphere.json): perpendicular -1.4375,
    parallel -1.625."""
    with open(os.path.join(GOLD, "two_sphere.json")) as f:
        g = json.load(f)
    L = 40.0
    F = np.array([[0.0, 0.0, -1.0], [0.0, 0.0, -1.0]])
    perp = orc.apply(np.array([[L / 2 - 1, 0, 0], [-(L / 2 - 1), 0, 0]]), F, 1.0, ETA1, box=L)
    np.testing.assert_allclose(perp[:, 2], g["rpy_perpendicular"]["2"], rtol=0, atol=2e-15)
    np.testing.assert_allclose(perp[:, :2], 0.0, atol=1e-16)
    par = orc.apply(np.array([[0, 0, L / 2 - 1], [0, 0, -(L / 2 - 1)]]), F, 1.0, ETA1, box=L)
    np.testing.assert_allclose(par[:, 2], g["rpy_parallel"]["2"], rtol=0, atol=2e-15)
    # oblique through an edge: the displacement seen is (2, 0, 2)/... = r 2 sqrt 2, 45 degrees
    ob = orc.apply(np.array([[L / 2 - 1, 0, L / 2 - 1], [-(L / 2 - 1), 0, -(L / 2 - 1)]]), F, 1.0,
                   ETA1, box=L)
    free = orc.apply(np.array([[-2.0, 0, -2.0], [0.0, 0, 0.0]]), F, 1.0, ETA1)
    np.testing.assert_allclose(ob, free, rtol=0, atol=2e-15)


@pytest.mark.parametrize("tensor", TENSORS)
def test_lattice_translations_of_single_particles_change_nothing(tensor):
    L = 17.0
    pos, F = _cloud(32, L, 7003)
    base = orc.apply(pos, F, 1.0, ETA1, tensor, box=L)
    rng = np.random.Generator(np.random.PCG64(7004))
    moved = pos + L * rng.integers(-3, 4, size=pos.shape)
    np.testing.assert_allclose(orc.apply(moved, F, 1.0, ETA1, tensor, box=L), base, rtol=0,
                               atol=1e-12)
    # rigid translation of everything by an arbitrary vector
    np.testing.assert_allclose(orc.apply(pos + np.array([3.3, -8.1, 0.7]), F, 1.0, ETA1, tensor,
                                         box=L), base, rtol=0, atol=1e-12)


def test_boxed_matrix_is_symmetric_and_matches_the_product():
    L = 13.0
    pos, F = _cloud(20, L, 7005, spread=2.0)
    M = orc.assemble(pos, 1.0, ETA1, orc.TENSOR_RPY, box=L)
    assert np.abs(M - M.T).max() < 1e-15     # rint is odd: d_ij = -d_ji
    v = orc.apply(pos, F, 1.0, ETA1, orc.TENSOR_RPY, box=L)
    np.testing.assert_allclose(M @ F.reshape(-1), v.reshape(-1), rtol=0, atol=1e-13)
    rows = np.array([3, 0, 19, 7])
    np.testing.assert_allclose(orc.apply_rows(pos, F, rows, 1.0, ETA1, box=L), v[rows], rtol=0,
                               atol=0)


@pytest.mark.parametrize("k", [3, 5])
def test_cubic_lattice_under_gravity_sediments_rigidly(k):
    """The paper's benchmark start is a lattice commensurate with the periodic box under uniform
    gravity.  On a simple-cubic lattice with an ODD number k of sites per edge no
    pair sits at exactly half a box, every site sees the same nearest-image neighbourhood with
    full cubic point symmetry, so all velocities are equal and vertical and the lattice
    translates rigidly; without the wrap the surface sites differ.  (The fcc lattice always has
    pairs at exactly L/2, where the nearest image is ambiguous: see the next test.)"""
    s = (1.0 / 0.1) ** (1.0 / 3.0)          # n = 0.1 a^-3
    g = (np.arange(k) - (k - 1) / 2.0) * s
    pos = np.stack(np.meshgrid(g, g, g, indexing="ij"), axis=-1).reshape(-1, 3)
    n, L = k ** 3, k * s
    F = wl.gravity_forces(n)
    v = orc.apply(pos, F, 1.0, ETA1, box=L)
    np.testing.assert_allclose(v, np.tile(v[0], (n, 1)), rtol=0, atol=1e-12)
    assert abs(v[0, 0]) < 1e-12 and abs(v[0, 1]) < 1e-12 and v[0, 2] < -1.0
    free = orc.apply(pos, F, 1.0, ETA1)
    assert np.abs(free - free[0]).max() > 1e-2
    p1, vl, _ = orc.step(pos, F, 1.0, ETA1, 1e-3, 25, orc.INT_EULER, box=L)
    np.testing.assert_allclose(p1 - pos, np.tile(25 * 1e-3 * v[0], (n, 1)), rtol=0, atol=1e-12)
    np.testing.assert_allclose(vl, v, rtol=0, atol=1e-12)


def test_fcc_workload_density_and_half_box_pairs():
    """workloads.fcc_lattice / fcc_box: N = 4 cells^3 sites at n = 0.1 a^-3.  Site
    separations are multiples of half a cell and L/2 = cells/2 cells, so pairs at exactly half a
    box always exist; fcc_lattice(..., jitter_seed) moves every site by a seeded offset, after
    which no pair sits on the decision boundary (closest: > 1e-8 L)."""
    cells = 3
    pos = wl.fcc_lattice(cells, 0.1)
    L = wl.fcc_box(cells, 0.1)
    assert pos.shape[0] == 4 * cells ** 3 and pos.shape[0] / L ** 3 == pytest.approx(0.1, rel=1e-12)
    d = pos[:, None, :] - pos[None, :, :]
    assert np.isclose(np.abs(d) / L, 0.5, atol=1e-12).any()
    nn = np.sqrt((d ** 2).sum(-1) + np.eye(pos.shape[0]) * 1e9).min()
    assert nn == pytest.approx((4.0 / 0.1) ** (1.0 / 3.0) / math.sqrt(2.0), rel=1e-12)  # > 2a
    jit = wl.fcc_lattice(cells, 0.1, jitter_seed=wl.SEED_BASE + 7, jitter=1e-2)
    assert np.abs(jit - pos).max() <= 1e-2 and np.abs(jit - pos).max() > 1e-3
    dj = jit[:, None, :] - jit[None, :, :]
    assert np.abs(np.abs(dj / L - np.rint(dj / L)) - 0.5).min() > 1e-8


@pytest.mark.parametrize("image", [orc.IMAGE_F32, orc.IMAGE_F64])
def test_image_decision_variants_agree_away_from_half_box(image):
    """DESIGN.md reading B2: the fp32 / fp64 decision rules pick the same image as the
    definition unless |d_alpha| is within rounding of L/2."""
    L = 19.0
    pos, F = _cloud(48, L, 7006, spread=2.5)
    pos = pos.astype(np.float32).astype(np.float64)  # fp32-representable, as on the fp32 path
    d = pos[:, None, :] - pos[None, :, :]
    frac = np.abs(d / L - np.rint(d / L))
    assert np.abs(frac - 0.5).min() > 1e-5           # no pair near the decision boundary
    want = orc.apply(pos, F, 1.0, ETA1, box=L)
    got = orc.apply(pos, F, 1.0, ETA1, box=L, image=image)
    # same images, and the displacement is the exact difference in every variant (reading B2:
    # only the decision n is taken in the kernel's precision)
    np.testing.assert_allclose(got, want, rtol=0, atol=1e-13)


@pytest.mark.parametrize("image", [orc.IMAGE_F32, orc.IMAGE_F64])
def test_image_decision_rule_against_exact_rational_arithmetic(image):
    """Reading B2 spelled out with fractions.Fraction: n = nearest integer, ties to even, of the
    EXACT product d * fl(1/fl(L)).  The exact fcc lattice supplies hundreds of coordinate pairs
    whose product is within an ulp of +-1/2, on either side of it."""
    from fractions import Fraction

    def rint_even(fr):
        fl = math.floor(fr)
        r = fr - fl
        if r != Fraction(1, 2):
            return fl if r < Fraction(1, 2) else fl + 1
        return fl if fl % 2 == 0 else fl + 1

    F = np.array([[1.0, 2.0, 3.0], [0.5, -1.0, 2.0]])
    checked, below, above = 0, 0, 0
    for cells in (3, 5, 6, 7):
        pos = wl.fcc_lattice(cells, 0.1)
        L = wl.fcc_box(cells, 0.1)
        if image == orc.IMAGE_F32:
            pos = pos.astype(np.float32).astype(np.float64)
            L = float(np.float32(L))
            inv = float(np.float32(1.0) / np.float32(L))
        else:
            inv = 1.0 / L
        xs = sorted(set(pos[:, 0]))
        for xa in xs:
            for xb in xs:
                d = float(np.float32(xa) - np.float32(xb)) if image == orc.IMAGE_F32 else xa - xb
                prod = Fraction(d) * Fraction(inv)
                if abs(abs(float(prod)) - 0.5) > 1e-6:
                    continue
                n = rint_even(prod)
                below += abs(prod) < Fraction(1, 2)
                above += abs(prod) > Fraction(1, 2)
                got = orc.apply(np.array([[xa, 0.25, 0.125], [xb, 0.0, 0.0]]), F, 1.0, ETA1,
                                box=L, image=image)
                # the decision uses the fp32 difference d; the displacement is exact: xa - xb - n L
                want = orc.apply(np.array([[(xa - xb) - n * L, 0.25, 0.125], [0.0, 0.0, 0.0]]), F,
                                 1.0, ETA1)
                np.testing.assert_allclose(got, want, rtol=0, atol=1e-14)
                checked += 1
    assert checked >= 40 and below > 0 and above > 0


def test_image_decision_at_exactly_half_a_box():
    """d = L/2 exactly: both images are nearest.  remainder() takes the even multiple (n = 0);
    the fp32 rule rounds d * fl32(1/L), and fl32(1/3) > 1/3 tips it to n = 1.  Same distance,
    opposite direction: the variants may differ here and only here."""
    L = 3.0
    F = np.array([[0.0, 0.0, -1.0], [1.0, 0.0, 0.0]])
    pos = np.array([[1.5, 0.0, 0.0], [0.0, 0.0, 0.0]])
    v_def = orc.apply(pos, F, 1.0, ETA1, box=L)
    v_f32 = orc.apply(pos, F, 1.0, ETA1, box=L, image=orc.IMAGE_F32)
    free_plus = orc.apply(pos, F, 1.0, ETA1)
    free_minus = orc.apply(np.array([[-1.5, 0.0, 0.0], [0.0, 0.0, 0.0]]), F, 1.0, ETA1)
    np.testing.assert_allclose(v_def, free_plus, rtol=0, atol=1e-15)
    np.testing.assert_allclose(v_f32[0], free_minus[0], rtol=0, atol=1e-15)


def test_box_argument_validation():
    pos, F = _cloud(4, 10.0, 7007)
    for bad in (-1.0, float("nan"), float("inf")):
        with pytest.raises(ValueError):
            orc.apply(pos, F, 1.0, ETA1, box=bad)
    with pytest.raises(ValueError):
        orc.apply(pos, F, 1.0, ETA1, box=10.0, image=7)
