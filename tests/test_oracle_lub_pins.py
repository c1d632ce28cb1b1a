"""Pins of the oracle's lubrication correction (Eq. 8).
CPU only; nothing here touches the CUDA path."""
import math

import numpy as np
import pytest

from oracle import sd_oracle as orc

ETA1 = 1.0 / (6.0 * math.pi)  # mu0 = 1 with a = 1


def _par(s):   # coefficient of rr^ in mu0 f_sing, Eq. (8)
    return 1.0 / (4.0 * s) - 9.0 / 40.0 * math.log(s)


def _per(s):   # coefficient of I - rr^
    return -math.log(s) / 6.0


def _cloud(n, side, seed):
    rng = np.random.Generator(np.random.PCG64(seed))
    return rng.uniform(-0.5 * side, 0.5 * side, size=(n, 3)), rng.normal(size=(n, 3))


def test_two_spheres_closed_forms_of_eq8():
    """Head-on approach feels [1/(4s) - 9/40 ln s] v_rel / mu0, sliding past -(1/6) ln s v_rel / mu0.
    s = 1/4, 1/2: 1/(4s) is exact, ln(1/4) = -2 ln 2, ln(1/2) = -ln 2."""
    ln2 = 0.6931471805599453
    for s, par, per in ((0.25, 1.0 + 0.45 * ln2, ln2 / 3.0), (0.5, 0.5 + 0.225 * ln2, ln2 / 6.0)):
        r = 2.0 + s
        pos = np.array([[0.0, 0.0, r], [0.0, 0.0, 0.0]])
        vel = np.array([[0.3, 0.0, -1.0], [0.0, 0.2, 0.5]])        # v_12 = (0.3, -0.2, -1.5)
        c = orc.lubrication(pos, vel, 1.0, ETA1)
        np.testing.assert_allclose(c[0], [per * 0.3, per * -0.2, par * -1.5], rtol=1e-15)
        np.testing.assert_allclose(c[1], -c[0], rtol=0, atol=0)    # action = -reaction
    # units: f_sing scales with 1/mu0 = 6 pi eta a, and s with r/a
    c2 = orc.lubrication(2.5 * np.array([[0.0, 0.0, 2.5], [0, 0, 0]]), vel, 2.5, 0.7)
    np.testing.assert_allclose(c2[0, 2], 6 * math.pi * 0.7 * 2.5 * _par(0.5) * -1.5, rtol=1e-14)


def test_cutoff_at_three_radii_and_clamp_at_contact():
    vel = np.array([[0.0, 1.0, 1.0], [0.0, 0.0, 0.0]])
    two = lambda r: orc.lubrication(np.array([[0.0, 0.0, r], [0, 0, 0]]), vel, 1.0, ETA1)[0]
    assert np.all(two(3.0) == 0.0) and np.all(two(3.5) == 0.0)     # s >= 1: truncated
    c = two(3.0 - 1e-9)                                            # just inside: ln s -> 0, 1/(4s) -> 1/4
    assert abs(c[1]) < 1e-9 and c[2] == pytest.approx(0.25, abs=1e-8)
    # contact and overlap: s clamped at LUB_SMIN (reading C2); the value is that of s = s_min
    want = [0.0, _per(orc.LUB_SMIN), _par(orc.LUB_SMIN)]
    for r in (2.0 + 0.5 * orc.LUB_SMIN, 2.0, 1.7, 0.3):
        np.testing.assert_allclose(two(r), want, rtol=1e-12)
    assert np.all(orc.lubrication(np.zeros((2, 3)), vel, 1.0, ETA1) == 0.0)  # r = 0: no direction


@pytest.mark.parametrize("box", [0.0, 9.5])
def test_momentum_galilei_dissipation_rotation(box):
    n = 60
    pos, vel = _cloud(n, 9.5, 8101)                                # ~0.07 a^-3: many pairs below 3a
    c = orc.lubrication(pos, vel, 1.0, ETA1, box=box)
    assert np.count_nonzero(np.abs(c).sum(axis=1)) > n // 2
    np.testing.assert_allclose(c.sum(axis=0), 0.0, atol=1e-9)     # pairwise antisymmetric
    u = np.array([0.4, -2.0, 1.1])
    np.testing.assert_allclose(orc.lubrication(pos, vel + u, 1.0, ETA1, box=box), c, atol=1e-9)
    assert np.all(orc.lubrication(pos, np.tile(u, (n, 1)), 1.0, ETA1, box=box) == 0.0)
    assert (vel * c).sum() > 0.0                                   # friction dissipates
    np.testing.assert_allclose(orc.lubrication(pos, 3.0 * vel, 1.0, ETA1, box=box), 3.0 * c, rtol=1e-11, atol=1e-11)
    if box == 0.0:
        q, _ = np.linalg.qr(np.random.Generator(np.random.PCG64(8102)).normal(size=(3, 3)))
        np.testing.assert_allclose(orc.lubrication(pos @ q.T, vel @ q.T, 1.0, ETA1), c @ q.T, atol=1e-9)


def test_friction_matrix_is_symmetric_positive_semidefinite_and_pairwise():
    """zeta_sing assembled column by column from unit velocities ("constructed from close
    particle pairs alone"): symmetric, PSD, zero on rigid translations; and equal to the sum of
    two-sphere blocks computed pair by pair."""
    n = 14
    pos, _ = _cloud(n, 5.5, 8103)
    Z = np.zeros((3 * n, 3 * n))
    for k in range(3 * n):
        e = np.zeros(3 * n)
        e[k] = 1.0
        Z[:, k] = orc.lubrication(pos, e.reshape(n, 3), 1.0, ETA1).reshape(-1)
    np.testing.assert_allclose(Z, Z.T, atol=1e-13)
    w = np.linalg.eigvalsh(Z)
    assert w.min() > -1e-11 and w.max() > 0.1
    assert np.abs(Z @ np.tile(np.eye(3), (n, 1))).max() < 1e-12
    Zp = np.zeros_like(Z)
    for i in range(n):
        for j in range(i + 1, n):
            d = pos[i] - pos[j]
            r = np.linalg.norm(d)
            if r >= 3.0:
                continue
            s = max(r - 2.0, orc.LUB_SMIN)
            rr = np.outer(d, d) / r ** 2
            blk = _par(s) * rr + _per(s) * (np.eye(3) - rr)
            for a_, b_, sg in ((i, i, 1), (j, j, 1), (i, j, -1), (j, i, -1)):
                Zp[3 * a_:3 * a_ + 3, 3 * b_:3 * b_ + 3] += sg * blk
    np.testing.assert_allclose(Z, Zp, atol=1e-12)


def test_nearest_image_pair_through_the_boundary_and_fp32_decision():
    L = 20.0
    pos = np.array([[L / 2 - 1.2, 0.0, 0.0], [-(L / 2 - 1.2), 0.0, 0.0]])   # 2.4 a apart through the face
    vel = np.array([[1.0, 0.5, 0.0], [0.0, 0.0, 0.0]])
    c = orc.lubrication(pos, vel, 1.0, ETA1, box=L)
    np.testing.assert_allclose(c[0], [_par(0.4) * 1.0, _per(0.4) * 0.5, 0.0], rtol=1e-13)
    assert np.all(orc.lubrication(pos, vel, 1.0, ETA1) == 0.0)
    # the fp32 decision variant only differs for pairs within rounding of r = 3a
    p, v = _cloud(80, 10.0, 8104)
    p = p.astype(np.float32).astype(np.float64)
    np.testing.assert_array_equal(orc.lubrication(p, v, 1.0, ETA1, decide_f32=True),
                                  orc.lubrication(p, v, 1.0, ETA1))
    # a pair just inside 3a in exact arithmetic whose r^2, accumulated in fp32, rounds up to 9
    rng = np.random.Generator(np.random.PCG64(8107))
    found = 0
    for _ in range(4000):
        u = rng.normal(size=3)
        d = (3.0 * (1.0 - 3e-8) * u / np.linalg.norm(u)).astype(np.float32)
        r2_32 = np.float32(np.float64(d[2]) * d[2] + np.float32(np.float64(d[1]) * d[1] + d[0] * d[0]))
        r2_64 = float((d.astype(np.float64) ** 2).sum())
        if r2_64 < 9.0 <= float(r2_32):
            edge = np.array([d.astype(np.float64), [0.0, 0.0, 0.0]])
            assert np.any(orc.lubrication(edge, vel, 1.0, ETA1) != 0.0)                  # inside in double
            assert np.all(orc.lubrication(edge, vel, 1.0, ETA1, decide_f32=True) == 0.0)  # outside in fp32
            found += 1
    assert found > 10


@pytest.mark.parametrize("integ", [orc.INT_EULER, orc.INT_MIDPOINT])
def test_step_with_lubrication_against_the_loop_written_out(integ):
    """sdo_step_lub == the paper's loop spelled out in numpy on top of the pinned
    apply() and lubrication(): F = F_ext - C(r, v_prev); v = M(r) F; r += dt v."""
    n = 12
    pos, _ = _cloud(n, 5.0, 8105)
    fext = np.tile([0.0, 0.0, -1.0], (n, 1)) + 0.3 * _cloud(n, 1.0, 8106)[1]
    dt, steps = 0.02, 5
    got_p, got_v = orc.step_lub(pos, np.zeros_like(pos), fext, 1.0, ETA1, dt, steps, integ)
    p, v = pos.copy(), np.zeros_like(pos)
    for _ in range(steps):
        v = orc.apply(p, fext - orc.lubrication(p, v, 1.0, ETA1), 1.0, ETA1)
        if integ == orc.INT_EULER:
            p = p + dt * v
        else:
            ph = p + 0.5 * dt * v
            v = orc.apply(ph, fext - orc.lubrication(ph, v, 1.0, ETA1), 1.0, ETA1)
            p = p + dt * v
    np.testing.assert_allclose(got_p, p, rtol=0, atol=1e-13)
    np.testing.assert_allclose(got_v, v, rtol=0, atol=1e-13)
    # the correction matters here and vanishes on the first product (v_prev = 0)
    free_p, _, _ = orc.step(pos, fext, 1.0, ETA1, dt, steps, integ)
    assert np.abs(free_p - p).max() > 1e-5
    p1, _ = orc.step_lub(pos, np.zeros_like(pos), fext, 1.0, ETA1, dt, 1, orc.INT_EULER)
    np.testing.assert_allclose(p1, orc.step(pos, fext, 1.0, ETA1, dt, 1, orc.INT_EULER)[0], atol=1e-15)


def test_lubrication_slows_the_approach_of_two_pushed_spheres():
    """The paper's motivation ("implementation of a hard core repulsion"): two spheres
    pushed together close their gap more slowly with the correction than without."""
    pos = np.array([[0.0, 0.0, 1.3], [0.0, 0.0, -1.3]])            # gap 0.6 a
    fext = np.array([[0.0, 0.0, -1.0], [0.0, 0.0, 1.0]])
    free, _, _ = orc.step(pos, fext, 1.0, ETA1, 0.01, 60, orc.INT_EULER)
    lub, _ = orc.step_lub(pos, np.zeros_like(pos), fext, 1.0, ETA1, 0.01, 60, orc.INT_EULER)
    gap = lambda p: p[0, 2] - p[1, 2] - 2.0
    assert 0.0 < gap(free) < gap(lub) < 0.6
    assert (0.6 - gap(lub)) < 0.75 * (0.6 - gap(free))
