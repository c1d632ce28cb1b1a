"""Pins of the CPU oracle against what the paper and the mathematics fix (CPU only).

Each test names the passage / closed form it checks.  Nothing here touches the CUDA path.
"""
import json
import math
import os

import numpy as np
import pytest

from oracle import sd_oracle as orc
from paper_1205_6333_b200 import workloads as wl

GOLD = os.path.join(os.path.dirname(__file__), "golden")
ETA1 = 1.0 / (6.0 * math.pi)  # mu0 = 1 with a = 1


def _gold(name):
    with open(os.path.join(GOLD, name)) as f:
        return json.load(f)


def _pair_block(d, a, eta, tensor):
    """3x3 block mu_12 for displacement d = r_1 - r_2, read off the assembled matrix."""
    pos = np.array([np.asarray(d, dtype=np.float64), [0.0, 0.0, 0.0]])
    return orc.assemble(pos, a, eta, tensor)[0:3, 3:6]


# ---- P1: single sphere, Stokes mobility mu0 = 1/(6 pi eta a) ---------------

@pytest.mark.parametrize("a,eta", [(1.0, ETA1), (0.37, 2.5), (3.0, 0.01)])
@pytest.mark.parametrize("tensor", [orc.TENSOR_RPY, orc.TENSOR_OSEEN])
def test_single_sphere_stokes_velocity(a, eta, tensor):
    F = np.array([[0.3, -1.7, 2.2]])
    for p in ([[0.0, 0.0, 0.0]], [[12.5, -3.0, 1e3]]):
        v = orc.apply(np.array(p), F, a, eta, tensor)
        np.testing.assert_allclose(v, F / (6.0 * math.pi * eta * a), rtol=1e-15)
    assert orc.mu0(a, eta) == pytest.approx(1.0 / (6.0 * math.pi * eta * a), rel=1e-15)


# ---- P2-P6: closed-form two-sphere sedimentation velocities --------------------------------

def _two_sphere(d, tensor):
    pos = np.array([np.asarray(d, dtype=np.float64), [0.0, 0.0, 0.0]])
    F = np.array([[0.0, 0.0, -1.0], [0.0, 0.0, -1.0]])
    return orc.apply(pos, F, 1.0, ETA1, tensor)


def test_two_spheres_rpy_parallel_and_perpendicular():
    g = _gold("two_sphere.json")
    for rs, vz in g["rpy_parallel"].items():
        v = _two_sphere([0.0, 0.0, float(rs)], orc.TENSOR_RPY)
        np.testing.assert_allclose(v[:, 2], vz, rtol=0, atol=2e-15)
        np.testing.assert_allclose(v[:, :2], 0.0, atol=1e-16)
    for rs, vz in g["rpy_perpendicular"].items():
        v = _two_sphere([float(rs), 0.0, 0.0], orc.TENSOR_RPY)
        np.testing.assert_allclose(v[:, 2], vz, rtol=0, atol=2e-15)
        np.testing.assert_allclose(v[:, :2], 0.0, atol=1e-16)  # no horizontal component


def test_two_spheres_rpy_oblique():
    g = _gold("two_sphere.json")["rpy_oblique45_r4"]
    s = 4.0 / math.sqrt(2.0)
    v = _two_sphere([s, 0.0, s], orc.TENSOR_RPY)
    np.testing.assert_allclose(v[:, 2], g["vz"], atol=1e-15)
    np.testing.assert_allclose(v[:, 0], g["vx"], atol=1e-15)  # identical for both spheres
    np.testing.assert_allclose(v[:, 1], 0.0, atol=1e-16)


def test_two_spheres_oseen():
    g = _gold("two_sphere.json")
    v = _two_sphere([0.0, 0.0, 4.0], orc.TENSOR_OSEEN)
    np.testing.assert_allclose(v[:, 2], g["oseen_parallel"]["4"], atol=1e-15)
    v = _two_sphere([0.0, 4.0, 0.0], orc.TENSOR_OSEEN)
    np.testing.assert_allclose(v[:, 2], g["oseen_perpendicular"]["4"], atol=1e-15)


def test_two_spheres_overlap_branch():
    g = _gold("two_sphere.json")
    v = _two_sphere([0.0, 0.0, 1.0], orc.TENSOR_RPY)
    np.testing.assert_allclose(v[:, 2], g["overlap_parallel"]["1"], atol=1e-15)
    v = _two_sphere([1.0, 0.0, 0.0], orc.TENSOR_RPY)
    np.testing.assert_allclose(v[:, 2], g["overlap_perpendicular"]["1"], atol=1e-15)
    # r -> 0: two coincident spheres move like one sphere under 2F
    for d in ([1e-9, 0.0, 0.0], [0.0, 0.0, 1e-9], [0.0, 0.0, 0.0]):
        v = _two_sphere(d, orc.TENSOR_RPY)
        np.testing.assert_allclose(v[:, 2], g["overlap_r0_limit"], atol=1e-8)
    # coincident centres: Oseen / unregularised RP contribute nothing (reading A5)
    for t in (orc.TENSOR_OSEEN, orc.TENSOR_RP_FAR):
        np.testing.assert_allclose(_two_sphere([0.0, 0.0, 0.0], t)[:, 2], -1.0, atol=0)


def test_overlap_branch_is_c1_continuous_at_2a():
    """Both RPY branches agree at r = 2a in value (A = 7/16, B r^2 = 3/16) and slope."""
    for a in (1.0, 0.7):
        eta = 1.0 / (6.0 * math.pi * a)  # mu0 = 1
        for u in ([1.0, 0.0, 0.0], [0.0, 0.6, 0.8], [1 / math.sqrt(3)] * 3):
            u = np.asarray(u)
            T2 = _pair_block(2.0 * a * u, a, eta, orc.TENSOR_RPY)
            want = 7.0 / 16.0 * np.eye(3) + 3.0 / 16.0 * np.outer(u, u)
            np.testing.assert_allclose(T2, want, atol=1e-15)
            h = 1e-6 * a
            Tm = _pair_block((2.0 * a - h) * u, a, eta, orc.TENSOR_RPY)       # overlap branch
            Tp = _pair_block((2.0 * a + h) * u, a, eta, orc.TENSOR_RPY)       # far branch
            Tmf = _pair_block((2.0 * a - h) * u, a, eta, orc.TENSOR_RP_FAR)   # far, continued
            np.testing.assert_allclose(Tm, T2, atol=2e-6)
            np.testing.assert_allclose(Tp, T2, atol=2e-6)
            # one-sided slopes agree to O(h)
            np.testing.assert_allclose((T2 - Tm) / h, (Tp - T2) / h, atol=1e-4)
            # and the two formulas differ only at second order in (2a - r)
            np.testing.assert_allclose(Tm, Tmf, atol=1e-10)


# ---- differential identities: Stokes flow is incompressible, T = (1 + a^2/3 lap) G ---------

def _fd_div(d, a, eta, tensor, h):
    div = np.zeros(3)
    for al in range(3):
        e = np.zeros(3)
        e[al] = h
        Tp = _pair_block(d + e, a, eta, tensor)
        Tm = _pair_block(d - e, a, eta, tensor)
        div += (Tp[al, :] - Tm[al, :]) / (2.0 * h)
    return div


@pytest.mark.parametrize("tensor,d", [
    (orc.TENSOR_OSEEN, [3.1, -1.2, 0.7]),
    (orc.TENSOR_RPY, [3.1, -1.2, 0.7]),        # far branch
    (orc.TENSOR_RPY, [0.5, 0.9, -0.4]),        # overlap branch (r = 1.10)
    (orc.TENSOR_RP_FAR, [0.5, 0.9, -0.4]),
])
def test_pair_tensor_is_divergence_free(tensor, d):
    """div_r T(r) = 0 for the Green's function of incompressible flow (Eq. 3)."""
    d = np.asarray(d)
    div = _fd_div(d, 1.0, ETA1, tensor, 1e-4)
    scale = np.abs(_pair_block(d, 1.0, ETA1, tensor)).max() / np.linalg.norm(d)
    assert np.abs(div).max() < 1e-7 * scale


def test_rotne_prager_is_laplacian_corrected_oseen():
    """First equality of Eq. (7b):  T = (1 + a^2/3 lap) G, by finite differences."""
    a, eta = 1.3, 0.21
    h = 2e-3
    for d in ([4.0, 1.0, -2.0], [0.3, 6.0, 0.5]):
        d = np.asarray(d)
        G0 = _pair_block(d, a, eta, orc.TENSOR_OSEEN)
        lap = -6.0 * G0
        for al in range(3):
            e = np.zeros(3)
            e[al] = h
            lap = lap + _pair_block(d + e, a, eta, orc.TENSOR_OSEEN) \
                      + _pair_block(d - e, a, eta, orc.TENSOR_OSEEN)
        lap /= h * h
        want = G0 + a * a / 3.0 * lap
        got = _pair_block(d, a, eta, orc.TENSOR_RPY)
        np.testing.assert_allclose(got, want, atol=2e-7 * np.abs(got).max())


def test_oseen_prefactor_and_far_field_limit():
    """G = (I + rr)/(8 pi eta r) (Eq. 4): trace = 4/(8 pi eta r); RP -> Oseen as a/r -> 0."""
    eta, a = 0.8, 0.5
    d = np.array([1.0, 2.0, -2.0])  # r = 3
    G = _pair_block(d, a, eta, orc.TENSOR_OSEEN)
    assert np.trace(G) == pytest.approx(4.0 / (8.0 * math.pi * eta * 3.0), rel=1e-14)
    np.testing.assert_allclose(G @ d, 2.0 / (8.0 * math.pi * eta * 3.0) * d, rtol=1e-14)
    far = 1e4 * d
    T = _pair_block(far, a, eta, orc.TENSOR_RPY)
    G = _pair_block(far, a, eta, orc.TENSOR_OSEEN)
    assert np.abs(T - G).max() < 1e-8 * np.abs(G).max()
    # trace of Eq. (7b): the a^3 term is traceless
    T3 = _pair_block(d, a, eta, orc.TENSOR_RPY)
    assert np.trace(T3) == pytest.approx(np.trace(_pair_block(d, a, eta, orc.TENSOR_OSEEN)),
                                         rel=1e-14)


# ---- P7 / P8: symmetry and positive definiteness ---------------

def test_assembled_matrix_is_symmetric():
    pos = wl.uniform_cube(48, 0.15, 7)
    for t in (orc.TENSOR_RPY, orc.TENSOR_OSEEN, orc.TENSOR_RP_FAR):
        M = orc.assemble(pos, 1.0, ETA1, t)
        np.testing.assert_allclose(M, M.T, rtol=4e-16, atol=0)  # up to one rounding
        np.testing.assert_array_equal(np.diag(M), 1.0)


def test_matrix_free_symmetry():
    pos = wl.uniform_cube(300, 0.05, 11)
    F, G = wl.normal_forces(300, 12), wl.normal_forces(300, 13)
    for t in (orc.TENSOR_RPY, orc.TENSOR_OSEEN):
        lhs = np.sum(G * orc.apply(pos, F, 1.0, ETA1, t))
        rhs = np.sum(F * orc.apply(pos, G, 1.0, ETA1, t))
        assert lhs == pytest.approx(rhs, rel=1e-12)


def test_positive_definite_by_cholesky():
    """'mu is positive definite if no pair of particle centres is closer than 2a';
    the RPY overlap branch keeps it so for overlapping spheres; the unregularised forms do not."""
    n = 64
    apart = wl.rsa_cube(n, 0.2, 21)
    assert wl.min_pair_distance(apart, 3.0) >= 2.0
    M = orc.assemble(apart, 1.0, ETA1, orc.TENSOR_RPY)
    np.linalg.cholesky(M)
    assert np.linalg.eigvalsh(M).min() > 0.05
    # far-only formula is the same matrix when nothing overlaps
    assert np.array_equal(M, orc.assemble(apart, 1.0, ETA1, orc.TENSOR_RP_FAR))

    close = wl.uniform_cube(n, 0.6, 22)
    assert wl.min_pair_distance(close, 2.0) < 0.5
    M = orc.assemble(close, 1.0, ETA1, orc.TENSOR_RPY)
    np.linalg.cholesky(M)
    assert np.linalg.eigvalsh(M).min() > 0.0
    for t in (orc.TENSOR_RP_FAR, orc.TENSOR_OSEEN):  # negative controls
        Mbad = orc.assemble(close, 1.0, ETA1, t)
        assert np.linalg.eigvalsh(Mbad).min() < 0.0
        with pytest.raises(np.linalg.LinAlgError):
            np.linalg.cholesky(Mbad)


# ---- P12: the product is the assembled matrix times the force vector ----------------------

@pytest.mark.parametrize("tensor", [orc.TENSOR_RPY, orc.TENSOR_OSEEN, orc.TENSOR_RP_FAR])
def test_product_equals_dense_matvec(tensor):
    n = 64
    pos = wl.uniform_cube(n, 0.3, 31)  # mixes both RPY branches
    F = wl.normal_forces(n, 32)
    M = orc.assemble(pos, 1.0, ETA1, tensor)
    want = (M @ F.reshape(-1)).reshape(n, 3)
    got = orc.apply(pos, F, 1.0, ETA1, tensor)
    np.testing.assert_allclose(got, want, atol=1e-13 * np.abs(want).max())


def test_pair_block_has_tensor_form_of_eq_7b():
    """mu_12 = mu0 [3a/4r (I + uu) + a^3/2r^3 (I - 3uu)]: eigenvalue along u is
    mu0 (3a/2r - a^3/r^3), transverse eigenvalues mu0 (3a/4r + a^3/2r^3)."""
    a, eta = 0.8, 0.4
    mu0 = 1.0 / (6.0 * math.pi * eta * a)
    d = np.array([2.0, -3.0, 6.0])  # r = 7
    r = 7.0
    T = _pair_block(d, a, eta, orc.TENSOR_RPY)
    w = np.sort(np.linalg.eigvalsh(T))
    lon = mu0 * (3 * a / (2 * r) - a ** 3 / r ** 3)
    tra = mu0 * (3 * a / (4 * r) + a ** 3 / (2 * r ** 3))
    np.testing.assert_allclose(w, sorted([lon, tra, tra]), rtol=1e-13)
    np.testing.assert_allclose(T @ d, lon * d, rtol=1e-13)


# ---- P9: invariances of Eq. (7) -------------------------------------------------------------

def test_invariances():
    n = 200
    pos = wl.uniform_cube(n, 0.2, 41)
    F = wl.normal_forces(n, 42)
    for t in (orc.TENSOR_RPY, orc.TENSOR_OSEEN):
        v = orc.apply(pos, F, 1.0, ETA1, t)
        scale = np.abs(v).max()
        # translation
        v2 = orc.apply(pos + np.array([100.0, -50.0, 25.0]), F, 1.0, ETA1, t)
        np.testing.assert_allclose(v2, v, atol=1e-11 * scale)
        # rotation
        Q, _ = np.linalg.qr(wl.normal_forces(3, 43))
        v3 = orc.apply(pos @ Q.T, F @ Q.T, 1.0, ETA1, t)
        np.testing.assert_allclose(v3, v @ Q.T, atol=1e-12 * scale)
        # linearity in F
        G = wl.normal_forces(n, 44)
        v4 = orc.apply(pos, 2.0 * F - 0.5 * G, 1.0, ETA1, t)
        np.testing.assert_allclose(v4, 2.0 * v - 0.5 * orc.apply(pos, G, 1.0, ETA1, t),
                                   atol=1e-12 * scale)
        # scaling (r, a) -> (lam r, lam a) at fixed eta: v -> v / lam
        lam = 3.0
        v5 = orc.apply(lam * pos, F, lam * 1.0, ETA1, t)
        np.testing.assert_allclose(v5, v / lam, atol=1e-12 * scale)
        # permutation of the particles permutes the rows (summation order does not matter)
        perm = np.random.Generator(np.random.PCG64(45)).permutation(n)
        v6 = orc.apply(pos[perm], F[perm], 1.0, ETA1, t)
        np.testing.assert_allclose(v6, v[perm], atol=1e-14 * scale)


def test_apply_rows_matches_apply_and_rejects_bad_arguments():
    n = 257
    pos, F = wl.uniform_cube(n, 0.1, 51), wl.normal_forces(n, 52)
    v = orc.apply(pos, F, 1.0, ETA1)
    rows = wl.row_subset(n, 40, 53)
    assert np.array_equal(orc.apply_rows(pos, F, rows, 1.0, ETA1), v[rows])
    with pytest.raises(ValueError):
        orc.apply_rows(pos, F, [n], 1.0, ETA1)
    with pytest.raises(ValueError):
        orc.apply(pos, F, -1.0, ETA1)
    with pytest.raises(ValueError):
        orc.apply(pos, F, 1.0, ETA1, 7)


# ---- P10 / P11: the periodic four-sphere cluster -------------------------

@pytest.fixture(scope="module")
def four_sphere_run():
    g = _gold("four_sphere.json")
    pos, F = wl.four_sphere()
    assert np.array_equal(pos, np.array(g["positions"], dtype=float))
    _, _, traj = orc.step(pos, F, 1.0, ETA1, g["dt"], 66000, orc.INT_MIDPOINT, rec_stride=1)
    return g, np.concatenate([pos[None], traj], axis=0)


def _crossings(t, y):
    s = np.nonzero(np.sign(y[:-1]) * np.sign(y[1:]) < 0)[0]
    return t[s] + (t[s + 1] - t[s]) * y[s] / (y[s] - y[s + 1])


def test_four_sphere_period_is_517(four_sphere_run):
    g, traj = four_sphere_run
    t = g["dt"] * np.arange(traj.shape[0])
    cr = _crossings(t, traj[:, 0, 2] - traj[:, 1, 2])  # all four in one horizontal plane
    np.testing.assert_allclose(cr[:3], g["probe_plane_crossings"], atol=2e-3)
    T = cr[2] - cr[0]
    assert abs(T - g["paper_T"]) < g["paper_T_tol"]          # paper: "about 517 tau_s"
    assert abs(T - g["probe_T_rpy"]) < 5e-3
    assert abs(cr[0] - T / 4.0) < 5e-3                         # quarter period
    # after one period the initial relative configuration is restored
    k = g["probe_return_step"]
    rel0 = traj[0] - traj[0].mean(axis=0)
    relk = traj[k] - traj[k].mean(axis=0)
    assert np.abs(relk - rel0).max() < 1e-3
    # after half a period: the horizontally mirrored configuration (couples swap roles)
    kh = int(round(0.5 * T / g["dt"]))
    relh = traj[kh] - traj[kh].mean(axis=0)
    assert abs(relh[0, 2] - relh[1, 2] + 10.0) < 5e-3       # couple {1,3} now below {2,4}
    x1 = traj[:, 0, 0]
    assert x1.min() == pytest.approx(g["probe_x1_range"][0], abs=2e-4)
    assert x1.max() == pytest.approx(g["probe_x1_range"][1], abs=2e-4)


def test_four_sphere_symmetries_hold_throughout(four_sphere_run):
    """x3 = -x1, y2 = -y4, z3 = z1, z4 = z2, y1 = y3 = x2 = x4 = 0."""
    _, traj = four_sphere_run
    assert np.abs(traj[:, 2, 0] + traj[:, 0, 0]).max() < 1e-12
    assert np.abs(traj[:, 1, 1] + traj[:, 3, 1]).max() < 1e-12
    assert np.abs(traj[:, 2, 2] - traj[:, 0, 2]).max() < 1e-9
    assert np.abs(traj[:, 3, 2] - traj[:, 1, 2]).max() < 1e-9
    for p, c in ((0, 1), (2, 1), (1, 0), (3, 0)):
        assert np.abs(traj[:, p, c]).max() < 1e-12
    zcm = traj[:, :, 2].mean(axis=1)
    assert np.all(np.diff(zcm) < 0)  # centre of mass sediments monotonically


def test_four_sphere_state_after_1e4_steps(four_sphere_run):
    g, traj = four_sphere_run
    k = g["steps"]
    np.testing.assert_allclose(traj[k, 0], g["probe_midpoint_r1"], atol=2e-9)
    np.testing.assert_allclose(traj[k, 1], g["probe_midpoint_r2"], atol=2e-9)
    pos, F = wl.four_sphere()
    pe, _, _ = orc.step(pos, F, 1.0, ETA1, g["dt"], k, orc.INT_EULER)
    np.testing.assert_allclose(pe[0], g["probe_euler_r1"], atol=2e-9)
    # second-order convergence of the midpoint rule, first order of Euler
    pm4, _, _ = orc.step(pos, F, 1.0, ETA1, g["dt"] / 4, 4 * k, orc.INT_MIDPOINT)
    assert np.abs(pm4 - traj[k]).max() < 5e-8
    assert 1e-4 < np.abs(pe - pm4).max() < 1e-2


def test_four_sphere_oseen_period_differs():
    """The paper's 517 tau_s needs the Rotne-Prager tensor; Oseen gives ~522.8 (reading A2)."""
    g = _gold("four_sphere.json")
    pos, F = wl.four_sphere()
    _, _, traj = orc.step(pos, F, 1.0, ETA1, g["dt"], 66000, orc.INT_MIDPOINT,
                          tensor=orc.TENSOR_OSEEN, rec_stride=1)
    t = g["dt"] * (1 + np.arange(traj.shape[0]))
    cr = _crossings(t, traj[:, 0, 2] - traj[:, 1, 2])
    assert abs((cr[2] - cr[0]) - g["probe_T_oseen"]) < 2e-2


def test_euler_step_is_r_plus_dt_v():
    """Step 1 of the paper's loop with velocities from step 3."""
    pos, F = wl.uniform_cube(50, 0.1, 61), wl.normal_forces(50, 62)
    dt = 0.125
    v = orc.apply(pos, F, 1.0, ETA1)
    p1, vlast, _ = orc.step(pos, F, 1.0, ETA1, dt, 1, orc.INT_EULER)
    assert np.array_equal(p1, pos + dt * v)
    assert np.array_equal(vlast, v)
    ph = pos + 0.5 * dt * v
    vh = orc.apply(ph, F, 1.0, ETA1)
    p2, vlast, _ = orc.step(pos, F, 1.0, ETA1, dt, 1, orc.INT_MIDPOINT)
    assert np.array_equal(p2, pos + dt * vh)
    assert np.array_equal(vlast, vh)
