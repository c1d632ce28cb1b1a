"""GPU parity of the periodic-box / nearest-image variant (PAPER.md:115
footnote 1) against the CPU oracle, through the C ABI (`sd_set_box`).

Tolerances are those of the free-space path (north_star): 1e-5 (fp32-Kahan), 1e-11 (fp64) on
max_i |v_gpu,i - v_ref,i| / |v_ref,i|.  The nearest-image index is an integer decided by floating
point.  Two kinds of comparison:
 * against the oracle's PLAIN definition (C99 `remainder`, IMAGE_DEFINITION) on clouds for which a
   CPU pre-check (tests/guards.py) asserts that no pair component lies within GUARD = 1e-3 a of
   half a box, products and trajectories alike -- a kernel that took a wrong image would fail;
 * where ties at |d| = L/2 are the point (the commensurate fcc lattice has thousands), both sides
   take the decision in the kernel's precision (reading B2): the oracle runs with
   IMAGE_F32 (resp. IMAGE_F64) on the same rounded inputs, box side included.
"""
import numpy as np
import pytest

import guards

from oracle import sd_oracle as orc
from paper_1205_6333_b200 import workloads as wl

pytestmark = pytest.mark.gpu

TOL = {"PREC_F32_KAHAN": 1e-5, "PREC_F64": 1e-11}
IMAGE = {"PREC_F32_KAHAN": orc.IMAGE_F32, "PREC_F64": orc.IMAGE_F64}
TENSOR = {"rpy": (0, orc.TENSOR_RPY), "oseen": (1, orc.TENSOR_OSEEN)}
GUARD = 1e-3   # a: distance every pair component keeps from half a box in the plain-definition tests


@pytest.fixture(scope="module")
def gpu():
    import torch
    from paper_1205_6333_b200 import sd
    assert torch.cuda.is_available()
    torch.cuda.set_device(0)
    sd.load_library()
    return torch, sd


def rel_err(got, want):
    return float(np.max(np.linalg.norm(got - want, axis=1) / np.linalg.norm(want, axis=1)))


def rounded(x, prec_name):
    dt = np.float64 if prec_name == "PREC_F64" else np.float32
    return wl.to_xyzw(x, dt)


def row_errs(got, want):
    return np.linalg.norm(got - want, axis=1) / np.linalg.norm(want, axis=1)


def fp32_oseen_row_tol(p, f, want, Ls):
    """Per-row tolerance for Oseen in fp32 on clouds with overlapping centres (DESIGN.md reading
    B6).  The fp32 kernels form d = fl(x_i - x_j) before the image shift: an absolute error of up
    to ulp(|d|)/2 per component that does not shrink with the image distance r, and Eq. (4) has no
    overlap branch to bound 1/r.  For a pair that meets through a face (|x_i - x_j| > L/2) at
    r < 2a the term c1 [F/r + (d.F) d/r^3] moves by at most 4 c1 |F_j| |delta| / r^2.  Rows without
    such a partner keep the plain 1e-5; the others (asserted to be under a tenth of the rows) get
    that bound on top."""
    tol = np.full(p.shape[0], TOL["PREC_F32_KAHAN"])
    ov = guards.pairs_in_shell(p, 0.0, 2.0 * wl.A, Ls)
    raw = p[ov[:, 0]] - p[ov[:, 1]]
    face = np.abs(raw).max(axis=1) > 0.5 * Ls
    ov, raw = ov[face], raw[face]
    r2 = ((raw - Ls * np.rint(raw / Ls)) ** 2).sum(axis=1)
    delta = np.sqrt(3.0) * 0.5 * np.spacing(np.abs(raw).max(axis=1).astype(np.float32)).astype(np.float64)
    c1 = 0.75 * wl.A * orc.mu0(wl.A, wl.ETA)
    for a, b in ((0, 1), (1, 0)):
        add = 4.0 * c1 * np.linalg.norm(f[ov[:, b]], axis=1) * delta / r2 / np.linalg.norm(want[ov[:, a]], axis=1)
        np.add.at(tol, ov[:, a], add)
    assert (tol > TOL["PREC_F32_KAHAN"]).mean() < 0.10
    return tol


def box_as_seen(L, prec_name):
    """The box side after the one rounding to the path's dtype (an input like pos and force)."""
    return float(np.float32(L)) if prec_name != "PREC_F64" else float(L)


def gpu_apply_box(torch, sd, pos, force, L, prec_name, tensor, expect_kernel=None,
                  dispatch=(-1, 0)):
    p, f = rounded(pos, prec_name), rounded(force, prec_name)
    ctx = sd.Context(pos.shape[0], wl.A, wl.ETA)
    ctx.set_precision(getattr(sd, prec_name))
    ctx.set_tensor(tensor)
    ctx.set_dispatch(*dispatch)
    ctx.set_box(L)
    assert ctx.box == L
    if expect_kernel is not None:
        assert expect_kernel in ctx.kernel_name, ctx.kernel_name
    dp, df = torch.from_numpy(p).cuda(), torch.from_numpy(f).cuda()
    dv = torch.full_like(dp, float("nan"))
    ctx.mobility_apply(dp, df, dv)
    torch.cuda.synchronize()
    out = dv.cpu().numpy()
    assert np.all(out[:, 3] == 0.0)
    assert ctx.launch_count >= 1
    ctx.close()
    return out[:, :3].astype(np.float64), p[:, :3].astype(np.float64), f[:, :3].astype(np.float64)


# ---- the paper's benchmark shape: fcc lattice, n = 0.1 a^-3, periodic box --------

@pytest.mark.parametrize("prec_name", ["PREC_F32_KAHAN", "PREC_F64"])
@pytest.mark.parametrize("tname", ["rpy", "oseen"])
@pytest.mark.parametrize("forces", ["gravity", "normal"])
@pytest.mark.parametrize("path", ["small_apply", "pairs_f"])
def test_fcc_4000_all_rows(gpu, prec_name, tname, forces, path):
    """N = 4000 through the one-launch kernel (forced) and through the tiled kernels (default)."""
    torch, sd = gpu
    cells = 10
    pos = wl.fcc_lattice(cells, 0.1, jitter_seed=wl.SEED_BASE + 20)
    L = wl.fcc_box(cells, 0.1)
    n = pos.shape[0]
    assert n == 4000
    F = wl.gravity_forces(n) if forces == "gravity" else wl.normal_forces(n, wl.SEED_BASE + 21)
    got, p, f = gpu_apply_box(torch, sd, pos, F, L, prec_name, TENSOR[tname][0], path,
                              dispatch=(1 << 20, 0) if path == "small_apply" else (-1, 0))
    want = orc.apply(p, f, wl.A, wl.ETA, TENSOR[tname][1], box=box_as_seen(L, prec_name),
                     image=IMAGE[prec_name])
    assert rel_err(got, want) <= TOL[prec_name]
    # the box matters: the free-space sum of the same cloud is far away
    assert rel_err(orc.apply(p, f, wl.A, wl.ETA, TENSOR[tname][1]), want) > 1e-2


@pytest.mark.parametrize("prec_name", ["PREC_F32_KAHAN", "PREC_F64"])
def test_exact_fcc_lattice_ties_at_half_a_box(gpu, prec_name):
    """The un-jittered lattice has thousands of pairs at exactly |d_alpha| = L/2 (up to the
    rounding of the coordinates): parity holds only if GPU and oracle break every such tie the
    same way, i.e. if the kernel's fma(d, 1/L, M) - M is the documented rint of the exact
    product.  Small path (N = 864) and tiled path (N = 10976, ragged last tile)."""
    torch, sd = gpu
    for cells, kern in ((6, "small_apply"), (14, "pairs_f")):
        pos = wl.fcc_lattice(cells, 0.1)
        L = wl.fcc_box(cells, 0.1)
        n = pos.shape[0]
        F = wl.normal_forces(n, wl.SEED_BASE + 22)
        got, p, f = gpu_apply_box(torch, sd, pos, F, L, prec_name, 0, kern)
        Ls = box_as_seen(L, prec_name)
        d = (p[:, None, 0] - p[None, :, 0]) / Ls
        assert (np.abs(np.abs(d) - 0.5) < 1e-6).sum() > n  # the ties are there
        want = orc.apply(p, f, wl.A, wl.ETA, box=Ls, image=IMAGE[prec_name])
        assert rel_err(got, want) <= TOL[prec_name]


# ---- against the plain definition (remainder), tie-free clouds (PAPER.md:115 footnote 1) ---------

@pytest.mark.parametrize("prec_name", ["PREC_F32_KAHAN", "PREC_F64"])
@pytest.mark.parametrize("tname", ["rpy", "oseen"])
@pytest.mark.parametrize("path", ["small_apply", "pairs_f"])
def test_plain_definition_fcc_in_a_larger_box_all_rows(gpu, prec_name, tname, path):
    """The benchmark lattice (N = 4000, jittered) in a box 2 % larger than the commensurate one: the
    lattice planes are cell/2 = 1.71 a apart and half a box falls 0.34 a from the nearest plane
    difference, so every image decision is far from a tie and the oracle's plain `remainder` rule
    is the reference.  One-launch kernel (forced) and tiled kernels."""
    torch, sd = gpu
    cells = 10
    pos = wl.fcc_lattice(cells, 0.1, jitter_seed=wl.SEED_BASE + 20)
    L = 1.02 * wl.fcc_box(cells, 0.1)
    n = pos.shape[0]
    F = wl.normal_forces(n, wl.SEED_BASE + 21)
    Ls = box_as_seen(L, prec_name)
    assert guards.half_box_margin(rounded(pos, prec_name)[:, :3].astype(np.float64), Ls) >= 0.3 > GUARD
    got, p, f = gpu_apply_box(torch, sd, pos, F, L, prec_name, TENSOR[tname][0], path,
                              dispatch=(1 << 20, 0) if path == "small_apply" else (-1, 0))
    want = orc.apply(p, f, wl.A, wl.ETA, TENSOR[tname][1], box=Ls, image=orc.IMAGE_DEFINITION)
    assert rel_err(got, want) <= TOL[prec_name]
    assert rel_err(orc.apply(p, f, wl.A, wl.ETA, TENSOR[tname][1]), want) > 1e-2


@pytest.mark.parametrize("prec_name", ["PREC_F32_KAHAN", "PREC_F64"])
@pytest.mark.parametrize("tname", ["rpy", "oseen"])
def test_plain_definition_uniform_cloud_with_overlaps_all_rows(gpu, prec_name, tname):
    """A uniform cloud (overlaps allowed, a third of the particles in neighbouring periodic copies)
    from which one member of every pair with a component within GUARD of half a box has been
    removed (CPU pre-check on the rounded coordinates): ~5300 particles, ragged tiles, overlapping
    pairs through the faces, all rows against the plain definition.
    Oseen in fp32: the rows with an overlapping partner through a face get the per-row bound of
    fp32_oseen_row_tol (reading B6), every other row the plain 1e-5; Rotne-Prager's overlap branch
    is bounded and stays within 1e-5 on all rows."""
    torch, sd = gpu
    n0 = 6000
    L = wl.cube_side(n0, 0.01)
    pos = wl.uniform_cube(n0, 0.01, wl.SEED_BASE + 33)
    shift = np.random.Generator(np.random.PCG64(wl.SEED_BASE + 34)).integers(-1, 2, size=(n0, 3))
    pos = pos + L * shift * (np.arange(n0) % 3 == 0)[:, None]
    Ls = box_as_seen(L, prec_name)
    p0 = rounded(pos, prec_name)[:, :3].astype(np.float64)
    keep = guards.drop_one_of_each(n0, guards.half_box_ties(p0, Ls, GUARD))
    pos = pos[keep]
    n = pos.shape[0]
    assert 4000 < n < n0 and n % 32 != 0
    assert guards.half_box_margin(p0[keep], Ls) >= GUARD
    F = wl.normal_forces(n, wl.SEED_BASE + 35)
    got, p, f = gpu_apply_box(torch, sd, pos, F, L, prec_name, TENSOR[tname][0], "_pbc")
    assert np.array_equal(p, p0[keep])
    want = orc.apply(p, f, wl.A, wl.ETA, TENSOR[tname][1], box=Ls, image=orc.IMAGE_DEFINITION)
    if tname == "oseen" and prec_name == "PREC_F32_KAHAN":
        assert np.all(row_errs(got, want) <= fp32_oseen_row_tol(p, f, want, Ls))
    else:
        assert rel_err(got, want) <= TOL[prec_name]
    # the cloud still has overlapping pairs (r < 2a), some of them through a face
    ov = guards.pairs_in_shell(p, 0.0, 2.0 * wl.A, Ls)
    assert ov.shape[0] > 50
    through = np.linalg.norm(p[ov[:, 0]] - p[ov[:, 1]], axis=1) > 0.5 * Ls
    assert through.sum() > 5


# ---- tiled packed kernels: random clouds with overlaps, ragged tails, images outside the box ----

@pytest.mark.parametrize("prec_name", ["PREC_F32_KAHAN", "PREC_F64"])
@pytest.mark.parametrize("tname", ["rpy", "oseen"])
def test_uniform_20000_tiled_all_rows(gpu, prec_name, tname):
    torch, sd = gpu
    n = 20000                                     # not a multiple of the 2048-record granularity
    L = wl.cube_side(n, 0.01)
    pos = wl.uniform_cube(n, 0.01, wl.SEED_BASE + 23)
    # a third of the particles sit in neighbouring periodic copies of the box
    shift = np.random.Generator(np.random.PCG64(wl.SEED_BASE + 24)).integers(-1, 2, size=(n, 3))
    pos = pos + L * shift * (np.arange(n) % 3 == 0)[:, None]
    F = wl.normal_forces(n, wl.SEED_BASE + 25)
    got, p, f = gpu_apply_box(torch, sd, pos, F, L, prec_name, TENSOR[tname][0], "_pbc")
    Ls = box_as_seen(L, prec_name)
    want = orc.apply(p, f, wl.A, wl.ETA, TENSOR[tname][1], box=Ls, image=IMAGE[prec_name])
    if tname == "oseen" and prec_name == "PREC_F32_KAHAN":
        assert np.all(row_errs(got, want) <= fp32_oseen_row_tol(p, f, want, Ls))
    else:
        assert rel_err(got, want) <= TOL[prec_name]
    if tname == "rpy":  # overlaps through the faces exist and take the r < 2a branch
        w = p - Ls * np.rint(p / Ls)
        face = np.abs(w).max(axis=1) > 0.5 * Ls - 1.0
        assert face.sum() > 100
        far = orc.apply_rows(p, f, np.nonzero(face)[0], wl.A, wl.ETA, orc.TENSOR_RP_FAR, box=Ls,
                             image=IMAGE[prec_name])
        assert rel_err(far, want[face]) > 1e-4


@pytest.mark.parametrize("n", [131072 + 777, 200000 + 555])  # the second: 256- (fp64: 128-) record tiles, careful pass
@pytest.mark.parametrize("prec_name", ["PREC_F32_KAHAN", "PREC_F64"])
def test_uniform_131849_eight_per_thread_sampled_rows(gpu, prec_name, n):
    torch, sd = gpu
    L = wl.cube_side(n, 0.01)
    pos = wl.uniform_cube(n, 0.01, wl.SEED_BASE + 26)
    F = wl.normal_forces(n, wl.SEED_BASE + 27)
    kern = "i8_rpy_kahan_pbc" if prec_name == "PREC_F32_KAHAN" else "f64_i4_rpy_pbc"
    got, p, f = gpu_apply_box(torch, sd, pos, F, L, prec_name, 0, kern)
    rows = wl.row_subset(n, 4096, wl.SEED_BASE + 28)
    rows[-1] = n - 1                               # the last particle of the ragged tail
    want = orc.apply_rows(p, f, rows, wl.A, wl.ETA, box=box_as_seen(L, prec_name),
                          image=IMAGE[prec_name])
    assert rel_err(got[rows], want) <= TOL[prec_name]
    assert np.all(np.isfinite(got))


def test_large_box_is_free_space_and_box_can_be_switched_off(gpu):
    torch, sd = gpu
    for n in (3000, 9000):
        pos = wl.uniform_cube(n, 0.01, wl.SEED_BASE + 29)
        F = wl.normal_forces(n, wl.SEED_BASE + 30)
        p, f = wl.to_xyzw(pos, np.float32), wl.to_xyzw(F, np.float32)
        dp, df = torch.from_numpy(p).cuda(), torch.from_numpy(f).cuda()
        ctx = sd.Context(n, wl.A, wl.ETA)
        ctx.set_dispatch(0, 0)                      # the same (tiled) kernel family with and without the box: the
        out = []                                    # one-launch kernels end at different N in the two cases
        for L in (0.0, 1.0e4, wl.cube_side(n, 0.01), 0.0):
            ctx.set_box(L)
            dv = torch.empty_like(dp)
            ctx.mobility_apply(dp, df, dv)
            torch.cuda.synchronize()
            out.append(dv.cpu().numpy()[:, :3].astype(np.float64))
        assert rel_err(out[1], out[0]) <= 1e-6      # every pair is its own nearest image
        assert rel_err(out[2], out[0]) > 1e-2
        assert np.array_equal(out[3], out[0])       # back in free space: same kernel, same bits
        with pytest.raises(sd.SdError):
            ctx.set_box(-1.0)
        with pytest.raises(sd.SdError):
            ctx.set_box(float("nan"))
        ctx.close()


# ---- sd_step in the box: the paper's benchmark run (Euler, dt = 0.001 tau_s, 100 steps) ----------
#
# The nearest-image rule is discontinuous: when a pair component crosses |d| = L/2 the pair
# tensor jumps, so two trajectories that differ in the last bit part ways by O(1e-3 a) as soon as
# one of them flips a pair the other does not.  The commensurate lattice keeps thousands of pair
# components within the jitter of L/2, and fp32 positions put a handful of them within an ulp.
# Long runs are therefore compared (a) in fp64 on the commensurate box and (b) in a box 2 % larger
# than the lattice, both sides deciding the way the kernel does; (b') in fp32 and fp64 against the
# PLAIN definition on a lattice that provably stays clear of the discontinuity (asserted on the
# oracle trajectory), every particle held to the tolerance; and (c) in fp32 on the commensurate
# box step by step, each step restarted from the GPU's own positions.

@pytest.mark.parametrize("prec_name,tol,scale", [("PREC_F64", 1e-9, 1.02), ("PREC_F64", 1e-9, 1.0)])
@pytest.mark.parametrize("cells,integ,steps,dt", [(2, "midpoint", 1000, 0.01),
                                                  (8, "midpoint", 30, 0.005),
                                                  (10, "euler", 100, 0.001),
                                                  (16, "midpoint", 5, 0.005)])
def test_step_in_periodic_box_fp64(gpu, prec_name, tol, scale, cells, integ, steps, dt):
    """(a), (b) in fp64.  N = 32 (one-launch stepper), 2048 (one launch per product), 4000 and 16384
    (tiled kernels).  Every particle obeys the tolerance."""
    torch, sd = gpu
    pos = wl.fcc_lattice(cells, 0.1, jitter_seed=wl.SEED_BASE + 31 + cells)
    L = scale * wl.fcc_box(cells, 0.1)
    n = pos.shape[0]
    p = rounded(pos, prec_name)
    ctx = sd.Context(n, wl.A, wl.ETA)
    ctx.set_precision(getattr(sd, prec_name))
    ctx.set_box(L)
    dp = torch.from_numpy(p).cuda()
    gi = sd.INT_EULER if integ == "euler" else sd.INT_MIDPOINT
    oi = orc.INT_EULER if integ == "euler" else orc.INT_MIDPOINT
    ctx.step(dp, dt, steps, gi, gravity=(0.0, 0.0, -1.0))
    dv = torch.empty_like(dp)
    ctx.get_velocity(dv)
    torch.cuda.synchronize()
    want, vlast, _ = orc.step(p[:, :3].astype(np.float64), wl.gravity_forces(n), wl.A, wl.ETA, dt,
                              steps, oi, box=box_as_seen(L, prec_name), image=IMAGE[prec_name])
    got = dp.cpu().numpy()[:, :3].astype(np.float64)
    assert np.abs(got - want).max() <= tol
    assert rel_err(dv.cpu().numpy()[:, :3].astype(np.float64), vlast) <= 10 * TOL[prec_name]
    # the suspension settled (|v| is several mu0 F with ~N^(2/3) neighbours inside L/2)
    assert (got[:, 2] - p[:, 2]).mean() < -steps * dt
    ctx.close()


@pytest.mark.parametrize("prec_name", ["PREC_F32_KAHAN", "PREC_F64"])
@pytest.mark.parametrize("edge,integ,steps,dt", [(3, "midpoint", 400, 0.01),
                                                 (11, "midpoint", 40, 0.005),
                                                 (15, "euler", 100, 0.001),
                                                 (25, "midpoint", 5, 0.005)])
def test_step_in_periodic_box_against_the_plain_definition(gpu, prec_name, edge, integ, steps, dt):
    """(b'): trajectories against the oracle's plain nearest-image rule (`remainder`), fp32 and
    fp64, ALL particles held to the tolerance.  Cloud: jittered simple-cubic lattice with an odd
    number of sites per edge in its commensurate box -- half a box falls midway between two lattice
    planes (1.08 a from the nearest pair component) and the lattice sediments almost rigidly, so
    no pair component comes near the discontinuity at |d| = L/2 during the run.  That is not
    assumed but asserted on the oracle trajectory: at every step boundary the margin exceeds GUARD
    plus the largest relative displacement any pair can make within one step.
    N = 27 (one-launch stepper), 1331 (one launch per product; >= 32 steps: CUDA-graph replay),
    3375 (tiled, 2 particles per thread, graph replay), 15625 (tiled, 4 per thread).
    Tolerance: the velocity tolerance of the product integrated over the run, 1e-5 |v|_max t (fp32;
    1e-11 in fp64), plus the rounding of the stored position word."""
    torch, sd = gpu
    pos = wl.sc_lattice(edge, 0.1, jitter_seed=wl.SEED_BASE + 40 + edge)
    L = wl.sc_box(edge, 0.1)
    n = pos.shape[0]
    p = rounded(pos, prec_name)
    p64 = p[:, :3].astype(np.float64)
    Ls = box_as_seen(L, prec_name)
    oi = orc.INT_EULER if integ == "euler" else orc.INT_MIDPOINT
    F = wl.gravity_forces(n)
    want2, _, traj = orc.step(p64, F, wl.A, wl.ETA, dt, steps + 2, oi, box=Ls,
                              image=orc.IMAGE_DEFINITION, rec_stride=1)
    states = np.concatenate([p64[None], traj])
    margin = min(guards.half_box_margin(q, Ls) for q in states)
    assert margin >= GUARD + guards.step_spread(states), (margin, guards.step_spread(states))
    want = traj[steps - 1]
    _, vlast, _ = orc.step(p64, F, wl.A, wl.ETA, dt, steps, oi, box=Ls, image=orc.IMAGE_DEFINITION)

    ctx = sd.Context(n, wl.A, wl.ETA)
    ctx.set_precision(getattr(sd, prec_name))
    ctx.set_box(L)
    dp = torch.from_numpy(p).cuda()
    gi = sd.INT_EULER if integ == "euler" else sd.INT_MIDPOINT
    ctx.step(dp, dt, steps, gi, gravity=(0.0, 0.0, -1.0))
    dv = torch.empty_like(dp)
    ctx.get_velocity(dv)
    torch.cuda.synchronize()
    got = dp.cpu().numpy()[:, :3].astype(np.float64)
    vmax = float(np.abs(vlast).max())
    eps = 2.0 ** -52 if prec_name == "PREC_F64" else 2.0 ** -23
    tol = TOL[prec_name] * vmax * steps * dt + eps * float(np.abs(want).max())
    assert np.abs(got - want).max() <= tol
    assert rel_err(dv.cpu().numpy()[:, :3].astype(np.float64), vlast) <= 10 * TOL[prec_name]
    assert (got[:, 2] - p64[:, 2]).mean() < -steps * dt
    # two more steps == one longer run (the state carried between calls is complete)
    ctx.step(dp, dt, 2, gi, gravity=(0.0, 0.0, -1.0))
    torch.cuda.synchronize()
    tol2 = TOL[prec_name] * vmax * (steps + 2) * dt + eps * float(np.abs(want2).max())
    assert np.abs(dp.cpu().numpy()[:, :3].astype(np.float64) - want2).max() <= tol2
    ctx.close()


@pytest.mark.parametrize("cells", [10, 11])
def test_fp32_euler_steps_on_the_commensurate_lattice_step_by_step(gpu, cells):
    """(c) above: the paper's benchmark shape itself in fp32.  Every Euler step starts from the
    positions the GPU holds (hi words; the low words are dropped on both sides by
    sd_reset_compensation), so GPU and oracle decide every image from identical fp32 numbers."""
    torch, sd = gpu
    pos = wl.fcc_lattice(cells, 0.1, jitter_seed=wl.SEED_BASE + 31 + cells)
    L = wl.fcc_box(cells, 0.1)
    n = pos.shape[0]
    ctx = sd.Context(n, wl.A, wl.ETA)
    ctx.set_box(L)
    dp = torch.from_numpy(wl.to_xyzw(pos, np.float32)).cuda()
    dv = torch.empty_like(dp)
    F = wl.gravity_forces(n)
    for _ in range(6):
        before = dp.cpu().numpy()[:, :3].astype(np.float64)
        ctx.reset_compensation()
        ctx.step(dp, 0.001, 1, sd.INT_EULER, gravity=(0.0, 0.0, -1.0))
        ctx.get_velocity(dv)
        torch.cuda.synchronize()
        want, vwant, _ = orc.step(before, F, wl.A, wl.ETA, 0.001, 1, orc.INT_EULER,
                                  box=float(np.float32(L)), image=orc.IMAGE_F32)
        assert rel_err(dv.cpu().numpy()[:, :3].astype(np.float64), vwant) <= 1e-5
        # positions: exact to the rounding of the stored fp32 word
        got = dp.cpu().numpy()[:, :3].astype(np.float64)
        assert np.abs(got - want).max() <= 1e-5 * 0.001 * np.abs(vwant).max() + 2.0 ** -24 * np.abs(want).max()
    ctx.close()


def test_box_at_bench_size_sampled_rows(gpu):
    """`bench.py --box` configuration (N = 1,048,576, fp32-Kahan, RPY, box = the cloud's own cube):
    4096 seeded rows against the oracle, plus a property that holds at any size: moving every
    particle by one box length along x leaves the velocities unchanged up to fp32 rounding."""
    torch, sd = gpu
    n = 1048576
    pos, force = wl.sweep(n)
    L = wl.cube_side(n, 0.01)
    got, p, f = gpu_apply_box(torch, sd, pos, force, L, "PREC_F32_KAHAN", 0, "i8_rpy_kahan_pbc")
    rows = wl.row_subset(n, 4096, wl.SEED_BASE + 90)
    want = orc.apply_rows(p, f, rows, wl.A, wl.ETA, box=float(np.float32(L)), image=orc.IMAGE_F32)
    assert rel_err(got[rows], want) <= TOL["PREC_F32_KAHAN"]
    assert np.all(np.isfinite(got))
    shifted = pos.copy()
    shifted[:, 0] += float(np.float32(L))
    got2, _, _ = gpu_apply_box(torch, sd, shifted, force, L, "PREC_F32_KAHAN", 0)
    # the shifted coordinates round differently in fp32 (|x| up to 1.5 L): input rounding, ~1e-4 a
    assert rel_err(got2[rows], got[rows]) <= 2e-3
