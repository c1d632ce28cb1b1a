"""GPU parity of the lubrication correction (Eq. 8) and of the
paper's full loop (forces corrected with the previous velocities) against the
CPU oracle, through the C ABI (`sd_lubrication_apply`, `sd_set_lubrication` + `sd_step`).

The cut-off r < 3a is a decision taken by floating point.  Two kinds of comparison:
 * against the oracle's PLAIN definition (`r < 3a` in double, `remainder` images) on clouds for
   which a CPU pre-check (tests/guards.py) asserts that no pair lies within GUARD = 1e-3 a of
   r = 3a -- products and whole trajectories, every particle held to the tolerance;
 * on clouds with pairs at any distance both sides take the decision in the kernel's arithmetic
   (reading C3; oracle `decide_f32`).
Accepted pairs are evaluated in fp64 on both sides, so the only fp32 error is the rounding of the
stored inputs and of the output.
"""
import numpy as np
import pytest

import guards

from oracle import sd_oracle as orc
from paper_1205_6333_b200 import workloads as wl

pytestmark = pytest.mark.gpu

IMAGE = {"PREC_F32_KAHAN": orc.IMAGE_F32, "PREC_F64": orc.IMAGE_F64}
GUARD = 1e-3   # a: distance every pair keeps from the cut-off r = 3a in the plain-definition tests


@pytest.fixture(scope="module")
def gpu():
    import torch
    from paper_1205_6333_b200 import sd
    assert torch.cuda.is_available()
    torch.cuda.set_device(0)
    sd.load_library()
    return torch, sd


def _dt(prec_name):
    return np.float64 if prec_name == "PREC_F64" else np.float32


def _row_err(got, want):
    scale = np.maximum(np.linalg.norm(want, axis=1), 1.0)
    return float(np.max(np.linalg.norm(got - want, axis=1) / scale))


@pytest.mark.parametrize("prec_name,tol", [("PREC_F32_KAHAN", 2e-7), ("PREC_F64", 1e-12)])
@pytest.mark.parametrize("boxed", [False, True])
@pytest.mark.parametrize("n,phi", [(50, 0.1), (1500, 0.05), (3000, 0.05), (4096, 0.2), (5000, 0.05),
                                   (40000, 0.05), (70001, 0.05), (50000, 0.3)])
def test_lubrication_apply_all_rows(gpu, prec_name, tol, boxed, n, phi):
    """Uniform clouds with overlaps allowed: pairs inside 3a (about 27 phi per sphere), in contact,
    overlapping (s clamped) and, when boxed, through the faces; per-particle external forces."""
    torch, sd = gpu
    dt = _dt(prec_name)
    L = wl.cube_side(n, phi)
    pos = wl.uniform_cube(n, phi, wl.SEED_BASE + 300 + n)
    if boxed:  # a third of the particles live in neighbouring periodic copies
        sh = np.random.Generator(np.random.PCG64(wl.SEED_BASE + 301)).integers(-1, 2, size=(n, 3))
        pos = pos + L * sh * (np.arange(n) % 3 == 0)[:, None]
    vel = wl.normal_forces(n, wl.SEED_BASE + 302 + n)
    fext = wl.normal_forces(n, wl.SEED_BASE + 303 + n)
    p, v, f = wl.to_xyzw(pos, dt), wl.to_xyzw(vel, dt), wl.to_xyzw(fext, dt)
    ctx = sd.Context(n, wl.A, wl.ETA)
    ctx.set_precision(getattr(sd, prec_name))
    if boxed:
        ctx.set_box(L)
    dp, dv, df = (torch.from_numpy(x).cuda() for x in (p, v, f))
    out = torch.full_like(dp, float("nan"))
    ctx.lubrication_apply(dp, dv, out, f_ext=df)
    out2 = torch.full_like(dp, float("nan"))
    ctx.lubrication_apply(dp, dv, out2, f_ext=df)
    torch.cuda.synchronize()
    got = out.cpu().numpy()
    assert np.array_equal(got, out2.cpu().numpy())            # deterministic despite the atomics
    assert np.all(got[:, 3] == 0.0)
    Ls = (float(np.float32(L)) if dt == np.float32 else L) if boxed else 0.0
    corr = orc.lubrication(p[:, :3].astype(np.float64), v[:, :3].astype(np.float64), wl.A, wl.ETA,
                           box=Ls, image=IMAGE[prec_name], decide_f32=(dt == np.float32))
    want = f[:, :3].astype(np.float64) - corr
    assert np.count_nonzero(np.abs(corr).sum(axis=1)) > 0.5 * n * min(1.0, 27 * phi * 0.5)
    assert _row_err(got[:, :3].astype(np.float64), want) <= tol
    # in place (force_out = f_ext) and with a uniform force instead of an array
    ctx.lubrication_apply(dp, dv, df, f_ext=df)
    out3 = torch.empty_like(dp)
    ctx.lubrication_apply(dp, dv, out3, gravity=(0.0, 0.0, -1.0))
    torch.cuda.synchronize()
    assert np.array_equal(df.cpu().numpy(), got)
    wantg = np.array([0.0, 0.0, -1.0]) - corr
    assert _row_err(out3.cpu().numpy()[:, :3].astype(np.float64), wantg) <= tol
    ctx.close()


@pytest.mark.parametrize("prec_name,tol", [("PREC_F32_KAHAN", 2e-7), ("PREC_F64", 1e-12)])
@pytest.mark.parametrize("boxed", [False, True])
@pytest.mark.parametrize("n0,phi", [(60, 0.1), (1500, 0.05), (3000, 0.05), (4096, 0.2), (5000, 0.05),
                                    (40000, 0.05), (70001, 0.05), (50000, 0.3)])
def test_lubrication_apply_against_the_plain_definition(gpu, prec_name, tol, boxed, n0, phi):
    """Eq. (8) with the cut-off decided as the paper states it (r < 3a, in double) and the plain
    `remainder` image: the same uniform clouds as above (overlaps, contacts, pairs through the
    faces) after one member of every pair within GUARD of r = 3a has been removed (CPU pre-check on
    the rounded coordinates; a component near half a box cannot matter here: such a pair is at
    least 4.5 a apart in either image).  All rows; every dispatch class: all pairs (N <= 1024), the
    one-launch grid (<= 4096), the cell grid with 32 / 8 / 1 lanes per particle (the last one with
    full queues at phi = 0.3)."""
    torch, sd = gpu
    dt = _dt(prec_name)
    L = wl.cube_side(n0, phi)
    pos = wl.uniform_cube(n0, phi, wl.SEED_BASE + 320 + n0)
    if boxed:
        sh = np.random.Generator(np.random.PCG64(wl.SEED_BASE + 321)).integers(-1, 2, size=(n0, 3))
        pos = pos + L * sh * (np.arange(n0) % 3 == 0)[:, None]
    Ls = (float(np.float32(L)) if dt == np.float32 else L) if boxed else 0.0
    p0 = wl.to_xyzw(pos, dt)[:, :3].astype(np.float64)
    near = guards.pairs_in_shell(p0, 3.0 * wl.A - GUARD, 3.0 * wl.A + GUARD, Ls)
    keep = guards.drop_one_of_each(n0, near)
    pos = pos[keep]
    n = pos.shape[0]
    assert n > 0.95 * n0
    assert guards.cutoff_margin(p0[keep], 3.0 * wl.A, Ls) >= GUARD
    vel = wl.normal_forces(n, wl.SEED_BASE + 322 + n0)
    fext = wl.normal_forces(n, wl.SEED_BASE + 323 + n0)
    p, v, f = wl.to_xyzw(pos, dt), wl.to_xyzw(vel, dt), wl.to_xyzw(fext, dt)
    ctx = sd.Context(n, wl.A, wl.ETA)
    ctx.set_precision(getattr(sd, prec_name))
    if boxed:
        ctx.set_box(L)
    dp, dv, df = (torch.from_numpy(x).cuda() for x in (p, v, f))
    out = torch.full_like(dp, float("nan"))
    ctx.lubrication_apply(dp, dv, out, f_ext=df)
    torch.cuda.synchronize()
    corr = orc.lubrication(p[:, :3].astype(np.float64), v[:, :3].astype(np.float64), wl.A, wl.ETA,
                           box=Ls, image=orc.IMAGE_DEFINITION, decide_f32=False)
    want = f[:, :3].astype(np.float64) - corr
    assert np.count_nonzero(np.abs(corr).sum(axis=1)) > 0.5 * n * min(1.0, 27 * phi * 0.5)
    assert _row_err(out.cpu().numpy()[:, :3].astype(np.float64), want) <= tol
    ctx.close()


@pytest.mark.parametrize("prec_name,tol", [("PREC_F32_KAHAN", 2e-7), ("PREC_F64", 1e-12)])
def test_lubrication_box_side_limits(gpu, prec_name, tol):
    """A pair inside 3a must have one nearest image: the box side has to exceed 6a.  The all-pairs
    kernel (N <= 1024, and up to 4096 when the box is too small for a grid) works from there on --
    checked against the plain definition in a box of 7a, where most pairs interact through a face --
    the cell grid above that size needs 9a."""
    torch, sd = gpu
    dt = _dt(prec_name)
    n = 40
    ctx = sd.Context(n, wl.A, wl.ETA)
    ctx.set_precision(getattr(sd, prec_name))
    z = torch.zeros((n, 4), device="cuda", dtype=torch.float64 if dt == np.float64 else torch.float32)
    for bad in (5.5, 6.0):
        ctx.set_box(bad)
        with pytest.raises(sd.SdError) as e:
            ctx.lubrication_apply(z, z.clone(), z.clone())
        assert e.value.status == sd.ERR_UNSUPPORTED
    L = 7.0
    ctx.set_box(L)
    pos = wl.rsa_cube(n, 4.0 / 3.0 * np.pi * n / L ** 3, wl.SEED_BASE + 340)   # fills the box of side L
    near = guards.pairs_in_shell(pos, 3.0 - GUARD, 3.0 + GUARD, L)
    assert near.shape[0] == 0
    vel = wl.normal_forces(n, wl.SEED_BASE + 341)
    p, v = wl.to_xyzw(pos, dt), wl.to_xyzw(vel, dt)
    out = torch.empty_like(z)
    ctx.lubrication_apply(torch.from_numpy(p).cuda(), torch.from_numpy(v).cuda(), out, gravity=(0.0, 0.0, -1.0))
    torch.cuda.synchronize()
    corr = orc.lubrication(p[:, :3].astype(np.float64), v[:, :3].astype(np.float64), wl.A, wl.ETA, box=L)
    assert np.count_nonzero(np.abs(corr).sum(axis=1)) > n // 2
    assert _row_err(out.cpu().numpy()[:, :3].astype(np.float64), np.array([0.0, 0.0, -1.0]) - corr) <= tol
    ctx.close()


@pytest.mark.parametrize("prec_name,tol", [("PREC_F32_KAHAN", 2e-7), ("PREC_F64", 1e-12)])
def test_lubrication_small_box_between_1024_and_4096_particles(gpu, prec_name, tol):
    """1024 < N <= 4096 in a box of 8a (two cells per edge: no grid): the all-pairs kernel, against
    the plain definition; N = 5000 in the same box is refused."""
    torch, sd = gpu
    dt = _dt(prec_name)
    n0, L = 1500, 8.0
    rng = np.random.Generator(np.random.PCG64(wl.SEED_BASE + 350))
    pos = rng.uniform(0.0, L, size=(n0, 3))           # heavily overlapping: s is clamped on most pairs
    Ls = float(np.float32(L)) if dt == np.float32 else L
    p0 = wl.to_xyzw(pos, dt)[:, :3].astype(np.float64)
    keep = guards.drop_one_of_each(n0, guards.pairs_in_shell(p0, 3.0 * wl.A - GUARD, 3.0 * wl.A + GUARD, Ls))
    pos = pos[keep][:1200]
    n = pos.shape[0]
    assert n > 1024
    vel = wl.normal_forces(n, wl.SEED_BASE + 351)
    p, v = wl.to_xyzw(pos, dt), wl.to_xyzw(vel, dt)
    ctx = sd.Context(n, wl.A, wl.ETA)
    ctx.set_precision(getattr(sd, prec_name))
    ctx.set_box(L)
    out = torch.full((n, 4), float("nan"), device="cuda", dtype=torch.float64 if dt == np.float64 else torch.float32)
    ctx.lubrication_apply(torch.from_numpy(p).cuda(), torch.from_numpy(v).cuda(), out, gravity=(0.0, 0.0, -1.0))
    torch.cuda.synchronize()
    corr = orc.lubrication(p[:, :3].astype(np.float64), v[:, :3].astype(np.float64), wl.A, wl.ETA,
                           box=Ls, image=orc.IMAGE_DEFINITION, decide_f32=False)
    assert _row_err(out.cpu().numpy()[:, :3].astype(np.float64), np.array([0.0, 0.0, -1.0]) - corr) <= tol
    ctx.close()
    ctx = sd.Context(5000, wl.A, wl.ETA)
    ctx.set_precision(getattr(sd, prec_name))
    ctx.set_box(L)
    z = torch.zeros((5000, 4), device="cuda", dtype=out.dtype)
    with pytest.raises(sd.SdError) as e:
        ctx.lubrication_apply(z, z.clone(), z.clone())
    assert e.value.status == sd.ERR_UNSUPPORTED
    ctx.close()


@pytest.mark.parametrize("prec_name,ptol,vtol", [("PREC_F32_KAHAN", 2e-5, 1e-4), ("PREC_F64", 1e-10, 1e-9)])
@pytest.mark.parametrize("n,integ,steps", [(2, "euler", 60), (300, "midpoint", 6), (300, "euler", 7),
                                           (3000, "euler", 5), (3000, "midpoint", 3)])
def test_step_with_lubrication_matches_the_papers_loop(gpu, prec_name, ptol, vtol, n, integ, steps):
    """sd_set_lubrication + sd_step against sdo_step_lub: N = 2 and 300 through the one-launch-per-
    product kernel, 3000 through the tiled kernels; random sequential addition with centre distances
    >= 2.6 a (every gap s >= 0.6: the paper's lagged-velocity scheme v_n = mu (F - zeta v_{n-1})
    diverges once |mu zeta| > 1, i.e. for gaps well below half a radius, on either side of the
    comparison), ~2 neighbours inside 3a per sphere, gravity + random forces; cold start.  Both
    sides decide the cut-off in the kernel's arithmetic; the long runs (CUDA-graph replay) against
    the plain definition are in test_long_runs_with_lubrication_against_the_plain_definition."""
    torch, sd = gpu
    dt_np = _dt(prec_name)
    if n == 2:
        pos = np.array([[0.0, 0.0, 1.3], [0.0, 0.0, -1.3]])
        fext = np.array([[0.0, 0.0, -1.0], [0.0, 0.0, 1.0]])     # pushed together, gap 0.6 a
    else:
        pos = wl.rsa_cube(n, 0.25, wl.SEED_BASE + 310 + n, a=1.3)
        fext = wl.gravity_forces(n) + 0.5 * wl.normal_forces(n, wl.SEED_BASE + 311 + n)
    p, f = wl.to_xyzw(pos, dt_np), wl.to_xyzw(fext, dt_np)
    dt = 0.01
    ctx = sd.Context(n, wl.A, wl.ETA)
    ctx.set_precision(getattr(sd, prec_name))
    ctx.set_lubrication(True)
    dp, df = torch.from_numpy(p).cuda(), torch.from_numpy(f).cuda()
    gi = sd.INT_EULER if integ == "euler" else sd.INT_MIDPOINT
    oi = orc.INT_EULER if integ == "euler" else orc.INT_MIDPOINT
    ctx.step(dp, dt, steps, gi, force=df)
    dv = torch.empty_like(dp)
    ctx.get_velocity(dv)
    torch.cuda.synchronize()
    p64, f64 = p[:, :3].astype(np.float64), f[:, :3].astype(np.float64)
    want_p, want_v = orc.step_lub(p64, np.zeros_like(p64), f64, wl.A, wl.ETA, dt, steps, oi,
                                  decide_f32=(dt_np == np.float32))
    got_p = dp.cpu().numpy()[:, :3].astype(np.float64)
    got_v = dv.cpu().numpy()[:, :3].astype(np.float64)
    assert np.abs(got_p - want_p).max() <= ptol
    assert _row_err(got_v, want_v) <= vtol
    # the correction is not a no-op on this input
    free_p, _, _ = orc.step(p64, f64, wl.A, wl.ETA, dt, steps, oi)
    assert np.abs(free_p - want_p).max() > 20 * ptol
    # continuing from the carried velocities == one longer run (state between calls is complete)
    ctx.step(dp, dt, 2, gi, force=df)
    torch.cuda.synchronize()
    want_p2, _ = orc.step_lub(p64, np.zeros_like(p64), f64, wl.A, wl.ETA, dt, steps + 2, oi,
                              decide_f32=(dt_np == np.float32))
    assert np.abs(dp.cpu().numpy()[:, :3].astype(np.float64) - want_p2).max() <= 2 * ptol
    ctx.close()


@pytest.mark.parametrize("prec_name", ["PREC_F32_KAHAN", "PREC_F64"])
@pytest.mark.parametrize("n,integ,steps,dt", [(300, "euler", 41, 5e-4), (300, "midpoint", 37, 5e-4),
                                              (3000, "euler", 35, 2e-4)])
def test_long_runs_with_lubrication_against_the_plain_definition(gpu, prec_name, n, integ, steps, dt):
    """Runs of 32 steps and more (captured CUDA graph of 16 steps per replay plus a direct tail)
    against sdo_step_lub with the cut-off decided in double (the paper's `r < 3a`), EVERY particle
    held to the tolerance.  The radial coefficient of Eq. (8) jumps by 1/(4 mu0) at r = 3a, so the
    cloud is built to stay clear of it: random sequential addition with centre distances >= 2.6 a
    and no pair between 2.8 a and 3.2 a, time steps short enough that no pair crosses that shell.
    Not assumed but asserted: the oracle trajectory is advanced step by step and at every step
    boundary every pair is at least GUARD + (largest relative displacement within one step) away
    from 3a.  Tolerance: the product's velocity tolerance integrated over the run, 1e-5 |v|_max t
    (fp32; 1e-10 in fp64: the lagged-velocity iteration amplifies rounding), plus the rounding of
    the stored position word."""
    torch, sd = gpu
    dt_np = _dt(prec_name)
    pos = wl.rsa_cube(n, 0.25, wl.SEED_BASE + 310 + n, a=1.3, shell=(2.8, 3.2))
    fext = wl.gravity_forces(n) + 0.5 * wl.normal_forces(n, wl.SEED_BASE + 311 + n)
    p, f = wl.to_xyzw(pos, dt_np), wl.to_xyzw(fext, dt_np)
    p64, f64 = p[:, :3].astype(np.float64), f[:, :3].astype(np.float64)
    oi = orc.INT_EULER if integ == "euler" else orc.INT_MIDPOINT
    # oracle, one step per call (the state between calls is (pos, vel)), plain definition
    states, q, v = [p64], p64, np.zeros_like(p64)
    for k in range(steps + 2):
        q, v = orc.step_lub(q, v, f64, wl.A, wl.ETA, dt, 1, oi, decide_f32=False)
        states.append(q)
        if k == steps - 1:
            want_p, want_v = q, v
    want_p2 = q
    one_call, _ = orc.step_lub(p64, np.zeros_like(p64), f64, wl.A, wl.ETA, dt, steps, oi)
    assert np.array_equal(one_call, want_p)
    states = np.asarray(states)
    margin = min(guards.cutoff_margin(s, 3.0 * wl.A) for s in states)
    assert margin >= GUARD + guards.step_spread(states), (margin, guards.step_spread(states))
    assert guards.pairs_in_shell(p64, 0.0, 3.0 * wl.A).shape[0] > n // 3    # lubrication pairs exist

    ctx = sd.Context(n, wl.A, wl.ETA)
    ctx.set_precision(getattr(sd, prec_name))
    ctx.set_lubrication(True)
    dp, df = torch.from_numpy(p).cuda(), torch.from_numpy(f).cuda()
    gi = sd.INT_EULER if integ == "euler" else sd.INT_MIDPOINT
    ctx.step(dp, dt, steps, gi, force=df)
    dv = torch.empty_like(dp)
    ctx.get_velocity(dv)
    torch.cuda.synchronize()
    got_p = dp.cpu().numpy()[:, :3].astype(np.float64)
    got_v = dv.cpu().numpy()[:, :3].astype(np.float64)
    vmax = float(np.abs(want_v).max())
    rel, eps = (1e-10, 2.0 ** -52) if prec_name == "PREC_F64" else (1e-5, 2.0 ** -23)
    tol = rel * vmax * steps * dt + eps * float(np.abs(want_p).max())
    assert np.abs(got_p - want_p).max() <= tol
    assert _row_err(got_v, want_v) <= (1e-9 if prec_name == "PREC_F64" else 1e-4)
    # the correction is not a no-op on this input
    free_p, _, _ = orc.step(p64, f64, wl.A, wl.ETA, dt, steps, oi)
    assert np.abs(free_p - want_p).max() > 100 * tol
    # continuing from the carried velocities == one longer run
    ctx.step(dp, dt, 2, gi, force=df)
    torch.cuda.synchronize()
    tol2 = rel * vmax * (steps + 2) * dt + eps * float(np.abs(want_p2).max())
    assert np.abs(dp.cpu().numpy()[:, :3].astype(np.float64) - want_p2).max() <= tol2
    ctx.close()


@pytest.mark.parametrize("prec_name", ["PREC_F32_KAHAN", "PREC_F64"])
@pytest.mark.parametrize("n,lub,boxed", [(300, True, False), (3000, True, False), (1331, False, True),
                                         (3375, False, True), (3375, True, True)])
def test_graph_replay_is_bit_identical_to_the_stepwise_loop(gpu, prec_name, n, lub, boxed):
    """sd_step replays a captured CUDA graph for runs of >= 32 constant-force steps; the same run
    issued as calls of 31 steps and fewer (never captured) must give the same bits, positions and
    velocities: the graph is a replay of the same launches, nothing else."""
    torch, sd = gpu
    dt_np = _dt(prec_name)
    if boxed:
        edge = round(n ** (1.0 / 3.0))
        dens = 0.04 if lub else 0.1   # lattice spacing 2.92 a: gaps of 0.9 a, inside the 3a cut-off
        pos = wl.sc_lattice(edge, dens, jitter_seed=wl.SEED_BASE + 40 + edge)
        L = wl.sc_box(edge, dens)
    else:
        pos = wl.rsa_cube(n, 0.25, wl.SEED_BASE + 310 + n, a=1.3)
        L = 0.0
    p = wl.to_xyzw(pos, dt_np)
    out = []
    for chunks in ((50,), (31, 19), (7, 31, 12)):
        ctx = sd.Context(n, wl.A, wl.ETA)
        ctx.set_precision(getattr(sd, prec_name))
        ctx.set_lubrication(lub)
        if boxed:
            ctx.set_box(L)
        dp = torch.from_numpy(p).cuda()
        for c in chunks:
            ctx.step(dp, 1e-3, c, sd.INT_MIDPOINT if n == 300 else sd.INT_EULER, gravity=(0.0, 0.3, -1.0))
        dv = torch.empty_like(dp)
        ctx.get_velocity(dv)
        torch.cuda.synchronize()
        out.append((dp.cpu().numpy(), dv.cpu().numpy()))
        ctx.close()
    for q, w in out[1:]:
        assert np.array_equal(q, out[0][0]) and np.array_equal(w, out[0][1])
    assert np.abs(out[0][0][:, :3] - p[:, :3]).max() > 1e-3


def test_graph_replay_follows_changes_of_arguments_and_settings(gpu):
    """sd_step replays a captured CUDA graph of 16 steps when the lubrication correction is on and
    the forces are constant.  Everything a capture bakes in -- dt, the position buffer, the force
    array / gravity, the integrator, the box, the position compensation -- must trigger a new
    capture when it changes.  fp64, N = 300, 34 steps per call, each call checked against the oracle
    continued from the state it left."""
    torch, sd = gpu
    n = 300
    pos = wl.rsa_cube(n, 0.25, wl.SEED_BASE + 310 + n, a=1.3)
    fext = wl.gravity_forces(n) + 0.5 * wl.normal_forces(n, wl.SEED_BASE + 311 + n)
    L = 1.5 * wl.cube_side(n, 0.25, a=1.3)
    ctx = sd.Context(n, wl.A, wl.ETA)
    ctx.set_precision(sd.PREC_F64)
    ctx.set_lubrication(True)
    state = {"p": pos.copy(), "v": np.zeros_like(pos)}

    def run(dp, dt, integ, force=None, gravity=None, box=0.0):
        f64 = fext if force is not None else wl.gravity_forces(n, gravity)
        ctx.step(dp, dt, 34, integ, force=force, gravity=gravity)
        torch.cuda.synchronize()
        oi = orc.INT_EULER if integ == sd.INT_EULER else orc.INT_MIDPOINT
        state["p"], state["v"] = orc.step_lub(state["p"], state["v"], f64, wl.A, wl.ETA, dt, 34, oi,
                                              box=box, image=orc.IMAGE_F64)
        state["calls"] = state.get("calls", 0) + 1
        err = np.abs(dp.cpu().numpy()[:, :3] - state["p"]).max()
        assert err <= 1e-9, f"call {state['calls']}: {err:.3e}"

    dp = torch.from_numpy(wl.to_xyzw(pos, np.float64)).cuda()
    df = torch.from_numpy(wl.to_xyzw(fext, np.float64)).cuda()
    run(dp, 0.002, sd.INT_EULER, force=df)
    run(dp, 0.002, sd.INT_EULER, force=df)                 # same key: replay
    run(dp, 0.001, sd.INT_EULER, force=df)                 # new dt
    run(dp, 0.001, sd.INT_MIDPOINT, force=df)              # new integrator
    dq = dp.clone()                                        # new position buffer
    run(dq, 0.001, sd.INT_MIDPOINT, force=df)
    run(dq, 0.001, sd.INT_EULER, gravity=(0.0, 0.3, -1.0))   # gravity instead of the force array
    run(dq, 0.001, sd.INT_EULER, gravity=(0.0, -0.3, -1.0))
    ctx.set_box(L)                                         # same kernels, new constants
    run(dq, 0.001, sd.INT_EULER, gravity=(0.0, -0.3, -1.0), box=L)
    ctx.set_lubrication(False)                             # and off again: plain loop
    ctx.step(dq, 0.001, 34, sd.INT_EULER, gravity=(0.0, -0.3, -1.0))
    torch.cuda.synchronize()
    want, _, _ = orc.step(state["p"], wl.gravity_forces(n, (0.0, -0.3, -1.0)), wl.A, wl.ETA, 0.001, 34,
                          orc.INT_EULER, box=L, image=orc.IMAGE_F64)
    assert np.abs(dq.cpu().numpy()[:, :3] - want).max() <= 1e-9
    ctx.close()


def test_previous_velocities_start_at_zero_in_recycled_memory(gpu):
    """Regression: the context-owned velocities ("of the previous step", reading C4) must be zero
    after sd_create even when cudaMalloc hands back the block a closed context left full of
    velocities (a missing memset showed up as order-dependent failures of the tests above)."""
    torch, sd = gpu
    n = 700
    pos = wl.rsa_cube(n, 0.25, wl.SEED_BASE + 333, a=1.3)
    p = wl.to_xyzw(pos, np.float32)
    for cycle in range(4):
        ctx = sd.Context(n, wl.A, wl.ETA)
        dv = torch.full((n, 4), float("nan"), device="cuda")
        ctx.get_velocity(dv)
        torch.cuda.synchronize()
        assert np.all(dv.cpu().numpy() == 0.0), f"cycle {cycle}"
        ctx.set_lubrication(True)
        dp = torch.from_numpy(p).cuda()
        ctx.step(dp, 0.01, 3, sd.INT_EULER, gravity=(0.0, 0.0, -1.0))   # leaves |v| ~ 10 behind
        ctx.get_velocity(dv)
        torch.cuda.synchronize()
        assert np.abs(dv.cpu().numpy()).max() > 1.0
        ctx.close()
