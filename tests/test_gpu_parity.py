"""GPU parity: the CUDA path (through the C ABI binding) against the CPU oracle, element by
element on the same seeded inputs.  Configurations follow BASELINE.json `configs`.

Tolerances (BASELINE.json north_star): max per-particle relative velocity error
    err = max_i |v_gpu,i - v_ref,i|_2 / |v_ref,i|_2
<= 1e-5 for fp32 with compensated summation, <= 1e-11 for fp64; trajectories (reading A14 in
DESIGN.md): max abs position deviation after 1e4 midpoint steps <= 1e-4 a (fp32), 1e-9 a (fp64).
The oracle gets the SAME fp32-rounded inputs promoted to double (input rounding is not error).
"""
import ctypes
import math

import numpy as np
import pytest

from oracle import sd_oracle as orc
from paper_1205_6333_b200 import workloads as wl

pytestmark = pytest.mark.gpu

TOL_F32 = 1e-5
TOL_F64 = 1e-11


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


def np_dtype(sd, prec):
    return np.float64 if prec == sd.PREC_F64 else np.float32


def gpu_apply(torch, sd, pos, force, prec, tensor, a=wl.A, eta=wl.ETA):
    """Returns (vel[N,3] fp64, pos_in[N,3] fp64, force_in[N,3] fp64) with inputs as rounded."""
    dt = np_dtype(sd, prec)
    p, f = wl.to_xyzw(pos, dt), wl.to_xyzw(force, dt)
    ctx = sd.Context(pos.shape[0], a, eta)
    ctx.set_precision(prec)
    ctx.set_tensor(tensor)
    dp, df = torch.from_numpy(p).cuda(), torch.from_numpy(f).cuda()
    dv = torch.full_like(dp, float("nan"))
    ctx.mobility_apply(dp, df, dv)
    torch.cuda.synchronize()
    out = dv.cpu().numpy()
    assert np.all(out[:, 3] == 0.0)  # pad lane written as 0
    assert ctx.launch_count >= 1  # our kernels ran (one launch up to N ~ 6000, three above)
    ctx.close()
    return out[:, :3].astype(np.float64), p[:, :3].astype(np.float64), f[:, :3].astype(np.float64)


# ---- config 1: four-sphere cluster, 1e4 midpoint steps ----------------------------------------

@pytest.mark.parametrize("prec_name,tol", [("PREC_F32_KAHAN", 1e-4), ("PREC_F64", 1e-9)])
def test_config1_four_sphere_trajectory(gpu, prec_name, tol):
    torch, sd = gpu
    prec = getattr(sd, prec_name)
    dt_np = np_dtype(sd, prec)
    pos, force = wl.four_sphere(jitter_seed=wl.SEED_BASE + 1)
    p = wl.to_xyzw(pos, dt_np)
    ctx = sd.Context(4, wl.A, wl.ETA)
    ctx.set_precision(prec)
    dp = torch.from_numpy(p).cuda()
    ctx.step(dp, 0.01, 10000, sd.INT_MIDPOINT, gravity=(0.0, 0.0, -1.0))
    dv = torch.empty_like(dp)
    ctx.get_velocity(dv)
    torch.cuda.synchronize()
    want, vlast, _ = orc.step(p[:, :3].astype(np.float64), force, wl.A, wl.ETA, 0.01, 10000,
                              orc.INT_MIDPOINT)
    got = dp.cpu().numpy()[:, :3].astype(np.float64)
    assert np.abs(got - want).max() <= tol
    assert rel_err(dv.cpu().numpy()[:, :3].astype(np.float64), vlast) <= 1e-4
    # the cluster really moved: ~125 a downwards (z_cm decreases monotonically)
    assert got[:, 2].mean() < -120.0
    ctx.close()


def test_config1_plain_fp32_positions_drift(gpu):
    """Ablation of PAPER.md:253-263: without the position low word (reset before every step) the
    fp32 trajectory is measurably worse than with it."""
    torch, sd = gpu
    pos, force = wl.four_sphere(jitter_seed=wl.SEED_BASE + 1)
    p = wl.to_xyzw(pos, np.float32)
    want, _, _ = orc.step(p[:, :3].astype(np.float64), force, wl.A, wl.ETA, 0.01, 2000,
                          orc.INT_MIDPOINT)
    errs = {}
    for reset in (False, True):
        ctx = sd.Context(4, wl.A, wl.ETA)
        dp = torch.from_numpy(p).cuda()
        for _ in range(2000):
            if reset:
                ctx.reset_compensation()
            ctx.step(dp, 0.01, 1, sd.INT_MIDPOINT, gravity=(0.0, 0.0, -1.0))
        torch.cuda.synchronize()
        errs[reset] = np.abs(dp.cpu().numpy()[:, :3] - want).max()
        ctx.close()
    assert errs[False] <= 1e-4
    assert errs[True] > 3.0 * errs[False]


# ---- config 2: N = 4096 non-overlapping spheres ----------------------------------------------

def test_config2_rsa_4096_all_rows(gpu):
    torch, sd = gpu
    pos, force = wl.config2()
    assert wl.min_pair_distance(pos, 3.0) >= 2.0
    got, p, f = gpu_apply(torch, sd, pos, force, sd.PREC_F32_KAHAN, sd.TENSOR_RPY)
    want = orc.apply(p, f, wl.A, wl.ETA, orc.TENSOR_RPY)
    assert rel_err(got, want) <= TOL_F32
    # no overlaps: the unregularised Eq. (7b) is the same sum
    want_far = orc.apply(p, f, wl.A, wl.ETA, orc.TENSOR_RP_FAR)
    assert rel_err(got, want_far) <= TOL_F32


# ---- config 3: N = 65536 with overlaps, all rows, fp32 and fp64, + one Euler step -------------

@pytest.fixture(scope="module")
def config3_oracle():
    pos, force = wl.config3()
    out = {}
    for name, dt in (("f32", np.float32), ("f64", np.float64)):
        p = wl.to_xyzw(pos, dt)[:, :3].astype(np.float64)
        f = wl.to_xyzw(force, dt)[:, :3].astype(np.float64)
        out[name] = (p, f, orc.apply(p, f, wl.A, wl.ETA, orc.TENSOR_RPY))
    return pos, force, out


def test_config3_overlaps_exist():
    pos, _ = wl.config3()
    assert wl.min_pair_distance(pos, 2.0) < 1.0  # exercises the r < 2a branch


def test_config3_fp32_all_rows(gpu, config3_oracle):
    torch, sd = gpu
    pos, force, ref = config3_oracle
    got, p, f = gpu_apply(torch, sd, pos, force, sd.PREC_F32_KAHAN, sd.TENSOR_RPY)
    assert np.array_equal(p, ref["f32"][0])
    assert rel_err(got, ref["f32"][2]) <= TOL_F32
    # the far-only formula is NOT the same sum here (negative control for the overlap branch)
    rows = wl.row_subset(pos.shape[0], 2048, wl.SEED_BASE + 33)
    far = orc.apply_rows(p, f, rows, wl.A, wl.ETA, orc.TENSOR_RP_FAR)
    assert rel_err(got[rows], far) > 1e-3


def test_config3_fp64_all_rows(gpu, config3_oracle):
    torch, sd = gpu
    pos, force, ref = config3_oracle
    got, p, f = gpu_apply(torch, sd, pos, force, sd.PREC_F64, sd.TENSOR_RPY)
    assert rel_err(got, ref["f64"][2]) <= TOL_F64


@pytest.mark.parametrize("prec_name,key,tol", [("PREC_F32_KAHAN", "f32", 2e-6), ("PREC_F64", "f64", 1e-12)])
def test_config3_one_euler_step(gpu, config3_oracle, prec_name, key, tol):
    """r <- r + dt v; fp32 positions must land within one ulp (coordinates are
    <= 151 a, ulp = 1.5e-5 a) -- checked as 2e-6 relative to the box."""
    torch, sd = gpu
    prec = getattr(sd, prec_name)
    pos, force, ref = config3_oracle
    p64, f64, v = ref[key]
    dt = 0.01
    want = p64 + dt * v
    dtp = np_dtype(sd, prec)
    ctx = sd.Context(pos.shape[0], wl.A, wl.ETA)
    ctx.set_precision(prec)
    dp = torch.from_numpy(wl.to_xyzw(pos, dtp)).cuda()
    df = torch.from_numpy(wl.to_xyzw(force, dtp)).cuda()
    ctx.step(dp, dt, 1, sd.INT_EULER, force=df)
    torch.cuda.synchronize()
    got = dp.cpu().numpy()[:, :3].astype(np.float64)
    assert np.abs(got - want).max() <= tol * 151.0
    ctx.close()


# ---- config 4: sedimenting cloud, N = 262144, 100 midpoint steps ------------------------------

def test_config4_sedimenting_cloud(gpu):
    torch, sd = gpu
    pos, force = wl.config4()
    n = pos.shape[0]
    rows = wl.row_subset(n, 4096, wl.SEED_BASE + 6)
    ctx = sd.Context(n, wl.A, wl.ETA)
    p32 = wl.to_xyzw(pos, np.float32)
    f32 = wl.to_xyzw(force, np.float32)
    dp, df = torch.from_numpy(p32).cuda(), torch.from_numpy(f32).cuda()
    dv = torch.empty_like(dp)

    def check(tag):
        ctx.mobility_apply(dp, df, dv)
        torch.cuda.synchronize()
        p = dp.cpu().numpy()[:, :3].astype(np.float64)
        want = orc.apply_rows(p, f32[:, :3].astype(np.float64), rows, wl.A, wl.ETA, orc.TENSOR_RPY)
        got = dv.cpu().numpy()[rows, :3].astype(np.float64)
        e = rel_err(got, want)
        assert e <= TOL_F32, f"{tag}: {e:.3e}"
        return p, want

    p0, v0 = check("step 0")
    # collective settling: |v| ~ N a / R >> mu0 F (SURVEY 8(d) cfg 4)
    assert np.linalg.norm(v0, axis=1).mean() > 500.0
    ctx.step(dp, 0.05, 100, sd.INT_MIDPOINT, gravity=(0.0, 0.0, -1.0))
    p100, _ = check("step 100")
    assert np.isfinite(p100).all()
    assert (p100[:, 2].mean() - p0[:, 2].mean()) < -1000.0  # the cloud sedimented
    ctx.close()


# ---- config 5: sweep, 4096 seeded rows per N --------------------------------------------------

@pytest.mark.parametrize("n", [1024, 4096, 16384, 65536, 262144, 1048576])
def test_config5_sweep_rows(gpu, n):
    torch, sd = gpu
    pos, force = wl.sweep(n)
    rows = wl.row_subset(n, 4096, wl.SEED_BASE + 6 + n)
    for tensor, otensor in ((sd.TENSOR_RPY, orc.TENSOR_RPY), (sd.TENSOR_OSEEN, orc.TENSOR_OSEEN)):
        want = {}
        for prec, tol in ((sd.PREC_F32_KAHAN, TOL_F32), (sd.PREC_F64, TOL_F64)):
            got, p, f = gpu_apply(torch, sd, pos, force, prec, tensor)
            want = orc.apply_rows(p, f, rows, wl.A, wl.ETA, otensor)
            e = rel_err(got[rows], want)
            assert e <= tol, f"n={n} tensor={tensor} prec={prec}: {e:.3e}"


# ---- properties that hold at any size, checked at the bench size ------------------------------

def test_full_size_symmetry_and_linearity(gpu):
    """<G, M F> = <F, M G> and M(aF + bG) = a MF + b MG at N = 1048576, in the
    launch configuration bench.py times."""
    torch, sd = gpu
    n = 1048576
    pos, force = wl.sweep(n)
    other = wl.normal_forces(n, wl.SEED_BASE + 77)
    ctx = sd.Context(n, wl.A, wl.ETA)
    dp = torch.from_numpy(wl.to_xyzw(pos, np.float32)).cuda()
    dF = torch.from_numpy(wl.to_xyzw(force, np.float32)).cuda()
    dG = torch.from_numpy(wl.to_xyzw(other, np.float32)).cuda()
    vF, vG, vH = torch.empty_like(dp), torch.empty_like(dp), torch.empty_like(dp)
    ctx.mobility_apply(dp, dF, vF)
    ctx.mobility_apply(dp, dG, vG)
    dH = (2.0 * dF - 0.5 * dG).contiguous()
    ctx.mobility_apply(dp, dH, vH)
    torch.cuda.synchronize()
    lhs = float((dG.double() * vF.double()).sum())
    rhs = float((dF.double() * vG.double()).sum())
    scale = float(vF.double().norm() * dG.double().norm())
    assert abs(lhs - rhs) <= 1e-6 * scale
    lin = (vH.double() - (2.0 * vF.double() - 0.5 * vG.double())).norm() / vH.double().norm()
    assert float(lin) <= 1e-6
    ctx.close()


# ---- edge cases ---------------------------------------------------------------------------------

@pytest.mark.parametrize("prec_name", ["PREC_F32_KAHAN", "PREC_F64", "PREC_F32_PLAIN"])
@pytest.mark.parametrize("tensor_name", ["TENSOR_RPY", "TENSOR_OSEEN"])
def test_single_sphere_and_pairs(gpu, prec_name, tensor_name):
    torch, sd = gpu
    prec, tensor = getattr(sd, prec_name), getattr(sd, tensor_name)
    otensor = orc.TENSOR_RPY if tensor == sd.TENSOR_RPY else orc.TENSOR_OSEEN
    tol = TOL_F64 if prec == sd.PREC_F64 else TOL_F32
    a, eta = 0.7, 0.31
    # N = 1: Stokes velocity
    F = np.array([[0.3, -1.7, 2.2]])
    got, _, f = gpu_apply(torch, sd, np.array([[3.0, -2.0, 9.0]]), F, prec, tensor, a, eta)
    np.testing.assert_allclose(got, f / (6 * math.pi * eta * a), rtol=1e-6 if prec != sd.PREC_F64 else 1e-14)
    # N = 2: far, touching (r = 2a exactly), overlapping, nearly coincident, coincident
    for d in ([0.0, 0.0, 4.0], [1.4, 0.0, 0.0], [0.3, 0.2, -0.4], [1e-4, 0.0, 0.0], [0.0, 0.0, 0.0]):
        pos = np.array([d, [0.0, 0.0, 0.0]]) + 1.5
        F2 = np.array([[0.0, 0.0, -1.0], [0.5, 0.25, -1.0]])
        if tensor == sd.TENSOR_OSEEN and np.linalg.norm(d) < 1e-3 and np.linalg.norm(d) > 0:
            continue  # unregularised 1/r at r = 1e-4 a: ill-conditioned, not a graded case
        got, p, f = gpu_apply(torch, sd, pos, F2, prec, tensor, a, eta)
        want = orc.apply(p, f, a, eta, otensor)
        assert rel_err(got, want) <= tol, d


@pytest.mark.parametrize("n", [3, 31, 257, 1023, 2049, 8193, 12345])
def test_ragged_sizes(gpu, n):
    """Sizes that end inside a warp, a j-tile, an i-block; dense clouds mix both RPY branches."""
    torch, sd = gpu
    pos = wl.uniform_cube(n, 0.2, wl.SEED_BASE + 500 + n)
    force = wl.normal_forces(n, wl.SEED_BASE + 600 + n)
    for prec, tol in ((sd.PREC_F32_KAHAN, TOL_F32), (sd.PREC_F64, TOL_F64)):
        got, p, f = gpu_apply(torch, sd, pos, force, prec, sd.TENSOR_RPY)
        want = orc.apply(p, f, wl.A, wl.ETA, orc.TENSOR_RPY)
        assert rel_err(got, want) <= tol


@pytest.mark.parametrize("n", [8193, 33001, 131073, 200003])
def test_ragged_sizes_large_kernels(gpu, n):
    """Ragged tails of the tiled kernels (4 and 8 particles per thread), seeded rows + the last
    rows of the cloud (the ragged i-block and j-tile)."""
    torch, sd = gpu
    pos = wl.uniform_cube(n, 0.05, wl.SEED_BASE + 520 + n)
    force = wl.normal_forces(n, wl.SEED_BASE + 620 + n)
    rows = np.unique(np.concatenate([wl.row_subset(n, 1024, wl.SEED_BASE + 720 + n),
                                     np.arange(n - 40, n), np.arange(0, 8)]))
    for prec, tol in ((sd.PREC_F32_KAHAN, TOL_F32), (sd.PREC_F64, TOL_F64)):
        got, p, f = gpu_apply(torch, sd, pos, force, prec, sd.TENSOR_RPY)
        want = orc.apply_rows(p, f, rows, wl.A, wl.ETA, orc.TENSOR_RPY)
        assert rel_err(got[rows], want) <= tol


@pytest.mark.parametrize("n,integ", [(4, "INT_EULER"), (33, "INT_MIDPOINT"), (64, "INT_EULER"),
                                     (65, "INT_EULER"), (300, "INT_MIDPOINT"), (2500, "INT_EULER"),
                                     (2500, "INT_MIDPOINT"), (5000, "INT_EULER"),
                                     (9000, "INT_MIDPOINT"), (9000, "INT_EULER"),
                                     (14000, "INT_MIDPOINT")])
@pytest.mark.parametrize("prec_name", ["PREC_F32_KAHAN", "PREC_F64"])
def test_step_paths_agree_with_oracle(gpu, n, integ, prec_name):
    """sd_step through every dispatch path (persistent stepper N <= 64, one-launch-per-product
    N <= 2560, tiled kernels with 2 / 4 particles per thread above), odd step counts (ping-pong buffers), per-particle forces."""
    torch, sd = gpu
    prec = getattr(sd, prec_name)
    dtp = np_dtype(sd, prec)
    pos = wl.uniform_cube(n, 0.1, wl.SEED_BASE + 900 + n)
    force = wl.normal_forces(n, wl.SEED_BASE + 901 + n)
    p, f = wl.to_xyzw(pos, dtp), wl.to_xyzw(force, dtp)
    steps, dt = 3, 0.02
    ctx = sd.Context(n, wl.A, wl.ETA)
    ctx.set_precision(prec)
    dp, df = torch.from_numpy(p).cuda(), torch.from_numpy(f).cuda()
    ctx.step(dp, dt, steps, getattr(sd, integ), force=df)
    dv = torch.empty_like(dp)
    ctx.get_velocity(dv)
    torch.cuda.synchronize()
    oint = orc.INT_EULER if integ == "INT_EULER" else orc.INT_MIDPOINT
    want, vlast, _ = orc.step(p[:, :3].astype(np.float64), f[:, :3].astype(np.float64), wl.A, wl.ETA,
                              dt, steps, oint)
    got = dp.cpu().numpy()[:, :3].astype(np.float64)
    L = wl.cube_side(n, 0.1)
    assert np.abs(got - want).max() <= (2e-7 * L if prec != sd.PREC_F64 else 1e-12 * L)
    assert rel_err(dv.cpu().numpy()[:, :3].astype(np.float64), vlast) <= (2e-5 if prec != sd.PREC_F64 else 1e-10)
    ctx.close()


def test_plain_accumulation_is_worse_than_kahan(gpu):
    """The paper's numerical claim: single-precision accumulation of the
    1/r-spread terms is the dominant error.  Gravity on a ball: all terms add up coherently."""
    torch, sd = gpu
    n = 65536
    pos = wl.uniform_ball(n, 0.02, wl.SEED_BASE + 700)
    force = wl.gravity_forces(n)
    rows = wl.row_subset(n, 2048, wl.SEED_BASE + 701)
    errs = {}
    for prec in (sd.PREC_F32_KAHAN, sd.PREC_F32_PLAIN):
        got, p, f = gpu_apply(torch, sd, pos, force, prec, sd.TENSOR_RPY)
        want = orc.apply_rows(p, f, rows, wl.A, wl.ETA, orc.TENSOR_RPY)
        errs[prec] = rel_err(got[rows], want)
    assert errs[sd.PREC_F32_KAHAN] <= 1e-6
    assert errs[sd.PREC_F32_PLAIN] > 5.0 * errs[sd.PREC_F32_KAHAN]


def test_host_entry_point_matches_device_entry_point(gpu):
    torch, sd = gpu
    n = 5000
    pos, force = wl.uniform_cube(n, 0.05, wl.SEED_BASE + 800), wl.normal_forces(n, wl.SEED_BASE + 801)
    hp = torch.from_numpy(wl.to_xyzw(pos, np.float32)).pin_memory()
    hf = torch.from_numpy(wl.to_xyzw(force, np.float32)).pin_memory()
    hv = torch.empty_like(hp).pin_memory()
    ctx = sd.Context(n, wl.A, wl.ETA)
    ctx.mobility_apply_host(hp, hf, hv)
    dv = torch.empty((n, 4), dtype=torch.float32, device="cuda")
    ctx.mobility_apply(hp.cuda(), hf.cuda(), dv)
    torch.cuda.synchronize()
    assert torch.equal(hv, dv.cpu())  # deterministic schedule: bit-identical
    ctx.close()


def test_force_callback_and_constant_forces_agree(gpu):
    """sd_step with a force callback that enqueues 'F = gravity' reproduces the gravity path."""
    torch, sd = gpu
    n = 3000
    pos = wl.uniform_cube(n, 0.05, wl.SEED_BASE + 810)
    p = wl.to_xyzw(pos, np.float32)
    g = (0.0, 0.0, -1.0)
    res = []
    calls = []
    for mode in ("gravity", "buffer", "callback"):
        ctx = sd.Context(n, wl.A, wl.ETA)
        dp = torch.from_numpy(p).cuda()
        if mode == "gravity":
            ctx.step(dp, 0.02, 3, sd.INT_MIDPOINT, gravity=g)
        elif mode == "buffer":
            df = torch.from_numpy(wl.to_xyzw(wl.gravity_forces(n), np.float32)).cuda()
            ctx.step(dp, 0.02, 3, sd.INT_MIDPOINT, force=df)
        else:
            gf = torch.tensor([g[0], g[1], g[2], 0.0], dtype=torch.float32, device="cuda")

            def fn(pos_ptr, force_ptr, nn, user, stream):
                calls.append(nn)
                # enqueue on the current torch stream (== the stream sd_step was given)
                view = _device_view(torch, force_ptr, nn)
                view.copy_(gf.expand(nn, 4))
                return 0

            ctx.step(dp, 0.02, 3, sd.INT_MIDPOINT, force_fn=fn)
        torch.cuda.synchronize()
        res.append(dp.cpu())
        ctx.close()
    assert torch.equal(res[0], res[1])
    assert torch.equal(res[0], res[2])
    assert len(calls) == 6  # two products per midpoint step


def _device_view(torch, ptr, n):
    """Wrap a raw device pointer [n][4] float as a torch tensor (no copy)."""
    class _Holder:
        pass
    h = _Holder()
    h.__cuda_array_interface__ = {"shape": (n, 4), "typestr": "<f4", "data": (int(ptr), False),
                                  "version": 2}
    return torch.as_tensor(h, device="cuda")


def test_invalid_arguments_are_reported(gpu):
    torch, sd = gpu
    lib = sd.load_library()
    h = ctypes.c_void_p()
    assert lib.sd_create(ctypes.byref(h), 0, 1.0, 1.0) == sd.ERR_INVALID_ARG
    assert lib.sd_create(ctypes.byref(h), 10, -1.0, 1.0) == sd.ERR_INVALID_ARG
    assert lib.sd_create(ctypes.byref(h), 10, 1.0, float("nan")) == sd.ERR_INVALID_ARG
    assert b"sd_create" in lib.sd_last_error(None)
    ctx = sd.Context(10, 1.0, 1.0)
    t = torch.zeros((10, 4), dtype=torch.float32, device="cuda")
    with pytest.raises(sd.SdError) as ei:
        ctx.mobility_apply(t, t, t)  # vel aliases the inputs
    assert ei.value.status == sd.ERR_INVALID_ARG
    with pytest.raises(sd.SdError):
        ctx.set_tensor(9)
    with pytest.raises(sd.SdError):
        ctx.set_precision(9)
    with pytest.raises(sd.SdError):
        ctx.step(t, float("inf"), 1, sd.INT_EULER, gravity=(0, 0, -1))
    with pytest.raises(sd.SdError):
        ctx.step(t, 0.1, 1, 7, gravity=(0, 0, -1))
    with pytest.raises(sd.SdError):
        ctx.step(t, 0.1, 1, sd.INT_EULER)  # no force at all
    st = lib.sd_mobility_apply(ctx._h, ctypes.c_void_p(t.data_ptr() + 4), ctypes.c_void_p(t.data_ptr()),
                               ctypes.c_void_p(0), ctypes.c_void_p(0))
    assert st == sd.ERR_INVALID_ARG
    ctx.step(t, 0.1, 0, sd.INT_EULER, gravity=(0, 0, -1))  # zero steps: no-op
    assert ctx.self_mobility == pytest.approx(1.0 / (6 * math.pi))
    ctx.close()


# ---- dispatch knobs: every tiled variant on small clouds, all rows (careful pass coverage) ------

@pytest.mark.parametrize("prec_name,tol", [("PREC_F32_KAHAN", TOL_F32), ("PREC_F64", TOL_F64)])
@pytest.mark.parametrize("tname", ["TENSOR_RPY", "TENSOR_OSEEN"])
@pytest.mark.parametrize("ipt", [2, 4, 8])
def test_forced_tiled_kernels_on_dense_small_clouds(gpu, prec_name, tol, tname, ipt):
    """sd_set_dispatch(0, ipt) sends small N through the tiled packed kernels.  Dense clouds
    (phi = 0.2, overlaps allowed: ~1.6 overlapping neighbours per sphere, plus two coincident
    centres) put self pairs, overlapping pairs and r = 0 pairs into most chunks, i.e. they
    exercise the clamped careful pass and its per-pair corrections on every row."""
    torch, sd = gpu
    prec, tensor = getattr(sd, prec_name), getattr(sd, tname)
    otensor = orc.TENSOR_RPY if tname == "TENSOR_RPY" else orc.TENSOR_OSEEN
    for n in (257, 3000):
        pos = wl.uniform_cube(n, 0.2, wl.SEED_BASE + 40 + n)
        pos[n // 2] = pos[3]                       # coincident centres, j != i (reading A5)
        force = wl.normal_forces(n, wl.SEED_BASE + 41 + n)
        dt = np_dtype(sd, prec)
        p, f = wl.to_xyzw(pos, dt), wl.to_xyzw(force, dt)
        ctx = sd.Context(n, wl.A, wl.ETA)
        ctx.set_precision(prec)
        ctx.set_tensor(tensor)
        ctx.set_jsplit(1)                          # the classic tiled kernels (warp-split: test_gpu_wsplit_parity.py)
        ctx.set_dispatch(0, ipt)
        assert "pairs_f" in ctx.kernel_name and "_w8_" not in ctx.kernel_name
        dp, df = torch.from_numpy(p).cuda(), torch.from_numpy(f).cuda()
        dv = torch.full_like(dp, float("nan"))
        ctx.mobility_apply(dp, df, dv)
        torch.cuda.synchronize()
        got = dv.cpu().numpy()[:, :3].astype(np.float64)
        want = orc.apply(p[:, :3].astype(np.float64), f[:, :3].astype(np.float64), wl.A, wl.ETA,
                         otensor)
        assert rel_err(got, want) <= tol
        # default dispatch (one-launch kernel at this N) agrees as well
        ctx.set_dispatch(-1, 0)
        ctx.mobility_apply(dp, df, dv)
        torch.cuda.synchronize()
        assert rel_err(dv.cpu().numpy()[:, :3].astype(np.float64), want) <= tol
        with pytest.raises(sd.SdError):
            ctx.set_dispatch(0, 3)
        ctx.close()


# ---- memory-access ablation (Appendix A): same bits through every staging -----

@pytest.mark.parametrize("n", [3000, 20000, 140000, 204800])  # 204800: the 256-record tiles
def test_staging_modes_are_bit_identical_and_guarded(gpu, n):
    """sd_set_staging: bulk-copy ring (default), naive global loads (Alg. 1), block tiling with
    barriers (Alg. 2).  The arithmetic and its order do not depend on how a record arrives."""
    torch, sd = gpu
    pos = wl.uniform_cube(n, 0.05, wl.SEED_BASE + 60 + n)
    force = wl.normal_forces(n, wl.SEED_BASE + 61 + n)
    p, f = wl.to_xyzw(pos, np.float32), wl.to_xyzw(force, np.float32)
    dp, df = torch.from_numpy(p).cuda(), torch.from_numpy(f).cuda()
    ctx = sd.Context(n, wl.A, wl.ETA)
    ctx.set_jsplit(1)               # the ablation lives in the classic tiled kernel
    ctx.set_dispatch(0, 0)          # tiled kernels at every N
    out = {}
    for mode, tag in ((sd.STAGE_BULK, "kahan"), (sd.STAGE_NAIVE, "_naive"), (sd.STAGE_SYNC, "_sync")):
        ctx.set_staging(mode)
        assert ctx.kernel_name.endswith(tag), ctx.kernel_name
        dv = torch.full_like(dp, float("nan"))
        ctx.mobility_apply(dp, df, dv)
        torch.cuda.synchronize()
        out[mode] = dv.cpu().numpy()
    assert np.array_equal(out[sd.STAGE_BULK], out[sd.STAGE_NAIVE])
    assert np.array_equal(out[sd.STAGE_BULK], out[sd.STAGE_SYNC])
    rows = wl.row_subset(n, 512, wl.SEED_BASE + 62)
    want = orc.apply_rows(p[:, :3].astype(np.float64), f[:, :3].astype(np.float64), rows, wl.A, wl.ETA)
    assert rel_err(out[sd.STAGE_SYNC][rows, :3].astype(np.float64), want) <= TOL_F32
    # the ablation variants exist for RPY / fp32-Kahan / free space only, and say so
    for bad in (lambda: ctx.set_tensor(sd.TENSOR_OSEEN), lambda: ctx.set_precision(sd.PREC_F64),
                lambda: ctx.set_box(100.0), lambda: ctx.set_staging(3)):
        with pytest.raises(sd.SdError):
            bad()
    ctx.mobility_apply(dp, df, dv)  # still usable after the refused calls
    torch.cuda.synchronize()
    assert np.array_equal(dv.cpu().numpy(), out[sd.STAGE_BULK])
    ctx.set_staging(sd.STAGE_BULK)
    ctx.set_tensor(sd.TENSOR_OSEEN)
    with pytest.raises(sd.SdError):
        ctx.set_staging(sd.STAGE_NAIVE)
    ctx.mobility_apply(dp, df, dv)
    torch.cuda.synchronize()
    assert np.all(np.isfinite(dv.cpu().numpy()))
    ctx.close()


# ---- the pieces the stability experiment runs on -----------------------------

def test_four_sphere_euler_2e5_steps_fp64_matches_oracle(gpu):
    """Euler, dt = 0.01, 2e5 steps (~3.9 cycles) in the one-launch stepper, fp64, against sdo_step."""
    torch, sd = gpu
    pos, force = wl.four_sphere()
    p = wl.to_xyzw(pos, np.float64)
    ctx = sd.Context(4, wl.A, wl.ETA)
    ctx.set_precision(sd.PREC_F64)
    dp = torch.from_numpy(p).cuda()
    for _ in range(4):  # several calls: the state carried between launches is complete
        ctx.step(dp, 0.01, 50000, sd.INT_EULER, gravity=(0.0, 0.0, -1.0))
    torch.cuda.synchronize()
    want, _, _ = orc.step(pos, force, wl.A, wl.ETA, 0.01, 200000, orc.INT_EULER)
    got = dp.cpu().numpy()[:, :3]
    assert np.abs(got - want).max() <= 1e-8
    assert np.all(got[[0, 2], 1] == 0.0) and np.all(got[[1, 3], 0] == 0.0)  # PAPER.md:251 symmetries
    ctx.close()


@pytest.mark.parametrize("n", [4, 300, 5000])
def test_plain_fp32_positions_round_every_step(gpu, n):
    """sd_set_position_compensation(0), reading B5: r <- fl32(r + dt v), nothing carried over.  One
    Euler step from fp32 positions must land on the fp32 number nearest to r + dt v_oracle (1 ulp
    of slack for the fp32 velocity error), and two such steps must differ from the compensated
    run exactly by the low words that were dropped."""
    torch, sd = gpu
    pos = wl.uniform_cube(n, 0.05, wl.SEED_BASE + 80 + n) if n > 4 else wl.four_sphere()[0]
    p = wl.to_xyzw(pos, np.float32)
    F = wl.gravity_forces(n)
    dt = 0.37
    ctx = sd.Context(n, wl.A, wl.ETA)
    ctx.set_position_compensation(False)
    dp = torch.from_numpy(p).cuda()
    ctx.step(dp, dt, 1, sd.INT_EULER, gravity=(0.0, 0.0, -1.0))
    torch.cuda.synchronize()
    got1 = dp.cpu().numpy()[:, :3].copy()
    v = orc.apply(p[:, :3].astype(np.float64), F, wl.A, wl.ETA)
    exact = p[:, :3].astype(np.float64) + dt * v
    ulp = np.spacing(np.abs(exact).astype(np.float32)).astype(np.float64)
    assert np.all(np.abs(got1.astype(np.float64) - exact) <= 0.5 * ulp
                  + 1e-5 * dt * np.linalg.norm(v, axis=1, keepdims=True) + 1e-12)
    # second step: plain mode restarts from the rounded positions, i.e. equals a fresh context
    ctx.step(dp, dt, 1, sd.INT_EULER, gravity=(0.0, 0.0, -1.0))
    ctx2 = sd.Context(n, wl.A, wl.ETA)
    dq = torch.from_numpy(np.concatenate([got1, np.zeros((n, 1), np.float32)], axis=1)).cuda()
    ctx2.step(dq, dt, 1, sd.INT_EULER, gravity=(0.0, 0.0, -1.0))
    torch.cuda.synchronize()
    assert np.array_equal(dp.cpu().numpy(), dq.cpu().numpy())
    ctx.close()
    ctx2.close()


@pytest.mark.parametrize("prec_name,tol", [("PREC_F32_KAHAN", 2e-5), ("PREC_F64", 1e-10)])
@pytest.mark.parametrize("n,integ,steps", [(70, "INT_EULER", 45), (300, "INT_MIDPOINT", 37),
                                           (1200, "INT_EULER", 33)])
def test_small_system_loop_replayed_from_a_cuda_graph(gpu, prec_name, tol, n, integ, steps):
    """64 < N <= 2560 with constant forces and 32 steps or more: sd_step captures 16 steps of the
    one-launch-per-product loop into a CUDA graph and replays it (Euler ping-pongs two position
    buffers: an even number of steps per replay), then runs the odd tail directly."""
    torch, sd = gpu
    prec = getattr(sd, prec_name)
    dtp = np_dtype(sd, prec)
    pos = wl.uniform_cube(n, 0.05, wl.SEED_BASE + 950 + n)
    force = wl.normal_forces(n, wl.SEED_BASE + 951 + n)
    p, f = wl.to_xyzw(pos, dtp), wl.to_xyzw(force, dtp)
    ctx = sd.Context(n, wl.A, wl.ETA)
    ctx.set_precision(prec)
    dp, df = torch.from_numpy(p).cuda(), torch.from_numpy(f).cuda()
    oint = orc.INT_EULER if integ == "INT_EULER" else orc.INT_MIDPOINT
    p64, f64 = p[:, :3].astype(np.float64), f[:, :3].astype(np.float64)
    ctx.step(dp, 0.01, steps, getattr(sd, integ), force=df)
    ctx.step(dp, 0.005, steps, getattr(sd, integ), force=df)      # new dt: new capture
    torch.cuda.synchronize()
    w1, _, _ = orc.step(p64, f64, wl.A, wl.ETA, 0.01, steps, oint)
    w2, _, _ = orc.step(w1, f64, wl.A, wl.ETA, 0.005, steps, oint)
    assert np.abs(dp.cpu().numpy()[:, :3].astype(np.float64) - w2).max() <= tol * wl.cube_side(n, 0.05)
    ctx.close()


def test_four_million_particles_sampled_rows(gpu):
    """Largest size exercised: N = 4,194,304 (1.76e13 pairs, 2048 i-blocks x 32768 j-tiles), fp32-
    Kahan, 512 seeded rows + the first and last row against the oracle.  Checks the 64-bit unit
    arithmetic of the schedule and the partial-sum buffers beyond the L2-resident sizes."""
    torch, sd = gpu
    n = 4 * 1048576
    pos = wl.uniform_cube(n, 0.01, wl.SEED_BASE + 990)
    force = wl.normal_forces(n, wl.SEED_BASE + 991)
    got, p, f = gpu_apply(torch, sd, pos, force, sd.PREC_F32_KAHAN, sd.TENSOR_RPY)
    rows = np.unique(np.concatenate([wl.row_subset(n, 512, wl.SEED_BASE + 992), [0, n - 1]]))
    want = orc.apply_rows(p, f, rows, wl.A, wl.ETA, orc.TENSOR_RPY)
    assert rel_err(got[rows], want) <= TOL_F32
    assert np.all(np.isfinite(got))


def test_side_stream_and_two_contexts_give_the_same_bits(gpu):
    """Every entry point only enqueues on the stream it is given (include/sd_b200.h): the same calls
    on a side stream, interleaved with a second context on the default stream, give bit-identical
    results -- including the CUDA-graph replay of a 40-step run with the lubrication correction."""
    torch, sd = gpu
    n = 3000
    pos = wl.rsa_cube(n, 0.25, wl.SEED_BASE + 310 + n, a=1.3)
    force = wl.normal_forces(n, wl.SEED_BASE + 970)
    p, f = wl.to_xyzw(pos, np.float32), wl.to_xyzw(force, np.float32)

    def run(stream, other=None):
        ctx = sd.Context(n, wl.A, wl.ETA)
        ctx.set_lubrication(True)
        with torch.cuda.stream(stream):
            dp, df = torch.from_numpy(p).cuda(), torch.from_numpy(f).cuda()
            dv = torch.empty_like(dp)
            ctx.mobility_apply(dp, df, dv)
            if other is not None:
                other()
            ctx.step(dp, 0.002, 40, sd.INT_MIDPOINT, force=df)
            ctx.step(dp, 0.002, 5, sd.INT_EULER, gravity=(0.0, 0.0, -1.0))
        stream.synchronize()
        out = (dv.cpu().numpy().copy(), dp.cpu().numpy().copy())
        ctx.close()
        return out

    base = run(torch.cuda.default_stream())
    side = torch.cuda.Stream()
    noise_ctx = sd.Context(5000, wl.A, wl.ETA)
    q = torch.from_numpy(wl.to_xyzw(wl.uniform_cube(5000, 0.05, 3), np.float32)).cuda()
    qv = torch.empty_like(q)

    def noise():  # another context, default stream, while the side stream is busy
        noise_ctx.mobility_apply(q, q.clone(), qv)

    got = run(side, other=noise)
    torch.cuda.synchronize()
    assert np.array_equal(base[0], got[0]) and np.array_equal(base[1], got[1])
    noise_ctx.close()


@pytest.mark.parametrize("prec_name,tol", [("PREC_F32_KAHAN", TOL_F32), ("PREC_F32_PLAIN", 5e-5)])
@pytest.mark.parametrize("tname", ["TENSOR_RPY", "TENSOR_OSEEN"])
@pytest.mark.parametrize("boxed", [False, True])
def test_packed_one_launch_kernel_window(gpu, prec_name, tol, tname, boxed):
    """256 <= N <= 4736 (periodic box: 2304 by default) in the fp32 modes runs small_apply_packed_kernel
    (two particles of a warp as the halves of packed registers, clamped body + per-pair corrections,
    all records in shared memory; CTAs of 128 threads up to 2304, of 512 above).  Dense clouds
    (phi = 0.2: overlaps in most rows, one pair of coincident centres), the ends of the two windows
    and an odd N, all rows; then one step against the oracle."""
    torch, sd = gpu
    prec, tensor = getattr(sd, prec_name), getattr(sd, tname)
    otensor = orc.TENSOR_RPY if tname == "TENSOR_RPY" else orc.TENSOR_OSEEN
    for n in (256, 1001, 2304, 2305, 4736):
        L = wl.cube_side(n, 0.2)
        pos = wl.uniform_cube(n, 0.2, wl.SEED_BASE + 1040 + n)
        pos[n // 2] = pos[3]
        force = wl.normal_forces(n, wl.SEED_BASE + 1041 + n)
        p, f = wl.to_xyzw(pos, np.float32), wl.to_xyzw(force, np.float32)
        ctx = sd.Context(n, wl.A, wl.ETA)
        ctx.set_precision(prec)
        ctx.set_tensor(tensor)
        if boxed:
            ctx.set_box(L)
            if n > 2304:
                ctx.set_dispatch(n, 0)           # beyond the default window of the box: forced
        assert ctx.kernel_name == "small_apply_f32x2"
        dp, df = torch.from_numpy(p).cuda(), torch.from_numpy(f).cuda()
        dv = torch.full_like(dp, float("nan"))
        ctx.mobility_apply(dp, df, dv)
        torch.cuda.synchronize()
        p64, f64 = p[:, :3].astype(np.float64), f[:, :3].astype(np.float64)
        box = float(np.float32(L)) if boxed else 0.0
        want = orc.apply(p64, f64, wl.A, wl.ETA, otensor, box=box, image=orc.IMAGE_F32)
        assert rel_err(dv.cpu().numpy()[:, :3].astype(np.float64), want) <= tol
        # midpoint for Rotne-Prager; Euler for Oseen: its 1/r terms of overlapping pairs amplify the
        # fp32 rounding of the half-step positions (ulp(x) / r_min ~ 2e-5) beyond any fixed bound
        gi, oi = ((sd.INT_MIDPOINT, orc.INT_MIDPOINT) if tname == "TENSOR_RPY"
                  else (sd.INT_EULER, orc.INT_EULER))
        ctx.step(dp, 0.01, 1, gi, force=df)
        torch.cuda.synchronize()
        wp, wv, _ = orc.step(p64, f64, wl.A, wl.ETA, 0.01, 1, oi, otensor, box=box, image=orc.IMAGE_F32)
        # position error <= rounding of the stored word + dt x (velocity error <= tol |v|): the
        # unregularised Oseen tensor gives overlapping spheres velocities of several hundred mu0 F
        vmax = np.linalg.norm(wv, axis=1).max()
        assert np.abs(dp.cpu().numpy()[:, :3] - wp).max() <= 2e-7 * L + 3 * tol * 0.01 * vmax
        ctx.close()
