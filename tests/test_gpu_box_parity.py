"""GPU parity of the periodic-box / nearest-image variant (PAPER.md:115
footnote 1) against the CPU oracle, through the C ABI (`sd_set_box`).

Tolerances are those of the free-space path (north_star): 1e-5 (fp32-Kahan), 1e-11 (fp64) on
max_i |v_gpu,i - v_ref,i| / |v_ref,i|.  The nearest-image index is an integer decided by floating
point, so both sides take that decision in the kernel's precision (reading B2): the
oracle runs with IMAGE_F32 (resp. IMAGE_F64) on the same rounded inputs, box side included.
"""
import numpy as np
import pytest

from oracle import sd_oracle as orc
from paper_1205_6333_b200 import workloads as wl

pytestmark = pytest.mark.gpu

TOL = {"PREC_F32_KAHAN": 1e-5, "PREC_F64": 1e-11}
IMAGE = {"PREC_F32_KAHAN": orc.IMAGE_F32, "PREC_F64": orc.IMAGE_F64}
TENSOR = {"rpy": (0, orc.TENSOR_RPY), "oseen": (1, orc.TENSOR_OSEEN)}


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
    assert rel_err(got, want) <= TOL[prec_name]
    if tname == "rpy":  # overlaps through the faces exist and take the r < 2a branch
        w = p - Ls * np.rint(p / Ls)
        face = np.abs(w).max(axis=1) > 0.5 * Ls - 1.0
        assert face.sum() > 100
        far = orc.apply_rows(p, f, np.nonzero(face)[0], wl.A, wl.ETA, orc.TENSOR_RP_FAR, box=Ls,
                             image=IMAGE[prec_name])
        assert rel_err(far, want[face]) > 1e-4


@pytest.mark.parametrize("prec_name", ["PREC_F32_KAHAN", "PREC_F64"])
def test_uniform_131849_eight_per_thread_sampled_rows(gpu, prec_name):
    torch, sd = gpu
    n = 131072 + 777
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
        out = []
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
# Long runs are therefore compared (a) in fp64 on the commensurate box, (b) in fp32 and fp64 in a
# box 2 % larger than the lattice, where no pair comes within 0.3 a of half a box, and (c) in fp32
# on the commensurate box step by step, each step restarted from the GPU's own positions.

@pytest.mark.parametrize("prec_name,tol,scale", [("PREC_F32_KAHAN", 1e-4, 1.02),
                                                 ("PREC_F64", 1e-9, 1.02),
                                                 ("PREC_F64", 1e-9, 1.0)])
@pytest.mark.parametrize("cells,integ,steps,dt", [(2, "midpoint", 1000, 0.01),
                                                  (8, "midpoint", 30, 0.005),
                                                  (10, "euler", 100, 0.001),
                                                  (16, "midpoint", 5, 0.005)])
def test_step_in_periodic_box(gpu, prec_name, tol, scale, cells, integ, steps, dt):
    """N = 32 (one-launch stepper), 2048 (one launch per product), 4000 and 16384 (tiled kernels
    with 2 and 4 particles per thread)."""
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
    perr = np.abs(got - want).max(axis=1)
    if prec_name == "PREC_F64":
        assert perr.max() <= tol
        assert rel_err(dv.cpu().numpy()[:, :3].astype(np.float64), vlast) <= 10 * TOL[prec_name]
    else:
        # fp32 positions differ from the oracle's by ~1e-6 a, so a pair component that crosses half
        # a box during the run (the jittered lattice is not in equilibrium in the larger box) may do
        # so one step apart on the two sides (reading B3); such a flip moves a few particles by
        # O(1e-4 a).  Everybody else obeys the tolerance.
        assert np.mean(perr <= tol) >= 0.995 and perr.max() <= 5e-3
    # the suspension settled (|v| is several mu0 F with ~N^(2/3) neighbours inside L/2)
    assert (got[:, 2] - p[:, 2]).mean() < -steps * dt
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
