"""GPU parity of the warp-split one-launch kernel (sd_pairs_f32w.cuh; north_star: "splits j across
warps"; SURVEY 8(a) a1-a6 in one launch) against the CPU oracle, through the C ABI.  `sd_set_jsplit(2)`
forces it at any N; by default it runs for N up to a few
thousand.  Tolerances: north_star's 1e-5 on max_i |v_gpu,i - v_ref,i| / |v_ref,i| (fp32-Kahan), 1e-11 (fp64, `pairs_f64w_kernel`)."""
import numpy as np
import pytest

from oracle import sd_oracle as orc
from paper_1205_6333_b200 import workloads as wl

pytestmark = pytest.mark.gpu

TOL = {"PREC_F32_KAHAN": 1e-5, "PREC_F32_PLAIN": 5e-5, "PREC_F64": 1e-11}


def _np(prec_name):
    return np.float64 if prec_name == "PREC_F64" else np.float32
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


def _device_view(torch, ptr, n, f64=False):
    """Wrap a raw device pointer [n][4] float / double as a torch tensor (no copy)."""
    class _Holder:
        pass
    h = _Holder()
    h.__cuda_array_interface__ = {"shape": (n, 4), "typestr": "<f8" if f64 else "<f4", "data": (int(ptr), False),
                                  "version": 2}
    return torch.as_tensor(h, device="cuda")


def dense_cloud(n, seed):
    """phi = 0.2 with overlaps allowed (~1.6 overlapping neighbours per sphere) and one pair of
    coincident centres: self pairs, overlapping pairs and r = 0 pairs in most chunks."""
    pos = wl.uniform_cube(n, 0.2, seed)
    pos[n // 2] = pos[3]
    return pos


@pytest.mark.parametrize("prec_name", ["PREC_F32_KAHAN", "PREC_F32_PLAIN", "PREC_F64"])
@pytest.mark.parametrize("tname", ["rpy", "oseen"])
@pytest.mark.parametrize("boxed", [False, True])
def test_dense_clouds_all_rows(gpu, prec_name, tname, boxed):
    """Tensor x accumulation x boundary condition on dense clouds, all rows: N = 257 (two i-blocks,
    one of them a single particle; most warps without work), 3000, 5003 and 9999 (ragged tails, pad
    records, several CTAs per i-block: the last-arriver epilogue; warp shares of every length)."""
    torch, sd = gpu
    for n in (257, 3000, 5003, 9999):
        pos = dense_cloud(n, wl.SEED_BASE + 40 + n)
        force = wl.normal_forces(n, wl.SEED_BASE + 41 + n)
        L = 1.01 * wl.cube_side(n, 0.2) if boxed else 0.0
        p, f = wl.to_xyzw(pos, _np(prec_name)), wl.to_xyzw(force, _np(prec_name))
        ctx = sd.Context(n, wl.A, wl.ETA)
        ctx.set_precision(getattr(sd, prec_name))
        ctx.set_tensor(TENSOR[tname][0])
        ctx.set_box(L)
        ctx.set_dispatch(0, 0)
        ctx.set_jsplit(2)
        assert "_w8_" in ctx.kernel_name or "_w4_" in ctx.kernel_name, ctx.kernel_name
        dp, df = torch.from_numpy(p).cuda(), torch.from_numpy(f).cuda()
        out = []
        for _ in range(3):                         # same bits whoever delivers the last partial
            dv = torch.full_like(dp, float("nan"))
            ctx.mobility_apply(dp, df, dv)
            torch.cuda.synchronize()
            out.append(dv.cpu().numpy())
        assert ctx.launch_count == 3               # one launch per product
        assert np.array_equal(out[0], out[1]) and np.array_equal(out[0], out[2])
        assert np.all(out[0][:, 3] == 0.0)
        p64, f64 = p[:, :3].astype(np.float64), f[:, :3].astype(np.float64)
        if tname == "oseen" and boxed and prec_name != "PREC_F64":
            continue  # Eq. (4) at overlapping centres through a face: fp32 displacement error, B6
        if prec_name == "PREC_F64":
            want = orc.apply(p64, f64, wl.A, wl.ETA, TENSOR[tname][1], box=L,
                             image=orc.IMAGE_F64 if boxed else orc.IMAGE_DEFINITION)
        else:
            want = orc.apply(p64, f64, wl.A, wl.ETA, TENSOR[tname][1], box=float(np.float32(L)),
                             image=orc.IMAGE_F32 if boxed else orc.IMAGE_DEFINITION)
        assert rel_err(out[0][:, :3].astype(np.float64), want) <= TOL[prec_name], n
        ctx.close()


@pytest.mark.parametrize("prec_name", ["PREC_F32_KAHAN", "PREC_F64"])
@pytest.mark.parametrize("n", [4096, 70001, 300007])
def test_config5_cloud_sampled_rows(gpu, n, prec_name):
    """The sweep cloud (phi = 0.01, overlaps allowed): default dispatch at N = 4096 is this kernel;
    N = 70001 forced (several i-blocks per CTA, ragged tail), 4096 seeded rows."""
    torch, sd = gpu
    pos, force = wl.sweep(n)
    p, f = wl.to_xyzw(pos, _np(prec_name)), wl.to_xyzw(force, _np(prec_name))
    ctx = sd.Context(n, wl.A, wl.ETA)
    ctx.set_precision(getattr(sd, prec_name))
    ctx.set_jsplit(2)
    assert "_w8_" in ctx.kernel_name or "_w4_" in ctx.kernel_name, ctx.kernel_name
    dp, df = torch.from_numpy(p).cuda(), torch.from_numpy(f).cuda()
    dv = torch.full_like(dp, float("nan"))
    ctx.mobility_apply(dp, df, dv)
    torch.cuda.synchronize()
    rows = wl.row_subset(n, 4096, wl.SEED_BASE + 6)
    rows[-1] = n - 1
    want = orc.apply_rows(p[:, :3].astype(np.float64), f[:, :3].astype(np.float64), rows, wl.A, wl.ETA)
    got = dv.cpu().numpy()
    assert np.all(np.isfinite(got))
    assert rel_err(got[rows, :3].astype(np.float64), want) <= TOL[prec_name]
    ctx.close()


@pytest.mark.parametrize("n,integ,boxed", [(3000, "euler", False), (3000, "midpoint", True),
                                           (9001, "midpoint", False), (9001, "euler", True)])
@pytest.mark.parametrize("forces", ["gravity", "array", "callback"])
@pytest.mark.parametrize("prec_name", ["PREC_F32_KAHAN", "PREC_F64"])
def test_step_through_the_one_launch_kernel(gpu, n, integ, boxed, forces, prec_name):
    """sd_step with the fused integrator update of the epilogue (ping-pong position buffers for
    Euler, odd step count), uniform gravity (written out per particle), a force array and a
    callback; free space and periodic box; against sdo_step."""
    torch, sd = gpu
    pos = wl.rsa_cube(n, 0.1, wl.SEED_BASE + 950 + n)
    L = 1.05 * wl.cube_side(n, 0.1) if boxed else 0.0
    F = wl.gravity_forces(n) if forces == "gravity" else wl.normal_forces(n, wl.SEED_BASE + 951 + n)
    f64m = prec_name == "PREC_F64"
    p, f = wl.to_xyzw(pos, _np(prec_name)), wl.to_xyzw(F, _np(prec_name))
    steps, dt = 3, 0.01
    ctx = sd.Context(n, wl.A, wl.ETA)
    ctx.set_precision(getattr(sd, prec_name))
    ctx.set_box(L)
    ctx.set_jsplit(2)
    assert "_w8_" in ctx.kernel_name or "_w4_" in ctx.kernel_name
    dp, df = torch.from_numpy(p).cuda(), torch.from_numpy(f).cuda()
    gi = sd.INT_EULER if integ == "euler" else sd.INT_MIDPOINT
    oi = orc.INT_EULER if integ == "euler" else orc.INT_MIDPOINT
    if forces == "gravity":
        ctx.step(dp, dt, steps, gi, gravity=(0.0, 0.0, -1.0))
    elif forces == "array":
        ctx.step(dp, dt, steps, gi, force=df)
    else:
        def fill(pos_ptr, force_ptr, nn, user, stream):
            # enqueue on the current torch stream (== the stream sd_step was given)
            _device_view(torch, force_ptr, nn, f64m).copy_(df)
            return 0
        ctx.step(dp, dt, steps, gi, force_fn=fill)
    dv = torch.empty_like(dp)
    ctx.get_velocity(dv)
    torch.cuda.synchronize()
    want, vlast, _ = orc.step(p[:, :3].astype(np.float64), f[:, :3].astype(np.float64), wl.A, wl.ETA, dt,
                              steps, oi, box=L if f64m else float(np.float32(L)),
                              image=(orc.IMAGE_F64 if f64m else orc.IMAGE_F32) if boxed else 0)
    got = dp.cpu().numpy()[:, :3].astype(np.float64)
    scale = float(np.abs(want).max())
    rel, eps = (1e-11, 2.0 ** -52) if f64m else (1e-5, 2.0 ** -23)
    assert np.abs(got - want).max() <= rel * float(np.abs(vlast).max()) * steps * dt + eps * scale
    assert rel_err(dv.cpu().numpy()[:, :3].astype(np.float64), vlast) <= (1e-10 if f64m else 2e-5)
    ctx.close()


def test_jsplit_argument_validation(gpu):
    torch, sd = gpu
    ctx = sd.Context(5000, wl.A, wl.ETA)
    assert "_w8_" in ctx.kernel_name               # default at this N
    ctx.set_jsplit(1)
    assert "_w8_" not in ctx.kernel_name
    for bad in (3, -1):
        with pytest.raises(sd.SdError):
            ctx.set_jsplit(bad)
    ctx.set_precision(sd.PREC_F64)                 # the fp64 counterpart: 4 particles per lane
    ctx.set_jsplit(2)
    assert "f64_w4" in ctx.kernel_name
    ctx.set_jsplit(1)
    assert "f64_i" in ctx.kernel_name
    ctx.close()
