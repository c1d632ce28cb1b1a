"""sd_mobility_apply_noalloc (include/sd_b200.h): the product for callers that cannot allocate device
memory.  Its scratch is a static 4-MiB device array inside the library, shared by every call, so the
checks are made on TWO calls in a row (different sizes and tensors: the second call finds the first
one's partial sums, tickets and schedule in the array) against the existing path
(`sd_mobility_apply` of a PREC_F32_KAHAN context) at that path's tolerance, north_star's 1e-5 on
max_i |v_i - v_ref,i| / |v_ref,i|.  Collected last on purpose (file name): the suite runs with
`pytest -x`.  Passes alone in a fresh process (the first call does the per-device set-up) and after
the other GPU tests."""
import numpy as np
import pytest

from paper_1205_6333_b200 import workloads as wl

pytestmark = pytest.mark.gpu

TOL = 1e-5


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


def _inputs(torch, n, seed):
    """phi = 0.2 with overlaps allowed and one pair of coincident centres: far pairs, overlapping
    pairs (RPY branch r < 2a) and an r = 0 pair; N(0,1) forces."""
    pos = wl.uniform_cube(n, 0.2, seed)
    pos[n // 2] = pos[3]
    frc = wl.normal_forces(n, seed + 1)
    return (torch.from_numpy(wl.to_xyzw(pos, np.float32)).cuda(), torch.from_numpy(wl.to_xyzw(frc, np.float32)).cuda())


def _existing_path(torch, sd, tensor, dp, df):
    n = dp.shape[0]
    ctx = sd.Context(n, wl.A, wl.ETA)
    ctx.set_tensor(tensor)
    ctx.set_precision(sd.PREC_F32_KAHAN)
    out = torch.full_like(dp, float("nan"))
    ctx.mobility_apply(dp, df, out)
    torch.cuda.synchronize()
    ctx.close()
    return out.cpu().numpy()[:, :3].astype(np.float64)


# (N, tensor) of the first and of the second call: one i-block shared by all CTAs then 64 i-blocks;
# ragged tails with pad records then a single CTA's worth; the maximum then a small one
@pytest.mark.parametrize("first,second", [((300, "TENSOR_RPY"), (16384, "TENSOR_OSEEN")),
                                          ((5003, "TENSOR_OSEEN"), (4, "TENSOR_RPY")),
                                          ((16384, "TENSOR_RPY"), (1031, "TENSOR_RPY"))])
def test_two_calls_in_a_row_match_the_existing_path(gpu, first, second):
    torch, sd = gpu
    cases = []
    for k, (n, tname) in enumerate((first, second)):
        dp, df = _inputs(torch, n, wl.SEED_BASE + 900 + 7 * n + k)
        cases.append((n, getattr(sd, tname), dp, df, _existing_path(torch, sd, getattr(sd, tname), dp, df)))
    outs = []
    for n, tensor, dp, df, _ in cases:          # back to back on one stream, no synchronisation between them
        out = torch.full_like(dp, float("nan"))
        sd.mobility_apply_noalloc(dp, df, out, wl.A, wl.ETA, tensor)
        outs.append(out)
    torch.cuda.synchronize()
    for (n, tensor, dp, df, want), out in zip(cases, outs):
        got = out.cpu().numpy()
        assert np.all(np.isfinite(got[:, :3]))
        assert rel_err(got[:, :3].astype(np.float64), want) <= TOL, (n, tensor)
    # the same call again gives the same bits: nothing of the previous call leaks into the next one
    n, tensor, dp, df, _ = cases[1]
    again = torch.full_like(dp, float("nan"))
    sd.mobility_apply_noalloc(dp, df, again, wl.A, wl.ETA, tensor)
    torch.cuda.synchronize()
    assert torch.equal(again[:, :3], outs[1][:, :3])


def test_no_device_memory_is_allocated(gpu):
    """Free device memory does not move across calls (after one warm-up call per kernel: loading a
    kernel's code is not an allocation of ours, but the driver may account for it)."""
    torch, sd = gpu
    n = 9999
    dp, df = _inputs(torch, n, wl.SEED_BASE + 950)
    out = torch.empty_like(dp)
    for tensor in (sd.TENSOR_RPY, sd.TENSOR_OSEEN):
        sd.mobility_apply_noalloc(dp, df, out, wl.A, wl.ETA, tensor)
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    for _ in range(3):
        for tensor in (sd.TENSOR_RPY, sd.TENSOR_OSEEN):
            sd.mobility_apply_noalloc(dp, df, out, wl.A, wl.ETA, tensor)
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert abs(free0 - free1) < (1 << 20)


def test_sizes_beyond_the_maximum_are_rejected(gpu):
    torch, sd = gpu
    nmax = sd.noalloc_max_particles()
    assert nmax == 16384
    z = torch.zeros((nmax + 1, 4), device="cuda", dtype=torch.float32)
    with pytest.raises(sd.SdError) as e:
        sd.mobility_apply_noalloc(z, z.clone(), z.clone(), wl.A, wl.ETA)
    assert e.value.status == sd.ERR_UNSUPPORTED
    assert "16384" in str(e.value)
    ok = torch.zeros((8, 4), device="cuda", dtype=torch.float32)
    with pytest.raises(sd.SdError) as e:                       # vel aliases pos
        sd.mobility_apply_noalloc(ok, ok.clone(), ok, wl.A, wl.ETA)
    assert e.value.status == sd.ERR_INVALID_ARG
    with pytest.raises(sd.SdError) as e:
        sd.mobility_apply_noalloc(ok, ok.clone(), ok.clone(), wl.A, -1.0)
    assert e.value.status == sd.ERR_INVALID_ARG
