"""Appendix A of the paper: minimal O(N^2) memory-access
kernels.  Oracle pins run on the CPU; the GPU test compares bit for bit (small-integer data make
every sum exact in fp32)."""
import math

import numpy as np
import pytest

from oracle import sd_oracle as orc

PATTERNS = [orc.ACC_LINEAR, orc.ACC_STRIDED, orc.ACC_UNORDERED]
SCHEMES = [orc.ACC_NAIVE, orc.ACC_SMALL_TILING, orc.ACC_TILING]


def _data(n, elem, seed):
    rng = np.random.Generator(np.random.PCG64(seed))
    shape = (n,) if elem == 1 else (n, 4)
    return rng.integers(0, 4, size=shape).astype(np.float32)


@pytest.mark.parametrize("n", [1000, 1310, 4096])
@pytest.mark.parametrize("elem", [1, 4])
def test_oracle_access_sums_closed_forms(n, elem):
    """k -> k p mod N is a permutation of 0..N-1 iff gcd(p, N) = 1, and so is k -> (k p + j M) mod N
    for every j: then the naive kernel makes every thread visit every element once, and thread j
    stores total + its own element, for all three patterns.  N = 1310 = 10 * 131 breaks it: the
    strided map then visits only every 131st element, 131 times each."""
    d = _data(n, elem, 9100 + n)
    val = d.sum(axis=1) if elem == 4 else d
    total = float(val.astype(np.float64).sum())
    for pattern in PATTERNS:
        got = orc.access_sums(d, pattern, orc.ACC_NAIVE)
        if pattern == orc.ACC_LINEAR or math.gcd(131, n) == 1:
            np.testing.assert_array_equal(got, total + val)
        elif pattern == orc.ACC_STRIDED:
            visited = val[(np.arange(n) * 131) % n].astype(np.float64).sum()
            np.testing.assert_array_equal(got, visited + val)
            assert visited != total
    # linear + any tiling: the tiles partition the array, so nothing changes
    for scheme in (orc.ACC_SMALL_TILING, orc.ACC_TILING, orc.ACC_BULK):
        np.testing.assert_array_equal(orc.access_sums(d, orc.ACC_LINEAR, scheme), total + val)
    # strided + tiling: the copying thread's id does not enter the map: same as naive
    np.testing.assert_array_equal(orc.access_sums(d, orc.ACC_STRIDED, orc.ACC_TILING),
                                  orc.access_sums(d, orc.ACC_STRIDED, orc.ACC_NAIVE))
    # unordered + tiling: all threads of a block store the same tile total (plus their own element)
    u = orc.access_sums(d, orc.ACC_UNORDERED, orc.ACC_SMALL_TILING) - val
    for b0 in range(0, n, 128):
        assert np.all(u[b0:b0 + 128] == u[b0])
    with pytest.raises(ValueError):
        orc.access_sums(d, orc.ACC_STRIDED, orc.ACC_BULK)


def test_oracle_unordered_tile_by_hand():
    """N = 40 (one block), small-tiling: tile m = 0 holds elements (131 n + 32 n) mod 40 for n < 32,
    tile m = 32 holds (131 (32 + n) + 32 n) mod 40 for n < 8; written out with python ints."""
    n = 40
    d = np.arange(n, dtype=np.float32) % 5
    idx = [(131 * k + 32 * k) % n for k in range(32)] + [(131 * (32 + k) + 32 * k) % n for k in range(8)]
    want = d.astype(np.float64) + float(sum(d[i] for i in idx))
    np.testing.assert_array_equal(orc.access_sums(d, orc.ACC_UNORDERED, orc.ACC_SMALL_TILING), want)


@pytest.mark.gpu
@pytest.mark.parametrize("elem", [1, 4])
@pytest.mark.parametrize("n", [1000, 4100, 20000])
def test_gpu_access_kernels_bit_exact(elem, n):
    import torch
    from paper_1205_6333_b200 import sd
    sd.load_library()
    torch.cuda.set_device(0)
    d = _data(n, elem, 9200 + n)
    dd = torch.from_numpy(d).cuda()
    for pattern in PATTERNS:
        for scheme in SCHEMES + [orc.ACC_BULK]:
            out = torch.full((n,), float("nan"), device="cuda")
            if scheme == orc.ACC_BULK and pattern != orc.ACC_LINEAR:
                with pytest.raises(sd.SdError):
                    sd.access_bench(dd, out, pattern, scheme, reps=1)
                continue
            ms = sd.access_bench(dd, out, pattern, scheme, reps=2)
            assert ms > 0.0
            want = orc.access_sums(d, pattern, scheme)
            assert want.max() < 2 ** 24                       # every partial sum is exact in fp32
            np.testing.assert_array_equal(out.cpu().numpy().astype(np.float64), want)

