"""Host logic of libsd_b200 without a GPU: the static work schedule of the tiled kernels
(sd_schedule_plan is the very code sd_create runs; DESIGN.md section 5.2 "Schedule" and "SM balance")."""
import numpy as np
import pytest

from paper_1205_6333_b200 import sd

CASES = [  # N, particles per block, tile, max CTAs, SMs
    (2561, 512, 128, 444, 148), (4000, 512, 128, 444, 148), (6000, 512, 32, 444, 148),
    (6000, 512, 128, 444, 148), (12288, 512, 128, 444, 148), (20000, 1024, 128, 296, 148),
    (65536, 2048, 128, 148, 148), (1048576, 2048, 128, 148, 148), (4194304, 2048, 128, 148, 148),
    (131849, 1024, 64, 148, 148), (3000, 256, 64, 444, 148), (777, 512, 128, 444, 148),
    (1, 512, 128, 444, 148), (100000, 2048, 128, 7, 3),
]


@pytest.mark.parametrize("n,ib,tj,max_ctas,nsm", CASES)
def test_schedule_covers_every_unit_once_and_names_the_right_slots(n, ib, tj, max_ctas, nsm):
    s = sd.schedule_plan(n, ib, tj, max_ctas, nsm)
    B, T, G = s["B"], s["T"], s["G"]
    assert B == -(-n // ib) and T == -(-n // tj) and G == min(B * T, max_ctas)
    u0 = np.array(s["cta_u0"], dtype=np.int64)
    assert u0[0] == 0 and u0[-1] == B * T and np.all(np.diff(u0) >= 1)
    sizes = np.diff(u0)
    assert sizes.max() - sizes.min() <= 1                      # equal pieces +-1 unit
    # block b's slots are exactly the pieces that intersect its unit range [b T, (b+1) T)
    first, nslots = np.array(s["blk_first"]), np.array(s["blk_nslots"])
    for b in (range(B) if B <= 64 else list(range(8)) + list(range(B - 8, B)) + [B // 2]):
        lo, hi = b * T, (b + 1) * T
        touching = [g for g in range(G) if u0[g] < hi and u0[g + 1] > lo]
        assert touching == list(range(first[b], first[b] + nslots[b]))
    assert s["max_slots"] == nslots.max()


@pytest.mark.parametrize("n,ib,tj,max_ctas,nsm", CASES)
def test_ctas_that_share_an_sm_own_consecutive_pieces_and_sms_are_balanced(n, ib, tj, max_ctas, nsm):
    s = sd.schedule_plan(n, ib, tj, max_ctas, nsm)
    G = s["G"]
    piece = np.array(s["cta_piece"])
    assert sorted(piece.tolist()) == list(range(G))            # a permutation of the pieces
    sizes = np.diff(np.array(s["cta_u0"], dtype=np.int64))
    loads = []
    for sm in range(min(nsm, G)):
        mine = piece[sm::nsm]                                  # CTAs sm, sm + nsm, ... share an SM
        assert np.all(np.diff(mine) == 1)                      # consecutive pieces
        loads.append(int(sizes[mine].sum()))
    ctas = [len(piece[sm::nsm]) for sm in range(min(nsm, G))]
    # SMs with the same number of CTAs carry the same number of units +-1
    for k in set(ctas):
        sel = [l for l, c in zip(loads, ctas) if c == k]
        assert max(sel) - min(sel) <= 1


def test_plain_map_would_resonate_at_6000():
    """Why the permutation exists (profiles/r01e_sweep.md history): N = 6000, 512-particle blocks,
    128-record tiles, 444 CTAs on 148 SMs: with piece = blockIdx some SMs would carry 6 units and
    others 3; with the balanced map every SM carries 3 or 4."""
    s = sd.schedule_plan(6000, 512, 128, 444, 148)
    sizes = np.diff(np.array(s["cta_u0"], dtype=np.int64))
    plain = [int(sizes[sm::148].sum()) for sm in range(148)]
    piece = np.array(s["cta_piece"])
    balanced = [int(sizes[piece[sm::148]].sum()) for sm in range(148)]
    assert max(plain) == 6 and min(plain) == 3
    assert max(balanced) == 4 and min(balanced) == 3


def test_schedule_plan_rejects_bad_arguments():
    for bad in ((0, 512, 128, 444, 148), (10, 0, 128, 444, 148), (10, 512, 0, 444, 148),
                (10, 512, 128, 0, 148), (10, 512, 128, 444, 0)):
        with pytest.raises(sd.SdError):
            sd.schedule_plan(*bad)
