"""CPU checks of the test-side geometry guards (tests/guards.py) and of the input generators the
plain-definition parity tests rely on: brute force on small clouds."""
import numpy as np

from paper_1205_6333_b200 import workloads as wl
import guards


def _brute_half_box(pos, L):
    d = pos[:, None, :] - pos[None, :, :]
    w = np.abs(d - L * np.rint(d / L))
    iu = np.triu_indices(pos.shape[0], 1)
    return 0.5 * L - w[iu], iu


def test_half_box_margin_and_ties_against_brute_force():
    rng = np.random.Generator(np.random.PCG64(wl.SEED_BASE + 700))
    for n, L in ((2, 5.0), (37, 11.0), (400, 23.5)):
        pos = rng.uniform(-1.7 * L, 1.7 * L, size=(n, 3))        # several boxes wide
        m, (ii, jj) = _brute_half_box(pos, L)
        assert abs(guards.half_box_margin(pos, L) - m.min()) < 1e-12
        guard = 5e-2
        hit = np.nonzero((m < guard).any(axis=1))[0]
        want = np.unique(np.stack([ii[hit], jj[hit]], axis=1), axis=0)
        got = guards.half_box_ties(pos, L, guard)
        assert np.array_equal(got, want)
        keep = guards.drop_one_of_each(n, got)
        if keep.sum() >= 2:
            assert guards.half_box_margin(pos[keep], L) >= guard


def test_cutoff_margin_and_shell_pairs_against_brute_force():
    rng = np.random.Generator(np.random.PCG64(wl.SEED_BASE + 701))
    pos = rng.uniform(-6.0, 6.0, size=(300, 3))
    for L in (0.0, 12.0):
        d = pos[:, None, :] - pos[None, :, :]
        if L > 0.0:
            d = d - L * np.rint(d / L)
        r = np.linalg.norm(d, axis=2)
        iu = np.triu_indices(300, 1)
        assert abs(guards.cutoff_margin(pos, 3.0, L) - np.abs(r[iu] - 3.0).min()) < 1e-12
        sel = (r[iu] >= 2.9) & (r[iu] <= 3.1)
        want = np.unique(np.stack([iu[0][sel], iu[1][sel]], axis=1), axis=0)
        got = np.unique(guards.pairs_in_shell(pos, 2.9, 3.1, L), axis=0)
        assert np.array_equal(got, want)


def test_step_spread():
    s = np.zeros((3, 4, 3))
    s[1, :, 2] = [0.0, 0.1, 0.2, 0.3]
    s[2] = s[1] + 1.0                                           # rigid shift: no relative motion
    assert abs(guards.step_spread(s) - 0.3) < 1e-15


def test_sc_lattice_with_odd_edge_keeps_half_a_spacing_from_half_a_box():
    for edge in (3, 9):
        pos = wl.sc_lattice(edge, 0.1, jitter_seed=wl.SEED_BASE + 702)
        L = wl.sc_box(edge, 0.1)
        assert pos.shape == (edge ** 3, 3)
        assert abs(edge ** 3 / L ** 3 - 0.1) < 1e-12
        sp = L / edge
        assert guards.half_box_margin(pos, L) >= 0.5 * sp - 2.1e-2   # two jitters of 1e-2
    # an even edge has pairs at half a box
    assert guards.half_box_margin(wl.sc_lattice(4, 0.1, jitter_seed=1), wl.sc_box(4, 0.1)) < 2.1e-2


def test_rsa_shell_leaves_no_pair_in_the_shell_and_keeps_the_plain_stream():
    n = 200
    plain = wl.rsa_cube(n, 0.25, wl.SEED_BASE + 703, a=1.3)
    assert np.array_equal(plain, wl.rsa_cube(n, 0.25, wl.SEED_BASE + 703, a=1.3, shell=None))
    pos = wl.rsa_cube(n, 0.25, wl.SEED_BASE + 703, a=1.3, shell=(2.8, 3.2))
    assert guards.pairs_in_shell(pos, 2.8, 3.2).shape[0] == 0
    assert guards.pairs_in_shell(pos, 0.0, 2.6 - 1e-12).shape[0] == 0
    assert guards.pairs_in_shell(pos, 2.6, 2.8).shape[0] > n // 10      # lubrication pairs remain
    assert guards.cutoff_margin(pos, 3.0) >= 0.2 - 1e-12
