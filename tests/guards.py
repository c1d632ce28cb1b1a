"""Test-side geometry checks (plain numpy / scipy, none of the method's arithmetic).

Two decisions of the path are taken by floating point and are discontinuous: the nearest-image
index at |d_c| = L/2 (PAPER.md:115 footnote 1; readings B2, B3) and the lubrication
cut-off at r = 3a (reading C3).  A comparison against the oracle's PLAIN
definition (C99 `remainder`, `r < 3a` in double) is only meaningful on inputs where no pair sits
within rounding of such a discontinuity; the functions below measure how far a cloud (or every
state of an oracle trajectory) stays away from them, and the parity tests assert that margin
before they hold every particle to the strict tolerance.
"""
from __future__ import annotations

import numpy as np
from scipy.spatial import cKDTree


def _circ(a, b, L):
    d = np.abs(a - b)
    return np.minimum(d, L - d)


def half_box_margin(pos: np.ndarray, L: float) -> float:
    """min over pairs (i != j) and components c of  L/2 - |nearest-image d_c| : the distance of the
    closest pair component to the discontinuity of the nearest-image rule.  O(N log N)."""
    pos = np.asarray(pos, dtype=np.float64)
    n = pos.shape[0]
    if n < 2:
        return float("inf")
    best = np.inf
    for c in range(3):
        u = np.mod(pos[:, c], L)
        s = np.sort(u)
        t = np.mod(u + 0.5 * L, L)           # where a partner at exactly half a box would sit
        k = np.searchsorted(s, t)
        lo, hi = s[(k - 1) % n], s[k % n]
        best = min(best, float(np.minimum(_circ(t, lo, L), _circ(t, hi, L)).min()))
    return best


def half_box_ties(pos: np.ndarray, L: float, guard: float) -> np.ndarray:
    """Pairs (i, j), i < j, with a component within `guard` of half a box: array [K, 2]."""
    pos = np.asarray(pos, dtype=np.float64)
    out = []
    for c in range(3):
        u = np.mod(pos[:, c], L)
        order = np.argsort(u, kind="stable")
        s = u[order]
        ext = np.concatenate([s - L, s, s + L])
        eo = np.concatenate([order, order, order])
        t = np.mod(u + 0.5 * L, L)
        k0 = np.searchsorted(ext, t - guard, side="left")
        k1 = np.searchsorted(ext, t + guard, side="right")
        for i in np.nonzero(k1 > k0)[0]:
            for j in eo[k0[i]:k1[i]]:
                if i != j:
                    out.append((min(i, int(j)), max(i, int(j))))
    if not out:
        return np.empty((0, 2), dtype=np.int64)
    return np.unique(np.asarray(out, dtype=np.int64), axis=0)


def pairs_in_shell(pos: np.ndarray, r_lo: float, r_hi: float, L: float = 0.0) -> np.ndarray:
    """Pairs (i, j), i < j, whose centre distance (nearest image when L > 0) lies in [r_lo, r_hi]."""
    pos = np.asarray(pos, dtype=np.float64)
    if L > 0.0:
        w = np.mod(pos, L)
        w[w >= L] = 0.0
        tree = cKDTree(w, boxsize=L)
        pr = tree.query_pairs(r_hi, output_type="ndarray")
        d = w[pr[:, 0]] - w[pr[:, 1]]
        d -= L * np.rint(d / L)
    else:
        tree = cKDTree(pos)
        pr = tree.query_pairs(r_hi, output_type="ndarray")
        d = pos[pr[:, 0]] - pos[pr[:, 1]]
    r = np.linalg.norm(d, axis=1)
    pr = pr[r >= r_lo]
    return np.sort(pr, axis=1)


def cutoff_margin(pos: np.ndarray, rc: float, L: float = 0.0, look: float = 1.0) -> float:
    """min over pairs of |r_ij - rc| (capped at `look`)."""
    pos = np.asarray(pos, dtype=np.float64)
    pr = pairs_in_shell(pos, max(rc - look, 0.0), rc + look, L)
    if pr.shape[0] == 0:
        return look
    d = pos[pr[:, 0]] - pos[pr[:, 1]]
    if L > 0.0:
        d -= L * np.rint(d / L)
    return float(min(look, np.abs(np.linalg.norm(d, axis=1) - rc).min()))


def drop_one_of_each(n: int, pairs: np.ndarray) -> np.ndarray:
    """Boolean keep-mask over n particles that removes one member (the higher index, unless the
    other is already gone) of every listed pair."""
    keep = np.ones(n, dtype=bool)
    for i, j in pairs:
        if keep[i] and keep[j]:
            keep[j] = False
    return keep


def step_spread(states: np.ndarray) -> float:
    """Upper bound on the relative displacement of any pair component during one step: the largest
    spread (max - min over the particles) of the per-step displacement, over steps and components.
    states: [K + 1, N, 3] positions at the step boundaries."""
    d = np.diff(np.asarray(states, dtype=np.float64), axis=0)
    return float((d.max(axis=1) - d.min(axis=1)).max()) if d.shape[0] else 0.0
