"""Pins of the parts of the oracle's S5 that closed forms do not reach: the pick-up window / metric / tie-break and the Phase B / C
control flow (S5; table T: n_sigma, w_max, max_gap, edge_margin; readings A5, A13, A33).

Every case is hand-built: clusters are placed at known offsets from a closed-form track, and the expected outcome follows from the
definition by arithmetic a reader can redo (no oracle value is stored).  Each test names the one-line mutations of
oracle/tpc_oracle.cpp it was checked to fail under.  Nothing here touches the CUDA path.
"""
import math

import numpy as np
import pytest

from oracle.oracle import Oracle
from tests import helpers as H

R = 152
X = H.row_x()                       # float64, rounded to fp32 by the oracle
ZMAX, VD = 250.0, 2.0               # vdrift = 2: z = 250 - 2 t is exact in fp32 for the z used here
SY, SZ = 0.1, 0.15
YEDGE = X * math.tan(math.pi / 18)


def _oracle(rows, bz=0.5, double=False, **params):
    """rows: {row: [(y, z), ...]} of ONE sector -> oracle with these clusters loaded (caller's order = list order)."""
    off = np.zeros(R + 1, np.int64)
    ys, ts = [], []
    for r in range(R):
        cl = rows.get(r, [])
        off[r + 1] = off[r] + len(cl)
        ys += [c[0] for c in cl]
        ts += [(ZMAX - c[1]) / VD for c in cl]
    o = Oracle(n_sectors=1, n_rows=R, row_x=X.astype(np.float32), sector_dphi=2 * math.pi / 18, z_max=ZMAX, t_frame=0.0,
               sigma_y=SY, sigma_z=SZ, bz=bz, vdrift=VD, double=double, **params)
    o.load(off, np.array(ys, np.float32), np.array(ts, np.float32))
    o.off = off
    return o


def _tri_diag(d):
    Cm = np.diag(np.array(d, dtype=np.float64))
    return np.array([Cm[a, b] for a in range(5) for b in range(a + 1)])


def _picked_original(o, row, pos):
    return -1 if pos < 0 else int(o.get("perm")[o.off[row] + pos])


# ------------------------------------------------------------------------------------------------ pick-up
# state at y = 0, z_rel = 0 with z_ref = 100: a cluster (dy, dz) sits at (dy, 100 + dz)
def _pick(cands, c00, c11, row=50, brute=False):
    o = _oracle({row: [(dy, 100.0 + dz) for dy, dz in cands]}).run("s1")
    pos = o.pickup([0.0, 0.0, 0.0, 0.0, 0.0], _tri_diag([c00, c11, 1.0, 1.0, 1.0]), 0, row, zref=100.0, brute=brute)
    return _picked_original(o, row, pos)


def test_pickup_window_is_n_sigma_times_sqrt_of_C_plus_sigma2():
    """w_y = 4 sqrt(C00 + sigma_y^2) = 4 sqrt(0.03 + 0.01) = 0.8; w_z = 4 sqrt(0.0175 + 0.0225) = 0.8.
    Fails under: sqrt(C) instead of sqrt(C + sigma^2) (0.693 / 0.529: the 0.79 candidates drop out); n_sigma = 3; sigma_y and
    sigma_z swapped (w_y = 0.917 admits 0.81)."""
    c00, c11 = 0.03, 0.0175
    assert _pick([(0.79, 0.0)], c00, c11) == 0
    assert _pick([(0.81, 0.0)], c00, c11) == -1
    assert _pick([(-0.79, 0.0)], c00, c11) == 0
    assert _pick([(-0.81, 0.0)], c00, c11) == -1
    assert _pick([(0.0, 0.79)], c00, c11) == 0
    assert _pick([(0.0, 0.81)], c00, c11) == -1
    assert _pick([(0.0, -0.79)], c00, c11) == 0
    assert _pick([(0.0, -0.81)], c00, c11) == -1
    # the two windows are independent intervals (a box, not an ellipse): the corner is inside
    assert _pick([(0.75, 0.75)], c00, c11) == 0


def test_pickup_window_is_capped_at_w_max():
    """C = 1: 4 sqrt(1.01) = 4.02 > w_max = 3.  Fails under: no cap; cap applied to one coordinate only."""
    assert _pick([(2.9, 0.0)], 1.0, 1.0) == 0
    assert _pick([(3.1, 0.0)], 1.0, 1.0) == -1
    assert _pick([(0.0, -2.9)], 1.0, 1.0) == 0
    assert _pick([(0.0, -3.1)], 1.0, 1.0) == -1


def test_pickup_metric_is_plain_squared_distance():
    """Candidates (0.5, 0) and (0, 0.6) with window half-widths 0.8 (y) and 2.0 (z): plain distance picks the first
    (0.25 < 0.36), a distance normalised by the window / by sqrt(C + sigma^2) picks the second ((0.5/0.2)^2 > (0.6/0.5)^2).
    Fails under: normalised metric; |dy| + |dz| would also pass -> second pair (0.5, 0.5) vs (0.0, 0.75): L1 1.0 vs 0.75 picks
    the second, L2 0.5 vs 0.5625 the first."""
    c00, c11 = 0.03, 0.25 - 0.0225
    assert _pick([(0.5, 0.0), (0.0, 0.6)], c00, c11) == 0
    assert _pick([(0.0, 0.6), (0.5, 0.0)], c00, c11) == 1
    assert _pick([(0.5, 0.5), (0.0, 0.75)], c00, c11) == 0


def test_pickup_tie_goes_to_the_lower_original_index_not_to_the_sorted_order():
    """(+1.2, 0) and (-1.2, 0) are exactly equidistant (window 4 sqrt(0.15 + 0.01) = 1.6).  With 1.6 cm bins (grid_scale) the
    cluster at negative y comes FIRST in the sorted (bin) order; it is given the HIGHER original index, and the pick must be
    original index 0.  Fails under: first-found-wins; tie-break on the sorted position; `<=` in the distance comparison."""
    for brute in (False, True):
        o = _oracle({50: [(1.2, 100.0), (-1.2, 100.0)]}, grid_scale=0.02).run("s1")
        assert list(o.get("perm")) == [1, 0]               # sorted order is the reverse of the caller's order
        pos = o.pickup([0.0, 0.0, 0.0, 0.0, 0.0], _tri_diag([0.15, 0.0175, 1.0, 1.0, 1.0]), 0, 50, zref=100.0, brute=brute)
        assert pos == 1 and _picked_original(o, 50, pos) == 0
        o = _oracle({50: [(-1.2, 100.0), (1.2, 100.0)]}, grid_scale=0.02).run("s1")
        pos = o.pickup([0.0, 0.0, 0.0, 0.0, 0.0], _tri_diag([0.15, 0.0175, 1.0, 1.0, 1.0]), 0, 50, zref=100.0, brute=brute)
        assert pos == 0 and _picked_original(o, 50, pos) == 0


def test_pickup_ignores_candidates_of_the_visited_bins_outside_the_window():
    """One unit with one cluster: the grid has a single 64 cm bin, so the candidate at 0.85 cm is visited and must be rejected by
    the window test itself (0.8); with a closer one present the closer one wins regardless of the order."""
    assert _pick([(0.85, 0.0)], 0.03, 0.0175) == -1
    assert _pick([(0.85, 0.0), (0.0, 0.5), (0.1, 0.85)], 0.03, 0.0175) == 1
    assert _pick([(0.85, 0.0), (0.0, 0.5), (0.1, 0.85)], 0.03, 0.0175, brute=True) == 1


def test_pickup_uses_z_relative_to_zref():
    """The state carries z - z_ref (reading N4): the same cluster is picked with z_ref = 100 and the state at z_rel = 0 as with
    z_ref = 60 and the state at z_rel = 40."""
    o = _oracle({50: [(0.2, 100.3), (0.2, 60.3)]}).run("s1")
    cov = _tri_diag([0.03, 0.0175, 1, 1, 1])
    a = o.pickup([0.0, 0.0, 0, 0, 0], cov, 0, 50, zref=100.0)
    b = o.pickup([0.0, 40.0, 0, 0, 0], cov, 0, 50, zref=60.0)
    assert _picked_original(o, 50, a) == 0 and _picked_original(o, 50, b) == 0


# ------------------------------------------------------------------------------------------------ Phase B / C control flow
def _track_rows(pt=3.0, charge=1, phi=0.03, tanl=0.4, bz=0.5, rows=range(R), y_shift=0.0):
    """Noise-free clusters of one primary on the given rows (closed-form helix from the origin, tests/helpers.py)."""
    out = {}
    for r in rows:
        st = H.helix_truth_at(X[r], pt, charge, phi, tanl, bz)
        out[r] = [(float(st[0]) + y_shift, float(st[1]))]
    return out


def _tracklet_rows(o):
    tl = o.tracklets()
    return [(int(tl["first"][i]), int(tl["last"][i]), int(tl["n"][i]), np.nonzero(tl["rowhit"][i] >= 0)[0]) for i in range(len(tl["n"]))]


def test_phase_b_bridges_max_gap_rows_and_stops_at_max_gap_plus_one():
    """A noise-free primary with rows 101..104 removed (4 = max_gap): every tracklet collects the whole track, 148 clusters on
    rows 0..151.  With rows 101..105 removed (5): the lower seeds stop at row 100, the upper seeds stop at row 106.
    Fails under: `gap >= max_gap` in Phase B or in Phase C; gap not reset after a pick-up (a second 4-row gap at 40..43)."""
    full = _track_rows()
    four = {r: c for r, c in full.items() if not (101 <= r <= 104) and not (40 <= r <= 43)}
    o = _oracle(four).run("s6")
    tls = _tracklet_rows(o)
    assert len(tls) >= 3                                    # chains: rows 1..38, 45..99, 106..150
    for first, last, n, rows in tls:
        assert (first, last, n) == (0, 151, 144), (first, last, n)
        assert set(rows) == set(four)
    assert len(o.tracks()["sector"]) == 1 and o.tracks()["cl_begin"][1] == 144

    five = {r: c for r, c in full.items() if not (101 <= r <= 105)}
    o = _oracle(five).run("s6")
    tls = _tracklet_rows(o)
    assert sorted({(f, l, n) for f, l, n, _ in tls}) == [(0, 100, 101), (106, 151, 46)]
    assert len(o.tracks()["sector"]) == 2


def test_max_gap_is_the_parameter_that_decides_it():
    full = _track_rows()
    five = {r: c for r, c in full.items() if not (101 <= r <= 105)}
    o = _oracle(five, max_gap=5).run("s6")
    assert {(f, l, n) for f, l, n, _ in _tracklet_rows(o)} == {(0, 151, 147)}


def _line_rows(y_at, rows, z=30.0):
    return {r: [(float(y_at(X[r])), z * X[r] / X[0])] for r in rows}


def test_phase_b_stops_at_the_sector_edge_plus_margin():
    """Bz = 0, a straight line y = 0.32 (x - 85) + 4: it crosses yedge(x) + 1 = 0.17633 x + 1 between two rows.  All rows up to
    `cut` carry a cluster (the seeds); above, only every second row does (no pair, hence no link, no seed and no ungated Phase A
    there: the clusters can only be collected by the outward pass), up to four rows BEYOND the edge (they would belong to the
    neighbour sector).  The outward pass must stop at the last populated row with |y| <= yedge + edge_margin.
    Fails under: margin dropped (stops earlier: second half of the test); no edge test (collects the rows beyond);
    the edge test applied after the pick-up instead of before it."""
    y_at = lambda x: 0.32 * (x - 85.0) + 4.0
    inside = [r for r in range(R) if abs(y_at(X[r])) <= YEDGE[r] + 1.0]
    r_last = max(inside)
    assert 20 < r_last < 140 and inside == list(range(r_last + 1))
    assert abs(y_at(X[r_last + 1])) - (YEDGE[r_last + 1] + 1.0) > 0.02 and YEDGE[r_last] + 1.0 - abs(y_at(X[r_last])) > 0.02   # not marginal
    r_last0 = max(r for r in range(R) if abs(y_at(X[r])) <= YEDGE[r])
    assert r_last0 <= r_last - 3
    cut = r_last0 - 12
    populated = [r for r in range(r_last + 5) if r <= cut or (r - cut) % 2 == 0]
    assert any(r > r_last for r in populated)
    rows = _line_rows(y_at, populated)
    want = max(r for r in populated if r <= r_last)
    o = _oracle(rows, bz=0.0).run("s6")
    tls = _tracklet_rows(o)
    assert len(tls) >= 1
    for first, last, n, hit_rows in tls:
        assert last == want and first == 0 and n == len([r for r in populated if r <= want]), (first, last, n, want)
    want0 = max(r for r in populated if r <= r_last0)
    assert want0 < want                                     # the margin matters
    o2 = _oracle(rows, bz=0.0, edge_margin=0.0).run("s6")
    assert {l for _, l, _, _ in _tracklet_rows(o2)} == {want0}


def test_phase_c_stops_at_the_sector_edge_below_the_first_assigned_row():
    """The mirror case: a line that ENTERS the sector from the side, y = -0.32 (x - 246) - 2 -> inside only above some row.
    All rows from `cut` up carry a cluster (the seeds); below, only every second row does (no links there), down to five rows
    OUTSIDE yedge + margin.  The inward pass collects the alternate rows inside and must stop at the first row outside.
    Fails under: `continue` instead of `break` below first_assigned (collects the rows outside); margin dropped."""
    y_at = lambda x: -0.32 * (x - 246.0) - 2.0
    inside = [r for r in range(R) if abs(y_at(X[r])) <= YEDGE[r] + 1.0]
    r_first = min(inside)
    assert 10 < r_first < 130 and inside == list(range(r_first, R))
    assert abs(y_at(X[r_first - 1])) - (YEDGE[r_first - 1] + 1.0) > 0.02 and YEDGE[r_first] + 1.0 - abs(y_at(X[r_first])) > 0.02
    r_first0 = min(r for r in range(R) if abs(y_at(X[r])) <= YEDGE[r])
    cut = r_first0 + 12
    populated = [r for r in range(r_first - 5, R) if r >= cut or (cut - r) % 2 == 0]
    assert any(r < r_first for r in populated)
    o = _oracle(_line_rows(y_at, populated), bz=0.0).run("s6")
    want = min(r for r in populated if r >= r_first)
    tls = _tracklet_rows(o)
    assert len(tls) >= 1
    for first, last, n, hit_rows in tls:
        assert first == want and last == R - 1 and n == len([r for r in populated if r >= want]), (first, last, n, want)
    want0 = min(r for r in populated if r >= r_first0)
    assert want0 > want
    o2 = _oracle(_line_rows(y_at, populated), bz=0.0, edge_margin=0.0).run("s6")
    assert {f for f, _, _, _ in _tracklet_rows(o2)} == {want0}


def test_a_track_that_leaves_and_re_enters_the_sector_is_two_tracklets():
    """A 0.967 GeV/c secondary (radius 645 cm) hugging the sector edge: inside yedge + margin on the low rows, OUTSIDE on the middle
    rows, inside again on the high rows (a circle can cross the edge line twice; a primary or a straight line cannot).  Clusters
    exist on all three parts (alternate rows only on and next to the outside part, so no links there).  By the definition the
    inward pass of the upper seeds BREAKS at the first outside row below first_assigned, and the outward pass of the lower seeds
    stops there as well: two families of tracklets, none spanning the outside part.
    Fails under: `continue` instead of `break` in Phase C below first_assigned (the upper tracklets jump the outside rows and
    collect the lower part: first = 0)."""
    st_at = lambda r: H.helix_truth_at(X[r], 0.967, 1, math.atan(0.301), 0.3, 0.5, vx=85.0, vy=13.0, vz=20.0)
    yy = np.array([st_at(r)[0] for r in range(R)])
    out = np.abs(yy) > YEDGE + 1.0
    ra, rb = int(np.nonzero(out)[0].min()) - 1, int(np.nonzero(out)[0].max()) + 1
    assert 20 < ra < rb - 10 < rb < 130 and out[ra + 1:rb].all() and not out[:ra + 1].any() and not out[rb:].any()
    for r in (ra, ra + 1, rb - 1, rb):
        assert abs(abs(yy[r]) - (YEDGE[r] + 1.0)) > 0.01     # not marginal
    populated = [r for r in range(R) if r <= ra - 8 or r >= rb + 8 or (r - ra) % 2 == 0]
    rows = {r: [(float(yy[r]), float(st_at(r)[1]))] for r in populated}
    o = _oracle(rows).run("s6")
    lo_last = max(r for r in populated if r <= ra)
    hi_first = min(r for r in populated if r >= rb)
    fams = {(f, l) for f, l, _, _ in _tracklet_rows(o)}
    assert fams == {(0, lo_last), (hi_first, R - 1)}, (fams, ra, rb)
    for f, l, n, hit_rows in _tracklet_rows(o):
        assert not out[hit_rows].any()                       # no cluster outside yedge + margin is collected


def test_phase_c_picks_up_what_phase_b_skipped_and_counts_it():
    """Row 150 holds no true cluster but one displaced by 1.5 cm in z.  Phase B arrives with a converged fit (window
    4 sqrt(C11 + 0.0225) < 0.8 cm): skip.  Phase C restarts at row 151 with C0 = diag(1, 2.25, 1, 1, 100): its window on row 150 is
    w_max = 3 cm, the cluster is taken (rows between first_assigned and r_out are searched, no gap counting there).
    Fails under: Phase C searching only below first_assigned; Phase C keeping Phase B's covariance (no reset to C0)."""
    full = _track_rows()
    y150, z150 = full[150][0]
    full[150] = [(y150, z150 + 1.5)]
    o = _oracle(full).run("s6")
    tl = o.tracklets()
    assert len(tl["n"]) >= 1
    for i in range(len(tl["n"])):
        if tl["last"][i] != 151:
            continue
        assert tl["rowhit"][i][150] == 0 and tl["n"][i] == 152 and tl["first"][i] == 0
    assert (tl["last"] == 151).sum() >= 1
    # the same cluster displaced by 3.5 cm is outside w_max for both passes
    full[150] = [(y150, z150 + 3.5)]
    tl = _oracle(full).run("s6").tracklets()
    sel = tl["last"] == 151
    assert sel.sum() >= 1 and np.all(tl["rowhit"][sel][:, 150] == -1) and np.all(tl["n"][sel] == 151)


def test_phase_c_gap_counts_only_below_the_first_assigned_row():
    """Rows 60..64 and 90..94 carry no cluster (5 > max_gap each) and the only chain long enough to seed is on rows 95..151 --
    rows 0..59 and 65..89 alternate (only the odd rows are populated there, so S2 finds no pair and S4 no seed).  Phase C comes down from
    151: first_assigned follows it through 65..89 (pick-ups reset the gap), the 5 empty rows 90..94 are below first_assigned = 95 ->
    stop.  With 4 empty rows (90..93) it goes on until the next 5-row hole at 60..64.
    Fails under: gap counted from r_out; gap not reset by a pick-up below first_assigned; first_assigned never lowered."""
    full = _track_rows()
    def build(hole_hi):
        rows = {}
        for r, c in full.items():
            if 60 <= r <= 64 or 90 <= r <= hole_hi:
                continue
            if r < 90 and r % 2 == 0:
                continue
            rows[r] = c
        return rows
    o = _oracle(build(94)).run("s6")
    assert {(f, l) for f, l, _, _ in _tracklet_rows(o)} == {(95, 151)}
    o = _oracle(build(93)).run("s6")
    got = {(f, l) for f, l, _, _ in _tracklet_rows(o)}
    assert got == {(65, 151)}, got          # row 94, four misses, then 89, 87, ... 65 (odd rows, one miss between); 64..60: five misses end the pass


def test_rows_the_inward_refit_never_reaches_are_cleared_reading_A33():
    """A hand-linked chain on rows 40..49 whose clusters lie on a line with dy/dx = 3.4 (sin phi = 0.959 > s_max = 0.95): Phase A
    follows the links without a gate until the fitted |sin phi| exceeds s_max (transport refused), Phase B is skipped, Phase C
    restarts from the last updated row r_out and its first inward transport is refused as well: stop_row = r_out - 1, so every
    row below r_out is cleared and the tracklet keeps exactly one cluster (n = 1, first = last = r_out).
    Fails under: the clearing loop removed (rows 40..r_out-1 keep their Phase-A clusters); clearing `< stop_row`."""
    rows = {r: [(3.4 * (X[r] - X[40]), 20.0)] for r in range(40, 50)}
    o = _oracle(rows).run("s1")
    N = int(o.off[-1])
    up = np.full(N, -1, np.int32); dn = np.full(N, -1, np.int32)
    for r in range(40, 49):
        up[o.off[r]] = 0                     # one cluster per row: sorted position 0
        dn[o.off[r + 1]] = 0
    o.set_links(up, dn)
    o.run_range("s4", "s5")
    tl = o.tracklets()
    assert len(tl["n"]) == 1
    r_out = int(tl["last"][0])
    assert 41 <= r_out <= 48                 # Phase A ran for at least one link and was stopped by s_max before the chain ended
    assert tl["n"][0] == 1 and tl["first"][0] == r_out
    assert list(np.nonzero(tl["rowhit"][0] >= 0)[0]) == [r_out]


def test_phase_a_follows_links_without_a_gate_and_phase_c_updates_assigned_rows_without_a_gate():
    """Hand-linked chain on a good track with ONE cluster displaced by 2.5 cm in z at row 70 (far outside any converged window,
    inside no from-origin S2 window): because it is linked, Phase A takes it, and Phase C -- which re-uses assigned clusters
    without searching -- keeps it: rowhit[70] is the displaced cluster and n = 152.  Fails under: a gate in Phase A; Phase C
    re-picking assigned rows."""
    full = _track_rows()
    y70, z70 = full[70][0]
    full[70] = [(y70, z70 + 2.5)]
    o = _oracle(full).run("s1")
    N = int(o.off[-1])
    up = np.full(N, -1, np.int32); dn = np.full(N, -1, np.int32)
    for r in range(60, 80):
        up[o.off[r]] = 0; dn[o.off[r + 1]] = 0
    o.set_links(up, dn)
    o.run_range("s4", "s5")
    tl = o.tracklets()
    assert len(tl["n"]) == 1 and tl["rowhit"][0][70] == 0 and tl["n"][0] == 152 and (tl["first"][0], tl["last"][0]) == (0, 151)
    assert tl["chi2"][0] > 100.0             # the outlier is in the fit
