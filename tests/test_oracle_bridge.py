"""Pins of the oracle's S4' seed bridging (NEXT-2 of SURVEY.md section 8(f); reading A39 of DESIGN.md): a start hit that
continues a lower chain across the rows a missing cluster takes out of the chain of mutual links is dropped, so that one
tracklet per track is built instead of one per chain piece.

Expected values come from hand-made inputs (clusters removed at known rows from noise-free tracks), set relations with
the S4 list, a brute-force probe, and generator truth -- not from the oracle's own formulas.
"""
import math

import numpy as np

from gen import workloads as W
from oracle.oracle import Oracle
from tests import helpers as H


def _tracks(n=40, seed=51, sigma=(0.0, 0.0), dropout=0.0, bz=0.5, pt=(0.5, 10.0)):
    p = W.Params(seed=seed, single_sector=1, mult_fixed=n, phi_lo=0.08, phi_hi=2 * math.pi / 18 - 0.08, bz=bz,
                 sigma_y=sigma[0], sigma_z=sigma[1], dropout=dropout, pt_lo=pt[0], pt_hi=pt[1], eta_max=0.5)
    return W.generate(p, "bridge")


def _remove(w, kill):
    """Copy of the workload without the clusters flagged in `kill` (CSR offsets rebuilt)."""
    keep = ~kill
    cnt = np.array([int(keep[w.unit_off[u]:w.unit_off[u + 1]].sum()) for u in range(len(w.unit_off) - 1)], dtype=np.int64)
    off = np.zeros(len(w.unit_off), dtype=np.int64); off[1:] = np.cumsum(cnt)
    return W.Workload(w.name, w.params, w.n_sectors, w.n_rows, w.row_x, off, w.y[keep].copy(), w.t[keep].copy(), w.q[keep].copy(),
                      w.label[keep].copy(), w.leg0[keep].copy(), w.particles, w.coll_t0, w.coll_mult)


def _row_of(w):
    row = np.zeros(w.n_clusters, dtype=np.int64)
    for u in range(len(w.unit_off) - 1):
        row[w.unit_off[u]:w.unit_off[u + 1]] = u % w.n_rows
    return row


def _starts(o):
    return list(zip(o.get("start_unit").tolist(), o.get("start_pos").tolist()))


def test_single_dropouts_leave_one_start_hit_per_track():
    """Noise-free tracks crossing all 152 rows, two clusters removed per track (rows 50 and 100): the chain of mutual links
    breaks into three pieces (S4: three start hits per track); with bridging over the 4 missing-link rows only the innermost
    piece keeps its start hit."""
    w0 = _tracks()
    row = _row_of(w0)
    full = [p for p in range(len(w0.particles["pt"])) if (w0.label == p).sum() == w0.n_rows]
    assert len(full) >= 20
    sel = np.isin(w0.label, full)
    w = _remove(w0, ~sel | (sel & ((row == 50) | (row == 100))))
    base = Oracle.for_workload(w, sigma_y=0.1, sigma_z=0.15).run("s4")
    assert len(_starts(base)) == 3 * len(full)
    br = Oracle.for_workload(w, sigma_y=0.1, sigma_z=0.15, bridge_rows=4, bridge_min=3).run("s4")
    s = _starts(br)
    assert len(s) == len(full) and all(u % w.n_rows == 1 for u, _ in s)      # one per track, on row 1 (row 0 holds no links)
    # a gap wider than bridge_rows is not bridged: rows 50..52 removed -> 6 rows without links
    w2 = _remove(w0, ~sel | (sel & ((row >= 50) & (row <= 52))))
    assert len(_starts(Oracle.for_workload(w2, sigma_y=0.1, sigma_z=0.15, bridge_rows=4).run("s4"))) == 2 * len(full)
    assert len(_starts(Oracle.for_workload(w2, sigma_y=0.1, sigma_z=0.15, bridge_rows=6).run("s4"))) == len(full)


def test_bridge_min_protects_short_lower_chains():
    """The lower chain must hold at least bridge_min clusters: with the dropout at row 8 the lower piece has 6 linked
    clusters (rows 1..6: row 0 carries no links, row 7 lost its pair), so bridge_min = 8 keeps both start hits and
    bridge_min = 6 drops the upper one."""
    w0 = _tracks()
    row = _row_of(w0)
    full = [p for p in range(len(w0.particles["pt"])) if (w0.label == p).sum() == w0.n_rows]
    sel = np.isin(w0.label, full)
    w = _remove(w0, ~sel | (sel & (row == 8)))
    n8 = len(_starts(Oracle.for_workload(w, sigma_y=0.1, sigma_z=0.15, bridge_rows=4, bridge_min=8).run("s4")))
    n6 = len(_starts(Oracle.for_workload(w, sigma_y=0.1, sigma_z=0.15, bridge_rows=4, bridge_min=6).run("s4")))
    assert n8 == 2 * len(full) and n6 == len(full)


def test_bridged_list_is_an_ordered_subset_and_off_means_s4():
    w = W.config(1)
    base = _starts(Oracle.for_workload(w).run("s4"))
    off = _starts(Oracle.for_workload(w, bridge_rows=0, bridge_min=8).run("s4"))
    br = _starts(Oracle.for_workload(w, bridge_rows=4, bridge_min=8).run("s4"))
    assert off == base
    assert len(br) < 0.8 * len(base) and br == sorted(br)
    it = iter(base)
    assert all(any(x == y for y in it) for x in br)             # subsequence of the S4 list


def test_bridge_probe_equals_brute_force_over_the_row():
    w = W.config(1)
    a = Oracle.for_workload(w, bridge_rows=5, bridge_min=6).run("s4")
    b = Oracle.for_workload(w, bridge_rows=5, bridge_min=6).run("s4", brute_links=True)
    assert _starts(a) == _starts(b)
    c = Oracle.for_workload(w, bridge_rows=5, bridge_min=6, grid_scale=0.37).run("s4")
    orig = lambda o: sorted((u, int(o.get("perm")[w.unit_off[u] + p])) for u, p in _starts(o))   # caller's cluster indices
    assert orig(a) == orig(c)                                     # independent of the bin size


def test_bridging_trades_few_tracks_for_fewer_tracklets():
    """The documented operating point (bridge_rows = 4, bridge_min = 8): at least a third fewer tracklets, efficiency versus
    generator truth within 0.3 % of S4's, no more fakes (C1 and a C2-shaped event at 20 % multiplicity)."""
    for w in (W.config(1), W.config(2, scale=0.2)):
        o0 = Oracle.for_workload(w).run("s6")
        o1 = Oracle.for_workload(w, bridge_rows=4, bridge_min=8).run("s6")
        m0, m1 = H.truth_metrics(w, o0.tracks()), H.truth_metrics(w, o1.tracks())
        assert len(o1.get("start_unit")) <= 0.72 * len(o0.get("start_unit"))
        assert m1["eff"] >= m0["eff"] - 0.003 and m1["fake_rate"] <= m0["fake_rate"] + 0.002, (m0["eff"], m1["eff"])


# ------------------------------------------------------------------ S4' with rescue wave (reading A39c)
def _fitted(o):
    return o.get("tl_first") >= 0


def test_rescue_variant_skips_only_seeds_whose_chain_is_used():
    """bridge_rescue = 1: the start list is S4's; the first wave is exactly the non-bridged start hits; a bridged start hit is
    left unfitted iff every cluster of its chain of links lies on a kept first-wave tracklet (recomputed here from the tracklets)."""
    w = W.config(1)
    base = Oracle.for_workload(w).run("s6")
    o = Oracle.for_workload(w, bridge_rows=4, bridge_min=3, bridge_rescue=1).run("s6")
    plain = Oracle.for_workload(w, bridge_rows=4, bridge_min=3).run("s4")
    assert _starts(o) == _starts(base)
    wave = o.get("start_wave"); fit = _fitted(o)
    assert [s for s, wv in zip(_starts(o), wave) if wv == 1] == _starts(plain)
    assert np.all(fit[wave == 1]) and 0 < fit[wave == 2].sum() < (wave == 2).sum()
    tl = o.tracklets(); R = w.n_rows; off = w.unit_off
    used = np.zeros(w.n_clusters, bool)
    for i in np.nonzero((wave == 1) & (tl["n"] >= 10))[0]:
        rows = np.nonzero(tl["rowhit"][i] >= 0)[0]
        rows = rows[(rows >= tl["first"][i]) & (rows <= tl["last"][i])]
        used[off[tl["sector"][i] * R + rows] + tl["rowhit"][i][rows]] = True
    up = o.get("clean_up")
    for i in np.nonzero(wave == 2)[0]:
        u, p = int(o.get("start_unit")[i]), int(o.get("start_pos")[i]); all_used = True
        while True:
            g = off[u] + p
            if not used[g]:
                all_used = False; break
            if up[g] < 0:
                break
            p = int(up[g]); u += 1
        assert fit[i] == (not all_used), i


def test_rescue_variant_on_hand_made_dropouts_and_truth():
    """Noise-free tracks with two removed clusters: one fitted tracklet per track instead of three, same tracks.  C1 and a
    C2-shaped event: at most 60 % of the tracklets fitted, efficiency within 0.1 % of S4's, no extra fakes."""
    w0 = _tracks()
    row = _row_of(w0)
    full = [p for p in range(len(w0.particles["pt"])) if (w0.label == p).sum() == w0.n_rows]
    sel = np.isin(w0.label, full)
    w = _remove(w0, ~sel | (sel & ((row == 50) | (row == 100))))
    a = Oracle.for_workload(w, sigma_y=0.1, sigma_z=0.15).run("s6")
    b = Oracle.for_workload(w, sigma_y=0.1, sigma_z=0.15, bridge_rows=4, bridge_min=3, bridge_rescue=1).run("s6")
    assert _fitted(a).sum() == 3 * len(full) and _fitted(b).sum() == len(full)
    ta, tb = a.tracks(), b.tracks()
    sets = lambda t: sorted(tuple(zip(t["cl_row"][t["cl_begin"][i]:t["cl_begin"][i + 1]].tolist(),
                                      t["cl_index"][t["cl_begin"][i]:t["cl_begin"][i + 1]].tolist())) for i in range(len(t["sector"])))
    assert len(ta["sector"]) == len(tb["sector"]) == len(full) and sets(ta) == sets(tb)     # same tracks (another duplicate may win)
    for w in (W.config(1), W.config(2, scale=0.2)):
        o0 = Oracle.for_workload(w).run("s6")
        o1 = Oracle.for_workload(w, bridge_rows=4, bridge_min=3, bridge_rescue=1).run("s6")
        m0, m1 = H.truth_metrics(w, o0.tracks()), H.truth_metrics(w, o1.tracks())
        assert _fitted(o1).sum() <= 0.6 * _fitted(o0).sum()
        assert m1["eff"] >= m0["eff"] - 0.001 and m1["fake_rate"] <= m0["fake_rate"] + 0.001, (m0["eff"], m1["eff"])
