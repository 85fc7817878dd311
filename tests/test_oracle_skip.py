"""Pins of the oracle's S2' (NEXT-2 as SURVEY.md section 8(f).2 wrote it: "links that may skip a row"; reading A45 of DESIGN.md;
`link_skip = 1`, off by default): a hit without an accepted pair on the adjacent rows may link over one missing row, so that a single
missing cluster no longer breaks the chain of mutual links.

Expected values come from hand-made inputs (clusters removed at known rows from noise-free tracks), an O(N^2) numpy restatement
written from the definition, set relations with the S2 tables, and generator truth -- not from the oracle's own formulas.
Fails under (checked by mutating oracle/tpc_oracle.cpp): level order swapped ((2,2) before (1,2)/(2,1)); windows not scaled with
the row distance; a / b of the adjacent rows used for a skipping pair; cleaner ignoring the row distance; Phase A transporting
one row for a two-row link.
"""
import math

import numpy as np

from gen import workloads as W
from oracle.oracle import Oracle
from tests import helpers as H
from tests.test_oracle_bridge import _remove, _row_of, _starts, _tracks


def _links_orig(w, o, names):
    """(up position, up distance, dn position, dn distance) re-expressed with ORIGINAL cluster indices, per original cluster."""
    R = w.n_rows
    perm = o.get("perm")
    up, dn, uk, dk = (o.get(n) for n in names)
    out = np.full((w.n_clusters, 4), -1, np.int64)
    for u in range(w.n_sectors * R):
        a, b = int(w.unit_off[u]), int(w.unit_off[u + 1])
        for p in range(b - a):
            g = a + int(perm[a + p])
            ku, kd = int(uk[a + p]), int(dk[a + p])
            if up[a + p] >= 0:
                out[g, 0] = perm[w.unit_off[u + ku] + up[a + p]]; out[g, 1] = ku
            if dn[a + p] >= 0:
                out[g, 2] = perm[w.unit_off[u - kd] + dn[a + p]]; out[g, 3] = kd
    return out


RAW = ("link_up", "link_dn", "link_up_k", "link_dn_k")
CLEAN = ("clean_up", "clean_dn", "clean_up_k", "clean_dn_k")


def test_single_dropouts_keep_one_chain_per_track():
    """Noise-free tracks crossing all 152 rows with the clusters of rows 50 and 100 removed: S2 breaks every chain into three
    pieces, S2' keeps ONE chain per track (1.0 tracklets per track); the links around a hole have row distance 2 on exactly
    the two clusters next to it.  Two adjacent missing rows (50, 51) are not bridged."""
    w0 = _tracks()
    row = _row_of(w0)
    full = [p for p in range(len(w0.particles["pt"])) if (w0.label == p).sum() == w0.n_rows]
    assert len(full) >= 20
    sel = np.isin(w0.label, full)
    w = _remove(w0, ~sel | (sel & ((row == 50) | (row == 100))))
    base = Oracle.for_workload(w, sigma_y=0.1, sigma_z=0.15).run("s4")
    assert len(_starts(base)) == 3 * len(full)
    sk = Oracle.for_workload(w, sigma_y=0.1, sigma_z=0.15, link_skip=1).run("s6")
    s = _starts(sk)
    assert len(s) == len(full) and all(u % w.n_rows == 1 for u, _ in s)
    r_of = _row_of(w)
    ck = _links_orig(w, sk, CLEAN)
    assert set(np.unique(r_of[ck[:, 1] == 2]).tolist()) == {49, 99} and set(np.unique(r_of[ck[:, 3] == 2]).tolist()) == {51, 101}
    assert (ck[:, 1] == 2).sum() == 2 * len(full)
    # every tracklet covers its whole track: 150 clusters, rows 0..151, the two holes empty
    tl = sk.tracklets()
    assert np.all(tl["n"] == 150) and np.all(tl["first"] == 0) and np.all(tl["last"] == 151)
    assert np.all(tl["rowhit"][:, 50] == -1) and np.all(tl["rowhit"][:, 100] == -1)
    assert len(sk.tracks()["sector"]) == len(full)
    w2 = _remove(w0, ~sel | (sel & ((row == 50) | (row == 51))))
    assert len(_starts(Oracle.for_workload(w2, sigma_y=0.1, sigma_z=0.15, link_skip=1).run("s4"))) == 2 * len(full)


def test_fit_through_skipping_links_recovers_the_helix():
    """Phase A transports over both rows of a skipping link in one step; the noise-free helix is still recovered to 1e-5
    (fp64 instance), which it would not be if the transport covered one row only."""
    w0 = _tracks(n=30, seed=52)
    row = _row_of(w0)
    full = [p for p in range(len(w0.particles["pt"])) if (w0.label == p).sum() == w0.n_rows]
    sel = np.isin(w0.label, full)
    w = _remove(w0, ~sel | (sel & ((row % 9) == 4)))
    o = Oracle.for_workload(w, double=True, sigma_y=0.1, sigma_z=0.15, link_skip=1).run("s6")
    tr = o.tracks()
    assert len(tr["sector"]) == len(full) == len(_starts(o))
    P = w.particles
    for i, (lab, frac) in enumerate(H.track_labels(w, tr)):
        assert frac == 1.0
        phl = H.wrap_pi(P["phi"][lab] - H.sector_alpha(0))
        truth = H.helix_truth_at(tr["x"][i], P["pt"][lab], P["charge"][lab], phl, abs(P["tanl"][lab]), w.params.bz)
        d = tr["par"][i] - truth
        assert np.all(np.abs(d[:4]) <= 1e-5) and abs(d[4]) <= 1e-5 * abs(truth[4]) + 1e-7, (i, d)


def test_links_of_s2_are_kept_and_grid_equals_brute_force():
    for w in (W.config(1, scale=0.1), W.generate(W.Params(seed=3, t_frame=200.0, rate_per_us=0.05, mult_mean=40.0, mult_cap=120,
                                                          sec_frac=0.2, noise_frac=0.02), "C3-tiny").sector_slice([0, 1, 18])):
        assert w.n_clusters < 6000
        base = Oracle.for_workload(w).run("s2")
        fast = Oracle.for_workload(w, link_skip=1).run("s4")
        slow = Oracle.for_workload(w, link_skip=1).run("s4", brute_links=True)
        for n in RAW + CLEAN + ("start_unit", "start_pos"):
            assert np.array_equal(fast.get(n), slow.get(n)), n
        had = base.get("link_up") >= 0                       # S2 is unchanged and final for the hits it linked
        assert np.array_equal(fast.get("link_up")[had], base.get("link_up")[had]) and np.all(fast.get("link_up_k")[had] == 1)
        assert np.array_equal(fast.get("link_dn")[had], base.get("link_dn")[had]) and np.all(fast.get("link_dn_k")[had] == 1)
        new = (fast.get("link_up") >= 0) & ~had
        assert new.sum() > 0.02 * w.n_clusters and np.all(fast.get("link_up_k")[new] + fast.get("link_dn_k")[new] >= 3)
        # bin-size invariance (original indices)
        ref = _links_orig(w, fast, RAW)
        for scale in (0.37, 2.9):
            assert np.array_equal(_links_orig(w, Oracle.for_workload(w, link_skip=1, grid_scale=scale).run("s2"), RAW), ref)


def test_mutual_links_carry_the_row_distance():
    w = W.config(1)
    o = Oracle.for_workload(w, link_skip=1).run("s4")
    R = w.n_rows
    cu, cd, ku, kd = (o.get(n) for n in CLEAN)
    n2 = 0
    for u in range(R):
        a, b = int(w.unit_off[u]), int(w.unit_off[u + 1])
        for h in range(b - a):
            if cu[a + h] >= 0:
                k = int(ku[a + h]); assert k in (1, 2)
                g = int(w.unit_off[u + k]) + int(cu[a + h])
                assert cd[g] == h and kd[g] == k
                n2 += k == 2
            else:
                assert ku[a + h] == 0
    assert n2 > 200
    # start hits = heads of chains of >= min_seed clusters, walking the row distances
    heads = []
    for u in range(R):
        a, b = int(w.unit_off[u]), int(w.unit_off[u + 1])
        for h in range(b - a):
            if cd[a + h] < 0 and cu[a + h] >= 0:
                n, uu, p = 1, u, h
                while cu[w.unit_off[uu] + p] >= 0:
                    k = int(ku[w.unit_off[uu] + p]); p = int(cu[w.unit_off[uu] + p]); uu += k; n += 1
                if n >= 3:
                    heads.append((u, h))
    assert heads == _starts(o)


def _restate(w, row_x, cut2, wy=1.5, wz=1.5, skip_cut2=None, **oracle_params):
    """O(N^2) restatement of S2' in numpy fp32 for the hits S2 left without a link, from the definition (reading A45).
    Returns the number of hits that got a skipping link.  skip_cut2: cut of the pairs that skip a row (default: the oracle's 1.75,
    which the callers that pass another cut2 set explicitly)."""
    base = Oracle.for_workload(w, cut2=cut2, **oracle_params).run("s2")
    skip_cut2 = cut2 if skip_cut2 is None else skip_cut2
    o = Oracle.for_workload(w, link_skip=1, cut2=cut2, skip_cut2=skip_cut2, **oracle_params).run("s2")
    got = _links_orig(w, o, RAW)
    base_up = _links_orig(w, base, RAW)[:, 0]
    f = np.float32
    X = np.asarray(row_x, np.float32).astype(np.float64)      # row_x is handed over as fp32
    z = (f(w.params.z_max) - f(w.params.vdrift) * w.t).astype(f)
    R = w.n_rows
    n_new = n_wide = 0
    for r in range(1, R - 1):
        for h in range(int(w.unit_off[r]), int(w.unit_off[r + 1])):
            if base_up[h] >= 0:
                continue
            y, zz = w.y[h], z[h]
            cand = {}
            for k in (1, 2):
                for sgn in (+1, -1):
                    rr = r + sgn * k
                    if rr < 0 or rr > R - 1:
                        cand[(sgn, k)] = []
                        continue
                    t_ = f(X[rr] / X[r])
                    yc, zc = f(y * t_), f(zz * t_)
                    hy, hz = f(k * wy), f(k * wz)
                    a0, b0 = int(w.unit_off[rr]), int(w.unit_off[rr + 1])
                    cand[(sgn, k)] = [i for i in range(a0, b0) if f(yc - hy) <= w.y[i] <= f(yc + hy) and f(zc - hz) <= z[i] <= f(zc + hz)]
            best = None
            for level in (((1, 2), (2, 1)), ((2, 2),)):
                for ku, kd in level:
                    if r + ku > R - 1 or r - kd < 0:
                        continue
                    A64, B64 = X[r + ku] - X[r], X[r] - X[r - kd]
                    A, B, lim = f(A64), f(B64), f(skip_cut2 * 0.5 * (A64 * A64 + B64 * B64))
                    for i in cand[(+1, ku)]:
                        for j in cand[(-1, kd)]:
                            ey = f(f(B * f(w.y[i] - y)) - f(A * f(y - w.y[j])))
                            ez = f(f(B * f(z[i] - zz)) - f(A * f(zz - z[j])))
                            D = f(f(ey * ey) + f(ez * ez))
                            if D < lim:
                                key = (float(D), ku, i - int(w.unit_off[r + ku]), j - int(w.unit_off[r - kd]), kd, i, j)
                                if best is None or key[:4] < best[:4]:
                                    best = key
                if best is not None:
                    break
            if best is None:
                assert tuple(got[h]) == (-1, -1, -1, -1), (r, h, got[h])
            else:
                assert tuple(got[h]) == (best[2], best[1], best[3], best[4]), (r, h, got[h], best)
                n_new += 1
                i, j, ku, kd = best[5], best[6], best[1], best[4]
                yu, yd = f(y * f(X[r + ku] / X[r])), f(y * f(X[r - kd] / X[r]))
                n_wide += (ku == 2 and abs(float(w.y[i]) - float(yu)) > wy) or (kd == 2 and abs(float(w.y[j]) - float(yd)) > wy)
    return n_new, n_wide


def test_numpy_restatement_of_the_skip_levels():
    n_new, _ = _restate(W.config(1, scale=0.1), H.row_x(), cut2=1.75)
    assert n_new > 40


def test_numpy_restatement_on_a_dense_cloud():
    """Rows 40..59 with 18 random clusters each in a 7 x 7 cm box and a loose cut (cut2 = 25): many candidates per window and
    many accepted pairs per level, among them links that exist only because the windows grow with the row distance and because
    every (k_u, k_d) level has its own threshold."""
    rng = np.random.default_rng(123)
    base = W.config(1, scale=0.05)
    R = base.n_rows
    off = np.zeros(R + 1, np.int64)
    ys, ts = [], []
    for r in range(R):
        n = 18 if 40 <= r < 60 and rng.uniform() > 0.25 else 0       # some rows stay empty
        off[r + 1] = off[r] + n
        ys += list(rng.uniform(-3.5, 3.5, n)); ts += list((base.params.z_max - rng.uniform(100.0, 107.0, n)) / base.params.vdrift)
    w = W.Workload("cloud", base.params, 1, R, base.row_x, off, np.array(ys, np.float32), np.array(ts, np.float32),
                   np.ones(len(ys), np.float32), -np.ones(len(ys), np.int32), np.zeros(len(ys), np.uint8), base.particles, base.coll_t0, base.coll_mult)
    n_new, n_wide = _restate(w, base.row_x, cut2=25.0)
    assert n_new > 30 and n_wide > 5
    # the pairs that skip a row have their own cut (skip_cut2): a stricter one links fewer hits, S2 itself (cut2) is untouched
    n_strict, _ = _restate(w, base.row_x, cut2=25.0, skip_cut2=6.0)
    assert 5 < n_strict < n_new


def test_exact_tie_between_the_two_one_sided_levels_goes_to_the_shorter_up_link():
    """Unit row pitch (exact in fp32), all clusters at z = 0: h = (0) on row 50; row 51: a dummy far away (original index 0) and
    u1 = +1.25; row 49: d1 = +1.25; row 52: u2 = -2.5; row 48: d2 = -2.5.  The adjacent pair (u1, d1) has ey = 2.5, D = 6.25 >= thr =
    1.75: rejected.  (k_u, k_d) = (1, 2): ey = 2 * 1.25 - 1 * 2.5 = 0 and (2, 1): ey = 1 * (-2.5) + 2 * 1.25 = 0, both exactly: the
    tie goes to k_u = 1 although u2 has the lower original index.  Fails under: k_u dropped from the key."""
    R = 152
    rows = {51: [(40.0, 0.0), (1.25, 0.0)], 49: [(1.25, 0.0)], 50: [(0.0, 0.0)], 52: [(-2.5, 0.0)], 48: [(-2.5, 0.0)]}
    off = np.zeros(R + 1, np.int64); ys, ts = [], []
    for r in range(R):
        cl = rows.get(r, [])
        off[r + 1] = off[r] + len(cl); ys += [c[0] for c in cl]; ts += [(250.0 - c[1]) / 2.0 for c in cl]
    X = (100.0 + np.arange(R)).astype(np.float32)
    o = Oracle(n_sectors=1, n_rows=R, row_x=X, sector_dphi=2 * math.pi / 18, z_max=250.0, t_frame=0.0, sigma_y=0.1, sigma_z=0.15,
               bz=0.5, vdrift=2.0, link_skip=1)
    o.load(off, np.array(ys, np.float32), np.array(ts, np.float32)); o.run("s2")
    h = int(off[50])
    perm = o.get("perm")
    up, dn, ku, kd = (o.get(n)[h] for n in RAW)
    assert (ku, kd) == (1, 2) and perm[off[51] + up] == 1 and perm[off[48] + dn] == 0


def test_every_level_has_its_own_threshold():
    """Unit pitch, z = 0: h = 0 on row 50, u1 = +1.25 on row 51, d2 = -0.25 on row 48, nothing else.  (1, 2): ey = 2 * 1.25 - 0.25 =
    2.25, D = 5.0625; thr_12 = cut2 * 0.5 * (1 + 4) = 4.375 < D < thr_22 = cut2 * 0.5 * (4 + 4) = 7: no link.  With d2 = -0.5: D = 4 <
    4.375: linked.  Fails under: one threshold for all levels."""
    R = 152
    X = (100.0 + np.arange(R)).astype(np.float32)
    for yd, linked in ((-0.25, False), (-0.5, True)):
        rows = {51: [(1.25, 0.0)], 50: [(0.0, 0.0)], 48: [(yd, 0.0)]}
        off = np.zeros(R + 1, np.int64); ys, ts = [], []
        for r in range(R):
            cl = rows.get(r, [])
            off[r + 1] = off[r] + len(cl); ys += [c[0] for c in cl]; ts += [(250.0 - c[1]) / 2.0 for c in cl]
        o = Oracle(n_sectors=1, n_rows=R, row_x=X, sector_dphi=2 * math.pi / 18, z_max=250.0, t_frame=0.0, sigma_y=0.1, sigma_z=0.15,
                   bz=0.5, vdrift=2.0, link_skip=1)
        o.load(off, np.array(ys, np.float32), np.array(ts, np.float32)); o.run("s2")
        h = int(off[50])
        assert (o.get("link_up")[h] >= 0) == linked and (o.get("link_up_k")[h], o.get("link_dn_k")[h]) == ((1, 2) if linked else (0, 0))


def test_skip_cut2_is_the_cut_of_the_skipping_pairs_only():
    """Same hand-made case as above with d2 = -0.5: D = 4 against thr_12 = skip_cut2 * 0.5 * (1 + 4): linked at 1.75 (4.375) and at
    1.61 (4.025), not at 1.59 (3.975); cut2 (the adjacent pairs) does not enter: cut2 = 0.1 / 100 change nothing here.  And the other
    way: an adjacent pair with D = 0.25 (u1 = +0.25, d1 = +0.25: ey = 0.5) is accepted by cut2 = 1.75 (thr = 1.75) whatever skip_cut2 is.
    Fails under: skip_cut2 ignored; skip_cut2 applied to the adjacent level."""
    R = 152
    X = (100.0 + np.arange(R)).astype(np.float32)
    def run(rows, **params):
        off = np.zeros(R + 1, np.int64); ys, ts = [], []
        for r in range(R):
            cl = rows.get(r, [])
            off[r + 1] = off[r] + len(cl); ys += [c[0] for c in cl]; ts += [(250.0 - c[1]) / 2.0 for c in cl]
        o = Oracle(n_sectors=1, n_rows=R, row_x=X, sector_dphi=2 * math.pi / 18, z_max=250.0, t_frame=0.0, sigma_y=0.1, sigma_z=0.15,
                   bz=0.5, vdrift=2.0, link_skip=1, **params)
        o.load(off, np.array(ys, np.float32), np.array(ts, np.float32)); o.run("s2")
        h = int(off[50])
        return int(o.get("link_up_k")[h]), int(o.get("link_dn_k")[h])
    skipping = {51: [(1.25, 0.0)], 50: [(0.0, 0.0)], 48: [(-0.5, 0.0)]}
    assert run(skipping) == (1, 2) and run(skipping, skip_cut2=1.61) == (1, 2) and run(skipping, skip_cut2=1.59) == (0, 0)
    assert run(skipping, cut2=0.1) == (1, 2) and run(skipping, cut2=100.0, skip_cut2=1.59) == (0, 0)
    adjacent = {51: [(0.25, 0.0)], 50: [(0.0, 0.0)], 49: [(0.25, 0.0)]}
    assert run(adjacent) == (1, 1) and run(adjacent, skip_cut2=1e-6) == (1, 1) and run(adjacent, cut2=0.1) == (0, 0)


def test_a_stricter_cut_for_skipping_pairs_keeps_the_efficiency():
    """Operating point DESIGN.md section 11.1 proposes: skip_cut2 = 0.4375 (a quarter of cut2).  Generator truth: efficiency not
    below the r+-1 path by more than 0.05 %, fewer fakes than with skip_cut2 = cut2, still at most 0.7 of the start hits."""
    for w in (W.config(1), W.config(3, scale=0.1)):
        b = Oracle.for_workload(w).run("s6")
        loose = Oracle.for_workload(w, link_skip=1).run("s6")
        tight = Oracle.for_workload(w, link_skip=1, skip_cut2=0.4375).run("s6")
        mb, ml, mt = (H.truth_metrics(w, o.tracks()) for o in (b, loose, tight))
        assert mt["eff"] >= mb["eff"] - 0.0005, (mb["eff"], mt["eff"])
        assert mt["fakes"] <= ml["fakes"] and len(_starts(loose)) <= len(_starts(tight)) <= 0.7 * len(_starts(b))


def test_fewer_tracklets_at_the_documented_efficiency():
    """Generator truth at the operating point DESIGN.md section 11 documents: about half the tracklets of S2, efficiency within
    0.2 % of it, fake rate below 1 %."""
    for w, max_ratio in ((W.config(1), 0.45), (W.config(3, scale=0.1), 0.6)):
        b = Oracle.for_workload(w).run("s6"); s = Oracle.for_workload(w, link_skip=1).run("s6")
        assert len(_starts(s)) <= max_ratio * len(_starts(b))
        mb, ms = H.truth_metrics(w, b.tracks()), H.truth_metrics(w, s.tracks())
        assert ms["eff"] >= mb["eff"] - 0.002 and ms["fake_rate"] <= 0.01, (mb["eff"], ms["eff"], ms["fake_rate"])
        tr = s.tracks()
        g = w.unit_off[tr["sector"].repeat(np.diff(tr["cl_begin"])) * w.n_rows + tr["cl_row"]] + tr["cl_index"]
        assert len(np.unique(g)) == len(g)
