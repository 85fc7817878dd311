"""Pins of the oracle's S8 (NEXT-4 of SURVEY.md section 8(f); "The tracker forms tubes of 1.5 cm around each
track, and marks unattached clusters as adjacent to the tube of the track with the highest transverse momentum it lies
in"; reading A40 of DESIGN.md).

The expected values come from an independent restatement in numpy that evaluates the closed-form helix of every track at
every pad row (no stepping, no grid), from brute force over whole rows, and from generator truth.
"""
import math

import numpy as np

from gen import workloads as W
from oracle.oracle import Oracle
from tests import helpers as H

TUBE = 1.5


def _restate(w, o, tr):
    """(status, track) per cluster from the definition: closed-form circle through the S6 state of each track."""
    R = w.n_rows
    X = w.row_x.astype(np.float64)
    cB = H.CB_PER_TESLA * float(np.float32(w.params.bz))
    z_all = o.get("z")                        # S0 output, caller's order
    N = w.n_clusters
    status = np.zeros(N, np.int32); track = np.full(N, -1, np.int32)
    first = o.tracklets()["first"]
    for i in range(len(tr["sector"])):
        a, b = tr["cl_begin"][i], tr["cl_begin"][i + 1]
        g = w.unit_off[tr["sector"][i] * R + tr["cl_row"][a:b]] + tr["cl_index"][a:b]
        status[g] = 1; track[g] = i
    best_q = np.full(N, np.inf)
    multi = np.zeros(N, np.int32)
    for i in range(len(tr["sector"])):
        y0, z0, s0, t0, q0 = tr["par"][i]
        if not np.isfinite(q0):
            continue
        sec = int(tr["sector"][i]); r0 = int(first[tr["tracklet"][i]]); r1 = int(tr["cl_row"][tr["cl_begin"][i + 1] - 1])
        k = cB * q0
        for r in range(r0, r1 + 1):
            s1 = s0 + k * (X[r] - X[r0])
            if abs(s1) > 0.95:
                break
            c0, c1 = math.sqrt(1 - s0 * s0), math.sqrt(1 - s1 * s1)
            if abs(k) > 1e-12:
                y = y0 + (c0 - c1) / k; z = z0 + t0 * (math.asin(s1) - math.asin(s0)) / k
            else:
                y = y0 + (X[r] - X[r0]) * s0 / c0; z = z0 + t0 * (X[r] - X[r0]) / c0
            lo, hi = int(w.unit_off[sec * R + r]), int(w.unit_off[sec * R + r + 1])
            d2 = (w.y[lo:hi].astype(np.float64) - y) ** 2 + (z_all[lo:hi] - z) ** 2
            for c in np.nonzero((d2 <= TUBE * TUBE) & (status[lo:hi] != 1))[0] + lo:
                multi[c] += 1
                if abs(q0) < best_q[c]:            # ascending track index: a tie keeps the lower index
                    best_q[c] = abs(q0); status[c] = 2; track[c] = i
    return status, track, multi


def test_tube_status_equals_closed_form_restatement():
    """Double instance on a dense single-sector event (tubes of neighbouring tracks overlap): identical status and track
    for every cluster, including the highest-pT rule where a cluster lies in several tubes."""
    w = W.generate(W.Params(seed=61, single_sector=1, mult_fixed=400, phi_lo=0.0, phi_hi=2 * math.pi / 18, noise_per_sector=3000,
                            dropout=0.08), "tube")
    o = Oracle.for_workload(w, double=True).run("s8")
    tr = o.tracks()
    st, tk = o.cluster_status()
    est, etk, multi = _restate(w, o, tr)
    assert (multi >= 2).sum() >= 20                                   # the highest-pT rule is exercised
    assert (st == 2).sum() >= 300 and (st == 0).sum() >= 1000
    assert np.array_equal(st, est) and np.array_equal(tk, etk), (np.nonzero(st != est)[0][:10], np.nonzero(tk != etk)[0][:10])


def test_tube_grid_lookup_equals_brute_force_and_is_grid_independent():
    w = W.config(1)
    oa = Oracle.for_workload(w).run("s8")
    a = oa.cluster_status()
    b = Oracle.for_workload(w).run("s8", brute_pickup=True).cluster_status()
    assert np.array_equal(a[0], b[0]) and np.array_equal(a[1], b[1])
    oc = Oracle.for_workload(w, grid_scale=0.41).run("s8")
    c = oc.cluster_status()
    assert np.array_equal(a[0], c[0])
    # another bin size renumbers the tracks (their order follows the sorted positions): compare the tracks' identities
    ident = lambda o: np.array([int(t["cl_row"][t["cl_begin"][i]]) * 100000 + int(t["cl_index"][t["cl_begin"][i]])
                                for t in [o.tracks()] for i in range(len(t["sector"]))] + [-1])
    assert np.array_equal(ident(oa)[a[1]], ident(oc)[c[1]])


def test_tube_status_against_generator_truth():
    """C1 (5 % dropout, 1000 noise clusters): attached = exactly the clusters of the track lists; what a track left behind of
    its own particle inside its row range lies a few sigma from the trajectory, far inside 1.5 cm, so it is adjacent -- to
    that track, or to a higher-pT track passing within 1.5 cm (those clusters were lost where tracks come close: the
    "moderate fake rate" of adjacent clusters); most of the uniform noise is in no tube; a wider tube never
    un-marks a cluster."""
    w = W.config(1)
    o = Oracle.for_workload(w).run("s8")
    tr = o.tracks(); st, tk = o.cluster_status()
    R = w.n_rows
    n_att = 0
    for i in range(len(tr["sector"])):
        a, b = tr["cl_begin"][i], tr["cl_begin"][i + 1]
        g = w.unit_off[tr["sector"][i] * R + tr["cl_row"][a:b]] + tr["cl_index"][a:b]
        assert np.all(st[g] == 1) and np.all(tk[g] == i)
        n_att += b - a
    assert (st == 1).sum() == n_att
    row = np.zeros(w.n_clusters, np.int64)
    for u in range(len(w.unit_off) - 1):
        row[w.unit_off[u]:w.unit_off[u + 1]] = u % R
    left = own = 0
    first = o.tracklets()["first"]
    for i, (lab, frac) in enumerate(H.track_labels(w, tr)):
        if lab < 0 or frac < 1.0:
            continue
        r0, r1 = first[tr["tracklet"][i]], tr["cl_row"][tr["cl_begin"][i + 1] - 1]
        sel = (w.label == lab) & (w.leg0 == 1) & (row >= r0) & (row <= r1) & (st != 1)
        left += sel.sum(); own += ((st[sel] == 2) & (tk[sel] == i)).sum()
        assert np.all(st[sel] == 2) and np.all(np.abs(tr["par"][tk[sel], 4]) <= abs(tr["par"][i][4]))
    assert left >= 20 and own >= 10, (left, own)
    noise = w.label < 0
    assert (st[noise] == 0).mean() > 0.8
    wide = Oracle.for_workload(w, tube=3.0).run("s8").cluster_status()[0]
    assert np.all((wide != 0) | (st == 0)) and (wide == 2).sum() > (st == 2).sum()
