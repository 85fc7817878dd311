"""Pins of the oracle's S10 (NEXT-3, second half, SURVEY.md section 8(f).3 "recognise returning legs / extra turns"
"looping tracks", "secondary legs of looping tracks below 200 MeV/c"; reading A46 of DESIGN.md): S6 tracks of one
sector that are successive turns of one looping particle are chained (prev), grouped under their first turn (root) and numbered (turn).

No formula of the oracle is re-typed: the expected turn numbers come from the generator's particle parameters through the closed form
pitch = 2 pi rho tan(lambda), rho = pT / (0.29979 B), the grouping from the generator's particle labels, the window logic from
noise-free events where the matches survive windows twenty times tighter.
Fails under (checked by mutating oracle/tpc_oracle.cpp): pitch without the 2 pi; pitch from q_B instead of the mean dz/ds sign
(n < 1 accepted); predecessor = largest n; no transport of B to x_A.
"""
import math

import numpy as np

from gen import workloads as W
from oracle.oracle import Oracle
from tests import helpers as H
from tests import parity as P


def _loopers(seed=61, n=160, sigma=(0.1, 0.15), dropout=0.05, noise=300):
    return W.generate(W.Params(seed=seed, mult_fixed=200, pt_lo=0.3, pt_hi=5.0, n_loopers=n, loop_pt_lo=0.07, loop_pt_hi=0.14, loop_turns=8,
                               sigma_y=sigma[0], sigma_z=sigma[1], dropout=dropout, noise_per_sector=noise), "loopers")


def _run(w, **params):
    o = Oracle.for_workload(w, **params).run("s6")        # (a geometry field such as sigma_y given explicitly overrides the workload's)
    o.run_range("s10", "s10")
    return o, o.tracks(), o.loopers()


def _check_turns(w):
    """Every link of a noise-free event joins two pure tracks of one particle whose turn numbers differ by the closed-form count."""
    o, tr, lp = _run(w, sigma_y=0.1, sigma_z=0.15)
    labs = H.track_labels(w, tr)
    Pt = w.particles
    linked = np.nonzero(lp["prev"] >= 0)[0]
    n_checked = n_multi = 0
    for b in linked:
        a = int(lp["prev"][b])
        assert labs[a][0] == labs[b][0] >= 0 and labs[a][1] == labs[b][1] == 1.0          # same particle, pure tracks
        lab = labs[b][0]
        rho = Pt["pt"][lab] / abs(H.CB_PER_TESLA * w.params.bz)                               # cm
        pitch = 2 * math.pi * rho * abs(Pt["tanl"][lab])
        # both tracks sit on the same branch of the same circle at (nearly) the same x: their z differ by whole turns
        dz = abs(tr["par"][b][1] - tr["par"][a][1])
        n_true = int(round(dz / pitch))
        if abs(dz / pitch - n_true) < 0.2 and abs(tr["x"][a] - tr["x"][b]) < 3.0:
            assert lp["turn"][b] - lp["turn"][a] == n_true >= 1, (a, b, dz / pitch, lp["turn"][a], lp["turn"][b])
            n_checked += 1
            n_multi += n_true >= 2
    return o, tr, lp, linked, n_checked, n_multi


def test_turn_numbers_follow_the_closed_form_pitch_on_noise_free_loopers():
    w = _loopers(sigma=(0.0, 0.0), dropout=0.0, noise=0)
    o, tr, lp, linked, n_checked, n_multi = _check_turns(w)
    assert n_checked > 100
    # the matches are not an accident of wide windows: they survive windows twenty times tighter in y, sin(phi), dz/ds and q/pT
    o2, tr2, lp2 = _run(w, sigma_y=0.1, sigma_z=0.15, loop_dy=0.05, loop_ds=0.005, loop_dt=0.005, loop_dq=0.025)
    both = (lp["prev"] >= 0) & (lp2["prev"] >= 0)
    assert both.sum() >= 0.9 * len(linked) and np.array_equal(lp["prev"][both], lp2["prev"][both])


def test_a_missing_turn_is_jumped_and_counted():
    """The clusters of the second turn (pitch < z <= 2 pitch) of every looper are removed: the third turn then follows the first
    with n = 2, and the turn numbers still add up to the closed-form count."""
    from tests.test_oracle_bridge import _remove
    w0 = _loopers(sigma=(0.0, 0.0), dropout=0.0, noise=0)
    Pt = w0.particles
    z = w0.params.z_max - w0.params.vdrift * w0.t.astype(np.float64)
    lab = w0.label
    pitch = np.where(lab >= 0, 2 * math.pi * Pt["pt"][np.maximum(lab, 0)] / abs(H.CB_PER_TESLA * w0.params.bz) * np.abs(Pt["tanl"][np.maximum(lab, 0)]), np.inf)
    kill = (lab >= 0) & (Pt["kind"][np.maximum(lab, 0)] == 2) & (z > pitch) & (z <= 2 * pitch)
    assert kill.sum() > 1000
    o, tr, lp, linked, n_checked, n_multi = _check_turns(_remove(w0, kill))
    assert n_checked > 60 and n_multi >= 20


def test_grouping_against_generator_labels_on_smeared_loopers():
    for w in (_loopers(), W.config(4)):
        o, tr, lp = _run(w)
        labs = H.track_labels(w, tr)
        linked = np.nonzero(lp["prev"] >= 0)[0]
        assert len(linked) > 100
        same = sum(1 for i in linked if labs[i][0] >= 0 and labs[i][0] == labs[lp["prev"][i]][0])
        assert same >= 0.98 * len(linked), (same, len(linked))                               # purity of the links
        groups = {}
        for i, (lab, frac) in enumerate(labs):
            if lab >= 0 and frac >= 0.9 and abs(tr["par"][i][4]) >= 5.0:
                groups.setdefault((lab, int(tr["sector"][i])), []).append(i)
        tot = ok = 0
        for ids in groups.values():
            if len(ids) >= 2:
                _, cnt = np.unique(lp["root"][ids], return_counts=True)
                tot += len(ids) - 1; ok += cnt.max() - 1
        assert tot > 100 and ok >= 0.9 * tot, (ok, tot)                                      # turns of one particle end up in one group


def test_structure_of_the_result():
    w = W.config(4)
    o, tr, lp = _run(w)
    prev, root, turn = lp["prev"], lp["root"], lp["turn"]
    n = len(prev)
    assert n == len(tr["sector"]) and np.all(root[root] == root) and np.all(turn[root == np.arange(n)] == 0)
    has = prev >= 0
    assert np.all(tr["sector"][has] == tr["sector"][prev[has]]) and np.all(root[has] == root[prev[has]])
    assert np.all(turn[has] > turn[prev[has]]) and np.all(turn[~has] == 0) and np.all(root[~has] == np.arange(n)[~has])
    q = np.abs(tr["par"][:, 4])
    assert np.all(q[has] >= 5.0) and np.all(q[prev[has]] >= 5.0)                             # below 200 MeV/c only
    assert turn.max() <= 20 * 10
    # nothing to group without loopers: C2 at 40 % (a central event of primaries and secondaries above 100 MeV/c)
    w2 = W.config(2, scale=0.4)
    o2, tr2, lp2 = _run(w2)
    assert (lp2["prev"] >= 0).sum() <= 0.002 * len(tr2["sector"])
    # the threshold is a parameter and applies to BOTH tracks: above every track's |q/pT| nothing is grouped; set between the
    # two |q/pT| of a linked pair, that link disappears whichever of the two is the slower one
    o3, tr3, lp3 = _run(w, loop_qmin=1e6)
    assert np.all(lp3["prev"] == -1)
    n_tested = 0
    for b in np.nonzero(has)[0]:
        a = int(prev[b])
        if abs(q[a] - q[b]) > 0.3 and n_tested < 6 and (q[a] < q[b]) == (n_tested % 2 == 0):
            o4, tr4, lp4 = _run(w, loop_qmin=0.5 * (q[a] + q[b]))
            assert lp4["prev"][b] != a
            n_tested += 1
    assert n_tested >= 4
