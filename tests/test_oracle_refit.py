"""Pins of the oracle's S7 ("improve the z-estimation"): refit of the clusters a
track owns after the selection (reading A37) and the collision time from the extrapolation to the beam line (reading A38).

Nothing here re-types the oracle's formulas: the expected values are the generator's collision times and closed-form
helix truth (tests/helpers.py), chi2 statistics, and invariances.
"""
import math

import numpy as np

from gen import workloads as W
from oracle.oracle import Oracle
from tests import helpers as H


def _frame(seed, sigma, dropout, t_frame=300.0, rate=0.02, mult=150, pt=(0.3, 10.0), bz=0.5):
    """One-sector continuous time frame: a few collisions at Poisson times, primaries only, no noise."""
    p = W.Params(seed=seed, single_sector=1, t_frame=t_frame, rate_per_us=rate, mult_mean=mult, mult_cap=4 * mult,
                 phi_lo=0.06, phi_hi=2 * math.pi / 18 - 0.06, bz=bz, sigma_y=sigma[0], sigma_z=sigma[1], dropout=dropout,
                 pt_lo=pt[0], pt_hi=pt[1])
    return W.generate(p, "refit")


def _pure(w, tr):
    return [(i, lab) for i, (lab, frac) in enumerate(H.track_labels(w, tr)) if lab >= 0 and frac == 1.0]


def test_refit_recovers_noise_free_helix_and_collision_time():
    """Double instance, noise-free hits: refitted state = closed-form helix (1e-5, reading A18) and t0 = the generator's
    collision time.  Tolerance of t0: (|dz| + S |d(dz/ds)|) / vdrift <= (1e-5 + 250 * 1e-5) / 2.58 = 1e-3 us."""
    w = _frame(41, (0.0, 0.0), 0.0)
    assert w.n_collisions >= 3 and float(np.ptp(w.coll_t0)) > 50.0         # collision times spread over the frame
    o = Oracle.for_workload(w, double=True, sigma_y=0.1, sigma_z=0.15).run("s7")
    tr, rf = o.tracks(), o.refit()
    P = w.particles
    n = 0
    for i, lab in _pure(w, tr):
        if rf["n"][i] < 40:
            continue
        phl = H.wrap_pi(P["phi"][lab] - H.sector_alpha(0))
        truth = H.helix_truth_at(rf["x"][i], P["pt"][lab], P["charge"][lab], phl, abs(P["tanl"][lab]), w.params.bz)
        truth[1] -= w.params.vdrift * P["t0"][lab]                          # scaled z of a collision at t0 (reading A6)
        d = rf["par"][i] - truth
        # z: the fp32 time stamps (t up to 550 us, half ulp 3e-5 us = 8e-5 cm per hit) set the floor, not the fit
        assert np.all(np.abs(d[[0, 2, 3]]) <= 1e-5) and abs(d[1]) <= 8e-5 and abs(d[4]) <= 1e-5 * abs(truth[4]) + 1e-7, (i, d)
        assert abs(rf["t0"][i] - P["t0"][lab]) <= 1e-3, (i, rf["t0"][i], P["t0"][lab])
        assert abs(rf["z0"][i] + w.params.vdrift * rf["t0"][i]) <= 1e-9 * max(1.0, abs(rf["z0"][i]))
        n += 1
    assert n >= 40


def test_refit_bz0_collision_time_is_straight_line_extrapolation():
    """Bz = 0: the arc to the beam line is the chord, z0 = z - (dz/ds) sqrt(x^2 + y^2) exactly."""
    w = _frame(42, (0.0, 0.0), 0.0, bz=0.0)
    o = Oracle.for_workload(w, double=True, sigma_y=0.1, sigma_z=0.15).run("s7")
    rf = o.refit()
    assert len(rf["n"]) >= 30
    for i in range(len(rf["n"])):
        y, z, _, t, q = rf["par"][i]
        assert q == 0.0
        z0 = z - t * math.hypot(rf["x"][i], y)
        assert abs(rf["z0"][i] - z0) <= 1e-9 * max(1.0, abs(z0))


def test_refit_chi2_ndf_and_t0_statistics_on_smeared_tracks():
    """fp32 parity instance, Gaussian-smeared hits with dropout.  After the refit EVERY pure track is a sample of the
    fit's statistics -- also the ones that lost clusters to a neighbour in S6 (the point of reading A37): mean chi2/ndf = 1
    +- 3/sqrt(sum ndf / 2), covariance SPD, ndf = 2 n - 5 with n = owned clusters; t0 unbiased with a sub-microsecond spread."""
    chi2 = 0.0; ndf = 0; dt = []; lost = 0
    for seed in (43, 44, 45):
        w = _frame(seed, (0.1, 0.15), 0.05, pt=(0.5, 10.0))
        o = Oracle.for_workload(w).run("s7")
        tr, rf = o.tracks(), o.refit()
        for i, lab in _pure(w, tr):
            nc = int(tr["cl_begin"][i + 1] - tr["cl_begin"][i])
            assert rf["n"][i] <= nc and rf["ndf"][i] == 2 * rf["n"][i] - 5
            if rf["n"][i] != nc or nc < 40:
                continue
            lost += tr["ndf"][i] != 2 * nc - 5
            tri = rf["cov"][i]; Cm = np.zeros((5, 5)); k = 0
            for a in range(5):
                for b in range(a + 1):
                    Cm[a, b] = Cm[b, a] = tri[k]; k += 1
            assert np.all(np.linalg.eigvalsh(Cm) > 0)
            chi2 += rf["chi2"][i]; ndf += int(rf["ndf"][i])
            dt.append(rf["t0"][i] - w.particles["t0"][lab])
    dt = np.array(dt)
    assert len(dt) >= 200 and lost >= 1
    assert abs(chi2 / ndf - 1.0) < 3.0 / math.sqrt(ndf / 2.0), chi2 / ndf
    assert dt.std() < 0.5 and abs(dt.mean()) < 3.0 * dt.std() / math.sqrt(len(dt)) + 1e-3, (dt.mean(), dt.std())


def test_refit_collision_time_follows_a_time_shift():
    """Shifting every cluster time by D shifts every t0 by D and leaves the other parameters alone (reading A6 / A38)."""
    w = _frame(46, (0.1, 0.15), 0.05)
    geo = w.geometry(); geo["t_frame"] = 1000.0
    D = 512.0
    a = Oracle(double=True, **geo); a.load(w.unit_off, w.y, w.t); a.run("s7")
    b = Oracle(double=True, **geo); b.load(w.unit_off, w.y, (w.t.astype(np.float64) + D).astype(np.float32)); b.run("s7")
    ta, tb, ra, rb = a.tracks(), b.tracks(), a.refit(), b.refit()
    key = lambda t, i: tuple(t["cl_index"][t["cl_begin"][i]:t["cl_begin"][i + 1]])
    ib = {key(tb, i): i for i in range(len(tb["sector"]))}
    n = 0
    for i in range(len(ta["sector"])):
        j = ib.get(key(ta, i))
        if j is None:
            continue
        # fp32 time stamps: t + 512 is rounded to 2^-14 us (6e-5 us, 1.6e-4 cm per hit); the extrapolation over ~1 m to the
        # beam line amplifies the resulting slope change a few times
        assert abs((rb["t0"][j] - ra["t0"][i]) - D) < 1e-3, (i, rb["t0"][j] - ra["t0"][i])
        sig = np.sqrt(ra["cov"][i][[0, 5, 9, 14]])           # that rounding moves the other parameters by a few % of their error
        assert np.all(np.abs(rb["par"][j][[0, 2, 3, 4]] - ra["par"][i][[0, 2, 3, 4]]) <= 0.05 * sig), (i, sig)
        n += 1
    assert n >= 0.8 * len(ta["sector"]) and n > 50


def test_refit_of_an_untouched_tracklet_reproduces_its_fit():
    """A track that owns every cluster of its tracklet: the refit runs over the same clusters, so n, ndf agree and the
    state agrees within a small fraction of its error (the two inward passes start from slightly different linearisations)."""
    w = _frame(47, (0.1, 0.15), 0.05)
    o = Oracle.for_workload(w, double=True).run("s7")
    tr, rf = o.tracks(), o.refit()
    n = 0
    for i in range(len(tr["sector"])):
        nc = int(tr["cl_begin"][i + 1] - tr["cl_begin"][i])
        if tr["ndf"][i] != 2 * nc - 5 or rf["n"][i] != nc:
            continue
        sig = np.sqrt(np.array([tr["cov"][i][0], tr["cov"][i][2], tr["cov"][i][5], tr["cov"][i][9], tr["cov"][i][14]]))
        assert rf["x"][i] == tr["x"][i] and rf["ndf"][i] == tr["ndf"][i]
        assert np.all(np.abs(rf["par"][i] - tr["par"][i]) <= 0.05 * sig), (i, (rf["par"][i] - tr["par"][i]) / sig)
        assert abs(rf["chi2"][i] - tr["chi2"][i]) <= 0.02 * max(1.0, tr["chi2"][i])
        n += 1
    assert n >= 50
