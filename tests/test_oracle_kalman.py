"""Pins of the oracle's Kalman part (S5 propagate / update / fit) and of the selector (S6) -- DESIGN.md section 6.

Closed forms, finite differences, textbook linear algebra and statistics; none of it calls the CUDA path.
"""
import math

import mpmath
import numpy as np
import pytest

from gen import workloads as W
from oracle.oracle import Oracle
from tests import helpers as H

GEO = dict(n_sectors=36, n_rows=152, row_x=H.row_x().astype(np.float32), sector_dphi=2 * math.pi / 18, z_max=250.0,
           t_frame=0.0, sigma_y=0.1, sigma_z=0.15, bz=0.5, vdrift=2.58)
CB = H.CB_PER_TESLA * 0.5


def _tri(Cm):
    return np.array([Cm[a, b] for a in range(5) for b in range(a + 1)])


def _full(tri):
    Cm = np.zeros((5, 5)); c = 0
    for a in range(5):
        for b in range(a + 1):
            Cm[a, b] = Cm[b, a] = tri[c]; c += 1
    return Cm


def _circle(par, dx):
    """Closed-form transport on a circle: y=y0+(cos0-cos1)/k, z=z0+t(phi1-phi0)/k, sin1=sin0+k dx.

    Evaluated with 60 digits (mpmath) so that the textbook form, which cancels badly at small k, is a usable reference.
    """
    mp = mpmath.mp.clone(); mp.dps = 60
    y, z, s, t, q = [mp.mpf(float(v)) for v in par]
    k = mp.mpf(CB) * q
    dx = mp.mpf(float(dx))
    s1 = s + k * dx
    if k == 0:
        c = mp.sqrt(1 - s * s)
        out = [y + dx * s / c, z + t * dx / c, s, t, q]
    else:
        out = [y + (mp.sqrt(1 - s * s) - mp.sqrt(1 - s1 * s1)) / k, z + t * (mp.asin(s1) - mp.asin(s)) / k, s1, t, q]
    return np.array([float(v) for v in out])


@pytest.fixture(scope="module")
def od():
    return Oracle(double=True, **GEO)


@pytest.fixture(scope="module")
def of():
    return Oracle(double=False, **GEO)


CASES = [  # y, z, sinphi, dz/ds, q/pT ; dx
    ((3.0, -7.0, 0.10, 0.7, 1.0), 1.066225), ((-12.0, 40.0, -0.35, -1.0, -9.5), 1.066225), ((0.5, 2.0, 0.6, 0.3, 0.1), 25.0),
    ((0.0, 0.0, 0.0, 1.02, -3.0), 161.0), ((1.0, 1.0, 0.2, 0.5, 3.0), -40.0), ((1.0, 1.0, -0.7, -0.5, 1e-6), 60.0),
    ((2.0, 3.0, 0.3, 0.9, 0.0), 80.0),
]


@pytest.mark.parametrize("par,dx", CASES)
def test_propagate_state_equals_closed_form_circle(od, of, par, dx):
    ok, p1, _ = od.propagate(par, _tri(np.eye(5)), dx)
    assert ok
    assert np.allclose(p1, _circle(par, dx), rtol=0, atol=2e-12 * max(1.0, abs(dx)))
    ok, pf, _ = of.propagate(par, _tri(np.eye(5)), dx)      # the fp32 instance follows the same formulas
    ref = _circle(par, dx)
    assert ok and np.allclose(pf, ref, rtol=3e-6, atol=3e-6 * max(1.0, abs(dx)))


def test_propagate_composition_and_round_trip(od):
    rng = np.random.default_rng(1)
    for _ in range(50):
        par = np.array([rng.uniform(-20, 20), rng.uniform(-100, 100), rng.uniform(-0.4, 0.4), rng.uniform(-1, 1), rng.uniform(-3, 3)])
        A = rng.normal(size=(5, 5)); C0 = A @ A.T * 1e-2
        d1, d2 = rng.uniform(0.5, 30), rng.uniform(0.5, 30)
        ok1, p1, c1 = od.propagate(par, _tri(C0), d1)
        ok2, p2, c2 = od.propagate(p1, c1, d2)
        ok3, p3, c3 = od.propagate(par, _tri(C0), d1 + d2)
        assert ok1 and ok2 and ok3
        assert np.allclose(p2, p3, rtol=0, atol=1e-10)
        assert np.allclose(c2, c3, rtol=1e-7, atol=1e-9)           # Jacobians compose: F(x1->x2) F(x0->x1) = F(x0->x2)
        okb, pb, cb = od.propagate(p1, c1, -d1)
        assert okb and np.allclose(pb, par, rtol=0, atol=1e-10) and np.allclose(cb, _tri(C0), rtol=1e-7, atol=1e-9)


@pytest.mark.parametrize("par,dx", CASES)
def test_propagate_jacobian_equals_finite_differences(od, par, dx):
    """C' = F C F^T with F probed column by column through rank-one covariances, against central differences of the circle."""
    par = np.array(par, dtype=np.float64)
    F_fd = np.zeros((5, 5))
    for j in range(5):
        h = 1e-6 * max(1.0, abs(par[j]))
        pp, pm = par.copy(), par.copy(); pp[j] += h; pm[j] -= h
        F_fd[:, j] = (_circle(pp, dx) - _circle(pm, dx)) / (2 * h)
    for j in range(5):
        e = np.zeros((5, 5)); e[j, j] = 1.0
        _, _, c = od.propagate(par, _tri(e), dx)
        assert np.allclose(_full(c), np.outer(F_fd[:, j], F_fd[:, j]), rtol=2e-6, atol=2e-7 * max(1.0, dx * dx))
    # off-diagonal signs: a full covariance
    A = np.arange(25, dtype=np.float64).reshape(5, 5) / 10 + np.eye(5); C0 = A @ A.T
    _, _, c = od.propagate(par, _tri(C0), dx)
    ref = F_fd @ C0 @ F_fd.T
    assert np.allclose(_full(c), ref, rtol=3e-6, atol=1e-6 * np.abs(ref).max())


def test_propagate_finite_at_zero_curvature_and_fails_beyond_s_max(od, of):
    for o in (od, of):
        ok, p, c = o.propagate((1.0, 2.0, 0.3, 0.5, 0.0), _tri(np.eye(5)), 30.0)
        assert ok and np.all(np.isfinite(p)) and np.all(np.isfinite(c))
        ok, _, _ = o.propagate((0.0, 0.0, 0.9, 0.0, -10.0), _tri(np.eye(5)), 20.0)      # sin(phi) would reach 1.05
        assert not ok
        ok, _, _ = o.propagate((0.0, 0.0, 0.96, 0.0, 0.0), _tri(np.eye(5)), 1.0)        # already beyond s_max = 0.95
        assert not ok
    bz0 = Oracle(double=True, **{**GEO, "bz": 0.0})
    ok, p, c = bz0.propagate((1.0, 2.0, 0.3, 0.5, 4.0), _tri(np.eye(5)), 30.0)
    cphi = math.sqrt(1 - 0.09)
    assert ok and np.allclose(p, [1.0 + 30 * 0.3 / cphi, 2.0 + 0.5 * 30 / cphi, 0.3, 0.5, 4.0], atol=1e-12)


def test_update_equals_textbook_kalman(od, of):
    rng = np.random.default_rng(2)
    Hm = np.zeros((2, 5)); Hm[0, 0] = Hm[1, 1] = 1
    Rm = np.diag([0.1 ** 2, 0.15 ** 2])
    for _ in range(20):
        A = rng.normal(size=(5, 5)); C0 = A @ A.T + 0.1 * np.eye(5)
        par = rng.normal(size=5); m = rng.normal(size=2)
        S = Hm @ C0 @ Hm.T + Rm; K = C0 @ Hm.T @ np.linalg.inv(S); res = m - Hm @ par
        p_ref = par + K @ res; C_ref = C0 - K @ Hm @ C0; chi2_ref = res @ np.linalg.inv(S) @ res
        p, c, chi2 = od.update(par, _tri(C0), m[0], m[1])
        assert np.allclose(p, p_ref, atol=1e-11) and np.allclose(_full(c), C_ref, atol=1e-10) and abs(chi2 - chi2_ref) < 1e-9 * max(1, chi2_ref)
        p, c, chi2 = of.update(par, _tri(C0), m[0], m[1])
        assert np.allclose(p, p_ref, atol=2e-4) and abs(chi2 - chi2_ref) < 1e-3 * max(1, chi2_ref)


# ------------------------------------------------------------------ S5 fit on generated tracks
def _clean_tracks(bz, n=60, seed=21, sigma=(0.0, 0.0), pt=(0.3, 10.0), dropout=0.0):
    p = W.Params(seed=seed, single_sector=1, mult_fixed=n, phi_lo=0.06, phi_hi=2 * math.pi / 18 - 0.06, bz=bz,
                 sigma_y=sigma[0], sigma_z=sigma[1], dropout=dropout, pt_lo=pt[0], pt_hi=pt[1])
    return W.generate(p, "fit")


def _truth_for_tracks(w, tr):
    """(track index, truth state at the track's x) for every track that is pure (one label)."""
    P = w.particles
    out = []
    for i, (lab, frac) in enumerate(H.track_labels(w, tr)):
        if lab < 0 or frac < 1.0:
            continue
        phl = H.wrap_pi(P["phi"][lab] - H.sector_alpha(0))
        truth = H.helix_truth_at(tr["x"][i], P["pt"][lab], P["charge"][lab], phl, abs(P["tanl"][lab]), w.params.bz)
        out.append((i, truth))
    return out


def test_fit_recovers_noise_free_helix_to_1e5():
    """Reading A18: double instance, noise-free hits (fp32-rounded inputs), tracks with >= 40 clusters."""
    w = _clean_tracks(bz=0.5)
    o = Oracle.for_workload(w, double=True, sigma_y=0.1, sigma_z=0.15).run("s6")
    tr = o.tracks()
    n = 0
    for i, truth in _truth_for_tracks(w, tr):
        if tr["cl_begin"][i + 1] - tr["cl_begin"][i] < 40:
            continue
        d = tr["par"][i] - truth
        assert abs(d[0]) <= 1e-5 and abs(d[1]) <= 1e-5 and abs(d[2]) <= 1e-5 and abs(d[3]) <= 1e-5, (i, d)
        assert abs(d[4]) <= 1e-5 * abs(truth[4]) + 1e-7, (i, d)
        n += 1
    assert n >= 40


def test_fit_straight_lines_bz0_exact():
    w = _clean_tracks(bz=0.0)
    o = Oracle.for_workload(w, double=True, sigma_y=0.1, sigma_z=0.15).run("s6")
    tr = o.tracks()
    pairs = _truth_for_tracks(w, tr)
    assert len(pairs) >= 55
    for i, truth in pairs:
        d = tr["par"][i] - truth
        assert np.all(np.abs(d[:4]) < 2e-5), (i, d)      # fp32-rounded inputs set the floor
        assert tr["par"][i][4] == 0.0                      # q/pT unobservable at Bz = 0: stays at the prior


def test_fit_chi2_and_pulls_on_smeared_tracks():
    """Gaussian-smeared tracks at C1's density: mean chi2/ndf = 1 +- 3/sqrt(sum ndf / 2), pulls ~ N(0,1), covariance SPD.

    Only tracks that own every cluster of their tracklet are used: the reported state is the tracklet's (reading A17), so
    a tracklet that lost clusters to a neighbour was fitted through foreign hits and is not a sample of the fit's statistics.
    """
    pulls, chi2, ndf = [], 0.0, 0
    for seed in (33, 34, 35):
        w = _clean_tracks(bz=0.5, n=150, seed=seed, sigma=(0.1, 0.15), pt=(0.5, 10.0), dropout=0.05)
        tr = Oracle.for_workload(w).run("s6").tracks()              # the fp32 parity instance
        for i, truth in _truth_for_tracks(w, tr):
            nc = tr["cl_begin"][i + 1] - tr["cl_begin"][i]
            if nc < 60 or tr["ndf"][i] != 2 * nc - 5:
                continue
            Cm = _full(tr["cov"][i])
            assert np.allclose(Cm, Cm.T) and np.all(np.linalg.eigvalsh(Cm) > 0)          # symmetric positive definite
            pulls.append((tr["par"][i] - truth) / np.sqrt(np.diag(Cm)))
            chi2 += tr["chi2"][i]; ndf += tr["ndf"][i]
    pulls = np.array(pulls)
    assert len(pulls) >= 200
    assert abs(chi2 / ndf - 1.0) < 3.0 / math.sqrt(ndf / 2.0), chi2 / ndf
    rms = np.sqrt((pulls ** 2).mean(axis=0))
    assert np.all(rms > 0.85) and np.all(rms < 1.15), rms
    assert np.all(np.abs(pulls.mean(axis=0)) < 0.2), pulls.mean(axis=0)


def test_s5_one_tracklet_per_start_hit_and_pickup_equals_brute_force():
    w = W.config(1, scale=0.25)
    a = Oracle.for_workload(w).run("s6")
    b = Oracle.for_workload(w).run("s6", brute_links=True, brute_pickup=True)
    ta, tb = a.tracklets(), b.tracklets()
    assert len(ta["n"]) == len(a.get("start_unit"))        # single hypothesis per seed
    assert np.array_equal(ta["rowhit"], tb["rowhit"]) and np.array_equal(ta["par"], tb["par"])
    assert np.array_equal(a.tracks()["cl_index"], b.tracks()["cl_index"])


def test_s5_continuous_mode_is_shift_invariant_in_time():
    """Reading A6: a collision at t0 != 0 is found exactly like the same collision at t0 = 0 (rigid shift in scaled z)."""
    w0 = W.config(1, scale=0.25)
    geo = w0.geometry(); geo["t_frame"] = 1000.0
    a = Oracle(**geo); a.load(w0.unit_off, w0.y, w0.t); a.run("s6")
    b = Oracle(**geo); b.load(w0.unit_off, w0.y, (w0.t.astype(np.float64) + 512.0).astype(np.float32)); b.run("s6")
    ta, tb = a.tracks(), b.tracks()
    # 512 us * 2.58 cm/us is not a power of two in cm, so bins and roundings differ; the physics must not
    na, nb = len(ta["sector"]), len(tb["sector"])
    assert na > 20 and abs(na - nb) <= max(1, na // 50)
    sa = {tuple(ta["cl_index"][ta["cl_begin"][i]:ta["cl_begin"][i + 1]]) for i in range(na)}
    sb = {tuple(tb["cl_index"][tb["cl_begin"][i]:tb["cl_begin"][i + 1]]) for i in range(nb)}
    assert len(sa & sb) >= 0.9 * na


# ------------------------------------------------------------------ S6
def _select_case(rows_a, rows_b, n_a, n_b, chi_a, chi_b):
    """Two hand-built tracklets over a workload whose rows each hold >= 1 hit; position 0 of every row is shared."""
    w = W.config(1, scale=0.25)
    o = Oracle.for_workload(w).run("s1")
    R = w.n_rows
    rh = np.full((2, R), -1, np.int32)
    for r in rows_a:
        rh[0, r] = 0
    for r in rows_b:
        rh[1, r] = 0
    return w, o, o.select([0, 0], [n_a, n_b], [chi_a, chi_b], rh)


def test_s6_more_hits_wins_then_chi2_then_index():
    # B has more hits: it takes the 8 shared clusters, A keeps 12 (>= min_hits) of its own
    w, o, tr = _select_case(range(0, 20), range(12, 40), 20, 28, 10.0, 300.0)
    assert list(tr["tracklet"]) == [0, 1]
    assert list(tr["cl_row"][tr["cl_begin"][0]:tr["cl_begin"][1]]) == list(range(0, 12))
    assert list(tr["cl_row"][tr["cl_begin"][1]:tr["cl_begin"][2]]) == list(range(12, 40))
    # equal hits: lower chi2/ndf wins; the loser falls under min_hits and disappears
    w, o, tr = _select_case(range(0, 15), range(6, 21), 15, 15, 30.0, 20.0)
    assert list(tr["tracklet"]) == [1] and list(tr["cl_row"]) == list(range(6, 21))
    # full tie: lower tracklet index wins
    w, o, tr = _select_case(range(0, 15), range(6, 21), 15, 15, 20.0, 20.0)
    assert list(tr["tracklet"]) == [0] and list(tr["cl_row"]) == list(range(0, 15))
    # cluster indices are the caller's (original) indices
    perm = o.get("perm")
    assert list(tr["cl_index"]) == [int(perm[w.unit_off[r]]) for r in range(0, 15)]
    assert list(tr["ndf"]) == [25]


def test_s6_tracklets_below_min_hits_own_nothing():
    w, o, tr = _select_case(range(0, 9), range(0, 30), 9, 30, 1.0, 500.0)
    assert list(tr["tracklet"]) == [1] and len(tr["cl_row"]) == 30


def test_s6_no_shared_clusters_and_order_invariance():
    w = W.config(1)
    o = Oracle.for_workload(w).run("s6")
    tr, tl = o.tracks(), o.tracklets()
    R = w.n_rows
    g = w.unit_off[tr["sector"].repeat(np.diff(tr["cl_begin"])) * R + tr["cl_row"]] + tr["cl_index"]
    assert len(np.unique(g)) == len(g)                        # every cluster in at most one track
    assert np.all(np.diff(tr["cl_begin"]) >= 10)
    for i in range(len(tr["sector"])):                         # ascending row inside a track
        assert np.all(np.diff(tr["cl_row"][tr["cl_begin"][i]:tr["cl_begin"][i + 1]]) > 0)
    # feed the same tracklets in reversed order: same tracks.  Exact key ties do occur (two start hits of one physical
    # track converge to the same tracklet) and flip the winner's index, so cluster sets are compared, and the winner's
    # index wherever the key is unique.
    M = len(tl["n"])
    rev = np.arange(M)[::-1]
    o2 = Oracle.for_workload(w).run("s1")
    tr2 = o2.select(tl["sector"][rev], tl["n"][rev], tl["chi2"][rev], tl["rowhit"][rev])
    s1 = {tuple(tr["cl_index"][tr["cl_begin"][i]:tr["cl_begin"][i + 1]]): int(tr["tracklet"][i]) for i in range(len(tr["sector"]))}
    s2 = {tuple(tr2["cl_index"][tr2["cl_begin"][i]:tr2["cl_begin"][i + 1]]): int(M - 1 - tr2["tracklet"][i]) for i in range(len(tr2["sector"]))}
    assert set(s1) == set(s2)
    keys = list(zip(tl["n"].tolist(), (tl["chi2"].astype(np.float32) / (2 * tl["n"] - 5).astype(np.float32)).tolist()))
    unique_key = {i for i in range(M) if keys.count(keys[i]) == 1}
    assert all(s2[c] == t for c, t in s1.items() if t in unique_key)
    assert sum(1 for t in s1.values() if t in unique_key) > 0.8 * len(s1)


# ------------------------------------------------------------------ end to end versus generator truth
def test_end_to_end_efficiency_c1():
    w = W.config(1)
    m = H.truth_metrics(w, Oracle.for_workload(w).run("s6").tracks())
    assert m["findable"] > 100 and m["eff"] >= 0.98 and m["fake_rate"] <= 0.02, m
