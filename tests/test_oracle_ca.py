"""Pins of the oracle's CA seeding part (S0-S4) against what mathematics fixes.

Nothing here touches the CUDA path.  Each test is chosen so that a plausible oracle mistake (dropped term, wrong sign,
off-by-one row, transposed up/down) fails it.
"""
import math

import numpy as np
import pytest

from gen import workloads as W
from oracle.oracle import Oracle
from tests import helpers as H


@pytest.fixture(scope="module")
def c1():
    return W.config(1)


@pytest.fixture(scope="module")
def c1_small():
    return W.config(1, scale=0.1)     # 20 tracks + 100 noise: ~1.7 k clusters, brute force is instant


@pytest.fixture(scope="module")
def c3_small():
    return W.generate(W.Params(seed=3, t_frame=200.0, rate_per_us=0.05, mult_mean=40.0, mult_cap=120, sec_frac=0.2,
                               noise_frac=0.02), "C3-tiny")


# ------------------------------------------------------------------ S0
def test_s0_affine_closed_form(c1):
    o = Oracle.for_workload(c1).run("s0")
    z = o.get("z")
    # fp32: product rounded, then subtracted
    ref = (np.float32(c1.params.z_max) - np.float32(c1.params.vdrift) * c1.t).astype(np.float64)
    assert np.array_equal(z, ref)
    # round trip with the generator's t = (z_max - |z|)/vdrift: z in [0, z_max] up to smearing / fp32 rounding
    assert z.min() > -1.0 and z.max() < c1.params.z_max + 1.0
    od = Oracle.for_workload(c1, double=True).run("s0")
    assert np.allclose(od.get("z"), c1.params.z_max - c1.params.vdrift * c1.t.astype(np.float64), rtol=0, atol=1e-12)


def test_s0_continuous_negative_z(c3_small):
    o = Oracle.for_workload(c3_small).run("s0")
    z = o.get("z")
    assert z.min() < -50.0           # later collisions sit at negative scaled z (reading A6)
    assert z.min() >= -c3_small.params.vdrift * c3_small.params.t_frame - 1.0


# ------------------------------------------------------------------ S1
def _check_grid(w, o):
    R = w.n_rows
    ys, zs, perm = o.get("ys"), o.get("zs"), o.get("perm")
    z = o.get("z")
    bin_off, bin_start = o.get("bin_off"), o.get("bin_start")
    ny, nz = o.get("grid_ny"), o.get("grid_nz")
    ylo, zlo, invs = o.get("grid_ylo"), o.get("grid_zlo"), o.get("grid_invs")
    n_checked = 0
    for u in range(w.n_sectors * R):
        a, b = w.unit_off[u], w.unit_off[u + 1]
        n = b - a
        bs = bin_start[bin_off[u]:bin_off[u + 1]]
        assert len(bs) == ny[u] * nz[u] + 1
        assert bs[0] == 0 and bs[-1] == n and np.all(np.diff(bs) >= 0)
        if n == 0:
            continue
        p = perm[a:b]
        assert np.array_equal(np.sort(p), np.arange(n))                     # bijection
        assert np.array_equal(ys[a:b], w.y[a:b][p].astype(np.float64))      # payload follows the permutation
        assert np.array_equal(zs[a:b], z[a:b][p])
        # recomputed bin (fp32 arithmetic restated here) equals the bin the hit sits in
        fy = (w.y[a:b][p] - np.float32(ylo[u])) * np.float32(invs[u])
        fz = (z[a:b][p].astype(np.float32) - np.float32(zlo[u])) * np.float32(invs[u])
        by = np.clip(np.where(fy > 0, fy, 0).astype(np.int64), 0, ny[u] - 1)
        bz = np.clip(np.where(fz > 0, fz, 0).astype(np.int64), 0, nz[u] - 1)
        bins = bz * ny[u] + by
        pos_bin = np.searchsorted(bs, np.arange(n), side="right") - 1
        assert np.array_equal(bins, pos_bin)
        # inside a bin: ascending original index
        same = bins[1:] == bins[:-1]
        assert np.all(p[1:][same] > p[:-1][same])
        n_checked += n
    assert n_checked == w.n_clusters


def test_s1_grid_invariants_triggered(c1):
    _check_grid(c1, Oracle.for_workload(c1).run("s1"))


def test_s1_grid_invariants_continuous(c3_small):
    _check_grid(c3_small, Oracle.for_workload(c3_small).run("s1"))


def test_s1_nonfinite_and_out_of_range_inputs_are_binned_by_clamp():
    w = W.config(1, scale=0.05)
    y = w.y.copy(); t = w.t.copy()
    y[0] = np.nan; y[1] = np.inf; y[2] = -np.inf; t[3] = np.nan; y[4] = 1e9; t[5] = -1e9
    o = Oracle(**w.geometry()); o.load(w.unit_off, y, t); o.run("s4")
    bs, bo = o.get("bin_start"), o.get("bin_off")
    for u in range(w.n_sectors * w.n_rows):
        assert bs[bo[u + 1] - 1] == w.unit_off[u + 1] - w.unit_off[u]
    # non-finite hits are never linked (every comparison with NaN is false; inf is outside every window)
    up, dn, perm = o.get("link_up"), o.get("link_dn"), o.get("perm")
    a, b = w.unit_off[0], w.unit_off[1]
    bad = {0, 1, 2, 3, 4, 5}
    pos_of_bad = [i for i in range(b - a) if perm[a + i] in bad]
    assert all(up[a + i] == -1 and dn[a + i] == -1 for i in pos_of_bad)


# ------------------------------------------------------------------ S2
def _links_in_original_index(w, o, up_name="link_up", dn_name="link_dn"):
    """Link tables re-expressed with original cluster indices on both ends (independent of sorted order)."""
    R = w.n_rows
    perm, up, dn = o.get("perm"), o.get(up_name), o.get(dn_name)
    up_o = np.full(w.n_clusters, -1, np.int64); dn_o = np.full(w.n_clusters, -1, np.int64)
    for u in range(w.n_sectors * R):
        a, b = w.unit_off[u], w.unit_off[u + 1]
        if b == a:
            continue
        r = u % R
        pu, pd = up[a:b], dn[a:b]
        tgt = a + perm[a:b]
        if r + 1 < R:
            au = w.unit_off[u + 1]
            up_o[tgt] = np.where(pu >= 0, perm[au + np.maximum(pu, 0)] if w.unit_off[u + 2] > au else -1, -1)
        if r > 0:
            ad = w.unit_off[u - 1]
            dn_o[tgt] = np.where(pd >= 0, perm[ad + np.maximum(pd, 0)] if a > ad else -1, -1)
    return up_o, dn_o


def test_s2_grid_search_equals_brute_force(c1_small, c3_small):
    for w in (c1_small, c3_small.sector_slice([0, 1, 18])):
        assert w.n_clusters < 6000
        fast = Oracle.for_workload(w).run("s2")
        slow = Oracle.for_workload(w).run("s2", brute_links=True)
        assert np.array_equal(fast.get("link_up"), slow.get("link_up"))
        assert np.array_equal(fast.get("link_dn"), slow.get("link_dn"))
        assert (fast.get("link_up") >= 0).sum() > 0.5 * w.n_clusters * 0.5


def test_s2_python_brute_force_restatement(c1_small):
    """O(N^2) restatement of S2 in numpy fp32, written from DESIGN.md section 4 (not from the oracle's code)."""
    w = c1_small
    o = Oracle.for_workload(w).run("s2")
    up_o, dn_o = _links_in_original_index(w, o)
    f = np.float32
    X = H.row_x().astype(np.float64)
    z = (f(w.params.z_max) - f(w.params.vdrift) * w.t).astype(f)
    wy, wz, cut2 = f(1.5), f(1.5), 1.75
    R = w.n_rows
    n_links = 0
    for r in range(1, R - 1):
        a, b = w.unit_off[r], w.unit_off[r + 1]
        au, bu = w.unit_off[r + 1], w.unit_off[r + 2]
        ad, bd = w.unit_off[r - 1], w.unit_off[r]
        xr, xu, xd = float(f(X[r])), float(f(X[r + 1])), float(f(X[r - 1]))    # row_x is handed over as fp32
        tu, td, A, B = f(xu / xr), f(xd / xr), f(xu - xr), f(xr - xd)
        thr = f(cut2 * 0.5 * ((xu - xr) ** 2 + (xr - xd) ** 2))
        for h in range(a, b):
            y, zz = w.y[h], z[h]
            cu = [i for i in range(au, bu) if f(y * tu) - wy <= w.y[i] <= f(y * tu) + wy and f(zz * tu) - wz <= z[i] <= f(zz * tu) + wz]
            cd = [i for i in range(ad, bd) if f(y * td) - wy <= w.y[i] <= f(y * td) + wy and f(zz * td) - wz <= z[i] <= f(zz * td) + wz]
            best = None
            for i in cu:
                for j in cd:
                    ey = f(B * f(w.y[i] - y)) - f(A * f(y - w.y[j]))
                    ez = f(B * f(z[i] - zz)) - f(A * f(zz - z[j]))
                    D = f(f(ey * ey) + f(ez * ez))
                    key = (float(D), i - au, j - ad)
                    if best is None or key < best:
                        best = key
            if best is not None and f(best[0]) < thr:
                assert (up_o[h], dn_o[h]) == (best[1], best[2])
                n_links += 1
            else:
                assert (up_o[h], dn_o[h]) == (-1, -1)
    assert n_links > 500


def test_s2_continuous_mode_restatement_with_unequal_row_pitch():
    """O(N^2) numpy-fp32 restatement of S2 for t_frame > 0, the mode the benchmark runs (reading A6: window centre z, half-width
    wzu_r = dzdx_max * (x_{r+1} - x_r) + wz0 upwards and wzd_r = dzdx_max * (x_r - x_{r-1}) + wz0 downwards), written from DESIGN.md
    section 4 and not from the oracle's code.  The row pitch alternates 0.75 / 1.5 cm so that wzu != wzd on every row, the weights
    a_r != b_r enter the residual, and the tracks carry collision-time shifts (z down to -900 cm) and slopes dz/dx up to 1.9, so
    that true neighbours lie between the smaller and the larger half-width.
    Fails under: wzu / wzd swapped; window centre z * x'/x as in triggered mode; a and b swapped in ey / ez; thr from the wrong pitch."""
    f = np.float32
    rng = np.random.default_rng(77)
    R = 40
    pitch = np.where(np.arange(R - 1) % 2 == 0, 0.75, 1.5)
    X = (90.0 + np.concatenate([[0.0], np.cumsum(pitch)])).astype(np.float32)
    t_frame, vd, zmax = 400.0, 2.5, 250.0
    rows_y = [[] for _ in range(R)]; rows_z = [[] for _ in range(R)]
    n_tracks = 40
    for k in range(n_tracks):                       # straight lines from the beam line (Bz plays no role in S2), shifted in z
        tphi = rng.uniform(-0.15, 0.15); dzdx = rng.uniform(1.3, 1.9) * rng.choice([-1, 1]) if k % 2 else rng.uniform(-0.8, 0.8)
        zshift = -rng.uniform(0.0, 900.0)
        for r in range(R):
            if rng.uniform() < 0.05:
                continue
            rows_y[r].append(X[r] * tphi + rng.normal(0, 0.1)); rows_z[r].append(X[r] * dzdx * 0.1 + 60.0 + zshift + dzdx * (X[r] - X[0]) + rng.normal(0, 0.15))
    for r in range(R):                              # noise
        for _ in range(15):
            rows_y[r].append(rng.uniform(-15, 15)); rows_z[r].append(rng.uniform(-990.0, 240.0))
    off = np.zeros(R + 1, np.int64); off[1:] = np.cumsum([len(v) for v in rows_y])
    y = np.concatenate([np.array(v, np.float32) for v in rows_y]); zz = np.concatenate([np.array(v, np.float64) for v in rows_z])
    t = ((zmax - zz) / vd).astype(np.float32)
    geo = dict(n_sectors=1, n_rows=R, row_x=X, sector_dphi=2 * math.pi / 18, z_max=zmax, t_frame=t_frame, sigma_y=0.1, sigma_z=0.15, bz=0.5, vdrift=vd)
    o = Oracle(**geo); o.load(off, y, t); o.run("s2")

    class _W:                                        # the slice of the Workload interface _links_in_original_index reads
        n_sectors, n_rows, unit_off, n_clusters = 1, R, off, len(y)
    up_o, dn_o = _links_in_original_index(_W, o)
    z = (f(zmax) - f(vd) * t).astype(f)              # S0, fp32: product rounded, then subtracted
    wy, dzdx_max, wz0, cut2 = f(1.5), 1.5, 0.75, 1.75
    Xd = X.astype(np.float64)
    n_links = n_between = 0
    for r in range(1, R - 1):
        a, b = off[r], off[r + 1]; au, bu = off[r + 1], off[r + 2]; ad, bd = off[r - 1], off[r]
        A64, B64 = Xd[r + 1] - Xd[r], Xd[r] - Xd[r - 1]
        tu, td, A, B = f(Xd[r + 1] / Xd[r]), f(Xd[r - 1] / Xd[r]), f(A64), f(B64)
        thr = f(cut2 * 0.5 * (A64 * A64 + B64 * B64))
        wzu, wzd = f(dzdx_max * A64 + wz0), f(dzdx_max * B64 + wz0)
        assert wzu != wzd
        for h in range(a, b):
            yh, zh = y[h], z[h]
            ycu, ycd = f(yh * tu), f(yh * td)
            cu = [i for i in range(au, bu) if f(ycu - wy) <= y[i] <= f(ycu + wy) and f(zh - wzu) <= z[i] <= f(zh + wzu)]
            cd = [i for i in range(ad, bd) if f(ycd - wy) <= y[i] <= f(ycd + wy) and f(zh - wzd) <= z[i] <= f(zh + wzd)]
            best = None
            for i in cu:
                for j in cd:
                    ey = f(f(B * f(y[i] - yh)) - f(A * f(yh - y[j])))
                    ez = f(f(B * f(z[i] - zh)) - f(A * f(zh - z[j])))
                    D = f(f(ey * ey) + f(ez * ez))
                    key = (float(D), i - au, j - ad)
                    if best is None or key < best:
                        best = key
            if best is not None and f(best[0]) < thr:
                assert (up_o[h], dn_o[h]) == (best[1], best[2]), (r, h)
                n_links += 1
                lo, hi = min(wzu, wzd), max(wzu, wzd)
                n_between += lo < abs(z[au + best[1]] - zh) <= hi or lo < abs(z[ad + best[2]] - zh) <= hi
            else:
                assert (up_o[h], dn_o[h]) == (-1, -1), (r, h)
    assert n_links > 800 and n_between > 100          # the unequal half-widths decide links here


def test_s2_invariant_under_bin_size(c1):
    ref = Oracle.for_workload(c1).run("s4")
    r_up, r_dn = _links_in_original_index(c1, ref)
    rc_up, rc_dn = _links_in_original_index(c1, ref, "clean_up", "clean_dn")
    for scale in (0.37, 2.9):
        o = Oracle.for_workload(c1, grid_scale=scale).run("s4")
        assert not np.array_equal(o.get("grid_ny"), ref.get("grid_ny"))
        up, dn = _links_in_original_index(c1, o)
        assert np.array_equal(up, r_up) and np.array_equal(dn, r_dn)
        cu, cd = _links_in_original_index(c1, o, "clean_up", "clean_dn")
        assert np.array_equal(cu, rc_up) and np.array_equal(cd, rc_dn)
        assert len(o.get("start_unit")) == len(ref.get("start_unit"))


def test_s2_invariant_under_input_permutation(c1_small):
    """Relabelling the input inside each (sector,row) relabels the links and nothing else (no exact D ties in smeared data)."""
    w = c1_small
    rng = np.random.default_rng(5)
    y2, t2 = w.y.copy(), w.t.copy()
    new_of_old = np.arange(w.n_clusters)
    for u in range(w.n_sectors * w.n_rows):
        a, b = w.unit_off[u], w.unit_off[u + 1]
        p = rng.permutation(b - a)          # new position i holds old p[i]
        y2[a:b] = w.y[a:b][p]; t2[a:b] = w.t[a:b][p]
        new_of_old[a + p] = np.arange(b - a)
    o1 = Oracle.for_workload(w).run("s2")
    o2 = Oracle(**w.geometry()); o2.load(w.unit_off, y2, t2); o2.run("s2")
    up1, dn1 = _links_in_original_index(w, o1)
    up2, dn2 = _links_in_original_index(w, o2)
    for u in range(w.n_rows):
        a, b = w.unit_off[u], w.unit_off[u + 1]
        for h in range(a, b):
            h2 = a + new_of_old[h]
            e_up = -1 if up1[h] < 0 else new_of_old[w.unit_off[u + 1] + up1[h]]
            e_dn = -1 if dn1[h] < 0 else new_of_old[w.unit_off[u - 1] + dn1[h]]
            assert (up2[h2], dn2[h2]) == (e_up, e_dn)


def _straight_line_workload(n_tracks=12, bz=0.0, seed=11):
    p = W.Params(seed=seed, single_sector=1, mult_fixed=n_tracks, phi_lo=0.02, phi_hi=2 * math.pi / 18 - 0.02, bz=bz,
                 sigma_y=0.0, sigma_z=0.0, dropout=0.0, pt_lo=1.0, pt_hi=10.0)
    return W.generate(p, "lines")


def test_s2_straight_lines_from_origin_link_to_true_neighbours():
    w = _straight_line_workload()
    o = Oracle.for_workload(w, double=True).run("s4")
    up_o, dn_o = _links_in_original_index(w, o)
    R = w.n_rows
    n = 0
    for r in range(1, R - 1):
        a, b = w.unit_off[r], w.unit_off[r + 1]
        for h in range(a, b):
            lab = w.label[h]
            iu = [i for i in range(w.unit_off[r + 1], w.unit_off[r + 2]) if w.label[i] == lab]
            idn = [i for i in range(w.unit_off[r - 1], w.unit_off[r]) if w.label[i] == lab]
            if len(iu) == 1 and len(idn) == 1:
                assert up_o[h] == iu[0] - w.unit_off[r + 1] and dn_o[h] == idn[0] - w.unit_off[r - 1]
                n += 1
    assert n > 100 * 12
    # one chain per track and sector: start hits = number of tracks with >= min_seed+... rows
    assert len(o.get("start_unit")) == len(set(w.label.tolist()))
    assert np.all(o.get("start_unit") % R == 1)     # rows 0 and R-1 never search, so chains start on row 1


def test_s2_collinearity_residual_is_zero_on_exact_lines():
    """D = 0 for three collinear points: a link exists even with cut2 shrunk to (almost) nothing."""
    w = _straight_line_workload()
    o = Oracle.for_workload(w, double=True, cut2=1e-6).run("s2")
    up = o.get("link_up")
    a, b = w.unit_off[1], w.unit_off[w.n_rows - 1]
    assert (up[a:b] >= 0).mean() > 0.98


# ------------------------------------------------------------------ S3 / S4
def test_s3_mutual_links_and_idempotence(c1):
    o = Oracle.for_workload(c1).run("s4")
    R = c1.n_rows
    up, dn, cu, cd = o.get("link_up"), o.get("link_dn"), o.get("clean_up"), o.get("clean_dn")
    n_mut = 0
    for u in range(c1.n_sectors * R):
        a, b = c1.unit_off[u], c1.unit_off[u + 1]
        for h in range(b - a):
            x = cu[a + h]
            if x >= 0:
                assert up[a + h] == x and cd[c1.unit_off[u + 1] + x] == h     # up'[h]=u  =>  dn'[u]=h
                n_mut += 1
            elif up[a + h] >= 0:
                assert dn[c1.unit_off[u + 1] + up[a + h]] != h               # removed only if non-mutual
            x = cd[a + h]
            if x >= 0:
                assert dn[a + h] == x and cu[c1.unit_off[u - 1] + x] == h
            elif dn[a + h] >= 0:
                assert up[c1.unit_off[u - 1] + dn[a + h]] != h
    assert n_mut > 0.5 * c1.n_clusters
    assert (cu >= 0).sum() == (cd >= 0).sum()          # links pair up
    assert (cu >= 0).sum() < (up >= 0).sum()           # the cleaner removed something


def test_s4_start_hits_are_chain_heads_of_min_seed(c1):
    for min_seed in (3, 5):
        o = Oracle.for_workload(c1, min_seed=min_seed).run("s4")
        R = c1.n_rows
        cu, cd = o.get("clean_up"), o.get("clean_dn")
        su, sp = o.get("start_unit"), o.get("start_pos")
        # independent chain census: walk every chain from its head
        heads = []
        for u in range(c1.n_sectors * R):
            a, b = c1.unit_off[u], c1.unit_off[u + 1]
            for h in range(b - a):
                if cd[a + h] < 0 and cu[a + h] >= 0:
                    n, uu, p = 1, u, h
                    while cu[c1.unit_off[uu] + p] >= 0:
                        p = cu[c1.unit_off[uu] + p]; uu += 1; n += 1
                    if n >= min_seed:
                        heads.append((u, h))
        assert heads == list(zip(su.tolist(), sp.tolist()))
        keys = su.astype(np.int64) * (1 << 32) + sp
        assert np.all(np.diff(keys) > 0)               # strictly ascending (sector,row,sorted pos)
    assert len(heads) > 100
