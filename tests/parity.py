"""GPU-vs-oracle comparison helpers (used by tests/test_gpu_parity.py and __graft_entry__.smoke()).

The oracle gets exactly the values the C ABI carries (geometry scalars rounded to fp32), so that both sides start from
identical numbers; tunables are doubles on both sides.
"""
from __future__ import annotations

import numpy as np

from oracle.oracle import Oracle

F32_KEYS = ("sector_dphi", "z_max", "t_frame", "sigma_y", "sigma_z", "bz", "vdrift")


def abi_geometry(w) -> dict:
    """Workload geometry with every scalar rounded to fp32, as tpc_create receives it."""
    g = dict(w.geometry())
    for k in F32_KEYS:
        g[k] = float(np.float32(g[k]))
    return g


def make_oracle(w, **params) -> Oracle:
    o = Oracle(double=False, **abi_geometry(w), **params)
    o.load(w.unit_off, w.y, w.t)
    return o


def compare_grid(w, o, trk, units=None) -> int:
    """Bit-exact S0/S1 tables: grid descriptor, bin_start, perm, sorted (y,z).  Returns the number of units compared."""
    R = w.n_rows
    ys, zs, perm = o.get("ys"), o.get("zs"), o.get("perm")
    bin_off, bin_start = o.get("bin_off"), o.get("bin_start")
    ny, nz, ylo, zlo, invs = o.get("grid_ny"), o.get("grid_nz"), o.get("grid_ylo"), o.get("grid_zlo"), o.get("grid_invs")
    units = range(w.n_sectors * R) if units is None else units
    k = 0
    for u in units:
        g = trk.grid(u // R, u % R)
        a, b = int(w.unit_off[u]), int(w.unit_off[u + 1])
        assert g["n"] == b - a and g["ny"] == ny[u] and g["nz"] == nz[u], (u, g["n"], g["ny"], g["nz"])
        assert np.float32(ylo[u]) == g["y_lo"] and np.float32(zlo[u]) == g["z_lo"] and np.float32(invs[u]) == g["inv_s"], u
        assert np.array_equal(g["bin_start"], bin_start[bin_off[u]:bin_off[u + 1]]), u
        assert np.array_equal(g["perm"], perm[a:b]), u
        # equal_nan: NaN inputs of degenerate cases stay NaN on both sides (the payload bits of a NaN are not part of the result)
        assert np.array_equal(g["yz"][:, 0], ys[a:b].astype(np.float32), equal_nan=True), u
        assert np.array_equal(g["yz"][:, 1], zs[a:b].astype(np.float32), equal_nan=True), u
        k += 1
    return k


def gather_links(w, trk, cleaned, with_rows=False):
    up = np.full(w.n_clusters, -2, np.int32)
    dn = np.full(w.n_clusters, -2, np.int32)
    uk = np.full(w.n_clusters, -2, np.int32); dk = np.full(w.n_clusters, -2, np.int32)
    R = w.n_rows
    for u in range(w.n_sectors * R):
        a, b = int(w.unit_off[u]), int(w.unit_off[u + 1])
        if b > a:
            if with_rows:
                up[a:b], dn[a:b], uk[a:b], dk[a:b] = trk.link_rows(u // R, u % R, cleaned)
            else:
                up[a:b], dn[a:b] = trk.links(u // R, u % R, cleaned)
    return (up, dn, uk, dk) if with_rows else (up, dn)


def compare_links(w, o, trk) -> dict:
    """Raw (S2) and cleaned (S3) link tables and the S4 start list; returns the differing-hit counts (bar: 0)."""
    out = {}
    for cleaned, (nu, nd) in ((False, ("link_up", "link_dn")), (True, ("clean_up", "clean_dn"))):
        up, dn, uk, dk = gather_links(w, trk, cleaned, with_rows=True)
        diff = (up != o.get(nu)) | (dn != o.get(nd)) | (uk != o.get(nu + "_k")) | (dk != o.get(nd + "_k"))   # positions and row distances
        out["cleaned" if cleaned else "raw"] = int(diff.sum())
    su, sp = trk.start_hits()
    out["start_equal"] = bool(np.array_equal(su, o.get("start_unit")) and np.array_equal(sp, o.get("start_pos")))
    out["n_start"] = int(len(su))
    return out


def track_sets(tr) -> dict:
    """(sector, frozenset of (row, cluster index)) -> track index."""
    d = {}
    for i in range(len(tr["sector"])):
        a, b = int(tr["cl_begin"][i]), int(tr["cl_begin"][i + 1])
        key = (int(tr["sector"][i]), tuple(zip(tr["cl_row"][a:b].tolist(), tr["cl_index"][a:b].tolist())))
        d[key] = i
    return d


_DCOV = np.array([0, 2, 5, 9, 14])
_TRI = [(a, b) for a in range(5) for b in range(a + 1)]


def _cov_ratio(co, cg, rel=1e-4) -> float:
    """Largest |dC_ab| / (rel * sqrt(C_aa C_bb)) over the 15 lower-triangle entries (scale-aware: off-diagonals pass through 0)."""
    co = np.asarray(co, dtype=np.float64); cg = np.asarray(cg, dtype=np.float64)
    dg = np.sqrt(np.abs(co[_DCOV]))
    scale = np.array([dg[a] * dg[b] for a, b in _TRI])
    return float(np.max(np.abs(co - cg) / (rel * scale + 1e-300)))


def compare_tracks(otr, gtr, rel=1e-4, sig=1e-3) -> dict:
    """Reading A31/A19: pair tracks by (sector, exact cluster set); parameters within rel*|oracle| or sig*sqrt(C_ii); the 15
    covariance entries within rel * sqrt(C_aa C_bb); chi2 within 1e-3 relative; ndf and x equal.
    Also reports how many pairs are bit-identical in every number (parameters, covariance, chi2)."""
    so, sg = track_sets(otr), track_sets(gtr)
    common = [k for k in so if k in sg]
    n_bad = n_cov_bad = n_exact = 0
    worst = worst_cov = 0.0
    for k in common:
        i, j = so[k], sg[k]
        po, pg = otr["par"][i].astype(np.float64), np.asarray(gtr["par"][j], dtype=np.float64)
        so_ = np.sqrt(np.abs(otr["cov"][i][_DCOV].astype(np.float64)))
        d = np.abs(po - pg)
        ok = (d <= rel * np.abs(po)) | (d <= sig * so_)
        worst = max(worst, float(np.max(d / np.maximum(rel * np.abs(po), sig * so_ + 1e-300))))
        c2o, c2g = float(otr["chi2"][i]), float(gtr["chi2"][j])
        if not ok.all() or abs(c2o - c2g) > 1e-3 * max(1.0, abs(c2o)) or int(otr["ndf"][i]) != int(gtr["ndf"][j]) or \
                float(otr["x"][i]) != float(gtr["x"][j]):
            n_bad += 1
        rc = _cov_ratio(otr["cov"][i], gtr["cov"][j], rel)
        worst_cov = max(worst_cov, rc)
        n_cov_bad += rc > 1.0
        n_exact += bool(np.array_equal(otr["par"][i].astype(np.float32), np.asarray(gtr["par"][j], dtype=np.float32)) and
                        np.array_equal(otr["cov"][i].astype(np.float32), np.asarray(gtr["cov"][j], dtype=np.float32)) and
                        np.float32(c2o) == np.float32(c2g))
    return dict(n_oracle=len(so), n_gpu=len(sg), identical_sets=len(common), frac_identical=len(common) / max(1, len(so)),
                param_mismatch=n_bad, worst_ratio=worst, cov_mismatch=int(n_cov_bad), worst_cov_ratio=worst_cov, bit_identical=n_exact)


def compare_tracklets(o, tl) -> dict:
    """S5 output before selection, tracklet by tracklet (same index = same start hit): n, first, last and the rowhit table must be
    equal; chi2, the 5 parameters and the 15 covariance entries of tracklets with n >= 1 are compared bit for bit (both sides
    spell the same fp32 operation order)."""
    ot = o.tracklets()
    M = len(ot["n"])
    assert len(tl["n"]) == M, (len(tl["n"]), M)
    fitted = ot["first"] >= 0
    out = dict(n_tracklets=M)
    out["n_diff"] = int((ot["n"] != tl["n"]).sum())
    out["range_diff"] = int(((ot["first"] != tl["first"]) | (ot["last"] != tl["last"]))[fitted].sum())
    out["rowhit_diff"] = int((ot["rowhit"] != tl["rowhit"]).any(axis=1).sum())
    f32 = np.float32
    out["chi2_diff"] = int((ot["chi2"].astype(f32) != tl["chi2"].astype(f32))[fitted & np.isfinite(ot["chi2"])].sum())
    out["par_diff"] = int((ot["par"].astype(f32) != tl["par"].astype(f32)).any(axis=1)[fitted].sum())
    out["cov_diff"] = int((ot["cov"].astype(f32) != tl["cov"].astype(f32)).any(axis=1)[fitted].sum())
    return out


def compare_refit(otr, orf, gtr, grf, rel=1e-4, sig=1e-3) -> dict:
    """S7 (readings A37/A38): refit results of tracks paired by (sector, exact cluster set).  n, ndf, x equal; parameters as in
    compare_tracks; chi2 within 1e-3 relative; z0 / t0 within rel*|oracle| or sig * the z error (t0 = -z0 / vdrift)."""
    so, sg = track_sets(otr), track_sets(gtr)
    common = [k for k in so if k in sg]
    n_bad = 0
    dcov = _DCOV
    for k in common:
        i, j = so[k], sg[k]
        po, pg = orf["par"][i].astype(np.float64), np.asarray(grf["par"][j], dtype=np.float64)
        so_ = np.sqrt(np.abs(orf["cov"][i][dcov].astype(np.float64)))
        d = np.abs(po - pg)
        ok = bool(((d <= rel * np.abs(po)) | (d <= sig * so_)).all())
        ok &= int(orf["n"][i]) == int(grf["n"][j]) and int(orf["ndf"][i]) == int(grf["ndf"][j]) and float(orf["x"][i]) == float(grf["x"][j])
        ok &= abs(float(orf["chi2"][i]) - float(grf["chi2"][j])) <= 1e-3 * max(1.0, abs(float(orf["chi2"][i])))
        ok &= _cov_ratio(orf["cov"][i], grf["cov"][j], rel) <= 1.0
        for name in ("z0", "t0"):
            a, b = float(orf[name][i]), float(grf[name][j])
            ok &= abs(a - b) <= max(rel * abs(a), sig * so_[1] * 10.0)   # z0 adds (dz/ds error) x (arc ~ 1 m) to the z error
        n_bad += not ok
    return dict(n_common=len(common), mismatch=n_bad)
