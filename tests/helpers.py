"""Test helpers: closed-form helix truth and truth matching.  Independent of oracle/ and of the CUDA path."""
from __future__ import annotations

import math

import numpy as np

CB_PER_TESLA = -0.00299792458   # 1/cm per (c/GeV) per Tesla ("curvature constant")


def row_x(n_rows=152, x_first=85.0, x_last=246.0):
    return np.array([x_first + r * (x_last - x_first) / (n_rows - 1) for r in range(n_rows)], dtype=np.float64)


def helix_truth_at(x, pt, charge, phi_local, tanl_drift, bz, vx=0.0, vy=0.0, vz=0.0):
    """Closed-form circle through (vx,vy) with local azimuth phi_local: state (y, z, sinphi, dz/ds, q/pT) at local x.

    sinphi(x) = sinphi0 + k (x - vx);  y = vy + (cosphi0 - cosphi1)/k;  z = vz + tanl * (phi1 - phi0)/k.
    """
    k = CB_PER_TESLA * bz * charge / pt
    s0, c0 = math.sin(phi_local), math.cos(phi_local)
    s1 = s0 + k * (x - vx)
    c1 = math.sqrt(1.0 - s1 * s1)
    if abs(k) > 0:
        y = vy + (c0 - c1) / k
        path = (math.asin(s1) - phi_local) / k
    else:
        y = vy + (x - vx) * s0 / c0
        path = (x - vx) / c0
    return np.array([y, vz + tanl_drift * path, s1, tanl_drift, charge / pt])


def wrap_pi(a):
    while a > math.pi:
        a -= 2 * math.pi
    while a <= -math.pi:
        a += 2 * math.pi
    return a


def sector_alpha(sector):
    return ((sector % 18) + 0.5) * (2 * math.pi / 18)


def track_labels(w, tracks):
    """Per track: (majority label, fraction of clusters carrying it)."""
    R = w.n_rows
    out = []
    for i in range(len(tracks["sector"])):
        a, b = tracks["cl_begin"][i], tracks["cl_begin"][i + 1]
        g = w.unit_off[tracks["sector"][i] * R + tracks["cl_row"][a:b]] + tracks["cl_index"][a:b]
        vals, cnt = np.unique(w.label[g], return_counts=True)
        j = cnt.argmax()
        out.append((int(vals[j]), cnt[j] / float(b - a)))
    return out


def truth_metrics(w, tracks, min_findable=30, purity=0.9):
    """Reading A26: matched iff >= 90 % of the clusters carry one label; findable = >= 30 leg-0 clusters in one sector."""
    labs = track_labels(w, tracks)
    matched = {}
    fakes = 0
    for i, (lab, frac) in enumerate(labs):
        if lab >= 0 and frac >= purity:
            matched.setdefault((lab, int(tracks["sector"][i])), []).append(i)
        else:
            fakes += 1
    P = w.particles
    findable = np.where(P["best_count"] >= min_findable)[0]
    found = sum(1 for p in findable if (int(p), int(P["best_sector"][p])) in matched)
    prim = [p for p in findable if P["kind"][p] == 0]
    found_prim = sum(1 for p in prim if (int(p), int(P["best_sector"][p])) in matched)
    clones = sum(len(v) - 1 for v in matched.values())
    n = len(labs)
    return dict(n_tracks=n, findable=len(findable), found=found, eff=found / max(1, len(findable)),
                eff_primary=found_prim / max(1, len(prim)), fakes=fakes, fake_rate=fakes / max(1, n), clones=clones,
                matched=matched)
