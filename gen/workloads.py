"""Seeded synthetic TPC workloads (inputs only; no track-finding arithmetic lives here).

Thin ctypes wrapper around gen/tpcgen.c plus the five presets that stand in for
BASELINE.json:configs[0..4] (readings A20-A25).  Both the oracle tests and the
CUDA library's tests / bench take their input bytes from here.
"""
from __future__ import annotations

import ctypes as C
import math
import os
import subprocess
from dataclasses import dataclass, field

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "libtpcgen.so")
_SRC = os.path.join(_HERE, "tpcgen.c")


def build(force: bool = False) -> str:
    """Compile gen/tpcgen.c -> gen/libtpcgen.so (gcc, OpenMP)."""
    if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < os.path.getmtime(_SRC):
        subprocess.check_call(["gcc", "-O2", "-fopenmp", "-shared", "-fPIC", "-w", _SRC, "-o", _SO, "-lm"])
    return _SO


class _Params(C.Structure):
    _fields_ = [
        ("seed", C.c_uint64), ("n_rows", C.c_int32), ("single_sector", C.c_int32),
        ("x_first", C.c_double), ("x_last", C.c_double), ("bz", C.c_double), ("vdrift", C.c_double),
        ("z_max", C.c_double), ("t_frame", C.c_double), ("sigma_y", C.c_double), ("sigma_z", C.c_double),
        ("dropout", C.c_double), ("rate_per_us", C.c_double), ("mult_fixed", C.c_int32),
        ("mult_mean", C.c_double), ("mult_cap", C.c_int32), ("pt_lo", C.c_double), ("pt_hi", C.c_double),
        ("eta_max", C.c_double), ("phi_lo", C.c_double), ("phi_hi", C.c_double), ("sec_frac", C.c_double),
        ("sec_rmax", C.c_double), ("n_loopers", C.c_int32), ("loop_pt_lo", C.c_double),
        ("loop_pt_hi", C.c_double), ("loop_turns", C.c_int32), ("noise_per_sector", C.c_int32),
        ("noise_frac", C.c_double),
    ]


_PF, _PI, _PD, _PL, _PB = (C.POINTER(C.c_float), C.POINTER(C.c_int32), C.POINTER(C.c_double),
                           C.POINTER(C.c_int64), C.POINTER(C.c_uint8))


class _Out(C.Structure):
    _fields_ = [
        ("n_sectors", C.c_int32), ("n_rows", C.c_int32), ("n_clusters", C.c_int64),
        ("n_particles", C.c_int32), ("n_collisions", C.c_int32),
        ("row_x", _PF), ("unit_off", _PL), ("y", _PF), ("t", _PF), ("q", _PF), ("label", _PI), ("leg0", _PB),
        ("p_collision", _PI), ("p_kind", _PI), ("p_charge", _PI),
        ("p_pt", _PD), ("p_tanl", _PD), ("p_phi", _PD), ("p_t0", _PD), ("p_vx", _PD), ("p_vy", _PD), ("p_vz", _PD),
        ("p_n_clusters", _PI), ("p_best_sector", _PI), ("p_best_count", _PI),
        ("coll_t0", _PD), ("coll_mult", _PI),
    ]


@dataclass
class Params:
    """Generator knobs; defaults are the common part of configs 1-5."""
    seed: int = 1
    n_rows: int = 152
    single_sector: int = 0
    x_first: float = 85.0
    x_last: float = 246.0
    bz: float = 0.5
    vdrift: float = 2.58
    z_max: float = 250.0
    t_frame: float = 0.0
    sigma_y: float = 0.1
    sigma_z: float = 0.15
    dropout: float = 0.05
    rate_per_us: float = 0.0
    mult_fixed: int = 0
    mult_mean: float = 800.0
    mult_cap: int = 5000
    pt_lo: float = 0.1
    pt_hi: float = 10.0
    eta_max: float = 0.9
    phi_lo: float = 0.0
    phi_hi: float = 2 * math.pi
    sec_frac: float = 0.0
    sec_rmax: float = 60.0
    n_loopers: int = 0
    loop_pt_lo: float = 0.05
    loop_pt_hi: float = 0.15
    loop_turns: int = 10
    noise_per_sector: int = 0
    noise_frac: float = 0.0


@dataclass
class Workload:
    """Clusters in CSR order of unit = sector*n_rows+row, plus generator truth."""
    name: str
    params: Params
    n_sectors: int
    n_rows: int
    row_x: np.ndarray          # float32 [n_rows]
    unit_off: np.ndarray       # int64 [n_sectors*n_rows+1]
    y: np.ndarray              # float32 [N] pad-y
    t: np.ndarray              # float32 [N] time (us)
    q: np.ndarray              # float32 [N] charge
    label: np.ndarray          # int32 [N] particle id, -1 noise
    leg0: np.ndarray           # uint8 [N]
    particles: dict = field(default_factory=dict)
    coll_t0: np.ndarray = None
    coll_mult: np.ndarray = None

    @property
    def n_clusters(self) -> int:
        return int(self.y.shape[0])

    @property
    def n_collisions(self) -> int:
        return int(self.coll_t0.shape[0])

    def geometry(self) -> dict:
        p = self.params
        return dict(n_sectors=self.n_sectors, n_rows=self.n_rows, row_x=self.row_x,
                    sector_dphi=float(np.float32(2 * math.pi / 18)), z_max=p.z_max, t_frame=p.t_frame,
                    sigma_y=p.sigma_y, sigma_z=p.sigma_z, bz=p.bz, vdrift=p.vdrift)

    def sector_slice(self, sectors) -> "Workload":
        """Same workload with only the given sectors populated (sectors are independent units)."""
        sectors = sorted(set(int(s) for s in sectors))
        R = self.n_rows
        keep = np.zeros(self.n_clusters, dtype=bool)
        cnt = np.zeros(self.n_sectors * R, dtype=np.int64)
        for s in sectors:
            a, b = self.unit_off[s * R], self.unit_off[(s + 1) * R]
            keep[a:b] = True
            cnt[s * R:(s + 1) * R] = np.diff(self.unit_off[s * R:(s + 1) * R + 1])
        off = np.zeros(self.n_sectors * R + 1, dtype=np.int64)
        np.cumsum(cnt, out=off[1:])
        return Workload(self.name + "/sectors" + ",".join(map(str, sectors)), self.params, self.n_sectors, R,
                        self.row_x, off, self.y[keep].copy(), self.t[keep].copy(), self.q[keep].copy(),
                        self.label[keep].copy(), self.leg0[keep].copy(), self.particles, self.coll_t0, self.coll_mult)


def _arr(ptr, n, dtype):
    if n == 0:
        return np.zeros(0, dtype=dtype)
    return np.ctypeslib.as_array(ptr, shape=(n,)).astype(dtype, copy=True)


def generate(params: Params, name: str = "custom") -> Workload:
    lib = C.CDLL(build())
    lib.tpcgen_generate.argtypes = [C.POINTER(_Params), C.POINTER(_Out)]
    lib.tpcgen_generate.restype = C.c_int
    lib.tpcgen_free.argtypes = [C.POINTER(_Out)]
    lib.tpcgen_free.restype = None
    cp = _Params(**{k: getattr(params, k) for k, _ in _Params._fields_})
    out = _Out()
    rc = lib.tpcgen_generate(C.byref(cp), C.byref(out))
    if rc != 0:
        raise RuntimeError(f"tpcgen_generate failed: {rc}")
    try:
        n, npart, nc = out.n_clusters, out.n_particles, out.n_collisions
        U = out.n_sectors * out.n_rows
        parts = {k[2:]: _arr(getattr(out, k), npart, dt) for k, dt in [
            ("p_collision", np.int32), ("p_kind", np.int32), ("p_charge", np.int32), ("p_pt", np.float64),
            ("p_tanl", np.float64), ("p_phi", np.float64), ("p_t0", np.float64), ("p_vx", np.float64),
            ("p_vy", np.float64), ("p_vz", np.float64), ("p_n_clusters", np.int32),
            ("p_best_sector", np.int32), ("p_best_count", np.int32)]}
        return Workload(name, params, out.n_sectors, out.n_rows, _arr(out.row_x, out.n_rows, np.float32),
                        _arr(out.unit_off, U + 1, np.int64), _arr(out.y, n, np.float32), _arr(out.t, n, np.float32),
                        _arr(out.q, n, np.float32), _arr(out.label, n, np.int32), _arr(out.leg0, n, np.uint8),
                        parts, _arr(out.coll_t0, nc, np.float64), _arr(out.coll_mult, nc, np.int32))
    finally:
        lib.tpcgen_free(C.byref(out))


def config_params(k: int, seed: int | None = None, scale: float = 1.0) -> Params:
    """Presets C1..C5 (BASELINE.json:configs[k-1]).  `scale` shrinks multiplicities / frame length for tests."""
    seed = k if seed is None else seed
    if k == 1:   # one sector, 200 primaries within the sector, 1000 noise clusters
        return Params(seed=seed, single_sector=1, mult_fixed=max(1, int(round(200 * scale))),
                      phi_lo=0.0, phi_hi=2 * math.pi / 18, noise_per_sector=int(round(1000 * scale)))
    if k == 2:   # one central Pb-Pb-like event, 36 sectors
        return Params(seed=seed, mult_fixed=max(1, int(round(5000 * scale))), sec_frac=0.2, noise_frac=0.02)
    if k == 3:   # 2 ms continuous time frame at 50 kHz
        return Params(seed=seed, t_frame=2000.0 * scale, rate_per_us=0.05, mult_mean=800.0, mult_cap=5000,
                      sec_frac=0.2, noise_frac=0.02)
    if k == 4:   # looper stress
        return Params(seed=seed, mult_fixed=max(1, int(round(1500 * scale))), pt_lo=0.15, pt_hi=10.0,
                      n_loopers=int(round(1500 * scale)), noise_per_sector=int(round(1000 * scale)))
    if k == 5:   # 10 ms continuous time frame
        return Params(seed=seed, t_frame=10000.0 * scale, rate_per_us=0.05, mult_mean=800.0, mult_cap=5000,
                      sec_frac=0.2, noise_frac=0.02)
    raise ValueError("config must be 1..5")


def config(k: int, seed: int | None = None, scale: float = 1.0) -> Workload:
    return generate(config_params(k, seed, scale), name=f"C{k}" + ("" if scale == 1.0 else f"@{scale:g}"))
