"""ctypes binding of the CPU oracle (oracle/tpc_oracle.cpp).

TEST INFRASTRUCTURE ONLY: imported by tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
--impl reference legs.  The product (paper_1905_05515_b200) never imports this module.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "libtpc_oracle.so")
_SRC = os.path.join(_HERE, "tpc_oracle.cpp")
_KINDS = {0: (C.c_int32, np.int32), 1: (C.c_int64, np.int64), 2: (C.c_double, np.float64), 3: (C.c_float, np.float32)}

STAGES = {"s0": 0, "s1": 1, "s2": 2, "s3": 3, "s4": 4, "s5": 5, "s6": 6, "s7": 7, "s8": 8, "s9": 9, "s10": 10}


_SO_PLAIN = os.path.join(_HERE, "libtpc_oracle_plain.so")


def _flags():
    hw = []
    try:
        with open("/proc/cpuinfo") as f:
            if " fma " in f.read():
                hw = ["-mfma"]
    except OSError:
        pass
    return ["g++", "-O2", "-ffp-contract=off"] + hw + ["-std=c++17", "-shared", "-fPIC"]


def build(force: bool = False) -> str:
    """g++ -O2 -ffp-contract=off: a product is rounded before it is added unless the source says std::fma (reading A43 of DESIGN.md:
    the S5 transport / update).  -mfma, when the host has the instruction, only makes std::fma the hardware instruction instead of a
    libm call; the result is the correctly rounded one either way.
    Also builds the test-only second instance (-DS5_PLAIN_ORDER -> libtpc_oracle_plain.so): the S5 transport / update in the
    operation order of SURVEY.md section 8(c) as first written (own division per entry, no fused multiply-add)."""
    for so, extra in ((_SO, []), (_SO_PLAIN, ["-DS5_PLAIN_ORDER"])):
        if force or not os.path.exists(so) or os.path.getmtime(so) < os.path.getmtime(_SRC):
            subprocess.check_call(_flags() + extra + [_SRC, "-o", so])
    return _SO


def build_sanitized() -> str:
    """The oracle with -fsanitize=address,undefined as a stand-alone check of its own memory safety (tests/test_oracle_sanitize.py
    runs it in a subprocess with libasan preloaded)."""
    so = os.path.join(_HERE, "libtpc_oracle_asan.so")
    if not os.path.exists(so) or os.path.getmtime(so) < os.path.getmtime(_SRC):
        subprocess.check_call(_flags() + ["-g", "-fsanitize=address,undefined", "-fno-omit-frame-pointer", _SRC, "-o", so])
    return so


_libs = {}


def _load(which: str = "default"):
    if which not in _libs:
        build()
        path = {"default": _SO, "plain": _SO_PLAIN}.get(which, which)     # or an explicit path (sanitized build)
        lib = C.CDLL(path)
        lib.orc_create.restype = C.c_void_p
        lib.orc_create.argtypes = [C.c_int, C.c_int, C.c_int, C.POINTER(C.c_float)] + [C.c_double] * 7
        lib.orc_destroy.argtypes = [C.c_void_p]
        lib.orc_set_param.argtypes = [C.c_void_p, C.c_char_p, C.c_double]
        lib.orc_load.argtypes = [C.c_void_p, C.POINTER(C.c_int64), C.POINTER(C.c_float), C.POINTER(C.c_float)]
        lib.orc_run.argtypes = [C.c_void_p, C.c_int, C.c_int]
        lib.orc_run_range.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_int]
        lib.orc_get.argtypes = [C.c_void_p, C.c_char_p, C.POINTER(C.c_void_p), C.POINTER(C.c_int64), C.POINTER(C.c_int)]
        lib.orc_propagate.argtypes = [C.c_void_p, C.POINTER(C.c_double), C.POINTER(C.c_double), C.c_double]
        lib.orc_update.argtypes = [C.c_void_p, C.POINTER(C.c_double), C.POINTER(C.c_double), C.c_double, C.c_double,
                                   C.POINTER(C.c_double)]
        lib.orc_pickup.argtypes = [C.c_void_p, C.POINTER(C.c_double), C.POINTER(C.c_double), C.c_int, C.c_int, C.c_double, C.c_int]
        lib.orc_set_links.argtypes = [C.c_void_p, C.POINTER(C.c_int32), C.POINTER(C.c_int32)]
        lib.orc_set_tracklets.argtypes = [C.c_void_p, C.c_int64, C.POINTER(C.c_int32), C.POINTER(C.c_int32),
                                          C.POINTER(C.c_double), C.POINTER(C.c_int32)]
        assert lib.orc_plain_order() == (1 if which == "plain" else 0) or which not in ("default", "plain")
        _libs[which] = lib
    return _libs[which]


def _fp(a, ct):
    return a.ctypes.data_as(C.POINTER(ct))


class Oracle:
    """One oracle context.  `double=False` is the fp32 parity reference, `double=True` the fp64 pin instance."""

    def __init__(self, n_sectors, n_rows, row_x, sector_dphi, z_max, t_frame, sigma_y, sigma_z, bz, vdrift,
                 double=False, plain_order=False, lib=None, **params):
        # plain_order: the test-only build with the S5 arithmetic in SURVEY section 8(c)'s first operation order (no fma, own divisions)
        self.lib = _load(lib if lib else ("plain" if plain_order else "default"))
        self.n_sectors, self.n_rows = int(n_sectors), int(n_rows)
        self.row_x = np.ascontiguousarray(row_x, dtype=np.float32)
        self.h = self.lib.orc_create(int(double), self.n_sectors, self.n_rows, _fp(self.row_x, C.c_float),
                                     float(sector_dphi), float(z_max), float(t_frame), float(sigma_y), float(sigma_z),
                                     float(bz), float(vdrift))
        for k, v in params.items():
            self.set_param(k, v)

    @classmethod
    def for_workload(cls, w, double=False, **params):
        geo = w.geometry()
        for k in list(params):          # a geometry field given explicitly overrides the workload's (e.g. sigma_y for noise-free input)
            if k in geo:
                geo[k] = params.pop(k)
        o = cls(double=double, **geo, **params)
        o.load(w.unit_off, w.y, w.t)
        return o

    def __del__(self):
        if getattr(self, "h", None):
            self.lib.orc_destroy(self.h)
            self.h = None

    def set_param(self, name, value):
        if self.lib.orc_set_param(self.h, name.encode(), float(value)) != 0:
            raise KeyError(name)

    def load(self, unit_off, y, t):
        self.unit_off = np.ascontiguousarray(unit_off, dtype=np.int64)
        y = np.ascontiguousarray(y, dtype=np.float32)
        t = np.ascontiguousarray(t, dtype=np.float32)
        assert self.unit_off.shape[0] == self.n_sectors * self.n_rows + 1 and y.shape[0] == self.unit_off[-1] == t.shape[0]
        self.lib.orc_load(self.h, _fp(self.unit_off, C.c_int64), _fp(y, C.c_float), _fp(t, C.c_float))

    def run(self, upto="s6", brute_links=False, brute_pickup=False):
        self.lib.orc_run(self.h, STAGES[upto], int(brute_links) | (int(brute_pickup) << 1))
        return self

    def run_range(self, first, upto, brute_links=False, brute_pickup=False):
        """Stages first..upto only (earlier ones have run or were set by hand: set_links)."""
        self.lib.orc_run_range(self.h, STAGES[first], STAGES[upto], int(brute_links) | (int(brute_pickup) << 1))
        return self

    def set_links(self, up, dn):
        """Hand-set cleaned link tables (sorted positions in rows r+1 / r-1, -1 none), for hand-built S4 / S5 cases."""
        up = np.ascontiguousarray(up, dtype=np.int32); dn = np.ascontiguousarray(dn, dtype=np.int32)
        assert up.shape[0] == dn.shape[0] == self.unit_off[-1]
        self.lib.orc_set_links(self.h, _fp(up, C.c_int32), _fp(dn, C.c_int32))

    def pickup(self, par, cov, sector, row, zref=0.0, brute=False):
        """S5 pick-up alone: sorted position of the cluster picked on (sector,row) for the state (par, cov), -1 none (S1 must have run)."""
        par = np.array(par, dtype=np.float64); cov = np.array(cov, dtype=np.float64)
        return int(self.lib.orc_pickup(self.h, _fp(par, C.c_double), _fp(cov, C.c_double), int(sector), int(row), float(zref), int(brute)))

    def get(self, name):
        p, n, k = C.c_void_p(), C.c_int64(), C.c_int()
        if self.lib.orc_get(self.h, name.encode(), C.byref(p), C.byref(n), C.byref(k)) != 0:
            raise KeyError(name)
        ct, dt = _KINDS[k.value]
        if n.value == 0:
            return np.zeros(0, dtype=dt)
        return np.ctypeslib.as_array(C.cast(p, C.POINTER(ct)), shape=(n.value,)).copy()

    # ---- single-step entry points for the closed-form pins ----
    def propagate(self, par, cov, dx):
        par = np.array(par, dtype=np.float64); cov = np.array(cov, dtype=np.float64)
        rc = self.lib.orc_propagate(self.h, _fp(par, C.c_double), _fp(cov, C.c_double), float(dx))
        return rc == 0, par, cov

    def update(self, par, cov, ym, zm):
        par = np.array(par, dtype=np.float64); cov = np.array(cov, dtype=np.float64); chi2 = C.c_double()
        self.lib.orc_update(self.h, _fp(par, C.c_double), _fp(cov, C.c_double), float(ym), float(zm), C.byref(chi2))
        return par, cov, chi2.value

    def select(self, sector, n_hits, chi2, rowhit):
        """S6 alone on hand-built tracklets (S1 must have run)."""
        sector = np.ascontiguousarray(sector, dtype=np.int32); n_hits = np.ascontiguousarray(n_hits, dtype=np.int32)
        chi2 = np.ascontiguousarray(chi2, dtype=np.float64); rowhit = np.ascontiguousarray(rowhit, dtype=np.int32)
        assert rowhit.shape == (sector.shape[0], self.n_rows)
        self.lib.orc_set_tracklets(self.h, sector.shape[0], _fp(sector, C.c_int32), _fp(n_hits, C.c_int32),
                                   _fp(chi2, C.c_double), _fp(rowhit, C.c_int32))
        return self.tracks()

    def tracks(self):
        d = {k: self.get("trk_" + k) for k in ("sector", "ndf", "tracklet", "cl_begin", "cl_row", "cl_index", "x", "par",
                                                "cov", "chi2")}
        d["par"] = d["par"].reshape(-1, 5); d["cov"] = d["cov"].reshape(-1, 15)
        return d

    def refit(self):
        """S7 (NEXT-1): refitted state of every S6 track over its owned clusters + collision-time estimate (run("s7") first)."""
        d = {k: self.get("rf_" + k) for k in ("n", "ndf", "x", "par", "cov", "chi2", "z0", "t0")}
        d["par"] = d["par"].reshape(-1, 5); d["cov"] = d["cov"].reshape(-1, 15)
        return d

    def cluster_status(self):
        """S8 (NEXT-4): (status, track) per cluster in the caller's order; status 0 none / 1 attached / 2 adjacent (run("s8") first)."""
        return self.get("cl_status"), self.get("cl_track")

    def merges(self):
        """S9 (NEXT-3): next / prev segment of every track across a sector boundary (-1 none), leaver flag, outer state (run("s9") first)."""
        return {"next": self.get("mg_next"), "prev": self.get("mg_prev"), "leaver": self.get("mg_leaver"),
                "outer": self.get("mg_outer").reshape(-1, 4)}

    def loopers(self):
        """S10 (NEXT-3, second half): per track the previous turn of the same looping particle (-1 none), the first turn of its group
        (itself if it follows nobody) and the number of turns after it (run("s10") first)."""
        return {"prev": self.get("lp_prev"), "root": self.get("lp_root"), "turn": self.get("lp_turn")}

    def tracklets(self):
        d = {k: self.get("tl_" + k) for k in ("n", "first", "last", "rowhit", "sector", "chi2", "x", "par", "cov", "zref")}
        d["par"] = d["par"].reshape(-1, 5); d["cov"] = d["cov"].reshape(-1, 15); d["rowhit"] = d["rowhit"].reshape(-1, self.n_rows)
        return d
