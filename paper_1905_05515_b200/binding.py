"""ctypes binding of include/tpc.h.  Same names as the C ABI; argument marshalling only.

PyTorch is used for device memory and streams: torch tensors (CUDA or CPU) and numpy arrays are accepted as cluster arrays,
and device results are wrapped as torch tensors without a copy.  The library is loaded from the in-tree
paper_1905_05515_b200/libtpc_b200.so; a missing library or a missing CUDA device raises (there is no CPU fallback).
"""
from __future__ import annotations

import ctypes as C
import os
from dataclasses import dataclass

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
# TPC_B200_LIB selects another build of the same library (tests/test_gpu_checked.py: the bounds-checked build); default: the product
_SO = os.environ.get("TPC_B200_LIB") or os.path.join(_HERE, "libtpc_b200.so")

ABI_SYMBOLS = [
    "tpc_abi_version", "tpc_checked_build", "tpc_create", "tpc_set_param", "tpc_set_stream", "tpc_load_clusters", "tpc_load_clusters_batch",
    "tpc_find_tracks", "tpc_find_tracks_device", "tpc_refit_tracks", "tpc_mark_clusters", "tpc_merge_tracks", "tpc_find_loopers", "tpc_find_loopers_noalloc", "tpc_clear", "tpc_destroy", "tpc_last_error", "tpc_get_timings", "tpc_measure_fp32_peak",
    "tpc_debug_get_grid", "tpc_debug_get_links", "tpc_debug_get_link_rows", "tpc_debug_get_start_hits", "tpc_debug_get_tracklets",
]

_PF, _PI, _PL = C.POINTER(C.c_float), C.POINTER(C.c_int32), C.POINTER(C.c_int64)


class TpcError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"tpc error {code}: {msg}")
        self.code = code


class _Geometry(C.Structure):
    _fields_ = [("n_sectors", C.c_int32), ("n_rows", C.c_int32), ("row_x", _PF), ("sector_dphi", C.c_float),
                ("z_max", C.c_float), ("t_frame", C.c_float), ("sigma_y", C.c_float), ("sigma_z", C.c_float)]


class _Tracks(C.Structure):
    _fields_ = [("n_tracks", C.c_int64), ("n_cluster_refs", C.c_int64), ("sector", C.c_void_p), ("x", C.c_void_p),
                ("par", C.c_void_p), ("cov", C.c_void_p), ("chi2", C.c_void_p), ("ndf", C.c_void_p), ("tracklet", C.c_void_p),
                ("cl_begin", C.c_void_p), ("cl_row", C.c_void_p), ("cl_index", C.c_void_p)]


class _Refit(C.Structure):
    _fields_ = [("n_tracks", C.c_int64)] + [(k, C.c_void_p) for k in ("n", "ndf", "x", "par", "cov", "chi2", "z0", "t0")] + \
               [("ms_refit", C.c_float)]


class _Marks(C.Structure):
    _fields_ = [("n_clusters", C.c_int64), ("status", C.c_void_p), ("track", C.c_void_p), ("ms_mark", C.c_float)]


class _Merges(C.Structure):
    _fields_ = [("n_tracks", C.c_int64), ("next", C.c_void_p), ("prev", C.c_void_p), ("ms_merge", C.c_float)]


class _Loopers(C.Structure):
    _fields_ = [("n_tracks", C.c_int64), ("prev", C.c_void_p), ("root", C.c_void_p), ("turn", C.c_void_p), ("ms_loopers", C.c_float)]


class _Timings(C.Structure):
    _fields_ = [(k, C.c_float) for k in ("ms_upload", "ms_grid", "ms_neighbours", "ms_clean_start", "ms_tracklets",
                                         "ms_selector", "ms_download", "ms_total")] + \
               [(k, C.c_int64) for k in ("n_clusters", "n_bins", "n_start_hits", "n_tracklets_kept", "n_tracks",
                                         "n_cluster_refs", "launches", "n_propagations", "n_updates", "n_pickups")]


class _GridView(C.Structure):
    _fields_ = [("n", C.c_int32), ("ny", C.c_int32), ("nz", C.c_int32), ("y_lo", C.c_float), ("z_lo", C.c_float),
                ("inv_s", C.c_float), ("yz", _PF), ("perm", _PI), ("bin_start", _PI)]


class _TrackletView(C.Structure):
    _fields_ = [("n_tracklets", C.c_int64), ("sector", _PI), ("start_row", _PI), ("n_hits", _PI), ("first_row", _PI),
                ("last_row", _PI), ("chi2", _PF), ("x", _PF), ("par", _PF), ("cov", _PF), ("rowhit", _PI)]


_lib = None


def lib_path() -> str:
    return _SO


def load_library():
    """Load libtpc_b200.so (raises if it has not been built: `python -m paper_1905_05515_b200.build`)."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(_SO):
        raise TpcError(-4, f"{_SO} is missing: build it with `python -m paper_1905_05515_b200.build` (no CPU fallback exists)")
    try:
        import torch  # noqa: F401  -- loads libcudart.so.12 that the library links against
    except Exception:
        pass
    lib = C.CDLL(_SO)
    vp = C.c_void_p
    lib.tpc_abi_version.restype = C.c_int
    lib.tpc_checked_build.restype = C.c_int
    lib.tpc_create.argtypes = [C.POINTER(_Geometry), C.c_float, C.c_float, C.POINTER(vp)]
    lib.tpc_set_param.argtypes = [vp, C.c_char_p, C.c_double]
    lib.tpc_set_stream.argtypes = [vp, vp]
    lib.tpc_load_clusters.argtypes = [vp, C.c_int, C.c_int, vp, vp, vp, C.c_int]
    lib.tpc_load_clusters_batch.argtypes = [vp, _PL, vp, vp, vp]
    lib.tpc_find_tracks.argtypes = [vp, C.POINTER(_Tracks)]
    lib.tpc_find_tracks_device.argtypes = [vp, C.POINTER(_Tracks)]
    lib.tpc_refit_tracks.argtypes = [vp, C.c_int, C.POINTER(_Refit)]
    lib.tpc_mark_clusters.argtypes = [vp, C.c_float, C.c_int, C.POINTER(_Marks)]
    lib.tpc_merge_tracks.argtypes = [vp, C.c_int, C.POINTER(_Merges)]
    lib.tpc_find_loopers.argtypes = [vp, C.c_int, C.POINTER(_Loopers)]
    lib.tpc_find_loopers_noalloc.argtypes = [vp, C.c_int64] + [C.c_void_p] * 6
    lib.tpc_clear.argtypes = [vp]
    lib.tpc_destroy.argtypes = [vp]
    lib.tpc_destroy.restype = None
    lib.tpc_last_error.argtypes = [vp]
    lib.tpc_last_error.restype = C.c_char_p
    lib.tpc_get_timings.argtypes = [vp, C.POINTER(_Timings)]
    lib.tpc_measure_fp32_peak.argtypes = [vp, C.POINTER(C.c_float)]
    lib.tpc_debug_get_grid.argtypes = [vp, C.c_int, C.c_int, C.POINTER(_GridView)]
    lib.tpc_debug_get_links.argtypes = [vp, C.c_int, C.c_int, C.c_int, C.POINTER(_PI), C.POINTER(_PI), C.POINTER(C.c_int32)]
    lib.tpc_debug_get_link_rows.argtypes = [vp, C.POINTER(C.POINTER(C.c_int8)), C.POINTER(C.POINTER(C.c_int8)), C.POINTER(C.c_int32)]
    lib.tpc_debug_get_start_hits.argtypes = [vp, C.POINTER(_PI), C.POINTER(_PI), C.POINTER(C.c_int64)]
    lib.tpc_debug_get_tracklets.argtypes = [vp, C.POINTER(_TrackletView)]
    _lib = lib
    return lib


def abi_symbols() -> list[str]:
    return list(ABI_SYMBOLS)


def _check(h, rc):
    if rc != 0:
        raise TpcError(rc, (load_library().tpc_last_error(h) or b"").decode())


def _ptr(a):
    """Raw address of a numpy array / torch tensor (float32, contiguous) or None; returns (address, keepalive)."""
    if a is None:
        return None, None
    if isinstance(a, np.ndarray):
        a = np.ascontiguousarray(a, dtype=np.float32)
        return a.ctypes.data, a
    import torch
    if isinstance(a, torch.Tensor):
        if a.dtype != torch.float32 or not a.is_contiguous():
            a = a.to(torch.float32).contiguous()
        return a.data_ptr(), a
    a = np.ascontiguousarray(a, dtype=np.float32)
    return a.ctypes.data, a


# ---- functions with the names of the C ABI ----------------------------------------------------------------------------
def tpc_create(n_sectors, n_rows, row_x, sector_dphi, z_max, t_frame, sigma_y, sigma_z, bz, vdrift):
    lib = load_library()
    rx = np.ascontiguousarray(row_x, dtype=np.float32)
    g = _Geometry(int(n_sectors), int(n_rows), rx.ctypes.data_as(_PF), float(sector_dphi), float(z_max), float(t_frame),
                  float(sigma_y), float(sigma_z))
    h = C.c_void_p()
    _check(None, lib.tpc_create(C.byref(g), float(bz), float(vdrift), C.byref(h)))
    return h


def tpc_set_param(h, name, value):
    _check(h, load_library().tpc_set_param(h, name.encode(), float(value)))


def tpc_set_stream(h, cuda_stream):
    _check(h, load_library().tpc_set_stream(h, C.c_void_p(int(cuda_stream) if cuda_stream else 0)))


def tpc_load_clusters(h, sector, row, pad_y, time, charge=None):
    py, k1 = _ptr(pad_y); pt, k2 = _ptr(time); pq, k3 = _ptr(charge)
    n = int(k1.shape[0]) if k1 is not None else 0
    _check(h, load_library().tpc_load_clusters(h, int(sector), int(row), py, pt, pq, n))
    return k1, k2, k3


def tpc_load_clusters_batch(h, unit_off, pad_y, time, charge=None):
    off = np.ascontiguousarray(unit_off, dtype=np.int64)
    py, k1 = _ptr(pad_y); pt, k2 = _ptr(time); pq, k3 = _ptr(charge)
    _check(h, load_library().tpc_load_clusters_batch(h, off.ctypes.data_as(_PL), py, pt, pq))
    return k1, k2, k3


def tpc_clear(h):
    _check(h, load_library().tpc_clear(h))


def tpc_destroy(h):
    load_library().tpc_destroy(h)


def tpc_get_timings(h) -> dict:
    t = _Timings()
    _check(h, load_library().tpc_get_timings(h, C.byref(t)))
    return {k: getattr(t, k) for k, _ in _Timings._fields_}


@dataclass
class Tracks:
    """Result of tpc_find_tracks (numpy views of library-owned pinned host arrays) or tpc_find_tracks_device (torch CUDA tensors,
    library-owned views).  Both stay valid until the next tpc_find_tracks* / tpc_clear / tpc_destroy on the context; use copy() to keep them."""
    n_tracks: int
    n_cluster_refs: int
    sector: object
    x: object
    par: object
    cov: object
    chi2: object
    ndf: object
    tracklet: object
    cl_begin: object
    cl_row: object
    cl_index: object

    def copy(self):
        """Owning copy (the arrays of a result are library-owned views and are overwritten by the next call)."""
        d = {k: (v.copy() if isinstance(v, np.ndarray) else v.clone()) for k, v in self.as_dict().items()}
        return Tracks(self.n_tracks, self.n_cluster_refs, **d)

    def as_dict(self):
        return {k: getattr(self, k) for k in ("sector", "x", "par", "cov", "chi2", "ndf", "tracklet", "cl_begin", "cl_row", "cl_index")}


_FIELDS = [("sector", np.int32, 1), ("x", np.float32, 1), ("par", np.float32, 5), ("cov", np.float32, 15), ("chi2", np.float32, 1),
           ("ndf", np.int32, 1), ("tracklet", np.int32, 1)]


def _host_array(addr, n, dtype):
    """Zero-copy numpy view of a library-owned host array (valid until the next tpc_find_tracks* / tpc_clear / tpc_destroy)."""
    if n == 0 or not addr:
        return np.zeros(0, dtype=dtype)
    ct = {np.int32: C.c_int32, np.float32: C.c_float, np.int64: C.c_int64}[dtype]
    return np.ctypeslib.as_array(C.cast(addr, C.POINTER(ct)), shape=(n,))


class _DevView:
    """Zero-copy view of library-owned device memory through __cuda_array_interface__."""
    def __init__(self, addr, n, dtype):
        self.__cuda_array_interface__ = {"shape": (n,), "typestr": np.dtype(dtype).str, "data": (int(addr), False), "version": 3,
                                         "strides": None}


def _dev_tensor(addr, n, dtype):
    import torch
    if n == 0 or not addr:
        return torch.zeros(0, dtype={np.int32: torch.int32, np.float32: torch.float32, np.int64: torch.int64}[dtype], device="cuda")
    return torch.as_tensor(_DevView(addr, n, dtype), device="cuda")


def _wrap(t: _Tracks, make) -> Tracks:
    nt, nr = int(t.n_tracks), int(t.n_cluster_refs)
    d = {}
    for name, dt, w in _FIELDS:
        a = make(getattr(t, name), nt * w, dt)
        d[name] = a.reshape(nt, w) if w > 1 else a
    d["cl_begin"] = make(t.cl_begin, nt + 1, np.int64)
    d["cl_row"] = make(t.cl_row, nr, np.int32)
    d["cl_index"] = make(t.cl_index, nr, np.int32)
    return Tracks(nt, nr, **d)


def tpc_find_tracks(h) -> Tracks:
    t = _Tracks()
    _check(h, load_library().tpc_find_tracks(h, C.byref(t)))
    return _wrap(t, _host_array)


def tpc_find_tracks_device(h) -> Tracks:
    t = _Tracks()
    _check(h, load_library().tpc_find_tracks_device(h, C.byref(t)))
    return _wrap(t, _dev_tensor)


_REFIT_FIELDS = [("n", np.int32, 1), ("ndf", np.int32, 1), ("x", np.float32, 1), ("par", np.float32, 5), ("cov", np.float32, 15),
                 ("chi2", np.float32, 1), ("z0", np.float32, 1), ("t0", np.float32, 1)]


def tpc_refit_tracks(h, device_result=False) -> dict:
    """S7: refit over the owned clusters + collision time of every track of the last tpc_find_tracks* call (zero-copy views)."""
    t = _Refit()
    _check(h, load_library().tpc_refit_tracks(h, 1 if device_result else 0, C.byref(t)))
    make = _dev_tensor if device_result else _host_array
    nt = int(t.n_tracks)
    d = {"n_tracks": nt, "ms_refit": float(t.ms_refit)}
    for name, dt, w in _REFIT_FIELDS:
        a = make(getattr(t, name), nt * w, dt)
        d[name] = a.reshape(nt, w) if w > 1 else a
    return d


def tpc_mark_clusters(h, tube_cm=1.5, device_result=False) -> dict:
    """S8: attachment status (0 none / 1 attached / 2 adjacent) and track of every cluster, caller's order (zero-copy views)."""
    t = _Marks()
    _check(h, load_library().tpc_mark_clusters(h, float(tube_cm), 1 if device_result else 0, C.byref(t)))
    make = _dev_tensor if device_result else _host_array
    n = int(t.n_clusters)
    return {"n_clusters": n, "ms_mark": float(t.ms_mark), "status": make(t.status, n, np.int32), "track": make(t.track, n, np.int32)}


def tpc_merge_tracks(h, device_result=False) -> dict:
    """S9: next / prev segment of every track across a sector boundary, -1 = none (zero-copy views)."""
    t = _Merges()
    _check(h, load_library().tpc_merge_tracks(h, 1 if device_result else 0, C.byref(t)))
    make = _dev_tensor if device_result else _host_array
    n = int(t.n_tracks)
    return {"n_tracks": n, "ms_merge": float(t.ms_merge), "next": make(t.next, n, np.int32), "prev": make(t.prev, n, np.int32)}


def tpc_find_loopers(h, device_result=False) -> dict:
    """S10: previous turn / first turn / turn number of every track (turns of one looping particle), zero-copy views."""
    t = _Loopers()
    _check(h, load_library().tpc_find_loopers(h, 1 if device_result else 0, C.byref(t)))
    make = _dev_tensor if device_result else _host_array
    n = int(t.n_tracks)
    return {"n_tracks": n, "ms_loopers": float(t.ms_loopers), "prev": make(t.prev, n, np.int32), "root": make(t.root, n, np.int32),
            "turn": make(t.turn, n, np.int32)}


NOALLOC_MAX_TRACKS = 262144   # TPC_NOALLOC_MAX_TRACKS of include/tpc.h


def tpc_find_loopers_noalloc(h, n_tracks, sector, x, par, prev, root, turn) -> None:
    """S10 without any allocation: raw pointers (ints) or objects with data_ptr() to caller-owned DEVICE arrays; the work is queued on
    the context's stream and the call returns without synchronising (include/tpc.h)."""
    ptr = lambda a: C.c_void_p(a.data_ptr() if hasattr(a, "data_ptr") else (int(a) if a is not None else 0))
    _check(h, load_library().tpc_find_loopers_noalloc(h, int(n_tracks), ptr(sector), ptr(x), ptr(par), ptr(prev), ptr(root), ptr(turn)))


class Tracker:
    """Context manager around one tpc_ctx, for the tests and bench.py."""

    def __init__(self, n_sectors, n_rows, row_x, sector_dphi, z_max, t_frame, sigma_y, sigma_z, bz, vdrift, stream=None, **params):
        self.n_sectors, self.n_rows = int(n_sectors), int(n_rows)
        self.h = tpc_create(n_sectors, n_rows, row_x, sector_dphi, z_max, t_frame, sigma_y, sigma_z, bz, vdrift)
        self._keep = []
        for k, v in params.items():
            tpc_set_param(self.h, k, v)
        if stream is not None:
            tpc_set_stream(self.h, stream)

    @classmethod
    def for_workload(cls, w, **params):
        return cls(**w.geometry(), **params)

    def close(self):
        if getattr(self, "h", None):
            tpc_destroy(self.h)
            self.h = None

    __del__ = close

    def __enter__(self):
        return self

    def __exit__(self, *a):
        self.close()

    def set_param(self, name, value):
        tpc_set_param(self.h, name, value)

    def set_stream(self, s):
        tpc_set_stream(self.h, s)

    def load(self, sector, row, pad_y, time, charge=None):
        self._keep.append(tpc_load_clusters(self.h, sector, row, pad_y, time, charge))

    def load_batch(self, unit_off, pad_y, time, charge=None):
        self._keep = [tpc_load_clusters_batch(self.h, unit_off, pad_y, time, charge)]

    def load_workload(self, w, per_unit=False):
        if not per_unit:
            return self.load_batch(w.unit_off, w.y, w.t, w.q)
        for u in range(self.n_sectors * self.n_rows):
            a, b = int(w.unit_off[u]), int(w.unit_off[u + 1])
            if b > a:
                self.load(u // self.n_rows, u % self.n_rows, w.y[a:b], w.t[a:b], w.q[a:b])

    def find_tracks(self) -> Tracks:
        return tpc_find_tracks(self.h)

    def find_tracks_device(self) -> Tracks:
        return tpc_find_tracks_device(self.h)

    def refit_tracks(self, device_result=False) -> dict:
        return tpc_refit_tracks(self.h, device_result)

    def mark_clusters(self, tube_cm=1.5, device_result=False) -> dict:
        return tpc_mark_clusters(self.h, tube_cm, device_result)

    def merge_tracks(self, device_result=False) -> dict:
        return tpc_merge_tracks(self.h, device_result)

    def find_loopers(self, device_result=False) -> dict:
        return tpc_find_loopers(self.h, device_result)

    def find_loopers_noalloc(self, n_tracks, sector, x, par, prev, root, turn) -> None:
        tpc_find_loopers_noalloc(self.h, n_tracks, sector, x, par, prev, root, turn)

    def clear(self):
        self._keep = []
        tpc_clear(self.h)

    def timings(self) -> dict:
        return tpc_get_timings(self.h)

    def measure_fp32_peak(self) -> float:
        """fp32 FMA-loop throughput of the device now, TFLOP/s (measurement utility of the library, not part of the path)."""
        v = C.c_float()
        _check(self.h, load_library().tpc_measure_fp32_peak(self.h, C.byref(v)))
        return float(v.value)

    # ---- parity / debug exports
    def grid(self, sector, row) -> dict:
        g = _GridView()
        _check(self.h, load_library().tpc_debug_get_grid(self.h, sector, row, C.byref(g)))
        n, nb = g.n, g.ny * g.nz
        yz = np.ctypeslib.as_array(g.yz, shape=(max(n, 1) * 2,))[:2 * n].copy().reshape(n, 2)
        return dict(n=n, ny=g.ny, nz=g.nz, y_lo=g.y_lo, z_lo=g.z_lo, inv_s=g.inv_s, yz=yz,
                    perm=np.ctypeslib.as_array(g.perm, shape=(max(n, 1),))[:n].copy(),
                    bin_start=np.ctypeslib.as_array(g.bin_start, shape=(nb + 1,)).copy())

    def links(self, sector, row, cleaned=True):
        up, dn, n = _PI(), _PI(), C.c_int32()
        _check(self.h, load_library().tpc_debug_get_links(self.h, sector, row, int(cleaned), C.byref(up), C.byref(dn), C.byref(n)))
        if n.value == 0:
            return np.zeros(0, np.int32), np.zeros(0, np.int32)
        return (np.ctypeslib.as_array(up, shape=(n.value,)).copy(), np.ctypeslib.as_array(dn, shape=(n.value,)).copy())

    def link_rows(self, sector, row, cleaned=True):
        """(up, dn, up_k, dn_k): link positions and their row distances (1; 2 = the link skips a row, link_skip only; 0 = no link)."""
        up, dn = self.links(sector, row, cleaned)
        a, b, n = C.POINTER(C.c_int8)(), C.POINTER(C.c_int8)(), C.c_int32()
        _check(self.h, load_library().tpc_debug_get_link_rows(self.h, C.byref(a), C.byref(b), C.byref(n)))
        m = len(up)
        if m == 0:
            return up, dn, np.zeros(0, np.int8), np.zeros(0, np.int8)
        return up, dn, np.ctypeslib.as_array(a, shape=(m,)).copy(), np.ctypeslib.as_array(b, shape=(m,)).copy()

    def start_hits(self):
        u, p, n = _PI(), _PI(), C.c_int64()
        _check(self.h, load_library().tpc_debug_get_start_hits(self.h, C.byref(u), C.byref(p), C.byref(n)))
        if n.value == 0:
            return np.zeros(0, np.int32), np.zeros(0, np.int32)
        return (np.ctypeslib.as_array(u, shape=(n.value,)).copy(), np.ctypeslib.as_array(p, shape=(n.value,)).copy())

    def tracklets(self) -> dict:
        v = _TrackletView()
        _check(self.h, load_library().tpc_debug_get_tracklets(self.h, C.byref(v)))
        M, R = int(v.n_tracklets), self.n_rows
        def arr(p, n):
            return np.ctypeslib.as_array(p, shape=(max(n, 1),))[:n].copy()
        return dict(n=arr(v.n_hits, M), sector=arr(v.sector, M), start_row=arr(v.start_row, M), first=arr(v.first_row, M),
                    last=arr(v.last_row, M), chi2=arr(v.chi2, M), x=arr(v.x, M), par=arr(v.par, M * 5).reshape(M, 5),
                    cov=arr(v.cov, M * 15).reshape(M, 15), rowhit=arr(v.rowhit, M * R).reshape(R, M).T.copy())
