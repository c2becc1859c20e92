"""ctypes front-end of the CPU oracle (oracle/tpc_oracle.cpp).  TEST INFRASTRUCTURE, not the product.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / ``--impl reference`` legs may import
this package.  It never imports the CUDA package and shares no code with it.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "tpc_oracle.cpp")
_LIB = os.path.join(_HERE, "libtpcoracle.so")


class Params(ctypes.Structure):
    """DESIGN.md 'Constants' (defaults via oracle_default_params)."""
    _fields_ = [
        ("err2_y", ctypes.c_double), ("err2_z", ctypes.c_double),
        ("nf_ty", ctypes.c_double), ("nf_tz", ctypes.c_double), ("nf_c", ctypes.c_double),
        ("nf_d2max", ctypes.c_double),
        ("kf_css0", ctypes.c_double), ("kf_ctt0", ctypes.c_double), ("kf_ckk0", ctypes.c_double),
        ("kf_smax", ctypes.c_double), ("road_nsig", ctypes.c_double), ("road_max", ctypes.c_double),
        ("max_gap", ctypes.c_int32), ("min_hits", ctypes.c_int32), ("seed_min_chain", ctypes.c_int32),
        ("pad", ctypes.c_int32),
        ("merge_chi2", ctypes.c_double), ("merge_max_row_gap", ctypes.c_int32), ("pad2", ctypes.c_int32),
        ("sector_dphi", ctypes.c_double),
        ("field_ar", ctypes.c_double), ("field_az", ctypes.c_double), ("ms_x0_inv", ctypes.c_double),
    ]


TRACKLET_DTYPE = np.dtype([
    ("start_gid", np.int64), ("sector", np.int32), ("start_row", np.int32), ("n_hits", np.int32),
    ("first_row", np.int32), ("last_row", np.int32), ("kept", np.int32), ("n_fit", np.int32),
    ("near_tie", np.int32), ("x", np.float64), ("p", np.float64, 5), ("c", np.float64, 15),
    ("chi2", np.float64)], align=True)
REFIT_DTYPE = np.dtype([
    ("first_track", np.int32), ("sector", np.int32), ("n_fit", np.int32), ("ok", np.int32),
    ("x", np.float64), ("p", np.float64, 5), ("c", np.float64, 15), ("chi2", np.float64)], align=True)
TRACK_DTYPE = np.dtype([
    ("start_gid", np.int64), ("cluster_offset", np.int64), ("sector", np.int32), ("n_clusters", np.int32),
    ("first_row", np.int32), ("last_row", np.int32), ("n_fit", np.int32), ("pad", np.int32),
    ("x", np.float64), ("p", np.float64, 5), ("c", np.float64, 15), ("chi2", np.float64)], align=True)


def build(force: bool = False) -> str:
    """g++ -O2 -ffp-contract=off (IEEE fp32/fp64; fused multiply-adds only where std::fma is written: DESIGN.md R-12)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        flags = ["-O2", "-std=c++17", "-ffp-contract=off", "-fPIC", "-shared", "-Wall"]
        try:   # std::fma is exact either way; with the FMA3 unit it is one instruction instead of a libm call
            if " fma " in open("/proc/cpuinfo").read():
                flags.append("-mfma")
        except OSError:
            pass
        subprocess.check_call(["g++"] + flags + ["-o", _LIB, _SRC])
    return _LIB


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = ctypes.CDLL(build())
        vp, i32, i64, dbl = ctypes.c_void_p, ctypes.c_int32, ctypes.c_int64, ctypes.c_double
        L.oracle_default_params.argtypes = [ctypes.POINTER(Params)]
        L.oracle_create.restype = vp
        L.oracle_create.argtypes = [i32, i32, vp, dbl, ctypes.POINTER(Params), i32]
        L.oracle_destroy.argtypes = [vp]
        L.oracle_run.argtypes = [vp, vp, vp, vp, i32]
        for name in ("oracle_n_clusters", "oracle_n_start_hits", "oracle_n_tracklets", "oracle_n_tracks",
                     "oracle_n_cluster_ids"):
            getattr(L, name).restype = i64
            getattr(L, name).argtypes = [vp]
        L.oracle_get_links.argtypes = [vp, i32, vp]
        L.oracle_get_tie_flags.argtypes = [vp, vp]
        L.oracle_get_start_hits.argtypes = [vp, vp]
        L.oracle_get_tracklets.argtypes = [vp, vp, vp]
        L.oracle_get_owners.argtypes = [vp, vp]
        L.oracle_get_tracks.argtypes = [vp, vp, vp]
        L.oracle_get_stage_seconds.argtypes = [vp, vp]
        L.oracle_sizeof_tracklet.restype = i32
        L.oracle_sizeof_track.restype = i32
        L.oracle_propagate.restype = i32
        L.oracle_propagate.argtypes = [i32, vp, vp, vp, dbl, dbl, dbl, vp]
        L.oracle_update.argtypes = [i32, vp, vp, vp, i32, dbl, dbl]
        L.oracle_merge.argtypes = [vp]
        L.oracle_n_merged.restype = i64
        L.oracle_n_merged.argtypes = [vp]
        L.oracle_get_merge.argtypes = [vp] + [vp] * 6
        L.oracle_scatter.argtypes = [vp, vp, dbl, dbl]
        L.oracle_refit.argtypes = [vp]
        L.oracle_sizeof_refit.restype = i32
        L.oracle_get_refits.argtypes = [vp, vp]
        assert L.oracle_sizeof_refit() == REFIT_DTYPE.itemsize, (L.oracle_sizeof_refit(), REFIT_DTYPE.itemsize)
        L.oracle_rotate.restype = i32
        L.oracle_rotate.argtypes = [i32, vp, vp, vp, dbl, dbl, dbl]
        L.oracle_chi2_5.restype = dbl
        L.oracle_chi2_5.argtypes = [i32, vp, vp]
        assert L.oracle_sizeof_tracklet() == TRACKLET_DTYPE.itemsize, (L.oracle_sizeof_tracklet(), TRACKLET_DTYPE.itemsize)
        assert L.oracle_sizeof_track() == TRACK_DTYPE.itemsize, (L.oracle_sizeof_track(), TRACK_DTYPE.itemsize)
        _lib = L
    return _lib


def default_params() -> Params:
    p = Params()
    lib().oracle_default_params(ctypes.byref(p))
    return p


class Result:
    """All stage outputs of one oracle run, in canonical (order-independent) form.

    links: row-local LOAD index of the linked hit in row r+1 (up) / r-1 (down), -1 none, indexed by
    event-global cluster id.  tracklets/tracks are keyed by ``start_gid`` (global id of the start hit).
    """
    pass


class Oracle:
    def __init__(self, n_sectors, n_rows, row_x, bz, params: Params | None = None, precision="float"):
        self.n_sectors, self.n_rows = int(n_sectors), int(n_rows)
        self._rx = np.ascontiguousarray(row_x, dtype=np.float32)
        self.use_double = 1 if precision == "double" else 0
        self._h = lib().oracle_create(self.n_sectors, self.n_rows, self._rx.ctypes.data, float(bz),
                                      ctypes.byref(params) if params is not None else None, self.use_double)

    def __del__(self):
        try:
            if self._h:
                lib().oracle_destroy(self._h)
                self._h = None
        except Exception:
            pass

    def run(self, row_counts, y, z, brute_force=False, fetch=True) -> Result | None:
        L = lib()
        rc = np.ascontiguousarray(row_counts, dtype=np.int32).reshape(-1)
        assert rc.size == self.n_sectors * self.n_rows
        y = np.ascontiguousarray(y, dtype=np.float32)
        z = np.ascontiguousarray(z, dtype=np.float32)
        assert y.size == int(rc.sum()) == z.size
        L.oracle_run(self._h, rc.ctypes.data, y.ctypes.data, z.ctypes.data, 1 if brute_force else 0)
        return self.fetch() if fetch else None

    def merge(self, res: "Result") -> "Result":
        """Phase II track merging (S7) on the tracks of the last run; adds the merge_* fields to ``res``."""
        L, h = lib(), self._h
        L.oracle_merge(h)
        n, m = res.tracks.size, int(L.oracle_n_merged(h))
        res.merge_next, res.merge_prev = np.empty(n, np.int32), np.empty(n, np.int32)
        res.merge_chi2, res.merge_tie = np.empty(n, np.float64), np.empty(n, np.uint8)
        res.merged_offset, res.merged_segs = np.empty(m + 1, np.int32), np.empty(n, np.int32)
        L.oracle_get_merge(h, res.merge_next.ctypes.data, res.merge_prev.ctypes.data, res.merge_chi2.ctypes.data,
                           res.merge_tie.ctypes.data, res.merged_offset.ctypes.data, res.merged_segs.ctypes.data)
        return res

    def refit(self, res: "Result") -> "Result":
        """Final fit of the merged tracks (S8) after merge(); adds res.refits (one per merged track)."""
        L, h = lib(), self._h
        L.oracle_refit(h)
        res.refits = np.empty(res.merged_offset.size - 1, dtype=REFIT_DTYPE)
        L.oracle_get_refits(h, res.refits.ctypes.data)
        return res

    def stage_seconds(self):
        s = np.zeros(6)
        lib().oracle_get_stage_seconds(self._h, s.ctypes.data)
        return dict(zip(("grid", "neighbours", "clean", "start_hits", "construct", "select"), s.tolist()))

    def fetch(self) -> Result:
        L, h = lib(), self._h
        r = Result()
        n = L.oracle_n_clusters(h)
        r.n_clusters = n
        links = []
        for which in range(4):
            a = np.empty(n, dtype=np.int32)
            L.oracle_get_links(h, which, a.ctypes.data)
            links.append(a)
        r.link_up, r.link_dn, r.link_up_clean, r.link_dn_clean = links
        r.tie_s2 = np.empty(n, dtype=np.uint8)
        L.oracle_get_tie_flags(h, r.tie_s2.ctypes.data)
        ns = L.oracle_n_start_hits(h)
        r.start_hits = np.empty(ns, dtype=np.int64)
        L.oracle_get_start_hits(h, r.start_hits.ctypes.data)
        m = L.oracle_n_tracklets(h)
        r.tracklets = np.empty(m, dtype=TRACKLET_DTYPE)
        r.row_hit = np.empty((m, self.n_rows), dtype=np.int32)
        L.oracle_get_tracklets(h, r.tracklets.ctypes.data, r.row_hit.ctypes.data)
        r.owner = np.empty(n, dtype=np.int64)
        L.oracle_get_owners(h, r.owner.ctypes.data)
        nt, nc = L.oracle_n_tracks(h), L.oracle_n_cluster_ids(h)
        r.tracks = np.empty(nt, dtype=TRACK_DTYPE)
        r.cluster_ids = np.empty(nc, dtype=np.int32)
        L.oracle_get_tracks(h, r.tracks.ctypes.data, r.cluster_ids.ctypes.data)
        return r


def run_event(ev, params: Params | None = None, precision="float", brute_force=False) -> Result:
    """Convenience: run the oracle on a datagen.Event-like object (duck-typed, no import of datagen)."""
    o = Oracle(ev.n_sectors, ev.n_rows, ev.row_x, ev.bz, params, precision)
    return o.run(ev.row_counts, ev.y, ev.z, brute_force)


def run_event_merged(ev, params: Params | None = None, precision="float") -> Result:
    """Phase I + Phase II merging on a datagen.Event-like object."""
    o = Oracle(ev.n_sectors, ev.n_rows, ev.row_x, ev.bz, params, precision)
    return o.merge(o.run(ev.row_counts, ev.y, ev.z))


def run_event_refit(ev, params: Params | None = None, precision="float") -> Result:
    """Phase I + Phase II (merging, final fit)."""
    o = Oracle(ev.n_sectors, ev.n_rows, ev.row_x, ev.bz, params, precision)
    return o.refit(o.merge(o.run(ev.row_counts, ev.y, ev.z)))


def scatter(p, c, length, x0_inv):
    """Covariance c[15] after multiple scattering over `length` cm (S8 process noise); returns the new c."""
    pa, ca = np.array(p, dtype=np.float64), np.array(c, dtype=np.float64).copy()
    lib().oracle_scatter(pa.ctypes.data, ca.ctypes.data, float(length), float(x0_inv))
    return ca


def rotate(x, p, c, beta, cb, smax=0.95, precision="double"):
    """Rotate a state into the frame turned by +beta about z; returns (ok, x', p'[5], c'[15])."""
    xa = np.array([x], dtype=np.float64)
    pa, ca = np.array(p, dtype=np.float64).copy(), np.array(c, dtype=np.float64).copy()
    ok = lib().oracle_rotate(1 if precision == "double" else 0, xa.ctypes.data, pa.ctypes.data, ca.ctypes.data,
                             float(beta), float(cb), float(smax))
    return bool(ok), float(xa[0]), pa, ca


def chi2_5(d, s15, precision="double"):
    da, sa = np.ascontiguousarray(d, dtype=np.float64), np.ascontiguousarray(s15, dtype=np.float64)
    return float(lib().oracle_chi2_5(1 if precision == "double" else 0, da.ctypes.data, sa.ctypes.data))


def propagate(x, p, c, x2, cb, smax=0.95, precision="double"):
    """One propagation step; returns (ok, x, p[5], c[15], J[5,5])."""
    xa = np.array([x], dtype=np.float64)
    pa = np.array(p, dtype=np.float64).copy()
    ca = np.array(c, dtype=np.float64).copy()
    J = np.zeros((5, 5))
    ok = lib().oracle_propagate(1 if precision == "double" else 0, xa.ctypes.data, pa.ctypes.data, ca.ctypes.data,
                                float(x2), float(cb), float(smax), J.ctypes.data)
    return bool(ok), float(xa[0]), pa, ca, J


def update(p, c, chi2, coord, m, e2, precision="double"):
    """One scalar Kalman update; returns (p, c, chi2)."""
    pa = np.array(p, dtype=np.float64).copy()
    ca = np.array(c, dtype=np.float64).copy()
    ch = np.array([chi2], dtype=np.float64)
    lib().oracle_update(1 if precision == "double" else 0, pa.ctypes.data, ca.ctypes.data, ch.ctypes.data,
                        int(coord), float(m), float(e2))
    return pa, ca, float(ch[0])
