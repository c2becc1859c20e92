"""Thin ctypes binding of libtpctrk.so: same names as include/tpctrk.h, argument marshalling only.

Every step of the hot path runs in the CUDA kernels; PyTorch is used for the workspace allocation and the
stream handle.  If the library is missing or there is no GPU, calls fail loudly: there is no CPU fallback.
"""
from __future__ import annotations

import ctypes
import os

import numpy as np

from . import build as _build

c_float_p = ctypes.POINTER(ctypes.c_float)


class tpc_params(ctypes.Structure):
    _fields_ = [
        ("err2_y", ctypes.c_float), ("err2_z", ctypes.c_float), ("nf_ty", ctypes.c_float), ("nf_tz", ctypes.c_float),
        ("nf_c", ctypes.c_float), ("nf_d2max", ctypes.c_float), ("kf_css0", ctypes.c_float),
        ("kf_ctt0", ctypes.c_float), ("kf_ckk0", ctypes.c_float), ("kf_smax", ctypes.c_float),
        ("road_nsig", ctypes.c_float), ("road_max", ctypes.c_float), ("max_gap", ctypes.c_int32),
        ("min_hits", ctypes.c_int32), ("seed_min_chain", ctypes.c_int32),
        ("max_tracklets_per_cluster", ctypes.c_float), ("grid_bins_per_hit", ctypes.c_float),
        ("merge_chi2", ctypes.c_float), ("merge_max_row_gap", ctypes.c_int32),
        ("field_ar", ctypes.c_float), ("field_az", ctypes.c_float), ("ms_x0_inv", ctypes.c_float),
    ]


class tpc_geometry(ctypes.Structure):
    _fields_ = [
        ("n_sectors", ctypes.c_int32), ("n_rows", ctypes.c_int32), ("row_x", c_float_p),
        ("sector_dphi", ctypes.c_float), ("z_max", ctypes.c_float), ("params", ctypes.POINTER(tpc_params)),
    ]


class tpc_stats(ctypes.Structure):
    _fields_ = [
        ("n_clusters", ctypes.c_int64), ("n_links", ctypes.c_int64), ("n_start_hits", ctypes.c_int64),
        ("n_tracklets", ctypes.c_int64), ("n_tracklet_hits", ctypes.c_int64), ("n_tracks", ctypes.c_int64),
        ("n_track_clusters", ctypes.c_int64), ("workspace_bytes_used", ctypes.c_int64),
        ("max_clusters", ctypes.c_int64), ("max_tracklets", ctypes.c_int64), ("n_output_refetches", ctypes.c_int64),
        ("merge_us", ctypes.c_float), ("n_merged_tracks", ctypes.c_int32), ("n_merge_links", ctypes.c_int32), ("refit_us", ctypes.c_float),
        ("kernel_us", ctypes.c_float * 8),
    ]


TRACK_DTYPE = np.dtype([
    ("sector", np.int32), ("n_clusters", np.int32), ("first_row", np.int32), ("last_row", np.int32),
    ("cluster_offset", np.int32), ("x", np.float32), ("p", np.float32, 5), ("c", np.float32, 15),
    ("chi2", np.float32), ("n_fit", np.int32)])
TRACKLET_DTYPE = np.dtype([
    ("start_gid", np.uint32), ("sector", np.int32), ("start_row", np.int32), ("n_hits", np.int32),
    ("first_row", np.int32), ("last_row", np.int32), ("n_fit", np.int32), ("x", np.float32),
    ("p", np.float32, 5), ("c", np.float32, 15), ("chi2", np.float32)])
MERGED_DTYPE = np.dtype([("n_segments", np.int32), ("n_clusters", np.int32), ("segment_offset", np.int32), ("first_track", np.int32)])
REFIT_DTYPE = np.dtype([("first_track", np.int32), ("sector", np.int32), ("n_fit", np.int32), ("ok", np.int32),
                        ("x", np.float32), ("p", np.float32, 5), ("c", np.float32, 15), ("chi2", np.float32)])
assert TRACK_DTYPE.itemsize == 112 and TRACKLET_DTYPE.itemsize == 116 and REFIT_DTYPE.itemsize == 104

TPC_OK, TPC_E_ARG, TPC_E_STATE, TPC_E_NOMEM, TPC_E_OVERFLOW, TPC_E_CUDA, TPC_E_LIMIT = 0, -1, -2, -3, -4, -5, -6
TPC_NO_ALLOC_MAX_TRACKS, TPC_NO_ALLOC_MAX_BINS = 65536, 16384
TPC_DUMP_LINKS, TPC_DUMP_START_HITS, TPC_DUMP_TRACKLETS, TPC_DUMP_OWNERS = 1, 2, 3, 4
KERNEL_NAMES = ("K1_sort_grid", "K2_neighbours", "K3K4_clean_start", "K5_construct", "K6a_weights", "K6b_select")

_lib = None


def library_path() -> str:
    return _build.LIB


def lib():
    """Load libtpctrk.so (building it if sources are newer).  Raises if it cannot be built or loaded."""
    global _lib
    if _lib is None:
        path = os.environ.get("TPCTRK_LIB")   # an explicitly given build of the same library (tuning experiments)
        if not path:
            path = _build.build() if (_build.needs_build() and os.path.exists(_build.SOURCES[0])) else _build.LIB
        L = ctypes.CDLL(path)
        vp, i32, i64 = ctypes.c_void_p, ctypes.c_int32, ctypes.c_int64
        L.tpc_default_params.argtypes = [ctypes.POINTER(tpc_params)]
        L.tpc_default_params.restype = None
        L.tpc_tracker_create.argtypes = [ctypes.POINTER(tpc_geometry), ctypes.c_float, ctypes.POINTER(vp)]
        L.tpc_tracker_destroy.argtypes = [vp]
        L.tpc_tracker_destroy.restype = None
        L.tpc_set_stream.argtypes = [vp, vp]
        L.tpc_set_kernel_timing.argtypes = [vp, ctypes.c_int]
        L.tpc_set_dependent_launch.argtypes = [vp, ctypes.c_int]
        L.tpc_set_output_prefetch.argtypes = [vp, ctypes.c_int]
        L.tpc_set_neighbour_staging.argtypes = [vp, ctypes.c_int]
        L.tpc_wait_input.argtypes = [vp]
        L.tpc_workspace_bytes.argtypes = [vp, i64]
        L.tpc_workspace_bytes.restype = ctypes.c_size_t
        L.tpc_set_workspace.argtypes = [vp, vp, ctypes.c_size_t]
        L.tpc_reset_event.argtypes = [vp]
        L.tpc_load_clusters.argtypes = [vp, i32, i32, i32, vp, vp, vp]
        L.tpc_load_event.argtypes = [vp, vp, vp, vp]
        L.tpc_track_sectors.argtypes = [vp]
        L.tpc_get_tracks.argtypes = [vp, ctypes.POINTER(vp), ctypes.POINTER(i32), ctypes.POINTER(vp), ctypes.POINTER(i64)]
        L.tpc_sync.argtypes = [vp]
        L.tpc_track_event_sliced.argtypes = [vp, vp, vp, vp, i32, ctypes.POINTER(vp), ctypes.POINTER(i32), ctypes.POINTER(vp),
                                             ctypes.POINTER(i64)]
        L.tpc_merge_tracks.argtypes = [vp]
        L.tpc_refit_tracks.argtypes = [vp]
        L.tpc_get_refit.argtypes = [vp, ctypes.POINTER(vp), ctypes.POINTER(i32)]
        L.tpc_get_merged.argtypes = [vp, ctypes.POINTER(vp), ctypes.POINTER(vp), ctypes.POINTER(vp), ctypes.POINTER(i32),
                                     ctypes.POINTER(vp), ctypes.POINTER(i32), ctypes.POINTER(vp)]
        L.tpc_get_stats.argtypes = [vp, ctypes.POINTER(tpc_stats)]
        L.tpc_debug_dump_bytes.argtypes = [vp, i32]
        L.tpc_debug_dump_bytes.restype = ctypes.c_size_t
        L.tpc_debug_dump.argtypes = [vp, i32, vp, ctypes.c_size_t]
        L.tpc_debug_check_guards.argtypes = [vp]
        L.tpc_strerror.argtypes = [i32]
        L.tpc_strerror.restype = ctypes.c_char_p
        L.tpc_last_cuda_error.argtypes = [vp]
        L.tpc_launches_per_track.argtypes = [vp]
        L.tpc_merge_links_no_alloc.argtypes = [i32, i32, ctypes.c_float, ctypes.c_float, ctypes.POINTER(tpc_params), vp, i32, vp,
                                               vp, vp, vp, vp, ctypes.POINTER(ctypes.c_int)]
        _lib = L
    return _lib


class TpcError(RuntimeError):
    def __init__(self, code, where, cuda=0):
        self.code = code
        msg = lib().tpc_strerror(code).decode()
        super().__init__(f"{where}: {msg} (code {code}" + (f", cudaError {cuda})" if cuda else ")"))


def default_params() -> tpc_params:
    p = tpc_params()
    lib().tpc_default_params(ctypes.byref(p))
    return p


def merge_links_no_alloc(n_sectors, n_rows, sector_dphi, bz_tesla, params, dev_tracks, n_tracks, dev_cluster_ids,
                         dev_next, dev_prev, dev_chi2, stream=None):
    """tpc_merge_links_no_alloc: K7's links for caller-owned DEVICE arrays (torch tensors or raw device pointers), its
    scratch in the library's static device array; allocates nothing.  Asynchronous on `stream` (a cudaStream_t as int)."""
    err = ctypes.c_int(0)
    dp = lambda a: a if isinstance(a, (int, type(None))) else a.data_ptr()
    rc = lib().tpc_merge_links_no_alloc(int(n_sectors), int(n_rows), float(sector_dphi), float(bz_tesla),
                                        ctypes.byref(params) if params is not None else None, dp(dev_tracks), int(n_tracks),
                                        dp(dev_cluster_ids), dp(dev_next), dp(dev_prev), dp(dev_chi2),
                                        int(stream) if stream else None, ctypes.byref(err))
    if rc != TPC_OK:
        raise TpcError(rc, "tpc_merge_links_no_alloc", err.value)


def _ptr(a):
    """Device pointer of a torch tensor, host pointer of a numpy array, or None."""
    if a is None:
        return None
    if hasattr(a, "data_ptr"):
        return ctypes.c_void_p(a.data_ptr())
    return ctypes.c_void_p(a.ctypes.data)


class Tracker:
    """Python mirror of the C API: one method per tpc_* call (same name without the prefix)."""

    def __init__(self, n_sectors, n_rows, row_x, bz, params: tpc_params | None = None, stream=None):
        self._L = lib()
        self._rx = np.ascontiguousarray(row_x, dtype=np.float32)
        self.n_sectors, self.n_rows = int(n_sectors), int(n_rows)
        self._params = params
        g = tpc_geometry(self.n_sectors, self.n_rows, self._rx.ctypes.data_as(c_float_p), float(np.deg2rad(20.0)),
                         250.0, ctypes.pointer(params) if params is not None else None)
        h = ctypes.c_void_p()
        self._check(self._L.tpc_tracker_create(ctypes.byref(g), ctypes.c_float(bz), ctypes.byref(h)), "tpc_tracker_create")
        self._h = h
        self._ws = None
        if stream is not None:
            self.set_stream(stream)

    def _check(self, rc, where, allow=()):
        if rc != TPC_OK and rc not in allow:
            cuda = self._L.tpc_last_cuda_error(self._h) if getattr(self, "_h", None) else 0
            raise TpcError(rc, where, cuda)
        return rc

    def destroy(self):
        if getattr(self, "_h", None):
            self._L.tpc_tracker_destroy(self._h)
            self._h = None
            self._ws = None

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass

    def set_stream(self, cuda_stream: int):
        self._check(self._L.tpc_set_stream(self._h, ctypes.c_void_p(cuda_stream)), "tpc_set_stream")

    def set_kernel_timing(self, on: bool):
        self._check(self._L.tpc_set_kernel_timing(self._h, 1 if on else 0), "tpc_set_kernel_timing")

    def set_dependent_launch(self, on: bool):
        self._check(self._L.tpc_set_dependent_launch(self._h, 1 if on else 0), "tpc_set_dependent_launch")

    def set_neighbour_staging(self, on: bool):
        self._check(self._L.tpc_set_neighbour_staging(self._h, 1 if on else 0), "tpc_set_neighbour_staging")

    def set_output_prefetch(self, on: bool):
        self._check(self._L.tpc_set_output_prefetch(self._h, 1 if on else 0), "tpc_set_output_prefetch")

    def wait_input(self):
        return self._check(self._L.tpc_wait_input(self._h), "tpc_wait_input")

    def workspace_bytes(self, max_clusters: int) -> int:
        return int(self._L.tpc_workspace_bytes(self._h, int(max_clusters)))

    def set_workspace(self, tensor):
        """tensor: a torch CUDA uint8 tensor (caller-owned device memory; kept alive here)."""
        self._ws = tensor
        self._check(self._L.tpc_set_workspace(self._h, ctypes.c_void_p(tensor.data_ptr()), tensor.numel() * tensor.element_size()),
                    "tpc_set_workspace")

    def allocate_workspace(self, max_clusters: int, device="cuda:0"):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("paper_1712_09430_b200 needs a CUDA device: there is no CPU fallback")
        nbytes = self.workspace_bytes(max_clusters)
        self.set_workspace(torch.empty(nbytes, dtype=torch.uint8, device=device))
        return nbytes

    def reset_event(self):
        self._check(self._L.tpc_reset_event(self._h), "tpc_reset_event")

    def load_clusters(self, sector, row, x, y, z):
        n = int(y.shape[0]) if y is not None else 0
        return self._check(self._L.tpc_load_clusters(self._h, int(sector), int(row), n, _ptr(x), _ptr(y), _ptr(z)),
                           "tpc_load_clusters")

    def load_event(self, row_counts, y, z):
        rc = np.ascontiguousarray(row_counts, dtype=np.int32).reshape(-1)
        assert rc.size == self.n_sectors * self.n_rows
        return self._check(self._L.tpc_load_event(self._h, rc.ctypes.data, _ptr(y), _ptr(z)), "tpc_load_event")

    def track_sectors(self):
        return self._check(self._L.tpc_track_sectors(self._h), "tpc_track_sectors")

    def sync(self):
        return self._check(self._L.tpc_sync(self._h), "tpc_sync")

    def get_tracks(self, copy=True, allow_overflow=False):
        tp, ip = ctypes.c_void_p(), ctypes.c_void_p()
        nt, nc = ctypes.c_int32(), ctypes.c_int64()
        rc = self._check(self._L.tpc_get_tracks(self._h, ctypes.byref(tp), ctypes.byref(nt), ctypes.byref(ip), ctypes.byref(nc)),
                         "tpc_get_tracks", allow=(TPC_E_OVERFLOW,) if allow_overflow else ())
        if nt.value:
            buf = (ctypes.c_char * (nt.value * TRACK_DTYPE.itemsize)).from_address(tp.value)
            tracks = np.frombuffer(buf, dtype=TRACK_DTYPE)
        else:
            tracks = np.zeros(0, dtype=TRACK_DTYPE)
        if nc.value:
            buf = (ctypes.c_char * (nc.value * 4)).from_address(ip.value)
            ids = np.frombuffer(buf, dtype=np.uint32)
        else:
            ids = np.zeros(0, dtype=np.uint32)
        if copy:
            tracks, ids = tracks.copy(), ids.copy()
        return (tracks, ids, rc) if allow_overflow else (tracks, ids)

    def track_event_sliced(self, row_counts, y, z, sectors_per_slice):
        """tpc_track_event_sliced -> (tracks, cluster ids) of the whole event, processed slice after slice."""
        rc = np.ascontiguousarray(row_counts, dtype=np.int32).reshape(-1)
        assert rc.size == self.n_sectors * self.n_rows
        tp, ip = ctypes.c_void_p(), ctypes.c_void_p()
        nt, nc = ctypes.c_int32(), ctypes.c_int64()
        self._check(self._L.tpc_track_event_sliced(self._h, rc.ctypes.data, _ptr(y), _ptr(z), int(sectors_per_slice), ctypes.byref(tp),
                                                   ctypes.byref(nt), ctypes.byref(ip), ctypes.byref(nc)), "tpc_track_event_sliced")
        tracks = np.frombuffer((ctypes.c_char * (nt.value * TRACK_DTYPE.itemsize)).from_address(tp.value), dtype=TRACK_DTYPE).copy() \
            if nt.value else np.zeros(0, dtype=TRACK_DTYPE)
        ids = np.frombuffer((ctypes.c_char * (nc.value * 4)).from_address(ip.value), dtype=np.uint32).copy() \
            if nc.value else np.zeros(0, dtype=np.uint32)
        return tracks, ids

    def merge_tracks(self):
        return self._check(self._L.tpc_merge_tracks(self._h), "tpc_merge_tracks")

    def get_merged(self):
        """-> dict(next, prev, chi2 per track; merged records; segments)."""
        nx, pv, ch, mg, sg = (ctypes.c_void_p() for _ in range(5))
        nt, nm = ctypes.c_int32(), ctypes.c_int32()
        self._check(self._L.tpc_get_merged(self._h, ctypes.byref(nx), ctypes.byref(pv), ctypes.byref(ch), ctypes.byref(nt),
                                           ctypes.byref(mg), ctypes.byref(nm), ctypes.byref(sg)), "tpc_get_merged")

        def arr(p, n, dt):
            if not n:
                return np.zeros(0, dtype=dt)
            buf = (ctypes.c_char * (n * np.dtype(dt).itemsize)).from_address(p.value)
            return np.frombuffer(buf, dtype=dt).copy()
        n, m = nt.value, nm.value
        return {"next": arr(nx, n, np.int32), "prev": arr(pv, n, np.int32), "chi2": arr(ch, n, np.float32),
                "merged": arr(mg, m, MERGED_DTYPE), "segments": arr(sg, n, np.int32)}

    def refit_tracks(self):
        return self._check(self._L.tpc_refit_tracks(self._h), "tpc_refit_tracks")

    def get_refit(self):
        """-> tpc_refit_track records, one per merged track (same order as get_merged()["merged"])."""
        rp, n = ctypes.c_void_p(), ctypes.c_int32()
        self._check(self._L.tpc_get_refit(self._h, ctypes.byref(rp), ctypes.byref(n)), "tpc_get_refit")
        if not n.value:
            return np.zeros(0, dtype=REFIT_DTYPE)
        buf = (ctypes.c_char * (n.value * REFIT_DTYPE.itemsize)).from_address(rp.value)
        return np.frombuffer(buf, dtype=REFIT_DTYPE).copy()

    def get_stats(self) -> dict:
        s = tpc_stats()
        self._check(self._L.tpc_get_stats(self._h, ctypes.byref(s)), "tpc_get_stats")
        d = {k: int(getattr(s, k)) for k, _ in tpc_stats._fields_ if k not in ("kernel_us", "merge_us", "refit_us")}
        d["merge_us"], d["refit_us"] = float(s.merge_us), float(s.refit_us)
        d["kernel_us"] = dict(zip(KERNEL_NAMES, [float(v) for v in s.kernel_us[:6]]))
        d["total_us"] = float(s.kernel_us[6])
        d["k6a_fused"] = bool(s.kernel_us[7] > 0.5)
        return d

    def debug_check_guards(self) -> int:
        rc = int(self._L.tpc_debug_check_guards(self._h))
        if rc < 0:
            self._check(rc, "tpc_debug_check_guards")
        return rc

    def launches_per_track(self) -> int:
        return int(self._L.tpc_launches_per_track(self._h))

    def debug_dump(self, stage):
        n = int(self._L.tpc_debug_dump_bytes(self._h, stage))
        buf = np.zeros(max(n, 1), dtype=np.uint8)
        self._check(self._L.tpc_debug_dump(self._h, stage, buf.ctypes.data, n), "tpc_debug_dump")
        buf = buf[:n]
        if stage == TPC_DUMP_LINKS:
            return buf.view(np.int32).reshape(4, -1)
        if stage in (TPC_DUMP_START_HITS, TPC_DUMP_OWNERS):
            return buf.view(np.uint32)
        m = n // (TRACKLET_DTYPE.itemsize + 4 * self.n_rows)
        recs = buf[:m * TRACKLET_DTYPE.itemsize].view(TRACKLET_DTYPE)
        row_hit = buf[m * TRACKLET_DTYPE.itemsize:].view(np.int32).reshape(m, self.n_rows)
        return recs, row_hit
