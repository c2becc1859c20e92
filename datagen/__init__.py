"""Seeded synthetic TPC events (the only module the oracle's tests and the CUDA path share).

Holds none of the tracker's arithmetic.  ``config_event(i, seed)`` builds the i-th workload of
BASELINE.json:configs (recipe: DESIGN.md "Input recipe"); ``event_from_hits``
wraps hand-made hits (closed-form pins) in the same container.  The heavy lifting is the plain-C
generator in ``gen.c`` (own RNG, fp64 maths, fp32 output), compiled on first use with gcc.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from dataclasses import dataclass, field

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "gen.c")
_LIB = os.path.join(_HERE, "libtpcgen.so")

N_SECTORS = 36
N_ROWS = 159
BZ = 0.5
SIGMA = 0.1


class _GenConfig(ctypes.Structure):
    _fields_ = [
        ("n_sectors", ctypes.c_int32), ("n_rows", ctypes.c_int32), ("n_events", ctypes.c_int32),
        ("n_primaries", ctypes.c_int32), ("n_secondaries", ctypes.c_int32), ("pt_mode", ctypes.c_int32),
        ("single_sector", ctypes.c_int32), ("z_shift", ctypes.c_int32),
        ("noise_frac", ctypes.c_double), ("sigma", ctypes.c_double), ("bz", ctypes.c_double),
        ("eta_max", ctypes.c_double), ("seed", ctypes.c_uint64),
    ]


def build(force: bool = False) -> str:
    """Compile gen.c -> libtpcgen.so (idempotent)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(["gcc", "-O2", "-fPIC", "-shared", "-std=c11", "-o", _LIB, _SRC, "-lm"])
    return _LIB


_lib = None


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        lib.tpcgen_generate.restype = ctypes.c_void_p
        lib.tpcgen_generate.argtypes = [ctypes.POINTER(_GenConfig), ctypes.c_void_p]
        lib.tpcgen_n_clusters.restype = ctypes.c_int64
        lib.tpcgen_n_clusters.argtypes = [ctypes.c_void_p]
        lib.tpcgen_n_tracks.restype = ctypes.c_int32
        lib.tpcgen_n_tracks.argtypes = [ctypes.c_void_p]
        lib.tpcgen_copy.restype = None
        lib.tpcgen_copy.argtypes = [ctypes.c_void_p, ctypes.c_int32] + [ctypes.c_void_p] * 5
        lib.tpcgen_free.restype = None
        lib.tpcgen_free.argtypes = [ctypes.c_void_p]
        lib.tpcgen_default_row_x.restype = None
        lib.tpcgen_default_row_x.argtypes = [ctypes.c_int32, ctypes.c_void_p]
        _lib = lib
    return _lib


def default_row_x(n_rows: int = N_ROWS) -> np.ndarray:
    """Pad-row x positions: 85.2 .. 246.0 cm, pitches 0.75/1.0/1.5 with two pitch jumps."""
    out = np.empty(n_rows, dtype=np.float32)
    _load().tpcgen_default_row_x(n_rows, out.ctypes.data)
    return out


@dataclass
class Event:
    """Clusters in (sector,row)-major order; index within a (sector,row) = load index."""
    n_sectors: int
    n_rows: int
    row_x: np.ndarray            # float32 [n_rows]
    bz: float
    row_counts: np.ndarray       # int32 [n_sectors, n_rows]
    y: np.ndarray                # float32 [N]
    z: np.ndarray                # float32 [N]
    truth: np.ndarray            # int32 [N], -1 noise
    tracks: np.ndarray = field(default_factory=lambda: np.zeros((0, 8)))  # vx,vy,vz,pt,q,phi0,eta,zshift
    name: str = ""

    def __post_init__(self):
        # the C ABI carries the field as a float (tpc_tracker_create): both sides get the value a float holds, so that
        # the curvature constant they derive from it is the same number
        self.bz = float(np.float32(self.bz))

    @property
    def n_clusters(self) -> int:
        return int(self.y.shape[0])

    @property
    def row_base(self) -> np.ndarray:
        """Exclusive prefix sum of row_counts over ascending (sector,row): event-global id base."""
        c = self.row_counts.reshape(-1).astype(np.int64)
        b = np.zeros(c.size + 1, dtype=np.int64)
        np.cumsum(c, out=b[1:])
        return b

    def x(self) -> np.ndarray:
        """Per-cluster x = row_x[row] exactly (R-13)."""
        rows = np.repeat(np.tile(np.arange(self.n_rows), self.n_sectors), self.row_counts.reshape(-1))
        return self.row_x[rows].astype(np.float32)

    def sector_row(self):
        """Per-cluster (sector,row) index arrays."""
        sr = np.repeat(np.arange(self.n_sectors * self.n_rows), self.row_counts.reshape(-1))
        return sr // self.n_rows, sr % self.n_rows

    def sector_slice(self, s: int) -> "Event":
        """The single-sector sub-event of sector s (sectors are independent)."""
        b = self.row_base
        lo, hi = int(b[s * self.n_rows]), int(b[(s + 1) * self.n_rows])
        return Event(1, self.n_rows, self.row_x, self.bz, self.row_counts[s:s + 1].copy(),
                     self.y[lo:hi].copy(), self.z[lo:hi].copy(), self.truth[lo:hi].copy(), self.tracks,
                     f"{self.name}/sector{s}")


CONFIGS = {
    # BASELINE.json:configs[i]; see DESIGN.md for the readings R-G1 / R-G2
    0: dict(n_events=1, n_primaries=200, n_secondaries=0, pt_mode=0, single_sector=1, z_shift=0, noise_frac=0.05),
    1: dict(n_events=1, n_primaries=100, n_secondaries=0, pt_mode=0, single_sector=0, z_shift=0, noise_frac=0.02),
    2: dict(n_events=1, n_primaries=1500, n_secondaries=150, pt_mode=1, single_sector=0, z_shift=0, noise_frac=0.10),
    3: dict(n_events=1, n_primaries=8000, n_secondaries=800, pt_mode=1, single_sector=0, z_shift=0, noise_frac=0.20),
    4: dict(n_events=20, n_primaries=8000, n_secondaries=800, pt_mode=1, single_sector=0, z_shift=1, noise_frac=0.20),
}
CONFIG_NAMES = {0: "single-sector", 1: "pp-like", 2: "peripheral-PbPb", 3: "central-PbPb", 4: "timeframe-20x-central"}


def generate(seed: int = 0, *, n_events=1, n_primaries=100, n_secondaries=0, pt_mode=0, single_sector=0,
             z_shift=0, noise_frac=0.0, sigma=SIGMA, bz=BZ, eta_max=0.9, row_x=None, name="custom") -> Event:
    lib = _load()
    rx = default_row_x() if row_x is None else np.ascontiguousarray(row_x, dtype=np.float32)
    cfg = _GenConfig(N_SECTORS, rx.shape[0], n_events, n_primaries, n_secondaries, pt_mode, single_sector, z_shift,
                     noise_frac, sigma, bz, eta_max, seed)
    h = lib.tpcgen_generate(ctypes.byref(cfg), rx.ctypes.data)
    try:
        n = lib.tpcgen_n_clusters(h)
        nt = lib.tpcgen_n_tracks(h)
        counts = np.zeros((N_SECTORS, rx.shape[0]), dtype=np.int32)
        y = np.zeros(n, dtype=np.float32)
        z = np.zeros(n, dtype=np.float32)
        truth = np.zeros(n, dtype=np.int32)
        tracks = np.zeros((nt, 8), dtype=np.float64)
        lib.tpcgen_copy(h, counts.size, counts.ctypes.data, y.ctypes.data, z.ctypes.data, truth.ctypes.data,
                        tracks.ctypes.data)
    finally:
        lib.tpcgen_free(h)
    return Event(N_SECTORS, rx.shape[0], rx, bz, counts, y, z, truth, tracks, name)


def config_event(i: int, seed: int = 0, scale: float = 1.0) -> Event:
    """Workload i of BASELINE.json:configs. ``scale`` multiplies the track counts (tests only)."""
    c = dict(CONFIGS[i])
    c["n_primaries"] = max(1, int(round(c["n_primaries"] * scale)))
    c["n_secondaries"] = int(round(c["n_secondaries"] * scale))
    return generate(seed, name=f"config{i}:{CONFIG_NAMES[i]}", **c)


def event_from_hits(hits, n_sectors: int = 1, row_x=None, bz: float = BZ, name: str = "hand-made") -> Event:
    """Build an Event from an iterable of (sector,row,y,z[,truth]); load order = order given per (sector,row)."""
    rx = default_row_x() if row_x is None else np.ascontiguousarray(row_x, dtype=np.float32)
    n_rows = rx.shape[0]
    hits = list(hits)
    keys = np.array([h[0] * n_rows + h[1] for h in hits], dtype=np.int64) if hits else np.zeros(0, np.int64)
    order = np.argsort(keys, kind="stable")
    counts = np.bincount(keys, minlength=n_sectors * n_rows).astype(np.int32).reshape(n_sectors, n_rows)
    y = np.array([hits[i][2] for i in order], dtype=np.float32)
    z = np.array([hits[i][3] for i in order], dtype=np.float32)
    truth = np.array([hits[i][4] if len(hits[i]) > 4 else -1 for i in order], dtype=np.int32)
    return Event(n_sectors, n_rows, rx, bz, counts, y, z, truth, np.zeros((0, 8)), name)


def findable_tracks(ev: Event, min_hits: int = 10):
    """Truth metric of SURVEY 8(c): (track id, sector) pairs with >= min_hits clusters in that sector."""
    sec, _ = ev.sector_row()
    m = ev.truth >= 0
    key = ev.truth[m].astype(np.int64) * ev.n_sectors + sec[m]
    uniq, cnt = np.unique(key, return_counts=True)
    return uniq[cnt >= min_hits], key, m


def efficiency(ev, cluster_ids, track_offsets, track_counts, min_hits=10):
    """Truth metric of DESIGN.md: cluster-to-track efficiency, track efficiency, clones, fakes.

    Pure bookkeeping on truth labels (no tracker arithmetic); used for oracle and GPU outputs alike by the tests.
    """
    truth = ev.truth
    sec = np.repeat(np.arange(ev.n_sectors * ev.n_rows), ev.row_counts.reshape(-1)) // ev.n_rows
    m = truth >= 0
    key_all = np.where(m, truth.astype(np.int64) * ev.n_sectors + sec, -1)
    uniq, cnt = np.unique(key_all[m], return_counts=True)
    findable = uniq[cnt >= min_hits]
    n_findable_clusters = int(cnt[cnt >= min_hits].sum())
    good = 0
    found = set()
    clones = fakes = 0
    for off, n in zip(track_offsets, track_counts):
        ids = cluster_ids[off:off + n]
        keys = key_all[ids]
        vals, c = np.unique(keys, return_counts=True)
        j = int(np.argmax(c))
        label = int(vals[j])
        if label < 0 or c[j] < 0.9 * n:
            fakes += 1
            if label < 0:
                continue
        if label in found:
            clones += 1
        found.add(label)
        if np.searchsorted(findable, label) < findable.size and findable[np.searchsorted(findable, label)] == label:
            good += int(c[j])
    found_findable = sum(1 for f in found if np.searchsorted(findable, f) < findable.size
                         and findable[np.searchsorted(findable, f)] == f)
    return dict(cluster_eff=good / max(1, n_findable_clusters), track_eff=found_findable / max(1, findable.size),
                n_findable=int(findable.size), clones=clones, fakes=fakes, n_tracks=len(track_counts))
