"""CPU-side checks of the boundary: libtpctrk.so loads, exports every symbol include/tpctrk.h declares, struct
layouts match the binding, and host-side argument/state validation works without a GPU (no compute calls)."""
import ctypes
import os
import re

import numpy as np
import pytest

from paper_1712_09430_b200 import binding

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_symbols():
    src = open(os.path.join(ROOT, "include", "tpctrk.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(tpc_[a-z_]+)\s*\(", src)))


def test_library_exports_every_declared_symbol():
    L = binding.lib()
    syms = declared_symbols()
    assert len(syms) >= 18 and "tpc_track_sectors" in syms and "tpc_load_clusters" in syms
    for s in syms:
        assert hasattr(L, s), f"{s} declared in include/tpctrk.h but not exported"


def test_struct_layouts_match_header():
    assert ctypes.sizeof(binding.tpc_params) == 22 * 4
    assert ctypes.sizeof(binding.tpc_stats) == 11 * 8 + 4 * 4 + 8 * 4
    assert binding.TRACK_DTYPE.itemsize == 112
    p = binding.default_params()
    assert abs(p.err2_y - 0.01) < 1e-9 and p.min_hits == 10 and p.max_gap == 4 and p.seed_min_chain == 3
    assert abs(p.nf_tz - 1.5) < 1e-9 and abs(p.kf_ckk0 - 100.0) < 1e-9 and abs(p.road_max - 2.0) < 1e-9
    assert abs(p.max_tracklets_per_cluster - 0.1) < 1e-7 and abs(p.grid_bins_per_hit - 2.0) < 1e-9


def test_create_validates_geometry():
    rx = np.linspace(85, 246, 159).astype(np.float32)
    t = binding.Tracker(36, 159, rx, 0.5)
    assert t.workspace_bytes(1000) > 0
    assert t.workspace_bytes(2_000_000) > t.workspace_bytes(1_000_000) > t.workspace_bytes(1000)
    t.destroy()
    for bad in (dict(n_sectors=0), dict(n_rows=2), dict(n_rows=300), dict(row_x=rx[::-1].copy())):
        kw = dict(n_sectors=36, n_rows=159, row_x=rx)
        kw.update(bad)
        with pytest.raises(binding.TpcError) as e:
            binding.Tracker(kw["n_sectors"], kw["n_rows"], kw["row_x"], 0.5)
        assert e.value.code == binding.TPC_E_ARG
    p = binding.default_params()
    p.seed_min_chain = 1
    with pytest.raises(binding.TpcError):
        binding.Tracker(36, 159, rx, 0.5, p)


def test_parameters_outside_their_domain_are_refused():
    """The kernels' branch-free reciprocal / square root assume positive finite variances and roads:
    anything else must be TPC_E_ARG at create, never silent garbage."""
    rx = np.linspace(85, 246, 159).astype(np.float32)
    bad = [("err2_y", 0.0), ("err2_z", -0.01), ("err2_y", float("nan")), ("kf_css0", 0.0), ("kf_ctt0", float("inf")),
           ("kf_ckk0", -1.0), ("road_nsig", 0.0), ("road_max", -2.0), ("road_max", float("nan")), ("kf_smax", 0.0),
           ("kf_smax", 1.0), ("kf_smax", 1.5), ("kf_smax", float("nan")), ("nf_ty", -1.0), ("nf_tz", float("nan")),
           ("nf_c", -0.5), ("nf_d2max", -1.0), ("min_hits", 0), ("max_gap", -1), ("max_tracklets_per_cluster", 0.0),
           ("grid_bins_per_hit", 0.1), ("grid_bins_per_hit", 100.0)]
    for name, val in bad:
        p = binding.default_params()
        setattr(p, name, val)
        with pytest.raises(binding.TpcError) as e:
            binding.Tracker(36, 159, rx, 0.5, p)
        assert e.value.code == binding.TPC_E_ARG, (name, val)
    with pytest.raises(binding.TpcError):
        binding.Tracker(36, 159, rx, float("nan"))
    # the defaults and a few legal corner values pass
    p = binding.default_params()
    p.nf_c, p.max_gap, p.kf_smax = 0.0, 0, 0.999
    binding.Tracker(36, 159, rx, 0.0, p).destroy()


def test_calls_out_of_order_fail_without_touching_the_gpu():
    rx = np.linspace(85, 246, 159).astype(np.float32)
    t = binding.Tracker(2, 159, rx, 0.5)
    y = np.zeros(4, dtype=np.float32)
    with pytest.raises(binding.TpcError) as e:
        t.load_clusters(0, 0, None, y, y)
    assert e.value.code == binding.TPC_E_STATE
    with pytest.raises(binding.TpcError) as e:
        t.track_sectors()
    assert e.value.code == binding.TPC_E_STATE
    with pytest.raises(binding.TpcError) as e:
        t.get_tracks()
    assert e.value.code == binding.TPC_E_STATE
    with pytest.raises(binding.TpcError) as e:
        t.load_clusters(5, 0, None, y, y)
    assert e.value.code == binding.TPC_E_ARG
    # the launch options are host state only: settable before any workspace exists, NULL handle is an argument error
    t.set_kernel_timing(True); t.set_kernel_timing(False)
    t.set_dependent_launch(False); t.set_dependent_launch(True)
    assert binding.lib().tpc_set_kernel_timing(None, 1) == binding.TPC_E_ARG
    assert binding.lib().tpc_set_dependent_launch(None, 1) == binding.TPC_E_ARG
    st = t.get_stats()
    assert st["n_clusters"] == 0 and st["n_tracks"] == 0
    assert st["k6a_fused"] is False
    assert binding.lib().tpc_strerror(binding.TPC_E_OVERFLOW).decode() == "tracklet capacity exceeded"


def test_no_cpu_fallback_in_product_path():
    """The package must not import the oracle, and allocate_workspace must refuse to run without CUDA."""
    import torch
    pkg = os.path.join(ROOT, "paper_1712_09430_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in txt and "from oracle" not in txt and "tpc_oracle" not in txt, f
    if not torch.cuda.is_available():
        t = binding.Tracker(1, 159, np.linspace(85, 246, 159).astype(np.float32), 0.5)
        with pytest.raises(RuntimeError):
            t.allocate_workspace(1000)


def test_header_is_plain_c():
    """include/tpctrk.h is a C header (C99, no torch or CUDA types): it compiles on its own with gcc and with g++."""
    import subprocess
    binding.lib()                                   # (builds the library if this test is the first to need it)
    hdr = os.path.join(ROOT, "include", "tpctrk.h")
    subprocess.check_call(["gcc", "-x", "c", "-std=c99", "-Wall", "-Wextra", "-pedantic", "-Werror", "-fsyntax-only", hdr])
    subprocess.check_call(["g++", "-x", "c++", "-std=c++17", "-Wall", "-Werror", "-fsyntax-only", hdr])
    # a C caller links against the library without any C++ or CUDA header
    src = '#include "tpctrk.h"\nint main(void) { tpc_params p; tpc_default_params(&p); return p.min_hits == 10 ? 0 : 1; }\n'
    import tempfile
    with tempfile.TemporaryDirectory() as d:
        c = os.path.join(d, "t.c")
        open(c, "w").write(src)
        exe = os.path.join(d, "t")
        libdir = os.path.dirname(binding.library_path())
        subprocess.check_call(["gcc", "-std=c99", "-I", os.path.join(ROOT, "include"), c, "-o", exe, "-L", libdir, "-ltpctrk",
                               "-Wl,-rpath," + libdir])
        assert subprocess.run([exe]).returncode == 0
