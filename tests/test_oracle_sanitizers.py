"""The oracle under AddressSanitizer and UndefinedBehaviorSanitizer ("oracle built with
-fsanitize=address,undefined"): every parity claim rests on oracle/tpc_oracle.cpp, so an out-of-bounds read or a
signed overflow in it must not go unnoticed.  A second build of the same source with the sanitizers on runs Phase I,
merging and the final fit (fp32 and fp64 instantiations, a full-TPC event, a single-sector event, an empty event and
hand-made tracks with holes) in a child process; any report aborts the child."""
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

CHILD = r"""
import sys
sys.path.insert(0, {root!r}); sys.path.insert(0, {root!r} + '/tests')
import oracle
oracle._LIB = {lib!r}                      # the sanitizer build (same source, same entry points)
import numpy as np
import datagen
from test_oracle_merge import hits_of_global_helix, BZ
n = 0
for cfg, seed in ((1, 0), (0, 3)):
    ev = datagen.config_event(cfg, seed=seed)
    for mode in ("float", "double"):
        res = oracle.run_event_refit(ev, None, mode)
        n += int(res.tracks.size)
rng = np.random.default_rng(5)
rx = datagen.default_row_x()
hits = hits_of_global_helix(rng, 0.6, 1, 1.2, 0.5, 0.1) + hits_of_global_helix(rng, 2.0, -1, 4.0, -0.3, 0.1, skip=lambda s, r: 60 <= r < 72)
ev = datagen.event_from_hits(hits, 36, rx, BZ)
prm = oracle.default_params()
prm.field_ar, prm.ms_x0_inv = -2e-6, 1.0 / 3000.0
n += int(oracle.run_event_refit(ev, prm, "float").refits.size)
empty = datagen.event_from_hits([], 36, rx, BZ)
assert oracle.run_event_refit(empty, None, "double").tracks.size == 0
one_row = datagen.event_from_hits([(0, 5, 0.1 * i, 10.0 + i) for i in range(50)], 1, rx, BZ)
assert oracle.run_event(one_row).tracks.size == 0
print("sanitized oracle ok", n)
"""


def _libasan():
    try:
        p = subprocess.run(["gcc", "-print-file-name=libasan.so"], capture_output=True, text=True, check=True).stdout.strip()
    except (OSError, subprocess.CalledProcessError):
        return None
    return p if os.path.isabs(p) and os.path.exists(p) else None


def test_oracle_runs_clean_under_address_and_undefined_behaviour_sanitizers(tmp_path):
    asan = _libasan()
    if asan is None:
        pytest.skip("no libasan beside this gcc")
    lib = str(tmp_path / "libtpcoracle_san.so")
    subprocess.check_call(["g++", "-O1", "-g", "-std=c++17", "-ffp-contract=off", "-fPIC", "-shared",
                           "-fsanitize=address,undefined", "-fno-sanitize-recover=undefined",
                           "-o", lib, os.path.join(ROOT, "oracle", "tpc_oracle.cpp")])
    env = dict(os.environ, LD_PRELOAD=asan, ASAN_OPTIONS="detect_leaks=0:abort_on_error=1", UBSAN_OPTIONS="print_stacktrace=1")
    r = subprocess.run([sys.executable, "-c", CHILD.format(root=ROOT, lib=lib)], env=env, capture_output=True, text=True, timeout=600)
    assert r.returncode == 0 and "sanitized oracle ok" in r.stdout, (r.stdout[-2000:], r.stderr[-4000:])
    assert "runtime error" not in r.stderr and "AddressSanitizer" not in r.stderr, r.stderr[-4000:]
