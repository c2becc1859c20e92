#!/usr/bin/env python
"""Writes tests/golden/oracle_counts.txt: stage counts and checksums of the ORACLE on the small seeded configs.

The paper (arxiv 1712.09430) prints no worked numerical example, so there is no value of the paper's to store here
(DESIGN.md section 2).  These numbers are regression pins of the oracle against itself over time: they are written by
this script, which calls only datagen/ (seeded inputs) and oracle/ - never the CUDA path - and they are compared in
tests/test_golden.py.  A change of the oracle's arithmetic has to regenerate them deliberately
(`python tests/golden/make_golden.py`) and say why in the commit message.
"""
import os
import sys
import zlib

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)
import datagen  # noqa: E402
import oracle  # noqa: E402

CASES = [(0, 0), (1, 0), (2, 0), (2, 1)]   # (config, seed)


def summarise(cfg, seed):
    ev = datagen.config_event(cfg, seed=seed)
    ref = oracle.run_event(ev)
    crc = lambda a: zlib.crc32(np.ascontiguousarray(a).tobytes()) & 0xFFFFFFFF
    order = np.argsort(ref.tracks["start_gid"]) if ref.tracks.size else np.zeros(0, np.int64)
    return {
        "n_clusters": ev.n_clusters,
        "n_links_raw": int((ref.link_up >= 0).sum()),
        "n_links_clean": int((ref.link_up_clean >= 0).sum()),
        "n_start_hits": int(ref.start_hits.size),
        "n_tracklets_kept": int(ref.tracklets["kept"].sum()),
        "n_tracklet_hits": int(ref.tracklets["n_hits"].sum()),
        "n_tracks": int(ref.tracks.size),
        "n_track_clusters": int(ref.cluster_ids.size),
        "crc_links_clean": crc(ref.link_up_clean.astype(np.int32)),
        "crc_start_hits": crc(np.sort(ref.start_hits).astype(np.int64)),
        "crc_cluster_ids": crc(np.sort(ref.cluster_ids).astype(np.int64)),
        "crc_track_n_clusters": crc(ref.tracks["n_clusters"][order].astype(np.int32)),
    }


def lines():
    out = ["# written by tests/golden/make_golden.py (oracle only); config seed key value"]
    for cfg, seed in CASES:
        for k, v in summarise(cfg, seed).items():
            out.append(f"{cfg} {seed} {k} {v}")
    return out


if __name__ == "__main__":
    with open(os.path.join(os.path.dirname(os.path.abspath(__file__)), "oracle_counts.txt"), "w") as f:
        f.write("\n".join(lines()) + "\n")
    print("written")
