"""GPU-vs-oracle comparison used by the -m gpu tests and __graft_entry__.smoke (test infrastructure).

Compares stage by stage in canonical (load-index / global-id) form: links after K2 and K3, start hits,
tracklets (row->hit table, state, covariance), owners, final tracks and cluster lists.
"""
import numpy as np

from paper_1712_09430_b200 import binding


def run_gpu(ev, params=None, max_clusters=None, device_input=False, tracker=None):
    import torch
    trk = tracker or binding.Tracker(ev.n_sectors, ev.n_rows, ev.row_x, ev.bz, params)
    if tracker is None:
        trk.set_stream(torch.cuda.current_stream().cuda_stream)
        trk.allocate_workspace(max_clusters if max_clusters is not None else max(ev.n_clusters, 1))
    if device_input:
        y = torch.from_numpy(ev.y).cuda()
        z = torch.from_numpy(ev.z).cuda()
        trk.load_event(ev.row_counts, y, z)
    else:
        trk.load_event(ev.row_counts, ev.y, ev.z)
    trk.track_sectors()
    tracks, ids = trk.get_tracks()
    return trk, tracks, ids


def compare(ev, trk, tracks, ids, ref, rtol=1e-4, atol=1e-5, check_links=True):
    """Assert parity with the oracle result ``ref``; returns a dict of summary numbers."""
    out = {}
    n = ev.n_clusters
    if check_links:
        links = trk.debug_dump(binding.TPC_DUMP_LINKS)
        # north_star: bit-exact except where the oracle's own candidates tie within 1e-6 (counted).  A raw link (S2)
        # may differ only at a hit the oracle flagged; a cleaned link (S3) of hit h is a function of the raw links of h
        # and of the hits h links to, so it may differ only where one of those is flagged.
        tie = ref.tie_s2 == 1
        allowed = tie.copy()
        rows = np.repeat(np.arange(ev.n_sectors * ev.n_rows), ev.row_counts.reshape(-1))
        base = ev.row_base
        for raw, step in ((ref.link_up, 1), (ref.link_dn, -1), (links[0], 1), (links[1], -1)):
            has = raw >= 0
            partner = base[np.clip(rows + step, 0, base.size - 2)] + np.maximum(raw, 0)
            allowed |= has & tie[np.clip(partner, 0, max(n - 1, 0))]
        for k, (g, o) in enumerate(zip(links, (ref.link_up, ref.link_dn, ref.link_up_clean, ref.link_dn_clean))):
            bad = np.nonzero(g != o)[0]
            ok = tie[bad] if k < 2 else allowed[bad]
            assert np.all(ok), f"links[{k}]: {int((~ok).sum())} mismatches without a near-tie, first {bad[~ok][:5]}"
            out[f"link_mismatch_{k}"] = int(bad.size)
        assert out["link_mismatch_0"] <= 1e-5 * max(n, 1) + 1
        out["near_tie_hits"] = int(tie.sum())
    starts = np.sort(trk.debug_dump(binding.TPC_DUMP_START_HITS).astype(np.int64))
    assert np.array_equal(starts, ref.start_hits), (starts.size, ref.start_hits.size)
    recs, row_hit = trk.debug_dump(binding.TPC_DUMP_TRACKLETS)
    order = np.argsort(recs["start_gid"].astype(np.int64))
    recs, row_hit = recs[order], row_hit[order]
    assert np.array_equal(recs["start_gid"].astype(np.int64), ref.tracklets["start_gid"])
    same_hits = (row_hit == ref.row_hit).all(axis=1)
    tied = ref.tracklets["near_tie"] == 1
    assert np.all(same_hits | tied), f"{(~same_hits & ~tied).sum()} tracklets differ without a near-tie"
    out["tracklet_mismatch"] = int((~same_hits).sum())
    out["near_tie_tracklets"] = int(tied.sum())
    assert out["tracklet_mismatch"] <= 1e-4 * max(1, recs.size) + 1
    s = same_hits
    for f in ("n_hits", "first_row", "last_row", "n_fit", "sector", "start_row"):
        assert np.array_equal(recs[f][s], ref.tracklets[f][s]), f
    assert np.allclose(recs["x"][s], ref.tracklets["x"][s], rtol=0, atol=1e-4)
    for f in ("p", "c", "chi2"):
        a, b = recs[f][s].astype(np.float64), ref.tracklets[f][s]
        err = np.abs(a - b) - (atol + rtol * np.abs(b))
        assert np.all(err <= 0), f"{f}: worst excess {err.max()}"
        out[f"max_abs_diff_{f}"] = float(np.abs(a - b).max()) if a.size else 0.0
        out[f"bitexact_{f}"] = bool(np.array_equal(a.astype(np.float32), b.astype(np.float32)))
    owners = trk.debug_dump(binding.TPC_DUMP_OWNERS).astype(np.int64)
    owners[owners == 0xFFFFFFFF] = -1
    if out["tracklet_mismatch"] == 0:
        assert np.array_equal(owners, ref.owner)
    # final tracks, keyed by first cluster id
    key_g = ids[tracks["cluster_offset"]].astype(np.int64) if tracks.size else np.zeros(0, np.int64)
    key_o = ref.cluster_ids[ref.tracks["cluster_offset"]].astype(np.int64) if ref.tracks.size else np.zeros(0, np.int64)
    og, oo = np.argsort(key_g), np.argsort(key_o)
    if out["tracklet_mismatch"] == 0:
        assert tracks.size == ref.tracks.size and np.array_equal(key_g[og], key_o[oo])
        tg, to = tracks[og], ref.tracks[oo]
        for f in ("sector", "n_clusters", "first_row", "last_row", "n_fit"):
            assert np.array_equal(tg[f], to[f]), f
        for f in ("x", "p", "c", "chi2"):
            a, b = tg[f].astype(np.float64), to[f]
            assert np.all(np.abs(a - b) <= atol + rtol * np.abs(b)), f
        # cluster lists
        for i in range(0, tg.size, max(1, tg.size // 2000)):
            a = ids[tg["cluster_offset"][i]: tg["cluster_offset"][i] + tg["n_clusters"][i]]
            b = ref.cluster_ids[to["cluster_offset"][i]: to["cluster_offset"][i] + to["n_clusters"][i]]
            assert np.array_equal(a.astype(np.int64), b.astype(np.int64))
        assert np.array_equal(np.sort(ids.astype(np.int64)), np.sort(ref.cluster_ids.astype(np.int64)))
    out["n_tracks"] = int(tracks.size)
    out["n_tracklets"] = int(recs.size)
    # no kernel wrote past the end of any workspace buffer (guard zones behind every buffer; tpctrk.h)
    out["guards_hit"] = trk.debug_check_guards()
    assert out["guards_hit"] == 0, f"{out['guards_hit']} workspace guard zones overwritten"
    return out
