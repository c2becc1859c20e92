"""Pins for the oracle's cellular-automaton seeding, selector and whole chain (S1-S4, S6).

PAPER.md:33 ("heuristics in a cellular automaton", seeds of 3..~10 clusters), :43 (best instance kept),
:60 (one hypothesis per hit).  No worked example in the paper, so: brute force, invariants, closed forms.
"""
import numpy as np
import pytest

import datagen
import oracle
from helpers import helix_hits

ROW_X = datagen.default_row_x()


def small_row_x(n):
    return ROW_X[:n].copy()


def brute_links_python(ev, prm):
    """Independent all-pairs neighbour search in pure numpy/Python (fp64), tiny inputs only."""
    n_rows = ev.n_rows
    base = ev.row_base
    y, z = ev.y.astype(np.float64), ev.z.astype(np.float64)
    x = ev.row_x.astype(np.float64)
    up = -np.ones(ev.n_clusters, dtype=np.int32)
    dn = -np.ones(ev.n_clusters, dtype=np.int32)
    for s in range(ev.n_sectors):
        for r in range(1, n_rows - 1):
            sr = s * n_rows + r
            b, bu, bd = base[sr], base[sr + 1], base[sr - 1]
            n, nu, nd = base[sr + 1] - b, base[sr + 2] - bu, b - bd
            if n == 0 or nu == 0 or nd == 0:
                continue
            dxu, dxd = x[r + 1] - x[r], x[r - 1] - x[r]
            wu, wd = -dxd / (dxu - dxd), dxu / (dxu - dxd)
            for h in range(n):
                best = None
                for u in range(nu):
                    if abs(y[bu + u] - y[b + h]) > prm.nf_ty * dxu + prm.nf_c:
                        continue
                    if abs(z[bu + u] - z[b + h]) > prm.nf_tz * dxu + prm.nf_c:
                        continue
                    for d in range(nd):
                        if abs(y[bd + d] - y[b + h]) > prm.nf_ty * -dxd + prm.nf_c:
                            continue
                        if abs(z[bd + d] - z[b + h]) > prm.nf_tz * -dxd + prm.nf_c:
                            continue
                        ey = y[b + h] - (wu * y[bu + u] + wd * y[bd + d])
                        ez = z[b + h] - (wu * z[bu + u] + wd * z[bd + d])
                        key = (ey * ey + ez * ez, u, d)
                        if best is None or key < best:
                            best = key
                if best is not None and best[0] <= prm.nf_d2max:
                    up[b + h], dn[b + h] = best[1], best[2]
    return up, dn


def random_tiny_event(rng, n_rows=10, n_per_row=64, lattice=True, empty_rows=()):
    hits = []
    for r in range(n_rows):
        if r in empty_rows:
            continue
        n = int(rng.integers(1, n_per_row + 1))
        for _ in range(n):
            y, z = rng.uniform(-6, 6), rng.uniform(0, 12)
            if lattice:   # coarse binary lattice: plenty of duplicates, exact ties and hits exactly on window edges
                y, z = round(y * 4) / 4, round(z * 4) / 4
            hits.append((0, r, y, z))
    return datagen.event_from_hits(hits, 1, small_row_x(n_rows))


@pytest.mark.parametrize("seed", range(6))
def test_grid_search_equals_brute_force_links(seed):
    """north_star self-check 1 on S2: grid == the oracle's own brute force == an independent Python all-pairs."""
    rng = np.random.default_rng(seed)
    ev = random_tiny_event(rng, lattice=(seed % 2 == 0), empty_rows=(3,) if seed == 4 else ())
    prm = oracle.default_params()
    for prec in ("double", "float"):
        rg = oracle.run_event(ev, prm, prec, brute_force=False)
        rb = oracle.run_event(ev, prm, prec, brute_force=True)
        assert np.array_equal(rg.link_up, rb.link_up) and np.array_equal(rg.link_dn, rb.link_dn)
        assert np.array_equal(rg.row_hit, rb.row_hit)
        assert np.array_equal(rg.cluster_ids, rb.cluster_ids)
    up, dn = brute_links_python(ev, prm)
    rd = oracle.run_event(ev, prm, "double", brute_force=False)
    assert np.array_equal(rd.link_up, up) and np.array_equal(rd.link_dn, dn)
    assert (up >= 0).sum() >= 3


def test_grid_equals_brute_force_full_chain_dense():
    """Same on a busy realistic sector (config 0 scaled down): every stage identical, grid vs brute."""
    ev = datagen.config_event(0, seed=5, scale=0.25).sector_slice(0)
    for prec in ("float", "double"):
        rg = oracle.run_event(ev, None, prec, brute_force=False)
        rb = oracle.run_event(ev, None, prec, brute_force=True)
        assert np.array_equal(rg.link_up, rb.link_up) and np.array_equal(rg.link_dn, rb.link_dn)
        assert np.array_equal(rg.start_hits, rb.start_hits)
        assert np.array_equal(rg.row_hit, rb.row_hit)
        assert np.array_equal(rg.tracklets["p"], rb.tracklets["p"])
        assert np.array_equal(rg.owner, rb.owner) and np.array_equal(rg.cluster_ids, rb.cluster_ids)
        assert rg.tracks.size > 20


def test_edge_cases_empty_and_single_row():
    rx = small_row_x(5)
    ev = datagen.event_from_hits([], 2, rx)
    r = oracle.run_event(ev)
    assert r.n_clusters == 0 and r.tracks.size == 0 and r.start_hits.size == 0
    ev = datagen.event_from_hits([(1, 2, 0.0, 1.0), (1, 2, 0.1, 1.0)], 2, rx)
    r = oracle.run_event(ev)
    assert np.all(r.link_up == -1) and np.all(r.link_dn == -1) and r.tracks.size == 0
    # first and last rows never carry links of their own
    hits = [(0, r_, 0.0, 5.0) for r_ in range(5)]
    r = oracle.run_event(datagen.event_from_hits(hits, 1, rx))
    assert list(r.link_up) == [-1, 0, 0, 0, -1] and list(r.link_dn) == [-1, 0, 0, 0, -1]
    assert list(r.link_up_clean) == [-1, 0, 0, -1, -1]       # row 3 -> row 4 is not reciprocated
    assert list(r.link_dn_clean) == [-1, -1, 0, 0, -1]
    assert list(r.start_hits) == [1]                          # chain rows 1-2-3 has 3 hits


def test_noise_free_straight_track_is_collinear_across_pitch_jumps():
    """S2 geometry: unequal pitches use the right interpolation weights: d2 < 1e-10 for every triplet (fp64)."""
    prm = oracle.default_params()
    prm.nf_d2max = 1e-10
    # dyadic slopes/offsets and a dyadic row_x keep the straight line exactly representable in fp32
    rx = np.concatenate([100 + 0.75 * np.arange(20), 120 + 1.0 * np.arange(20), 142.5 + 1.5 * np.arange(20)]).astype(np.float32)
    hits = [(0, r, 0.5 + 0.25 * (float(x) - 100.0), 10 + 0.5 * (float(x) - 100.0)) for r, x in enumerate(rx)]
    ev = datagen.event_from_hits(hits, 1, rx)
    r = oracle.run_event(ev, prm, "double")
    assert np.all(r.link_up[1:-1] == 0) and np.all(r.link_dn[1:-1] == 0)
    # a wrong (equal-weight) interpolation would leave 0.2 cm residuals at the two pitch jumps
    prm.nf_d2max = 0.25
    r = oracle.run_event(ev, prm, "double")
    assert r.tracks.size == 1 and r.tracks[0]["n_clusters"] == rx.size


def test_slope_window_inside_outside():
    """|dy/dx| just inside / outside NF_TY*dx + NF_C links / does not link (inclusive test)."""
    rx = np.array([100.0, 101.0, 102.0], dtype=np.float32)
    for dy, expect in ((1.5, True), (1.5 + 2 ** -10, False)):
        hits = [(0, 0, -dy, 0.0), (0, 1, 0.0, 0.0), (0, 2, dy, 0.0)]
        r = oracle.run_event(datagen.event_from_hits(hits, 1, rx), None, "double")
        assert (r.link_up[1] == 0) == expect
    for dz, expect in ((2.0, True), (2.0 + 2 ** -10, False)):
        hits = [(0, 0, 0.0, 50 - dz), (0, 1, 0.0, 50.0), (0, 2, 0.0, 50 + dz)]
        r = oracle.run_event(datagen.event_from_hits(hits, 1, rx), None, "double")
        assert (r.link_up[1] == 0) == expect


def test_tie_break_prefers_smaller_load_index():
    rx = np.array([100.0, 101.0, 102.0], dtype=np.float32)
    # two identical up-candidates and two identical down-candidates: (u,d) = (0,0) must win
    hits = [(0, 0, 0.0, 0.0), (0, 0, 0.0, 0.0), (0, 1, 0.0, 0.0), (0, 2, 0.0, 0.0), (0, 2, 0.0, 0.0)]
    r = oracle.run_event(datagen.event_from_hits(hits, 1, rx))
    assert r.link_up[2] == 0 and r.link_dn[2] == 0


@pytest.fixture(scope="module")
def busy():
    ev = datagen.config_event(2, seed=1)
    return ev, oracle.run_event(ev)


def test_cleaner_invariants(busy):
    ev, r = busy
    base = ev.row_base
    sr = np.repeat(np.arange(ev.n_sectors * ev.n_rows), ev.row_counts.reshape(-1))
    h = np.arange(ev.n_clusters) - base[sr]
    has_up = r.link_up_clean >= 0
    tgt = base[sr[has_up] + 1] + r.link_up_clean[has_up]
    assert np.array_equal(r.link_dn_clean[tgt], h[has_up])           # up => reciprocal down
    has_dn = r.link_dn_clean >= 0
    tgt = base[sr[has_dn] - 1] + r.link_dn_clean[has_dn]
    assert np.array_equal(r.link_up_clean[tgt], h[has_dn])           # down => reciprocal up
    # cleaned links are a subset of the raw links, and cleaning is idempotent
    assert np.all((r.link_up_clean == r.link_up) | (r.link_up_clean == -1))
    up2 = np.where(has_up, r.link_up_clean, -1)
    assert np.array_equal(up2, r.link_up_clean)
    # chains are disjoint: no hit is the up-target of two hits
    tgt = base[sr[has_up] + 1] + r.link_up_clean[has_up]
    assert np.unique(tgt).size == tgt.size


def test_start_hits_equal_chains_of_three(busy):
    """S4: #start hits == #maximal chains with >= 3 hits, counted independently by walking the links."""
    ev, r = busy
    base = ev.row_base
    sr = np.repeat(np.arange(ev.n_sectors * ev.n_rows), ev.row_counts.reshape(-1))
    heads = np.nonzero((r.link_dn_clean < 0) & (r.link_up_clean >= 0))[0]
    starts = []
    for g in heads:
        n, cur = 1, g
        while r.link_up_clean[cur] >= 0:
            cur = base[sr[cur] + 1] + r.link_up_clean[cur]
            n += 1
        if n >= 3:
            starts.append(g)
    assert np.array_equal(np.array(starts), r.start_hits)
    assert np.all(r.link_dn_clean[r.start_hits] < 0)
    lens = []
    assert r.start_hits.size > 1000


def test_selector_invariants(busy):
    ev, r = busy
    # every hit in at most one output track; one per row, ascending; >= MIN_HITS
    assert np.unique(r.cluster_ids).size == r.cluster_ids.size
    sr = np.repeat(np.arange(ev.n_sectors * ev.n_rows), ev.row_counts.reshape(-1))
    for t in r.tracks[:: max(1, r.tracks.size // 300)]:
        ids = r.cluster_ids[t["cluster_offset"]: t["cluster_offset"] + t["n_clusters"]]
        rows = sr[ids] % ev.n_rows
        assert t["n_clusters"] >= 10 and np.all(np.diff(rows) > 0) and np.all(sr[ids] // ev.n_rows == t["sector"])
        assert rows[0] == t["first_row"] and rows[-1] == t["last_row"]
        assert np.all(r.owner[ids] == t["start_gid"])
    # owner(h) = best key among kept tracklets containing h, recomputed independently with numpy
    base = ev.row_base
    kept = np.nonzero(r.tracklets["kept"])[0]
    best = {}
    for ti in kept:
        tr = r.tracklets[ti]
        rows = np.nonzero(r.row_hit[ti] >= 0)[0]
        assert rows.size == tr["n_hits"]
        for g in base[tr["sector"] * ev.n_rows + rows] + r.row_hit[ti][rows]:
            key = (-tr["n_hits"], tr["start_gid"])
            if g not in best or key < best[g]:
                best[g] = key
    own = -np.ones(ev.n_clusters, dtype=np.int64)
    for g, key in best.items():
        own[g] = key[1]
    assert np.array_equal(own, r.owner)


def test_results_do_not_depend_on_load_order():
    """Canonical-ness: permuting the load order inside every (sector,row) permutes the results consistently."""
    ev = datagen.config_event(2, seed=2)
    r1 = oracle.run_event(ev)
    rng = np.random.default_rng(0)
    base = ev.row_base
    perm = np.arange(ev.n_clusters)
    for i in range(base.size - 1):
        perm[base[i]:base[i + 1]] = base[i] + rng.permutation(base[i + 1] - base[i])
    ev2 = datagen.Event(ev.n_sectors, ev.n_rows, ev.row_x, ev.bz, ev.row_counts, ev.y[perm], ev.z[perm], ev.truth[perm])
    r2 = oracle.run_event(ev2)
    # the same physical tracks come out (compare as sets of coordinates): tie-breaks on load index only matter
    # for exact fp ties, which smeared data does not have
    def track_sets(ev_, r_):
        out = set()
        for t in r_.tracks:
            ids = r_.cluster_ids[t["cluster_offset"]: t["cluster_offset"] + t["n_clusters"]]
            out.add((t["sector"], tuple(np.round(ev_.y[ids].astype(np.float64), 6)), tuple(ev_.z[ids].tolist())))
        return out
    assert track_sets(ev, r1) == track_sets(ev2, r2)
    assert (r1.link_up >= 0).sum() == (r2.link_up >= 0).sum()


def test_z_shift_invariance():
    """R-3: a common z shift (time-frame pile-up) changes no link and no assignment."""
    rng = np.random.default_rng(3)
    hits = []
    for trk in range(30):
        rows, y, z = helix_hits(ROW_X, 85.2, rng.uniform(-10, 10), rng.uniform(5, 100), rng.uniform(-0.3, 0.3),
                                rng.uniform(-0.8, 0.8), rng.choice([-1, 1]) / rng.uniform(0.3, 5), 0.5)
        q = 2.0 ** -8     # lattice so that the +64 cm shift is exact in fp32
        hits += [(0, int(r), float(np.round((a + rng.normal() * 0.1) / q) * q),
                  float(np.round((b + rng.normal() * 0.1) / q) * q)) for r, a, b in zip(rows, y, z)]
    ev = datagen.event_from_hits(hits, 1, ROW_X)
    ev2 = datagen.Event(1, ev.n_rows, ev.row_x, ev.bz, ev.row_counts, ev.y, (ev.z - 64.0).astype(np.float32), ev.truth)
    assert np.array_equal(ev2.z.astype(np.float64) + 64.0, ev.z.astype(np.float64))
    a, b = oracle.run_event(ev, None, "double"), oracle.run_event(ev2, None, "double")
    assert np.array_equal(a.link_up, b.link_up) and np.array_equal(a.link_dn, b.link_dn)
    assert np.array_equal(a.row_hit, b.row_hit) and np.array_equal(a.cluster_ids, b.cluster_ids)
    assert a.tracks.size >= 25


def test_clean_single_track_events_are_found_with_all_clusters():
    """north_star self-check 3: one generated track, no noise clusters, no smear: every track-in-sector with
    >= MIN_HITS rows whose seedable part is along x is found as exactly one track holding ALL its clusters."""
    n_checked = 0
    for seed in range(60):
        ev = datagen.generate(seed, n_primaries=1, pt_mode=0, noise_frac=0.0, sigma=0.0)
        res = oracle.run_event(ev, None, "double")
        sec, row = ev.sector_row()
        pt = ev.tracks[0, 3]
        for s in np.unique(sec):
            ids = np.nonzero(sec == s)[0]
            if ids.size < 10:
                continue
            # seedable: somewhere three consecutive rows with |dy/dx| <= 1 (DESIGN.md NF_TY), no row gaps in the piece
            rows = row[ids]
            order = np.argsort(rows)
            ids, rows = ids[order], rows[order]
            slope = np.abs(np.diff(ev.y[ids].astype(np.float64)) / np.diff(ev.row_x[rows].astype(np.float64)))
            contiguous = np.all(np.diff(rows) == 1)
            if not contiguous or slope.max() > 1.0:
                continue          # steep looper legs are outside the seeding acceptance
            tr = res.tracks[res.tracks["sector"] == s]
            assert tr.size == 1, (seed, s, pt, tr.size)
            t = tr[0]
            got = res.cluster_ids[t["cluster_offset"]: t["cluster_offset"] + t["n_clusters"]]
            assert np.array_equal(np.sort(got), np.sort(ids)), (seed, s, pt)
            n_checked += 1
    assert n_checked >= 40


def test_busy_event_efficiency_sanity():
    """Not a contract (SURVEY 8(c) 'whole chain, busy'): the tracker actually tracks."""
    ev = datagen.config_event(2, seed=0)
    r = oracle.run_event(ev)
    e = datagen.efficiency(ev, r.cluster_ids, r.tracks["cluster_offset"], r.tracks["n_clusters"])
    assert e["cluster_eff"] > 0.96 and e["track_eff"] > 0.9
    assert e["fakes"] <= 0.01 * e["n_tracks"] and e["clones"] <= 0.01 * e["n_tracks"]
