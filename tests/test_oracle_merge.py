"""Pins for the oracle's Phase-II track merging (S7; "merges track segments inside the sector
for the case that there is a gap which the track following did not cover ... track parameters at the border of the
sectors are compared and matching tracks are merged"; Table 1: "Matching Covariance").

The paper gives no formula; the rotation of a state between sector frames, its Jacobian and the chi2 distance are
pinned against plain geometry (a circle in the global frame, expressed in two sector frames), group properties, a
finite-difference Jacobian and numpy's linear algebra; the decision logic against hand-made events.
"""
import numpy as np
import pytest

import datagen
import oracle
from helpers import CB_PER_T, tri, untri

ROW_X = datagen.default_row_x()
DPHI = np.deg2rad(20.0)
BZ = 0.5
CB = CB_PER_T * BZ


def rand_state(rng):
    p = np.array([rng.uniform(-8, 8), rng.uniform(10, 200), rng.uniform(-0.4, 0.4), rng.uniform(-1, 1), rng.uniform(-3, 3)])
    a = rng.normal(size=(5, 5)) * np.array([0.05, 0.05, 0.01, 0.01, 0.05])[:, None]
    return p, a @ a.T + np.diag([1e-4, 1e-4, 1e-6, 1e-6, 1e-4])


def global_circle(x, p, alpha):
    """Global description of the track through local state p at local x in the frame rotated by alpha: point, direction
    angle, curvature (signed), z, dz/ds."""
    y, z, s, t, k = p
    ca, sa = np.cos(alpha), np.sin(alpha)
    gx, gy = x * ca - y * sa, x * sa + y * ca
    phi = np.arcsin(s) + alpha
    return gx, gy, phi, k * CB, z, t, k


def state_in_frame(gc, alpha, x_plane):
    """Local state (y, z, sin phi, dz/ds, q/pT) of the global circle gc in the frame rotated by alpha at local x = x_plane
    (plain geometry: follow the circle from its reference point to the plane)."""
    gx, gy, phi, kap, z, t, k = gc
    ca, sa = np.cos(alpha), np.sin(alpha)
    lx, ly = gx * ca + gy * sa, -gx * sa + gy * ca          # the point in the local frame
    lphi = phi - alpha
    s0 = np.sin(lphi)
    s1 = s0 + kap * (x_plane - lx)
    if abs(kap) > 1e-12:
        y1 = ly + (np.cos(np.arcsin(s0)) - np.cos(np.arcsin(s1))) / kap
        arc = (np.arcsin(s1) - np.arcsin(s0)) / kap
    else:
        y1 = ly + (x_plane - lx) * s0 / np.sqrt(1 - s0 * s0)
        arc = (x_plane - lx) / np.sqrt(1 - s0 * s0)
    return np.array([y1, z + t * arc, s1, t, k])


# ------------------------------------------------------------------ rotation of a state between sector frames
def test_rotation_equals_the_same_circle_seen_from_the_other_frame():
    rng = np.random.default_rng(0)
    for _ in range(200):
        p, C = rand_state(rng)
        x = rng.uniform(90, 240)
        beta = rng.choice([-1, 1]) * DPHI
        ok, x2, p2, _ = oracle.rotate(x, p, untri(C), beta, CB)
        assert ok
        gc = global_circle(x, p, 0.0)
        ref = state_in_frame(gc, beta, x2)                 # the same circle at the plane the rotation ended on
        assert abs(x2 - (x * np.cos(beta) + p[0] * np.sin(beta))) < 1e-12
        assert np.allclose(p2, ref, rtol=0, atol=1e-11), p2 - ref


def test_rotation_there_and_back_and_group_property():
    rng = np.random.default_rng(1)
    for _ in range(100):
        p, C = rand_state(rng)
        x = rng.uniform(90, 240)
        ok1, x1, p1, c1 = oracle.rotate(x, p, untri(C), DPHI, CB)
        ok2, x2, p2, c2 = oracle.rotate(x1, p1, c1, -DPHI, CB)
        assert ok1 and ok2
        # back in the old frame but at another plane (the point has not moved): same point, direction, covariance of
        # the point-like quantities; compare after propagating back to x
        okp, _, p3, c3, _ = oracle.propagate(x2, p2, c2, x, CB)
        assert okp and np.allclose(p3, p, atol=1e-10) and np.allclose(c3, untri(C), rtol=1e-8, atol=1e-14)
        # two small rotations = one: a + b
        a, b = 0.13, 0.219
        _, xa, pa, ca_ = oracle.rotate(x, p, untri(C), a, CB)
        _, xb, pb, cb_ = oracle.rotate(xa, pa, ca_, b, CB)
        _, xc, pc, cc_ = oracle.rotate(x, p, untri(C), a + b, CB)
        okp, _, pb2, cb2, _ = oracle.propagate(xb, pb, cb_, xc, CB)
        assert okp and np.allclose(pb2, pc, atol=1e-10) and np.allclose(cb2, cc_, rtol=1e-7, atol=1e-14)


def test_rotation_jacobian_vs_finite_differences_of_the_geometry():
    """C' = J C J^T with J = d(state in the new frame at its fixed plane) / d(state in the old frame at its fixed
    plane), J from five-point differences of the plain circle geometry."""
    rng = np.random.default_rng(2)
    for _ in range(50):
        p, C = rand_state(rng)
        x = rng.uniform(90, 240)
        beta = rng.choice([-1, 1]) * DPHI
        ok, x2, p2, c2 = oracle.rotate(x, p, untri(C), beta, CB)
        f = lambda q: state_in_frame(global_circle(x, q, 0.0), beta, x2)
        J = np.zeros((5, 5))
        h = 1e-4
        for j in range(5):
            d = np.zeros(5)
            d[j] = h
            J[:, j] = (-f(p + 2 * d) + 8 * f(p + d) - 8 * f(p - d) + f(p - 2 * d)) / (12 * h)
        ref = J @ C @ J.T
        assert np.allclose(tri(c2), ref, rtol=1e-6, atol=1e-12), np.abs(tri(c2) - ref).max()


def test_rotation_fails_for_tracks_that_do_not_move_along_the_new_x():
    p = np.array([0.0, 0.0, 0.94, 0.0, 0.0])
    assert not oracle.rotate(100.0, p, np.zeros(15), -DPHI, CB)[0]        # sin(phi + 20 deg) > smax
    assert oracle.rotate(100.0, p, np.zeros(15), DPHI, CB)[0]


def test_chi2_is_the_mahalanobis_distance():
    rng = np.random.default_rng(3)
    for _ in range(100):
        _, S = rand_state(rng)
        d = rng.normal(size=5) * 0.05
        ref = float(d @ np.linalg.solve(S, d))
        assert abs(oracle.chi2_5(d, untri(S)) - ref) < 1e-9 * max(1.0, ref)
    assert oracle.chi2_5(np.ones(5), untri(-np.eye(5))) > 1e29         # not positive definite: never a match


# ------------------------------------------------------------------ the merger on events
def hits_of_global_helix(rng, pt, q, phi0, eta, sigma, n_sectors=36, skip=None):
    """Clusters of one primary from the origin in every sector it crosses (plain geometry, fp64), smeared by sigma."""
    kap = -q * 0.299792458e-2 * BZ / pt
    hits = []
    for s in range(18):
        alpha = (s + 0.5) * DPHI
        lphi0 = phi0 - alpha
        s0 = np.sin(lphi0)
        if np.cos(lphi0) <= 0:
            continue
        for r, x in enumerate(ROW_X.astype(np.float64)):
            s1 = s0 + kap * x
            if abs(s1) >= 0.999:
                break
            y = (np.cos(lphi0) - np.sqrt(1 - s1 * s1)) / kap
            if abs(y) > x * np.tan(DPHI / 2):
                continue
            arc = (np.arcsin(s1) - np.arcsin(s0)) / kap
            z = arc * np.sinh(eta)
            if skip and skip(s, r):
                continue
            hits.append((s, r, y + rng.normal() * sigma, z + rng.normal() * sigma))
    return hits


def test_a_track_crossing_a_sector_border_is_merged_and_strangers_are_not():
    rng = np.random.default_rng(5)
    n_cross = n_ok = 0
    chi = []
    for _ in range(60):
        pt, q = rng.uniform(0.35, 1.5), rng.choice([-1, 1])
        hits = hits_of_global_helix(rng, pt, q, rng.uniform(0.2, 6.0), rng.uniform(0.2, 0.8), 0.1)
        ev = datagen.event_from_hits(hits, 36, ROW_X, BZ)
        res = oracle.run_event_merged(ev, None, "double")
        if res.tracks.size != 2 or res.tracks["sector"][0] == res.tracks["sector"][1]:
            continue                                     # (stays in one sector, or a piece is too short to be a track)
        n_cross += 1
        inner = int(np.argmin(res.tracks["first_row"]))
        if res.merge_next[inner] == 1 - inner and res.merge_prev[1 - inner] == inner:
            n_ok += 1
            chi.append(res.merge_chi2[inner])
            assert res.merged_offset.tolist() == [0, 2] and res.merged_segs.tolist() == [inner, 1 - inner]
    assert n_cross >= 20 and n_ok >= 0.9 * n_cross, (n_cross, n_ok)
    assert 2.0 < np.mean(chi) < 9.0, np.mean(chi)        # 5 degrees of freedom, covariances honest: about 5
    # two different particles in neighbouring sectors: nothing to merge
    # (stiff tracks along the centres of sectors 0 and 1; the second one only on the outer rows, so that the row order
    # "outer segment starts above the end of the inner one" would allow a merge - the parameters do not)
    hits = hits_of_global_helix(rng, 5.0, 1, 0.5 * DPHI, 0.4, 0.1, skip=lambda s, r: r >= 70) + \
        hits_of_global_helix(rng, 5.0, 1, 1.5 * DPHI, 0.45, 0.1, skip=lambda s, r: r < 80)
    res = oracle.run_event_merged(datagen.event_from_hits(hits, 36, ROW_X, BZ), None, "double")
    assert res.tracks.size == 2 and set(res.tracks["sector"]) == {0, 1}
    assert np.all(res.merge_next == -1) and res.merged_offset.size == 3


def test_a_gap_the_track_following_did_not_cover_is_merged_inside_the_sector():
    """PAPER.md:45 first case.  A straight-ish track with 12 pad rows removed (max_gap = 4: Phase I ends both
    segments at the hole); the merger joins them; with merge_max_row_gap below the hole it does not."""
    rng = np.random.default_rng(6)
    hits = hits_of_global_helix(rng, 2.0, 1, 0.5 * DPHI, 0.5, 0.1, skip=lambda s, r: 60 <= r < 72)
    ev = datagen.event_from_hits(hits, 36, ROW_X, BZ)
    res = oracle.run_event_merged(ev, None, "double")
    assert res.tracks.size == 2 and set(res.tracks["sector"]) == {0}
    inner = int(np.argmin(res.tracks["first_row"]))
    assert res.tracks["last_row"][inner] == 59 and res.tracks["first_row"][1 - inner] == 72
    assert res.merge_next[inner] == 1 - inner and res.merge_prev[1 - inner] == inner and res.merge_next[1 - inner] == -1
    assert res.merged_offset.tolist() == [0, 2]
    prm = oracle.default_params()
    prm.merge_max_row_gap = 12
    assert np.all(oracle.run_event_merged(ev, prm, "double").merge_next == -1)      # 72 - 59 = 13 rows
    prm.merge_max_row_gap = 13
    assert oracle.run_event_merged(ev, prm, "double").merge_next[inner] == 1 - inner
    prm = oracle.default_params()
    prm.merge_chi2 = 1e-6
    assert np.all(oracle.run_event_merged(ev, prm, "double").merge_next == -1)      # the cut is applied


def test_merge_links_are_mutual_and_chains_partition_the_tracks():
    ev = datagen.config_event(2, seed=1)
    res = oracle.run_event_merged(ev)
    n = res.tracks.size
    nxt, prv = res.merge_next, res.merge_prev
    has = nxt >= 0
    assert has.sum() > 50                                             # a peripheral event has crossings
    assert np.array_equal(prv[nxt[has]], np.nonzero(has)[0])          # mutual
    assert np.unique(nxt[has]).size == has.sum()                      # nobody is continued by two segments
    assert np.array_equal(np.sort(res.merged_segs), np.arange(n))     # every segment in exactly one merged track
    assert res.merged_offset[-1] == n and res.merged_offset.size - 1 == n - has.sum()
    t = res.tracks
    a, b = np.nonzero(has)[0], nxt[has]
    assert np.all(t["first_row"][b] > t["last_row"][a]) and np.all(t["first_row"][b] - t["last_row"][a] <= 40)
    side = t["sector"] // 18
    assert np.all(side[a] == side[b])
    ds = (t["sector"][b] % 18 - t["sector"][a] % 18) % 18
    assert np.all((ds == 0) | (ds == 1) | (ds == 17))
    assert np.all(res.merge_chi2[has] <= 50.0)
    # merging is (almost always) right: the two segments carry the same majority truth label
    def label(i):
        ids = res.cluster_ids[t["cluster_offset"][i]: t["cluster_offset"][i] + t["n_clusters"][i]]
        v, c = np.unique(ev.truth[ids], return_counts=True)
        return v[np.argmax(c)]
    same = sum(label(i) == label(j) for i, j in zip(a, b))
    assert same >= 0.97 * a.size, (same, a.size)
