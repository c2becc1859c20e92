"""Pins for the control logic of the oracle's tracklet constructor and selector (S5 steps 2-5, S6).

The paper gives no formula for these ("extrapolates the track ... adding the closest cluster in
each ... row"; :43 "best instance is selected"), so every rule is a DESIGN.md reading; each test below fails for a
plausible slip in oracle/tpc_oracle.cpp (off-by-one in the gap counter, a counter shared between legs, a search inside
leg C, 9 instead of 10 hits, a road without the measurement variance, a circular road, a lost tie-break, a wrong
re-initialisation of the inward pass).  Hand-made tracks on exact lattices; expected values come from counting rows
by hand, from the closed-form covariance of a linear fit, or from an independent numpy filter (trigonometric circle
propagation + finite-difference Jacobian) - never from the oracle itself.
"""
import numpy as np
import pytest

import datagen
import oracle
from helpers import CB_PER_T, helix_hits, state_at, tri

ROW_X = datagen.default_row_x()
Y0, Z0, DZ = 0.0, 40.0, 0.25     # the straight test track: y = 0, z = 40 + 0.25 * (x - x_0), all exact in fp32


def line_hits(rows, y=Y0, sector=0):
    return [(sector, int(r), float(y), float(np.float32(Z0 + DZ * (float(ROW_X[r]) - float(ROW_X[0]))))) for r in rows]


def run(hits, params=None, bz=0.0, precision="double", n_sectors=1):
    ev = datagen.event_from_hits(hits, n_sectors, ROW_X, bz)
    return ev, oracle.run_event(ev, params, precision)


def tracklet_of_start_row(res, row):
    i = np.nonzero(res.tracklets["start_row"] == row)[0]
    assert i.size == 1, (row, res.tracklets["start_row"])
    return res.tracklets[i[0]], res.row_hit[i[0]]


# ------------------------------------------------------------------ gaps: leg B (outward), S5 step 3
@pytest.mark.parametrize("hole,bridged", [(0, True), (1, True), (4, True), (5, False), (6, False)])
def test_leg_b_bridges_max_gap_empty_rows_and_stops_at_the_next(hole, bridged):
    """Rows 9..30 hold the track (chain 10..29, row 30 taken by the first search), then `hole` empty rows, then two
    more hits (too few for a seed of their own).  max_gap = 4: four empty rows are crossed, the fifth ends the leg."""
    far = [31 + hole, 32 + hole]
    ev, res = run(line_hits(list(range(9, 31)) + far))
    assert res.start_hits.size == 1
    t, rh = tracklet_of_start_row(res, 10)
    assert t["last_row"] == (far[1] if bridged else 30)
    assert t["n_hits"] == 22 + (2 if bridged else 0)
    assert (rh[far[0]] >= 0) == bridged and (rh[far[1]] >= 0) == bridged
    assert np.all(rh[31:31 + hole] == -1)


def test_max_gap_parameter_is_the_number_of_empty_rows_crossed():
    prm = oracle.default_params()
    prm.max_gap = 2
    for hole, bridged in ((2, True), (3, False)):
        _, res = run(line_hits(list(range(9, 31)) + [31 + hole, 32 + hole]), prm)
        t, _ = tracklet_of_start_row(res, 10)
        assert (t["last_row"] > 30) == bridged


# ------------------------------------------------------------------ gaps: leg D (inward, below the seed), step 4
@pytest.mark.parametrize("hole,bridged", [(4, True), (5, False)])
def test_leg_d_counts_gaps_from_zero_at_the_seed_row(hole, bridged):
    """Track on rows 40..60 and 64..66; row 39 holds only a hit 0.9 cm beside the line: near enough to give the hit of
    row 40 its (non-reciprocal) down-link, so that row 40 is the start hit (r0 = 40), but outside leg D's ~0.5 cm
    road, so the first row below the seed is already a row without hit.  `hole` such rows (39 and the empty ones
    below), then two more hits.  Leg B bridged a 3-row hole (61..63) on the way out and leg C passes it on the way in:
    were the counter shared between the legs, counted inside leg C, or not restarted at r0, the 4-row hole below the
    seed would not be crossed (3 + 4 > max_gap)."""
    upper = list(range(40, 61)) + [64, 65, 66]          # 64..66: picked up by leg B, no seed of their own
    low = [39 - hole, 38 - hole]
    ev, res = run(line_hits(upper + low) + line_hits([39], y=0.9))
    assert res.start_hits.size == 1
    t, rh = tracklet_of_start_row(res, 40)
    assert t["last_row"] == 66 and np.all(rh[61:64] == -1) and np.all(rh[64:67] >= 0)
    assert rh[39] == -1
    assert t["first_row"] == (low[1] if bridged else 40)
    assert t["n_hits"] == 24 + (2 if bridged else 0)
    # the inward pass updates with every assigned hit except the outermost one (its starting point)
    assert t["n_fit"] == t["n_hits"] - 1


def test_leg_c_does_not_search_rows_the_outward_pass_left_empty():
    """A decoy in row 62, 1.0 cm beside the track: outside leg B's road there (4*sqrt(C_yy + err2) ~ 0.5 cm after 20
    hits) but inside leg C's (the inward pass has only seen rows 66..64 when it crosses row 62, C_yy is still large
    and the road is capped at road_max = 2 cm).  S5 step 4: between r0 and the top, rows without a hit are neither
    searched nor counted as gaps - the decoy must not be picked up."""
    upper = list(range(40, 61)) + [64, 65, 66]
    hits = line_hits(upper) + line_hits([62], y=1.0)
    ev, res = run(hits)
    t, rh = tracklet_of_start_row(res, 41)
    assert rh[62] == -1 and t["n_hits"] == 24 and t["last_row"] == 66
    # (the same decoy 0.2 cm beside the track IS taken, by leg B: the search itself works in that row)
    _, res2 = run(line_hits(upper) + line_hits([62], y=0.2))
    t2, rh2 = tracklet_of_start_row(res2, 41)
    assert rh2[62] == 0 and t2["n_hits"] == 25


# ------------------------------------------------------------------ min_hits: kept tracklets and owned hits (S5.5, S6)
@pytest.mark.parametrize("n,kept", [(9, False), (10, True), (11, True)])
def test_a_tracklet_needs_min_hits_hits(n, kept):
    _, res = run(line_hits(range(20, 20 + n)))
    assert res.tracklets.size == 1 and res.tracklets[0]["n_hits"] == n
    assert bool(res.tracklets[0]["kept"]) == kept
    assert res.tracks.size == (1 if kept else 0)
    if kept:
        assert res.tracks[0]["n_clusters"] == n
    prm = oracle.default_params()
    prm.min_hits = n + 1
    assert run(line_hits(range(20, 20 + n)), prm)[1].tracks.size == 0
    prm.min_hits = n
    assert run(line_hits(range(20, 20 + n)), prm)[1].tracks.size == 1


@pytest.mark.parametrize("k,emitted", [(9, False), (10, True)])
def test_a_track_needs_min_hits_owned_hits(k, emitted):
    """Track 1 on rows 1..40 at y = 0; track 2 runs 0.3 cm beside it on rows 1..k and ends there.  Tracklet 2 follows
    its own k hits, then - the road is ~0.5 cm - track 1's hits up to row 40: both tracklets have 40 hits, the tie goes
    to the smaller start-hit id (track 1 is loaded first), so tracklet 2 owns exactly its own k hits."""
    hits = []
    for r in range(1, 41):
        hits += line_hits([r])
        if r <= k:
            hits += line_hits([r], y=0.3)
    ev, res = run(hits)
    assert res.tracklets.size == 2 and np.all(res.tracklets["n_hits"] == 40) and np.all(res.tracklets["kept"] == 1)
    assert res.tracks.size == (2 if emitted else 1)
    first = res.tracks[np.argmin(res.tracks["start_gid"])]
    assert first["n_clusters"] == 40
    if emitted:
        second = res.tracks[np.argmax(res.tracks["start_gid"])]
        ids = res.cluster_ids[second["cluster_offset"]: second["cluster_offset"] + second["n_clusters"]]
        assert second["n_clusters"] == k and np.allclose(ev.y[ids], 0.3)
        assert second["first_row"] == 1 and second["last_row"] == k
    assert np.unique(res.cluster_ids).size == res.cluster_ids.size          # one hypothesis per hit


# ------------------------------------------------------------------ road size and shape (S5 step 3, R-7)
def linear_fit_variance(x_hits, x_pred, e2, slope_var0):
    """Variance of the predicted coordinate at x_pred of a straight-line fit: the first hit enters as the prior
    (variance e2 on the intercept, slope_var0 on the slope), the others as measurements of variance e2.
    Information form, nothing recursive: P = (P0^-1 + sum h h^T / e2)^-1, var = (1, dx) P (1, dx)^T."""
    x0 = x_hits[0]
    info = np.diag([1.0 / e2, 1.0 / slope_var0])
    for x in x_hits[1:]:
        h = np.array([1.0, x - x0])
        info += np.outer(h, h) / e2
    P = np.linalg.inv(info)
    g = np.array([1.0, x_pred - x0])
    return float(g @ P @ g)


def probe_event(dy, dz):
    """Chain on rows 10..15 (hits on rows 9..15), one probe hit in row 16 displaced by (dy, dz) from the line."""
    hits = line_hits(range(9, 16))
    zline = Z0 + DZ * (float(ROW_X[16]) - float(ROW_X[0]))
    hits.append((0, 16, float(np.float32(dy)), float(np.float32(zline + dz))))
    return hits


EPS = 3e-5      # [cm] z ~ 43 cm is stored in fp32 (ulp 4e-6) and the fitted line carries that rounding


def below(v):
    return float(v - EPS)


def above(v):
    return float(v + EPS)


def test_road_is_nsig_sigma_of_prediction_plus_measurement_and_rectangular():
    """Bz = 0, track along x: the filter is exactly linear, so the predicted variances at row 16 are those of a
    straight-line fit through rows 10..15 (slope priors css0 = 1 on sin(phi) = dy/dx, ctt0 = 10 on dz/ds = dz/dx).
    A hit at road -/+ epsilon is taken / not taken; so is one in the corner of the rectangle (outside the ellipse)."""
    prm = oracle.default_params()
    xs = ROW_X[10:16].astype(np.float64)
    x16 = float(ROW_X[16])
    cyy = linear_fit_variance(xs, x16, prm.err2_y, prm.kf_css0)
    czz = linear_fit_variance(xs, x16, prm.err2_z, prm.kf_ctt0)
    ry = prm.road_nsig * np.sqrt(cyy + prm.err2_y)
    rz = prm.road_nsig * np.sqrt(czz + prm.err2_z)
    assert 0.4 < ry < 1.0 and 0.4 < rz < 1.0 and ry < prm.road_max          # (not capped: this pins the formula)
    assert prm.road_nsig * np.sqrt(cyy) < 0.9 * ry                            # dropping err2 would move the edge by > 10 %

    def taken(dy, dz):
        _, res = run(probe_event(dy, dz))
        t, rh = tracklet_of_start_row(res, 10)
        return rh[16] == 0

    for sgn in (1.0, -1.0):
        assert taken(sgn * below(ry), 0.0) and not taken(sgn * above(ry), 0.0)
        assert taken(0.0, sgn * below(rz)) and not taken(0.0, sgn * above(rz))
    assert taken(0.95 * ry, 0.95 * rz) and taken(-0.95 * ry, 0.95 * rz)        # rectangle, not ellipse
    assert not taken(above(ry), 0.5 * rz) and not taken(0.5 * ry, -above(rz))


def test_road_is_capped_at_road_max():
    prm = oracle.default_params()
    prm.road_nsig = 20.0           # 20 sigma of the prediction at row 16 is > 2 cm in both coordinates
    xs = ROW_X[10:16].astype(np.float64)
    assert prm.road_nsig * np.sqrt(linear_fit_variance(xs, float(ROW_X[16]), prm.err2_y, prm.kf_css0) + prm.err2_y) > 2.05

    def taken(dy, dz):
        _, res = run(probe_event(dy, dz), prm)
        return tracklet_of_start_row(res, 10)[1][16] == 0

    assert taken(below(2.0), 0.0) and not taken(above(2.0), 0.0)
    assert taken(0.0, -below(2.0)) and not taken(0.0, -above(2.0))
    prm.road_max = 1.0
    assert taken(below(1.0), below(1.0)) and not taken(above(1.0), 0.0)


def test_closest_hit_wins_and_equal_distances_go_to_the_smaller_load_index():
    """Row 32 holds two hits at y = +1.5 and y = -1.5 around a prediction at exactly y = 0 (all hits on the line have
    y = 0, so the fitted y and sin(phi) stay exactly 0): equal distances, the smaller load index wins whatever the
    order in which the grid visits them (they sit in different bins; the one at -1.5 is visited first)."""
    prm = oracle.default_params()
    prm.road_nsig = 40.0           # road = road_max = 2 cm
    zl = lambda r: float(np.float32(Z0 + DZ * (float(ROW_X[r]) - float(ROW_X[0]))))
    for first, second in ((1.5, -1.5), (-1.5, 1.5)):
        hits = line_hits(range(9, 31)) + [(0, 32, first, zl(32)), (0, 32, second, zl(32))]
        for brute in (False, True):
            ev = datagen.event_from_hits(hits, 1, ROW_X, 0.0)
            res = oracle.Oracle(1, ev.n_rows, ev.row_x, 0.0, prm, "double").run(ev.row_counts, ev.y, ev.z, brute)
            t, rh = tracklet_of_start_row(res, 10)
            assert rh[32] == 0, (first, brute)
    # and a strictly closer hit wins whatever its index
    hits = line_hits(range(9, 31)) + [(0, 32, 1.5, zl(32)), (0, 32, -1.25, zl(32)), (0, 32, 1.75, zl(32))]
    _, res = run(hits, prm)
    assert tracklet_of_start_row(res, 10)[1][32] == 1


# ------------------------------------------------------------------ the inward pass: independent numpy filter
def numpy_propagate(p, C, x, x2, bz):
    """Exact circle transport of (y, z, sin phi, dz/ds, q/pT) with trigonometric formulas (helpers.state_at) and a
    five-point finite-difference Jacobian: a different route to the same model than the oracle's algebraic one."""
    f = lambda q: state_at(x2, x, q[0], q[1], q[2], q[3], q[4], bz)
    J = np.zeros((5, 5))
    h = 1e-4     # five-point stencil: truncation ~h^4, and large enough for the (cos - cos) / kappa cancellation
    for j in range(5):
        d = np.zeros(5)
        d[j] = h
        J[:, j] = (-f(p + 2 * d) + 8 * f(p + d) - 8 * f(p - d) + f(p - 2 * d)) / (12 * h)
    return f(p), J @ C @ J.T


def numpy_update(p, C, chi2, ym, zm, e2y, e2z):
    for i, m, e2 in ((0, ym, e2y), (1, zm, e2z)):
        H = np.zeros(5)
        H[i] = 1.0
        S = C[i, i] + e2
        K = C[:, i] / S
        r = m - p[i]
        p = p + K * r
        C = C - np.outer(K, H @ C)
        chi2 += r * r / S
    return p, C, chi2


@pytest.mark.parametrize("with_decoy", [False, True])
def test_output_state_is_the_inward_filter_restarted_at_the_outermost_hit(with_decoy):
    """S5 steps 1, 2, 4 replayed by an independent numpy filter on noisy single helices whose hits are all assigned:
    outward pass from the first link (direction from the first two hits, q/pT = 0, diagonal prior), remember
    (sin phi, dz/ds, q/pT) after the update with the outermost hit, restart there at that hit's coordinates with the
    diagonal prior and chi2 = 0, filter inward.  A different restart (state before the update, fitted instead of
    measured y/z, covariance or chi2 not reset) moves the result by ~1e-3, the test allows 2e-6."""
    rng = np.random.default_rng(21)
    prm = oracle.default_params()
    bz = 0.5
    checked = 0
    for _ in range(16):
        pt = 0.4 * 10 ** rng.uniform(0, 1)
        k = rng.choice([-1.0, 1.0]) / pt
        rows, y, z = helix_hits(ROW_X, float(ROW_X[0]), rng.uniform(-5, 5), rng.uniform(20, 90), rng.uniform(-0.2, 0.2),
                                rng.uniform(-0.7, 0.7), k, bz, smax=0.6)
        rows, y, z = rows[5:75], y[5:75], z[5:75]            # no pitch jump needed: rows 5..74
        if rows.size < 70:
            continue
        y = (y + rng.normal(size=y.size) * 0.1).astype(np.float32)
        z = (z + rng.normal(size=z.size) * 0.1).astype(np.float32)
        hits = [(0, int(r), float(a), float(b)) for r, a, b in zip(rows, y, z)]
        if with_decoy:
            # a hit 0.7 cm beside the track in the row above its last hit: the last hit gets a (non-reciprocal) up-link,
            # so the link chain - leg A - reaches it, and leg B finds nothing (the decoy is outside the road): the
            # restart then takes (sin phi, dz/ds, q/pT) as leg A left them
            hits.append((0, int(rows[-1]) + 1, float(y[-1]) + 0.7, float(z[-1])))
        ev = datagen.event_from_hits(hits, 1, ROW_X, bz)
        res = oracle.run_event(ev, None, "double")
        full = [i for i in range(res.tracklets.size) if res.tracklets[i]["n_hits"] == rows.size]
        if not full:
            continue                                        # (a noisy chain may split; only fully assigned ones pin)
        t = res.tracklets[full[0]]
        r0 = int(t["start_row"])
        x = ROW_X.astype(np.float64)
        yy = dict(zip(rows.tolist(), y.astype(np.float64)))
        zz = dict(zip(rows.tolist(), z.astype(np.float64)))
        # outward pass from r0
        dx, dy, dz = x[r0 + 1] - x[r0], yy[r0 + 1] - yy[r0], zz[r0 + 1] - zz[r0]
        ell = np.hypot(dx, dy)
        p = np.array([yy[r0], zz[r0], dy / ell, dz / ell, 0.0])
        C0 = np.diag([prm.err2_y, prm.err2_z, prm.kf_css0, prm.kf_ctt0, prm.kf_ckk0])
        C, chi2 = C0.copy(), 0.0
        for r in range(r0 + 1, int(rows[-1]) + 1):
            p, C = numpy_propagate(p, C, x[r - 1], x[r], bz)
            p, C, chi2 = numpy_update(p, C, chi2, yy[r], zz[r], prm.err2_y, prm.err2_z)
        top = int(rows[-1])
        p = np.array([yy[top], zz[top], p[2], p[3], p[4]])
        C, chi2, nfit = C0.copy(), 0.0, 0
        for r in range(top - 1, int(rows[0]) - 1, -1):
            p, C = numpy_propagate(p, C, x[r + 1], x[r], bz)
            p, C, chi2 = numpy_update(p, C, chi2, yy[r], zz[r], prm.err2_y, prm.err2_z)
            nfit += 1
        assert t["n_fit"] == nfit and t["first_row"] == rows[0] and t["last_row"] == top
        assert abs(t["x"] - x[int(rows[0])]) < 1e-6
        scale = np.array([1.0, 1.0, 1.0, 1.0, 10.0])
        assert np.all(np.abs(t["p"] - p) < 2e-6 * scale), t["p"] - p
        Cref = np.array([C[i, j] for i in range(5) for j in range(i + 1)])
        assert np.allclose(t["c"], Cref, rtol=2e-4, atol=1e-9), np.abs(t["c"] - Cref).max()
        assert abs(t["chi2"] - chi2) < 1e-4 * max(1.0, chi2)
        checked += 1
    assert checked >= 6
