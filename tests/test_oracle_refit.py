"""Pins for the oracle's final track fit (S8; "the full track is refit using the full Kalman
filter.  A polynomial approximation of the magnetic field avoids the slow memory access to a field map").

The refit is an iteration, so the oracle follows it step by step; what it must reach is pinned from outside: the
analytic helix for noise-free tracks across a sector border, unit pulls for noisy ones, the Phase-I estimate where both
see the same clusters, tracks integrated numerically (RK4) through a field that falls off with r^2, and tracks that
scatter in the gas by the angles the Highland formula gives (simulated from first principles: kicks in azimuth and dip).
"""
import numpy as np
import pytest

import datagen
import oracle
from helpers import CB_PER_T, tri
from test_oracle_merge import BZ, DPHI, ROW_X, hits_of_global_helix

CB = CB_PER_T * BZ


def truth_state(pt, q, phi0, eta, sector, x):
    """Local state (y, z, sin phi, dz/ds, q/pT) at local x of a primary from the origin, in the frame of `sector`."""
    kap = -q * 0.299792458e-2 * BZ / pt
    lphi0 = phi0 - (sector % 18 + 0.5) * DPHI
    s0 = np.sin(lphi0)
    s1 = s0 + kap * x
    y = (np.cos(lphi0) - np.sqrt(1 - s1 * s1)) / kap
    arc = (np.arcsin(s1) - np.arcsin(s0)) / kap
    return np.array([y, arc * np.sinh(eta), s1, np.sinh(eta), kap / CB])


def crossing_events(rng, n, sigma):
    out = []
    while len(out) < n:
        pt, q = rng.uniform(0.4, 1.5), rng.choice([-1, 1])
        phi0, eta = rng.uniform(0.2, 6.0), rng.uniform(0.2, 0.8)
        hits = hits_of_global_helix(rng, pt, q, phi0, eta, sigma)
        ev = datagen.event_from_hits(hits, 36, ROW_X, BZ)
        res = oracle.run_event_refit(ev, None, "double")
        if res.tracks.size == 2 and res.merged_offset.size == 2 and res.refits[0]["ok"]:
            out.append((ev, res, (pt, q, phi0, eta)))
    return out


def test_noise_free_tracks_across_a_sector_border_are_recovered():
    rng = np.random.default_rng(11)
    for ev, res, (pt, q, phi0, eta) in crossing_events(rng, 15, 0.0):
        r = res.refits[0]
        assert r["n_fit"] == res.tracks["n_clusters"].sum() - 1          # every cluster but the starting one
        inner = res.tracks[r["first_track"]]
        assert r["sector"] == inner["sector"] and abs(r["x"] - ROW_X[inner["first_row"]]) < 1e-6
        ref = truth_state(pt, q, phi0, eta, r["sector"], r["x"])
        err = np.abs(r["p"] - ref)
        err[4] /= 10.0
        assert err.max() < 2e-5, err               # inputs are fp32-rounded


def test_pulls_of_merged_tracks_and_gain_over_one_segment():
    rng = np.random.default_rng(12)
    pulls, gain = [], []
    for ev, res, (pt, q, phi0, eta) in crossing_events(rng, 250, 0.1):
        r = res.refits[0]
        ref = truth_state(pt, q, phi0, eta, r["sector"], r["x"])
        C = tri(r["c"])
        pulls.append((r["p"] - ref) / np.sqrt(np.diag(C)))
        inner = res.tracks[r["first_track"]]
        if abs(inner["x"] - r["x"]) < 1e-6:
            gain.append(tri(inner["c"])[4, 4] / C[4, 4])
    pulls = np.array(pulls)
    rms = np.sqrt((pulls ** 2).mean(axis=0))
    assert np.all(rms > 0.85) and np.all(rms < 1.2), rms
    assert np.all(np.abs(pulls.mean(axis=0)) < 4.0 / np.sqrt(len(pulls))), pulls.mean(axis=0)
    # the merged track's lever arm is longer than its inner segment's: the variance of q/pT shrinks
    assert np.median(gain) > 2.0, np.median(gain)


def test_one_segment_refit_equals_the_phase_one_estimate():
    """Same clusters, same model, other starting point of the linearisation: the two least-squares estimates agree to a
    small fraction of their standard deviation."""
    ev = datagen.config_event(1, seed=3)
    res = oracle.run_event_refit(ev, None, "double")
    n = 0
    for m in range(res.refits.size):
        if res.merged_offset[m + 1] - res.merged_offset[m] != 1 or not res.refits[m]["ok"]:
            continue
        t, r = res.tracks[res.refits[m]["first_track"]], res.refits[m]
        if abs(t["x"] - r["x"]) > 1e-6 or t["n_clusters"] < 30:
            continue
        sig = np.sqrt(np.diag(tri(t["c"])))
        assert np.all(np.abs(r["p"] - t["p"]) < 0.05 * sig), (r["p"] - t["p"]) / sig
        assert np.allclose(r["c"], t["c"], rtol=0.05, atol=1e-9)
        n += 1
    assert n >= 20


def rk4_track(pt, q, y0, s0, t, ar, rows_x, z0=20.0, h=0.05):
    """Hits of a track in sector-local coordinates integrated through Bz(r) = BZ (1 + ar r^2) with RK4 in x."""
    k = q / pt

    def f(x, u):
        y, s, z = u
        c = np.sqrt(1 - s * s)
        kap = k * CB * (1 + ar * (x * x + y * y))
        return np.array([s / c, kap, t / c])
    x, u = float(rows_x[0]), np.array([y0, s0, z0])
    out = [(x, u[0], u[2], u[1])]
    for xr in rows_x[1:]:
        nstep = max(1, int(np.ceil((xr - x) / h)))
        hh = (xr - x) / nstep
        for _ in range(nstep):
            k1 = f(x, u); k2 = f(x + hh / 2, u + hh / 2 * k1); k3 = f(x + hh / 2, u + hh / 2 * k2); k4 = f(x + hh, u + hh * k3)
            u = u + hh / 6 * (k1 + 2 * k2 + 2 * k3 + k4)
            x += hh
        out.append((xr, u[0], u[2], u[1]))
    return out, k


def test_polynomial_field_is_used():
    """Tracks integrated through a field that falls by 12 % from the axis to r = 250 cm.  Refit with the matching
    polynomial: q/pT unbiased within its errors; refit with the constant field: biased by several standard deviations."""
    rng = np.random.default_rng(13)
    ar = -2.0e-6
    x = ROW_X.astype(np.float64)
    pull_poly, pull_const = [], []
    for _ in range(60):
        pt, q = rng.uniform(1.5, 3.0), rng.choice([-1, 1])
        pts, k = rk4_track(pt, q, rng.uniform(-3, 3), rng.uniform(-0.05, 0.05), rng.uniform(-0.5, 0.5), ar, x)
        hits = [(0, r, yy + rng.normal() * 0.1, zz + rng.normal() * 0.1) for r, (xx, yy, zz, ss) in enumerate(pts)
                if abs(yy) < xx * np.tan(DPHI / 2)]
        ev = datagen.event_from_hits(hits, 36, ROW_X, BZ)
        for a, acc in ((ar, pull_poly), (0.0, pull_const)):
            prm = oracle.default_params()
            prm.field_ar = a
            res = oracle.run_event_refit(ev, prm, "double")
            if res.refits.size != 1 or not res.refits[0]["ok"] or res.refits[0]["n_fit"] < 100:
                continue
            r = res.refits[0]
            acc.append((r["p"][4] - k) / np.sqrt(r["c"][14]))
    assert len(pull_poly) >= 40 and len(pull_const) >= 40
    rms = lambda v: float(np.sqrt(np.mean(np.square(v))))
    assert abs(np.mean(pull_poly)) < 0.5 and rms(pull_poly) < 1.5, (np.mean(pull_poly), rms(pull_poly))
    assert rms(pull_const) > 3.0, rms(pull_const)           # (the bias has the sign of the charge)


def scattered_track(rng, pt, q, y0, s0, t, x0_inv, rows_x, z0=20.0):
    """Helix steps between pad rows with a multiple-scattering kick after each step: theta0 = 0.0136 / p sqrt(L / X0)
    (Highland without the log term), split into two orthogonal plane angles; the azimuth turns by theta1 / cos(lambda),
    the dip by theta2."""
    k = q / pt
    y, s, z, tt = y0, s0, z0, t
    out = [(y, z)]
    for i in range(1, len(rows_x)):
        dx = rows_x[i] - rows_x[i - 1]
        kap = k * CB
        s2 = s + kap * dx
        c, c2 = np.sqrt(1 - s * s), np.sqrt(1 - s2 * s2)
        dy = dx * (s + s2) / (c + c2)
        arc = (np.arcsin(s2) - np.arcsin(s)) / kap
        y, z, s = y + dy, z + tt * arc, s2
        out.append((y, z))
        L = abs(arc) * np.sqrt(1 + tt * tt)
        p = np.sqrt(1 + tt * tt) / abs(k)
        th0 = 0.0136 / p * np.sqrt(L * x0_inv)
        th1, th2 = rng.normal() * th0, rng.normal() * th0
        lam = np.arctan(tt)
        phi = np.arcsin(s) + th1 / np.cos(lam)
        lam2 = lam + th2
        k = k * np.cos(lam) / np.cos(lam2)              # |p| unchanged: q/pT = (q/p) / cos(lambda)
        s, tt = np.sin(phi), np.tan(lam2)
    return out, k, s, tt


def test_scattering_covariance_equals_sampled_kicks():
    """The covariance the oracle adds for a path L == the sample covariance of (sin phi, dz/ds, q/pT) after random
    kicks: azimuth turned by theta1 / cos(lambda), dip by theta2, |p| unchanged (first principles, 400k samples)."""
    rng = np.random.default_rng(15)
    for s, t, k in ((0.3, 0.9, 2.0), (-0.5, -0.4, -1.2), (0.0, 1.5, 0.7)):
        L, x0_inv = 40.0, 1.0 / 300.0
        p_inv = abs(k) / np.sqrt(1 + t * t)
        th0 = 0.0136 * p_inv * np.sqrt(L * x0_inv)
        n = 400000
        th1, th2 = rng.normal(size=n) * th0, rng.normal(size=n) * th0
        lam = np.arctan(t)
        s_new = np.sin(np.arcsin(s) + th1 / np.cos(lam))
        t_new = np.tan(lam + th2)
        k_new = k * np.cos(lam) / np.cos(lam + th2)
        ref = np.cov(np.stack([s_new, t_new, k_new]))
        c = tri(oracle.scatter([0.0, 0.0, s, t, k], np.zeros(15), L, x0_inv))[2:, 2:]
        assert np.allclose(c, ref, rtol=0.03, atol=1e-2 * th0 * th0), (c, ref)
        assert np.all(tri(oracle.scatter([0.0, 0.0, s, t, k], np.zeros(15), L, 0.0)) == 0)


def test_multiple_scattering_noise_gives_unit_pulls():
    """Soft tracks in a dense 'gas' (X0 = 300 cm): with the matching process noise the refit's pulls are ~1, without
    it the covariance is far too small."""
    rng = np.random.default_rng(14)
    x0_inv = 1.0 / 300.0
    x = ROW_X.astype(np.float64)[:100]
    pulls = {True: [], False: []}
    for _ in range(300):
        pt, q = rng.uniform(0.5, 0.9), rng.choice([-1, 1])
        y0, s0, t = rng.uniform(-2, 2), rng.uniform(-0.05, 0.05), rng.choice([-1, 1]) * rng.uniform(0.8, 1.1)   # steep in z: the (1+t^2) factors count
        pts, k_end, s_end, t_end = scattered_track(rng, pt, q, y0, s0, t, x0_inv, x)
        hits = [(0, r, yy + rng.normal() * 0.1, zz + rng.normal() * 0.1) for r, (yy, zz) in enumerate(pts)
                if abs(yy) < x[r] * np.tan(DPHI / 2)]
        ev = datagen.event_from_hits(hits, 36, ROW_X, BZ)
        for with_ms in (True, False):
            prm = oracle.default_params()
            prm.ms_x0_inv = x0_inv if with_ms else 0.0
            res = oracle.run_event_refit(ev, prm, "double")
            if res.refits.size != 1 or not res.refits[0]["ok"] or res.refits[0]["n_fit"] < 60 or res.refits[0]["x"] > x[0] + 1e-6:
                continue
            r = res.refits[0]
            ref = np.array([y0, 20.0, s0, t, q / pt])          # the state at the innermost row (before any scattering)
            pulls[with_ms].append((r["p"] - ref) / np.sqrt(np.diag(tri(r["c"]))))
    a, b = np.array(pulls[True]), np.array(pulls[False])
    assert len(a) >= 150 and len(b) >= 150
    rms_a, rms_b = np.sqrt((a ** 2).mean(axis=0)), np.sqrt((b ** 2).mean(axis=0))
    assert np.all(rms_a[2:] > 0.8) and np.all(rms_a[2:] < 1.2), rms_a
    assert np.all(rms_b[2:] > 1.6), rms_b
