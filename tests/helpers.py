"""Closed-form helpers for the pins: analytic helices in the sector-local frame (numpy, fp64).

Independent of oracle/ and of the CUDA path: plain circle geometry, used as the 'other thing' the
oracle is pinned to.
"""
import numpy as np

CB_PER_T = -0.299792458e-2


def helix_hits(row_x, x0, y0, z0, s0, t, k, bz, smax=0.9):
    """Exact crossings of a circle (curvature kappa = k*CB) with the pad rows.

    State at x0: y0, z0, s0 = sin(phi), t = dz/ds (s = arc length in xy), k = q/pT.
    Returns rows, y, z (fp64) for rows where |sin phi| < smax on the whole way from x0.
    """
    kap = k * CB_PER_T * bz
    rows, ys, zs = [], [], []
    phi0 = np.arcsin(s0)
    for r, x in enumerate(np.asarray(row_x, dtype=np.float64)):
        s = s0 + kap * (x - x0)
        if abs(s) >= smax:
            continue
        phi = np.arcsin(s)
        if abs(kap) > 1e-14:
            y = y0 + (np.cos(phi0) - np.cos(phi)) / kap
            arc = (phi - phi0) / kap
        else:
            y = y0 + (x - x0) * s0 / np.sqrt(1 - s0 * s0)
            arc = (x - x0) / np.sqrt(1 - s0 * s0)
        rows.append(r)
        ys.append(y)
        zs.append(z0 + t * arc)
    return np.array(rows), np.array(ys), np.array(zs)


def state_at(x, x0, y0, z0, s0, t, k, bz):
    """Exact state (y,z,s,t,k) of the same helix at x."""
    kap = k * CB_PER_T * bz
    s = s0 + kap * (x - x0)
    phi0, phi = np.arcsin(s0), np.arcsin(s)
    if abs(kap) > 1e-14:
        y = y0 + (np.cos(phi0) - np.cos(phi)) / kap
        arc = (phi - phi0) / kap
    else:
        y = y0 + (x - x0) * s0 / np.sqrt(1 - s0 * s0)
        arc = (x - x0) / np.sqrt(1 - s0 * s0)
    return np.array([y, z0 + t * arc, s, t, k])


def tri(c15):
    """15-element lower triangle -> full 5x5."""
    m = np.zeros((5, 5))
    k = 0
    for i in range(5):
        for j in range(i + 1):
            m[i, j] = m[j, i] = c15[k]
            k += 1
    return m


def untri(m):
    return np.array([m[i, j] for i in range(5) for j in range(i + 1)])
