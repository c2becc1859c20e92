"""The seeded generator (datagen/): shapes and structure of BASELINE.json:configs, determinism."""
import numpy as np

import datagen


def test_default_geometry():
    rx = datagen.default_row_x()
    assert rx.shape == (159,) and abs(rx[0] - 85.2) < 1e-5 and abs(rx[-1] - 246.0) < 1e-4
    d = np.diff(rx.astype(np.float64))
    assert np.all(d > 0) and abs(d[62] - 3.3) < 1e-4 and abs(d[126] - 1.5) < 1e-4


def test_configs_have_the_nominal_sizes_and_are_deterministic():
    nominal = {0: 29e3, 1: 15.5e3, 2: 271e3}
    for i, n in nominal.items():
        a, b = datagen.config_event(i, seed=0), datagen.config_event(i, seed=0)
        assert abs(a.n_clusters - n) < 0.05 * n
        assert np.array_equal(a.y, b.y) and np.array_equal(a.z, b.z) and np.array_equal(a.row_counts, b.row_counts)
        c = datagen.config_event(i, seed=1)
        assert c.n_clusters != a.n_clusters or not np.array_equal(a.y, c.y)


def test_structure_sides_acceptance_noise_and_shuffle():
    ev = datagen.config_event(2, seed=0)
    sec, row = ev.sector_row()
    side = np.where(sec < 18, 1.0, -1.0)
    trk = ev.truth >= 0
    # z on the sector's side (up to the 0.1 cm smear), |y| within the 20-degree sector up to the smear
    assert np.all(ev.z[trk] * side[trk] > -0.6)
    assert np.all(np.abs(ev.y[trk]) <= ev.row_x[row[trk]] * np.tan(np.pi / 18) + 0.6)
    frac = (~trk).sum() / trk.sum()
    assert abs(frac - 0.10) < 0.002
    # one cluster per (track, sector, row)
    key = (ev.truth[trk].astype(np.int64) * 36 + sec[trk]) * 159 + row[trk]
    assert np.unique(key).size == key.size
    # load index carries no track information: within rows, truth ids are not sorted
    base = ev.row_base
    big = np.argmax(ev.row_counts.reshape(-1))
    t = ev.truth[base[big]:base[big + 1]]
    assert not np.all(np.diff(t[t >= 0]) >= 0)


def test_time_frame_overlaps_events_with_z_offsets():
    ev = datagen.generate(0, n_events=3, n_primaries=200, n_secondaries=20, pt_mode=1, z_shift=1, noise_frac=0.2)
    assert np.unique(ev.tracks[:, 7]).size == 3 and ev.tracks[:, 7].max() < 250
    sec, _ = ev.sector_row()
    assert ev.z[sec < 18].min() < -20 and ev.z[sec >= 18].max() > 20   # apparent z crosses the central electrode


def test_event_from_hits_keeps_load_order():
    ev = datagen.event_from_hits([(0, 1, 1.0, 2.0), (0, 0, 3.0, 4.0), (0, 1, 5.0, 6.0)], 1, datagen.default_row_x()[:3])
    assert ev.row_counts.tolist() == [[1, 2, 0]] and ev.y.tolist() == [3.0, 1.0, 5.0]
