"""Input generators (fdc_inputs): machine-independent math, DB closed forms (pin P5), phantoms."""
import math

import numpy as np
import pytest

import fdc_inputs as fi


def test_det_math_matches_libm():
    L = fi._load()
    rng = np.random.default_rng(7)
    for x in np.concatenate([rng.uniform(1e-6, 1.0, 200), rng.uniform(1.0, 300.0, 200)]):
        assert abs(L.fdcgen_ln(x) - math.log(x)) <= 4e-16 * max(1.0, abs(math.log(x)))
    for x in rng.uniform(-20.0, 20.0, 400):
        assert abs(L.fdcgen_exp(x) / math.exp(x) - 1.0) < 1e-14
    for x in rng.uniform(-10.0, 10.0, 400):
        assert abs(L.fdcgen_sin(x) - math.sin(x)) < 1e-15
        assert abs(L.fdcgen_cos(x) - math.cos(x)) < 1e-15


def test_generator_philox_kat():
    import os
    L = fi._load()
    path = os.path.join(os.path.dirname(__file__), "golden", "philox_kat.txt")
    rows = [l.split() for l in open(path) if l.strip() and not l.startswith("#")]
    assert len(rows) == 3
    for r in rows:
        v = [int(x, 16) for x in r]
        c = np.array(v[0:4], dtype=np.uint32); k = np.array(v[4:6], dtype=np.uint32); o = np.zeros(4, dtype=np.uint32)
        L.fdcgen_philox(c.ctypes.data, k.ctypes.data, o.ctypes.data)
        assert list(o) == v[6:10]


def test_trackdb_closed_forms(wl1_small):
    """P5: per-track sum dE == nominal energy; end depth ~ Bragg-Kleeman range; 1 mm steps;
    E is the start-of-step energy and non-increasing; first step exactly (0,0,1 mm)."""
    db = wl1_small.db
    off = db.track_off.astype(np.int64)
    assert db.n_tracks == 200 and list(db.bin_first) == [0, 200]
    R = 0.022 * 100.0 ** 1.77          # mm (configs[0]: R = 0.0022 E^1.77 cm)
    depths = []
    for j in range(db.n_tracks):
        s = slice(off[j], off[j + 1])
        dE = db.dE[s].astype(np.float64)
        assert abs(dE.sum() - 100.0) < 2e-5
        E = db.E[s].astype(np.float64)
        assert E[0] == 100.0 and np.all(np.diff(E) <= 0)
        assert np.allclose(E[1:], 100.0 - np.cumsum(dE)[:-1], atol=1e-4)
        assert E[-1] - dE[-1] == 0.0 and (E[:-1] - dE[:-1]).min() >= 0.5
        l = np.sqrt(db.dx[s].astype(np.float64) ** 2 + db.dy[s] ** 2 + db.dz[s] ** 2)
        assert np.allclose(l[:-1], 1.0, atol=1e-6) and 0 < l[-1] <= 1.0 + 1e-6
        assert (db.dx[s][0], db.dy[s][0], db.dz[s][0]) == (0.0, 0.0, 1.0)
        assert np.all(dE > 0)
        depths.append(db.dz[s].astype(np.float64).sum())
    depths = np.array(depths)
    # straggling 1 %/step -> range spread ~0.1 mm; detour from scattering < 1 %
    assert abs(depths.mean() - R) < 0.012 * R
    assert depths.std() < 0.5
    # path length == range within straggling
    # steps per track ~ 77
    assert 75 <= np.diff(off).min() and np.diff(off).max() <= 79


def test_trackdb_scattering_scale(wl1_small):
    """Highland: projected angle per 1 mm water step at 100 MeV is about 1.5 mrad (theta0 =
    13.6/(p beta c) sqrt(x/X0)(1+0.038 ln(x/X0)), X0 = 360.8 mm)."""
    db = wl1_small.db
    off = db.track_off.astype(np.int64)
    th = []
    for j in range(db.n_tracks):
        s = slice(off[j], off[j + 1])
        th.append(db.dx[s][1] / db.dz[s][1])      # direction after the first step's scatter
    T = 100.0; M = 938.272
    pbc = (T * T + 2 * T * M) / (T + M)
    xr = 1.0 / 360.8
    th0 = 13.6 / pbc * math.sqrt(xr) * (1 + 0.038 * math.log(xr))
    th = np.array(th)
    assert abs(th.mean()) < 4 * th0 / math.sqrt(len(th))
    assert abs(th.std() / th0 - 1.0) < 0.2


def test_lazy_db_equals_full_db():
    full = fi.make_trackdb(102, 140.0, 1.0, 21, 5)
    lazy = fi.make_trackdb(102, 140.0, 1.0, 21, 5, bins=[10])
    a, b = int(full.bin_first[10]), int(full.bin_first[11])
    s = slice(int(full.track_off[a]), int(full.track_off[b]))
    assert list(lazy.bin_first) == [0] * 11 + [5] * 11
    for name in ("dx", "dy", "dz", "dE", "E"):
        assert np.array_equal(getattr(full, name)[s], getattr(lazy, name))


def test_phantoms():
    p1 = fi.make_phantom("uniform", (8, 8, 8), (2, 2, 2))
    assert p1.hu.dtype == np.int16 and not p1.hu.any()
    p2 = fi.workload(2, n_protons=10, tracks_per_bin=2).phantom
    assert p2.dims == (128, 128, 128)
    z = p2.hu[:, 5, 7]
    assert np.all(z[:30] == 0) and np.all(z[30:60] == -750) and np.all(z[60:80] == 1000) and np.all(z[80:] == 0)
    p3 = fi.make_phantom("thorax", (64, 64, 32), (8.0, 8.0, 8.0), seed=203, noise_sigma=0.0)
    assert set(np.unique(p3.hu)) == {-1000, -800, 0, 700}
    p3n = fi.make_phantom("thorax", (64, 64, 32), (8.0, 8.0, 8.0), seed=203, noise_sigma=20.0)
    body = p3.hu == 0
    d = (p3n.hu[body].astype(np.float64) - 0.0)
    assert abs(d.mean()) < 4 * 20 / math.sqrt(d.size) + 0.01 and abs(d.std() - 20.0) < 1.0
    assert p3n.hu.min() >= -1000
    # same seed -> same bytes; different seed -> different
    assert np.array_equal(p3n.hu, fi.make_phantom("thorax", (64, 64, 32), (8.0, 8.0, 8.0), seed=203, noise_sigma=20.0).hu)
    assert not np.array_equal(p3n.hu, fi.make_phantom("thorax", (64, 64, 32), (8.0, 8.0, 8.0), seed=204, noise_sigma=20.0).hu)


def test_plans():
    w3 = fi.workload(3, n_protons=11760, tracks_per_bin=2)
    assert len(w3.beamlets) == 24 * 49 and int(w3.beamlets["n_protons"].sum()) == 11760
    assert np.all(w3.beamlets["n_protons"] == 10)
    assert len(fi.bins_hit(w3.beamlets, 70.0, 1.0)) == 24
    b = w3.beamlets[0]
    assert tuple(b["dir"]) == (0.0, 1.0, 0.0) and tuple(b["origin"]) == (256.0, -144.0, 128.0)
    bl4 = fi.make_plan((512.0, 512.0, 256.0), [0, 120, 240], [100.0], [0.0], 4.0, 10)
    assert len(bl4) == 3 and list(bl4["n_protons"]) == [3, 3, 4]
    for b in bl4:
        e1, e2, d = (b[k].astype(np.float64) for k in ("e1", "e2", "dir"))
        assert np.allclose(np.cross(e1, e2), d, atol=1e-6) and abs(np.linalg.norm(d) - 1) < 1e-6
    assert list(fi.split_even(10, 4)) == [2, 3, 2, 3]
