"""Pins of the oracle's gamma index (Gamma(3 %, 3 mm), Low et al. 1998).  No GPU.

G1  identical distributions: Gamma = 0 everywhere
G2  uniform field scaled by (1 + delta): Gamma = delta / dose_tol everywhere (the distance term cannot help)
G3  one hot voxel displaced by one voxel: Gamma = displacement / dist_tol at both voxels
G4  linear ramp with a constant offset: the closed-form minimum over whole-voxel shifts
G5  bounds: 0 <= Gamma <= |D_eval - D_ref| / dD at the same voxel; a larger search window never raises Gamma
"""
import numpy as np
import pytest

import oracle


def test_identical_and_scaled():
    rng = np.random.default_rng(1)
    d = rng.random((6, 7, 8)).astype(np.float32) + 0.5
    g, frac, n = oracle.gamma_index(d, d, (2.0, 2.0, 2.0))
    assert not g.any() and frac == 1.0 and n == d.size
    u = np.full((5, 5, 5), 2.0, dtype=np.float32)
    for delta in (0.015, 0.03, 0.06):
        g, frac, n = oracle.gamma_index(u, u * np.float32(1 + delta), (1.0, 1.0, 1.0))
        expect = (float(np.float32(2.0) * np.float32(1 + delta)) - 2.0) / (float(np.float32(0.03)) * 2.0)
        assert np.allclose(g, expect, rtol=1e-6) and frac == (1.0 if expect <= 1 else 0.0)


def test_displaced_hot_voxel():
    ref = np.zeros((7, 7, 7), dtype=np.float32); ev = ref.copy()
    ref[3, 3, 3] = 1.0; ev[3, 3, 4] = 1.0                      # moved by one voxel of 2 mm along x
    g, _, _ = oracle.gamma_index(ref, ev, (2.0, 2.0, 2.0), search_mm=4.0)
    assert g[3, 3, 3] == pytest.approx(2.0 / 3.0, rel=1e-6)     # reach the displaced peak: distance only
    assert g[3, 3, 4] == pytest.approx(2.0 / 3.0, rel=1e-6)     # a zero neighbour at 2 mm
    assert g[0, 0, 0] == 0.0
    g1, _, _ = oracle.gamma_index(ref, ev, (2.0, 2.0, 2.0), search_mm=1.0)      # window of one voxel: no escape
    assert g1[3, 3, 3] == pytest.approx(1.0 / 0.03, rel=1e-5)


def test_ramp_with_offset():
    nx, s, slope, off = 41, 1.0, 0.02, 0.05
    x = np.arange(nx, dtype=np.float32)
    ref = np.tile((1.0 + slope * x).astype(np.float32), (3, 3, 1))
    ev = (ref + np.float32(off)).astype(np.float32)
    g, _, _ = oracle.gamma_index(ref, ev, (s, s, s), dose_tol_frac=0.03, dist_tol_mm=3.0, search_mm=3.0)
    dD = float(np.float32(0.03)) * float(ref.max())
    # shifting by k voxels changes the evaluated dose by slope*k: minimise over k = -3..3 (interior voxel)
    best = min(np.sqrt((k * s / 3.0) ** 2 + ((off + slope * k) / dD) ** 2) for k in range(-3, 4))
    assert g[1, 1, 20] == pytest.approx(best, rel=1e-4)
    assert best < off / dD                                       # the distance term does help on a ramp


def test_bounds_and_window_monotonicity():
    rng = np.random.default_rng(2)
    ref = (rng.random((8, 9, 10)) + 0.2).astype(np.float32)
    ev = (ref * (1 + 0.05 * rng.standard_normal(ref.shape))).astype(np.float32)
    sp = (2.0, 1.5, 2.5)
    g3, f3, n3 = oracle.gamma_index(ref, ev, sp, search_mm=3.0)
    g6, f6, n6 = oracle.gamma_index(ref, ev, sp, search_mm=6.0)
    dD = float(np.float32(0.03)) * float(ref.max())
    same = np.abs(ev.astype(np.float64) - ref.astype(np.float64)) / dD
    assert np.all(g3 >= 0) and np.all(g3 <= same.astype(np.float32) * (1 + 1e-6) + 1e-7)
    assert np.all(g6 <= g3) and f6 >= f3 and n3 == n6 == ref.size
    gc, fc, nc = oracle.gamma_index(ref, ev, sp, cutoff_frac=0.5)
    assert nc == int((ref > np.float32(0.5) * ref.max()).sum()) and np.array_equal(gc, g3)
