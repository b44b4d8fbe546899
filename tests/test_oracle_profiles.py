"""Pins of the oracle's profile comparators (R16, R17).  No GPU.

PR1  a grid that depends on one coordinate only: the profile along that axis is the function itself whatever the
     thickness; along another axis it is constant; a separable ramp a*x + b*y + c*z gives the closed form
     (mean of an arithmetic progression over the bundle) on every axis
PR2  hand values on a 3 x 4 x 5 grid, including a bundle clipped by the grid edge (fewer columns in the mean)
PR3  the energy grid: integer sum times 2^-24 over the count, exact; the profile over the full cross-section
     integrates to the grid's total energy (Fig. 2 plots deposited energy against depth)
RM1  closed forms of the RMS difference: identical -> 0; uniform reference scaled by (1 + d) -> d; one voxel off
     by e in a grid of n voxels -> (e / max) / sqrt(n); a box of height 1 shifted by one voxel along x ->
     sqrt(2 * face area / n)
RM2  invariances: a common scale factor on both grids leaves it unchanged; swapping the roles changes only the
     normalisation (ratio of the two maxima)
"""
import numpy as np
import pytest

import oracle


def test_pr1_one_coordinate_and_separable_ramp():
    nz, ny, nx = 6, 7, 9
    z, y, x = np.meshgrid(np.arange(nz), np.arange(ny), np.arange(nx), indexing="ij")
    fy = (3.0 + 0.25 * y * y).astype(np.float32)                      # depends on y only
    for hw in ((0, 0), (2, 2), (2, 0), (5, 9)):
        assert np.array_equal(oracle.profile(fy, 1, 4, 3, *hw), (3.0 + 0.25 * np.arange(ny) ** 2).astype(np.float32).astype(np.float64))
        # along x (a = y, b = z): constant, equal to the mean of fy over the y range of the bundle
        y0, y1 = max(0, 3 - hw[0]), min(ny - 1, 3 + hw[0])
        want = np.mean([float(np.float32(3.0 + 0.25 * k * k)) for k in range(y0, y1 + 1)])
        assert np.allclose(oracle.profile(fy, 0, 3, 2, *hw), want, rtol=1e-15)
    a, b, c = 0.5, 2.0, -0.25                                          # exactly representable: sums are exact
    ramp = (a * x + b * y + c * z + 10.0).astype(np.float32)
    # axis 2 (z): a = x, b = y; bundle x in [2, 6], y in [1, 5] around (4, 3) with half width 2
    got = oracle.profile(ramp, 2, 4, 3, 2, 2)
    assert np.array_equal(got, a * 4 + b * 3 + c * np.arange(nz) + 10.0)
    # axis 0 (x): a = y, b = z; the bundle is clipped at y = 0: y in [0, 2] around fixed_a = 0
    got = oracle.profile(ramp, 0, 0, 3, 2, 1)
    assert np.array_equal(got, a * np.arange(nx) + b * 1.0 + c * 3 + 10.0)


def test_pr2_hand_values_and_clipping():
    v = np.arange(3 * 4 * 5, dtype=np.float32).reshape(3, 4, 5)        # value = x + 5 y + 20 z
    assert np.array_equal(oracle.profile(v, 0, 1, 2, 0, 0), [45, 46, 47, 48, 49])          # y = 1, z = 2
    assert np.array_equal(oracle.profile(v, 1, 4, 0, 0, 0), [4, 9, 14, 19])                # x = 4, z = 0
    assert np.array_equal(oracle.profile(v, 2, 0, 3, 0, 0), [15, 35, 55])                  # x = 0, y = 3
    # x = 4 is the last column: half width 1 on x keeps x in {3, 4} (2 columns, not 3); z in {0, 1}
    got = oracle.profile(v, 1, 4, 0, 1, 1)
    want = [np.mean([xx + 5 * yy + 20 * zz for zz in (0, 1) for xx in (3, 4)]) for yy in range(4)]
    assert np.array_equal(got, want)


def test_pr3_energy_grid_profile_integrates_to_the_total():
    rng = np.random.default_rng(5)
    g = rng.integers(0, 1 << 40, size=(5, 6, 7), dtype=np.uint64)
    nz, ny, nx = g.shape
    p = oracle.profile(g, 1, nx // 2, nz // 2, nx, nz)                 # the whole cross-section at each depth y
    per_y = g.sum(axis=(0, 2), dtype=np.uint64).astype(np.float64) * 2.0 ** -24 / float(nx * nz)
    assert np.array_equal(p, per_y)
    assert np.sum(p) * nx * nz == pytest.approx(float(g.sum(dtype=np.uint64)) * 2.0 ** -24, rel=1e-14)
    one = oracle.profile(g, 0, 2, 3, 0, 0)
    assert np.array_equal(one, g[3, 2, :].astype(np.float64) * 2.0 ** -24)


def test_rm1_closed_forms():
    rng = np.random.default_rng(6)
    ref = (rng.random((5, 6, 7)) + 0.5).astype(np.float32)
    assert oracle.rms_diff(ref, ref) == (0.0, float(ref.max()))
    u = np.full((4, 5, 6), 2.0, dtype=np.float32)
    for d in (0.005, 0.03):
        ev = (u * np.float32(1 + d)).astype(np.float32)
        want = (float(ev[0, 0, 0]) - 2.0) / 2.0
        assert oracle.rms_diff(u, ev)[0] == pytest.approx(want, rel=1e-14)
    ev = ref.copy(); ev[2, 3, 4] += np.float32(0.125)
    e = float(ev[2, 3, 4]) - float(ref[2, 3, 4])
    assert oracle.rms_diff(ref, ev)[0] == pytest.approx(e / float(ref.max()) / np.sqrt(ref.size), rel=1e-14)
    box = np.zeros((8, 8, 10), dtype=np.float32); box[2:6, 2:6, 3:7] = 1.0
    sh = np.roll(box, 1, axis=2)                                       # moved by one voxel along x
    # differs by 1 on the two 4 x 4 faces the shift uncovers / covers
    assert oracle.rms_diff(box, sh)[0] == pytest.approx(np.sqrt(2 * 16 / box.size), rel=1e-15)


def test_rm2_invariances():
    rng = np.random.default_rng(7)
    ref = (rng.random((4, 5, 6)) + 0.1).astype(np.float32)
    ev = (ref + 0.01 * rng.standard_normal(ref.shape)).astype(np.float32)
    r, m = oracle.rms_diff(ref, ev)
    r4, m4 = oracle.rms_diff(ref * np.float32(4), ev * np.float32(4))   # power of two: exact
    assert r4 == r and m4 == 4 * m
    rs, ms = oracle.rms_diff(ev, ref)
    assert rs * ms == pytest.approx(r * m, rel=1e-13)
