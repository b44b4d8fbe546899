"""Pins P2 (water identity vs Siddon), P3 (range scaling), P4 (brute-force walker), P5 (Bragg peak
depth), P10 (slab consistency) -- DESIGN.md §3.4 / SURVEY §8(c)."""
import math

import numpy as np
import pytest
from scipy.spatial.transform import Rotation

import fdc_inputs as fi
import oracle

Q24 = float(2 ** 24)


# ------------------------------------------------------------------ P2: independent Siddon voxelisation
def siddon_track(p0, steps, dE, dims, sp):
    """Energy per voxel (MeV, f64) of one polyline p0 + cumsum(steps) in a uniform-water grid, by
    Siddon's merged list of parametric plane crossings on each whole segment (not incremental)."""
    nx, ny, nz = dims
    out = {}
    p = np.array(p0, dtype=np.float64)
    for d, e in zip(steps, dE):
        q = p + d
        alphas = [0.0, 1.0]
        for a in range(3):
            if d[a] != 0.0:
                lo, hi = sorted((p[a], q[a]))
                k0 = math.ceil(lo / sp[a] - 1e-12); k1 = math.floor(hi / sp[a] + 1e-12)
                for k in range(k0, k1 + 1):
                    al = (k * sp[a] - p[a]) / d[a]
                    if 0.0 < al < 1.0:
                        alphas.append(al)
        alphas = np.unique(np.array(alphas))
        for a0, a1 in zip(alphas[:-1], alphas[1:]):
            mid = p + 0.5 * (a0 + a1) * d
            idx = tuple(int(math.floor(mid[a] / sp[a])) for a in range(3))
            if all(0 <= idx[a] < (nx, ny, nz)[a] for a in range(3)):
                out[idx] = out.get(idx, 0.0) + e * (a1 - a0)
            else:
                return out, False
        p = q
    return out, True


@pytest.mark.parametrize("origin", [(64.0, 64.0, 0.0), (63.1, 64.7, 0.0)])
def test_p2_water_identity_vs_siddon(origin):
    """All-water phantom, azimuth off, point source: the grid equals the n_j-weighted sum of each
    database track's own voxelisation (water tracks are re-traced unscaled)."""
    w = fi.workload(1, n_protons=600, tracks_per_bin=12)
    origin = tuple(float(np.float32(x)) for x in origin)         # the beamlet stores float32
    bl = fi.single_beamlet(origin, 100.0, 0.0, 600)
    g64, st = oracle.run(w.phantom, w.table, w.db, bl, seed=8, flags=0, f64=True)
    g32, st32 = oracle.run(w.phantom, w.table, w.db, bl, seed=8, flags=0)
    s = oracle.sample(w.phantom, w.table, w.db, bl, seed=8, n=600, flags=0)
    counts = np.bincount(s["track"], minlength=w.db.n_tracks)
    off = w.db.track_off.astype(np.int64)
    exp = np.zeros(g64.shape, dtype=np.float64)
    for j in range(w.db.n_tracks):
        sl = slice(off[j], off[j + 1])
        steps = np.stack([w.db.dx[sl], w.db.dy[sl], w.db.dz[sl]], axis=1).astype(np.float64)
        vox, inside = siddon_track(origin, steps, w.db.dE[sl].astype(np.float64), w.phantom.dims, w.phantom.spacing)
        assert inside
        for (ix, iy, iz), e in vox.items():
            exp[iz, iy, ix] += counts[j] * e
    got64 = g64.astype(np.float64) / Q24
    # f64 rules: only the 2^-24 MeV cumulative rounding (<= 1 quantum per share) separates the two
    assert np.abs(got64 - exp).max() <= 600 * 4 / Q24 + 1e-9
    # f32 contract: float rounding of positions moves face crossings by ~1e-5 mm; a sub-step that
    # runs within that distance of a face (the source sits on two faces) can change voxel outright
    got32 = g32.astype(np.float64) / Q24
    assert np.abs(got32 - exp).sum() <= 2e-4 * exp.sum()
    assert np.abs(got32 - exp).max() <= 1e-3 * exp.max()
    assert st32["grid_sum"] == st["grid_sum"] == st["q_replayed"]


# ------------------------------------------------------------------ P3: range scaling
def test_p3_range_scaling_bit_identical():
    """Material with rho*s = 1/2 and t = s on spacing 2h, with origin / spot / sigma doubled, gives
    the same integer grid as water on spacing h (scaling by 2 is exact in binary floating point)."""
    db = fi.make_trackdb(77, 100.0, 1.0, 1, 40)
    water = np.array([(-1000.0, 1.0, 1.0, 1.0), (3000.0, 1.0, 1.0, 1.0)], dtype=fi.KNOT_DTYPE)
    half = np.array([(-1000.0, 0.25, 2.0, 2.0), (3000.0, 0.25, 2.0, 2.0)], dtype=fi.KNOT_DTYPE)
    ph1 = fi.make_phantom("uniform", (48, 48, 96), (1.0, 1.0, 1.0))
    ph2 = fi.make_phantom("uniform", (48, 48, 96), (2.0, 2.0, 2.0))
    bl1 = fi.single_beamlet((24.3, 23.9, 0.0), 100.0, 3.0, 500); bl1["spot_u_mm"] = 1.5
    bl2 = fi.single_beamlet((48.6, 47.8, 0.0), 100.0, 6.0, 500); bl2["spot_u_mm"] = 3.0
    bl2["origin"] = 2 * bl1["origin"]
    g1, s1 = oracle.run(ph1, water, db, bl1, seed=21)
    g2, s2 = oracle.run(ph2, half, db, bl2, seed=21)
    assert np.array_equal(g1, g2)
    assert s1 == s2
    # the Gy grids differ by the voxel mass ratio (2^3 * 0.25 = 2)
    d1 = oracle.to_gy(g1, ph1, water); d2 = oracle.to_gy(g2, ph2, half)
    nz = d1 > 0
    assert np.allclose(d1[nz] / d2[nz], 2.0, rtol=1e-6)


@pytest.mark.parametrize("rho,s", [(0.8, 1.0), (1.0, 1.25), (1.85, 1.0), (0.5, 0.9)])
def test_p3_range_scales_as_inverse_rho_s(rho, s):
    """north_star: range in uniform material of density rho scales as 1/(rho x stopping-power ratio)."""
    db = fi.make_trackdb(78, 100.0, 1.0, 1, 60)
    ph = fi.make_phantom("uniform", (24, 24, 400), (2.0, 2.0, 0.5))
    bl = fi.single_beamlet((24.0, 24.0, 0.0), 100.0, 0.0, 400)
    def r80(tab):
        g, st = oracle.run(ph, tab, db, bl, seed=3)
        idd = g.sum(axis=(1, 2)).astype(np.float64)
        k = int(idd.argmax())
        j = k + int(np.argmax(idd[k:] < 0.8 * idd[k]))          # first slab past the peak below 80 %
        return (j + 0.5) * 0.5
    water = np.array([(-1000.0, 1.0, 1.0, 1.0), (3000.0, 1.0, 1.0, 1.0)], dtype=fi.KNOT_DTYPE)
    mat = np.array([(-1000.0, rho, s, s), (3000.0, rho, s, s)], dtype=fi.KNOT_DTYPE)
    rw, rm = r80(water), r80(mat)
    assert abs(rw - 0.022 * 100 ** 1.77) < 1.5                      # Bragg-Kleeman range, configs[0]
    assert abs(rm - rw / (rho * s)) <= 0.5 / (rho * s) + 0.5        # within one slab


def test_p5_config1_bragg_peak_depth(wl1_small):
    """Config 1 integral depth dose peaks in the 2 mm slab containing about R(100 MeV) = 76 mm."""
    w = wl1_small
    g, st = oracle.run(w.phantom, w.table, w.db, w.beamlets, 1)
    idd = g.sum(axis=(1, 2)).astype(np.float64)
    assert int(idd.argmax()) in (37, 38)
    assert idd[40:].sum() == 0 and idd[0] / idd.max() < 0.3
    # entrance dE/dx at 100 MeV from Bragg-Kleeman: dE/dx = E^(1-p) / (alpha p) = 0.74 MeV/mm
    assert idd[0] / Q24 / w.n_protons / 2.0 == pytest.approx(100 ** (1 - 1.77) / (0.022 * 1.77), rel=0.02)


# ------------------------------------------------------------------ P4: brute-force walker
def brute_force(ph, lut_w, lut_f, db, start, k0, k_end, dl_we=1e-3, max_geo=0.002):
    """Independent f64 walker: advances in small water-equivalent increments, looks the voxel up
    from the position at each increment's midpoint, deposits dE*dl/l there; the deflection scaling
    is applied with an axis-angle rotation (trigonometric), not the closed form."""
    nx, ny, nz = ph.dims
    sp = np.array(ph.spacing)
    p = start["p"].astype(np.float64).copy()
    R = start["R"].astype(np.float64).copy()
    out = {}
    def voxel(q):
        idx = np.floor(q / sp).astype(int)
        if np.any(idx < 0) or np.any(idx >= np.array([nx, ny, nz])):
            return None
        return tuple(idx)
    def mat(idx):
        return int(ph.hu[idx[2], idx[1], idx[0]]) + 1024
    u_prev = None
    for k in range(k0, k_end):
        d = np.array([db.dx[k], db.dy[k], db.dz[k]], dtype=np.float64)
        l = np.linalg.norm(d); u = d / l
        e = float(db.dE[k])
        v0 = voxel(p)
        if v0 is None:
            return out
        if u_prev is not None:
            f = float(lut_f[mat(v0)])
            if f != 1.0:
                c = u_prev @ u
                wv = c * u_prev + f * (u - c * u_prev); wv /= np.linalg.norm(wv)
                axis = np.cross(u, wv); sn = np.linalg.norm(axis)
                if sn > 0:
                    R = R @ Rotation.from_rotvec(axis / sn * math.atan2(sn, u @ wv)).as_matrix()
        u_prev = u
        g = R @ u
        rem = l
        while rem > 1e-15:
            v = voxel(p + 1e-9 * g)
            if v is None:
                return out
            wm = float(lut_w[mat(v)])
            step_we = min(dl_we, rem, max_geo * wm)
            q = p + g * (step_we / wm)
            vm = voxel(0.5 * (p + q))
            if vm is None:
                return out
            out[vm] = out.get(vm, 0.0) + e * step_we / l
            p = q; rem -= step_we
    return out


@pytest.mark.parametrize("cfg,protons", [(2, [0, 1, 2]), (3, [5, 4500])])
def test_p4_brute_force(cfg, protons, wl2_small, wl3_small):
    w = {2: wl2_small, 3: wl3_small}[cfg]
    rho, lw, lf = oracle.material_lut(w.table)
    off = w.db.track_off.astype(np.int64)
    for i in protons:
        s = oracle.sample(w.phantom, w.table, w.db, w.beamlets, w.seed, first=i, n=1)
        start = {"p": s["p"][0], "R": s["R"][0]}
        j = int(s["track"][0]); k0 = int(s["k0"][0])
        ref = brute_force(w.phantom, lw, lf, w.db, start, k0, int(off[j + 1]))
        g, st = oracle.run(w.phantom, w.table, w.db, w.beamlets, w.seed, first=i, n=1, f64=True)
        got = g.astype(np.float64) / Q24
        exp = np.zeros_like(got)
        for (ix, iy, iz), e in ref.items():
            exp[iz, iy, ix] = e
        emax = float(w.db.dE[k0:off[j + 1]].max())
        # each face crossing can misplace at most one increment's energy (1e-3 of a step)
        assert np.abs(got - exp).max() < 6e-3 * emax
        assert abs(got.sum() - exp.sum()) < 2e-3 * emax
        # the f32 contract lands within float rounding of the same answer
        g32, _ = oracle.run(w.phantom, w.table, w.db, w.beamlets, w.seed, first=i, n=1)
        assert np.abs(g32.astype(np.float64) / Q24 - exp).max() < 2e-2 * emax


# ------------------------------------------------------------------ P10: slab consistency
def test_p10_slab_consistency(wl2_small):
    """Config 2 central integral depth dose vs a water run mapped through W(z) = int w dz:
    IDD_slab(z) dz = IDD_water(W) dW, i.e. IDD_slab(z) = w(z) IDD_water(W(z))."""
    w = wl2_small
    n = 1500
    bl = w.beamlets.copy(); bl["n_protons"] = n
    g_s, st_s = oracle.run(w.phantom, w.table, w.db, bl, seed=5, n=n)
    wat = fi.make_phantom("uniform", (128, 128, 160), (1.0, 1.0, 1.0))
    g_w, st_w = oracle.run(wat, w.table, w.db, bl, seed=5, n=n)
    idd_s = g_s.sum(axis=(1, 2)).astype(np.float64) / Q24 / n
    idd_w = g_w.sum(axis=(1, 2)).astype(np.float64) / Q24 / n
    rho, lw, lf = oracle.material_lut(w.table)
    wz = lw[w.phantom.hu[:, 0, 0].astype(int) + 1024].astype(np.float64)
    W_edges = np.concatenate([[0.0], np.cumsum(wz)])
    cum_w = np.concatenate([[0.0], np.cumsum(idd_w)])
    pred = np.interp(W_edges[1:], np.arange(161), cum_w) - np.interp(W_edges[:-1], np.arange(161), cum_w)
    assert W_edges[-1] == pytest.approx(30 + 30 * 0.26 + 20 * 1.85 + 48, rel=1e-6)      # 122.8 mm (A17)
    sel = pred > 0.05
    assert np.all(np.abs(idd_s[sel] - pred[sel]) / pred[sel] < 0.03)
    assert abs(idd_s.sum() - pred.sum()) / pred.sum() < 0.005
