"""Pins of R14, the re-alignment of a sub-track that starts deep in a database track (PAPER.md:L71
"selecting the trajectory and step where the track-repeating algorithm should start").

RA1  a start at the first step, or a straight track, is unchanged (bit-identical grid)
RA2  a track deflected before the start step: with the flag the first replayed step runs exactly along
     the beam; without it, along the deflected direction (closed form, one remaining step)
RA3  single-energy database, energies far below it (deep starts): energy is conserved and the dose of a
     single re-used track stays on the beam axis with the flag, off it without
"""
import numpy as np
import pytest

import fdc_inputs as fi
import oracle
from test_oracle_pins import hand_db, table_uniform, uniform_phantom

RA = oracle.FLAG_REALIGN_START


def test_realign_is_identity_for_straight_tracks_and_first_step(wl2_small):
    ph = uniform_phantom(16, 1.0)
    db = hand_db([[(0, 0, 1.0, 1.0)] * 8])
    bl = fi.single_beamlet((5.5, 6.5, 0.0), 97.5, 0.0, 3)                    # starts at step 3 (E: 100, 99, 98, 97 ...)
    g0, s0 = oracle.run(ph, table_uniform(1.0), db, bl, 3, flags=1)
    g1, s1 = oracle.run(ph, table_uniform(1.0), db, bl, 3, flags=1 | RA)
    assert s0["proton_steps"] == 15 and np.array_equal(g0, g1)
    w = wl2_small                                                           # 150 MeV into the 150 MeV bin: k0 = first step = (0,0,1)
    g0, _ = oracle.run(w.phantom, w.table, w.db, w.beamlets, w.seed, n=200)
    g1, _ = oracle.run(w.phantom, w.table, w.db, w.beamlets, w.seed, n=200, flags=1 | RA)
    assert np.array_equal(g0, g1)


def test_first_replayed_step_runs_along_the_beam():
    th = 0.2
    db = hand_db([[(0, 0, 1.0, 1.0), (0, 0, 1.0, 1.0), (np.sin(th), 0.0, np.cos(th), 1.0)]])
    ph = uniform_phantom(16, 1.0)
    d = np.float32([0.6, 0.0, 0.8]); e1 = np.float32([0.8, 0.0, -0.6]); e2 = np.float32([0.0, 1.0, 0.0])
    p0 = np.float32([4.25, 7.5, 3.25])
    bl = fi.single_beamlet(tuple(p0), 98.0, 0.0, 1, e1=tuple(e1), e2=tuple(e2), d=tuple(d))   # E[2] = 98 <= 98: k0 = 2
    out = {}
    for name, flags in (("plain", 0), ("realign", RA)):
        g, st, tr, es = oracle.run_trace(ph, table_uniform(1.0), db, bl, 1, flags=flags)
        assert st["proton_steps"] == 1 and st["stopped"] == 1
        out[name] = es[0, :3].astype(np.float64)
    assert np.allclose(out["realign"], p0.astype(np.float64) + d.astype(np.float64), atol=2e-6)
    tilted = np.sin(th) * e1.astype(np.float64) + np.cos(th) * d.astype(np.float64)          # R0 (sin, 0, cos)
    assert np.allclose(out["plain"], p0.astype(np.float64) + tilted, atol=2e-6)


def test_deep_starts_in_a_single_energy_database():
    base = fi.workload(1, n_protons=1, tracks_per_bin=1)                    # ONE 100 MeV track (the paper's single-energy DB, L57)
    n = 400
    res = {}
    for name, flags in (("plain", 0), ("realign", RA)):                      # azimuth off: every proton replays the same sub-track
        bl = fi.single_beamlet((64.0, 64.0, 0.0), 40.0, 0.0, n)              # 40 MeV: starts about 60 steps into the track
        g, st = oracle.run(base.phantom, base.table, base.db, bl, 5, flags=flags)
        assert st["grid_sum"] + st["q_escaped"] == st["q_replayed"] and st["stopped"] == n
        assert abs(st["q_replayed"] / n / 2 ** 24 - 40.0) < 1.5               # the gap E0 - E[k0] is below one step's loss
        zz, yy, xx = np.nonzero(g)
        wgt = g[zz, yy, xx].astype(np.float64)
        cx = ((xx + 0.5) * 2.0 * wgt).sum() / wgt.sum(); cy = ((yy + 0.5) * 2.0 * wgt).sum() / wgt.sum()
        res[name] = (np.hypot(cx - 64.0, cy - 64.0), ((zz + 0.5) * 2.0 * wgt).sum() / wgt.sum())
    # 60 steps of multiple scattering have tilted the track by some tens of mrad: un-aligned it drifts off the axis
    assert res["realign"][0] < res["plain"][0]
    assert res["realign"][1] >= res["plain"][1] - 0.5                          # and does not lose depth
