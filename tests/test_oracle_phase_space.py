"""Pins of the oracle's phase-space source (R12; "phase-space array").  No GPU.

PS1  the frame rule gives a right-handed orthonormal frame for any unit direction; (x, y) for +z
PS2  a phase-space array made of the start points of a beamlet plan reproduces that plan's grid and
     counters exactly (ties the phase-space path to the beamlet path, itself pinned by P1-P10)
PS3  divergent beam with an energy spread: conservation, additivity over sub-arrays, misses
"""
import numpy as np

import fdc_inputs as fi
import oracle


def test_frame_rule():
    e1, e2 = oracle.frame_rule((0, 0, 1))
    assert tuple(e1) == (1, 0, 0) and tuple(e2) == (0, 1, 0)
    e1, e2 = oracle.frame_rule((0, 1, 0))
    assert tuple(e1) == (1, 0, 0) and tuple(e2) == (0, 0, -1)
    rng = np.random.default_rng(5)
    for _ in range(200):
        d = rng.normal(size=3); d = (d / np.linalg.norm(d)).astype(np.float32)
        e1, e2 = oracle.frame_rule(d)
        d64, a, b = d.astype(np.float64), e1.astype(np.float64), e2.astype(np.float64)
        assert abs(a @ a - 1) < 1e-6 and abs(b @ b - 1) < 1e-6
        assert abs(a @ d64) < 1e-6 and abs(b @ d64) < 1e-6 and abs(a @ b) < 1e-6
        assert np.allclose(np.cross(a, b), d64, atol=1e-6)              # e1 x e2 = dir, as in the beamlet frames


def particles(pos, dirs, energy):
    ps = np.zeros(len(pos), dtype=oracle.PARTICLE_DTYPE)
    ps["pos"] = pos; ps["dir"] = dirs; ps["energy_mev"] = energy
    return ps


def test_phase_space_reproduces_a_beamlet_plan(wl2_small):
    w = wl2_small                                                           # 150 MeV, +z, sigma 5 mm, frame (x, y)
    smp = oracle.sample(w.phantom, w.table, w.db, w.beamlets, w.seed, first=0, n=w.n_protons)
    p = smp["p"] if isinstance(smp, dict) else smp[3]
    ps = particles(np.asarray(p, dtype=np.float32).reshape(-1, 3), np.tile(np.float32([0, 0, 1]), (w.n_protons, 1)), 150.0)
    for flags in (1, 0):
        g0, st0 = oracle.run(w.phantom, w.table, w.db, w.beamlets, w.seed, flags=flags)
        g1, st1 = oracle.run_phase_space(w.phantom, w.table, w.db, ps, w.seed, first_id=0, flags=flags)
        assert np.array_equal(g0, g1)
        assert all(st0[k] == st1[k] for k in st0)


def cone(n, seed, e_lo=141.0, e_hi=150.0, half_angle=0.05):
    rng = np.random.default_rng(seed)
    th = half_angle * np.sqrt(rng.random(n)); ph = 2 * np.pi * rng.random(n)
    d = np.stack([np.sin(th) * np.cos(ph), np.sin(th) * np.sin(ph), np.cos(th)], 1)
    d = (d / np.linalg.norm(d, axis=1, keepdims=True)).astype(np.float32)
    pos = np.tile(np.float32([64.0, 64.0, -50.0]), (n, 1)) + rng.normal(0, 2.0, (n, 3)).astype(np.float32) * np.float32([1, 1, 0])
    return particles(pos, d, rng.uniform(e_lo, e_hi, n).astype(np.float32))


def test_divergent_beam_with_energy_spread():
    w = fi.workload(2, n_protons=10, tracks_per_bin=100, lazy_db=False)      # all 21 bins 140-160 MeV
    ps = cone(600, 3)
    g, st = oracle.run_phase_space(w.phantom, w.table, w.db, ps, 77)
    assert st["protons"] == 600 == st["missed"] + st["escaped"] + st["stopped"]
    assert st["grid_sum"] + st["q_escaped"] == st["q_replayed"]
    ga, sa = oracle.run_phase_space(w.phantom, w.table, w.db, ps[:250], 77, first_id=0)
    gb, sb = oracle.run_phase_space(w.phantom, w.table, w.db, ps[250:], 77, first_id=250)
    assert np.array_equal(ga + gb, g) and sa["deposits"] + sb["deposits"] == st["deposits"]
    # the random-number identity is first_id + m: another offset gives another (valid) result
    gc, sc = oracle.run_phase_space(w.phantom, w.table, w.db, ps, 77, first_id=1000)
    assert not np.array_equal(gc, g) and sc["grid_sum"] + sc["q_escaped"] == sc["q_replayed"]
    # starts deeper in a track for lower energies: less energy replayed per proton on average
    lo = oracle.run_phase_space(w.phantom, w.table, w.db, cone(300, 4, 141.0, 142.0), 9)[1]
    hi = oracle.run_phase_space(w.phantom, w.table, w.db, cone(300, 4, 158.0, 159.0), 9)[1]
    assert lo["q_replayed"] < hi["q_replayed"]
    # pointing away from the grid: missed, nothing tallied
    away = particles(np.float32([[64, 64, -10]]), np.float32([[0, 0, -1]]), 150.0)
    g2, s2 = oracle.run_phase_space(w.phantom, w.table, w.db, away, 1)
    assert s2["missed"] == 1 and not g2.any()
