"""Pins of R15, histories with several trajectories.  No GPU.

SE1  an empty secondary table changes nothing
SE2  closed form: a secondary branching from a straight primary deposits where the primary stood, along the
     database x axis carried through the primary's frame
SE3  energy: with nobody escaping, the grid holds the primary's energy from its start step plus the energy of
     every secondary that branches at or after that step; a proton that joins after a branch skips it
SE4  a primary that escapes before the branch step never starts the secondary
SE5  additivity, conservation and ordered squares tallies on random worlds with random secondaries
"""
import numpy as np

import fdc_inputs as fi
import oracle
from test_oracle_pins import table_uniform, uniform_phantom


def db_with_secondaries(primaries, secondaries, e_min=100.0):
    """primaries: list of step lists [(dx,dy,dz,dE)...] (one bin); secondaries: list of (parent, step, steps)."""
    dx, dy, dz, dE, E, off = [], [], [], [], [], [0]
    for tr in primaries + [s[2] for s in secondaries]:
        e = e_min
        for (a, b, c, d) in tr:
            dx.append(a); dy.append(b); dz.append(c); dE.append(d); E.append(e); e -= d
        off.append(len(dx))
    f = lambda v: np.array(v, dtype=np.float32)
    n_p = len(primaries)
    db = fi.TrackDB(f(dx), f(dy), f(dz), f(dE), f(E), np.array(off, dtype=np.uint64), np.array([0, n_p], dtype=np.uint32), e_min, 1.0)
    n_tr = n_p + len(secondaries)
    order = sorted(range(len(secondaries)), key=lambda i: (secondaries[i][0], secondaries[i][1]))
    first = np.zeros(n_tr + 1, dtype=np.uint32); track, step = [], []
    for i in order:
        first[secondaries[i][0] + 1] += 1; track.append(n_p + i); step.append(secondaries[i][1])
    first = np.cumsum(first).astype(np.uint32)
    return db, (first, np.array(track, dtype=np.uint32), np.array(step, dtype=np.uint32))


Q = lambda e: int(np.rint(np.float32(e) * np.float32(2 ** 24)))


def test_empty_table_is_the_plain_run(wl2_small):
    w = wl2_small
    sec = (np.zeros(w.db.n_tracks + 1, np.uint32), np.zeros(0, np.uint32), np.zeros(0, np.uint32))
    g0, s0 = oracle.run(w.phantom, w.table, w.db, w.beamlets, w.seed, n=300)
    g1, s1 = oracle.run_secondaries(w.phantom, w.table, w.db, sec, w.beamlets, w.seed, n=300)
    assert np.array_equal(g0, g1) and all(s0[k] == s1[k] for k in s0)


def test_secondary_starts_where_the_parent_stood():
    ph = uniform_phantom(16, 1.0)
    prim = [[(0, 0, 1.0, 1.0)] * 4]
    secs = [(0, 1, [(1.0, 0, 0, 0.5), (1.0, 0, 0, 0.25), (1.0, 0, 0, 0.125)])]        # after the primary's second step, along database x
    db, sec = db_with_secondaries(prim, secs)
    bl = fi.single_beamlet((5.5, 6.5, 0.25), 100.0, 0.0, 1)                            # frame (x, y, z), azimuth off
    g, st = oracle.run_secondaries(ph, table_uniform(1.0), db, sec, bl, 1, flags=0)
    exp = np.zeros_like(g)
    for k in range(4):                                                                 # primary: z from 0.25 + k to 1.25 + k
        exp[k, 6, 5] += int(np.rint(Q(1.0) * np.float32(np.float32(0.75) * np.float32(1.0))))
        exp[k + 1, 6, 5] += Q(1.0) - int(np.rint(Q(1.0) * np.float32(0.75)))
    # the secondary starts at (5.5, 6.5, 2.25) in voxel (5, 6, 2): x from 5.5: half a voxel, then whole voxels
    for k, e in enumerate((0.5, 0.25, 0.125)):
        a = int(np.rint(Q(e) * np.float32(0.5)))
        exp[2, 6, 5 + k] += a; exp[2, 6, 6 + k] += Q(e) - a
    assert np.array_equal(g, exp)
    assert st["proton_steps"] == 7 and st["stopped"] == 1 and st["q_replayed"] == 4 * Q(1.0) + Q(0.5) + Q(0.25) + Q(0.125)


def test_energy_bookkeeping_and_late_joiners():
    ph = uniform_phantom(32, 2.0)
    prim = [[(0, 0, 1.0, 1.0)] * 10]
    secs = [(0, 2, [(0.6, 0, 0.8, 2.0)] * 2), (0, 6, [(0, 0.6, 0.8, 3.0)]), (0, 6, [(0, -1.0, 0, 0.5)])]
    db, sec = db_with_secondaries(prim, secs)
    for e0, k0 in ((100.0, 0), (97.5, 3), (93.0, 7)):                                  # E = 100, 99, 98, ...: joins at step k0
        bl = fi.single_beamlet((31.0, 33.0, 1.0), e0, 0.0, 5)
        g, st = oracle.run_secondaries(ph, table_uniform(1.0), db, sec, bl, 3, flags=1)
        q_sec = sum(sum(Q(s[3]) for s in steps) for (_, step, steps) in secs if step >= k0)
        assert st["escaped"] == 0 and st["stopped"] == 5
        assert st["q_replayed"] == 5 * ((10 - k0) * Q(1.0) + q_sec) == st["grid_sum"]
        assert st["proton_steps"] == 5 * ((10 - k0) + sum(len(steps) for (_, step, steps) in secs if step >= k0))


def test_escape_before_the_branch():
    ph = uniform_phantom(4, 1.0)                                                       # 4 mm deep: the primary leaves during its 4th step
    prim = [[(0, 0, 1.0, 1.0)] * 8]
    secs = [(0, 1, [(1.0, 0, 0, 0.5)]), (0, 6, [(1.0, 0, 0, 0.5)])]
    db, sec = db_with_secondaries(prim, secs)
    bl = fi.single_beamlet((1.5, 1.5, 0.5), 100.0, 0.0, 1)
    g, st = oracle.run_secondaries(ph, table_uniform(1.0), db, sec, bl, 1, flags=0)
    assert st["escaped"] == 1 and st["proton_steps"] == 4 + 1                            # the first secondary ran, the second never started
    assert st["grid_sum"] + st["q_escaped"] == st["q_replayed"] == 8 * Q(1.0) + Q(0.5)


def random_secondaries(rng, db, n_primary_bins_tracks):
    """Random secondary table for a random-world database: a few of the primaries get 1-3 secondaries whose
    trajectories are appended to the step arrays."""
    n_p = db.n_tracks
    dx, dy, dz, dE, E = (list(a) for a in (db.dx, db.dy, db.dz, db.dE, db.E))
    off = list(db.track_off)
    recs = []
    for j in range(n_p):
        ln = int(off[j + 1] - off[j])
        if ln == 0 or rng.random() < 0.4:
            continue
        for step in sorted(int(rng.integers(0, ln)) for _ in range(int(rng.integers(1, 4)))):
            e = 20.0
            for _ in range(int(rng.integers(1, 6))):
                d = rng.normal(size=3) * rng.uniform(0.1, 1.5)
                de = float(rng.uniform(0, 1.0))
                dx.append(d[0]); dy.append(d[1]); dz.append(d[2]); dE.append(de); E.append(e); e -= de
            off.append(len(dx)); recs.append((j, step))
    f = lambda v: np.array(v, dtype=np.float32)
    db2 = fi.TrackDB(f(dx), f(dy), f(dz), f(dE), f(E), np.array(off, dtype=np.uint64), db.bin_first.copy(), db.e_min, db.e_bin)
    first = np.zeros(len(off), dtype=np.uint32)
    for (j, _) in recs:
        first[j + 1] += 1
    first = np.cumsum(first).astype(np.uint32)
    return db2, (first, np.arange(n_p, n_p + len(recs), dtype=np.uint32), np.array([s for (_, s) in recs], dtype=np.uint32))


def test_random_worlds_with_secondaries():
    from random_worlds import random_case
    rng = np.random.default_rng(11)
    started = 0
    for case in range(40):
        w = random_case(rng)
        db2, sec = random_secondaries(rng, w.db, None)
        flags = int(rng.choice([0, 1, 33]))
        g, sv, sh, st = oracle.run_secondaries(w.phantom, w.table, db2, sec, w.beamlets, w.seed, flags=flags, squares=True)
        assert st["grid_sum"] + st["q_escaped"] == st["q_replayed"], case
        assert st["protons"] == st["missed"] + st["escaped"] + st["stopped"], case
        assert np.all(sv <= sh), case
        h = w.n_protons // 2
        ga, sa = oracle.run_secondaries(w.phantom, w.table, db2, sec, w.beamlets, w.seed, first=0, n=h, flags=flags)
        gb, sb = oracle.run_secondaries(w.phantom, w.table, db2, sec, w.beamlets, w.seed, first=h, n=w.n_protons - h, flags=flags)
        assert np.array_equal(ga + gb, g), case
        g0, s0 = oracle.run(w.phantom, w.table, db2, w.beamlets, w.seed, flags=flags)       # the same primaries without their secondaries
        assert np.all(g >= g0) and st["proton_steps"] >= s0["proton_steps"]
        started += st["proton_steps"] - s0["proton_steps"]
    assert started > 1000
