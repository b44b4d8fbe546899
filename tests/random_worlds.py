"""Small random worlds for the degenerate-input tests (oracle conservation on the CPU, GPU parity on the box).
Input generation only: no arithmetic of the method."""
import numpy as np

import fdc_inputs as fi


def random_case(rng):
    """A small random world: ragged grid (axes of 1-9 voxels, unequal spacings), HU from vacuum to metal,
    a hand-made database with several energy bins (some empty), tracks of 1-12 steps that include
    zero-length steps, steps much longer and much shorter than a voxel and deflections beyond 90
    degrees, and a few oblique beamlets that start inside, outside or miss the grid."""
    dims = tuple(int(rng.integers(1, 10)) for _ in range(3))
    sp = tuple(float(np.float32(rng.choice([0.5, 1.0, 1.7, 2.0, 3.3]))) for _ in range(3))
    ph = fi.make_phantom("uniform", dims, sp)
    ph.hu[...] = rng.choice(np.array([-1000, -990, -800, -50, 0, 30, 400, 1500, 3071, -1024], dtype=np.int16), size=ph.hu.shape)
    n_bins, e_min = 4, 50.0
    dx, dy, dz, dE, E, off, binf = [], [], [], [], [], [0], [0]
    for b in range(n_bins):
        ntr = 0 if b == 2 else int(rng.integers(1, 5))                       # bin 2 stays empty
        for _ in range(ntr):
            e = e_min + b
            for k in range(int(rng.integers(1, 13))):
                kind = rng.integers(0, 6)
                if kind == 0:
                    d = np.zeros(3)
                elif kind == 1:
                    d = rng.normal(size=3) * 1.5                            # any direction (deflections beyond 90 degrees)
                elif kind == 2:
                    d = np.array([0.0, 0.0, 1.0]) * 10.0 ** rng.uniform(-4, 1)
                else:
                    d = np.array([rng.normal() * 0.2, rng.normal() * 0.2, 1.0]) * rng.uniform(0.05, 1.2)
                de = float(rng.uniform(0, 1.5)) if rng.random() > 0.1 else 0.0
                dx.append(d[0]); dy.append(d[1]); dz.append(d[2]); dE.append(de); E.append(e)
                e -= de * rng.uniform(0.0, 1.0)                              # E only has to be non-increasing
            off.append(len(dx))
        binf.append(len(off) - 1)
    f = lambda v: np.array(v, dtype=np.float32)
    db = fi.TrackDB(f(dx), f(dy), f(dz), f(dE), f(E), np.array(off, dtype=np.uint64), np.array(binf, dtype=np.uint32), e_min, 1.0)
    bls = []
    ext = np.array(dims) * np.array(sp)
    for _ in range(int(rng.integers(1, 4))):
        d = rng.normal(size=3); d /= np.linalg.norm(d)
        a = np.cross(d, rng.normal(size=3)); a /= np.linalg.norm(a); bb = np.cross(d, a)   # e1 x e2 = d
        origin = ext * (rng.uniform(0.05, 0.95, size=3) if rng.random() < 0.7 else rng.uniform(-0.5, 1.5, size=3))
        energy = float(rng.choice([50.0, 50.5, 51.0, 53.0, 49.0, 52.6]))      # never bin 2 (51 < E <= 52)
        bl = fi.single_beamlet(tuple(origin.astype(np.float32)), energy, float(rng.choice([0.0, 0.7])), int(rng.integers(20, 200)),
                               e1=tuple(a.astype(np.float32)), e2=tuple(bb.astype(np.float32)), d=tuple(d.astype(np.float32)))
        bls.append(bl)
    bl = np.concatenate(bls)
    table = np.array([(-1000.0, 0.001, 1.0, 1.0), (-800.0, 0.2, 1.02, 0.9), (0.0, 1.0, 1.0, 1.0), (1500.0, 2.0, 0.95, 1.3), (3000.0, 4.5, 0.9, 2.0)],
                     dtype=fi.KNOT_DTYPE)
    return fi.Workload("fuzz", ph, table, db, bl, int(bl["n_protons"].sum()), int(rng.integers(1, 2 ** 40)))
