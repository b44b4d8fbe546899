"""Seeded synthetic inputs for the track-repeating hot path (track DB, phantoms, beam plans).

Serves BOTH the oracle and the CUDA path with identical bytes; holds none of the method's
arithmetic.  The heavy generators are in ``gen.c`` (built here with gcc, OpenMP);
this file marshals numpy arrays and defines the five workload presets that stand in for
``BASELINE.json:configs[0..4]`` (the paper's CT and GEANT4 database are not
available: PAPER.md:L57, L61, L98).
"""
from __future__ import annotations

import ctypes
import math
import os
import subprocess
from dataclasses import dataclass, field

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "gen.c")
_LIB = os.path.join(_HERE, "libfdcgen.so")
_lib = None


def build(force: bool = False) -> str:
    """Compile gen.c -> libfdcgen.so (in-tree).  -ffp-contract=off: see gen.c header."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + ".tmp.%d" % os.getpid()
        subprocess.check_call(["gcc", "-O2", "-ffp-contract=off", "-fno-fast-math", "-fopenmp",
                               "-shared", "-fPIC", "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        L = ctypes.CDLL(build())
        L.fdcgen_tracks_capacity.restype = ctypes.c_int64
        L.fdcgen_tracks_capacity.argtypes = [ctypes.c_double, ctypes.c_double, ctypes.c_int,
                                             ctypes.c_int, ctypes.c_void_p]
        L.fdcgen_tracks.restype = ctypes.c_int64
        L.fdcgen_tracks.argtypes = [ctypes.c_uint64, ctypes.c_double, ctypes.c_double, ctypes.c_int,
                                    ctypes.c_int, ctypes.c_void_p] + [ctypes.c_void_p] * 7
        L.fdcgen_phantom.restype = None
        L.fdcgen_phantom.argtypes = [ctypes.c_int, ctypes.c_uint64, ctypes.c_int, ctypes.c_int,
                                     ctypes.c_int, ctypes.c_double, ctypes.c_double, ctypes.c_double,
                                     ctypes.c_int, ctypes.c_double, ctypes.c_void_p]
        for f in ("fdcgen_ln", "fdcgen_exp", "fdcgen_sin", "fdcgen_cos"):
            getattr(L, f).restype = ctypes.c_double
            getattr(L, f).argtypes = [ctypes.c_double]
        L.fdcgen_philox.restype = None
        L.fdcgen_philox.argtypes = [ctypes.c_void_p] * 3
        _lib = L
    return _lib


# ----------------------------------------------------------------------------- containers
@dataclass
class TrackDB:
    """SoA track-step store binned by incident energy (BASELINE.json north_star (1))."""
    dx: np.ndarray
    dy: np.ndarray
    dz: np.ndarray
    dE: np.ndarray
    E: np.ndarray            # kinetic energy at the START of each step
    track_off: np.ndarray    # uint64, n_tracks+1
    bin_first: np.ndarray    # uint32, n_bins+1, into track ids
    e_min: float
    e_bin: float

    @property
    def n_steps(self) -> int:
        return int(self.dx.shape[0])

    @property
    def n_tracks(self) -> int:
        return int(self.track_off.shape[0] - 1)

    @property
    def n_bins(self) -> int:
        return int(self.bin_first.shape[0] - 1)


@dataclass
class Phantom:
    hu: np.ndarray           # int16, shape (nz, ny, nx): x fastest
    spacing: tuple           # (sx, sy, sz) mm

    @property
    def dims(self):
        nz, ny, nx = self.hu.shape
        return nx, ny, nz


BEAMLET_DTYPE = np.dtype([("origin", "<f4", 3), ("e1", "<f4", 3), ("e2", "<f4", 3), ("dir", "<f4", 3),
                          ("energy_mev", "<f4"), ("spot_u_mm", "<f4"), ("spot_v_mm", "<f4"),
                          ("sigma_mm", "<f4"), ("n_protons", "<u8")], align=True)
KNOT_DTYPE = np.dtype([("hu", "<f4"), ("density_g_cc", "<f4"), ("mass_spr", "<f4"),
                       ("mass_scpr", "<f4")], align=True)


@dataclass
class Workload:
    name: str
    phantom: Phantom
    table: np.ndarray        # KNOT_DTYPE
    db: TrackDB
    beamlets: np.ndarray     # BEAMLET_DTYPE
    n_protons: int
    seed: int
    notes: dict = field(default_factory=dict)


# ----------------------------------------------------------------------------- generators
def make_trackdb(seed: int, e_min: float, e_bin: float, n_bins: int, tracks_per_bin: int,
                 bins=None) -> TrackDB:
    """Track database per configs[0]'s recipe.  ``bins`` (iterable of bin indices) restricts
    generation to those bins; the others stay empty (same tracks either way)."""
    L = _load()
    mask = None
    if bins is not None:
        mask = np.zeros(n_bins, dtype=np.uint8)
        mask[np.asarray(sorted(set(int(b) for b in bins)), dtype=np.int64)] = 1
    mptr = mask.ctypes.data if mask is not None else None
    cap = L.fdcgen_tracks_capacity(e_min, e_bin, n_bins, tracks_per_bin, mptr)
    ntr = tracks_per_bin * (int(mask.sum()) if mask is not None else n_bins)
    arrs = [np.empty(cap, dtype=np.float32) for _ in range(5)]
    track_off = np.empty(ntr + 1, dtype=np.uint64)
    bin_first = np.empty(n_bins + 1, dtype=np.uint32)
    n = L.fdcgen_tracks(seed, e_min, e_bin, n_bins, tracks_per_bin, mptr,
                        *[a.ctypes.data for a in arrs], track_off.ctypes.data, bin_first.ctypes.data)
    assert 0 < n <= cap
    dx, dy, dz, dE, E = [a[:n] for a in arrs]
    return TrackDB(dx, dy, dz, dE, E, track_off, bin_first, float(e_min), float(e_bin))


def make_phantom(kind: str, dims, spacing, seed: int = 0, hu0: int = 0,
                 noise_sigma: float = 0.0) -> Phantom:
    L = _load()
    nx, ny, nz = dims
    hu = np.empty((nz, ny, nx), dtype=np.int16)
    k = {"uniform": 0, "slab": 1, "thorax": 2}[kind]
    L.fdcgen_phantom(k, seed, nx, ny, nz, *[float(s) for s in spacing], int(hu0),
                     float(noise_sigma), hu.ctypes.data)
    return Phantom(hu, tuple(float(s) for s in spacing))


def material_table(kind: str = "config2") -> np.ndarray:
    """HU -> (density, mass stopping-power ratio, mass scattering-power ratio) knots.

    'config2': BASELINE.json configs[1] density knots; s = 1 (reading A3: linear stopping-power
    ratio = density); scattering-power ratio knots are this build's choice (reading A4).
    'water': single material, all ones."""
    if kind == "water":
        rows = [(-1000.0, 1.0, 1.0, 1.0), (3000.0, 1.0, 1.0, 1.0)]
    elif kind == "config2":
        rows = [(-1000.0, 0.001, 1.0, 1.0), (-750.0, 0.26, 1.0, 1.0), (0.0, 1.0, 1.0, 1.0),
                (1000.0, 1.85, 1.0, 1.20), (2000.0, 2.3, 1.0, 1.30)]
    else:
        raise ValueError(kind)
    return np.array(rows, dtype=KNOT_DTYPE)


def split_even(n: int, parts: int) -> np.ndarray:
    """n_b = floor(N(b+1)/B) - floor(N b/B)."""
    b = np.arange(parts + 1, dtype=object)
    edges = np.array([(n * int(x)) // parts for x in b], dtype=np.uint64)
    return (edges[1:] - edges[:-1]).astype(np.uint64)


def _gantry_frame(g_deg: int):
    """A19: gantry angle rotates about z: dir=(sin g, cos g, 0), e1=(0,0,1), e2=(cos g,-sin g,0)."""
    h = math.sqrt(3.0) / 2.0
    sc = {0: (0.0, 1.0), 120: (h, -0.5), 240: (-h, -0.5)}[g_deg]
    s, c = sc
    return (0.0, 0.0, 1.0), (c, -s, 0.0), (s, c, 0.0)


def make_plan(extent, gantries, layers_mev, spot_offsets, sigma, n_protons) -> np.ndarray:
    """Field list -> beamlets, ordered field-major, layer, spot_u, spot_v (A19, A20).
    Isocentre = grid centre; source plane 400 mm upstream; equal protons per beamlet."""
    iso = np.array(extent, dtype=np.float64) * 0.5
    rows = []
    for g in gantries:
        e1, e2, d = _gantry_frame(g)
        origin = iso - 400.0 * np.array(d)
        for E in layers_mev:
            for su in spot_offsets:
                for sv in spot_offsets:
                    rows.append((origin, e1, e2, d, E, su, sv, sigma, 0))
    bl = np.zeros(len(rows), dtype=BEAMLET_DTYPE)
    for i, r in enumerate(rows):
        bl[i] = r
    bl["n_protons"] = split_even(n_protons, len(rows))
    return bl


def single_beamlet(origin, energy, sigma, n_protons, e1=(1, 0, 0), e2=(0, 1, 0), d=(0, 0, 1)):
    bl = np.zeros(1, dtype=BEAMLET_DTYPE)
    bl[0] = (origin, e1, e2, d, energy, 0.0, 0.0, sigma, n_protons)
    return bl


def bins_hit(beamlets: np.ndarray, e_min: float, e_bin: float) -> list:
    """Energy bins a plan touches (for lazy DB generation): smallest nominal energy >= E0,
    evaluated in float32 like the method does -- duplicated here only to decide
    which bins to GENERATE; a wrong guess shows up as FDC_ERANGE, never as a wrong dose."""
    e = beamlets["energy_mev"].astype(np.float32)
    x = (e - np.float32(e_min)) / np.float32(e_bin)
    return sorted(set(int(v) for v in np.maximum(np.ceil(x), 0).astype(np.int64)))


# ----------------------------------------------------------------------------- presets
_FULL = {1: 100_000, 2: 1_000_000, 3: 10_000_000, 4: 50_000_000, 5: 200_000_000}


def workload(cfg: int, n_protons: int | None = None, tracks_per_bin: int | None = None,
             lazy_db: bool = True) -> Workload:
    """Preset ``cfg`` in 1..5 = BASELINE.json configs[cfg-1].

    ``n_protons`` / ``tracks_per_bin`` override the full sizes (reduced-size parity cases);
    ``lazy_db`` builds only the energy bins the plan touches (identical tracks)."""
    n = _FULL[cfg] if n_protons is None else int(n_protons)
    if cfg == 1:
        ph = make_phantom("uniform", (64, 64, 64), (2.0, 2.0, 2.0), hu0=0)
        tpb = 2000 if tracks_per_bin is None else tracks_per_bin
        db = make_trackdb(101, 100.0, 1.0, 1, tpb)
        bl = single_beamlet((64.0, 64.0, 0.0), 100.0, 0.0, n)
        return Workload("config1_water64", ph, material_table("config2"), db, bl, n, 1)
    if cfg == 2:
        ph = make_phantom("slab", (128, 128, 128), (1.0, 1.0, 1.0))
        tpb = 10_000 if tracks_per_bin is None else tracks_per_bin
        bl = single_beamlet((64.0, 64.0, 0.0), 150.0, 5.0, n)
        bins = bins_hit(bl, 140.0, 1.0) if lazy_db else None
        db = make_trackdb(102, 140.0, 1.0, 21, tpb, bins)
        return Workload("config2_slab128", ph, material_table("config2"), db, bl, n, 2)
    if cfg in (3, 4):
        ph = make_phantom("thorax", (256, 256, 128), (2.0, 2.0, 2.0), seed=203, noise_sigma=20.0)
        layers = [100.0 + l * 100.0 / 23.0 for l in range(24)]
        if cfg == 3:
            bl = make_plan((512.0, 512.0, 256.0), [0], layers, [-15.0 + 5.0 * i for i in range(7)], 4.0, n)
        else:
            bl = make_plan((512.0, 512.0, 256.0), [0, 120, 240], layers,
                           [-20.0 + 5.0 * i for i in range(9)], 4.0, n)
        tpb = 10_000 if tracks_per_bin is None else tracks_per_bin
        bins = bins_hit(bl, 70.0, 1.0) if lazy_db else None
        db = make_trackdb(103, 70.0, 1.0, 181, tpb, bins)
        return Workload("config%d_thorax256" % cfg, ph, material_table("config2"), db, bl, n, cfg)
    if cfg == 5:
        ph = make_phantom("thorax", (512, 512, 256), (1.0, 1.0, 1.0), seed=205, noise_sigma=20.0)
        layers = [70.0 + l * 160.0 / 39.0 for l in range(40)]
        bl = make_plan((512.0, 512.0, 256.0), [0, 120, 240], layers,
                       [-20.0 + 5.0 * i for i in range(9)], 4.0, n)
        tpb = 20_000 if tracks_per_bin is None else tracks_per_bin
        bins = bins_hit(bl, 70.0, 1.0) if lazy_db else None
        db = make_trackdb(105, 70.0, 1.0, 181, tpb, bins)
        return Workload("config5_thorax512", ph, material_table("config2"), db, bl, n, 5)
    raise ValueError("cfg must be 1..5")


# ----------------------------------------------------------------------------- secondaries (R15), synthetic
def add_secondaries(db: TrackDB, seed: int, fraction: float = 1.0):
    """A synthetic secondary table for a generated database (stands in for the secondary
    trajectories of the paper's GEANT4 histories).  Recipe, per primary track j with at least
    8 steps, with probability `fraction`: one secondary; it branches at the end of step b = floor(u1 (len - 4));
    it carries E_s = (0.1 + 0.3 u2) E[b]; its steps are the tail of another primary p of the same database,
    from that track's first step with E <= E_s on, rotated as a whole so that its first step leaves at polar
    angle 10 + 30 u3 degrees and azimuth 2 pi u4 from the parent's direction of step b.  u1..u4 and p from
    numpy's PCG64 seeded by `seed`.  Returns (db with the secondary tracks appended past the last bin,
    (sec_first, sec_track, sec_step)).  Input preparation only: float64 numpy, rounded to float32."""
    rng = np.random.default_rng(seed)
    off = db.track_off.astype(np.int64)
    n_p = db.n_tracks
    lens = off[1:] - off[:-1]
    cand = np.nonzero(lens >= 8)[0]
    cand = cand[rng.random(len(cand)) < fraction]
    D = np.stack([db.dx, db.dy, db.dz], 1).astype(np.float64)
    new_steps, new_dE, new_E, new_len, step_of = [], [], [], [], []
    pool = np.nonzero(lens > 0)[0]
    for j in cand:
        u = rng.random(4)
        b = int(u[0] * (lens[j] - 4))
        e_s = (0.1 + 0.3 * u[1]) * float(db.E[off[j] + b])
        p = int(pool[rng.integers(len(pool))])
        Ep = db.E[off[p]:off[p + 1]]
        k = int(np.searchsorted(-Ep, -np.float32(e_s), side="left"))          # first step with E <= E_s (E non-increasing)
        if k >= lens[p]:
            continue
        seg = D[off[p] + k:off[p + 1]]
        a = seg[0] / max(np.linalg.norm(seg[0]), 1e-30)                       # its own first direction
        d = D[off[j] + b]; d = d / max(np.linalg.norm(d), 1e-30)              # the parent's direction at the branch
        th, ph = np.deg2rad(10.0 + 30.0 * u[2]), 2.0 * np.pi * u[3]
        e1 = np.cross(d, [1.0, 0.0, 0.0] if abs(d[0]) < 0.9 else [0.0, 1.0, 0.0]); e1 /= np.linalg.norm(e1); e2 = np.cross(d, e1)
        t = np.cos(th) * d + np.sin(th) * (np.cos(ph) * e1 + np.sin(ph) * e2)  # where the secondary leaves
        v = np.cross(a, t); c = float(a @ t)
        vx = np.array([[0, -v[2], v[1]], [v[2], 0, -v[0]], [-v[1], v[0], 0]])
        Rm = np.eye(3) + vx + vx @ vx / (1.0 + c) if c > -0.999999 else -np.eye(3)
        new_steps.append(seg @ Rm.T); new_dE.append(db.dE[off[p] + k:off[p + 1]]); new_E.append(Ep[k:])
        new_len.append(len(seg)); step_of.append((int(j), b))
    if not new_len:
        return db, (np.zeros(n_p + 1, np.uint32), np.zeros(0, np.uint32), np.zeros(0, np.uint32))
    S = np.concatenate(new_steps).astype(np.float32)
    db2 = TrackDB(np.concatenate([db.dx, S[:, 0]]), np.concatenate([db.dy, S[:, 1]]), np.concatenate([db.dz, S[:, 2]]),
                  np.concatenate([db.dE] + new_dE).astype(np.float32), np.concatenate([db.E] + new_E).astype(np.float32),
                  np.concatenate([db.track_off, db.track_off[-1] + np.cumsum(new_len).astype(np.uint64)]).astype(np.uint64),
                  db.bin_first.copy(), db.e_min, db.e_bin)
    first = np.zeros(db2.n_tracks + 1, dtype=np.int64)
    for (j, _) in step_of:
        first[j + 1] += 1
    first = np.cumsum(first).astype(np.uint32)                                 # candidates ascend in j: the table is already ordered
    return db2, (first, np.arange(n_p, n_p + len(step_of), dtype=np.uint32), np.array([b for (_, b) in step_of], dtype=np.uint32))
