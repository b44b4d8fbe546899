"""ctypes loader for the oracle (oracle/oracle.cpp).  TEST INFRASTRUCTURE, NOT PRODUCT.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this.  It imports nothing from paper_1011_2188_b200 (the CUDA path) and vice versa.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "oracle.cpp")
_LIB = os.path.join(_HERE, "liboracle.so")
_lib = None

FLAG_RANDOM_AZIMUTH = 1
FLAG_REALIGN_START = 32


class TrackDBStruct(ctypes.Structure):
    _fields_ = [("dx", ctypes.c_void_p), ("dy", ctypes.c_void_p), ("dz", ctypes.c_void_p),
                ("dE", ctypes.c_void_p), ("E", ctypes.c_void_p), ("n_steps", ctypes.c_uint64),
                ("track_off", ctypes.c_void_p), ("n_tracks", ctypes.c_uint32),
                ("bin_first", ctypes.c_void_p), ("n_bins", ctypes.c_uint32),
                ("e_min", ctypes.c_float), ("e_bin", ctypes.c_float)]


class StatsStruct(ctypes.Structure):
    _fields_ = [(n, ctypes.c_uint64) for n in ("protons", "proton_steps", "deposits", "missed", "escaped",
                                               "stopped", "grid_sum", "q_replayed", "q_escaped")]

    def as_dict(self):
        return {n: int(getattr(self, n)) for n, _ in self._fields_}


def build(force: bool = False) -> str:
    """g++ -O2 -ffp-contract=off (the arithmetic contract)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + ".tmp.%d" % os.getpid()
        subprocess.check_call(["g++", "-std=c++17", "-O2", "-ffp-contract=off", "-fno-fast-math",
                               "-shared", "-fPIC", "-o", tmp, _SRC])
        os.replace(tmp, _LIB)
    return _LIB


def lib():
    global _lib
    if _lib is None:
        L = ctypes.CDLL(build())
        L.oracle_signed_unit.restype = ctypes.c_float
        L.oracle_signed_unit.argtypes = [ctypes.c_uint32]
        L.oracle_ln.restype = ctypes.c_double
        L.oracle_ln.argtypes = [ctypes.c_double]
        L.oracle_energy_bin.restype = ctypes.c_int
        L.oracle_energy_bin.argtypes = [ctypes.c_float] * 3
        _lib = L
    return _lib


def _p(a):
    return ctypes.c_void_p(a.ctypes.data)


def philox(ctr, key):
    c = np.asarray(ctr, dtype=np.uint32); k = np.asarray(key, dtype=np.uint32); o = np.zeros(4, dtype=np.uint32)
    lib().oracle_philox4x32_10(_p(c), _p(k), _p(o))
    return o


def material_lut(table):
    t = np.ascontiguousarray(table)
    rho, w, f = (np.zeros(4096, dtype=np.float32) for _ in range(3))
    lib().oracle_material_lut(_p(t), ctypes.c_int(len(t)), _p(rho), _p(w), _p(f))
    return rho, w, f


def _db_struct(db):
    arrs = [np.ascontiguousarray(a, dtype=np.float32) for a in (db.dx, db.dy, db.dz, db.dE, db.E)]
    off = np.ascontiguousarray(db.track_off, dtype=np.uint64)
    bf = np.ascontiguousarray(db.bin_first, dtype=np.uint32)
    s = TrackDBStruct(*[a.ctypes.data for a in arrs], arrs[0].shape[0], off.ctypes.data, off.shape[0] - 1,
                      bf.ctypes.data, bf.shape[0] - 1, db.e_min, db.e_bin)
    return s, (arrs, off, bf)


def _common_args(phantom, table, db, beamlets):
    hu = np.ascontiguousarray(phantom.hu, dtype=np.int16)
    nx, ny, nz = phantom.dims
    t = np.ascontiguousarray(table)
    bl = np.ascontiguousarray(beamlets)
    dbs, keep = _db_struct(db)
    args = [_p(hu), ctypes.c_int(nx), ctypes.c_int(ny), ctypes.c_int(nz)] + \
           [ctypes.c_float(s) for s in phantom.spacing] + \
           [_p(t), ctypes.c_int(len(t)), ctypes.byref(dbs), _p(bl), ctypes.c_uint32(len(bl))]
    return args, (hu, t, bl, dbs, keep)


def _range_args(first, n, stride, seed, flags):
    return [ctypes.c_uint64(first), ctypes.c_uint64(n), ctypes.c_uint64(stride), ctypes.c_uint64(seed),
            ctypes.c_uint32(flags)]


def run(phantom, table, db, beamlets, seed, first=0, n=None, stride=1, flags=FLAG_RANDOM_AZIMUTH,
        grid=None, f64=False, end_state=False):
    """Whole path, single thread.  Returns (grid u64 [nz,ny,nx], stats dict[, end_state])."""
    if n is None:
        n = int(beamlets["n_protons"].sum()) - first
    if grid is None:
        grid = np.zeros(phantom.hu.shape, dtype=np.uint64)
    st = StatsStruct()
    a, keep = _common_args(phantom, table, db, beamlets)
    a += _range_args(first, n, stride, seed, flags) + [_p(grid), ctypes.byref(st)]
    es = None
    if f64:
        es = np.zeros((n, 6), dtype=np.float64) if end_state else None
        a.append(_p(es) if es is not None else None)
        rc = lib().oracle_run_f64(*a)
    else:
        rc = lib().oracle_run(*a)
    if rc != 0:
        raise RuntimeError("oracle_run failed rc=%d" % rc)
    d = st.as_dict()
    d["grid_sum"] = int(grid.sum(dtype=np.uint64))
    return (grid, d, es) if (f64 and end_state) else (grid, d)


PARTICLE_DTYPE = np.dtype([("pos", "<f4", 3), ("dir", "<f4", 3), ("energy_mev", "<f4"), ("reserved", "<f4")], align=True)


def run_phase_space(phantom, table, db, particles, seed, first_id=0, flags=FLAG_RANDOM_AZIMUTH):
    """R12: the path started from a phase-space array.  Returns (grid, stats)."""
    ps = np.ascontiguousarray(particles, dtype=PARTICLE_DTYPE)
    grid = np.zeros(phantom.hu.shape, dtype=np.uint64)
    st = StatsStruct()
    a, keep = _common_args(phantom, table, db, np.zeros(0, dtype=ps.dtype))
    a = a[:-2] + [_p(ps), ctypes.c_uint64(len(ps)), ctypes.c_uint64(first_id), ctypes.c_uint64(seed), ctypes.c_uint32(flags),
                  _p(grid), ctypes.byref(st)]
    rc = lib().oracle_run_phase_space(*a)
    if rc != 0:
        raise RuntimeError("oracle_run_phase_space failed rc=%d" % rc)
    d = st.as_dict()
    d["grid_sum"] = int(grid.sum(dtype=np.uint64))
    return grid, d


def frame_rule(d):
    d = np.ascontiguousarray(d, dtype=np.float32); e1 = np.zeros(3, np.float32); e2 = np.zeros(3, np.float32)
    lib().oracle_frame_rule(_p(d), _p(e1), _p(e2))
    return e1, e2


def run_sq(phantom, table, db, beamlets, seed, first=0, n=None, stride=1, flags=FLAG_RANDOM_AZIMUTH, by_history=True):
    """Whole path plus the sum-of-squares tallies (R10).  Returns (grid, sq_by_visit,
    sq_by_history or None, stats): u64 grids [nz,ny,nx]; squares in quanta of 2^-32 MeV^2."""
    if n is None:
        n = int(beamlets["n_protons"].sum()) - first
    grid = np.zeros(phantom.hu.shape, dtype=np.uint64)
    sqv = np.zeros(phantom.hu.shape, dtype=np.uint64)
    sqh = np.zeros(phantom.hu.shape, dtype=np.uint64) if by_history else None
    st = StatsStruct()
    a, keep = _common_args(phantom, table, db, beamlets)
    a += _range_args(first, n, stride, seed, flags) + [_p(grid), _p(sqv), _p(sqh) if by_history else None, ctypes.byref(st)]
    rc = lib().oracle_run_sq(*a)
    if rc != 0:
        raise RuntimeError("oracle_run_sq failed rc=%d" % rc)
    d = st.as_dict()
    d["grid_sum"] = int(grid.sum(dtype=np.uint64))
    return grid, sqv, sqh, d


def run_secondaries(phantom, table, db, sec, beamlets, seed, first=0, n=None, stride=1, flags=FLAG_RANDOM_AZIMUTH, squares=False):
    """R15: histories with secondaries.  sec = (sec_first[n_tracks+1], sec_track[n_sec], sec_step[n_sec]) uint32.
    Returns (grid, stats) or (grid, sq_by_visit, sq_by_history, stats) with squares=True."""
    if n is None:
        n = int(beamlets["n_protons"].sum()) - first
    sf, stt, sst = (np.ascontiguousarray(a, dtype=np.uint32) for a in sec)
    assert len(sf) == db.n_tracks + 1 and len(stt) == len(sst) == int(sf[-1])
    grid = np.zeros(phantom.hu.shape, dtype=np.uint64)
    sqv = np.zeros(phantom.hu.shape, dtype=np.uint64) if squares else None
    sqh = np.zeros(phantom.hu.shape, dtype=np.uint64) if squares else None
    st = StatsStruct()
    a, keep = _common_args(phantom, table, db, beamlets)
    a = a[:-2] + [_p(sf), _p(stt) if len(stt) else None, _p(sst) if len(sst) else None] + a[-2:]
    a += _range_args(first, n, stride, seed, flags) + [_p(grid), _p(sqv) if squares else None, _p(sqh) if squares else None, ctypes.byref(st)]
    rc = lib().oracle_run_secondaries(*a)
    if rc != 0:
        raise RuntimeError("oracle_run_secondaries failed rc=%d" % rc)
    d = st.as_dict()
    d["grid_sum"] = int(grid.sum(dtype=np.uint64))
    return (grid, sqv, sqh, d) if squares else (grid, d)


# ---------------------------------------------------------------- PAPER.md §2.4, eq. (1), (2), mean uncertainty (numpy f64)
E_QUANTUM = 2.0 ** -24      # MeV per unit of the energy grid
SQ_QUANTUM = 2.0 ** -32     # MeV^2 per unit of the squares grid


def sigma_history(grid, sq, n_histories):
    """Eq. (2) (sums over all N primaries: reading A11), per voxel, of the MEAN energy per
    history: sigma = sqrt(max(0, (sum e^2 / N - (sum e / N)^2)) / (N - 1)).  Returns (mean, sigma) in MeV."""
    N = float(n_histories)
    m1 = (grid.astype(np.float64) * E_QUANTUM) / N
    m2 = (sq.astype(np.float64) * SQ_QUANTUM) / N
    var = (m2 - m1 * m1) / (N - 1.0)
    return m1, np.sqrt(np.maximum(var, 0.0))


def sigma_batch(grids):
    """Eq. (1): n independent batches D_i -> (mean, sqrt(sum (D_i - mean)^2 / (n (n - 1)))), MeV."""
    n = len(grids)
    D = [g.astype(np.float64) * E_QUANTUM for g in grids]
    mean = D[0].copy()
    for d in D[1:]:
        mean = mean + d
    mean = mean / float(n)
    ss = np.zeros_like(mean)
    for d in D:
        ss = ss + (d - mean) * (d - mean)
    return mean, np.sqrt(ss / float(n * (n - 1)))


def mean_uncertainty(mean, sigma, rho):
    """average of sigma/D over the voxels whose DOSE (energy / density; the voxel volume is
    common) exceeds half the maximum dose.  Returns (value, number of voxels averaged)."""
    dose = mean / rho.astype(np.float64)
    sel = dose > 0.5 * dose.max()
    rel = sigma[sel] / mean[sel]
    return float(rel.mean()), int(sel.sum())


def density(phantom, table):
    """rho (f32) per voxel from the material LUT (R1)."""
    rho, w, f = material_lut(table)
    return rho[np.clip(phantom.hu.astype(np.int32), -1024, 3071) + 1024]


def run_trace(phantom, table, db, beamlets, seed, first=0, n=1, stride=1, flags=FLAG_RANDOM_AZIMUTH, cap=1 << 20):
    """f32 run recording every deposit: returns grid, stats, (voxel, share, step), end_state[n,6]."""
    grid = np.zeros(phantom.hu.shape, dtype=np.uint64)
    st = StatsStruct()
    vox = np.zeros(cap, dtype=np.uint64); share = np.zeros(cap, dtype=np.uint64); step = np.zeros(cap, dtype=np.uint32)
    ntr = ctypes.c_uint64(0)
    es = np.zeros((n, 6), dtype=np.float32)
    a, keep = _common_args(phantom, table, db, beamlets)
    a += _range_args(first, n, stride, seed, flags) + [_p(grid), ctypes.byref(st), _p(vox), _p(share), _p(step),
                                                        ctypes.c_uint64(cap), ctypes.byref(ntr), _p(es)]
    rc = lib().oracle_run_trace(*a)
    if rc != 0:
        raise RuntimeError("oracle_run_trace failed rc=%d" % rc)
    k = int(ntr.value)
    d = st.as_dict(); d["grid_sum"] = int(grid.sum(dtype=np.uint64))
    return grid, d, (vox[:k], share[:k], step[:k]), es


def sample(phantom, table, db, beamlets, seed, first=0, n=1, stride=1, flags=FLAG_RANDOM_AZIMUTH):
    """R2-R6 only: per-proton start state."""
    out = dict(beamlet=np.zeros(n, np.uint32), track=np.zeros(n, np.uint32), k0=np.zeros(n, np.uint64),
               p=np.zeros((n, 3), np.float32), R=np.zeros((n, 3, 3), np.float32), iv=np.zeros((n, 3), np.int32),
               missed=np.zeros(n, np.int32), csg=np.zeros((n, 4), np.float32))
    a, keep = _common_args(phantom, table, db, beamlets)
    a += _range_args(first, n, stride, seed, flags)
    a += [_p(out[k]) for k in ("beamlet", "track", "k0", "p", "R", "iv", "missed", "csg")]
    rc = lib().oracle_sample(*a)
    if rc != 0:
        raise RuntimeError("oracle_sample failed rc=%d" % rc)
    return out


def to_gy(grid, phantom, table):
    hu = np.ascontiguousarray(phantom.hu, dtype=np.int16)
    g = np.ascontiguousarray(grid, dtype=np.uint64)
    t = np.ascontiguousarray(table)
    dose = np.zeros(hu.shape, dtype=np.float32)
    lib().oracle_to_gy(_p(g), _p(hu), ctypes.c_uint64(g.size), *[ctypes.c_float(s) for s in phantom.spacing],
                       _p(t), ctypes.c_int(len(t)), _p(dose))
    return dose


# ---------------------------------------------------------------- PAPER.md:L94 gamma index (Low et al. 1998), numpy f64
def gamma_index(dose_ref, dose_eval, spacing, dose_tol_frac=0.03, dist_tol_mm=3.0, search_mm=None, cutoff_frac=0.0):
    """Discrete gamma index of dose_eval against dose_ref (both [nz,ny,nx] f32), the definition written out:
    Gamma(r) = min over voxels r' with |r' - r| <= search_mm (offsets in whole voxels, inside the grid) of
               sqrt(|r' - r|^2 / dist_tol^2 + (D_eval(r') - D_ref(r))^2 / dD^2),   dD = dose_tol_frac * max(D_ref)
    (global dose criterion; no interpolation between voxels).  Arithmetic in f64 in this order:
    d2 = ((ox*sx)^2 + (oy*sy)^2) + (oz*sz)^2;  g2 = (diff*diff) * (1/dD^2) + d2 * (1/dist_tol^2).
    Returns (gamma f32 map, pass fraction = share of voxels with D_ref > cutoff_frac*max(D_ref) whose
    gamma <= 1, number of such voxels)."""
    ref = np.asarray(dose_ref, dtype=np.float32).astype(np.float64)
    ev = np.asarray(dose_eval, dtype=np.float32).astype(np.float64)
    sx, sy, sz = (float(np.float32(s)) for s in spacing)
    search = float(np.float32(dist_tol_mm if search_mm is None else search_mm))
    dmax = float(ref.max())
    dD = float(np.float32(dose_tol_frac)) * dmax
    c_dose = 1.0 / (dD * dD)
    c_dist = 1.0 / (float(np.float32(dist_tol_mm)) * float(np.float32(dist_tol_mm)))
    rx, ry, rz = int(np.floor(search / sx)), int(np.floor(search / sy)), int(np.floor(search / sz))
    nz, ny, nx = ref.shape
    g2 = np.full(ref.shape, np.inf)
    for oz in range(-rz, rz + 1):
        for oy in range(-ry, ry + 1):
            for ox in range(-rx, rx + 1):
                d2 = ((ox * sx) * (ox * sx) + (oy * sy) * (oy * sy)) + (oz * sz) * (oz * sz)
                if d2 > search * search:
                    continue
                # destination (reference) slices and source (evaluated, shifted by the offset) slices
                z0, z1 = max(0, -oz), min(nz, nz - oz); y0, y1 = max(0, -oy), min(ny, ny - oy); x0, x1 = max(0, -ox), min(nx, nx - ox)
                if z0 >= z1 or y0 >= y1 or x0 >= x1:
                    continue
                diff = ev[z0 + oz:z1 + oz, y0 + oy:y1 + oy, x0 + ox:x1 + ox] - ref[z0:z1, y0:y1, x0:x1]
                cand = (diff * diff) * c_dose + d2 * c_dist
                sub = g2[z0:z1, y0:y1, x0:x1]
                np.minimum(sub, cand, out=sub)
    gamma = np.sqrt(g2).astype(np.float32)
    sel = ref > float(np.float32(cutoff_frac)) * dmax
    n = int(sel.sum())
    return gamma, (float((gamma[sel] <= 1.0).sum()) / n if n else 0.0), n


# ---------------------------------------------------------------- PAPER.md:L104-108 profile comparators, numpy f64
def profile(values, axis, fixed_a, fixed_b, half_width_a=2, half_width_b=2):
    """R16 (Fig. 2-3: depth and cross-field profiles, "each profile is calculated along a five voxel
    thick line").  values: [nz,ny,nx] array (a dose grid, f32; or the u64 energy grid, then the result is in MeV).
    The line runs along `axis` (0 = x, 1 = y, 2 = z) through the voxel whose indices on the other two axes (a = the
    lower-numbered one, b = the other) are (fixed_a, fixed_b); it is thickened to the columns with
    |a - fixed_a| <= half_width_a and |b - fixed_b| <= half_width_b that lie inside the grid, and out[k] is the
    mean over those columns: summed in f64 with b outer and a inner, then divided by their number.  The energy
    grid is summed as integers and multiplied once by 2^-24.  Returns float64 [n_axis]."""
    v = np.asarray(values)
    nz, ny, nx = v.shape
    n = (nx, ny, nz)
    ia, ib = (1 if axis == 0 else 0), (1 if axis == 2 else 2)
    assert 0 <= fixed_a < n[ia] and 0 <= fixed_b < n[ib]
    a0, a1 = max(0, fixed_a - half_width_a), min(n[ia] - 1, fixed_a + half_width_a)
    b0, b1 = max(0, fixed_b - half_width_b), min(n[ib] - 1, fixed_b + half_width_b)
    is_int = v.dtype.kind in "ui"
    acc = np.zeros(n[axis], dtype=np.uint64 if is_int else np.float64)
    for b in range(b0, b1 + 1):
        for a in range(a0, a1 + 1):
            idx = [None, None, None]                       # numpy index order is (z, y, x) = axes (2, 1, 0)
            idx[2 - axis] = slice(None); idx[2 - ia] = a; idx[2 - ib] = b
            col = v[tuple(idx)]
            acc = acc + (col.astype(np.uint64) if is_int else col.astype(np.float64))
    cnt = float((a1 - a0 + 1) * (b1 - b0 + 1))
    return (acc.astype(np.float64) * E_QUANTUM if is_int else acc) / cnt


def rms_diff(dose_ref, dose_eval):
    """R17 ("the difference between the GFDC- and GEANT4-calculated doses for each voxel in the
    anatomic phantom divided by the maximum GEANT4 voxel dose has a RMS value of 0.5 %"):
    sqrt(mean over ALL voxels of ((eval - ref) * (1 / max(ref)))^2), f64.  Returns (rms, max(ref))."""
    ref = np.asarray(dose_ref, dtype=np.float32).astype(np.float64)
    ev = np.asarray(dose_eval, dtype=np.float32).astype(np.float64)
    dmax = float(ref.max())
    x = (ev - ref) * (1.0 / dmax)
    return float(np.sqrt(np.sum(x * x) / float(x.size))), dmax
