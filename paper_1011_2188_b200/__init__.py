"""Thin ctypes binding over the C-ABI of include/fdc.h (libfdc.so, CUDA kernels for sm_100a).

Same names as the C functions; argument marshalling only -- every stage of the path (sampling,
track selection, transport, deposit, Gy conversion) runs in the library's kernels.  torch is used
for device memory and the stream, nothing else.  There is NO CPU fallback: a missing library or
a non-sm_100 device raises.
"""
from __future__ import annotations

import ctypes
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.environ.get("FDC_LIB") or os.path.join(_HERE, "libfdc.so")      # FDC_LIB: another build of the same library

FDC_RANDOM_AZIMUTH = 1
FDC_DOSE_TO_HOST = 2
FDC_NO_SORT = 4
FDC_NO_AGGREGATE = 8
FDC_TALLY_SQUARES = 16
FDC_REALIGN_START = 32
FDC_DIAG_REDS = 64
FDC_SORT_SPATIAL = 128
FDC_NO_LAT = 256
FDC_PRIVATE_TALLY = 512
FDC_WARP_AGGREGATE = 1024
FDC_MAT_TILED = 2048
FDC_MAT_LINEAR = 4096
FDC_SQUARES_BY_HISTORY = 8192

FDC_NOALLOC_MAX_BATCHES = 32          # fdc_uncertainty_batch_noalloc: what its fixed scratch holds

FDC_OK, FDC_EINVAL, FDC_ENOTRACKS, FDC_ERANGE, FDC_ENOMEM, FDC_ECUDA, FDC_EARCH = 0, -1, -2, -3, -4, -5, -6
FDC_WSEGMENTED = 1                    # positive codes are warnings: outputs valid (include/fdc.h)

EXPORTS = ["fdc_create", "fdc_load_tracks", "fdc_run", "fdc_to_gy", "fdc_get_edep_fixed", "fdc_set_edep_fixed", "fdc_edep_device_ptr",
           "fdc_get_stats", "fdc_reset", "fdc_destroy", "fdc_strerror", "fdc_last_error",
           "fdc_get_sq_fixed", "fdc_set_sq_fixed", "fdc_uncertainty_history", "fdc_uncertainty_batch", "fdc_run_phase_space", "fdc_gamma_index",
           "fdc_profile", "fdc_rms_diff", "fdc_set_secondaries", "fdc_uncertainty_batch_noalloc",
           "fdc_last_call_info", "fdc_trace_reds"]          # the last two: diagnostics (include/fdc.h)

BEAMLET_DTYPE = np.dtype([("origin", "<f4", 3), ("e1", "<f4", 3), ("e2", "<f4", 3), ("dir", "<f4", 3),
                          ("energy_mev", "<f4"), ("spot_u_mm", "<f4"), ("spot_v_mm", "<f4"),
                          ("sigma_mm", "<f4"), ("n_protons", "<u8")], align=True)
PARTICLE_DTYPE = np.dtype([("pos", "<f4", 3), ("dir", "<f4", 3), ("energy_mev", "<f4"), ("reserved", "<f4")], align=True)
KNOT_DTYPE = np.dtype([("hu", "<f4"), ("density_g_cc", "<f4"), ("mass_spr", "<f4"), ("mass_scpr", "<f4")], align=True)


class FdcError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__("fdc error %d: %s" % (code, msg))
        self.code = code


class FdcWarning(RuntimeWarning):
    """A positive return code of the library: the call did its work, its outputs are valid."""


class _TrackDB(ctypes.Structure):
    _fields_ = [("dx", ctypes.c_void_p), ("dy", ctypes.c_void_p), ("dz", ctypes.c_void_p), ("dE", ctypes.c_void_p),
                ("E", ctypes.c_void_p), ("n_steps", ctypes.c_uint64), ("track_off", ctypes.c_void_p),
                ("n_tracks", ctypes.c_uint32), ("bin_first", ctypes.c_void_p), ("n_bins", ctypes.c_uint32),
                ("e_min_mev", ctypes.c_float), ("e_bin_mev", ctypes.c_float)]


class _CallInfo(ctypes.Structure):
    _fields_ = [("ms_total", ctypes.c_float), ("ms_transport", ctypes.c_float), ("ms_sort", ctypes.c_float), ("ms_gy", ctypes.c_float),
                ("launches", ctypes.c_uint32), ("sq_history_flushes", ctypes.c_uint32), ("h2d_bytes", ctypes.c_uint64), ("d2h_bytes", ctypes.c_uint64),
                ("reds_sent", ctypes.c_uint64), ("reds_traced", ctypes.c_uint64)]


class _Stats(ctypes.Structure):
    _fields_ = [(n, ctypes.c_uint64) for n in ("protons", "proton_steps", "deposits", "missed", "escaped", "stopped",
                                               "grid_sum", "q_replayed", "q_escaped")]


_lib = None


def lib():
    """Load libfdc.so (built in-tree by build.py / __graft_entry__.build()).  Fails loudly if absent."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError("%s not found: build it with `python -m paper_1011_2188_b200.build` "
                              "(there is no CPU fallback)" % LIB_PATH)
        L = ctypes.CDLL(LIB_PATH)
        vp, i32, u32, u64, f32 = ctypes.c_void_p, ctypes.c_int, ctypes.c_uint32, ctypes.c_uint64, ctypes.c_float
        L.fdc_create.restype = i32
        L.fdc_create.argtypes = [ctypes.POINTER(vp), i32, vp, vp, i32, i32, i32, f32, f32, f32, vp, i32, i32]
        L.fdc_load_tracks.restype = i32
        L.fdc_load_tracks.argtypes = [vp, ctypes.POINTER(_TrackDB), i32]
        L.fdc_run.restype = i32
        L.fdc_run.argtypes = [vp, vp, u32, u64, u64, u64, u64, u32, vp]
        L.fdc_get_edep_fixed.restype = i32
        L.fdc_get_edep_fixed.argtypes = [vp, vp, i32]
        L.fdc_set_edep_fixed.restype = i32
        L.fdc_set_edep_fixed.argtypes = [vp, vp, i32]
        L.fdc_get_stats.restype = i32
        L.fdc_get_stats.argtypes = [vp, ctypes.POINTER(_Stats)]
        L.fdc_reset.restype = i32
        L.fdc_reset.argtypes = [vp]
        L.fdc_destroy.restype = None
        L.fdc_destroy.argtypes = [vp]
        L.fdc_strerror.restype = ctypes.c_char_p
        L.fdc_strerror.argtypes = [i32]
        L.fdc_last_error.restype = ctypes.c_char_p
        L.fdc_last_error.argtypes = [vp]
        L.fdc_last_call_info.restype = i32
        L.fdc_last_call_info.argtypes = [vp, ctypes.POINTER(_CallInfo)]
        L.fdc_trace_reds.restype = i32
        L.fdc_trace_reds.argtypes = [vp, vp, u64]
        L.fdc_to_gy.restype = i32
        L.fdc_to_gy.argtypes = [vp, vp, i32]
        L.fdc_edep_device_ptr.restype = i32
        L.fdc_edep_device_ptr.argtypes = [vp, ctypes.POINTER(vp), ctypes.POINTER(vp)]
        L.fdc_profile.restype = i32
        L.fdc_profile.argtypes = [vp, vp, i32, i32, i32, i32, i32, vp, i32]
        L.fdc_rms_diff.restype = i32
        L.fdc_rms_diff.argtypes = [vp, vp, vp, ctypes.POINTER(ctypes.c_double), ctypes.POINTER(ctypes.c_double)]
        for f in (L.fdc_get_sq_fixed, L.fdc_set_sq_fixed):
            f.restype = i32
            f.argtypes = [vp, vp, i32]
        L.fdc_run_phase_space.restype = i32
        L.fdc_run_phase_space.argtypes = [vp, vp, u64, i32, u64, u64, u32, vp]
        L.fdc_set_secondaries.restype = i32
        L.fdc_set_secondaries.argtypes = [vp, vp, vp, vp, u32]
        L.fdc_gamma_index.restype = i32
        L.fdc_gamma_index.argtypes = [vp, vp, vp, f32, f32, f32, f32, vp, ctypes.POINTER(ctypes.c_double), ctypes.POINTER(u64)]
        L.fdc_uncertainty_history.restype = i32
        L.fdc_uncertainty_history.argtypes = [vp, u64, vp, i32, ctypes.POINTER(ctypes.c_double), ctypes.POINTER(u64)]
        L.fdc_uncertainty_batch.restype = i32
        L.fdc_uncertainty_batch.argtypes = [vp, vp, i32, u64, vp, i32, ctypes.POINTER(ctypes.c_double), ctypes.POINTER(u64)]
        L.fdc_uncertainty_batch_noalloc.restype = i32
        L.fdc_uncertainty_batch_noalloc.argtypes = [vp, vp, i32, u64, vp, ctypes.POINTER(ctypes.c_double), ctypes.POINTER(u64)]
        _lib = L
    return _lib


def _ptr(x):
    """Pointer of a numpy array (host) or torch tensor (host or device); None -> NULL."""
    if x is None:
        return None
    if isinstance(x, np.ndarray):
        assert x.flags["C_CONTIGUOUS"]
        return ctypes.c_void_p(x.ctypes.data)
    assert x.is_contiguous()
    return ctypes.c_void_p(x.data_ptr())


def _is_device(x):
    return (not isinstance(x, np.ndarray)) and x.is_cuda


class _DeviceArray:
    """A borrowed device array as a __cuda_array_interface__ object (so torch can alias it without a copy)."""

    def __init__(self, ptr, shape, typestr, owner):
        self.__cuda_array_interface__ = {"shape": tuple(shape), "typestr": typestr, "data": (int(ptr), False), "version": 3, "strides": None}
        self._owner = owner


class Fdc:
    """One fdc_ctx.  Methods mirror the C-ABI one to one."""

    def __init__(self, hu, spacing, table, device: int = 0, stream=None):
        """fdc_create.  hu: int16 [nz,ny,nx] numpy array (copied) or CUDA torch tensor (read during the call)."""
        import torch
        self._lib = lib()
        self._h = ctypes.c_void_p(None)
        self._keep = []
        nz, ny, nx = hu.shape
        self.shape = (nz, ny, nx)
        self.device = device
        self._torch = torch
        if stream is None:
            stream = torch.cuda.current_stream(device)
        self.stream = stream
        table = np.ascontiguousarray(table, dtype=KNOT_DTYPE)
        if _is_device(hu):
            self._keep.append(hu)
        h = ctypes.c_void_p(None)
        rc = self._lib.fdc_create(ctypes.byref(h), device, ctypes.c_void_p(stream.cuda_stream), _ptr(hu), nx, ny, nz,
                                  float(spacing[0]), float(spacing[1]), float(spacing[2]), _ptr(table), len(table),
                                  1 if _is_device(hu) else 0)
        if rc != 0:
            raise FdcError(rc, self._lib.fdc_strerror(rc).decode())
        self._h = h

    def _check(self, rc):
        if rc > 0:
            import warnings
            warnings.warn(FdcWarning("fdc warning %d: %s: %s" % (rc, self._lib.fdc_strerror(rc).decode(), self._lib.fdc_last_error(self._h).decode())), stacklevel=3)
            return
        if rc != 0:
            raise FdcError(rc, "%s: %s" % (self._lib.fdc_strerror(rc).decode(), self._lib.fdc_last_error(self._h).decode()))

    def fdc_load_tracks(self, dx, dy, dz, dE, E, track_off, bin_first, e_min, e_bin):
        """Step arrays: all numpy (host) or all CUDA torch tensors; offsets: numpy."""
        dev = _is_device(dx)
        assert all(_is_device(a) == dev for a in (dy, dz, dE, E))
        track_off = np.ascontiguousarray(track_off, dtype=np.uint64)
        bin_first = np.ascontiguousarray(bin_first, dtype=np.uint32)
        n = int(dx.shape[0])
        db = _TrackDB(_ptr(dx).value, _ptr(dy).value, _ptr(dz).value, _ptr(dE).value, _ptr(E).value, n,
                      track_off.ctypes.data, len(track_off) - 1, bin_first.ctypes.data, len(bin_first) - 1,
                      float(e_min), float(e_bin))
        self._check(self._lib.fdc_load_tracks(self._h, ctypes.byref(db), 1 if dev else 0))

    def fdc_set_secondaries(self, sec_first, sec_track, sec_step):
        """R15 secondary table (numpy uint32 arrays); empty sec_track removes it."""
        sf = np.ascontiguousarray(sec_first, dtype=np.uint32); stt = np.ascontiguousarray(sec_track, dtype=np.uint32)
        sst = np.ascontiguousarray(sec_step, dtype=np.uint32)
        assert len(stt) == len(sst)
        self._check(self._lib.fdc_set_secondaries(self._h, _ptr(sf), _ptr(stt) if len(stt) else None, _ptr(sst) if len(sst) else None, len(stt)))

    def fdc_run(self, beamlets, first_proton, n_protons, proton_stride, seed, flags=FDC_RANDOM_AZIMUTH, dose_gy=None):
        """dose_gy: None, a CUDA float32 tensor [nz,ny,nx], or a host numpy/pinned-torch float32 array."""
        bl = np.ascontiguousarray(beamlets, dtype=BEAMLET_DTYPE)
        flags = int(flags) & ~FDC_DOSE_TO_HOST
        if dose_gy is not None and not _is_device(dose_gy):
            flags |= FDC_DOSE_TO_HOST
        self._check(self._lib.fdc_run(self._h, _ptr(bl), len(bl), int(first_proton), int(n_protons), int(proton_stride),
                                      int(seed), flags, _ptr(dose_gy)))

    def fdc_run_phase_space(self, particles, first_id, seed, flags=FDC_RANDOM_AZIMUTH, dose_gy=None):
        """particles: numpy array of PARTICLE_DTYPE (host, copied) or a CUDA uint8/float32 tensor holding
        n x 32 bytes in that layout (borrowed for the call)."""
        if isinstance(particles, np.ndarray):
            ps = np.ascontiguousarray(particles, dtype=PARTICLE_DTYPE); n = len(ps); dev = 0
        else:
            ps = particles; n = particles.numel() * particles.element_size() // PARTICLE_DTYPE.itemsize; dev = 1
            assert particles.is_cuda and particles.is_contiguous()
        flags = int(flags) & ~FDC_DOSE_TO_HOST
        if dose_gy is not None and not _is_device(dose_gy):
            flags |= FDC_DOSE_TO_HOST
        self._check(self._lib.fdc_run_phase_space(self._h, _ptr(ps), n, dev, int(first_id), int(seed), flags, _ptr(dose_gy)))

    def fdc_to_gy(self, dose_gy):
        """Stage 5 alone: the grid as it stands -> Gy into a CUDA float32 tensor or a host float32 array."""
        self._check(self._lib.fdc_to_gy(self._h, _ptr(dose_gy), 1 if _is_device(dose_gy) else 0))

    def fdc_edep_device_ptr(self):
        """The context's own grids as torch int64 CUDA tensors aliasing the library's memory (borrowed: valid until
        fdc_destroy): (energy grid, squares grid or None).  For the in-place all-reduce over GPUs."""
        e = ctypes.c_void_p(None); q = ctypes.c_void_p(None)
        self._check(self._lib.fdc_edep_device_ptr(self._h, ctypes.byref(e), ctypes.byref(q)))
        torch = self._torch
        mk = lambda p: torch.as_tensor(_DeviceArray(p, self.shape, "<i8", self), device=torch.device("cuda", self.device))
        return mk(e.value), (mk(q.value) if q.value else None)

    def fdc_profile(self, values, axis, fixed_a, fixed_b, half_width_a=2, half_width_b=2, out=None):
        """values: CUDA float32 tensor [nz,ny,nx] or None (the energy grid, MeV).  Returns the profile (host float64
        numpy array of n_axis entries, or `out`, a CUDA float64 tensor, filled)."""
        n_axis = self.shape[2 - axis]
        if out is None:
            out = np.empty(n_axis, dtype=np.float64)
        assert values is None or _is_device(values)
        self._check(self._lib.fdc_profile(self._h, _ptr(values), int(axis), int(fixed_a), int(fixed_b), int(half_width_a), int(half_width_b),
                                          _ptr(out), 1 if _is_device(out) else 0))
        return out

    def fdc_rms_diff(self, dose_ref, dose_eval):
        """CUDA float32 tensors [nz,ny,nx].  Returns (rms of (eval - ref) / max(ref) over all voxels, max(ref))."""
        assert _is_device(dose_ref) and _is_device(dose_eval)
        r = ctypes.c_double(0.0); m = ctypes.c_double(0.0)
        self._check(self._lib.fdc_rms_diff(self._h, _ptr(dose_ref), _ptr(dose_eval), ctypes.byref(r), ctypes.byref(m)))
        return r.value, m.value

    def fdc_get_edep_fixed(self, out=None):
        """Raw grid; out: CUDA int64 tensor, or None -> new host numpy uint64 [nz,ny,nx]."""
        if out is None:
            out = np.empty(self.shape, dtype=np.uint64)
        self._check(self._lib.fdc_get_edep_fixed(self._h, _ptr(out), 1 if _is_device(out) else 0))
        return out

    def fdc_set_edep_fixed(self, grid):
        """Overwrite the raw grid from a CUDA int64 tensor or a host numpy uint64 array."""
        self._check(self._lib.fdc_set_edep_fixed(self._h, _ptr(grid), 1 if _is_device(grid) else 0))

    def fdc_get_sq_fixed(self, out=None):
        """Sum-of-squares grid (FDC_TALLY_SQUARES); out as in fdc_get_edep_fixed."""
        if out is None:
            out = np.empty(self.shape, dtype=np.uint64)
        self._check(self._lib.fdc_get_sq_fixed(self._h, _ptr(out), 1 if _is_device(out) else 0))
        return out

    def fdc_set_sq_fixed(self, grid):
        self._check(self._lib.fdc_set_sq_fixed(self._h, _ptr(grid), 1 if _is_device(grid) else 0))

    def fdc_uncertainty_history(self, n_histories, rel_sigma=None):
        """Eq. (2).  rel_sigma: None, a CUDA float32 tensor or a host float32 array [nz,ny,nx] (filled).
        Returns (mean relative uncertainty over voxels above half the maximum dose, their number)."""
        m = ctypes.c_double(0.0); c = ctypes.c_uint64(0)
        self._check(self._lib.fdc_uncertainty_history(self._h, int(n_histories), _ptr(rel_sigma),
                                                      1 if (rel_sigma is not None and _is_device(rel_sigma)) else 0,
                                                      ctypes.byref(m), ctypes.byref(c)))
        return m.value, int(c.value)

    def fdc_uncertainty_batch(self, batch_grids, histories_per_batch, rel_sigma=None):
        """Eq. (1).  batch_grids: list of CUDA int64 tensors [nz,ny,nx] (one energy grid per batch)."""
        assert all(_is_device(g) and g.is_contiguous() for g in batch_grids)
        ptrs = (ctypes.c_void_p * len(batch_grids))(*[g.data_ptr() for g in batch_grids])
        m = ctypes.c_double(0.0); c = ctypes.c_uint64(0)
        self._check(self._lib.fdc_uncertainty_batch(self._h, ctypes.cast(ptrs, ctypes.c_void_p), len(batch_grids), int(histories_per_batch),
                                                    _ptr(rel_sigma), 1 if (rel_sigma is not None and _is_device(rel_sigma)) else 0,
                                                    ctypes.byref(m), ctypes.byref(c)))
        return m.value, int(c.value)

    def fdc_uncertainty_batch_noalloc(self, batch_grids, histories_per_batch, rel_sigma=None):
        """Eq. (1) for callers that must not cause a device allocation while they run (all device memory handed to
        their own arena, or no room for the device-wide wait a cudaMalloc / cudaFree can bring): same results as
        fdc_uncertainty_batch, scratch in a fixed 512-byte array inside the library, at most FDC_NOALLOC_MAX_BATCHES
        grids.  rel_sigma: None or a CUDA float32 tensor [nz,ny,nx] the caller owns.  One scratch array per device:
        calls that overlap on the GPU race.  Make the first call on a device during set-up (include/fdc.h)."""
        assert all(_is_device(g) and g.is_contiguous() for g in batch_grids)
        assert rel_sigma is None or (_is_device(rel_sigma) and rel_sigma.is_contiguous())
        ptrs = (ctypes.c_void_p * len(batch_grids))(*[g.data_ptr() for g in batch_grids])
        m = ctypes.c_double(0.0); c = ctypes.c_uint64(0)
        self._check(self._lib.fdc_uncertainty_batch_noalloc(self._h, ctypes.cast(ptrs, ctypes.c_void_p), len(batch_grids),
                                                            int(histories_per_batch), _ptr(rel_sigma), ctypes.byref(m), ctypes.byref(c)))
        return m.value, int(c.value)

    def fdc_gamma_index(self, dose_ref, dose_eval, dose_tol_frac=0.03, dist_tol_mm=3.0, search_mm=None, cutoff_frac=0.0, gamma_out=None):
        """dose_ref, dose_eval, gamma_out: CUDA float32 tensors [nz,ny,nx].  Returns (pass fraction, voxels evaluated)."""
        assert _is_device(dose_ref) and _is_device(dose_eval) and (gamma_out is None or _is_device(gamma_out))
        pf = ctypes.c_double(0.0); c = ctypes.c_uint64(0)
        self._check(self._lib.fdc_gamma_index(self._h, _ptr(dose_ref), _ptr(dose_eval), float(dose_tol_frac), float(dist_tol_mm),
                                              float(dist_tol_mm if search_mm is None else search_mm), float(cutoff_frac),
                                              _ptr(gamma_out), ctypes.byref(pf), ctypes.byref(c)))
        return pf.value, int(c.value)

    def fdc_get_stats(self) -> dict:
        s = _Stats()
        self._check(self._lib.fdc_get_stats(self._h, ctypes.byref(s)))
        return {n: int(getattr(s, n)) for n, _ in s._fields_}

    def fdc_reset(self):
        self._check(self._lib.fdc_reset(self._h))

    def fdc_last_call_info(self) -> dict:
        """Diagnostics: device times, launches and host<->device bytes of the most recent run / fdc_to_gy."""
        ci = _CallInfo()
        self._check(self._lib.fdc_last_call_info(self._h, ctypes.byref(ci)))
        return {"total_ms": ci.ms_total, "transport_ms": ci.ms_transport, "sort_ms": ci.ms_sort, "gy_ms": ci.ms_gy, "launches": int(ci.launches),
                "h2d_bytes": int(ci.h2d_bytes), "d2h_bytes": int(ci.d2h_bytes), "reds_sent": int(ci.reds_sent), "reds_traced": int(ci.reds_traced),
                "sq_history_flushes": int(ci.sq_history_flushes)}

    def fdc_trace_reds(self, trace=None):
        """Diagnostics: a CUDA int32/uint32 tensor that FDC_DIAG_REDS runs fill with voxel indices (None removes it)."""
        if trace is None:
            self._trace = None
            self._check(self._lib.fdc_trace_reds(self._h, None, 0))
        else:
            assert trace.is_cuda and trace.is_contiguous() and trace.element_size() == 4
            self._trace = trace
            self._check(self._lib.fdc_trace_reds(self._h, _ptr(trace), trace.numel()))

    def fdc_destroy(self):
        if self._h:
            self._lib.fdc_destroy(self._h)
            self._h = ctypes.c_void_p(None)
            self._keep = []

    def __del__(self):
        try:
            self.fdc_destroy()
        except Exception:
            pass
