"""ctypes binding of libfdcpeaks.so (csrc/bench_peaks.cu): the roofline microbenchmarks bench.py needs for its
denominators.  Measurement tooling -- not part of the method, not linked into libfdc.so."""
from __future__ import annotations

import ctypes
import os

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libfdcpeaks.so")
EXPORTS = ["fdcpeaks_red_u64", "fdcpeaks_red_replay"]
_lib = None


def lib():
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError("%s not found: build it with `python -m paper_1011_2188_b200.build`" % LIB_PATH)
        L = ctypes.CDLL(LIB_PATH)
        i32, u32, u64, vp = ctypes.c_int, ctypes.c_uint32, ctypes.c_uint64, ctypes.c_void_p
        L.fdcpeaks_red_u64.restype = i32
        L.fdcpeaks_red_u64.argtypes = [i32, u64, u64, i32, ctypes.POINTER(ctypes.c_double)]
        L.fdcpeaks_red_replay.restype = i32
        L.fdcpeaks_red_replay.argtypes = [i32, vp, u64, u64, u32, i32, ctypes.POINTER(ctypes.c_double)]
        _lib = L
    return _lib


def red_u64(device: int, footprint_bytes: int, n_ops: int, mode: int = 0) -> float:
    """u64 reductions per second: mode 0 uniform over the footprint, 1 lanes of a warp on 4 words, 2 on one word."""
    out = ctypes.c_double(0.0)
    rc = lib().fdcpeaks_red_u64(device, footprint_bytes, n_ops, mode, ctypes.byref(out))
    if rc != 0:
        raise RuntimeError("fdcpeaks_red_u64 failed: %d" % rc)
    return out.value


def red_replay(device: int, trace, n_addr: int, n_words: int, passes: int, shuffled: bool) -> float:
    """Replays the first n_addr entries of a traced voxel-index list (CUDA int32 tensor) `passes` times."""
    assert trace.is_cuda and trace.is_contiguous() and trace.element_size() == 4 and n_addr <= trace.numel()
    out = ctypes.c_double(0.0)
    rc = lib().fdcpeaks_red_replay(device, ctypes.c_void_p(trace.data_ptr()), n_addr, n_words, passes, 1 if shuffled else 0, ctypes.byref(out))
    if rc != 0:
        raise RuntimeError("fdcpeaks_red_replay failed: %d" % rc)
    return out.value
