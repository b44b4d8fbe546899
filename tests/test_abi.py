"""Host-side checks that need no GPU: the C-ABI library builds, loads and exports every symbol
include/fdc.h declares; the binding's struct layouts match the header's."""
import ctypes
import os
import re

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared():
    text = open(os.path.join(ROOT, "include", "fdc.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(fdc_[a-z0-9_]+)\s*\(", text)))


def test_library_builds_loads_and_exports_every_declared_symbol():
    from paper_1011_2188_b200 import build
    path = build.build()
    L = ctypes.CDLL(path)
    names = _declared()
    assert {"fdc_create", "fdc_load_tracks", "fdc_run", "fdc_get_edep_fixed", "fdc_get_stats", "fdc_reset",
            "fdc_destroy", "fdc_strerror", "fdc_last_error"} <= set(names)
    for n in names:
        assert hasattr(L, n), n
    import paper_1011_2188_b200 as fdc
    assert sorted(fdc.EXPORTS) == names
    fdc.lib()                                   # argtypes wiring
    assert fdc.lib().fdc_strerror(0) == b"ok" and b"sm_100" in fdc.lib().fdc_strerror(fdc.FDC_EARCH)


def test_struct_layouts_match_header():
    import paper_1011_2188_b200 as fdc
    import fdc_inputs as fi
    assert fdc.BEAMLET_DTYPE.itemsize == 72 and fdc.BEAMLET_DTYPE.fields["n_protons"][1] == 64
    assert fdc.KNOT_DTYPE.itemsize == 16
    assert fi.BEAMLET_DTYPE == fdc.BEAMLET_DTYPE and fi.KNOT_DTYPE == fdc.KNOT_DTYPE
    assert ctypes.sizeof(fdc._TrackDB) == 88 and ctypes.sizeof(fdc._Stats) == 72
    assert ctypes.sizeof(fdc._CallInfo) == 56 and fdc._CallInfo.h2d_bytes.offset == 24      # fdc_call_info


def test_peaks_library_is_separate_and_exports_its_symbols():
    """The roofline microbenchmarks are measurement tooling: their own library, nothing of them in libfdc.so."""
    from paper_1011_2188_b200 import build, peaks
    L = ctypes.CDLL(build.build())
    P = ctypes.CDLL(build.PEAKS_LIB)
    for n in peaks.EXPORTS:
        assert hasattr(P, n) and not hasattr(L, n), n
    assert not hasattr(L, "fdc_peak_red_u64")
    peaks.lib()


def test_build_line_carries_the_arithmetic_contract():
    from paper_1011_2188_b200 import build
    assert "-fmad=false" in build.NVCC_FLAGS and "arch=compute_100a,code=sm_100a" in build.NVCC_FLAGS
    assert not any("fast_math" in f for f in build.NVCC_FLAGS)


def test_sass_of_the_transport_kernel():
    """cuobjdump of the built library: the code is sm_100a, the deposit is a 64-bit RED (R8), and the
    kernel holds separate FMUL / FADD beside the FFMAs the source asks for by name (-fmad=false: no contraction)."""
    import shutil
    import subprocess
    from paper_1011_2188_b200 import build
    cu = shutil.which("cuobjdump") or "/usr/local/cuda/bin/cuobjdump"
    if not os.path.exists(cu):
        import pytest
        pytest.skip("cuobjdump not installed")
    out = subprocess.run([cu, "-sass", "-fun", "k_transport", build.build()], capture_output=True, text=True, timeout=300).stdout
    if "k_transport" not in out:                                   # older cuobjdump: -fun wants the mangled name
        out = subprocess.run([cu, "-sass", build.build()], capture_output=True, text=True, timeout=600).stdout
    assert "sm_100a" in out or "SM100" in out.upper() or "sm_100" in out
    assert re.search(r"RED(G)?\.E\.ADD\.64", out), "no 64-bit reduction in the SASS"
    assert "FMUL" in out and "FADD" in out and "FFMA" in out


def test_product_does_not_touch_the_oracle():
    for dirpath, _, files in os.walk(os.path.join(ROOT, "paper_1011_2188_b200")):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h", ".cpp")):
                src = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in src and "from oracle" not in src
                assert not re.search(r'#include\s*[<"][^>"]*oracle', src)
                assert "liboracle" not in src and "fdc_inputs" not in src
