"""pytest configuration: the `gpu` marker and shared small workloads."""
import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")


@pytest.fixture(scope="session")
def wl1_small():
    """config 1 geometry, reduced: 200 tracks, 2000 protons."""
    import fdc_inputs as fi
    return fi.workload(1, n_protons=2000, tracks_per_bin=200)


@pytest.fixture(scope="session")
def wl2_small():
    """config 2 (slabs), reduced: 300 tracks per bin, 3000 protons."""
    import fdc_inputs as fi
    return fi.workload(2, n_protons=3000, tracks_per_bin=300)


@pytest.fixture(scope="session")
def wl3_small():
    """config 3 (thorax, 1176 beamlets), reduced: 50 tracks per bin, 4704 protons (4 per beamlet)."""
    import fdc_inputs as fi
    return fi.workload(3, n_protons=4704, tracks_per_bin=50)
