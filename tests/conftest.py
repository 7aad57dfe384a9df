import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")


@pytest.fixture(scope="session")
def curand_shim():
    """NVIDIA's own curand_Philox4x32_10 (header host path) as a ctypes library."""
    import ctypes
    here = os.path.dirname(os.path.abspath(__file__))
    src = os.path.join(here, "curand_philox_shim.cpp")
    out = os.path.join(here, "libcurand_philox_shim.so")
    inc = "/usr/local/cuda/include"
    if not os.path.exists(os.path.join(inc, "curand_philox4x32_x.h")):
        pytest.skip("cuRAND header not on this machine")
    if not os.path.exists(out) or os.path.getmtime(out) < os.path.getmtime(src):
        subprocess.run(["g++", "-O2", "-shared", "-fPIC", "-I" + inc, src, "-o", out], check=True)
    return ctypes.CDLL(out)
