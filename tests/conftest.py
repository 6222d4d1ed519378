import ctypes
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")


@pytest.fixture(scope="session")
def curand_pin(tmp_path_factory):
    """cuRAND's curand_Philox4x32_10 compiled for the host (tests/curand_pin.cpp)."""
    src = os.path.join(ROOT, "tests", "curand_pin.cpp")
    so = str(tmp_path_factory.mktemp("pin") / "curand_pin.so")
    cuda_inc = os.path.join(os.environ.get("CUDA_HOME", "/usr/local/cuda"), "include")
    subprocess.check_call(["g++", "-O2", "-shared", "-fPIC", "-I" + cuda_inc, "-o", so, src])
    lib = ctypes.CDLL(so)
    lib.curand_philox_host.argtypes = [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_long]
    lib.curand_philox_host.restype = None
    return lib
