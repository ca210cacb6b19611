import ctypes
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
for p in (ROOT, os.path.join(ROOT, "oracle"), os.path.dirname(os.path.abspath(__file__))):
    if p not in sys.path:
        sys.path.insert(0, p)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")
    config.addinivalue_line("markers", "slow: long-running statistical check")


def _has_gpu():
    try:
        import torch
        return torch.cuda.is_available()
    except Exception:
        return False


def pytest_collection_modifyitems(config, items):
    if _has_gpu():
        return
    skip = pytest.mark.skip(reason="no CUDA device")
    for it in items:
        if "gpu" in it.keywords:
            it.add_marker(skip)


@pytest.fixture(scope="session")
def curand_pin(tmp_path_factory):
    """The toolkit's own Philox4x32-10 routines, built for the host (tests/pins/curand_philox_shim.cpp)."""
    cuda = os.environ.get("CUDA_HOME", "/usr/local/cuda")
    src = os.path.join(ROOT, "tests", "pins", "curand_philox_shim.cpp")
    out = str(tmp_path_factory.mktemp("pins") / "libcurand_pin.so")
    subprocess.check_call(["g++", "-O1", "-shared", "-fPIC", f"-I{cuda}/include", src,
                           f"-L{cuda}/lib64", "-lcurand", f"-Wl,-rpath,{cuda}/lib64", "-o", out])
    lib = ctypes.CDLL(out)
    u32p = ctypes.POINTER(ctypes.c_uint32)
    lib.pin_curand_philox4x32_10.argtypes = [u32p, u32p, u32p]
    lib.pin_curand_philox4x32_10.restype = None
    lib.pin_curand_host_generate.argtypes = [ctypes.c_ulonglong, ctypes.c_ulonglong, u32p, ctypes.c_size_t]
    lib.pin_curand_host_generate_uniform.argtypes = [ctypes.c_ulonglong, ctypes.c_ulonglong, ctypes.POINTER(ctypes.c_float), ctypes.c_size_t]
    return lib
