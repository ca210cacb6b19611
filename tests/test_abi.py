"""The C-ABI library builds, loads and exports every symbol include/muca.h declares (no GPU, no compute calls)."""
import ctypes
import os
import re

import pytest

import paper_1707_00919_b200 as mb
from paper_1707_00919_b200 import binding as B

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_symbols():
    text = open(os.path.join(ROOT, "include", "muca.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(muca_[a-z_0-9]+)\s*\(", text)))


def test_header_and_binding_list_agree():
    assert declared_symbols() == sorted(B.EXPORTS)


def test_library_exports_every_declared_symbol():
    lib = ctypes.CDLL(mb.lib_path()) if os.path.exists(mb.lib_path()) else mb.lib()
    for name in declared_symbols():
        assert hasattr(lib, name), f"{name} is declared in include/muca.h but not exported"


def test_host_only_entry_points():
    lib = mb.lib()
    assert b"sm_100a" in lib.muca_version()
    # workspace: packed spins + energies + threshold table + histogram, 256-byte aligned pieces
    for L, W in ((8, 128), (32, 16384), (128, 8192)):
        n = mb.workspace_bytes(L, W)
        assert n >= W * L * L // 8 + 4 * W + (L * L + 1) * 40 and n % 256 == 0
    assert mb.workspace_bytes(12, 32) == 0 and mb.workspace_bytes(32, 0) == 0
    w, p = ctypes.c_int(), ctypes.c_int()
    assert lib.muca_suggest_walkers(12, ctypes.byref(w), ctypes.byref(p)) == -1
    assert lib.muca_suggest_walkers(32, None, ctypes.byref(p)) == -1
    import torch
    if not torch.cuda.is_available():                            # no device: MUCA_ECUDA, never a made-up number
        assert lib.muca_suggest_walkers(32, ctypes.byref(w), ctypes.byref(p)) == -2
    # bad arguments are rejected before any CUDA call
    h = ctypes.c_void_p()
    assert lib.muca_create(ctypes.byref(h), 7, 32, 1) == -1 and not h
    assert lib.muca_create_in(ctypes.byref(h), 32, 0, 1, 0, None, 0, None) == -1 and not h


def test_no_cpu_fallback():
    import torch
    if torch.cuda.is_available():
        pytest.skip("CUDA present")
    with pytest.raises(mb.MucaError):
        mb.Muca(8, 32, 1)


def test_product_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_1707_00919_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert "muca_oracle" not in src and "oracle/" not in src.replace("shares nothing with oracle/", "").replace(
                    "Shares nothing with oracle/", "").replace("imported by neither oracle/", ""), f


def test_onsager_stand_in_is_close_to_the_exact_density_of_states():
    # workloads.onsager_log_dos (bench.py's weights for spread walkers at L = 128, where the tree has no exact g(E)):
    # against the exact finite-lattice g(E) of tests/golden/ it must be flat-histogram quality, i.e. off by a few units
    # of ln g over hundreds of units of range, symmetric in E, and largest in the middle
    import math
    import numpy as np
    from paper_1707_00919_b200.workloads import onsager_log_dos
    for L in (16, 32):
        with open(os.path.join(ROOT, "tests", "golden", f"ising_dos_L{L}.txt")) as f:
            g = [int(x) for x in f if not x.startswith("#")]
        approx = onsager_log_dos(L)
        exact = np.array([math.log(v) if v > 0 else np.nan for v in g])
        d = exact - approx
        assert approx.shape == (L * L + 1,) and np.all(np.isfinite(approx))
        assert np.nanmax(np.abs(d)) < 4.5, (L, np.nanmin(d), np.nanmax(d))
        assert np.allclose(approx, approx[::-1]) and np.argmax(approx) == L * L // 2
        assert abs(approx[L * L // 2] - L * L * math.log(2.0)) < 1e-3 and abs(approx[0]) < 1e-3
