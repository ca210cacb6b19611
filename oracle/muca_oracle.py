"""ctypes wrapper of the CPU oracle (oracle/muca_oracle.cpp).

TEST INFRASTRUCTURE — NOT PRODUCT CODE.  Only tests/, __graft_entry__.smoke()
and bench.py's cpu_baseline / --impl reference legs may import this module.
It imports nothing from paper_1707_00919_b200 and nothing there imports it.

Argument marshalling only; all arithmetic lives in muca_oracle.cpp, where each
function cites the PAPER.md passage (or DESIGN.md reading R<n>) it follows.
"""
import ctypes as C
import os
import sys

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
if _HERE not in sys.path:
    sys.path.insert(0, _HERE)
import build as _build  # noqa: E402  (oracle/build.py)

_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(_build.build())
        u32p = C.POINTER(C.c_uint32)
        u64p = C.POINTER(C.c_uint64)
        f64p = C.POINTER(C.c_double)
        i8p = C.POINTER(C.c_int8)
        i32p = C.POINTER(C.c_int32)
        L.oracle_philox4x32_10.argtypes = [u32p, u32p, u32p]
        L.oracle_philox4x32_10.restype = None
        L.oracle_energy.argtypes = [C.c_int, i8p]
        L.oracle_energy.restype = C.c_int
        L.oracle_thresholds.argtypes = [C.c_int, f64p, u32p]
        L.oracle_weight_update.argtypes = [C.c_int, f64p, u64p]
        L.oracle_create.argtypes = [C.c_int, C.c_int, C.c_uint64, C.c_uint32]
        L.oracle_create.restype = C.c_void_p
        L.oracle_destroy.argtypes = [C.c_void_p]
        L.oracle_destroy.restype = None
        L.oracle_set_log_weights.argtypes = [C.c_void_p, f64p, C.c_int]
        L.oracle_get_log_weights.argtypes = [C.c_void_p, f64p, C.c_int]
        L.oracle_run_iteration.argtypes = [C.c_void_p, C.c_int, C.c_int, u64p, C.c_int, C.c_int]
        L.oracle_run_iteration_random_site.argtypes = [C.c_void_p, C.c_uint64, C.c_uint64, u64p, C.c_int, C.c_int]
        L.oracle_run_iteration_random_site_expf.argtypes = [C.c_void_p, C.c_uint64, C.c_uint64, u64p, C.c_int, C.c_int]
        L.oracle_exp32.argtypes = [C.c_float]
        L.oracle_exp32.restype = C.c_float
        L.oracle_uniform32.argtypes = [C.c_uint32]
        L.oracle_uniform32.restype = C.c_float
        L.oracle_update_weights.argtypes = [C.c_void_p]
        L.oracle_update_weights_with.argtypes = [C.c_void_p, u64p, C.c_int]
        L.oracle_get_energies.argtypes = [C.c_void_p, i32p, C.c_int]
        L.oracle_get_spins.argtypes = [C.c_void_p, i8p, C.c_uint64]
        L.oracle_set_spins.argtypes = [C.c_void_p, i8p, C.c_uint64]
        L.oracle_get_iteration.argtypes = [C.c_void_p]
        L.oracle_get_iteration.restype = C.c_uint32
        L.oracle_set_iteration.argtypes = [C.c_void_p, C.c_uint32]
        L.oracle_max_threads.restype = C.c_int
        _lib = L
    return _lib


def _p(a, t):
    return a.ctypes.data_as(C.POINTER(t))


def max_threads() -> int:
    return int(lib().oracle_max_threads())


def philox4x32_10(ctr, key) -> np.ndarray:
    c = np.ascontiguousarray(ctr, dtype=np.uint32)
    k = np.ascontiguousarray(key, dtype=np.uint32)
    assert c.shape == (4,) and k.shape == (2,)
    out = np.empty(4, dtype=np.uint32)
    lib().oracle_philox4x32_10(_p(c, C.c_uint32), _p(k, C.c_uint32), _p(out, C.c_uint32))
    return out


def energy(spins_2d) -> int:
    s = np.ascontiguousarray(spins_2d, dtype=np.int8)
    assert s.ndim == 2 and s.shape[0] == s.shape[1]
    return int(lib().oracle_energy(s.shape[0], _p(s, C.c_int8)))


def thresholds(logw) -> np.ndarray:
    """uint32 [n_bins, 5]: acceptance threshold for slot j and a = 0..4 antiparallel neighbours."""
    w = np.ascontiguousarray(logw, dtype=np.float64)
    out = np.empty((w.size, 5), dtype=np.uint32)
    rc = lib().oracle_thresholds(w.size, _p(w, C.c_double), _p(out, C.c_uint32))
    assert rc == 0
    return out


def weight_update(logw, H) -> np.ndarray:
    w = np.array(logw, dtype=np.float64, copy=True)
    h = np.ascontiguousarray(H, dtype=np.uint64)
    assert w.size == h.size
    lib().oracle_weight_update(w.size, _p(w, C.c_double), _p(h, C.c_uint64))
    return w


class Oracle:
    """One oracle instance: W walkers on L x L lattices (global ids walker_offset .. +W-1)."""

    def __init__(self, L: int, n_walkers: int, seed: int, walker_offset: int = 0):
        self._h = lib().oracle_create(L, n_walkers, C.c_uint64(seed & (2**64 - 1)), walker_offset)
        if not self._h:
            raise ValueError("oracle_create rejected (L even >= 4, n_walkers > 0 required)")
        self.L, self.N, self.W = L, L * L, n_walkers
        self.n_bins = self.N + 1

    def close(self):
        if self._h:
            lib().oracle_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def set_log_weights(self, logw):
        w = np.ascontiguousarray(logw, dtype=np.float64)
        if lib().oracle_set_log_weights(self._h, _p(w, C.c_double), w.size) != 0:
            raise ValueError("n_bins mismatch")

    def get_log_weights(self) -> np.ndarray:
        out = np.empty(self.n_bins, dtype=np.float64)
        assert lib().oracle_get_log_weights(self._h, _p(out, C.c_double), out.size) == 0
        return out

    def run_iteration(self, therm_sweeps: int, sweeps: int, n_threads: int = 1) -> np.ndarray:
        H = np.zeros(self.n_bins, dtype=np.uint64)
        rc = lib().oracle_run_iteration(self._h, therm_sweeps, sweeps, _p(H, C.c_uint64), H.size,
                                        n_threads)
        if rc != 0:
            raise ValueError(f"oracle_run_iteration failed rc={rc}")
        return H

    def run_iteration_random_site(self, therm_updates: int, updates: int, n_threads: int = 1) -> np.ndarray:
        """The paper's own scheme (R22): same random site for all walkers, per-walker acceptance stream; counts in updates."""
        H = np.zeros(self.n_bins, dtype=np.uint64)
        rc = lib().oracle_run_iteration_random_site(self._h, C.c_uint64(therm_updates), C.c_uint64(updates),
                                                    _p(H, C.c_uint64), H.size, n_threads)
        if rc != 0:
            raise ValueError(f"oracle_run_iteration_random_site failed rc={rc}")
        return H

    def run_iteration_random_site_expf(self, therm_updates: int, updates: int, n_threads: int = 1) -> np.ndarray:
        """The same with the paper's single-precision acceptance U < exp32(omega_f[j'] - omega_f[j]) (R23)."""
        H = np.zeros(self.n_bins, dtype=np.uint64)
        rc = lib().oracle_run_iteration_random_site_expf(self._h, C.c_uint64(therm_updates), C.c_uint64(updates),
                                                         _p(H, C.c_uint64), H.size, n_threads)
        if rc != 0:
            raise ValueError(f"oracle_run_iteration_random_site_expf failed rc={rc}")
        return H

    def update_weights(self):
        assert lib().oracle_update_weights(self._h) == 0

    def update_weights_with(self, H):
        h = np.ascontiguousarray(H, dtype=np.uint64)
        assert lib().oracle_update_weights_with(self._h, _p(h, C.c_uint64), h.size) == 0

    def get_energies(self) -> np.ndarray:
        out = np.empty(self.W, dtype=np.int32)
        assert lib().oracle_get_energies(self._h, _p(out, C.c_int32), out.size) == 0
        return out

    def get_spins(self) -> np.ndarray:
        out = np.empty((self.W, self.L, self.L), dtype=np.int8)
        assert lib().oracle_get_spins(self._h, _p(out, C.c_int8), out.size) == 0
        return out

    def set_spins(self, spins):
        s = np.ascontiguousarray(spins, dtype=np.int8)
        assert s.size == self.W * self.N
        assert lib().oracle_set_spins(self._h, _p(s, C.c_int8), s.size) == 0

    @property
    def iteration(self) -> int:
        return int(lib().oracle_get_iteration(self._h))

    @iteration.setter
    def iteration(self, n: int):
        lib().oracle_set_iteration(self._h, n)
