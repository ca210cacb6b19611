"""ctypes binding of libmuca_b200.so -- same names as include/muca.h, argument marshalling only.

PyTorch supplies the device workspace (a uint8 CUDA tensor) and the CUDA stream; every step of the
path runs inside the library's kernels.  There is no CPU fallback: constructing a `Muca` without a
CUDA device, or without the compiled library, raises `MucaError`.
"""
import ctypes as C
import os

import numpy as np

from . import build as _build

MUCA_OK = 0
MUCA_KERNEL_AUTO, MUCA_KERNEL_RESIDENT, MUCA_KERNEL_STREAMED, MUCA_KERNEL_STREAMED_PAIRS = 0, 1, 2, 3
MUCA_OPT_KERNEL, MUCA_OPT_THREADS_PER_BLOCK, MUCA_OPT_MAX_SWEEPS_PER_LAUNCH, MUCA_OPT_WALKERS_PER_WARP = 1, 2, 3, 4
MUCA_OPT_UPDATE_SCHEME = 5
MUCA_OPT_TABLE_WINDOW_ROWS = 6
MUCA_OPT_ACCEPTANCE = 8
MUCA_ACCEPT_THRESHOLD, MUCA_ACCEPT_EXPF32 = 0, 1
MUCA_OPT_ROLE_MAP = 7
MUCA_SCHEME_TYPEWRITER, MUCA_SCHEME_RANDOM_SITE = 0, 1

# every symbol include/muca.h declares (tests/test_abi.py checks the header against this list and the .so)
EXPORTS = (
    "muca_workspace_bytes", "muca_suggest_walkers", "muca_create", "muca_create_in", "muca_destroy", "muca_set_option",
    "muca_set_log_weights", "muca_get_log_weights", "muca_run_iteration", "muca_get_histogram",
    "muca_update_weights", "muca_update_weights_with", "muca_get_energies", "muca_get_spins", "muca_set_spins",
    "muca_unpack_spins_device", "muca_get_thresholds", "muca_get_iteration", "muca_set_iteration",
    "muca_last_sweep_ms", "muca_last_error", "muca_debug_philox", "muca_version",
    "muca_flatness", "muca_schedule", "muca_converge", "muca_production", "muca_run_iteration_random_site", "muca_window_stats",
    "muca_debug_philox_static", "muca_abi_version",
)
MUCA_ABI_VERSION = 3            # include/muca.h: the enum values and signatures this file was written against
MUCA_PHILOX_STATIC_MAX = 4096   # include/muca.h: rows the library's fixed staging array holds


class Flatness(C.Structure):
    """muca_flatness_t (include/muca.h)."""
    _fields_ = [("j_lo", C.c_int), ("j_hi", C.c_int), ("width", C.c_int), ("d_k", C.c_double), ("d_c", C.c_double),
                ("n_updates", C.c_uint64)]


class IterationLog(C.Structure):
    """muca_iteration_log_t (include/muca.h)."""
    _fields_ = [("w", C.c_int), ("therm_sweeps", C.c_int), ("sweeps", C.c_int), ("flat", Flatness),
                ("sweep_ms", C.c_double)]


class MucaError(RuntimeError):
    pass


_lib = None


def checked() -> bool:
    """MUCA_CHECKED=1 in the environment selects the self-checking build of the library (build.py LIB_CHECKED)."""
    return os.environ.get("MUCA_CHECKED", "0") not in ("", "0")


def lib_path() -> str:
    return _build.LIB_CHECKED if checked() else _build.LIB


def lib():
    """Load libmuca_b200.so (building it in-tree with nvcc if it is missing or stale)."""
    global _lib
    if _lib is not None:
        return _lib
    try:
        path = _build.build(checked=checked())
    except _build.NvccMissing as e:   # no compiler here: a library built elsewhere is used as it is; a compile ERROR propagates
        if not os.path.exists(lib_path()):
            raise MucaError(f"{os.path.basename(lib_path())} is not built and cannot be built here: {e}") from e
        path = lib_path()
    L = C.CDLL(path)
    # The constants at the top of this file are raw integers: a library with another numbering (an older build found on
    # the path) would silently run a different kernel or option.  Refuse it instead.
    have = L.muca_abi_version() if hasattr(L, "muca_abi_version") else None
    if have != MUCA_ABI_VERSION:
        raise MucaError(f"{os.path.basename(path)} has ABI version {have}, this binding was written against {MUCA_ABI_VERSION} "
                        f"(include/muca.h MUCA_ABI_VERSION): rebuild the library (python -m paper_1707_00919_b200.build --force)")
    vp, u32p, u64p = C.c_void_p, C.POINTER(C.c_uint32), C.POINTER(C.c_uint64)
    f64p, i8p, i32p = C.POINTER(C.c_double), C.POINTER(C.c_int8), C.POINTER(C.c_int32)
    L.muca_suggest_walkers.argtypes = [C.c_int, C.POINTER(C.c_int), C.POINTER(C.c_int)]
    L.muca_workspace_bytes.argtypes = [C.c_int, C.c_int]
    L.muca_workspace_bytes.restype = C.c_size_t
    L.muca_create.argtypes = [C.POINTER(vp), C.c_int, C.c_int, C.c_uint64]
    L.muca_create_in.argtypes = [C.POINTER(vp), C.c_int, C.c_int, C.c_uint64, C.c_uint32, vp, C.c_size_t, vp]
    L.muca_destroy.argtypes = [vp]
    L.muca_destroy.restype = None
    L.muca_set_option.argtypes = [vp, C.c_int, C.c_int]
    L.muca_set_log_weights.argtypes = [vp, f64p, C.c_int]
    L.muca_get_log_weights.argtypes = [vp, f64p, C.c_int]
    L.muca_run_iteration.argtypes = [vp, C.c_int, C.c_int, u64p, C.c_int]
    L.muca_get_histogram.argtypes = [vp, u64p, C.c_int]
    L.muca_update_weights.argtypes = [vp]
    L.muca_update_weights_with.argtypes = [vp, u64p, C.c_int]
    L.muca_get_energies.argtypes = [vp, i32p, C.c_int]
    L.muca_get_spins.argtypes = [vp, i8p, C.c_size_t]
    L.muca_set_spins.argtypes = [vp, i8p, C.c_size_t]
    L.muca_unpack_spins_device.argtypes = [vp, vp, C.c_size_t]
    L.muca_get_thresholds.argtypes = [vp, u32p, C.c_size_t]
    L.muca_get_iteration.argtypes = [vp, u32p]
    L.muca_set_iteration.argtypes = [vp, C.c_uint32]
    L.muca_last_sweep_ms.argtypes = [vp, f64p, C.POINTER(C.c_int)]
    L.muca_last_error.argtypes = [vp]
    L.muca_last_error.restype = C.c_char_p
    L.muca_debug_philox.argtypes = [u32p, u32p, u32p, C.c_int]
    L.muca_debug_philox_static.argtypes = [u32p, u32p, u32p, C.c_int]
    L.muca_version.restype = C.c_char_p
    L.muca_flatness.argtypes = [u64p, C.c_int, C.c_int, C.POINTER(Flatness)]
    L.muca_schedule.argtypes = [C.c_int, C.c_int, C.c_int, f64p, C.POINTER(C.c_int), C.POINTER(C.c_int),
                                C.POINTER(C.c_int), C.POINTER(C.c_int)]
    L.muca_run_iteration_random_site.argtypes = [vp, C.c_uint64, C.c_uint64, u64p, C.c_int]
    L.muca_window_stats.argtypes = [vp, C.POINTER(C.c_int), C.POINTER(C.c_int)]
    L.muca_production.argtypes = [vp, C.c_int, C.c_int, C.c_int, f64p, f64p, u64p, C.c_int]
    L.muca_converge.argtypes = [vp, C.c_int, C.c_double, C.POINTER(IterationLog), C.c_int, C.POINTER(C.c_int),
                                C.POINTER(C.c_int)]
    _lib = L
    return L


def _p(a, t):
    return a.ctypes.data_as(C.POINTER(t))


def suggest_walkers(L: int):
    """muca_suggest_walkers: (n_walkers, pairs_per_sm) that load the current device fully and evenly."""
    w, p = C.c_int(), C.c_int()
    rc = lib().muca_suggest_walkers(L, C.byref(w), C.byref(p))
    if rc != MUCA_OK:
        raise MucaError(f"muca_suggest_walkers failed rc={rc}")
    return w.value, p.value


def workspace_bytes(L: int, n_walkers: int) -> int:
    return int(lib().muca_workspace_bytes(L, n_walkers))


def debug_philox(ctr, key) -> np.ndarray:
    """Philox4x32-10 evaluated on the device for rows of (ctr[4], key[2])."""
    c = np.ascontiguousarray(ctr, dtype=np.uint32).reshape(-1, 4)
    k = np.ascontiguousarray(key, dtype=np.uint32).reshape(-1, 2)
    out = np.empty_like(c)
    rc = lib().muca_debug_philox(_p(c, C.c_uint32), _p(k, C.c_uint32), _p(out, C.c_uint32), c.shape[0])
    if rc != MUCA_OK:
        raise MucaError(f"muca_debug_philox failed rc={rc}")
    return out


def debug_philox_static(ctr, key) -> np.ndarray:
    """muca_debug_philox_static: what debug_philox computes, for a caller that must not allocate device memory.

    debug_philox makes the library cudaMalloc and cudaFree its staging buffers on every call.  Inside a process whose
    GPU memory belongs to someone else (torch's caching allocator holding most of the HBM, a fixed memory partition)
    that allocation can fail, and it stalls all streams of the device while it runs.  This variant stages the rows in a
    fixed 160 KiB array inside the library instead and allocates nothing; in exchange it takes at most
    MUCA_PHILOX_STATIC_MAX rows per call, and calls share that array (one at a time; the library holds a lock).  The
    first call on a device also looks the array's address up: make it at set-up, before any stream capture."""
    c = np.ascontiguousarray(ctr, dtype=np.uint32).reshape(-1, 4)
    k = np.ascontiguousarray(key, dtype=np.uint32).reshape(-1, 2)
    if c.shape[0] != k.shape[0]:
        raise MucaError(f"muca_debug_philox_static: {c.shape[0]} counter rows but {k.shape[0]} key rows")
    out = np.empty_like(c)
    rc = lib().muca_debug_philox_static(_p(c, C.c_uint32), _p(k, C.c_uint32), _p(out, C.c_uint32), c.shape[0])
    if rc == -4:
        raise MucaError(f"muca_debug_philox_static: {c.shape[0]} rows do not fit the library's fixed staging array "
                        f"(at most MUCA_PHILOX_STATIC_MAX = {MUCA_PHILOX_STATIC_MAX} per call); nothing was computed")
    if rc != MUCA_OK:
        raise MucaError(f"muca_debug_philox_static failed rc={rc}")
    return out


def flatness(H, w: int) -> dict:
    """muca_flatness: width, d_k (Eq. (6)), d_c (Eq. (A.1)) of a histogram against Q = 1/w (host only)."""
    h = np.ascontiguousarray(H, dtype=np.uint64)
    f = Flatness()
    rc = lib().muca_flatness(_p(h, C.c_uint64), h.size, int(w), C.byref(f))
    if rc != MUCA_OK:
        raise MucaError(f"muca_flatness failed rc={rc}")
    return {k: getattr(f, k) for k, _ in Flatness._fields_}


def schedule(L: int, n_walkers: int, w_prev: int, n_updates: float = 0.0, full_range: int = 0):
    """muca_schedule: (w, therm_sweeps, sweeps, n_updates, full_range) of the next iteration (Eq. (7); host only)."""
    nu, fr, w, th, sw = C.c_double(n_updates), C.c_int(full_range), C.c_int(), C.c_int(), C.c_int()
    rc = lib().muca_schedule(L, n_walkers, int(w_prev), C.byref(nu), C.byref(fr), C.byref(w), C.byref(th), C.byref(sw))
    if rc != MUCA_OK:
        raise MucaError(f"muca_schedule failed rc={rc}")
    return w.value, th.value, sw.value, nu.value, fr.value


class Muca:
    """W walkers on L x L lattices on the current CUDA device (global walker ids walker_offset .. +W-1)."""

    def __init__(self, L: int, n_walkers: int, seed: int, walker_offset: int = 0, device=None):
        import torch
        if not torch.cuda.is_available():
            raise MucaError("no CUDA device: libmuca_b200 has no CPU fallback")
        self._lib = lib()
        self.device = torch.device("cuda", torch.cuda.current_device()) if device is None else torch.device(device)
        nbytes = workspace_bytes(L, n_walkers)
        if nbytes == 0:
            raise MucaError(f"unsupported (L={L}, n_walkers={n_walkers}): L in {{8,16,32,64,128}}, n_walkers >= 1")
        with torch.cuda.device(self.device):
            self._workspace = torch.empty(nbytes + 256, dtype=torch.uint8, device=self.device)
            ptr = (self._workspace.data_ptr() + 255) // 256 * 256
            self._stream = torch.cuda.current_stream(self.device)
            h = C.c_void_p()
            rc = self._lib.muca_create_in(C.byref(h), L, n_walkers, C.c_uint64(seed & (2 ** 64 - 1)),
                                          C.c_uint32(walker_offset), C.c_void_p(ptr), nbytes,
                                          C.c_void_p(self._stream.cuda_stream))
        if rc != MUCA_OK or not h:
            raise MucaError(f"muca_create_in failed rc={rc}")
        self._h = h
        self.L, self.N, self.W = L, L * L, n_walkers
        self.n_bins = self.N + 1
        self.seed, self.walker_offset = seed, walker_offset

    # -- lifetime
    def close(self):
        if getattr(self, "_h", None):
            self._lib.muca_destroy(self._h)
            self._h = None
            self._workspace = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()

    def _check(self, rc, what):
        if rc != MUCA_OK:
            msg = self._lib.muca_last_error(self._h)
            raise MucaError(f"{what} failed rc={rc}: {msg.decode() if msg else ''}")

    # -- include/muca.h, one method per entry point
    def set_option(self, option: int, value: int):
        self._check(self._lib.muca_set_option(self._h, option, value), "muca_set_option")

    def set_log_weights(self, logw):
        w = np.ascontiguousarray(logw, dtype=np.float64)
        self._check(self._lib.muca_set_log_weights(self._h, _p(w, C.c_double), w.size), "muca_set_log_weights")

    def get_log_weights(self) -> np.ndarray:
        out = np.empty(self.n_bins, dtype=np.float64)
        self._check(self._lib.muca_get_log_weights(self._h, _p(out, C.c_double), out.size), "muca_get_log_weights")
        return out

    def run_iteration(self, therm_sweeps: int, sweeps: int) -> np.ndarray:
        H = np.empty(self.n_bins, dtype=np.uint64)
        self._check(self._lib.muca_run_iteration(self._h, therm_sweeps, sweeps, _p(H, C.c_uint64), H.size),
                    "muca_run_iteration")
        return H

    def get_histogram(self) -> np.ndarray:
        H = np.empty(self.n_bins, dtype=np.uint64)
        self._check(self._lib.muca_get_histogram(self._h, _p(H, C.c_uint64), H.size), "muca_get_histogram")
        return H

    def update_weights(self):
        self._check(self._lib.muca_update_weights(self._h), "muca_update_weights")

    def update_weights_with(self, H_total):
        h = np.ascontiguousarray(H_total, dtype=np.uint64)
        self._check(self._lib.muca_update_weights_with(self._h, _p(h, C.c_uint64), h.size), "muca_update_weights_with")

    def get_energies(self, out: np.ndarray = None) -> np.ndarray:
        if out is None:
            out = np.empty(self.W, dtype=np.int32)
        assert out.dtype == np.int32 and out.size == self.W and out.flags.c_contiguous
        self._check(self._lib.muca_get_energies(self._h, _p(out, C.c_int32), out.size), "muca_get_energies")
        return out

    def get_spins(self, out: np.ndarray = None) -> np.ndarray:
        if out is None:
            out = np.empty((self.W, self.L, self.L), dtype=np.int8)
        assert out.dtype == np.int8 and out.size == self.W * self.N and out.flags.c_contiguous
        self._check(self._lib.muca_get_spins(self._h, _p(out, C.c_int8), out.size), "muca_get_spins")
        return out

    def set_spins(self, spins):
        s = np.ascontiguousarray(spins, dtype=np.int8)
        self._check(self._lib.muca_set_spins(self._h, _p(s, C.c_int8), s.size), "muca_set_spins")

    def unpack_spins_device(self):
        """int8 CUDA tensor [W, L, L] of +1/-1, produced on the context's stream (no host copy)."""
        import torch
        out = torch.empty((self.W, self.L, self.L), dtype=torch.int8, device=self.device)
        self._check(self._lib.muca_unpack_spins_device(self._h, C.c_void_p(out.data_ptr()), out.numel()),
                    "muca_unpack_spins_device")
        return out

    def get_thresholds(self) -> np.ndarray:
        out = np.empty((self.n_bins, 5), dtype=np.uint32)
        self._check(self._lib.muca_get_thresholds(self._h, _p(out, C.c_uint32), out.size), "muca_get_thresholds")
        return out

    @property
    def iteration(self) -> int:
        n = C.c_uint32()
        self._check(self._lib.muca_get_iteration(self._h, C.byref(n)), "muca_get_iteration")
        return int(n.value)

    @iteration.setter
    def iteration(self, n: int):
        self._check(self._lib.muca_set_iteration(self._h, C.c_uint32(n)), "muca_set_iteration")

    def run_iteration_random_site(self, therm_updates: int, updates: int) -> np.ndarray:
        """muca_run_iteration_random_site: the paper's own scheme (same random site in all walkers); counts in updates."""
        H = np.empty(self.n_bins, dtype=np.uint64)
        self._check(self._lib.muca_run_iteration_random_site(self._h, C.c_uint64(therm_updates), C.c_uint64(updates),
                                                             _p(H, C.c_uint64), self.n_bins), "muca_run_iteration_random_site")
        return H

    def converge(self, max_iterations: int, d_flat: float = 1e-4):
        """muca_converge: the paper's weight iteration until d_k < d_flat.  Returns (log records, converged)."""
        cap = max(int(max_iterations), 1)
        log = (IterationLog * cap)()
        n, conv = C.c_int(), C.c_int()
        self._check(self._lib.muca_converge(self._h, int(max_iterations), float(d_flat), log, cap, C.byref(n), C.byref(conv)),
                    "muca_converge")
        out = []
        for r in log[:n.value]:
            d = {"w": r.w, "therm_sweeps": r.therm_sweeps, "sweeps": r.sweeps, "sweep_ms": r.sweep_ms}
            d.update({k: getattr(r.flat, k) for k, _ in Flatness._fields_})
            out.append(d)
        return out, bool(conv.value)

    def production(self, n_calls: int, therm_sweeps: int, sweeps: int):
        """muca_production: fixed-weight calls + jackknife.  Returns (ln_omega, err, histograms[n_calls, n_bins])."""
        ln_om, err = np.empty(self.n_bins, dtype=np.float64), np.empty(self.n_bins, dtype=np.float64)
        Hs = np.empty((max(int(n_calls), 0), self.n_bins), dtype=np.uint64)
        self._check(self._lib.muca_production(self._h, int(n_calls), int(therm_sweeps), int(sweeps), _p(ln_om, C.c_double),
                                              _p(err, C.c_double), _p(Hs, C.c_uint64), self.n_bins), "muca_production")
        return ln_om, err, Hs

    def window_stats(self):
        a, b = C.c_int(), C.c_int()
        self._check(self._lib.muca_window_stats(self._h, C.byref(a), C.byref(b)), "muca_window_stats")
        return int(a.value), int(b.value)

    def last_sweep_ms(self):
        ms, k = C.c_double(), C.c_int()
        self._check(self._lib.muca_last_sweep_ms(self._h, C.byref(ms), C.byref(k)), "muca_last_sweep_ms")
        return float(ms.value), int(k.value)
