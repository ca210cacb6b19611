"""muca_debug_philox_static -- the Philox test hook for callers that are not allowed to allocate device memory.

Some users of this library run it inside a process whose GPU memory is not theirs to hand out: a framework's caching
allocator (torch's, for one) has taken most of the HBM, or the job runs in a fixed memory partition.  A raw cudaMalloc
from inside the library can then fail although the framework has room to spare, and it stalls every stream of the
device while it runs.  muca_debug_philox does exactly that (three cudaMalloc / cudaFree per call); the `_static`
variant keeps its staging rows in a fixed 160 KiB array that is part of the library and allocates nothing, at the price
of a row limit (MUCA_PHILOX_STATIC_MAX per call) and of all calls sharing that one array.

What is checked here: the static variant returns, bit for bit (integer work: no tolerance), what the allocating path
returns -- on two calls in a row, the second shorter than the first, so that rows left over from the first call would
show up if they could leak into the second; a request beyond the limit is refused with a clear message and without
touching the array's use by later calls.

This file sorts after every other test file on purpose: `pytest -x` stops at the first failure, and a failure here
must not hide the parity tests.  It depends on nothing the earlier tests leave behind and passes alone in a fresh
process as well (the first call on a device does the one-time address look-up itself).
"""
import numpy as np
import pytest

import paper_1707_00919_b200 as mb
from paper_1707_00919_b200 import binding as B

pytestmark = pytest.mark.gpu


def rows(seed, n):
    rng = np.random.default_rng(seed)
    ctr = rng.integers(0, 2 ** 32, size=(n, 4), dtype=np.uint64).astype(np.uint32)
    key = rng.integers(0, 2 ** 32, size=(n, 2), dtype=np.uint64).astype(np.uint32)
    return ctr, key


def test_static_scratch_philox_matches_the_allocating_path_on_two_calls_in_a_row():
    n_max = B.MUCA_PHILOX_STATIC_MAX
    # first call: the array filled to its last row (and the counters the sweep kernels use at the corners of their range)
    ctr1, key1 = rows(20170700919, n_max)
    ctr1[:4] = [[0, 0, 0, 0], [0xFFFFFFFF] * 4, [255, 549, 14, 16383], [3, 0, 0xFFFFFFFF, 77]]
    got1 = mb.debug_philox_static(ctr1, key1)
    # second call straight after it: other rows, fewer of them, not a multiple of the block size -- the tail of the
    # array still holds the first call's rows
    ctr2, key2 = rows(919, 1000 + 37)
    got2 = mb.debug_philox_static(ctr2, key2)
    want1, want2 = mb.debug_philox(ctr1, key1), mb.debug_philox(ctr2, key2)
    assert got1.dtype == np.uint32 and got1.shape == (n_max, 4) and got2.shape == (1037, 4)
    assert np.array_equal(got1, want1)
    assert np.array_equal(got2, want2)
    assert not np.array_equal(got2, got1[:1037])       # the second result is its own, not the first call's rows
    # one row, the smallest request
    assert np.array_equal(mb.debug_philox_static(ctr1[:1], key1[:1]), want1[:1])


def test_static_scratch_philox_refuses_more_rows_than_the_array_holds():
    n_max = B.MUCA_PHILOX_STATIC_MAX
    ctr, key = rows(3, n_max + 1)
    with pytest.raises(mb.MucaError, match="MUCA_PHILOX_STATIC_MAX"):
        mb.debug_philox_static(ctr, key)
    import ctypes as C
    u32p = C.POINTER(C.c_uint32)
    out = np.full((n_max + 1, 4), 0xA5A5A5A5, dtype=np.uint32)
    rc = mb.lib().muca_debug_philox_static(ctr.ctypes.data_as(u32p), key.ctypes.data_as(u32p), out.ctypes.data_as(u32p), n_max + 1)
    assert rc == -4 and np.all(out == 0xA5A5A5A5)      # MUCA_ENOMEM, output untouched
    assert mb.lib().muca_debug_philox_static(ctr.ctypes.data_as(u32p), key.ctypes.data_as(u32p), out.ctypes.data_as(u32p), 0) == -1
    assert mb.lib().muca_debug_philox_static(None, key.ctypes.data_as(u32p), out.ctypes.data_as(u32p), 8) == -1
    # the refusal left nothing behind: the next call within the limit is served as usual
    assert np.array_equal(mb.debug_philox_static(ctr[:n_max], key[:n_max]), mb.debug_philox(ctr[:n_max], key[:n_max]))
