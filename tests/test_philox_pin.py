"""P1 — pin the oracle's Philox4x32-10 to the CUDA toolkit's own routines (Ref. [41]).

Two independent library implementations (tests/pins/curand_philox_shim.cpp):
  * curand_Philox4x32_10(uint4, uint2) from curand_philox4x32_x.h, compiled for the host;
  * libcurand's host generator CURAND_RNG_PSEUDO_PHILOX4_32_10, whose i-th group of four
    outputs (offset 0, i < 4096) is Philox(ctr = (0, 0, i, 0), key = (seed_lo, seed_hi)).
"""
import ctypes

import numpy as np

import muca_oracle as mo

U32P = ctypes.POINTER(ctypes.c_uint32)


def _curand(lib, ctr, key):
    c = np.asarray(ctr, dtype=np.uint32)
    k = np.asarray(key, dtype=np.uint32)
    out = np.zeros(4, dtype=np.uint32)
    lib.pin_curand_philox4x32_10(c.ctypes.data_as(U32P), k.ctypes.data_as(U32P), out.ctypes.data_as(U32P))
    return out


def test_philox_matches_toolkit_routine_random_inputs(curand_pin):
    rng = np.random.default_rng(20170700919)
    for _ in range(2000):
        ctr = rng.integers(0, 2**32, size=4, dtype=np.uint64).astype(np.uint32)
        key = rng.integers(0, 2**32, size=2, dtype=np.uint64).astype(np.uint32)
        assert np.array_equal(mo.philox4x32_10(ctr, key), _curand(curand_pin, ctr, key))


def test_philox_matches_toolkit_routine_structured_inputs(curand_pin):
    # the counters the method actually uses: (i>>2, sweep, iteration, walker), and the init domain
    for seed in (170700919, 1, 0xDEADBEEFCAFEF00D, 0, 2**64 - 1):
        key = [seed & 0xFFFFFFFF, seed >> 32]
        for ctr in ([0, 0, 0, 0], [1, 0, 0, 0], [0, 1, 0, 0], [0, 0, 1, 0], [0, 0, 0, 1],
                    [255, 549, 14, 16383], [4095, 69, 4, 8191], [3, 0, 0xFFFFFFFF, 77],
                    [0xFFFFFFFF] * 4):
            assert np.array_equal(mo.philox4x32_10(ctr, key), _curand(curand_pin, ctr, key))


def test_philox_matches_curand_host_generator(curand_pin):
    for seed in (170700919, 0xDEADBEEFCAFEF00D):
        n_groups = 4096
        out = np.zeros(4 * n_groups, dtype=np.uint32)
        rc = curand_pin.pin_curand_host_generate(seed, 0, out.ctypes.data_as(U32P), out.size)
        assert rc == 0
        key = [seed & 0xFFFFFFFF, seed >> 32]
        for i in list(range(64)) + [100, 1000, 4095]:
            assert np.array_equal(mo.philox4x32_10([0, 0, i, 0], key), out[4 * i:4 * i + 4]), i


def test_philox_is_a_bijection_on_a_small_slice():
    # a counter-based generator maps distinct counters to distinct outputs (Ref. [41]); 4096 counters, no collision
    key = [123, 456]
    seen = set()
    for x in range(4096):
        seen.add(tuple(int(v) for v in mo.philox4x32_10([x, 0, 0, 0], key)))
    assert len(seen) == 4096


def test_philox_word_statistics():
    # crude equidistribution check of the 32-bit words: mean ~ 2^31, each bit ~ 1/2
    key = [170700919, 0]
    words = np.concatenate([mo.philox4x32_10([x, 7, 3, 11], key) for x in range(4000)]).astype(np.float64)
    assert abs(words.mean() / 2**32 - 0.5) < 0.01
    bits = (np.concatenate([mo.philox4x32_10([x, 7, 3, 11], key) for x in range(2000)])[:, None]
            >> np.arange(32, dtype=np.uint32)[None, :]) & 1
    assert np.all(np.abs(bits.mean(axis=0) - 0.5) < 0.03)
