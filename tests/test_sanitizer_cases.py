"""Small parity cases, one per default kernel and launch shape, sized to run under compute-sanitizer.

`compute-sanitizer --tool racecheck|memcheck python -m pytest tests/test_sanitizer_cases.py -q -m gpu` slows the
kernels by two to three orders of magnitude, so every case is a few blocks and a few sweeps; each still crosses a
block border, has a ragged last warp and compares H, E and spins with the oracle (SURVEY 5 "race detection";
PAPER.md:119: the histogram is the method's only shared state, resolved by atomics).  Summaries: profiles/.
"""
import numpy as np
import pytest

import muca_oracle as mo
import paper_1707_00919_b200 as mb
from paper_1707_00919_b200 import binding as B

pytestmark = pytest.mark.gpu


def pair(L, W, therm, sweeps, iters=2, options=(), random_site=False):
    g, o = mb.Muca(L, W, 20260411, walker_offset=3), mo.Oracle(L, W, 20260411, walker_offset=3)
    try:
        for k, v in options:
            g.set_option(k, v)
        for it in range(iters):
            if random_site:
                Hg, Ho = g.run_iteration_random_site(therm, sweeps), o.run_iteration_random_site(therm, sweeps, n_threads=mo.max_threads())
            else:
                Hg, Ho = g.run_iteration(therm, sweeps), o.run_iteration(therm, sweeps, n_threads=mo.max_threads())
            assert np.array_equal(Hg, Ho), f"it{it}: H differs in slots {np.nonzero(Hg != Ho)[0][:8]}"
            g.update_weights(); o.update_weights()
        assert np.array_equal(g.get_energies(), o.get_energies())
        assert np.array_equal(g.get_spins(), o.get_spins())
        return g.window_stats()
    finally:
        g.close(); o.close()


# resident kernel (L <= 32): 1, 2 and 4 walker/deviate warp pairs per block, ragged last warp, unused lanes parked
@pytest.mark.parametrize("L,W,tpb,wpw", [(8, 70, 32, 0), (16, 150, 64, 0), (32, 270, 128, 0), (32, 119, 128, 28), (32, 40, 0, 0)])
def test_resident_pairs(L, W, tpb, wpw):
    opts = [(B.MUCA_OPT_THREADS_PER_BLOCK, tpb)] if tpb else []
    if wpw:
        opts.append((B.MUCA_OPT_WALKERS_PER_WARP, wpw))
    pair(L, W, 1, 2, options=tuple(opts))


# paired streamed kernel: L = 64 with the whole table in shared memory, L = 128 with the default window
@pytest.mark.parametrize("L,W", [(64, 75), (128, 41)])
def test_streamed_pairs(L, W):
    pair(L, W, 1, 2 if L == 64 else 1)


# L = 128 with a forced 300-row window: sentinel rows, and (with walkers starting 45 slots wide) the snapshot fallback
def test_window_sentinels_and_fallback():
    windowed, fallbacks = pair(128, 41, 1, 2, iters=3, options=((B.MUCA_OPT_TABLE_WINDOW_ROWS, 300),))
    assert windowed + fallbacks > 0


# a split iteration (several launches share the global histogram)
def test_split_launches():
    pair(32, 70, 1, 3, options=((B.MUCA_OPT_MAX_SWEEPS_PER_LAUNCH, 1),))


# the paper's own update scheme
@pytest.mark.parametrize("L,W", [(16, 70), (32, 140)])
def test_random_site(L, W):
    pair(L, W, 100, 700, random_site=True)
