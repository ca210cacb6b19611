"""Convergence protocol (Eq. (6), (7), (A.1)).

not gpu: the oracle's numpy restatement is pinned against closed forms, scipy's relative entropy and exact integer
         arithmetic; the library's host functions (muca_flatness, muca_schedule: no device needed) must agree with it.
gpu    : muca_converge (library, CUDA sweeps) against the oracle driven through the same protocol: identical
         schedules, widths and histogram sums, d_k / d_c within 1e-12, final omega within 1e-12.
"""
import math
from fractions import Fraction

import numpy as np
import pytest

import muca_convergence as mc
import muca_oracle as mo
import paper_1707_00919_b200 as mb


# ------------------------------------------------------------------------------------------------ oracle pins
def test_flatness_closed_forms():
    n_bins = 65                                   # L = 8
    H = np.zeros(n_bins, dtype=np.uint64)
    H[20:30] = 7                                  # flat over m = 10 slots: d_k = ln(w / m) for any w (Eq. (6))
    for w in (10, 13, 65):
        f = mc.flatness(H, w)
        assert (f["j_lo"], f["j_hi"], f["width"], f["n_updates"]) == (20, 29, 10, 70)
        assert abs(f["d_k"] - math.log(w / 10)) < 1e-14
    # two-level histogram, by hand: P = (3/4, 1/4), Q = 1/2 -> d_k = 3/4 ln(3/2) + 1/4 ln(1/2)
    H[:] = 0; H[4], H[6] = 3, 1
    assert abs(mc.flatness(H, 2)["d_k"] - (0.75 * math.log(1.5) + 0.25 * math.log(0.5))) < 1e-15
    # Chebyshev distance (Eq. (A.1)): exactly flat over the N - 1 = 63 accessible slots -> 0; one of them doubled
    H[:] = 5; H[1] = H[63] = 0
    assert mc.flatness(H, 65)["d_c"] == 0.0 and mc.flatness(H, 65)["width"] == 65
    H[10] = 10
    m = Fraction(int(H.sum()), 63)
    assert abs(mc.flatness(H, 65)["d_c"] - float(Fraction(10) / m - 1)) < 1e-15
    # w = 0: the reference width is max(own width, 10)  (R19)
    H[:] = 0; H[30:50] = 3
    assert abs(mc.flatness(H)["d_k"]) < 1e-15 and abs(mc.flatness(H[:40])["d_k"] - math.log(10 / 10)) < 1e-15
    H[:] = 0; H[30:34] = 3
    assert abs(mc.flatness(H)["d_k"] - math.log(10 / 4)) < 1e-15
    H[:] = 9; H[1] = H[63] = 0                     # flat over the whole axis: the 63 accessible slots are the reference
    assert abs(mc.flatness(H)["d_k"]) < 1e-15 and abs(mc.flatness(H, 65)["d_k"] - math.log(65 / 63)) < 1e-14
    H[:] = 0
    assert mc.flatness(H, 10) == {"j_lo": -1, "j_hi": -1, "width": 0, "d_k": 0.0, "d_c": 0.0, "n_updates": 0}


def test_flatness_against_scipy_relative_entropy():
    from scipy.stats import entropy               # entropy(p, q) = sum p ln(p / q): the library routine for Eq. (6)
    rng = np.random.default_rng(5)
    for n_bins, w in ((65, 40), (257, 257), (1025, 600)):
        H = rng.integers(0, 1000, n_bins).astype(np.uint64)
        H[rng.random(n_bins) < 0.3] = 0
        H[1] = H[n_bins - 2] = 0
        visited = H > 0
        P = H[visited] / H.sum()
        d_ref = entropy(P, np.full(P.size, 1.0 / w))      # scipy normalises q: undo it with the analytic constant
        d_ref += math.log(w / P.size)
        assert abs(mc.flatness(H, w)["d_k"] - d_ref) < 1e-12


def test_schedule_against_exact_arithmetic():
    import mpmath as mp
    mp.mp.dps = 50
    for L, W, w_prev in ((8, 128, 0), (8, 128, 37), (16, 4096, 200), (32, 16384, 1025), (32, 26624, 700), (64, 32768, 4097)):
        N = L * L
        w = max(w_prev, 10)
        n_up = int(mp.floor(6 * mp.mpf(w) ** mp.mpf("2.25") / W)) + 1            # Eq. (7), truncated, + 1
        got = mc.schedule(L, W, w_prev)
        assert got == (w, max(1, math.ceil(30 * w / N)), max(1, math.ceil(n_up / N)), float(n_up), int(w >= N + 1))
    # whole range covered: Eq. (7) once, then x 1.1 (truncated, + 1) per iteration
    w, th, sw, n0, full = mc.schedule(8, 128, 65)
    assert full == 1 and n0 == math.floor(6 * 65 ** 2.25 / 128) + 1
    _, _, sw1, n1, full1 = mc.schedule(8, 128, 65, n0, full)
    assert n1 == math.floor(1.1 * n0) + 1 and sw1 == math.ceil(n1 / 64) and full1 == 1
    # the range shrank again (possible in principle): back to Eq. (7)
    assert mc.schedule(8, 128, 60, n1, 0)[3] == math.floor(6 * 60 ** 2.25 / 128) + 1
    # paper's example sizes: W = 26 624 walkers, L = 32: N_therm = 30 * 1025 flips -> 31 sweeps
    assert mc.schedule(32, 26624, 1025)[1] == 31


def test_oracle_converges_to_a_flat_histogram_L8():
    # the protocol itself: L = 8 reaches d_k < 1e-4 and the weights then reproduce the exact density of states
    o = mo.Oracle(8, 256, 11)
    log, conv = mc.converge(o, 90, 1e-4, n_threads=mo.max_threads())
    assert conv and log[-1]["width"] == 65 and log[-1]["d_c"] < 0.2
    assert all(r["n_updates"] == 256 * 64 * r["sweeps"] for r in log)
    widths = [r["width"] for r in log]
    assert widths[0] < 65 and max(widths) == 65          # the range grows from the initial peak to the whole axis
    o.close()


# ------------------------------------------------------------------------------------------------ library host functions
def test_library_host_functions_match_the_oracle_protocol():
    rng = np.random.default_rng(9)
    for n_bins, w in ((65, 10), (257, 100), (1025, 1025), (4097, 3000), (257, 0), (1025, 0)):
        H = rng.integers(0, 50000, n_bins).astype(np.uint64)
        H[rng.random(n_bins) < 0.2] = 0
        H[1] = H[n_bins - 2] = 0
        a, b = mb.flatness(H, w), mc.flatness(H, w)
        assert all(a[k] == b[k] for k in ("j_lo", "j_hi", "width", "n_updates"))
        assert abs(a["d_k"] - b["d_k"]) < 1e-12 and abs(a["d_c"] - b["d_c"]) < 1e-12
    assert mb.flatness(np.zeros(65, dtype=np.uint64), 10)["width"] == 0
    for L, W in ((8, 128), (16, 4096), (32, 16384), (64, 32768), (128, 8192)):
        n_up, full = 0.0, 0
        for w_prev in (0, 5, 11, L * L // 3, L * L, L * L + 1, L * L + 1, L * L + 1):
            a = mb.schedule(L, W, w_prev, n_up, full)
            assert a == mc.schedule(L, W, w_prev, n_up, full)
            n_up, full = a[3], a[4]
    with pytest.raises(mb.MucaError):
        mb.schedule(12, 10, 0)


# ------------------------------------------------------------------------------------------------ GPU parity
@pytest.mark.gpu
@pytest.mark.parametrize("L,W,seed,max_it,random_site", [(8, 128, 170700919, 60, False), (16, 512, 1, 25, False), (32, 300, 7, 8, False),
                                                         (8, 128, 170700919, 60, True), (16, 512, 1, 25, True)])
def test_gpu_converge_matches_oracle(L, W, seed, max_it, random_site):
    from paper_1707_00919_b200 import binding as B
    g, o = mb.Muca(L, W, seed), mo.Oracle(L, W, seed)
    try:
        if random_site:                          # the paper's own update scheme and units (R22)
            g.set_option(B.MUCA_OPT_UPDATE_SCHEME, B.MUCA_SCHEME_RANDOM_SITE)
        lg, cg = g.converge(max_it, 1e-4)
        lo, co = mc.converge(o, max_it, 1e-4, n_threads=mo.max_threads(), random_site=random_site)
        assert cg == co and len(lg) == len(lo)
        for a, b in zip(lg, lo):
            for k in ("w", "therm_sweeps", "sweeps", "j_lo", "j_hi", "width", "n_updates"):
                assert a[k] == b[k], (k, a, b)
            assert abs(a["d_k"] - b["d_k"]) < 1e-12 and abs(a["d_c"] - b["d_c"]) < 1e-12
        assert np.max(np.abs(g.get_log_weights() - o.get_log_weights())) <= 1e-12
        assert np.array_equal(g.get_energies(), o.get_energies())
        assert np.array_equal(g.get_spins(), o.get_spins())
        assert g.iteration == len(lg)
    finally:
        g.close(); o.close()
