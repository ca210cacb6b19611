"""Pins of the CPU oracle against what the paper and the mathematics fix (no GPU, no product code).

P2 brute force 2^16 states (L=4)       -> energy function, slot indexing, forbidden slots
thresholds vs arbitrary precision      -> acceptance table (PAPER.md:109 min(1, exp[w(E')-w(E)]))
init mapping vs toolkit Philox         -> R1 indexing
P5 omega == 0 closed form              -> sweep order, flip logic, H timing (independent of the RNG)
P4 invariants                          -> bookkeeping
P6 omega = -beta E                     -> acceptance = textbook canonical Metropolis, exact <E>, P(E)
P7 omega = -ln g_exact                 -> flat histogram (the paper's timing workload)
P3 whole recursion vs exact ln g       -> Eq. (4) + everything, max |d ln g| < 0.05 (north_star)
P8 Eq. (4)                             -> weight update on hand-made H
"""
import ctypes
import itertools
import math
import os

import mpmath as mp
import numpy as np
import pytest

import exact_dos
import muca_oracle as mo

GOLDEN = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


def golden_g(L):
    with open(os.path.join(GOLDEN, f"ising_dos_L{L}.txt")) as f:
        return [int(x) for x in f if not x.startswith("#")]


def ln_g_from(g):
    return np.array([float(mp.log(v)) if v > 0 else -np.inf for v in g])


# ------------------------------------------------------------------ P2 -----
def test_bruteforce_L4_density_of_states():
    L, N = 4, 16
    counts = np.zeros(N + 1, dtype=np.int64)
    for bits in range(1 << N):
        s = np.array([1 - 2 * ((bits >> i) & 1) for i in range(N)], dtype=np.int8).reshape(L, L)
        E = mo.energy(s)
        assert E % 4 == 0 and -2 * N <= E <= 2 * N
        counts[(E + 2 * N) // 4] += 1
    # values fixed by enumeration and, independently, by the closed form
    assert counts.tolist() == [2, 0, 32, 64, 424, 1728, 6688, 13568, 20524,
                               13568, 6688, 1728, 424, 64, 32, 0, 2]
    assert counts.tolist() == golden_g(4)
    assert counts.tolist() == exact_dos.exact_g(4)


def test_energy_special_configurations():
    for L in (4, 6, 8, 16):
        N = L * L
        up = np.ones((L, L), dtype=np.int8)
        assert mo.energy(up) == -2 * N and mo.energy(-up) == -2 * N          # ground states
        cb = np.fromfunction(lambda y, x: 1 - 2 * ((x + y) % 2), (L, L)).astype(np.int8)
        assert mo.energy(cb) == 2 * N                                           # antiferromagnetic ceiling
        one = up.copy(); one[1, 2] = -1
        assert mo.energy(one) == -2 * N + 8                                     # single flip costs 4 bonds: dE = 8
        stripes = np.fromfunction(lambda y, x: 1 - 2 * (y % 2), (L, L)).astype(np.int8)
        assert mo.energy(stripes) == 0                                          # horizontal bonds -N, vertical +N
        # a transposed-operand / missing-direction mistake shows up on an anisotropic configuration
        col = up.copy(); col[:, 0] = -1
        assert mo.energy(col) == -2 * N + 4 * L


def test_golden_dos_matches_closed_form_L8():
    assert exact_dos.exact_g(8) == golden_g(8)
    g16 = golden_g(16)
    assert sum(g16) == 2 ** 256 and g16 == g16[::-1] and g16[:4] == [2, 0, 512, 1024]


# ----------------------------------------------------------- thresholds -----
def test_thresholds_against_arbitrary_precision():
    rng = np.random.default_rng(7)
    n_bins = 65
    logw = np.cumsum(rng.normal(0, 1.5, n_bins))       # rough table with large and small ratios
    logw[10] = logw[8]                                   # an exact tie: d = 0 -> always accept
    logw[40] = logw[38] - 30.0                           # p ~ 1e-13 < 2^-32 -> clamps to T = 1, t = 0
    t = mo.thresholds(logw)
    assert t.shape == (n_bins, 5)
    n_exact = n_total = 0
    with mp.workdps(60):
        for j in range(n_bins):
            for a in range(5):
                jp = j + 2 - a
                if a == 2:
                    want = 0xFFFFFFFF
                elif jp < 0 or jp >= n_bins:
                    want = 0
                else:
                    d = float(logw[jp]) - float(logw[j])     # one IEEE subtraction (R7)
                    if d >= 0:
                        want = 0xFFFFFFFF
                    else:
                        T = int(mp.floor(mp.exp(mp.mpf(d)) * 2 ** 32))
                        T = min(max(T, 1), 2 ** 32)
                        want = T - 1
                n_total += 1
                got = int(t[j, a])
                assert abs(got - want) <= 1, (j, a, got, want)   # libm exp is within 1 ulp
                n_exact += got == want
    assert n_exact >= n_total - 1
    assert t[10, 4] == 0xFFFFFFFF and t[8, 0] == 0xFFFFFFFF      # tie, both directions
    assert t[38, 0] == 0                                          # clamped tiny probability
    assert t[0, 3] == 0 and t[0, 4] == 0 and t[n_bins - 1, 0] == 0 and t[n_bins - 1, 1] == 0


def test_thresholds_direction_and_probability():
    # omega = -beta*E: moving UP in energy by dE has p = exp(-beta dE); moving down is always accepted.
    beta, n_bins = 0.25, 17
    E = -32 + 4 * np.arange(n_bins)
    t = mo.thresholds(-beta * E)
    for a, dE in ((0, 8), (1, 4)):                       # a antiparallel neighbours -> dE = 8 - 4a
        p = (t[5, a].astype(np.float64) + 1) / 2 ** 32
        assert abs(p - math.exp(-beta * dE)) < 1e-9
    assert t[5, 3] == 0xFFFFFFFF and t[5, 4] == 0xFFFFFFFF and t[5, 2] == 0xFFFFFFFF


# ------------------------------------------------------------- init ---------
def test_init_mapping_against_toolkit_philox(curand_pin):
    U32P = ctypes.POINTER(ctypes.c_uint32)
    L, W, seed, off = 16, 5, 0xDEADBEEFCAFEF00D, 1000
    o = mo.Oracle(L, W, seed, walker_offset=off)
    spins = o.get_spins().reshape(W, -1)
    key = np.array([seed & 0xFFFFFFFF, seed >> 32], dtype=np.uint32)
    for w in range(W):
        for i in range(L * L):
            ctr = np.array([i >> 7, 0, 0xFFFFFFFF, off + w], dtype=np.uint32)
            out = np.zeros(4, dtype=np.uint32)
            curand_pin.pin_curand_philox4x32_10(ctr.ctypes.data_as(U32P), key.ctypes.data_as(U32P),
                                                out.ctypes.data_as(U32P))
            bit = (int(out[(i >> 5) & 3]) >> (i & 31)) & 1
            assert spins[w, i] == 1 - 2 * bit
    E = o.get_energies()
    for w in range(W):
        assert E[w] == mo.energy(spins[w].reshape(L, L))


def test_init_is_uniform():
    L, W = 16, 2000
    o = mo.Oracle(L, W, 170700919)
    s = o.get_spins().astype(np.float64)
    assert abs(s.mean()) < 0.01
    E = o.get_energies().astype(np.float64)
    # independent +-1 spins: <E> = 0, var E = number of bonds = 2N
    assert abs(E.mean()) < 4 * math.sqrt(2 * L * L / W)
    assert abs(E.var() / (2 * L * L) - 1) < 0.15
    # walkers differ from each other
    assert len({s[w].tobytes() for w in range(50)}) == 50


# ------------------------------------------------------------------ P5 -----
def _numpy_energy(s):
    return int(-(s * np.roll(s, -1, 1)).sum() - (s * np.roll(s, -1, 0)).sum())


def test_zero_weights_closed_form():
    """omega == 0: every proposal accepted -> site i is flipped at step i, whatever the RNG says."""
    L, W, therm, sweeps = 6, 7, 1, 2
    N = L * L
    o = mo.Oracle(L, W, 42)
    s0 = o.get_spins().copy()
    E0 = o.get_energies().copy()
    H = o.run_iteration(therm, sweeps)
    want = np.zeros(N + 1, dtype=np.uint64)
    for w in range(W):
        s = s0[w].copy()
        for sweep in range(therm + sweeps):
            for i in range(N):                      # typewriter order, x fastest (R3)
                s[i // L, i % L] *= -1
                if sweep >= therm:
                    want[(_numpy_energy(s) + 2 * N) // 4] += 1
    assert np.array_equal(H, want)
    sign = -1 if (therm + sweeps) % 2 else 1
    assert np.array_equal(o.get_spins(), sign * s0)
    assert np.array_equal(o.get_energies(), E0)
    assert o.iteration == 1


# ------------------------------------------------------------------ P4 -----
@pytest.mark.parametrize("L,W,seed", [(8, 64, 170700919), (16, 32, 1), (6, 10, 0xDEADBEEFCAFEF00D)])
def test_invariants_over_iterations(L, W, seed):
    N = L * L
    o = mo.Oracle(L, W, seed)
    for it in range(4):
        H = o.run_iteration(3, 25, n_threads=2)
        assert int(H.sum()) == W * 25 * N                 # every attempt recorded once
        assert H[1] == 0 and H[N - 1] == 0                # forbidden +-(2N-4)
        E = o.get_energies()
        s = o.get_spins()
        for w in range(W):
            assert E[w] == _numpy_energy(s[w].astype(np.int64))
        assert np.all(E % 4 == 0) and np.all(np.abs(E) <= 2 * N)
        assert set(np.unique(s).tolist()) <= {-1, 1}
        o.update_weights()
    assert o.iteration == 4


def test_result_does_not_depend_on_thread_count_or_partition():
    L, W, seed = 8, 48, 99
    a = mo.Oracle(L, W, seed)
    b = mo.Oracle(L, W, seed)
    c0 = mo.Oracle(L, 16, seed, walker_offset=0)
    c1 = mo.Oracle(L, 32, seed, walker_offset=16)
    for it in range(3):
        Ha = a.run_iteration(2, 20, n_threads=1)
        Hb = b.run_iteration(2, 20, n_threads=5)
        Hc = c0.run_iteration(2, 20) + c1.run_iteration(2, 20)      # H = sum_i H_i
        assert np.array_equal(Ha, Hb) and np.array_equal(Ha, Hc)
        a.update_weights(); b.update_weights()
        c0.update_weights_with(Hc); c1.update_weights_with(Hc)
        assert np.array_equal(a.get_log_weights(), c0.get_log_weights())
    assert np.array_equal(a.get_spins(), b.get_spins())
    assert np.array_equal(a.get_spins(), np.concatenate([c0.get_spins(), c1.get_spins()]))
    assert np.array_equal(a.get_energies(), np.concatenate([c0.get_energies(), c1.get_energies()]))


# ------------------------------------------------------------------ P8 -----
def test_weight_update_eq4():
    logw = np.array([0.5, -1.0, 2.0, 0.0, 3.25])
    H = np.array([1, 0, 10, 2 ** 40, 7], dtype=np.uint64)
    out = mo.weight_update(logw, H)
    want = [0.5 - 0.0, -1.0, 2.0 - math.log(10), 0.0 - 40 * math.log(2), 3.25 - math.log(7)]
    assert np.allclose(out, want, rtol=0, atol=1e-12)
    assert out[1] == -1.0                                  # unvisited bin untouched (R8)
    # W/H really is the estimator of 1/Omega: flat sampling of g under W gives H ~ g W => W/H ~ 1/g
    g = np.array([2.0, 32.0, 64.0, 424.0])
    lw = np.log([3.0, 0.1, 5.0, 1.0])
    Hs = np.round(1e6 * g * np.exp(lw)).astype(np.uint64)
    new = mo.weight_update(lw, Hs)
    est = -new - (-new).max()
    assert np.allclose(est, np.log(g) - np.log(g).max(), atol=1e-4)
