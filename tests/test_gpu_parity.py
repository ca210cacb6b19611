"""GPU parity: libmuca_b200 (CUDA, through the C ABI) against the CPU oracle, element by element.

Bars (BASELINE.json north_star): bit-exact H, per-walker E, final spins, thresholds; omega within 1e-12
absolute.  All inputs are seeded and synthetic (paper_1707_00919_b200/workloads.py).
"""
import numpy as np
import pytest

import muca_oracle as mo
import paper_1707_00919_b200 as mb
from paper_1707_00919_b200 import binding as B
from paper_1707_00919_b200.workloads import CONFIGS, EXTRA_SEEDS, PRIMARY_SEED

pytestmark = pytest.mark.gpu
LOGW_TOL = 1e-12   # north_star: "double log-weights must agree within 1e-12 absolute"


def energy_numpy(spins):
    """E = -sum_<ij> s_i s_j on the periodic lattice, written with numpy rolls (independent of both sides)."""
    s = spins.astype(np.int32)
    return -(s * np.roll(s, -1, axis=2)).sum(axis=(1, 2)) - (s * np.roll(s, -1, axis=1)).sum(axis=(1, 2))


def compare_state(g, o, tag=""):
    Eg, Eo = g.get_energies(), o.get_energies()
    assert np.array_equal(Eg, Eo), f"{tag}: energies differ at walkers {np.nonzero(Eg != Eo)[0][:8]}"
    sg, so = g.get_spins(), o.get_spins()
    assert sg.shape == so.shape
    if not np.array_equal(sg, so):
        bad = np.nonzero((sg != so).reshape(sg.shape[0], -1).any(axis=1))[0]
        raise AssertionError(f"{tag}: spins differ for walkers {bad[:8]} ({bad.size} of {sg.shape[0]})")
    for a in range(0, sg.shape[0], 4096):                      # chunked: 128 MiB of spins at configs 4 and 5
        assert np.array_equal(energy_numpy(sg[a:a + 4096]), Eg[a:a + 4096]), f"{tag}: tracked E != recomputed E"


def run_pair(L, W, seed, iterations, therm, sweeps, offset=0, options=(), threads=None, check_every=True):
    """Free-running pair: both sides apply their own Eq. (4) update each iteration."""
    threads = threads or mo.max_threads()
    g = mb.Muca(L, W, seed, walker_offset=offset)
    for k, v in options:
        g.set_option(k, v)
    o = mo.Oracle(L, W, seed, walker_offset=offset)
    try:
        compare_state(g, o, "init")
        N = L * L
        for it in range(iterations):
            assert np.array_equal(g.get_thresholds(), mo.thresholds(o.get_log_weights())), f"it{it}: thresholds"
            Hg = g.run_iteration(therm, sweeps)
            Ho = o.run_iteration(therm, sweeps, n_threads=threads)
            assert Hg.dtype == np.uint64 and int(Hg.sum()) == W * sweeps * N
            assert np.array_equal(Hg, Ho), f"it{it}: H differs in slots {np.nonzero(Hg != Ho)[0][:8]}"
            assert Hg[1] == 0 and Hg[N - 1] == 0                       # unreachable slots
            if check_every or it == iterations - 1:
                compare_state(g, o, f"it{it}")
            g.update_weights()
            o.update_weights()
            assert np.max(np.abs(g.get_log_weights() - o.get_log_weights())) <= LOGW_TOL
            assert g.iteration == o.iteration == it + 1
    finally:
        g.close()
        o.close()


# ---------------------------------------------------------------------------------------------------
def test_device_philox_matches_oracle_philox():
    rng = np.random.default_rng(1)
    ctr = rng.integers(0, 2 ** 32, size=(4096, 4), dtype=np.uint64).astype(np.uint32)
    key = rng.integers(0, 2 ** 32, size=(4096, 2), dtype=np.uint64).astype(np.uint32)
    ctr[:4] = [[0, 0, 0, 0], [0xFFFFFFFF] * 4, [255, 549, 14, 16383], [3, 0, 0xFFFFFFFF, 77]]
    got = mb.debug_philox(ctr, key)
    for i in list(range(64)) + [1000, 4095]:
        assert np.array_equal(got[i], mo.philox4x32_10(ctr[i], key[i])), i


@pytest.mark.parametrize("L", [8, 16, 32, 64, 128])
@pytest.mark.parametrize("W,offset", [(1, 0), (37, 5), (160, 1000)])
def test_init_matches_oracle(L, W, offset):
    for seed in (PRIMARY_SEED,) + EXTRA_SEEDS[1:]:
        g, o = mb.Muca(L, W, seed, walker_offset=offset), mo.Oracle(L, W, seed, walker_offset=offset)
        compare_state(g, o, f"L{L} W{W}")
        assert np.all(g.get_log_weights() == 0.0) and g.iteration == 0
        g.close(); o.close()


def test_thresholds_bit_exact_for_rough_weights():
    rng = np.random.default_rng(3)
    g = mb.Muca(16, 32, 1)
    logw = np.cumsum(rng.normal(0, 2.0, g.n_bins))
    logw[40] = logw[38]
    logw[100] = logw[98] - 40.0
    g.set_log_weights(logw)
    assert np.array_equal(g.get_log_weights(), logw)
    assert np.array_equal(g.get_thresholds(), mo.thresholds(logw))
    g.close()


# config 1 in full, all three seeds
@pytest.mark.parametrize("seed", (PRIMARY_SEED,) + EXTRA_SEEDS)
def test_config1_L8_full(seed):
    c = CONFIGS[0]
    run_pair(c.L, c.n_walkers, seed, c.iterations, c.therm_sweeps, c.sweeps)


# config 2 in full, all three seeds (2.8e9 attempts on the oracle per seed: seconds on 16 threads)
@pytest.mark.parametrize("seed", (PRIMARY_SEED,) + EXTRA_SEEDS)
def test_config2_L16_full(seed):
    c = CONFIGS[1]
    run_pair(c.L, c.n_walkers, seed, c.iterations, c.therm_sweeps, c.sweeps, check_every=False)


# configs 3-5 at reduced walker count / sweeps, several tiles and a ragged tail, default launch configuration
@pytest.mark.parametrize("L,W,iters,therm,sweeps", [
    (32, 32 * 5 + 7, 6, 5, 40),
    (64, 64 * 2 + 19, 4, 3, 12),
    (128, 32 * 2 + 9, 3, 2, 5),
])
def test_configs345_reduced(L, W, iters, therm, sweeps):
    for seed in (PRIMARY_SEED,) + EXTRA_SEEDS:
        run_pair(L, W, seed, iters, therm, sweeps, offset=11)


# configs 3-5 at FULL size in the launch configuration bench.py times (library defaults).  The walkers are
# independent given the weights, so the oracle follows sampled walker ranges one by one (same global
# ids, the library's omega injected before every iteration); what cannot be sampled is checked through the
# invariants: sum(H), the unreachable slots, tracked E == recomputed E for every walker.
@pytest.mark.parametrize("name", ["L32_w16384", "L64_w32768", "L128_w8192"])
def test_full_size_configs_sampled_walkers(name):
    c = next(x for x in CONFIGS if x.name == name)
    W, N = c.n_walkers, c.N
    starts = sorted({0, 27, W // 3 + 5, W // 2 - 3, W - 6})        # first / inner / last walkers, across warp and block borders
    width = 6
    g = mb.Muca(c.L, W, c.seed)
    oracles = [mo.Oracle(c.L, width, c.seed, walker_offset=w0) for w0 in starts]
    try:
        for it in range(c.iterations):
            logw = g.get_log_weights()
            H = g.run_iteration(c.therm_sweeps, c.sweeps)
            assert int(H.sum()) == W * c.sweeps * N and H[1] == 0 and H[N - 1] == 0
            for o in oracles:
                o.set_log_weights(logw)
                o.run_iteration(c.therm_sweeps, c.sweeps, n_threads=mo.max_threads())
            g.update_weights()
            assert np.max(np.abs(g.get_log_weights() - (logw - np.where(H > 0, np.log(np.maximum(H, 1).astype(np.float64)), 0.0)))) <= LOGW_TOL
        E, spins = g.get_energies(), g.get_spins()
        for w0, o in zip(starts, oracles):
            assert np.array_equal(E[w0:w0 + width], o.get_energies()), f"{name}: energies of walkers {w0}.."
            assert np.array_equal(spins[w0:w0 + width], o.get_spins()), f"{name}: spins of walkers {w0}.."
        step = 4096                                                  # tracked E == recomputed E, all walkers
        for a in range(0, W, step):
            assert np.array_equal(energy_numpy(spins[a:a + step]), E[a:a + step])
    finally:
        g.close()
        for o in oracles:
            o.close()


# configs 3-5 at FULL size, ALL walkers, in the launch configuration bench.py times: H is a sum over all walkers
# (Fig. 1), so a merge error that keeps sum(H) -- a bin dropped in one block and counted twice in another,
# a lane without a walker leaking into a real bin -- shows only when the whole histogram is compared.  The oracle needs
# 10-35 s per full-size iteration, so it replays the first, a middle and the last iteration of the config from the
# library's own state before that iteration (spins, omega, iteration counter) and must reproduce the full H, every
# energy and every spin.  Chained with test_full_size_configs_sampled_walkers (sampled walkers followed through every
# iteration from the initial state) this covers the whole run.
@pytest.mark.parametrize("name", ["L32_w16384", "L64_w32768", "L128_w8192"])
def test_full_size_configs_all_walkers_replayed(name):
    c = next(x for x in CONFIGS if x.name == name)
    W, N = c.n_walkers, c.N
    replay = sorted({0, c.iterations // 2, c.iterations - 1})
    g = mb.Muca(c.L, W, c.seed)
    o = mo.Oracle(c.L, W, c.seed)
    try:
        compare_state(g, o, f"{name}: init")
        for it in range(c.iterations):
            if it in replay:
                logw = g.get_log_weights()
                o.set_spins(g.get_spins())
                o.set_log_weights(logw)
                o.iteration = g.iteration
                assert np.array_equal(o.get_energies(), g.get_energies()), f"{name} it{it}: energies before the replay"
                assert np.array_equal(g.get_thresholds(), mo.thresholds(logw)), f"{name} it{it}: thresholds"
            Hg = g.run_iteration(c.therm_sweeps, c.sweeps)
            assert int(Hg.sum()) == W * c.sweeps * N and Hg[1] == 0 and Hg[N - 1] == 0
            if it in replay:
                Ho = o.run_iteration(c.therm_sweeps, c.sweeps, n_threads=mo.max_threads())
                assert np.array_equal(Hg, Ho), f"{name} it{it}: H differs in slots {np.nonzero(Hg != Ho)[0][:8]}"
                compare_state(g, o, f"{name} it{it}")
                o.update_weights()
            g.update_weights()
            if it in replay:
                assert np.max(np.abs(g.get_log_weights() - o.get_log_weights())) <= LOGW_TOL
    finally:
        g.close()
        o.close()


# every kernel variant / block size must give the same chains
@pytest.mark.parametrize("L,kernel,tpb", [
    (8, B.MUCA_KERNEL_RESIDENT, 64), (16, B.MUCA_KERNEL_RESIDENT, 128),
    (32, B.MUCA_KERNEL_RESIDENT, 64), (32, B.MUCA_KERNEL_RESIDENT, 128), (32, B.MUCA_KERNEL_RESIDENT, 96),
    (16, B.MUCA_KERNEL_RESIDENT, 32), (32, B.MUCA_KERNEL_STREAMED, 32),
    (32, B.MUCA_KERNEL_STREAMED, 96),
    (64, B.MUCA_KERNEL_RESIDENT, 32), (64, B.MUCA_KERNEL_STREAMED, 32), (64, B.MUCA_KERNEL_STREAMED, 64),
    (128, B.MUCA_KERNEL_RESIDENT, 32), (128, B.MUCA_KERNEL_STREAMED, 64), (16, B.MUCA_KERNEL_STREAMED, 64),
    (32, B.MUCA_KERNEL_STREAMED_PAIRS, 96), (64, B.MUCA_KERNEL_STREAMED_PAIRS, 64), (64, B.MUCA_KERNEL_STREAMED_PAIRS, 256),
    (128, B.MUCA_KERNEL_STREAMED_PAIRS, 32),
])
def test_kernel_variants(L, kernel, tpb):
    W = 2 * tpb + 13
    sweeps = {8: 30, 16: 20, 32: 10, 64: 5, 128: 3}[L]
    run_pair(L, W, PRIMARY_SEED, 3, 2, sweeps,
             options=((B.MUCA_OPT_KERNEL, kernel), (B.MUCA_OPT_THREADS_PER_BLOCK, tpb)))


# resident kernel, L <= 32: any number of walkers per warp (the default spreads the walkers over all SMs) and
# 1, 2 or 4 walker/deviate warp pairs per block give the same chains
@pytest.mark.parametrize("L,W,tpb,wpw", [
    (8, 128, 0, 0), (8, 77, 32, 5), (16, 300, 64, 17), (16, 4096, 0, 0), (32, 333, 128, 28), (32, 200, 32, 1),
    (32, 1000, 0, 0),
])
def test_resident_walkers_per_warp(L, W, tpb, wpw):
    opts = [(B.MUCA_OPT_KERNEL, B.MUCA_KERNEL_RESIDENT)]
    if tpb:
        opts.append((B.MUCA_OPT_THREADS_PER_BLOCK, tpb))
    if wpw:
        opts.append((B.MUCA_OPT_WALKERS_PER_WARP, wpw))
    run_pair(L, W, EXTRA_SEEDS[1], 3, 2, {8: 30, 16: 12, 32: 6}[L], offset=3, options=tuple(opts), check_every=False)


# L = 128 default: a WINDOW of the threshold table in shared memory; an iteration in which a walker leaves the window is
# repeated from a snapshot with the L1 kernel.  Small forced windows exercise that fallback; the chains must not change.
@pytest.mark.parametrize("kernel", [B.MUCA_KERNEL_STREAMED_PAIRS])
@pytest.mark.parametrize("L,W,rows,iters,therm,sweeps,expect_fallback", [
    (128, 70, 0, 3, 2, 5, False), (128, 70, 600, 4, 2, 6, None), (64, 150, 300, 6, 3, 12, None),
    (32, 200, 120, 8, 5, 40, True), (32, 100, 40, 3, 2, 10, None),
])
def test_windowed_table_and_fallback(L, W, rows, iters, therm, sweeps, expect_fallback, kernel):
    g, o = mb.Muca(L, W, PRIMARY_SEED, walker_offset=4), mo.Oracle(L, W, PRIMARY_SEED, walker_offset=4)
    try:
        g.set_option(B.MUCA_OPT_KERNEL, kernel)
        if rows:
            g.set_option(B.MUCA_OPT_TABLE_WINDOW_ROWS, rows)
        for it in range(iters):
            Hg, Ho = g.run_iteration(therm, sweeps), o.run_iteration(therm, sweeps, n_threads=mo.max_threads())
            assert np.array_equal(Hg, Ho), f"it{it}: H differs in slots {np.nonzero(Hg != Ho)[0][:8]}"
            compare_state(g, o, f"it{it}")
            g.update_weights(); o.update_weights()
        windowed, fallbacks = g.window_stats()
        if expect_fallback is True:
            assert windowed > 0 and fallbacks > 0, (windowed, fallbacks)
        if expect_fallback is False:
            assert windowed == iters and fallbacks == 0, (windowed, fallbacks)
    finally:
        g.close(); o.close()


# Walkers spread over more table rows than the window holds (L = 128 in every production run): the library sorts the
# walkers by energy, gives every block a window of its own and cuts the iteration into launches of a few sweeps
# (muca.cu run_sorted).  Walkers are started all over the energy range.  Cases:
#   L = 32, forced 600-row window, exact flat-histogram weights (every walker diffuses slowly from where it starts);
#   L = 64, forced 1500 rows, omega = 0 at the start, Eq. (4) updates;
#   L = 128 with the window the library itself picks (~5500 of the 16385 rows: the shape production runs take), omega = 0
#     at the start, Eq. (4) updates;
#   "quench", L = 64 and L = 128: omega = -E (a canonical ensemble far below T_c) pulls the disordered walkers down by
#     hundreds of slots per sweep, far beyond the 6 sigma of diffusion the launches are sized for: walkers DO leave their
#     windows, so launches are undone from the snapshot and repeated with the plain kernel (undone > 0 is asserted).
@pytest.mark.parametrize("L,W,rows,sweeps,weights,expect_undone", [
    (32, 200, 600, 8, "exact", False), (64, 150, 1500, 6, "zero", False), (128, 200, 0, 6, "zero", False),
    (64, 150, 1500, 6, "quench", True), (128, 200, 0, 4, "quench", True),
])
def test_sorted_windows_for_widely_spread_walkers(L, W, rows, sweeps, weights, expect_undone):
    import os
    N = L * L
    rng = np.random.default_rng(5)
    p = np.linspace(0.0, 0.5, W)[:, None]                       # walker k: a fraction p_k of its spins down -> E from -2N up to ~0
    spins = np.where(rng.random((W, N)) < p, -1, 1).astype(np.int8)
    if L != 64:                                                 # every second walker times a checkerboard: E -> -E, up to +2N
        yy, xx = np.divmod(np.arange(N), L)
        spins[1::2] *= np.where((xx + yy) % 2 == 0, 1, -1).astype(np.int8)[None, :]
    g, o = mb.Muca(L, W, PRIMARY_SEED, walker_offset=9), mo.Oracle(L, W, PRIMARY_SEED, walker_offset=9)
    try:
        g.set_spins(spins); o.set_spins(spins)
        if weights == "exact":                                  # omega = -ln g
            with open(os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", f"ising_dos_L{L}.txt")) as f:
                gE = [int(x) for x in f if not x.startswith("#")]
            import mpmath as mp
            w = np.array([-float(mp.log(v)) if v > 0 else 0.0 for v in gE])
            g.set_log_weights(w); o.set_log_weights(w)
        if weights == "quench":                                 # omega(E) = -beta E, beta = 1
            w = -1.0 * (-2.0 * N + 4.0 * np.arange(N + 1))
            g.set_log_weights(w); o.set_log_weights(w)
        g.set_option(B.MUCA_OPT_KERNEL, B.MUCA_KERNEL_STREAMED_PAIRS)
        if rows:
            g.set_option(B.MUCA_OPT_TABLE_WINDOW_ROWS, rows)
        E0 = g.get_energies()
        assert (E0.max() - E0.min()) // 4 > (rows if rows else 6000)   # one window cannot hold them (L = 128: < 5600 rows fit)
        for it in range(3):
            Hg, Ho = g.run_iteration(2, sweeps), o.run_iteration(2, sweeps, n_threads=mo.max_threads())
            assert np.array_equal(Hg, Ho), f"it{it}: H differs in slots {np.nonzero(Hg != Ho)[0][:8]}"
            compare_state(g, o, f"it{it}")
            if weights != "quench":
                g.update_weights(); o.update_weights()
        windowed, undone = g.window_stats()
        assert windowed > 0, (windowed, undone)                 # launches with per-block windows did run
        if expect_undone:
            assert undone > 0, (windowed, undone)               # ... and some were undone and repeated
    finally:
        g.close(); o.close()


def test_split_launches_give_the_same_iteration():
    # an iteration split into several launches (the uint32-bin overflow guard) is the same Markov chain
    run_pair(32, 70, PRIMARY_SEED, 3, 3, 9, options=((B.MUCA_OPT_MAX_SWEEPS_PER_LAUNCH, 2),))
    run_pair(128, 40, PRIMARY_SEED, 2, 1, 4, options=((B.MUCA_OPT_MAX_SWEEPS_PER_LAUNCH, 1),))


def test_edge_cases_zero_sweeps_and_single_walker():
    g, o = mb.Muca(16, 1, 5), mo.Oracle(16, 1, 5)
    H = g.run_iteration(0, 0)
    assert H.sum() == 0 and g.iteration == 1
    o.run_iteration(0, 0)
    compare_state(g, o)
    g.update_weights()
    assert np.all(g.get_log_weights() == 0.0)                 # H == 0 everywhere: omega unchanged (R8)
    Hg, Ho = g.run_iteration(3, 0), o.run_iteration(3, 0)     # thermalisation only: nothing recorded
    assert Hg.sum() == 0 and np.array_equal(Hg, Ho)
    compare_state(g, o)
    Hg, Ho = g.run_iteration(0, 4), o.run_iteration(0, 4)
    assert np.array_equal(Hg, Ho) and Hg.sum() == 4 * 256
    compare_state(g, o)
    g.close(); o.close()


@pytest.mark.parametrize("L", [8, 32, 64])
def test_degenerate_configurations_and_canonical_weights(L):
    # ground states (slot 0), antiferromagnetic ceiling (slot N), stripes; omega = -beta*E exercises genuine
    # rejections at the edges of the table (moves to unreachable / out-of-range slots never occur)
    N, W = L * L, 48
    yy, xx = np.mgrid[0:L, 0:L]
    pats = [np.ones((L, L)), -np.ones((L, L)), 1 - 2 * ((xx + yy) % 2), 1 - 2 * (yy % 2), 1 - 2 * (xx % 2)]
    spins = np.stack([pats[w % len(pats)] for w in range(W)]).astype(np.int8)
    E_axis = -2 * N + 4 * np.arange(N + 1)
    for beta in (0.0, 0.4, -0.3):
        g, o = mb.Muca(L, W, 99), mo.Oracle(L, W, 99)
        g.set_spins(spins); o.set_spins(spins)
        compare_state(g, o, "set_spins")
        assert g.get_energies()[0] == -2 * N and g.get_energies()[2] == 2 * N
        g.set_log_weights(-beta * E_axis); o.set_log_weights(-beta * E_axis)
        for it in range(2):
            Hg, Ho = g.run_iteration(1, 6), o.run_iteration(1, 6, n_threads=mo.max_threads())
            assert np.array_equal(Hg, Ho)
            compare_state(g, o, f"beta{beta} it{it}")
        g.close(); o.close()


def test_injected_weights_mode():
    # the harness may inject the oracle's omega each iteration (muca_set_log_weights) instead of muca_update_weights
    L, W = 32, 96
    g, o = mb.Muca(L, W, 7), mo.Oracle(L, W, 7)
    for it in range(4):
        g.set_log_weights(o.get_log_weights())
        Hg, Ho = g.run_iteration(2, 20), o.run_iteration(2, 20, n_threads=mo.max_threads())
        assert np.array_equal(Hg, Ho)
        o.update_weights()
    compare_state(g, o)
    g.close(); o.close()


def test_sharded_walkers_are_independent_of_the_split():
    # two contexts with walker_offset 0 / 50 reproduce one context of 120 walkers (R16); H adds up
    L, seed = 16, PRIMARY_SEED
    whole, a, b = mb.Muca(L, 120, seed), mb.Muca(L, 50, seed, 0), mb.Muca(L, 70, seed, 50)
    for it in range(3):
        Hw = whole.run_iteration(2, 15)
        Hs = a.run_iteration(2, 15) + b.run_iteration(2, 15)
        assert np.array_equal(Hw, Hs)
        whole.update_weights(); a.update_weights_with(Hs); b.update_weights_with(Hs)
        assert np.array_equal(whole.get_log_weights(), a.get_log_weights())
    assert np.array_equal(whole.get_spins(), np.concatenate([a.get_spins(), b.get_spins()]))
    assert np.array_equal(whole.get_energies(), np.concatenate([a.get_energies(), b.get_energies()]))
    for x in (whole, a, b):
        x.close()


def test_unpack_device_matches_host_readback():
    g = mb.Muca(64, 33, 3)
    g.run_iteration(1, 2)
    assert np.array_equal(g.unpack_spins_device().cpu().numpy(), g.get_spins())
    g.close()


def test_suggested_walker_count_loads_the_device_evenly():
    # SURVEY 8(f)4 / PAPER.md:179, :201: the suggested W is the first optimum of the time per flip -- not slower per flip
    # than one warp per SM less (idle lanes) or one warp per SM more (a second, nearly empty round of blocks)
    import torch
    n_sm = torch.cuda.get_device_properties(0).multi_processor_count
    for Lx, px in ((8, 4), (16, 4), (32, 4), (64, 8), (128, 4)):   # include/muca.h: pairs_per_sm of the default kernel per L
        Wx, pairs = mb.suggest_walkers(Lx)
        assert pairs == px and Wx == n_sm * px * 32, (Lx, Wx, pairs)
    L = 32
    W, pairs = mb.suggest_walkers(L)

    def ns_per_flip(Wx):
        g = mb.Muca(L, Wx, PRIMARY_SEED)
        try:
            best = 1e30
            for _ in range(3):
                g.run_iteration(2, 30)
                best = min(best, g.last_sweep_ms()[0])
            return best * 1e6 / (Wx * L * L * 32)
        finally:
            g.close()

    # a timing on whatever GPU the suite runs on: 10 % of slack (measured: one warp per SM more costs a second round of
    # blocks, +86 % per flip; one less leaves the time unchanged and wastes 25 % of the lanes, +32 % per flip: profiles/r02_flips_over_W_L32.txt)
    t_opt, t_less, t_more = ns_per_flip(W), ns_per_flip(W - 32 * n_sm), ns_per_flip(W + 32 * n_sm)
    assert t_opt <= 1.10 * min(t_less, t_more), (t_opt, t_less, t_more)


def test_context_on_an_explicit_device():
    # the context remembers its device: results do not depend on which device is current when the calls are made
    import torch
    dev = torch.device("cuda", torch.cuda.device_count() - 1)
    g, o = mb.Muca(16, 100, 5, device=dev), mo.Oracle(16, 100, 5)
    try:
        torch.cuda.set_device(0)
        assert np.array_equal(g.run_iteration(2, 10), o.run_iteration(2, 10, n_threads=mo.max_threads()))
        compare_state(g, o, "explicit device")
    finally:
        g.close(); o.close()


def test_error_paths():
    with pytest.raises(mb.MucaError):
        mb.Muca(12, 32, 1)
    with pytest.raises(mb.MucaError):
        mb.Muca(32, 0, 1)
    g = mb.Muca(8, 32, 1)
    with pytest.raises(mb.MucaError):
        g.set_log_weights(np.zeros(10))
    with pytest.raises(mb.MucaError):
        g.run_iteration(-1, 5)
    with pytest.raises(mb.MucaError):
        g.set_option(99, 1)
    g.iteration = 0xFFFFFFFF
    with pytest.raises(mb.MucaError):
        g.run_iteration(1, 1)
    g.close()


def test_randomized_configurations():
    # seeded random mix of lattice sizes, walker counts (ragged warps), global offsets, kernel variants, launch splits,
    # forced table windows, walkers per warp, walkers started all over the energy range (the sorted per-block windows),
    # smooth non-zero weights, both update schemes, both acceptance forms of the random-site scheme and optional weight
    # updates: every combination must give the oracle's chains bit for bit.  (The same generator ran 208 450 trials as a
    # soak during round 2 without a mismatch: profiles/r02_soak.txt.)
    import random
    rng = random.Random(20261106)
    stats = {"windowed": 0, "undone": 0, "expf": 0, "spread": 0, "random_site": 0}
    for trial in range(120):
        L = rng.choice([8, 16, 32, 32, 64, 64, 128])
        W = rng.choice([1, 3, 31, 32, 33, 64, 97, 130, 257, 300])
        if L == 128:
            W = min(W, 97)
        seed, off = rng.getrandbits(64), rng.choice([0, 0, 5, 1000, 2 ** 31])
        kernel = rng.choice([B.MUCA_KERNEL_AUTO, B.MUCA_KERNEL_RESIDENT, B.MUCA_KERNEL_STREAMED, B.MUCA_KERNEL_STREAMED_PAIRS,
                             B.MUCA_KERNEL_STREAMED_PAIRS])
        g, o = mb.Muca(L, W, seed, walker_offset=off), mo.Oracle(L, W, seed, walker_offset=off)
        tag = [trial, L, W, kernel]
        try:
            g.set_option(B.MUCA_OPT_KERNEL, kernel)
            if rng.random() < 0.4:                                   # walkers all over the energy range, -2N .. +2N
                N = L * L
                nr = np.random.default_rng(rng.getrandbits(32))
                p = np.linspace(0.0, 0.5, W)[:, None]
                spins = np.where(nr.random((W, N)) < p, -1, 1).astype(np.int8)
                yy, xx = np.divmod(np.arange(N), L)
                spins[1::2] *= np.where((xx + yy) % 2 == 0, 1, -1).astype(np.int8)[None, :]
                g.set_spins(spins); o.set_spins(spins); tag.append("spread"); stats["spread"] += 1
                if rng.random() < 0.5:
                    w = -0.002 * (np.arange(N + 1) - N / 2.0) ** 2 * (64.0 / N)   # smooth weights, maximum in the middle
                    g.set_log_weights(w); o.set_log_weights(w); tag.append("weights")
            if rng.random() < 0.3:
                g.set_option(B.MUCA_OPT_MAX_SWEEPS_PER_LAUNCH, rng.choice([1, 2, 3])); tag.append("split")
            if L >= 32 and kernel in (B.MUCA_KERNEL_AUTO, B.MUCA_KERNEL_STREAMED_PAIRS) and rng.random() < 0.6:
                rows = rng.choice([40, 60, 100, 300, 600, 1000, 2000]); g.set_option(B.MUCA_OPT_TABLE_WINDOW_ROWS, rows); tag.append(("window", rows))
            if L <= 32 and kernel in (B.MUCA_KERNEL_AUTO, B.MUCA_KERNEL_RESIDENT) and rng.random() < 0.5:
                wpw = rng.choice([1, 7, 16, 28, 32]); g.set_option(B.MUCA_OPT_WALKERS_PER_WARP, wpw); tag.append(("wpw", wpw))
            expf = rng.random() < 0.5                                # the paper's fp32 acceptance (random-site scheme only, R23)
            if expf:
                g.set_option(B.MUCA_OPT_ACCEPTANCE, B.MUCA_ACCEPT_EXPF32); tag.append("expf32")
            for it in range(rng.choice([1, 2, 4])):
                if rng.random() < 0.3:
                    u0, u1 = rng.choice([0, 17, 100, 255, 256, 257]), rng.choice([0, 1, 999, 4001, 1024, 1023])
                    Hg = g.run_iteration_random_site(u0, u1)
                    Ho = (o.run_iteration_random_site_expf if expf else o.run_iteration_random_site)(u0, u1, n_threads=mo.max_threads())
                    stats["random_site"] += 1; stats["expf"] += int(expf)
                else:
                    th, sw = rng.choice([0, 1, 3]), rng.choice([0, 1, 2, 5, 9] if L < 128 else [0, 1, 2, 3])
                    Hg, Ho = g.run_iteration(th, sw), o.run_iteration(th, sw, n_threads=mo.max_threads())
                assert np.array_equal(Hg, Ho), (tag, it)
                if rng.random() < 0.7:
                    g.update_weights(); o.update_weights()
            compare_state(g, o, str(tag))
            assert np.max(np.abs(g.get_log_weights() - o.get_log_weights())) <= LOGW_TOL, tag
            a, b = g.window_stats(); stats["windowed"] += a; stats["undone"] += b
        finally:
            g.close(); o.close()
    # the mix did reach the paths it is there for
    assert stats["spread"] >= 30 and stats["windowed"] >= 10 and stats["expf"] >= 10 and stats["random_site"] > stats["expf"], stats
