"""The paper's own update scheme (R22): the same random site in all
walkers, per-walker acceptance stream, work counted in updates.

not gpu: pins of the oracle's variants -- omega == 0 closed form (every update accepted: the final configuration is
         the initial one with every site flipped as often as the shared site stream drew it, the stream recomputed
         from the pinned Philox), canonical weights against the exact g(E) at L = 4, invariants.
gpu    : muca_run_iteration_random_site against the oracle, bit for bit.
"""
import os

import mpmath as mp
import numpy as np
import pytest

import muca_oracle as mo
import paper_1707_00919_b200 as mb

GOLDEN = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")
THREADS = max(1, min(8, mo.max_threads()))


def site_stream(seed, iteration, n_updates, N):
    """i_u of R22 from the (pinned) Philox routine: word (u & 3) of Philox((u >> 2, u >> 34, n, 0xFFFFFFFF), key) mod N."""
    key = np.array([seed & 0xFFFFFFFF, seed >> 32], dtype=np.uint32)
    out = np.empty(n_updates, dtype=np.int64)
    for q in range((n_updates + 3) // 4):
        r = mo.philox4x32_10(np.array([q & 0xFFFFFFFF, q >> 32, iteration, 0xFFFFFFFF], dtype=np.uint32), key)
        out[4 * q:4 * q + 4] = (r.astype(np.int64) % N)[:n_updates - 4 * q]
    return out


def energy_numpy(spins):
    s = spins.astype(np.int32)
    return -(s * np.roll(s, -1, axis=2)).sum(axis=(1, 2)) - (s * np.roll(s, -1, axis=1)).sum(axis=(1, 2))


@pytest.mark.parametrize("L,W,seed", [(4, 5, 3), (8, 16, 170700919), (6, 3, 0xDEADBEEFCAFEF00D)])
def test_zero_weights_closed_form(L, W, seed):
    # omega == 0: t = 0xFFFFFFFF everywhere, every update is accepted whatever the walker's own deviate is
    N, therm, updates = L * L, 37, 451
    o = mo.Oracle(L, W, seed)
    s0 = o.get_spins().copy()
    H = o.run_iteration_random_site(therm, updates, n_threads=THREADS)
    sites = site_stream(seed, 0, therm + updates, N)
    flips = np.bincount(sites, minlength=N).reshape(L, L) % 2
    assert np.array_equal(o.get_spins(), s0 * (1 - 2 * flips).astype(np.int8)[None])
    assert int(H.sum()) == W * updates and H[1] == 0 and H[N - 1] == 0
    assert np.array_equal(energy_numpy(o.get_spins()), o.get_energies()) and o.iteration == 1
    # the histogram is the energy trajectory of that deterministic sequence, replayed here with numpy
    Hn = np.zeros(N + 1, dtype=np.uint64)
    s = s0.astype(np.int32).copy()
    for u, i in enumerate(sites):
        s[:, i // L, i % L] *= -1
        if u >= therm:
            np.add.at(Hn, (energy_numpy(s) + 2 * N) // 4, 1)
    assert np.array_equal(H, Hn)
    o.close()


@pytest.mark.parametrize("beta", [0.25, -0.1])
def test_canonical_weights_reproduce_boltzmann_distribution(beta):
    # omega = -beta E: random-site Metropolis satisfies detailed balance -> P(E) = g(E) exp(-beta E) / Z, exact g(E) at L = 4
    L, N, W = 4, 16, 512
    with open(os.path.join(GOLDEN, "ising_dos_L4.txt")) as f:
        g = np.array([float(x) for x in f if not x.startswith("#")])
    E = -2 * N + 4 * np.arange(N + 1)
    o = mo.Oracle(L, W, 5)
    o.set_log_weights(-beta * E)
    H = o.run_iteration_random_site(50 * N, 2000 * N, n_threads=THREADS)
    P, Pe = H / H.sum(), g * np.exp(-beta * E)
    Pe /= Pe.sum()
    assert np.abs(P - Pe).max() < 2e-3 and abs((P * E).sum() - (Pe * E).sum()) < 0.05
    o.close()


def test_walkers_share_sites_but_not_decisions():
    # the sites visited are the same in all walkers; with non-trivial weights the decisions differ
    L, N, W = 8, 64, 8
    o = mo.Oracle(L, W, 9)
    o.set_log_weights(-0.4 * (-2 * N + 4 * np.arange(N + 1)))
    s0 = o.get_spins().copy()
    o.run_iteration_random_site(0, 5)
    changed = (o.get_spins() != s0).reshape(W, N)
    sites = set(site_stream(9, 0, 5, N).tolist())
    assert all(set(np.nonzero(changed[w])[0].tolist()) <= sites for w in range(W))
    assert len({tuple(c) for c in changed}) > 1
    o.close()


# ------------------------------------------------------------------------------------------------ fp32 acceptance (R23)
def test_exp32_against_arbitrary_precision():
    # PAPER.md:109 "a single precision version of the exponential function"; R23: a fixed sequence of fp32 operations
    L = mo.lib()
    xs = np.concatenate([np.linspace(-24.0, 0.0, 20001), -np.logspace(-12, 1.3, 500), [-24.0, -1e-30, -0.0, -0.6931472, -23.99999]])
    worst = 0.0
    for d in xs.astype(np.float32):
        v, ref = L.oracle_exp32(float(d)), mp.exp(mp.mpf(float(d)))
        worst = max(worst, abs(float((mp.mpf(v) - ref) / ref)))
    assert worst < 2.0 * 2.0 ** -23, worst                     # 2 ulp
    assert L.oracle_exp32(-24.5) == 0.0 and L.oracle_exp32(-1e30) == 0.0 and L.oracle_exp32(-0.0) == 1.0
    ys = np.array([L.oracle_exp32(float(d)) for d in np.linspace(-24, 0, 3001).astype(np.float32)])
    assert np.all(np.diff(ys) >= -2.0 ** -23 * ys[1:])          # monotone up to its own rounding


def test_uniform32_is_curands_mapping(curand_pin):
    # the Philox word -> (0, 1] as curand_uniform does it: compared with what libcurand's host generator returns for
    # the same raw words
    n = 1 << 16
    raw = np.zeros(n, dtype=np.uint32)
    uni = np.zeros(n, dtype=np.float32)
    import ctypes
    assert curand_pin.pin_curand_host_generate(77, 0, raw.ctypes.data_as(ctypes.POINTER(ctypes.c_uint32)), n) == 0
    assert curand_pin.pin_curand_host_generate_uniform(77, 0, uni.ctypes.data_as(ctypes.POINTER(ctypes.c_float)), n) == 0
    L = mo.lib()
    mine = np.array([L.oracle_uniform32(int(x)) for x in raw], dtype=np.float32)
    assert np.array_equal(mine, uni)
    assert L.oracle_uniform32(0) == 2.0 ** -33 and L.oracle_uniform32(2 ** 32 - 1) == 1.0


@pytest.mark.parametrize("beta", [0.25, -0.1])
def test_fp32_acceptance_reproduces_boltzmann_distribution(beta):
    # the same canonical check as above with U < exp32(omega_f[j'] - omega_f[j])
    L, N, W = 4, 16, 512
    with open(os.path.join(GOLDEN, "ising_dos_L4.txt")) as f:
        g = np.array([float(x) for x in f if not x.startswith("#")])
    E = -2 * N + 4 * np.arange(N + 1)
    o = mo.Oracle(L, W, 5)
    o.set_log_weights(-beta * E)
    H = o.run_iteration_random_site_expf(50 * N, 2000 * N, n_threads=THREADS)
    P, Pe = H / H.sum(), g * np.exp(-beta * E)
    Pe /= Pe.sum()
    assert np.abs(P - Pe).max() < 2e-3 and abs((P * E).sum() - (Pe * E).sum()) < 0.05
    assert H[1] == 0 and H[N - 1] == 0 and int(H.sum()) == W * 2000 * N
    assert np.array_equal(energy_numpy(o.get_spins()), o.get_energies())
    o.close()


def test_fp32_and_threshold_acceptance_agree_where_no_rounding_is_involved():
    # omega == 0: every weight difference is 0 -> accepted in both forms; omega with steps of -100 per slot: a move
    # up in omega is always accepted, a move down never (exp(-100) < 2^-33 in fp32, T = floor(exp(-100) 2^32) -> 1, i.e.
    # accepted only for the deviate 0): the two chains coincide (no deviate is 0 in these short runs)
    for logw in (np.zeros(65), -100.0 * np.arange(65)):
        a, b = mo.Oracle(8, 40, 11), mo.Oracle(8, 40, 11)
        a.set_log_weights(logw); b.set_log_weights(logw)
        Ha, Hb = a.run_iteration_random_site(10, 4000), b.run_iteration_random_site_expf(10, 4000)
        assert np.array_equal(Ha, Hb) and np.array_equal(a.get_spins(), b.get_spins())
        a.close(); b.close()


# ------------------------------------------------------------------------------------------------ GPU parity
@pytest.mark.gpu
@pytest.mark.parametrize("L,W,offset,therm,updates", [(8, 131, 0, 50, 3000), (16, 300, 7, 101, 5000), (32, 200, 1000, 333, 20001),
                                                      (64, 150, 3, 10, 9000), (128, 40, 0, 7, 6000)])
def test_gpu_random_site_matches_oracle(L, W, offset, therm, updates):
    g, o = mb.Muca(L, W, 170700919, walker_offset=offset), mo.Oracle(L, W, 170700919, walker_offset=offset)
    try:
        for it in range(3):
            Hg = g.run_iteration_random_site(therm, updates)
            Ho = o.run_iteration_random_site(therm, updates, n_threads=mo.max_threads())
            assert int(Hg.sum()) == W * updates and np.array_equal(Hg, Ho), f"it{it}"
            g.update_weights(); o.update_weights()
        assert np.array_equal(g.get_energies(), o.get_energies())
        assert np.array_equal(g.get_spins(), o.get_spins())
        assert np.max(np.abs(g.get_log_weights() - o.get_log_weights())) <= 1e-12 and g.iteration == 3
        # mixing the two schemes on one context keeps the chains identical, too
        Hg, Ho = g.run_iteration(1, 3), o.run_iteration(1, 3, n_threads=mo.max_threads())
        assert np.array_equal(Hg, Ho) and np.array_equal(g.get_spins(), o.get_spins())
    finally:
        g.close(); o.close()


@pytest.mark.gpu
@pytest.mark.parametrize("L,W,offset,therm,updates", [(8, 131, 0, 50, 3000), (16, 300, 7, 101, 5000), (32, 200, 1000, 333, 20001),
                                                      (64, 150, 3, 10, 9000), (128, 40, 0, 7, 6000)])
def test_gpu_random_site_fp32_acceptance_matches_oracle(L, W, offset, therm, updates):
    # MUCA_OPT_ACCEPTANCE = EXPF32 (R23): same chains as the oracle's fp32 variant, bit for bit
    from paper_1707_00919_b200 import binding as B
    g, o = mb.Muca(L, W, 170700919, walker_offset=offset), mo.Oracle(L, W, 170700919, walker_offset=offset)
    try:
        g.set_option(B.MUCA_OPT_ACCEPTANCE, B.MUCA_ACCEPT_EXPF32)
        for it in range(4):
            Hg = g.run_iteration_random_site(therm, updates)
            Ho = o.run_iteration_random_site_expf(therm, updates, n_threads=mo.max_threads())
            assert int(Hg.sum()) == W * updates and np.array_equal(Hg, Ho), f"it{it}"
            g.update_weights(); o.update_weights()
        assert np.array_equal(g.get_energies(), o.get_energies())
        assert np.array_equal(g.get_spins(), o.get_spins())
        # back to thresholds on the same context
        g.set_option(B.MUCA_OPT_ACCEPTANCE, B.MUCA_ACCEPT_THRESHOLD)
        assert np.array_equal(g.run_iteration_random_site(3, 500), o.run_iteration_random_site(3, 500, n_threads=mo.max_threads()))
    finally:
        g.close(); o.close()


@pytest.mark.gpu
def test_gpu_random_site_zero_updates_and_errors():
    g = mb.Muca(16, 33, 1)
    H = g.run_iteration_random_site(0, 0)
    assert H.sum() == 0 and g.iteration == 1
    H = g.run_iteration_random_site(5, 0)
    assert H.sum() == 0
    g.iteration = 0xFFFFFFFF
    with pytest.raises(mb.MucaError):
        g.run_iteration_random_site(1, 1)
    g.close()
