"""Soak: seeded random mix of all knobs against the oracle (the generator of tests/test_gpu_parity.py::test_randomized_configurations
extended by the round-2 paths: fp32 acceptance, spread walkers + forced windows (sorted per-block windows), suggest_walkers-sized blocks)."""
import sys, os, random, time
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))   # run as: python tests/soak_gpu.py <seed> <max trials> <seconds>
sys.path.insert(0, ROOT); sys.path.insert(0, os.path.join(ROOT, "oracle"))
import numpy as np
import muca_oracle as mo
import paper_1707_00919_b200 as mb
from paper_1707_00919_b200 import binding as B
seed0, n_trials, budget = int(sys.argv[1]), int(sys.argv[2]), float(sys.argv[3])
rng = random.Random(seed0)
t0 = time.time(); done = 0; stats = {"windowed": 0, "undone": 0, "expf": 0, "spread": 0}
for trial in range(n_trials):
    if time.time() - t0 > budget: break
    L = rng.choice([8, 16, 32, 32, 64, 64, 128])
    W = rng.choice([1, 3, 31, 32, 33, 64, 97, 130, 257, 300])
    if L == 128: W = min(W, 97)
    seed, off = rng.getrandbits(64), rng.choice([0, 0, 5, 1000, 2 ** 31])
    kernel = rng.choice([0, 1, 2, 3, 3])
    g, o = mb.Muca(L, W, seed, walker_offset=off), mo.Oracle(L, W, seed, walker_offset=off)
    tag = [trial, L, W, kernel]
    try:
        g.set_option(B.MUCA_OPT_KERNEL, kernel)
        if rng.random() < 0.4:                                   # walkers all over the energy range
            N = L * L
            nr = np.random.default_rng(rng.getrandbits(32))
            p = np.linspace(0.0, 0.5, W)[:, None]
            spins = np.where(nr.random((W, N)) < p, -1, 1).astype(np.int8)
            yy, xx = np.divmod(np.arange(N), L)
            spins[1::2] *= np.where((xx + yy) % 2 == 0, 1, -1).astype(np.int8)[None, :]
            g.set_spins(spins); o.set_spins(spins); tag.append("spread"); stats["spread"] += 1
            if rng.random() < 0.5:
                w = -0.002 * (np.arange(N + 1) - N / 2.0) ** 2 * (64.0 / N)   # some smooth weights
                g.set_log_weights(w); o.set_log_weights(w); tag.append("weights")
        if rng.random() < 0.3:
            g.set_option(B.MUCA_OPT_MAX_SWEEPS_PER_LAUNCH, rng.choice([1, 2, 3])); tag.append("split")
        if L >= 32 and kernel in (0, 3) and rng.random() < 0.6:
            rows = rng.choice([40, 60, 100, 300, 600, 1000, 2000]); g.set_option(B.MUCA_OPT_TABLE_WINDOW_ROWS, rows); tag.append(("window", rows))
        if L <= 32 and kernel in (0, 1) and rng.random() < 0.5:
            wpw = rng.choice([1, 7, 16, 28, 32]); g.set_option(B.MUCA_OPT_WALKERS_PER_WARP, wpw); tag.append(("wpw", wpw))
        expf = rng.random() < 0.5
        if expf: g.set_option(B.MUCA_OPT_ACCEPTANCE, B.MUCA_ACCEPT_EXPF32)
        for it in range(rng.choice([1, 2, 4])):
            if rng.random() < 0.3:
                u0, u1 = rng.choice([0, 17, 100, 255, 256, 257]), rng.choice([0, 1, 999, 4001, 1024, 1023])
                Hg = g.run_iteration_random_site(u0, u1)
                Ho = (o.run_iteration_random_site_expf if expf else o.run_iteration_random_site)(u0, u1, n_threads=mo.max_threads())
                stats["expf"] += int(expf)
            else:
                th, sw = rng.choice([0, 1, 3]), rng.choice([0, 1, 2, 5, 9] if L < 128 else [0, 1, 2, 3])
                Hg, Ho = g.run_iteration(th, sw), o.run_iteration(th, sw, n_threads=mo.max_threads())
            assert np.array_equal(Hg, Ho), (tag, it)
            if rng.random() < 0.7:
                g.update_weights(); o.update_weights()
        assert np.array_equal(g.get_energies(), o.get_energies()), tag
        assert np.array_equal(g.get_spins(), o.get_spins()), tag
        assert np.max(np.abs(g.get_log_weights() - o.get_log_weights())) <= 1e-12, tag
        a, b = g.window_stats(); stats["windowed"] += a; stats["undone"] += b
        done += 1
    finally:
        g.close(); o.close()
print(f"soak seed {seed0}: {done} trials OK in {time.time() - t0:.0f} s; {stats}")
