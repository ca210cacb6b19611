"""Statistical pins of the CPU oracle against exact results for the 2D Ising model (no GPU, no product code).

P6  omega = -beta*E      -> canonical ensemble: P(E) = g(E) exp(-beta E)/Z with the exact g(E)
P7  omega = -ln g_exact  -> flat histogram; KL divergence d_k (Eq. 6) tiny; ln g recovered
P3  whole recursion      -> W^(n+1) = W^(n)/H^(n) (Eq. 4) from omega = 0 converges to the
                            exact density of states: max |ln g_est - ln g_exact| < 0.05 (north_star bar)
The estimate is ln g_est(E) = ln H(E) - omega(E), normalised so that sum g_est = 2^N.
"""
import os

import mpmath as mp
import numpy as np
import pytest

import muca_oracle as mo

GOLDEN = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")
THREADS = max(1, min(8, mo.max_threads()))


def ln_g_exact(L):
    with open(os.path.join(GOLDEN, f"ising_dos_L{L}.txt")) as f:
        g = [int(x) for x in f if not x.startswith("#")]
    return np.array([float(mp.log(v)) if v > 0 else -np.inf for v in g])


def ln_g_estimate(H, logw, N):
    m = H > 0
    e = np.full(H.shape, -np.inf)
    e[m] = np.log(H[m].astype(np.float64)) - logw[m]
    mx = e[m].max()
    return e - (mx + np.log(np.exp(e[m] - mx).sum())) + N * np.log(2.0)


@pytest.mark.parametrize("beta", [0.3, -0.15])
def test_canonical_weights_reproduce_boltzmann_distribution(beta):
    L, N, W, sweeps = 4, 16, 512, 2000
    E = -2 * N + 4 * np.arange(N + 1)
    g = np.exp(ln_g_exact(L))
    o = mo.Oracle(L, W, 5)
    o.set_log_weights(-beta * E)
    H = o.run_iteration(50, sweeps, n_threads=THREADS)
    P = H / H.sum()
    Pe = g * np.exp(-beta * E)
    Pe /= Pe.sum()
    assert np.abs(P - Pe).max() < 2e-3
    assert abs((P * E).sum() - (Pe * E).sum()) < 0.05
    assert H[1] == 0 and H[N - 1] == 0


@pytest.mark.parametrize("L,W,therm,sweeps", [(8, 1024, 200, 1000), (16, 1024, 1500, 3000)])
def test_exact_weights_give_flat_histogram(L, W, therm, sweeps):
    N = L * L
    lg = ln_g_exact(L)
    ok = np.isfinite(lg)
    logw = np.where(ok, -lg, 0.0)
    o = mo.Oracle(L, W, 6)
    o.set_log_weights(logw)
    H = o.run_iteration(therm, sweeps, n_threads=THREADS)
    assert np.all(H[~ok] == 0) and np.all(H[ok] > 0)
    P = H[ok] / H.sum()
    d_k = float((P * np.log(P * ok.sum())).sum())          # Eq. (6) with Q = 1/N_bins, N_bins = L^2 - 1
    assert d_k < 1e-3
    assert np.abs(ln_g_estimate(H, logw, N)[ok] - lg[ok]).max() < 0.05


def _recursion(L, W, schedule, seed=170700919):
    N = L * L
    lg = ln_g_exact(L)
    o = mo.Oracle(L, W, seed)
    errs = []
    for therm, sweeps in schedule:
        H = o.run_iteration(therm, sweeps, n_threads=THREADS)
        vis = H > 0
        assert np.all(np.isfinite(lg[vis]))                 # never visits a forbidden slot
        est = ln_g_estimate(H, o.get_log_weights(), N)
        errs.append((int(vis.sum()), float(np.abs(est[vis] - lg[vis]).max())))
        o.update_weights()
    return errs


def test_weight_recursion_converges_to_exact_dos_L8():
    errs = _recursion(8, 2048, [(20, 1000)] * 6)
    assert errs[-1][0] == 63 and errs[-2][0] == 63          # all L^2 - 1 accessible bins
    assert errs[-1][1] < 0.05 and errs[-2][1] < 0.05


@pytest.mark.slow
def test_weight_recursion_converges_to_exact_dos_L16():
    errs = _recursion(16, 4096, [(50, 300)] * 13 + [(100, 1000), (100, 3000)])
    assert errs[-1][0] == 255
    assert errs[-1][1] < 0.05, errs
