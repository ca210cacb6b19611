"""Production run with fixed weights + jackknife (Fig. 7).

not gpu: the oracle's numpy restatement is pinned: the jackknife against the textbook standard error of a mean, the
         log-sum-exp against scipy, the estimator against H = c g(E) exp(omega) built from the exact density of states,
         and the whole chain (oracle: converge, then production) against the exact ln g at L = 8.
gpu    : muca_production (library) against the oracle: identical call histograms, ln Omega and errors within 1e-10,
         same NaN pattern; and the paper's Fig. 7 check on the GPU at L = 16 (and L = 32 when the golden file exists).
"""
import os

import mpmath as mp
import numpy as np
import pytest

import muca_convergence as mc
import muca_oracle as mo
import muca_production as mpr
import paper_1707_00919_b200 as mb

GOLDEN = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


def ln_g_exact(L):
    with open(os.path.join(GOLDEN, f"ising_dos_L{L}.txt")) as f:
        g = [int(x) for x in f if not x.startswith("#")]
    return np.array([float(mp.log(v)) if v > 0 else np.nan for v in g])


# ------------------------------------------------------------------------------------------------ oracle pins
def test_jackknife_of_a_mean_is_the_standard_error():
    rng = np.random.default_rng(2)
    x = rng.normal(3.0, 2.0, size=(40, 5))
    n = x.shape[0]
    full, err = mpr.jackknife(x, lambda s: s / (n if np.allclose(s, x.sum(axis=0)) else n - 1))
    assert np.allclose(full, x.mean(axis=0), atol=1e-14)
    assert np.allclose(err, x.std(axis=0, ddof=1) / np.sqrt(n), rtol=1e-12)     # textbook identity for a linear estimator


def test_log_sum_exp_against_scipy():
    from scipy.special import logsumexp
    rng = np.random.default_rng(3)
    a = rng.normal(0, 300, 1000)
    assert abs(mpr.log_sum_exp(a) - logsumexp(a)) < 1e-10


@pytest.mark.parametrize("L", [4, 8, 16])
def test_estimator_recovers_the_exact_density_of_states(L):
    # a histogram exactly proportional to g(E) exp(omega(E)) must give ln g back, whatever omega and c
    lg = ln_g_exact(L)
    ok = np.isfinite(lg)
    rng = np.random.default_rng(4)
    logw = np.cumsum(rng.normal(0, 0.5, lg.size)) - np.where(ok, lg, 0.0)
    H = np.zeros(lg.size)
    H[ok] = np.exp(lg[ok] + logw[ok] + 17.3)
    est = mpr.ln_omega_estimate(H, logw, L)
    assert np.all(np.isnan(est[~ok])) and np.max(np.abs(est[ok] - lg[ok])) < 1e-9
    assert abs(mpr.log_sum_exp(est[ok]) - L * L * np.log(2.0)) < 1e-9            # sum exp = 2^N


def test_oracle_production_run_agrees_with_the_exact_solution_L8():
    L = 8
    o = mo.Oracle(L, 512, 21)
    log, conv = mc.converge(o, 120, 1e-4, n_threads=mo.max_threads())
    assert conv
    ln_om, err, Hs = mpr.production(o, 20, 20, 400, n_threads=mo.max_threads())
    lg = ln_g_exact(L)
    ok = np.isfinite(lg)
    assert Hs.shape == (20, 65) and np.all(np.isnan(ln_om[~ok])) and not np.any(np.isnan(ln_om[ok]))
    delta = np.abs(ln_om[ok] - lg[ok])
    assert delta.max() < 0.05                                                    # north_star bar for L <= 16
    assert np.mean(delta < 3 * err[ok]) > 0.9 and np.all(err[ok] > 0) and err[ok].max() < 0.05
    o.close()


# ------------------------------------------------------------------------------------------------ GPU parity
@pytest.mark.gpu
@pytest.mark.parametrize("L,W,iters,n_calls,therm,sweeps", [(8, 128, 12, 5, 3, 40), (16, 300, 6, 4, 2, 10), (32, 200, 3, 3, 1, 4)])
def test_gpu_production_matches_oracle(L, W, iters, n_calls, therm, sweeps):
    g, o = mb.Muca(L, W, 33), mo.Oracle(L, W, 33)
    try:
        for _ in range(iters):                                    # a few weight iterations first: non-trivial omega
            g.run_iteration(2, 10); g.update_weights()
            o.run_iteration(2, 10, n_threads=mo.max_threads()); o.update_weights()
        a_ln, a_err, a_H = g.production(n_calls, therm, sweeps)
        b_ln, b_err, b_H = mpr.production(o, n_calls, therm, sweeps, n_threads=mo.max_threads())
        assert np.array_equal(a_H, b_H)
        assert np.array_equal(np.isnan(a_ln), np.isnan(b_ln)) and np.array_equal(np.isnan(a_err), np.isnan(b_err))
        assert np.nanmax(np.abs(a_ln - b_ln)) < 1e-10 and np.nanmax(np.abs(a_err - b_err)) < 1e-10
        assert np.array_equal(g.get_log_weights(), o.get_log_weights())          # weights untouched by the production run
        assert g.iteration == o.iteration == iters + n_calls
        assert np.array_equal(g.get_spins(), o.get_spins())
    finally:
        g.close(); o.close()
    with pytest.raises(mb.MucaError):
        mb.Muca(8, 32, 1).production(1, 1, 1)


@pytest.mark.gpu
@pytest.mark.parametrize("L,W,n_calls,sweeps,bar", [(16, 4096, 100, 200, 0.05), (32, 16384, 100, 1000, 0.02)])
def test_gpu_density_of_states_against_the_exact_solution(L, W, n_calls, sweeps, bar):
    # the paper's Fig. 7 on the GPU: weight iteration to d_k < 1e-4, then a production run of 100 calls (long enough
    # that successive calls decorrelate: with 300 sweeps per call at L = 32 the jackknife errors come out too small)
    if not os.path.exists(os.path.join(GOLDEN, f"ising_dos_L{L}.txt")):
        pytest.skip(f"no exact density of states for L = {L} under tests/golden")
    g = mb.Muca(L, W, 170700919)
    try:
        log, conv = g.converge(600, 1e-4)
        assert conv
        ln_om, err, Hs = g.production(n_calls, 30, sweeps)
        lg = ln_g_exact(L)
        ok = np.isfinite(lg)
        assert not np.any(np.isnan(ln_om[ok])) and np.all(np.isnan(ln_om[~ok]))
        delta = np.abs(ln_om[ok] - lg[ok])
        assert delta.max() < bar, delta.max()
        assert np.mean(delta < 3 * err[ok]) > 0.9                                  # statistical agreement within error bars
    finally:
        g.close()
