"""TEST INFRASTRUCTURE -- plain numpy restatement of the paper's production run.

Only tests/, __graft_entry__.smoke() and bench.py's CPU legs may import this module; it shares no code with the
CUDA library.  Passages followed: "we divide the total number of attempted spin flips into 100 individual calls to
the multicanonical simulation function [with fixed weights] and use the resulting individual histograms to determine
error bars from a jackknife analysis [46]"; the estimate is ln Omega(E) = ln H(E) - omega(E) (H sampled
with weight W = exp(omega)), normalised so that sum_E exp[ln Omega(E)] = 2^(L^2), all
in logarithms.  Readings (R21): the estimate uses the SUM of the call histograms; jackknife block k leaves
call k out; a slot counts only if every leave-one-out histogram visited it (else NaN); every block is normalised on
its own before the spread is taken.
"""
import numpy as np


def log_sum_exp(a):
    m = np.max(a)
    return float(m + np.log(np.sum(np.exp(a - m))))


def ln_omega_estimate(H, logw, L):
    """ln Omega(E_j) from one histogram sampled with weights exp(logw); NaN on unvisited slots."""
    H = np.asarray(H, dtype=np.float64)
    out = np.full(H.size, np.nan)
    v = H > 0
    out[v] = np.log(H[v]) - np.asarray(logw, dtype=np.float64)[v]
    out[v] += L * L * np.log(2.0) - log_sum_exp(out[v])          # sum exp(ln Omega) = 2^N
    return out


def jackknife(blocks, estimator):
    """Generic delete-one jackknife [46]: blocks (n, ...) summed except one; returns (estimate on all, error)."""
    blocks = np.asarray(blocks)
    n = blocks.shape[0]
    total = blocks.sum(axis=0)
    full = estimator(total)
    loo = np.stack([estimator(total - blocks[k]) for k in range(n)])
    mean = loo.mean(axis=0)
    err = np.sqrt((n - 1) / n * np.sum((loo - mean) ** 2, axis=0))
    return full, err


def production(oracle, n_calls, therm_sweeps, sweeps, n_threads=1):
    """n_calls fixed-weight calls on an oracle context. Returns (ln_omega, err, histograms[n_calls, n_bins])."""
    logw = oracle.get_log_weights()
    Hs = np.stack([oracle.run_iteration(therm_sweeps, sweeps, n_threads=n_threads) for _ in range(n_calls)])
    ln_om, err = jackknife(Hs.astype(np.float64), lambda H: ln_omega_estimate(H, logw, oracle.L))
    return ln_om, err, Hs
