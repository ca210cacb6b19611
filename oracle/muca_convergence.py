"""TEST INFRASTRUCTURE -- plain numpy / Python restatement of the paper's convergence protocol.

Only tests/, __graft_entry__.smoke() and bench.py's CPU legs may import this module; it shares no code with the
CUDA library (paper_1707_00919_b200/csrc).  Passages followed (PAPER.md = /root/reference/PAPER.md):
  flatness : Eq. (6), PAPER.md:134-152  d_k = sum_x P(x) ln(P(x)/Q(x)),  P = H / N_updates,  Q = 1/w,
             empty bins do not contribute;  w = max(w', 10), w' = width (in units of dE) of the range covered in the
             previous iteration.   Eq. (A.1), PAPER.md:252  d_c = max_x |H(x)/m - 1|,  m = N_updates / N_bins,
             N_bins = L^2 - 1 accessible energies.
  schedule : Eq. (7), PAPER.md:152  N_updates = 6 w^z / W, z = 2.25, "truncated to an integer value and increased
             by 1"; once w = L^2 + 1 it grows by a factor 1.1 per iteration;  N_therm = 30 w.
  converge : "The simulation ends if after an iteration we find that d_k < 1e-4".
Readings (R18-R20): flips per walker are rounded UP to whole sweeps (at least one); the width counts the
slots from the first to the last visited one, so that the whole range is w = L^2 + 1 as the paper states; "the
previous iteration" is the one just finished when flatness is judged and the next one is scheduled, and for Q only the
accessible slots of the covered range count (with an older, narrower width, or with the two unreachable slots counted,
Q = 1/w is not normalised over the support of P: d_k turns negative at once, resp. never falls below ln((N+1)/(N-1))); the first iteration
with w = L^2 + 1 still uses Eq. (7), the factor 1.1 applies from the next one on.
"""
import math

import numpy as np


def flatness(H, w=0):
    """w >= 1: width of the flat reference Q = 1/w; w = 0: max(accessible slots in the range of this histogram, 10) (R19)."""
    H = np.asarray(H, dtype=np.float64)
    n_bins = H.size
    N = n_bins - 1
    total = H.sum()
    visited = np.nonzero(H)[0]
    if visited.size == 0:
        return {"j_lo": -1, "j_hi": -1, "width": 0, "d_k": 0.0, "d_c": 0.0, "n_updates": 0}
    width = int(visited[-1] - visited[0] + 1)
    if w == 0:
        forbidden_inside = sum(1 for j in (1, N - 1) if visited[0] <= j <= visited[-1])
        w = max(width - forbidden_inside, 10)
    P = H[visited] / total
    Q = 1.0 / w
    d_k = float(np.sum(P * np.log(P / Q)))
    accessible = np.ones(n_bins, dtype=bool)
    accessible[[1, N - 1]] = False
    m = total / (N - 1)
    d_c = float(np.max(np.abs(H[accessible] / m - 1.0)))
    return {"j_lo": int(visited[0]), "j_hi": int(visited[-1]), "width": int(visited[-1] - visited[0] + 1),
            "d_k": d_k, "d_c": d_c, "n_updates": int(total)}


def schedule(L, n_walkers, w_prev, n_updates=0.0, full_range=0):
    """-> (w, therm_sweeps, sweeps, n_updates, full_range) of the next iteration."""
    N = L * L
    w = max(w_prev, 10)
    full = w >= N + 1
    if full and full_range:
        n_up = math.floor(1.1 * n_updates) + 1
    else:
        n_up = math.floor(6.0 * w ** 2.25 / n_walkers) + 1
    n_therm = 30 * w
    therm_sweeps = max(1, -(-n_therm // N))
    sweeps = max(1, -(-int(n_up) // N))
    return w, therm_sweeps, sweeps, float(n_up), int(full)


def converge(oracle, max_iterations, d_flat=1e-4, n_threads=1, random_site=False):
    """Drive an oracle context (muca_oracle.Oracle) through the weight iteration. Returns (log, converged).
    random_site: the paper's own update scheme and units (30 w and N_updates attempted flips per walker, no rounding)."""
    log, w_prev, n_up, full, conv = [], 0, 0.0, 0, False
    while len(log) < max_iterations and not conv:
        w, th, sw, n_up, full = schedule(oracle.L, oracle.W, w_prev, n_up, full)
        if random_site:
            H = oracle.run_iteration_random_site(30 * w, int(n_up), n_threads=n_threads)
        else:
            H = oracle.run_iteration(th, sw, n_threads=n_threads)
        fl = flatness(H)
        oracle.update_weights()
        rec = {"w": w, "therm_sweeps": th, "sweeps": sw}
        rec.update(fl)
        log.append(rec)
        w_prev = fl["width"]
        conv = fl["d_k"] < d_flat
    return log, conv
