"""Run the paper's weight iteration to convergence on the current CUDA device and print a summary.

    python -m paper_1707_00919_b200.converge [--L 32] [--walkers 16384] [--seed 170700919] [--d-flat 1e-4] [--max-iterations 1000]

Everything runs inside libmuca_b200 (muca_converge: Eq. (7) schedule, sweeps, Eq. (6) flatness, Eq. (4) update;
PAPER.md:130-157); this module only parses arguments and prints the iteration log as JSON lines.
"""
import argparse
import json
import time

from .binding import MUCA_OPT_UPDATE_SCHEME, MUCA_SCHEME_RANDOM_SITE, Muca


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--L", type=int, default=32)
    ap.add_argument("--walkers", type=int, default=16384)
    ap.add_argument("--seed", type=int, default=170700919)
    ap.add_argument("--d-flat", type=float, default=1e-4)
    ap.add_argument("--max-iterations", type=int, default=1000)
    ap.add_argument("--random-site", action="store_true", help="the paper's own update scheme and units (muca.h: MUCA_SCHEME_RANDOM_SITE)")
    ap.add_argument("--log", action="store_true", help="print one JSON line per iteration")
    a = ap.parse_args()
    g = Muca(a.L, a.walkers, a.seed)
    if a.random_site:
        g.set_option(MUCA_OPT_UPDATE_SCHEME, MUCA_SCHEME_RANDOM_SITE)
    t0 = time.perf_counter()
    log, converged = g.converge(a.max_iterations, a.d_flat)
    wall = time.perf_counter() - t0
    g.close()
    if a.log:
        for i, r in enumerate(log):
            print(json.dumps({"iteration": i, **r}))
    N = a.L * a.L
    full = [i for i, r in enumerate(log) if r["width"] == N + 1]
    sweeps = sum(r["sweeps"] + r["therm_sweeps"] for r in log)
    if a.random_site:      # updates per walker: 30 w thermalisation + N_updates recorded ones, in sweeps of N updates
        sweeps = sum(30 * r["w"] + r["n_updates"] // a.walkers for r in log) / N
    print(json.dumps({
        "L": a.L, "walkers": a.walkers, "scheme": "random_site" if a.random_site else "typewriter", "seed": a.seed, "d_flat": a.d_flat, "converged": converged, "iterations": len(log),
        "first_full_range_iteration": full[0] if full else None, "wall_s": wall,
        "sweep_kernel_s": sum(r["sweep_ms"] for r in log) * 1e-3, "sweeps_per_walker": sweeps,
        "flip_attempts": int(sweeps * a.walkers * N), "last_d_k": log[-1]["d_k"] if log else None,
        "last_d_c": log[-1]["d_c"] if log else None}))


if __name__ == "__main__":
    main()
