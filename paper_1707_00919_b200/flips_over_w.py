"""Time per spin flip over the number of walkers -- the analogue of the paper's Fig. 2 (Sec. 3.1).

    python -m paper_1707_00919_b200.flips_over_w --L 32 [--weights tests/golden/ising_dos_L32.txt] [--random-site]

The paper measures, for L = 16, 32, 64, the time per spin flip of equilibrated walkers under the exact weights as a
function of W and reads off the walker count that fills the device.  This prints the same curve for
libmuca_b200: for W in steps of half a warp per SM up to `--max-warps-per-sm`, a context of W walkers is created, the
weights are set, and `--repeats` iterations of (therm + sweeps) sweeps are timed with the library's own CUDA events
(muca_last_sweep_ms); the best one counts.  Columns: W, warps per SM, ms per iteration, flips/s, ns per flip.
`--walkers W` times that one walker count instead (e.g. `--walkers 16384 --therm 550 --sweeps 0` against `--therm 0
--sweeps 550`: what recording the histogram costs the sweep kernel).

Weights: `--weights FILE` reads the exact density of states g(E_j), one integer per line, '#' comments (the files under
tests/golden/ for L <= 32; any file of that format will do) and sets omega = -ln g, the paper's protocol.  Without it
omega = 0 is used for the first iteration and Eq. (4) updates after each (the start-up regime bench.py times).
Marshalling and a loop only: every flip runs in the library's kernels.
"""
import argparse
import math

import numpy as np

from .binding import (MUCA_ACCEPT_EXPF32, MUCA_OPT_ACCEPTANCE, Muca, suggest_walkers)


def read_log_weights(path: str, n_bins: int) -> np.ndarray:
    g = [int(x) for x in open(path) if x.strip() and not x.startswith("#")]
    if len(g) != n_bins:
        raise SystemExit(f"{path}: {len(g)} values, expected N + 1 = {n_bins}")
    return np.array([-math.log(v) if v > 0 else 0.0 for v in g])   # math.log takes integers far beyond double range (g ~ 2^N)


def main():
    import torch
    ap = argparse.ArgumentParser(description=__doc__, formatter_class=argparse.RawDescriptionHelpFormatter)
    ap.add_argument("--L", type=int, default=32)
    ap.add_argument("--weights", default=None, help="file with the exact g(E_j), one integer per line")
    ap.add_argument("--therm", type=int, default=2)
    ap.add_argument("--sweeps", type=int, default=None, help="measured sweeps per iteration (default: 200 / 60 / 20 / 10 for L <= 16 / 32 / 64 / 128)")
    ap.add_argument("--repeats", type=int, default=3)
    ap.add_argument("--max-warps-per-sm", type=float, default=None, help="default: twice the suggested count")
    ap.add_argument("--random-site", action="store_true", help="the paper's own update scheme (same random site in all walkers)")
    ap.add_argument("--expf32", action="store_true", help="with --random-site: the paper's single-precision acceptance")
    ap.add_argument("--walkers", type=int, default=None, help="time this one walker count instead of the scan")
    ap.add_argument("--seed", type=int, default=170700919)
    a = ap.parse_args()
    L, N = a.L, a.L * a.L
    sweeps = a.sweeps if a.sweeps is not None else (200 if L <= 16 else 60 if L == 32 else 20 if L == 64 else 10)
    n_sm = torch.cuda.get_device_properties(torch.cuda.current_device()).multi_processor_count
    w_opt, pairs = suggest_walkers(L)
    top = a.max_warps_per_sm if a.max_warps_per_sm is not None else 2.0 * pairs
    logw = read_log_weights(a.weights, N + 1) if a.weights else None
    scheme = ("random site" + (", fp32 acceptance" if a.expf32 else "")) if a.random_site else "typewriter"
    print(f"# L={L} n_sm={n_sm} suggested W={w_opt} ({pairs} warp pairs per SM); scheme: {scheme}; weights: "
          f"{'-ln g from ' + a.weights if a.weights else 'omega = 0, then Eq. (4) after every iteration'}; "
          f"{a.repeats} iterations of ({a.therm} + {sweeps}) sweeps, best one; "
          "columns: W, warps per SM, ms per iteration, flips/s, ns per flip")
    counts = [a.walkers] if a.walkers else [int(round(0.5 * h * 32 * n_sm)) for h in range(1, int(2 * top + 1e-9) + 1)]
    for W in counts:
        wps = W / (32.0 * n_sm)
        g = Muca(L, W, a.seed)
        try:
            if logw is not None:
                g.set_log_weights(logw)
            if a.random_site and a.expf32:
                g.set_option(MUCA_OPT_ACCEPTANCE, MUCA_ACCEPT_EXPF32)
            best = float("inf")
            for _ in range(a.repeats):
                if a.random_site:
                    g.run_iteration_random_site(a.therm * N, sweeps * N)
                else:
                    g.run_iteration(a.therm, sweeps)
                best = min(best, g.last_sweep_ms()[0])
                if logw is None:
                    g.update_weights()
        finally:
            g.close()
        flips = W * N * (a.therm + sweeps)
        print(f"{W:7d} {wps:6.2f} {best:9.3f} {flips / (best * 1e-3):.4e} {best * 1e6 / flips:.6f}", flush=True)


if __name__ == "__main__":
    main()
