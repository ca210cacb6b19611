#!/usr/bin/env python
"""bench.py -- spin-flip attempts/sec of the parallel-MUCA hot path on B200 (BASELINE.json metric).

A "step" is one pass of the whole hot path over one seeded synthetic job: create + initialise the walkers
(a0), then `iterations` x [threshold build (a1), thermalisation + measured sweeps (a2, a3), histogram merge
(a4), Eq. (4) weight update (a5)], then the unpack of the final configurations (a6).
  value : whole-job flip attempts / device time, state resident in HBM (final spins unpacked on the device)
  e2e   : same job through the C ABI with HOST buffers (thresholds H2D and H D2H every iteration, final
          energies and spins D2H into host arrays inside the timed region)
Workload at N=1: BASELINE.json configs[2] (L=32, 16384 walkers, 15 x (50 + 500) sweeps) -- the config the
north_star target is quoted on.  N>1: every rank runs that many walkers (weak scaling) with global walker
ids and one all-reduce of H per iteration.

`--impl reference` times the CPU oracle (oracle/) on the host cores on a bounded walker sample of the same
workload; there is no installable reference implementation (the paper's code is not available).
"""
import argparse
import json
import os
import sys
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
for p in (ROOT, os.path.join(ROOT, "oracle")):
    if p not in sys.path:
        sys.path.insert(0, p)

import numpy as np  # noqa: E402

METRIC = "spin-flip attempts/sec"
UNIT = "flips/s"
# algorithmic integer work per flip attempt and the roofline of the binding pipe.
# Per attempted flip: 1/4 Philox4x32-10 call (4 IMAD.WIDE on the FMA-heavy pipe + 4.5 LOP3) and ~11.5 instructions of
# site update = 20 thread-instructions, of which 11.7 can only run on the 16-lane ALU pipe (LOP3/IADD3/SHF/SEL/ISETP).
ALU_OPS_PER_FLIP = 11.7             # binding pipe: ALU, 16 lanes per scheduler per clock (profiles/r01_ubench_pipes.txt)
OPS_PER_FLIP = 20.0                 # all thread-instructions (issue slots: 32 lanes per scheduler per clock)
SCHED_PER_SM, ALU_LANES, ISSUE_LANES = 4, 16, 32
# Counters of ONE sweep-kernel launch per workload, copied by hand from the ncu --set full captures under profiles/ into
# that JSON file (dram__bytes_read.sum + dram__bytes_write.sum, pipe and issue utilisation; profiles/README.md names the
# captures): read at run time, nothing is measured under the profiler here.  The file records the commit and the sha256
# of csrc/ (paper_1707_00919_b200.build.csrc_sha256) it was captured from; when the sources have changed since, the
# entry is still printed, with "stale": true beside it.
NCU_SUMMARY = os.path.join(ROOT, "profiles", "r03_ncu_summary.json")


def ncu_summary(workload):
    try:
        with open(NCU_SUMMARY) as f:
            doc = json.load(f)
        entry = doc.get(workload)
        if entry is None:
            return None
        from paper_1707_00919_b200 import build as lib_build
        return dict(entry, stale=(entry.get("captured_from") or {}).get("csrc_sha256") != lib_build.csrc_sha256())
    except Exception:
        return None


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", default="L32_w16384")
    ap.add_argument("--ref-walkers", type=int, default=128, help="walker sample of the reference / cpu_baseline legs")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-other-configs", action="store_true", help="skip the untimed legs on configs 4 and 5")
    return ap.parse_args()


def peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(path) as f:
            return json.load(f), "measured"
    except Exception:
        return {"hbm_gbs": 6650.0, "sm_max_mhz": 1965.0}, "fallback"


# ------------------------------------------------------------------------------------------------ oracle legs
def oracle_job(cfg, n_walkers, n_threads, iterations=None):
    """The oracle, as it stands, on the first n_walkers walkers of the workload. Returns (flips, seconds)."""
    import muca_oracle as mo
    iters = cfg.iterations if iterations is None else iterations
    t0 = time.perf_counter()
    o = mo.Oracle(cfg.L, n_walkers, cfg.seed)
    for _ in range(iters):
        o.run_iteration(cfg.therm_sweeps, cfg.sweeps, n_threads=n_threads)
        o.update_weights()
    o.get_energies(); o.get_spins()
    dt = time.perf_counter() - t0
    o.close()
    return iters * n_walkers * cfg.N * (cfg.therm_sweeps + cfg.sweeps), dt


def run_reference(args, cfg):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import muca_oracle as mo
    cores = mo.max_threads()
    W = args.ref_walkers
    for _ in range(min(args.warmup, 1)):
        oracle_job(cfg, W, cores, iterations=1)
    flips = secs = 0.0
    for _ in range(args.steps):
        f, s = oracle_job(cfg, W, cores)
        flips += f; secs += s
    v = flips / secs
    sample = f"first {W} of {cfg.n_walkers} walkers, full schedule {cfg.iterations} x ({cfg.therm_sweeps}+{cfg.sweeps}) sweeps"
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * secs / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "int32", "data": "synthetic",
        "config": {"workload": cfg.name, "L": cfg.L, "n_walkers": W, "iterations": cfg.iterations,
                   "therm_sweeps": cfg.therm_sweeps, "sweeps": cfg.sweeps, "note": "CPU oracle, OpenMP over walkers"},
        "cpu_baseline": {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }))


# ------------------------------------------------------------------------------------------------ clocks
class ClockSampler:
    """SM clock and throttle reasons through NVML, sampled from the MAIN thread between the kernels of the timed
    region (after every iteration).  A background thread polling NVML contends with the CUDA calls of the job for a
    driver lock: single queries then took up to 0.8 s and stalled kernel launches (profiles/README.md)."""

    def __init__(self, index):
        self.sm, self.reasons, self.max_mhz = [], set(), None
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
            nv = pynvml
            self.names = {nv.nvmlClocksEventReasonHwSlowdown: "hw_slowdown", nv.nvmlClocksEventReasonHwThermalSlowdown: "hw_thermal_slowdown",
                          nv.nvmlClocksEventReasonSwThermalSlowdown: "sw_thermal_slowdown", nv.nvmlClocksEventReasonSwPowerCap: "sw_power_cap"} \
                if hasattr(nv, "nvmlClocksEventReasonHwSlowdown") else \
                {nv.nvmlClocksThrottleReasonHwSlowdown: "hw_slowdown", nv.nvmlClocksThrottleReasonHwThermalSlowdown: "hw_thermal_slowdown",
                 nv.nvmlClocksThrottleReasonSwThermalSlowdown: "sw_thermal_slowdown", nv.nvmlClocksThrottleReasonSwPowerCap: "sw_power_cap"}
        except Exception:
            self.nv = None

    def sample(self):
        if self.nv is None:
            return
        nv = self.nv
        try:
            self.sm.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
            try:
                r = nv.nvmlDeviceGetCurrentClocksEventReasons(self.h)
            except Exception:
                r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
            for bit, name in self.names.items():
                if r & bit:
                    self.reasons.add(name)
        except Exception:
            pass

    def result(self):
        return {"sm_mhz": float(np.median(self.sm)) if self.sm else None, "sm_max_mhz": self.max_mhz,
                "reasons": sorted(self.reasons), "samples": len(self.sm),
                "how": "NVML from the main thread after every iteration of the timed steps"}


# ------------------------------------------------------------------------------------------------ the other configs
def other_configs(mb, cfg_main, peak, f_max_hz, device_index):
    """north_star: "throughput is reported on each config".  The headline legs time ONE workload; here, after them and
    outside their timed regions, the two other large configs run two jobs each, and L = 128 once more in the regime of a
    production run (walkers spread over the whole energy range -> sorted per-block table windows).
    Sweep kernels only: the library's own CUDA events around the launches of every iteration (muca_last_sweep_ms)."""
    from paper_1707_00919_b200.workloads import by_name, onsager_log_dos
    res = {}

    def entry(c, W, flips, ms, launches, sampler, what, extra=None):
        fps = flips / (ms * 1e-3)
        e = {"value": fps, "unit": UNIT, "c_flip_cycles": W * f_max_hz / fps, "frac": fps * ALU_OPS_PER_FLIP / 1e12 / peak,
             "sweep_ms": ms, "launches": launches, "clocks": sampler.result(), "what": what}
        e.update(extra or {})
        return e

    for name in ("L64_w32768", "L128_w8192"):
        if name == cfg_main.name:
            continue
        c = by_name(name)
        sampler = ClockSampler(device_index)
        ms = 0.0; launches = 0; steps = 2
        for _ in range(steps):
            g = mb.Muca(c.L, c.n_walkers, c.seed)
            for _ in range(c.iterations):
                g.run_iteration(c.therm_sweeps, c.sweeps)
                m, k = g.last_sweep_ms()
                ms += m; launches += k
                sampler.sample()
                g.update_weights()
            g.close()
        res[name] = entry(c, c.n_walkers, steps * mb.total_flips(c), ms, launches, sampler,
                          f"{steps} jobs of {c.iterations} x ({c.therm_sweeps}+{c.sweeps}) sweeps, sweep kernels only")
    # L = 128, walkers spread from -2N to +2N (walker k: a fraction k/2W of its spins down, every second walker times a
    # checkerboard), weights omega(E) = -N s(E/N) from the infinite-lattice entropy (workloads.onsager_log_dos: no exact
    # g(E) exists in the tree for L = 128), close enough to flat-histogram weights to keep them spread: 3 x (20 + 50) sweeps
    c = by_name("L128_w8192")
    W, N, L = c.n_walkers, c.N, c.L
    rng = np.random.default_rng(c.seed)
    spins = np.empty((W, N), dtype=np.int8)
    pk = np.linspace(0.0, 0.5, W, dtype=np.float32)
    for a in range(0, W, 1024):
        spins[a:a + 1024] = np.where(rng.random((min(1024, W - a), N), dtype=np.float32) < pk[a:a + 1024, None], -1, 1)
    yy, xx = np.divmod(np.arange(N), L)
    spins[1::2] *= np.where((xx + yy) % 2 == 0, 1, -1).astype(np.int8)[None, :]
    g = mb.Muca(L, W, c.seed)
    g.set_spins(spins)
    g.set_log_weights(-onsager_log_dos(L))
    sampler = ClockSampler(device_index)
    ms = 0.0; launches = 0
    g.run_iteration(c.therm_sweeps, c.sweeps)                                  # untimed first call
    for _ in range(3):
        g.run_iteration(c.therm_sweeps, c.sweeps)
        m, k = g.last_sweep_ms()
        ms += m; launches += k
        sampler.sample()
    E = g.get_energies()
    windowed, undone = g.window_stats()
    g.close()
    res["L128_w8192_spread"] = entry(c, W, 3 * W * N * (c.therm_sweeps + c.sweeps), ms, launches, sampler,
                                     "walkers spread over the whole energy range, fixed weights -N s_Onsager(E/N), 3 x "
                                     f"({c.therm_sweeps}+{c.sweeps}) sweeps: sorted per-block table windows; the time "
                                     "includes the host's sorting and the snapshots between the launches",
                                     {"slots_spanned": int((E.max() - E.min()) // 4), "windowed_iterations": windowed,
                                      "undone_launches": undone})
    return res


# ------------------------------------------------------------------------------------------------ our arm
def run_ours(args, cfg):
    import torch
    import torch.distributed as dist
    import paper_1707_00919_b200 as mb

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (libmuca_b200 has no CPU fallback)")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    W = cfg.n_walkers                      # per rank: weak scaling
    offset = rank * W
    flips_per_step = mb.total_flips(cfg, W)
    table_bytes = cfg.n_bins * 8 * 4
    hist_bytes = cfg.n_bins * 8

    h_E = np.empty(W, dtype=np.int32)
    h_spins_t = torch.empty((W, cfg.L, cfg.L), dtype=torch.int8).pin_memory()
    h_spins = h_spins_t.numpy()
    l2_flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)

    stats = {"sweep_ms": 0.0, "sweep_launches": 0, "launches": 0}
    sampler = ClockSampler(local)

    def job(e2e: bool, record: bool):
        # ShardedMuca (paper_1707_00919_b200/parallel.py) is the N > 1 path the tests cover (tests/test_parallel_gloo.py):
        # contiguous walker ranges with global ids, one all-reduce of H per iteration -- the method's one exchange,
        # PAPER.md:87 --, the same Eq. (4) on every rank.  At N = 1 it is the plain context plus a copy of H.
        sm = mb.ShardedMuca(cfg.L, world * W, cfg.seed)                        # a0 (init kernel)
        g = sm.engine
        assert (sm.offset, sm.count) == (offset, W)
        n_launch = 1
        for _ in range(cfg.iterations):
            sm.run_iteration(cfg.therm_sweeps, cfg.sweeps)                     # a1-a4 (+ H2D table, D2H H), all-reduce(H)
            ms, k = g.last_sweep_ms()
            n_launch += k
            if record:
                stats["sweep_ms"] += ms; stats["sweep_launches"] += k
                sampler.sample()                                               # clocks line of the contract (see ClockSampler)
            sm.update_weights()                                                # a5
        if e2e:
            g.get_energies(h_E)
            g.get_spins(h_spins)                                               # a6: unpack kernel + D2H
        else:
            g.unpack_spins_device()                                            # a6: unpack kernel, stays in HBM
        n_launch += 1
        if record:
            stats["launches"] += n_launch
        sm.close()

    def timed(e2e: bool, steps: int, record: bool):
        total_ms = 0.0
        for _ in range(steps):
            l2_flush.fill_(1)                                                  # flush L2 between timed steps
            torch.cuda.synchronize()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            job(e2e, record)
            e1.record()
            torch.cuda.synchronize()
            total_ms += e0.elapsed_time(e1)
        return total_ms

    for _ in range(max(args.warmup, 3)):
        job(False, False)

    def bracket():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()

    job(True, False)
    sampler.sample()            # first NVML queries outside the timed region
    sampler.sm.clear(); sampler.reasons.clear()
    bracket()
    ms_dev = timed(False, args.steps, True)
    bracket()
    ms_e2e = timed(True, args.steps, False)
    bracket()

    t = torch.tensor([ms_dev, ms_e2e], dtype=torch.float64, device=dev)
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    ms_dev, ms_e2e = float(t[0]), float(t[1])
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    pk, pk_kind = peaks()
    f_max_hz = float(pk.get("sm_max_mhz", 1965.0)) * 1e6
    SM_COUNT = torch.cuda.get_device_properties(dev).multi_processor_count
    ncu = ncu_summary(cfg.name) if world == 1 else None
    value = world * flips_per_step * args.steps / (ms_dev * 1e-3)
    e2e_v = world * flips_per_step * args.steps / (ms_e2e * 1e-3)
    # dominant kernel: the sweep kernel (one launch per iteration)
    flips_per_launch = mb.flips_per_iteration(cfg, W) * cfg.iterations * args.steps / max(stats["sweep_launches"], 1)
    avg_launch_s = stats["sweep_ms"] * 1e-3 / max(stats["sweep_launches"], 1)
    kern_flips_s = flips_per_launch / avg_launch_s
    achieved = kern_flips_s * ALU_OPS_PER_FLIP / 1e12
    peak = SM_COUNT * SCHED_PER_SM * ALU_LANES * f_max_hz / 1e12
    issue_peak = SM_COUNT * SCHED_PER_SM * ISSUE_LANES * f_max_hz / 1e12
    kernel = "muca::sweep_kernel_v6<%d>" % cfg.L if cfg.L <= 32 else "muca::sweep_kernel_s6<%d>" % cfg.L
    clk = sampler.result()
    f_run_hz = (clk["sm_mhz"] or 0.0) * 1e6
    roofline = {
        "bound": "alu", "achieved": achieved, "peak": peak, "unit": "T lane-ops/s on the ALU pipe", "frac": achieved / peak,
        "frac_kind": "ALGORITHMIC: flips/s x 11.7 ALU-only instructions per attempted flip (DESIGN.md 6.2) over the ALU-pipe "
                     "peak at sm_max_mhz; the instructions actually executed and the pipe utilisation ncu measured are under 'ncu'",
        "frac_at_sampled_clock": achieved / (SM_COUNT * SCHED_PER_SM * ALU_LANES * f_run_hz / 1e12) if f_run_hz else None,
        "traffic": ncu.get("dram_bytes_per_launch") if ncu else None,
        "ncu": ncu,
        "kernel": kernel, "kernel_flips_per_s": kern_flips_s,
        "ops_per_flip": ALU_OPS_PER_FLIP, "avg_launch_ms": avg_launch_s * 1e3, "kernel_share_of_step": stats["sweep_ms"] / ms_dev,
        "c_flip_cycles": W * f_max_hz / kern_flips_s,
        "peak_source": f"{SM_COUNT} SM x {SCHED_PER_SM} schedulers x {ALU_LANES} ALU lanes x sm_max_mhz ({pk_kind} MEASURED_PEAKS.json clock); "
                       "11.7 ALU-only instructions per attempted flip (DESIGN.md 6.2)",
        "issue": {"achieved": kern_flips_s * OPS_PER_FLIP / 1e12, "peak": issue_peak, "unit": "T thread-instructions/s",
                  "frac": kern_flips_s * OPS_PER_FLIP / 1e12 / issue_peak, "ops_per_flip": OPS_PER_FLIP},
        "hbm": {"algorithmic_bytes_per_flip": 0.0 if cfg.L <= 32 else 0.25, "peak_gbs": pk.get("hbm_gbs"),
                "algorithmic_lattice_gbs": (0.0 if cfg.L <= 32 else 0.25) * kern_flips_s / 1e9,
                "ncu_dram_gbs": ncu["dram_bytes_per_launch"] / avg_launch_s / 1e9 if ncu and ncu.get("dram_bytes_per_launch") else None,
                "note": "algorithmic_lattice_gbs = 0.25 B per flip (every packed word of a streamed lattice read and written "
                        "once per sweep) x flips/s: traffic between the SMs and L2, which holds the 16 MiB of lattices of "
                        "configs 4 and 5; ncu_dram_gbs = what ncu saw at the DRAM interface for one launch over the launch "
                        "time measured here.  Lattices are shared-memory resident for L <= 32."},
    }
    out = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": max(args.warmup, 3),
        "ms_per_step": ms_dev / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "int32", "data": "synthetic",
        "config": {"workload": cfg.name, "L": cfg.L, "n_walkers_per_gpu": W, "iterations": cfg.iterations,
                   "therm_sweeps": cfg.therm_sweeps, "sweeps": cfg.sweeps, "seed": cfg.seed,
                   "flips_per_step_per_gpu": flips_per_step, "l2": "flushed between timed steps (256 MiB write)",
                   "parallelism": f"walkers x{world}, one all-reduce(H) per iteration" if world > 1 else "1 GPU"},
        "clocks": clk,
        "e2e": {"value": e2e_v, "unit": UNIT,
                "h2d_bytes_per_step": cfg.iterations * table_bytes,
                "d2h_bytes_per_step": cfg.iterations * hist_bytes + h_E.nbytes + h_spins.nbytes,
                "ms_per_step": ms_e2e / args.steps},
        "gpu_launches": stats["launches"],
        "roofline": roofline,
    }
    if world == 1:
        # secondary workload (the paper's Fig. 2 protocol): after the configured iterations,
        # three measured-only iterations with the weights frozen (broad histogram, little bin contention)
        g = mb.Muca(cfg.L, W, cfg.seed)
        for _ in range(cfg.iterations):
            g.run_iteration(cfg.therm_sweeps, cfg.sweeps)
            g.update_weights()
        fz = []
        for _ in range(3):
            g.run_iteration(0, cfg.sweeps)
            fz.append(W * cfg.N * cfg.sweeps / (g.last_sweep_ms()[0] * 1e-3))
        g.close()
        out["frozen_weights"] = {"value": float(np.median(fz)), "unit": UNIT,
                                 "what": f"sweep kernel only, 3 x {cfg.sweeps} measured sweeps after the {cfg.iterations} "
                                         "configured iterations, weights not updated (outside the timed region)"}
    if world == 1 and not args.no_other_configs:
        out["other_configs"] = other_configs(mb, cfg, peak, f_max_hz, local)
    if world == 1 and not args.no_cpu_baseline:
        import muca_oracle as mo
        cores = mo.max_threads()
        Wb = args.ref_walkers
        f, s = oracle_job(cfg, Wb, cores, iterations=3)
        out["cpu_baseline"] = {"value": f / s, "unit": UNIT, "cores": cores, "kind": "oracle",
                               "sample": f"first {Wb} of {cfg.n_walkers} walkers, 3 of {cfg.iterations} iterations x "
                                         f"({cfg.therm_sweeps}+{cfg.sweeps}) sweeps, OpenMP over walkers"}
        f1, s1 = oracle_job(cfg, max(Wb // 8, 8), 1, iterations=1)
        out["cpu_baseline"]["single_thread_value"] = f1 / s1
    print(json.dumps(out))
    if world > 1:
        dist.destroy_process_group()


def main():
    args = parse()
    from paper_1707_00919_b200.workloads import by_name
    cfg = by_name(args.config)
    if args.impl == "reference":
        run_reference(args, cfg)
    else:
        run_ours(args, cfg)


if __name__ == "__main__":
    main()
