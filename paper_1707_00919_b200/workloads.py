"""Seeded synthetic workloads (BASELINE.json `configs`) -- data only, none of the method's arithmetic.

Shared by tests/, bench.py and __graft_entry__.py; imported by neither oracle/ nor csrc/.
The paper's workload IS synthetic: L x L Ising walkers started from random spins (our reading R1) and
omega == 0, with weights updated after every iteration; there is no dataset.
"""
from dataclasses import dataclass

PRIMARY_SEED = 170700919
EXTRA_SEEDS = (1, 0xDEADBEEFCAFEF00D)   # the second exercises the high key word


@dataclass(frozen=True)
class Config:
    name: str
    L: int
    n_walkers: int
    iterations: int
    therm_sweeps: int
    sweeps: int
    seed: int = PRIMARY_SEED

    @property
    def N(self) -> int:
        return self.L * self.L

    @property
    def n_bins(self) -> int:
        return self.N + 1


# BASELINE.json configs[0..4]
CONFIGS = (
    Config("L8_w128", 8, 128, 8, 10, 100),
    Config("L16_w4096", 16, 4096, 12, 20, 200),
    Config("L32_w16384", 32, 16384, 15, 50, 500),
    Config("L64_w32768", 64, 32768, 10, 50, 200),
    Config("L128_w8192", 128, 8192, 5, 20, 50),
)


def by_name(name: str) -> Config:
    for c in CONFIGS:
        if c.name == name:
            return c
    raise KeyError(name)


def flips_per_iteration(c: Config, n_walkers: int = None) -> int:
    """Spin-flip attempts of one iteration: thermalisation attempts count."""
    w = c.n_walkers if n_walkers is None else n_walkers
    return w * c.N * (c.therm_sweeps + c.sweeps)


def total_flips(c: Config, n_walkers: int = None) -> int:
    return c.iterations * flips_per_iteration(c, n_walkers)
