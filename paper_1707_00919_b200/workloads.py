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


def onsager_log_dos(L: int):
    """Synthetic stand-in for ln g(E_j), j = 0..N, where no exact density of states is at hand (L = 128): N s(E_j / N) with
    s the entropy per spin of the INFINITE square-lattice Ising model, from Onsager's internal energy
        u(beta) = -coth(2 beta) [1 + (2/pi) (2 tanh^2(2 beta) - 1) K(k)],  k = 2 sinh(2 beta) / cosh^2(2 beta),
    integrated as ds = beta du from s(u = 0) = ln 2 and mirrored to E > 0.  Against the exact finite-lattice g(E) it is off
    by less than 4 in ln g over the whole range at L = 32 (and by O(ln N) in general): -onsager_log_dos(L) as omega gives a
    histogram flat within two orders of magnitude, which is all bench.py needs to keep walkers spread over all energies.
    Input data only: the method itself never uses it."""
    import numpy as np
    from scipy.special import ellipk
    N = L * L
    b = np.linspace(1e-6, 3.0, 600001)
    t = np.tanh(2.0 * b)
    k = 2.0 * np.sinh(2.0 * b) / np.cosh(2.0 * b) ** 2
    u = -(1.0 / t) * (1.0 + (2.0 / np.pi) * (2.0 * t * t - 1.0) * ellipk(np.minimum(k * k, 1.0 - 1e-15)))
    s = np.log(2.0) + np.concatenate([[0.0], np.cumsum(0.5 * (b[1:] + b[:-1]) * np.diff(u))])
    e = (-2.0 * N + 4.0 * np.arange(N + 1)) / N
    return N * np.interp(-np.abs(e), u[::-1], s[::-1])
