"""Multi-GPU sharding of the walkers (Fig. 1: independent walkers, one histogram sum per iteration).

One process per GPU.  Walkers are split into contiguous ranges; every rank passes the GLOBAL id of its
first walker to the library (R16), so the Markov chains -- hence H, E, spins -- do not depend
on the number of ranks.  The only exchange of the method is the histogram sum: one all-reduce of
N+1 integers per iteration (8 KiB at L=32) through torch.distributed (NCCL over NVLink on GPUs, gloo
in the CPU tests); every rank then applies Eq. (4) to the same total and so holds identical weights.
Integer sums are exact: the result is bit-identical for any rank count.
"""
import numpy as np


def shard_range(n_total: int, rank: int, world: int):
    """Contiguous split: the first (n_total % world) ranks get one extra walker. Returns (offset, count)."""
    if not (0 <= rank < world) or n_total < world:
        raise ValueError("need 0 <= rank < world <= n_total")
    base, extra = divmod(n_total, world)
    count = base + (1 if rank < extra else 0)
    offset = rank * base + min(rank, extra)
    return offset, count


class ShardedMuca:
    """All ranks call every method collectively.

    engine_factory(L, n_walkers, seed, walker_offset) -> object with run_iteration / update_weights_with /
    set_log_weights / get_log_weights / get_energies / get_spins (default: the CUDA library binding `Muca`).
    """

    def __init__(self, L: int, n_walkers_total: int, seed: int, group=None, engine_factory=None):
        import torch.distributed as dist
        self._dist = dist
        self.group = group
        if dist.is_available() and dist.is_initialized():
            self.rank, self.world = dist.get_rank(group), dist.get_world_size(group)
        else:
            self.rank, self.world = 0, 1
        self.offset, self.count = shard_range(n_walkers_total, self.rank, self.world)
        if engine_factory is None:
            from .binding import Muca
            engine_factory = Muca
        self.engine = engine_factory(L, self.count, seed, self.offset)
        self.L, self.N, self.n_bins = L, L * L, L * L + 1
        self.n_walkers_total = n_walkers_total
        self.H_total = np.zeros(self.n_bins, dtype=np.uint64)

    def _allreduce_sum(self, H_local: np.ndarray) -> np.ndarray:
        if self.world == 1:
            return H_local.copy()
        import torch
        dist = self._dist
        t = torch.from_numpy(H_local.astype(np.int64))       # counts < 2^63
        backend = dist.get_backend(self.group)
        if backend == "nccl":
            t = t.cuda()
        dist.all_reduce(t, op=dist.ReduceOp.SUM, group=self.group)
        return t.cpu().numpy().astype(np.uint64)

    def run_iteration(self, therm_sweeps: int, sweeps: int) -> np.ndarray:
        H_local = self.engine.run_iteration(therm_sweeps, sweeps)
        self.H_total = self._allreduce_sum(np.asarray(H_local, dtype=np.uint64))
        return self.H_total

    def update_weights(self):
        self.engine.update_weights_with(self.H_total)

    def set_log_weights(self, logw):
        self.engine.set_log_weights(logw)

    def get_log_weights(self):
        return self.engine.get_log_weights()

    def get_energies(self):
        return self.engine.get_energies()

    def get_spins(self):
        return self.engine.get_spins()

    def close(self):
        if hasattr(self.engine, "close"):
            self.engine.close()
