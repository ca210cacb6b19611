"""N>1 path on CPU: world_size-2 gloo run of the walker sharding + histogram all-reduce + Eq. (4).

The CUDA library cannot run here, so the per-rank engine is the CPU oracle behind the same interface
(tests may use the oracle); what is under test is the host logic of paper_1707_00919_b200/parallel.py:
the split, the global walker ids, the all-reduce and the identical weight update on every rank.
"""
import os
import sys

import numpy as np
import pytest
import torch.multiprocessing as mp

import muca_oracle as mo
from paper_1707_00919_b200.parallel import ShardedMuca, shard_range

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_shard_range_partitions_exactly():
    for n, world in ((16384, 8), (100, 3), (7, 7), (129, 2)):
        parts = [shard_range(n, r, world) for r in range(world)]
        assert parts[0][0] == 0 and sum(c for _, c in parts) == n
        for (o1, c1), (o2, _) in zip(parts, parts[1:]):
            assert o1 + c1 == o2
        assert max(c for _, c in parts) - min(c for _, c in parts) <= 1
    with pytest.raises(ValueError):
        shard_range(2, 0, 3)


class OracleEngine:
    def __init__(self, L, W, seed, offset):
        self.o = mo.Oracle(L, W, seed, walker_offset=offset)

    def run_iteration(self, t, s):
        return self.o.run_iteration(t, s)

    def update_weights_with(self, H):
        self.o.update_weights_with(H)

    def set_log_weights(self, w):
        self.o.set_log_weights(w)

    def get_log_weights(self):
        return self.o.get_log_weights()

    def get_energies(self):
        return self.o.get_energies()

    def get_spins(self):
        return self.o.get_spins()


def _worker(rank, world, port, out_dir):
    for p in (ROOT, os.path.join(ROOT, "oracle"), os.path.join(ROOT, "tests")):
        if p not in sys.path:
            sys.path.insert(0, p)
    import torch.distributed as dist
    dist.init_process_group("gloo", init_method=f"tcp://127.0.0.1:{port}", rank=rank, world_size=world)
    try:
        sm = ShardedMuca(16, 101, 170700919, engine_factory=OracleEngine)
        Hs = []
        for _ in range(3):
            Hs.append(sm.run_iteration(2, 12))
            sm.update_weights()
        np.savez(os.path.join(out_dir, f"r{rank}.npz"), H=np.stack(Hs), logw=sm.get_log_weights(),
                 E=sm.get_energies(), spins=sm.get_spins(), offset=sm.offset, count=sm.count)
    finally:
        dist.destroy_process_group()


def test_two_ranks_reproduce_the_single_process_run(tmp_path):
    port = 29500 + (os.getpid() % 2000)
    mp.spawn(_worker, args=(2, port, str(tmp_path)), nprocs=2, join=True)
    r0, r1 = np.load(tmp_path / "r0.npz"), np.load(tmp_path / "r1.npz")
    ref = mo.Oracle(16, 101, 170700919)
    Hs = []
    for _ in range(3):
        Hs.append(ref.run_iteration(2, 12))
        ref.update_weights()
    assert (int(r0["offset"]), int(r0["count"]), int(r1["offset"]), int(r1["count"])) == (0, 51, 51, 50)
    assert np.array_equal(r0["H"], np.stack(Hs)) and np.array_equal(r1["H"], r0["H"])       # summed histograms
    assert np.array_equal(r0["logw"], ref.get_log_weights()) and np.array_equal(r1["logw"], r0["logw"])
    assert np.array_equal(np.concatenate([r0["E"], r1["E"]]), ref.get_energies())
    assert np.array_equal(np.concatenate([r0["spins"], r1["spins"]]), ref.get_spins())


# ------------------------------------------------------------------------------------------------ the same with the CUDA library
def _gpu_worker(rank, world, port, out_dir, backend="gloo"):
    for p in (ROOT, os.path.join(ROOT, "oracle"), os.path.join(ROOT, "tests")):
        if p not in sys.path:
            sys.path.insert(0, p)
    import torch
    import torch.distributed as dist
    torch.cuda.set_device(rank % torch.cuda.device_count())     # one process per GPU where there are several
    dist.init_process_group(backend, init_method=f"tcp://127.0.0.1:{port}", rank=rank, world_size=world)
    try:
        sm = ShardedMuca(32, 301, 170700919)                    # default engine: the CUDA library binding
        Hs = []
        for _ in range(3):
            Hs.append(sm.run_iteration(2, 10))
            sm.update_weights()
        np.savez(os.path.join(out_dir, f"r{rank}.npz"), H=np.stack(Hs), logw=sm.get_log_weights(),
                 E=sm.get_energies(), spins=sm.get_spins(), offset=sm.offset, count=sm.count)
        sm.close()
    finally:
        dist.destroy_process_group()


@pytest.mark.gpu
@pytest.mark.parametrize("backend", ["gloo", "nccl"])
def test_two_ranks_with_the_cuda_library_reproduce_the_oracle(tmp_path, backend):
    # ShardedMuca with its default engine (libmuca_b200 through the binding) in two processes -- on two GPUs where the box
    # has them, otherwise both on cuda:0 --, histogram sum over gloo: global walker ids make the chains independent of
    # the split (R16), so the result is the single-process oracle's.  This is the path bench.py takes for --gpus N > 1.
    # The nccl variant (the all-reduce on device tensors, as bench.py runs it under torchrun) needs a GPU per rank: NCCL
    # refuses two ranks on one device, so on a one-GPU box it is skipped and only the gloo variant runs.
    import torch
    if backend == "nccl" and torch.cuda.device_count() < 2:
        pytest.skip("NCCL needs one GPU per rank; this box has one")
    port = 31500 + (os.getpid() % 2000) + (0 if backend == "gloo" else 2000)
    mp.spawn(_gpu_worker, args=(2, port, str(tmp_path), backend), nprocs=2, join=True)
    r0, r1 = np.load(tmp_path / "r0.npz"), np.load(tmp_path / "r1.npz")
    ref = mo.Oracle(32, 301, 170700919)
    Hs = []
    for _ in range(3):
        Hs.append(ref.run_iteration(2, 10, n_threads=mo.max_threads()))
        ref.update_weights()
    assert (int(r0["offset"]), int(r0["count"]), int(r1["offset"]), int(r1["count"])) == (0, 151, 151, 150)
    assert np.array_equal(r0["H"], np.stack(Hs)) and np.array_equal(r1["H"], r0["H"])
    assert np.max(np.abs(r0["logw"] - ref.get_log_weights())) <= 1e-12 and np.array_equal(r1["logw"], r0["logw"])
    assert np.array_equal(np.concatenate([r0["E"], r1["E"]]), ref.get_energies())
    assert np.array_equal(np.concatenate([r0["spins"], r1["spins"]]), ref.get_spins())
