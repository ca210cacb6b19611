"""paper_1707_00919_b200 -- B200-native hot path of parallel multicanonical simulation (arXiv 1707.00919).

The product is the C-ABI library ``libmuca_b200.so`` (include/muca.h; CUDA for sm_100a in csrc/).
This package is the thin Python binding: argument marshalling only, every step of the path runs in
the library.  PyTorch is used for device memory, streams and torch.distributed -- plumbing only.
"""
from .binding import Muca, MucaError, lib, lib_path, workspace_bytes, suggest_walkers, debug_philox, debug_philox_static, flatness, schedule  # noqa: F401
from .workloads import CONFIGS, Config, flips_per_iteration, total_flips  # noqa: F401
from .parallel import ShardedMuca, shard_range  # noqa: F401

__all__ = ["Muca", "MucaError", "lib", "lib_path", "workspace_bytes", "suggest_walkers", "debug_philox", "debug_philox_static", "flatness", "schedule", "CONFIGS", "Config",
           "flips_per_iteration", "total_flips", "ShardedMuca", "shard_range"]
