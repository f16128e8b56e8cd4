"""Started by tests/test_abi_and_sharding.py through shard.torchrun_argv (the command bench.py --gpus N runs when
it has to spawn its own ranks): every rank joins a gloo group from the torchrun environment, the ranks take the
max of a per-rank time the way bench.py does, and rank 0 prints one JSON line."""
import json
import os
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

import torch.distributed as dist  # noqa: E402

from paper_2606_06386_b200 import shard  # noqa: E402

if __name__ == "__main__":
    dist.init_process_group("gloo")
    rank, world = dist.get_rank(), dist.get_world_size()
    ms = shard.max_over_ranks(10.0 + rank)
    lo, hi = shard.shard_bounds(1184, rank, world)
    dist.barrier()
    if rank == 0:
        print(json.dumps({"n_gpus": world, "ms": ms, "rate": shard.aggregate_rate(1184, world, ms), "first": [lo, hi],
                          "args": sys.argv[1:], "master": os.environ.get("MASTER_ADDR")}))
    dist.destroy_process_group()
