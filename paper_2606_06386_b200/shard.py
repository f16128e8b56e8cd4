"""Host-side logic of the multi-GPU form: the batch shards across ranks with no data-path collective
(every division is independent: one instance per block).  Nothing here touches
limbs; it is index arithmetic plus the max-over-ranks reduction of device times that bench.py reports.
Works on any torch.distributed backend (nccl on GPUs, gloo in the CPU tests)."""
from __future__ import annotations


def shard_bounds(batch: int, rank: int, world: int) -> tuple[int, int]:
    """Contiguous slice [lo, hi) of a batch of `batch` instances owned by `rank` of `world`:
    sizes differ by at most one, earlier ranks take the larger slices, the slices tile the batch."""
    if world < 1 or not (0 <= rank < world) or batch < 0:
        raise ValueError("bad shard request")
    base, extra = divmod(batch, world)
    lo = rank * base + min(rank, extra)
    return lo, lo + base + (1 if rank < extra else 0)


def rank_seed(seed: int, rank: int) -> int:
    """Seed of the batch a rank draws in the weak-scaling benchmark (each rank its own problems)."""
    return int(seed) + int(rank)


def max_over_ranks(value: float, device=None) -> float:
    """MAX all-reduce of a scalar (a device time in ms); identity when not distributed."""
    import torch
    import torch.distributed as dist

    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device if device is not None else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def aggregate_rate(units_per_rank: int, world: int, ms_max: float) -> float:
    """Whole-job throughput: units all ranks processed divided by the slowest rank's time."""
    return world * units_per_rank / (ms_max * 1e-3)


def free_port() -> int:
    import socket

    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    return port


def torchrun_argv(nproc: int, script: str, script_args, port: int | None = None, python: str | None = None) -> list:
    """Command line that starts `script` as `nproc` ranks of one node, one process per GPU, rendezvous on
    127.0.0.1 (the container hostname may not resolve): what `bench.py --gpus N` runs when it was not itself
    started under torchrun."""
    import sys

    if nproc < 1:
        raise ValueError("nproc must be >= 1")
    return [python or sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(int(nproc)),
            "--master-addr", "127.0.0.1", "--master-port", str(port if port is not None else free_port()),
            script] + list(script_args)
