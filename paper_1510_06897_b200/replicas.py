"""Multi-GPU plumbing of the benchmark: the overlap path on one lattice does not shard without a halo exchange per
stencil application, so N GPUs run N independent replicas -- one process per GPU, each with
its own right-hand side (propagator-style workload), no data-path collective.  torch.distributed carries only the
barrier and the max-over-ranks of the device time (NCCL on GPUs; gloo in the CPU tests).  No method arithmetic here."""
from __future__ import annotations

import os


def world():
    """(rank, local_rank, world_size) from the torchrun environment (1 process = 1 GPU)."""
    return (int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0")),
            int(os.environ.get("WORLD_SIZE", "1")))


def rhs_seed_offset(rank: int) -> int:
    """Replica r applies the operator to its own seeded right-hand side: seed offset r (0 keeps the N = 1 inputs)."""
    return int(rank)


def max_over_ranks(value: float, dist=None, device="cpu") -> float:
    """MAX all-reduce of a per-rank scalar (the timed region's milliseconds); identity without a process group."""
    if dist is None:
        return float(value)
    import torch
    t = torch.tensor([float(value)], device=device, dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def aggregate_rate(units_per_rank: float, ms_local: float, world_size: int, dist=None, device="cpu"):
    """Whole-job throughput of a weak-scaling replica run: every rank processed `units_per_rank` units in its own
    `ms_local`; the job took the slowest rank's time.  Returns (units/s over all ranks, max ms)."""
    ms = max_over_ranks(ms_local, dist, device)
    return world_size * units_per_rank / (ms * 1e-3), ms
