"""Multi-GPU plumbing: independent replicas, one process per GPU, no data-path collective.

The paper's parameter-level parallelism (rotational averages, pathways, delay
times are independent propagations).  torch.distributed is used for the barrier and the
max-over-ranks reduction of the timing only; works with nccl (GPU) and gloo (CPU tests).
"""
import numpy as np


def replica_sigma0(w, rank):
    """Initial matrix of replica `rank`: the excitation starts on site (rank mod N)."""
    s = np.zeros((w.N, w.N), dtype=np.complex128)
    s[rank % w.N, rank % w.N] = 1.0
    return s


def barrier(world):
    if world > 1:
        import torch.distributed as dist
        dist.barrier()


def max_over_ranks(value, world):
    """MAX-reduce a python float over all ranks (device tensor for nccl, cpu tensor for gloo)."""
    if world <= 1:
        return float(value)
    import torch
    import torch.distributed as dist
    dev = "cuda" if dist.get_backend() == "nccl" else "cpu"
    t = torch.tensor([float(value)], dtype=torch.float64, device=dev)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def aggregate_throughput(units_per_rank, seconds_per_rank, world):
    """Whole-job value: units all ranks processed / max-over-ranks time."""
    return units_per_rank * world / max_over_ranks(seconds_per_rank, world)
