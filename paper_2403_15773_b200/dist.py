"""Multi-rank bookkeeping for the benchmark (torch.distributed plumbing only).

The timing protocol of the bench contract, for both multi-GPU modes of bench.py: "replicas only" (the
default: every rank steps its own copy of the workload, no data-path collective) and the z-slab
decomposition of ONE domain (slabs.py; the halo planes are pushed by the step kernels themselves).
What crosses ranks here: a barrier on both sides of the timed region, the MAX over ranks of the device
time, and the whole-job throughput = units processed by all ranks / that time.
Works with any backend (nccl on GPUs, gloo in the CPU tests).
"""
import torch
import torch.distributed as dist


def world():
    return dist.get_world_size() if dist.is_available() and dist.is_initialized() else 1


def barrier():
    if world() > 1:
        dist.barrier()


def max_over_ranks(value, device="cpu"):
    """MAX over ranks of a Python float (e.g. milliseconds measured with CUDA events)."""
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    if world() > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def sum_over_ranks(value, device="cpu"):
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    if world() > 1:
        dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return float(t.item())


def job_throughput(units_local, seconds_local, device="cpu"):
    """Whole-job throughput: all ranks' units divided by the slowest rank's time."""
    return sum_over_ranks(units_local, device) / max_over_ranks(seconds_local, device)
