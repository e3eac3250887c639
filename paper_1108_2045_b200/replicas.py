"""Replicas-only multi-GPU logic (the path has no exchange step).

Every rank solves its own independent problem; the only cross-rank traffic is the aggregation of the
timing for the bench line: the step time of the job is the MAX over ranks, the value is the units all
ranks processed divided by that time.  Backend-agnostic (nccl on GPUs, gloo in the CPU tests).
"""


def init(backend, device=None):
    """(rank, world) from the torchrun environment; initialises the process group when world > 1."""
    import os
    import torch.distributed as dist
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    if world > 1 and not dist.is_initialized():
        kw = {"device_id": device} if (device is not None and backend == "nccl") else {}
        dist.init_process_group(backend, **kw)
    return rank, world


def max_over_ranks(values, device="cpu"):
    """element-wise MAX over ranks of a list of floats (a no-op for a single process)."""
    import torch
    import torch.distributed as dist
    t = torch.tensor(list(values), dtype=torch.float64, device=device)
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(x) for x in t]


def barrier():
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        dist.barrier()


def job_value(units_per_rank_step, steps, world, total_ms_max):
    """whole-job throughput: units all ranks processed / max-over-ranks time (weak scaling)."""
    return units_per_rank_step * steps * world / (total_ms_max * 1e-3)
