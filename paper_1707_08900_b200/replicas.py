"""Host-side bookkeeping of the "replicas only" multi-GPU mode.

The path of north_star runs on one GPU: with N ranks every rank advances its own copy of the workload and
nothing of the data path crosses ranks.  What the ranks do share is the timing protocol of bench.py: a barrier on
both sides of the timed region, the MAX over ranks of the device time, and value = cells of all ranks x steps /
that time.  These helpers hold that logic so that it can be tested on CPU with the gloo backend (world size 2).
No method arithmetic lives here.
"""
import torch
import torch.distributed as dist


def world():
    """(rank, world_size) of the initialised process group, (0, 1) without one."""
    if dist.is_available() and dist.is_initialized():
        return dist.get_rank(), dist.get_world_size()
    return 0, 1


def barrier(device=None):
    """Rendezvous of all ranks, then a device synchronize when a CUDA device is given."""
    if world()[1] > 1:
        dist.barrier()
    if device is not None and torch.device(device).type == "cuda":
        torch.cuda.synchronize(device)


def max_over_ranks(ms, device="cpu"):
    """MAX over ranks of a per-rank device time in milliseconds (every rank gets the result)."""
    t = torch.tensor([float(ms)], dtype=torch.float64, device=device)
    if world()[1] > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_value(cells_per_rank, steps, ms_max, world_size):
    """Mcell-updates/s of the whole job: every rank advanced cells_per_rank cells by `steps` full RK3 steps
    within the slowest rank's ms_max milliseconds (weak scaling: per-rank work is fixed)."""
    if ms_max <= 0:
        raise ValueError("ms_max must be positive")
    return world_size * cells_per_rank * steps / (ms_max * 1e-3) / 1e6
