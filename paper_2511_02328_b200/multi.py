"""Multi-GPU plumbing: the path shards by independent units with NO data-path
collective.  A unit is one observation (one filterbank dedispersed over the whole DM grid) -- the way
the paper runs its four antenna streams side by side -- so every rank owns whole units
and `torch.distributed` is used only for the barrier around the timed region and for the max-over-
ranks of the device time.  Works with backend "nccl" (one process per GPU) and "gloo" (CPU tests).
"""
import os

import torch
import torch.distributed as dist


def env_world():
    """(rank, local_rank, world_size) from the torchrun environment (1 process if absent)."""
    return (int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0")),
            int(os.environ.get("WORLD_SIZE", "1")))


def init(backend=None):
    """Initialise the default process group when launched under torchrun; no-op for one process."""
    rank, local_rank, world = env_world()
    if world > 1 and not dist.is_initialized():
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        os.environ.setdefault("MASTER_PORT", "29500")
        if backend is None:
            backend = "nccl" if torch.cuda.is_available() else "gloo"
        dist.init_process_group(backend=backend, rank=rank, world_size=world)
    return rank, local_rank, world


def shard_units(n_units, rank, world):
    """Contiguous, balanced ownership of `n_units` independent units: the slice of rank `rank`."""
    if not (0 <= rank < world) or n_units < 0:
        raise ValueError("bad shard request")
    base, rem = divmod(n_units, world)
    lo = rank * base + min(rank, rem)
    return range(lo, lo + base + (1 if rank < rem else 0))


def barrier():
    if dist.is_initialized():
        dist.barrier()


def _device():
    if dist.is_initialized() and dist.get_backend() == "nccl":
        return torch.device("cuda", torch.cuda.current_device())
    return torch.device("cpu")


def max_over_ranks(value):
    """Max of a float over all ranks (the job's time is the slowest rank's device time)."""
    if not dist.is_initialized():
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=_device())
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def sum_over_ranks(value):
    """Sum of a float over all ranks (units of work processed by the whole job)."""
    if not dist.is_initialized():
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=_device())
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return float(t.item())


def job_throughput(units_this_rank, seconds_this_rank):
    """Whole-job throughput: units all ranks processed / max-over-ranks time."""
    total = sum_over_ranks(units_this_rank)
    t = max_over_ranks(seconds_this_rank)
    return total / t, t


def finalize():
    if dist.is_initialized():
        dist.destroy_process_group()
