"""Multi-GPU plumbing.  Two ways to use N GPUs, both without a reduction:

  * independent units (the default of bench.py --gpus N): a unit is one observation dedispersed over the whole
    DM grid -- the way the paper runs its four antenna streams side by side.  Every rank owns
    whole units; no collective touches the data.
  * ONE observation split by DM rows: DM trials are independent, so rank r computes the
    contiguous row range `shard_rows(ndm, r, world)` with a plan made by ddsp_plan_create_rows (d_max over the
    whole list, so every shard has the same nsamp_out); the only exchange step is ONE broadcast of the input
    from the rank that holds it (`broadcast_input`: NCCL over NVLink / NVSwitch on GPUs), outputs stay sharded.

`torch.distributed` also provides the barrier around the timed region and the max-over-ranks of the device
time.  Works with backend "nccl" (one process per GPU) and "gloo" (CPU tests).
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


def shard_rows(ndm, rank, world):
    """(row_begin, row_count) of rank `rank` when `ndm` DM rows are split into contiguous, balanced ranges
    (row_count may be 0 when there are more ranks than rows)."""
    r = shard_units(ndm, rank, world)
    return r.start, len(r)


def broadcast_input(x, src=0):
    """The one exchange step of the DM-row split: the filterbank of rank `src` is copied into every rank's `x`
    (same shape and dtype everywhere), in place.  NCCL for CUDA tensors, gloo for CPU tensors."""
    if dist.is_initialized() and dist.get_world_size() > 1:
        dist.broadcast(x, src=src)
    return x


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
