"""Multi-GPU = replicas only: requests are independent, every GPU holds the whole
backbone and all task extensions and takes its own batch; there is no data-path collective.
The only cross-rank steps are the bench's barrier and the max-over-ranks of the device time.
Host logic only; covered by world_size-2 gloo tests on CPU (tests/test_replicas.py).
"""
import os

import torch
import torch.distributed as dist


def env_world():
    """(rank, local_rank, world_size) from the torchrun environment (1 process if unset)."""
    return int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0")), int(os.environ.get("WORLD_SIZE", "1"))


def init(backend=None):
    """Initialise torch.distributed when WORLD_SIZE > 1 (nccl on GPU boxes, gloo otherwise)."""
    rank, local_rank, world = env_world()
    if world > 1 and not dist.is_initialized():
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        os.environ.setdefault("MASTER_PORT", "29511")
        backend = backend or ("nccl" if torch.cuda.is_available() else "gloo")
        kw = {}
        if backend == "nccl":
            torch.cuda.set_device(local_rank)
            kw["device_id"] = torch.device("cuda", local_rank)
        dist.init_process_group(backend, rank=rank, world_size=world, **kw)
    return rank, local_rank, world


def barrier():
    if dist.is_initialized():
        dist.barrier()


def max_over_ranks(value: float, device=None) -> float:
    """MAX all-reduce of one float (device time in ms); identity for a single process."""
    if not dist.is_initialized():
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device or "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def sum_over_ranks(value: float, device=None) -> float:
    if not dist.is_initialized():
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device or "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return float(t.item())


def shard_requests(n_req: int, rank: int, world: int):
    """Contiguous slice of request indices rank `rank` serves when ONE batch is split across
    replicas (strong scaling helper; the bench uses weak scaling = one full batch per replica)."""
    base, rem = divmod(n_req, world)
    lo = rank * base + min(rank, rem)
    return lo, lo + base + (1 if rank < rem else 0)


def whole_job_throughput(units_per_rank: float, steps: int, ms_max: float, world: int) -> float:
    """Units all ranks processed / the max-over-ranks time."""
    return units_per_rank * world * steps / (ms_max * 1e-3)


def finalize():
    if dist.is_initialized():
        dist.destroy_process_group()
