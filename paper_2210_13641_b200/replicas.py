"""Multi-GPU plumbing for replicas-only scaling: the hot path runs on one
GPU (BASELINE.json: "Everything runs on one GPU"), so N GPUs run N independent fields with no
data-path collective.  torch.distributed is used only for the timing barrier and for the
max-over-ranks / sum-over-ranks reductions of the reported numbers."""
import os

import torch
import torch.distributed as dist


def init_from_env(backend=None):
    """Join the process group torchrun described in the environment (no-op for world size 1)."""
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if world > 1 and not dist.is_initialized():
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        os.environ.setdefault("MASTER_PORT", "29500")
        if backend is None:
            backend = "nccl" if torch.cuda.is_available() else "gloo"
        kw = {}
        if backend == "nccl":
            torch.cuda.set_device(local_rank)
            kw["device_id"] = torch.device("cuda", local_rank)
        dist.init_process_group(backend=backend, rank=rank, world_size=world, **kw)
    return rank, local_rank, world


def barrier():
    if dist.is_initialized():
        dist.barrier()


def _reduce(value, op):
    if not dist.is_initialized():
        return float(value)
    dev = "cuda" if dist.get_backend() == "nccl" else "cpu"
    t = torch.tensor([float(value)], dtype=torch.float64, device=dev)
    dist.all_reduce(t, op=op)
    return float(t.item())


def max_over_ranks(value):
    return _reduce(value, dist.ReduceOp.MAX)


def sum_over_ranks(value):
    return _reduce(value, dist.ReduceOp.SUM)


def aggregate_throughput(units_this_rank, elapsed_s_this_rank):
    """Whole-job throughput of independent replicas: all units / the slowest rank's time."""
    total = sum_over_ranks(units_this_rank)
    t = max_over_ranks(elapsed_s_this_rank)
    return total / t if t > 0 else 0.0, total, t


def shutdown():
    if dist.is_initialized():
        dist.destroy_process_group()
