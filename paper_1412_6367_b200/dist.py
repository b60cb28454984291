"""Host-side plumbing for running N independent replicas, one process per GPU.

Frames are independent ("working with multiple detectors simultaneously"), so the path shards by frame
with NO data-path collective: each rank owns a contiguous block of the frame stream and its own copy of the matrix.
torch.distributed is used only for the start/stop barrier and for the max-over-ranks of the device time.
"""
from __future__ import annotations

import os


def env_world():
    """(rank, local_rank, world_size) from the torchrun environment (1-process defaults)."""
    return (int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0")),
            int(os.environ.get("WORLD_SIZE", "1")))


def shard_frames(total_frames: int, rank: int, world_size: int):
    """Contiguous block [start, stop) of the frame stream owned by `rank`; blocks differ by at most one frame."""
    if world_size < 1 or not (0 <= rank < world_size) or total_frames < 0:
        raise ValueError("bad shard arguments")
    base, extra = divmod(total_frames, world_size)
    start = rank * base + min(rank, extra)
    return start, start + base + (1 if rank < extra else 0)


def init(backend: str | None = None):
    """Initialise the default process group when launched under torchrun with WORLD_SIZE > 1; returns
    (rank, local_rank, world_size)."""
    rank, local_rank, world = env_world()
    if world > 1:
        import torch
        import torch.distributed as dist
        if not dist.is_initialized():
            os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
            os.environ.setdefault("MASTER_PORT", "29511")
            if backend is None:
                backend = "nccl" if torch.cuda.is_available() else "gloo"
            dist.init_process_group(backend=backend, rank=rank, world_size=world)
    return rank, local_rank, world


def barrier():
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized():
        dist.barrier()


def reduce_scalar(value: float, op: str = "max", device=None) -> float:
    """max / sum of a host scalar over all ranks (identity for a single process)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()):
        return float(value)
    if device is None:
        device = torch.device("cuda", torch.cuda.current_device()) if dist.get_backend() == "nccl" else "cpu"
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX if op == "max" else dist.ReduceOp.SUM)
    return float(t.item())


def aggregate_throughput(units_this_rank: float, ms_this_rank: float):
    """Whole-job throughput: units processed by all ranks / max-over-ranks time.  Returns (units/s, ms)."""
    total_units = reduce_scalar(units_this_rank, "sum")
    ms = reduce_scalar(ms_this_rank, "max")
    return (total_units / (ms * 1e-3) if ms > 0 else 0.0), ms


def finalize():
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized():
        dist.destroy_process_group()
