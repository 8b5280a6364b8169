"""Multi-GPU launch logic: replicas only.

Tracks are independent and the paper's own multi-GPU mode is one host thread per
device with no exchange, so there is no collective on the data path.  Under torchrun
every rank fits its own replica of the batch; the only communication is the barrier around the timed
region and the MAX-over-ranks of the device time.  Backend-agnostic (nccl on GPUs, gloo in the CPU
tests)."""
from __future__ import annotations

import os


def rank_world() -> tuple:
    """(rank, local_rank, world) from the torchrun environment; (0, 0, 1) when launched plainly."""
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", rank))
    return rank, local, world


def init(backend: str):
    """Join the process group named by the environment; returns torch.distributed or None (world 1)."""
    _, _, world = rank_world()
    if world <= 1:
        return None
    import torch.distributed as dist
    os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
    if not dist.is_initialized():
        dist.init_process_group(backend)
    return dist


def max_over_ranks(ms_local: float, dist, device=None) -> float:
    """Slowest rank's time: the job is done when the last replica is."""
    if dist is None:
        return float(ms_local)
    import torch
    t = torch.tensor([ms_local], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def job_throughput(n_tracks_per_rank: int, ms_local: float, dist, device=None) -> tuple:
    """Whole-job tracks/s = tracks fitted by all replicas / max-over-ranks time.  Ranks may carry
    different track counts (the count is summed), the time is the slowest rank's."""
    ms = max_over_ranks(ms_local, dist, device)
    if dist is None:
        total = int(n_tracks_per_rank)
    else:
        import torch
        c = torch.tensor([int(n_tracks_per_rank)], dtype=torch.int64, device=device)
        dist.all_reduce(c, op=dist.ReduceOp.SUM)
        total = int(c.item())
    return total / (ms * 1e-3), ms, total
