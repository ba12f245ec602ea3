"""Multi-GPU host logic: the path shards with NO data-path exchange.

Every output D[d][t] is independent, and the paper's own multi-GPU suggestion is
"allocation of a sub-set of beams to each GPU".  One process per GPU; each rank
dedisperses its own beams with its own plan.  The only collective is the MAX of the per-rank step
time used for reporting (torch.distributed: NCCL on GPUs, gloo in the CPU tests).
"""
from __future__ import annotations

import os
from typing import List, Optional, Tuple

import torch
import torch.distributed as dist


def shard_beams(nbeams: int, world_size: int, rank: int) -> List[int]:
    """Contiguous, balanced split of beam indices 0..nbeams-1; ranks beyond nbeams get nothing."""
    if nbeams < 0 or world_size <= 0 or not (0 <= rank < world_size):
        raise ValueError("bad shard request")
    base, extra = divmod(nbeams, world_size)
    lo = rank * base + min(rank, extra)
    hi = lo + base + (1 if rank < extra else 0)
    return list(range(lo, hi))


def env_rank() -> Tuple[int, int, int]:
    """(rank, local_rank, world_size) from the torchrun environment (1 process when absent)."""
    return (int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0")),
            int(os.environ.get("WORLD_SIZE", "1")))


def init_process_group(backend: Optional[str] = None) -> bool:
    """Initialise torch.distributed from MASTER_ADDR/MASTER_PORT when WORLD_SIZE > 1.  Returns True if initialised."""
    rank, local_rank, world = env_rank()
    if world <= 1:
        return False
    if dist.is_initialized():
        return True
    os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
    if backend is None:
        backend = "nccl" if torch.cuda.is_available() else "gloo"
    kw = {}
    if backend == "nccl":
        torch.cuda.set_device(local_rank)
        kw["device_id"] = torch.device("cuda", local_rank)
    dist.init_process_group(backend=backend, rank=rank, world_size=world, **kw)
    return True


def barrier() -> None:
    if dist.is_available() and dist.is_initialized():
        dist.barrier()


def max_over_ranks(value: float) -> float:
    """MAX of a host scalar over all ranks (identity when not distributed)."""
    if not (dist.is_available() and dist.is_initialized()):
        return float(value)
    dev = "cuda" if dist.get_backend() == "nccl" else "cpu"
    t = torch.tensor([float(value)], dtype=torch.float64, device=dev)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def sum_over_ranks(value: float) -> float:
    if not (dist.is_available() and dist.is_initialized()):
        return float(value)
    dev = "cuda" if dist.get_backend() == "nccl" else "cpu"
    t = torch.tensor([float(value)], dtype=torch.float64, device=dev)
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return float(t.item())


def job_throughput(units_this_rank: float, ms_this_rank: float) -> Tuple[float, float]:
    """Whole-job throughput: units summed over ranks / the slowest rank's time.  -> (units_per_s, max_ms)."""
    total = sum_over_ranks(units_this_rank)
    ms = max_over_ranks(ms_this_rank)
    return (total / (ms * 1e-3) if ms > 0 else 0.0), ms
