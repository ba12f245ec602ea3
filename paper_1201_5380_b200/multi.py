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


# ---- the other two exchange-free splits ----------------------------

def shard_dm_slabs(ndm: int, world_size: int, rank: int, align: int = 16) -> Tuple[int, int]:
    """DM slab [lo, hi) of rank `rank`: contiguous (a rank's delay spread stays compact), balanced in units of
    `align` trials (the kernel's DM block), the last slab taking the ragged rest.  The input is replicated, the
    outputs are disjoint rows: no exchange.  Ranks beyond the number of blocks get an empty slab."""
    if ndm < 0 or world_size <= 0 or align <= 0 or not (0 <= rank < world_size):
        raise ValueError("bad shard request")
    nblk = -(-ndm // align)
    base, extra = divmod(nblk, world_size)
    lo = rank * base + min(rank, extra)
    hi = lo + base + (1 if rank < extra else 0)
    return min(lo * align, ndm), min(hi * align, ndm)


def shard_time_slabs(nsamps: int, world_size: int, rank: int, max_delay: int, align: int = 128) -> Tuple[int, int, int, int]:
    """Time slab of rank `rank` ("time-division multiplexing"): output samples [t_lo, t_hi) and the
    input samples [t_lo, in_hi) it reads, in_hi = t_hi + max_delay -- a halo of max_delay samples that the next
    rank reads too, so nothing is exchanged.  Slab starts are multiples of `align` samples (128 keeps the start of a
    2-bit row slab 16-byte aligned for the bulk copies).  -> (t_lo, t_hi, t_lo, in_hi)."""
    if nsamps < 0 or world_size <= 0 or align <= 0 or max_delay < 0 or not (0 <= rank < world_size):
        raise ValueError("bad shard request")
    nunits = -(-nsamps // align)
    base, extra = divmod(nunits, world_size)
    lo = rank * base + min(rank, extra)
    hi = lo + base + (1 if rank < extra else 0)
    t_lo, t_hi = min(lo * align, nsamps), min(hi * align, nsamps)
    return t_lo, t_hi, t_lo, (t_hi + max_delay if t_hi > t_lo else t_lo)


def gather_dm_rows(local_rows: torch.Tensor, ndm: int, world_size: int, align: int = 16) -> torch.Tensor:
    """Optional assembly of the whole transform on every rank from DM slabs (only when one consumer wants all of
    it; the transform itself needs no collective): all_gather of the slabs, padded to the largest one.
    local_rows: [hi - lo, nsamps] of this rank's slab (shard_dm_slabs).  -> [ndm, nsamps]."""
    if not (dist.is_available() and dist.is_initialized()):
        return local_rows
    bounds = [shard_dm_slabs(ndm, world_size, r, align) for r in range(world_size)]
    most = max(hi - lo for lo, hi in bounds)
    nsamps = local_rows.shape[1]
    pad = torch.zeros((most, nsamps), dtype=local_rows.dtype, device=local_rows.device)
    pad[: local_rows.shape[0]] = local_rows
    parts = [torch.empty_like(pad) for _ in range(world_size)]
    dist.all_gather(parts, pad)
    return torch.cat([parts[r][: hi - lo] for r, (lo, hi) in enumerate(bounds)], dim=0)
