"""Multi-GPU plumbing of the CPRA loop: one process per GPU, no data-path collective.

The paper runs N_r independent random restarts of the whole loop and keeps the best (PAPER.md:64,
Step C; N_r = 100 in PAPER.md:104-106).  Restarts share the measured data and differ only in their
random initial phases, so they are the unit the path shards by: every rank runs its own restart(s)
of the full N_p-projection problem on its own GPU (weak scaling), the measured data is broadcast
once before the timed region, and the only cross-rank traffic inside a run is the timing reduction
(max over ranks) and the gather of the per-restart scalar errors that Step C ranks.  Sharding the
projections n of ONE restart across GPUs would need a halo exchange per mix; it
is not built.

`torch.distributed` only (NCCL on GPUs, gloo in the CPU tests); nothing here touches the kernels."""
from __future__ import annotations

import os
from typing import List, Sequence

import torch
import torch.distributed as dist


def env_world():
    """(rank, local_rank, world_size) from the torchrun environment (1 process if absent)."""
    return (int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0")),
            int(os.environ.get("WORLD_SIZE", "1")))


def init(backend: str | None = None) -> tuple[int, int, int]:
    """Initialise the default process group when WORLD_SIZE > 1.  Returns (rank, local_rank, world)."""
    rank, local_rank, world = env_world()
    if world > 1 and not dist.is_initialized():
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        os.environ.setdefault("MASTER_PORT", "29511")
        if backend is None:
            backend = "nccl" if torch.cuda.is_available() else "gloo"
        if backend == "nccl":
            torch.cuda.set_device(local_rank)
            dist.init_process_group(backend, rank=rank, world_size=world,
                                    device_id=torch.device("cuda", local_rank))
        else:
            dist.init_process_group(backend, rank=rank, world_size=world)
    return rank, local_rank, world


def shutdown():
    if dist.is_initialized():
        dist.destroy_process_group()


def restarts_of_rank(n_restarts: int, rank: int, world: int) -> List[int]:
    """Restart ids (seeds of the random initial phases) this rank runs: contiguous blocks, the
    first n_restarts % world ranks take one more."""
    if n_restarts < 0 or world < 1 or not 0 <= rank < world:
        raise ValueError("bad restart partition")
    base, extra = divmod(n_restarts, world)
    lo = rank * base + min(rank, extra)
    return list(range(lo, lo + base + (1 if rank < extra else 0)))


def broadcast_arrays(tensors: Sequence[torch.Tensor], src: int = 0) -> None:
    """Broadcast the measured data (intensities, masks, supports) from `src`, in place."""
    if dist.is_initialized() and dist.get_world_size() > 1:
        for t in tensors:
            dist.broadcast(t, src)


def barrier(device=None):
    if dist.is_initialized() and dist.get_world_size() > 1:
        if device is not None and torch.device(device).type == "cuda":
            dist.barrier(device_ids=[torch.device(device).index])
        else:
            dist.barrier()


def max_over_ranks(value: float, device="cpu") -> float:
    """The slowest rank's time: every multi-GPU number is the max over ranks."""
    if not (dist.is_initialized() and dist.get_world_size() > 1):
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def sum_over_ranks(value: float, device="cpu") -> float:
    if not (dist.is_initialized() and dist.get_world_size() > 1):
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return float(t.item())


def gather_restart_errors(errors: Sequence[float], restart_ids: Sequence[int], device="cpu"):
    """All ranks' (restart id, global error) pairs, sorted by error: the ranking Step C starts
    from ("episodes with the lowest reconstruction error").  Returns a list of
    (restart id, error) on every rank."""
    pairs = [(int(i), float(e)) for i, e in zip(restart_ids, errors)]
    if dist.is_initialized() and dist.get_world_size() > 1:
        out = [None] * dist.get_world_size()
        dist.all_gather_object(out, pairs)
        pairs = [p for chunk in out for p in chunk]
    return sorted(pairs, key=lambda p: (p[1], p[0]))
