"""Multi-GPU plumbing of the CPRA loop: one process per GPU, no data-path collective.

The paper runs N_r independent random restarts of the whole loop and keeps the best (PAPER.md:64,
Step C; N_r = 100 in PAPER.md:104-106).  Restarts share the measured data and differ only in their
random initial phases, so they are the unit the path shards by: every rank runs its own restart(s)
of the full N_p-projection problem on its own GPU (weak scaling), the measured data is broadcast
once before the timed region, and the only cross-rank traffic inside a run is the timing reduction
(max over ranks) and the gather of the per-restart scalar errors that Step C ranks.  Sharding the
projections n of ONE restart across GPUs would need a halo exchange per mix; it
is not built.  Step C across ranks (`merge_across_ranks`): every rank keeps the N_l best of ITS restarts in
its own device bank (cpra_merge_offer); the N_l best of all ranks are then moved to rank 0 (point-to-point
sends of whole episodes, once per run, outside any timed region) and merged there by cpra_merge_finish.

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


def select_global_best(local_errors: Sequence[float], n_keep: int):
    """[(rank, slot, error)] of the n_keep lowest errors over all ranks' banks (ties: lower rank, lower slot).
    `local_errors`: this rank's bank errors in slot order (only the kept ones)."""
    mine = [float(e) for e in local_errors]
    if dist.is_initialized() and dist.get_world_size() > 1:
        allv = [None] * dist.get_world_size()
        dist.all_gather_object(allv, mine)
    else:
        allv = [mine]
    flat = [(e, r, s) for r, errs in enumerate(allv) for s, e in enumerate(errs)]
    flat.sort()
    return [(r, s, e) for e, r, s in flat[:max(0, int(n_keep))]]


def merge_across_ranks(plan, n_keep: int, n_ref: int = 0):
    """Step C over all ranks.  `plan` is each rank's Plan (or any object with merge_errors /
    merge_get / merge_begin / merge_offer / merge_finish) whose bank holds the best of that rank's restarts.
    The n_keep best episodes of all ranks are collected in rank 0's bank and merged there.
    Returns merge_finish's result on rank 0, None elsewhere."""
    rank = dist.get_rank() if dist.is_initialized() else 0
    E, cnt = plan.merge_errors()
    kept = int(cnt.reshape(-1)[0])
    errs = [float(x) for x in E.reshape(-1)[:kept].tolist()]
    chosen = select_global_best(errs, n_keep)
    # copy this rank's chosen episodes out of the bank before rank 0 re-uses its bank
    local = {s: plan.merge_get(s) for r, s, _ in chosen if r == rank}
    if rank == 0:
        plan.merge_begin(n_keep)
    for r, s, e in chosen:
        if r == 0:
            if rank == 0:
                plan.merge_offer(local[s], e)
        elif rank == r:
            dist.send(torch.view_as_real(local[s]).contiguous(), dst=0)
        elif rank == 0:
            buf = torch.empty_like(torch.view_as_real(next(iter(local.values())) if local else plan.merge_get(0)))
            dist.recv(buf, src=r)
            plan.merge_offer(torch.view_as_complex(buf), e)
    return plan.merge_finish(n_ref) if rank == 0 else None
