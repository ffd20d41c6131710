"""Multi-GPU host logic: replicas over independent initial states (no data-path collective).

The path shards by state only: "random initial states are distributed over MPI processes" (section 2.4.2);
every rank holds a replica of H and propagates its own seeded states.  Nothing is exchanged during propagation; the only
collectives are the timing reduction (max over ranks) and, when a caller wants all correlation functions in one place, a
gather of corr[n_state][n_step] (kilobytes).  torch.distributed is plumbing here (nccl on the GPUs, gloo in the CPU tests);
this module holds none of the method's arithmetic and works on CPU tensors as well as CUDA tensors.
"""
from __future__ import annotations

import os
from dataclasses import dataclass
from typing import List, Optional

import torch
import torch.distributed as dist


@dataclass(frozen=True)
class Shard:
    rank: int
    world: int
    first_state: int     # index of this rank's first state in the global seeded sequence (sub-stream id of psi0 / LDOS site index)
    n_state: int         # states this rank propagates


def env_rank_world():
    return int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1")), int(os.environ.get("LOCAL_RANK", "0"))


def weak_shard(n_state_per_rank: int, rank: int, world: int) -> Shard:
    """Weak scaling (bench.py): per-rank work fixed, rank r takes global states [r*B, (r+1)*B)."""
    assert 0 <= rank < world and n_state_per_rank >= 0
    return Shard(rank, world, rank * n_state_per_rank, n_state_per_rank)


def strong_shard(n_state_total: int, rank: int, world: int) -> Shard:
    """Strong scaling: a fixed set of states split as evenly as possible, the first (total % world) ranks take one more."""
    assert 0 <= rank < world and n_state_total >= 0
    q, r = divmod(n_state_total, world)
    n = q + (1 if rank < r else 0)
    first = rank * q + min(rank, r)
    return Shard(rank, world, first, n)


def _active() -> bool:
    return dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1


def barrier(device: Optional[torch.device] = None) -> None:
    if device is not None and device.type == "cuda":
        torch.cuda.synchronize(device)
    if _active():
        dist.barrier()
    if device is not None and device.type == "cuda":
        torch.cuda.synchronize(device)


def max_over_ranks(values: List[float], device="cpu") -> List[float]:
    """Element-wise max over ranks of a short list of device-measured times."""
    t = torch.tensor(values, dtype=torch.float64, device=device)
    if _active():
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(v) for v in t.cpu()]


def sum_over_ranks(values: List[float], device="cpu") -> List[float]:
    t = torch.tensor(values, dtype=torch.float64, device=device)
    if _active():
        dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return [float(v) for v in t.cpu()]


def whole_job_rate(local_units: float, local_seconds: float, device="cpu") -> float:
    """Units all ranks processed / max-over-ranks time (the bench contract's `value`)."""
    total = sum_over_ranks([local_units], device)[0]
    worst = max_over_ranks([local_seconds], device)[0]
    return total / worst if worst > 0 else float("nan")


def gather_corr(corr: torch.Tensor, shard: Shard) -> Optional[torch.Tensor]:
    """All ranks' corr[n_state_r][n_step] stacked in global state order on rank 0 (None elsewhere).  Ragged shards allowed."""
    if not _active():
        return corr
    counts = [torch.zeros(1, dtype=torch.int64, device=corr.device) for _ in range(shard.world)]
    dist.all_gather(counts, torch.tensor([corr.shape[0]], dtype=torch.int64, device=corr.device))
    n_max = max(int(c) for c in counts)
    pad = torch.zeros((n_max,) + tuple(corr.shape[1:]), dtype=corr.dtype, device=corr.device)
    pad[: corr.shape[0]] = corr
    # complex tensors travel as (re, im) pairs: not every backend reduces/gathers complex dtypes
    buf = torch.view_as_real(pad).contiguous() if pad.is_complex() else pad
    parts = [torch.empty_like(buf) for _ in range(shard.world)]
    dist.all_gather(parts, buf)
    if shard.rank != 0:
        return None
    out = []
    for c, p in zip(counts, parts):
        p = torch.view_as_complex(p) if corr.is_complex() else p
        out.append(p[: int(c)])
    return torch.cat(out, dim=0)
