"""Multi-GPU plumbing: one process per GPU, DM trials sharded over ranks, NO data-path collective.

DM trials are independent time series ("5925 DM trials"), so the path shards by trial
(``inputs.shard_trials``): every rank owns a plan and its own planes; the only communication is the
barrier around the timed region, the max-over-ranks of the device time and the gather of the small
per-trial candidate counts.  ``torch.distributed`` (nccl on GPUs, gloo in the CPU tests) is used for
exactly that.
"""
from __future__ import annotations

import os
from dataclasses import dataclass


@dataclass
class Ctx:
    rank: int
    world: int
    local_rank: int
    backend: str
    active: bool   # a process group exists


def init_from_env(backend: str = "nccl") -> Ctx:
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if world <= 1:
        return Ctx(0, 1, 0, backend, False)
    import torch
    import torch.distributed as dist
    os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
    if backend == "nccl":
        torch.cuda.set_device(local)
        dist.init_process_group(backend="nccl", rank=rank, world_size=world,
                                device_id=torch.device("cuda", local))
    else:
        dist.init_process_group(backend=backend, rank=rank, world_size=world)
    return Ctx(rank, world, local, backend, True)


def _dev(ctx: Ctx):
    import torch
    return torch.device("cuda", ctx.local_rank) if ctx.backend == "nccl" else torch.device("cpu")


def barrier(ctx: Ctx):
    if ctx.active:
        import torch.distributed as dist
        dist.barrier()


def max_over_ranks(ctx: Ctx, value: float) -> float:
    if not ctx.active:
        return float(value)
    import torch
    import torch.distributed as dist
    t = torch.tensor([float(value)], dtype=torch.float64, device=_dev(ctx))
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def sum_over_ranks(ctx: Ctx, value: float) -> float:
    if not ctx.active:
        return value
    import torch
    import torch.distributed as dist
    t = torch.tensor([float(value)], dtype=torch.float64, device=_dev(ctx))
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    v = float(t.item())
    return int(round(v)) if isinstance(value, int) else v


def gather_dicts(ctx: Ctx, d: dict) -> dict:
    """Union of small per-rank dicts (e.g. trial -> candidate count) on every rank."""
    if not ctx.active:
        return dict(d)
    import torch.distributed as dist
    parts = [None] * ctx.world
    dist.all_gather_object(parts, d)
    out = {}
    for p in parts:
        out.update(p)
    return out


def finalize(ctx: Ctx):
    if ctx.active:
        import torch.distributed as dist
        dist.destroy_process_group()
