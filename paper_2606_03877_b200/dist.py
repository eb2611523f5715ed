"""Multi-GPU plumbing (S:Sec.8(e)): the render shards by VIEW -- rays and views are
independent problems and the scene (<= 320 MB) is replicated -- so there is no data-path collective.
One process per GPU; torch.distributed is used only for the rendezvous, the barrier around the
timed region and the max-over-ranks of the device times.  Pure host logic: testable with gloo on CPU.
"""
from __future__ import annotations

import os

import torch
import torch.distributed as dist


def env_rank_world() -> tuple[int, int, int]:
    """(rank, local_rank, world_size) from the torchrun environment; (0, 0, 1) when run plainly."""
    return (int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0")),
            int(os.environ.get("WORLD_SIZE", "1")))


def init(backend: str, device: torch.device | None = None) -> None:
    """Joins the process group described by RANK / WORLD_SIZE / MASTER_ADDR / MASTER_PORT."""
    if dist.is_initialized():
        return
    kw = {}
    if backend == "nccl" and device is not None:
        kw["device_id"] = device
    dist.init_process_group(backend, **kw)


def shutdown() -> None:
    if dist.is_initialized():
        dist.destroy_process_group()


def shard_range(n: int, rank: int, world: int) -> range:
    """Contiguous, balanced shard of n independent units (views, tile rows): sizes differ by at most
    one, every unit belongs to exactly one rank, empty when there are more ranks than units."""
    if n < 0 or world < 1 or not 0 <= rank < world:
        raise ValueError("bad shard arguments")
    lo = (n * rank) // world
    hi = (n * (rank + 1)) // world
    return range(lo, hi)


def barrier() -> None:
    if dist.is_initialized() and dist.get_world_size() > 1:
        dist.barrier()


def max_over_ranks(values: list[float], device: torch.device | str = "cpu") -> list[float]:
    """Element-wise maximum over all ranks (the job's time is its slowest rank's)."""
    t = torch.tensor(values, dtype=torch.float64, device=device)
    if dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(x) for x in t.cpu()]


def sum_over_ranks(values: list[float], device: torch.device | str = "cpu") -> list[float]:
    """Element-wise sum over all ranks (units processed by the whole job)."""
    t = torch.tensor(values, dtype=torch.float64, device=device)
    if dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return [float(x) for x in t.cpu()]


def render_views_sharded(render_batch, cams, gather: bool = True):
    """View-sharded render (S:Sec.8(e), Sec.8(f) NEXT-4): every rank renders its contiguous share of the batch of
    poses with `render_batch(cams_subset) -> tuple of tensors [v, ...]` (e.g. `Scene.render_batch` on its own
    replica of the scene) -- no collective on the data path.  With gather=True the shares are then assembled into
    the full batch on every rank by ONE all-gather of the output tensors (33 MB per 1080p rgba view); gather=False
    returns (this rank's views as a range, its outputs)."""
    rank, world = (dist.get_rank(), dist.get_world_size()) if dist.is_initialized() else (0, 1)
    n = len(cams)
    mine = shard_range(n, rank, world)
    outs = render_batch([cams[i] for i in mine]) if len(mine) else None
    if not gather or world == 1:
        return mine, outs
    sizes = [len(shard_range(n, r, world)) for r in range(world)]
    # shapes of one view's outputs from any rank that has a view (rank 0 always has one when n >= 1)
    meta = [None]
    if rank == 0:
        meta = [[(tuple(t.shape[1:]), t.dtype) if t is not None else None for t in outs]]
    dist.broadcast_object_list(meta, src=0)
    full = []
    for j, m in enumerate(meta[0]):
        if m is None:
            full.append(None)
            continue
        shape, dtype = m
        dev = outs[j].device if outs is not None else (torch.device("cuda", torch.cuda.current_device())
                                                        if dist.get_backend() == "nccl" else torch.device("cpu"))
        pad = torch.zeros((max(sizes),) + shape, dtype=dtype, device=dev)
        if outs is not None:
            pad[:len(mine)] = outs[j]
        parts = [torch.empty_like(pad) for _ in range(world)]
        dist.all_gather(parts, pad)
        full.append(torch.cat([parts[r][:sizes[r]] for r in range(world)], dim=0))
    return range(n), tuple(full)
