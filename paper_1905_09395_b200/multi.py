"""One process per GPU: rank setup and the max-over-ranks timing reduction.

STEV shards over cells with no exchange step (cells are independent; the paper's own multi-device
version is future work), so there is NO data-path collective: torch.distributed is used only for the
barrier that brackets the timed region and for reducing times / counters to rank 0.  Backend: nccl on GPUs, gloo in
the CPU tests.
"""
from __future__ import annotations

import dataclasses
import os


@dataclasses.dataclass
class RankContext:
    rank: int
    world: int
    local_rank: int
    device: object
    backend: str | None


def init(n_gpus_requested: int = 1, backend: str | None = None) -> RankContext:
    """Reads RANK / LOCAL_RANK / WORLD_SIZE / MASTER_* (torchrun); a plain `python` launch is world 1."""
    import torch
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if world == 1 and n_gpus_requested > 1:
        raise SystemExit(f"--gpus {n_gpus_requested} needs one process per GPU: launch with "
                         f"python -m torch.distributed.run --nproc-per-node {n_gpus_requested} ...")
    use_cuda = torch.cuda.is_available() and backend != "gloo"
    device = torch.device(f"cuda:{local}") if use_cuda else torch.device("cpu")
    if use_cuda:
        torch.cuda.set_device(device)
    be = None
    if world > 1:
        import torch.distributed as dist
        be = backend or ("nccl" if use_cuda else "gloo")
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        os.environ.setdefault("MASTER_PORT", "29511")
        kw = {"device_id": device} if be == "nccl" else {}
        dist.init_process_group(backend=be, rank=rank, world_size=world, **kw)
    return RankContext(rank=rank, world=world, local_rank=local, device=device, backend=be)


def barrier(ctx: RankContext) -> None:
    if ctx.world > 1:
        import torch.distributed as dist
        dist.barrier()


def _reduce(ctx: RankContext, value: float, op: str) -> float:
    if ctx.world == 1:
        return value
    import torch
    import torch.distributed as dist
    t = torch.tensor([value], dtype=torch.float64, device=ctx.device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX if op == "max" else dist.ReduceOp.SUM)
    return float(t.item())


def max_over_ranks(ctx: RankContext, value: float) -> float:
    return _reduce(ctx, value, "max")


def sum_over_ranks(ctx: RankContext, value) -> int:
    return int(round(_reduce(ctx, float(value), "sum")))


def finish(ctx: RankContext) -> None:
    if ctx.world > 1:
        import torch.distributed as dist
        dist.barrier()
        dist.destroy_process_group()
