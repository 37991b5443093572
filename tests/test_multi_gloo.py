"""The N>1 host logic on CPU: world-size-2 gloo.  Cells shard over ranks with no data-path collective
(DESIGN.md section 9); what needs checking is that the interleaved shards tile the global field exactly once and that
the max-over-ranks / sum-over-ranks reductions bench.py relies on behave."""
import os
import socket

import numpy as np


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank: int, world: int, port: int, out_dir: str):
    os.environ.update(RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE=str(world), MASTER_ADDR="127.0.0.1",
                      MASTER_PORT=str(port))
    from paper_1905_09395_b200 import multi
    from stev_inputs.configs import make_workload
    ctx = multi.init(world, backend="gloo")
    assert ctx.rank == rank and ctx.world == world and ctx.backend == "gloo"
    n_per_rank = 3 * 4096
    w = make_workload(1, n_per_rank, rank=rank, world=world, weak=True)
    assert w.n_cells == n_per_rank
    multi.barrier(ctx)
    t_max = multi.max_over_ranks(ctx, 10.0 + rank)
    total = multi.sum_over_ranks(ctx, w.n_cells)
    np.savez(os.path.join(out_dir, f"rank{rank}.npz"), T=w.T, Y=w.Y, blocks=w.blocks, t_max=t_max, total=total)
    multi.finish(ctx)


def test_two_ranks_shard_the_field_without_overlap(tmp_path):
    import torch.multiprocessing as mp
    from stev_inputs.configs import make_workload
    world, port = 2, _free_port()
    mp.spawn(_worker, args=(world, port, str(tmp_path)), nprocs=world, join=True)
    r = [np.load(tmp_path / f"rank{k}.npz") for k in range(world)]
    assert float(r[0]["t_max"]) == float(r[1]["t_max"]) == 11.0          # max over ranks, same on every rank
    assert int(r[0]["total"]) == int(r[1]["total"]) == 2 * 3 * 4096      # sum over ranks
    assert sorted(np.concatenate([r[0]["blocks"], r[1]["blocks"]]).tolist()) == list(range(6))
    assert r[0]["blocks"].tolist() == [0, 2, 4] and r[1]["blocks"].tolist() == [1, 3, 5]  # interleaved
    full = make_workload(1, 6 * 4096)                                   # the same global field in one process
    for k in range(world):
        for pos, b in enumerate(r[k]["blocks"]):
            sl = slice(int(b) * 4096, (int(b) + 1) * 4096)
            np.testing.assert_array_equal(r[k]["T"][pos * 4096:(pos + 1) * 4096], full.T[sl])
            np.testing.assert_array_equal(r[k]["Y"][:, pos * 4096:(pos + 1) * 4096], full.Y[:, sl])


def test_single_process_context_is_world_one():
    from paper_1905_09395_b200 import multi
    for k in ("RANK", "WORLD_SIZE", "LOCAL_RANK"):
        os.environ.pop(k, None)
    ctx = multi.init(1, backend="gloo")
    assert (ctx.rank, ctx.world) == (0, 1)
    assert multi.max_over_ranks(ctx, 3.5) == 3.5 and multi.sum_over_ranks(ctx, 7) == 7
    multi.barrier(ctx)
    multi.finish(ctx)
