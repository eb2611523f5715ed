"""Host-side multi-process logic (S:Sec.8(e)): world_size-2 gloo on CPU.  The render needs no
collective; what is covered is the view sharding and the max/sum-over-ranks of the bench numbers."""
import os
import socket

import pytest
import torch
import torch.multiprocessing as mp

from paper_2606_03877_b200 import dist as msdist


def test_shard_range_partitions_every_count():
    for world in (1, 2, 3, 4, 8):
        for n in (0, 1, 2, 7, 8, 9, 64):
            seen = []
            sizes = []
            for r in range(world):
                sh = msdist.shard_range(n, r, world)
                seen += list(sh)
                sizes.append(len(sh))
            assert seen == list(range(n))                  # contiguous, disjoint, complete, ordered
            assert max(sizes) - min(sizes) <= 1            # balanced
    with pytest.raises(ValueError):
        msdist.shard_range(4, 2, 2)


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank: int, world: int, port: int, n_views: int, out):
    os.environ.update(RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE=str(world),
                      MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    assert msdist.env_rank_world() == (rank, rank, world)
    msdist.init("gloo")
    mine = msdist.shard_range(n_views, rank, world)
    msdist.barrier()
    ms = 10.0 + 5.0 * rank                                  # this rank's device time
    t_max, = msdist.max_over_ranks([ms])
    units, = msdist.sum_over_ranks([float(len(mine))])
    out.put((rank, list(mine), t_max, units))
    msdist.barrier()
    msdist.shutdown()


@pytest.mark.timeout(120)
def test_two_ranks_shard_views_and_reduce_times():
    world, n_views = 2, 8                                   # CFG5: 8 poses
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, n_views, out)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(out.get(timeout=100) for _ in range(world))
    for p in procs:
        p.join(timeout=30)
        assert p.exitcode == 0
    assert res[0][1] + res[1][1] == list(range(n_views))
    assert all(r[2] == 15.0 for r in res)                   # max over ranks, identical on every rank
    assert all(r[3] == float(n_views) for r in res)         # whole-job units


def _render_worker(rank: int, world: int, port: int, out):
    """Each rank renders its share of CFG5's 8 poses (shrunk) -- here with the CPU oracle standing in for the GPU
    replica -- and the shares are assembled by render_views_sharded's single all-gather."""
    import numpy as np
    from oracle import mso
    from paper_2606_03877_b200 import synth
    os.environ.update(RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE=str(world),
                      MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    msdist.init("gloo")
    cfg = synth.shrink(synth.CONFIGS["cfg5"], 24, 14)
    sc, cams = synth.make_scene(cfg), synth.make_cameras(cfg)
    orc = mso.OracleScene(sc)

    def render_batch(sub):
        r = [orc.render(c, cfg.height, cfg.width, 4, n_threads=2) for c in sub]
        return (torch.from_numpy(np.stack([x[0] for x in r])), torch.from_numpy(np.stack([x[1] for x in r])),
                torch.from_numpy(np.stack([x[2] for x in r])))

    views, full = msdist.render_views_sharded(render_batch, cams)
    mine, part = msdist.render_views_sharded(render_batch, cams, gather=False)
    ref = render_batch(cams) if rank == 0 else None
    ok = True
    if rank == 0:
        ok = all(torch.equal(a, b) for a, b in zip(full, ref))
    ok = ok and list(views) == list(range(len(cams))) and all(
        torch.equal(p, f[mine.start:mine.stop]) for p, f in zip(part, full))
    out.put((rank, list(mine), bool(ok)))
    msdist.barrier()
    msdist.shutdown()


@pytest.mark.timeout(300)
@pytest.mark.parametrize("world", [2, 3])
def test_view_sharded_render_equals_the_single_rank_batch_bitwise(world):
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_render_worker, args=(r, world, port, out)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(out.get(timeout=280) for _ in range(world))
    for p in procs:
        p.join(timeout=30)
        assert p.exitcode == 0
    assert sum((r[1] for r in res), []) == list(range(8))    # the shards partition CFG5's 8 poses
    assert all(r[2] for r in res)                            # gathered batch == single-rank batch, bitwise
