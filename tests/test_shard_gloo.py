"""The N>1 host logic on CPU: world_size-2 gloo group, contiguous exposure shards that
cover the batch exactly once, max/sum over ranks as bench.py uses them, and shard-wise
results equal to the unsharded result (the oracle stands in for the kernels here: the
data path has no collective, so sharding must not change a single pixel)."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

import dfr_synth as S
from paper_2505_03932_b200.shard import max_over_ranks, shard_range, sum_over_ranks


def test_shard_range_covers_once():
    for n in (1, 2, 5, 32, 33, 1024):
        for world in (1, 2, 3, 8):
            got = [k for r in range(world) for k in shard_range(n, world, r)]
            assert got == list(range(n))
            sizes = [len(shard_range(n, world, r)) for r in range(world)]
            assert max(sizes) - min(sizes) <= 1
    with pytest.raises(ValueError):
        shard_range(4, 2, 2)


def _worker(rank, world, port, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import oracle
    w = S.config2(batch=3, n=96, nstars=20)
    mine = shard_range(3, world, rank)
    out = oracle.reproject(w.images[mine.start:mine.stop], w.src_wcs[mine.start:mine.stop], w.tgt_wcs,
                           w.shape_out, 1) if len(mine) else np.zeros((0, 96, 96), np.float32)
    dist.barrier()
    elapsed = 1.0 + rank                                  # pretend timings
    mx = max_over_ranks(elapsed)
    units = sum_over_ranks(float(len(mine)))
    gathered = [None] * world
    dist.all_gather_object(gathered, (mine.start, out))
    if rank == 0:
        full = np.concatenate([g[1] for g in sorted(gathered, key=lambda t: t[0])])
        ref = oracle.reproject(w.images, w.src_wcs, w.tgt_wcs, w.shape_out, 1)
        q.put((mx, units, bool(np.array_equal(np.nan_to_num(full, nan=-1), np.nan_to_num(ref, nan=-1)))))
    dist.destroy_process_group()


def test_two_rank_gloo_sharding():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    mx, units, same = q.get(timeout=120)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert mx == 2.0 and units == 3.0 and same
