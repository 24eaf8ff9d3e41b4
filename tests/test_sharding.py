"""Host logic of the multi-GPU path: contiguous batch slices, no data-path
collective.  world_size-2 gloo test on CPU; the per-rank compute is stood in for by a function of
the slice so that gather order and ragged sizes are what is tested (Procedure 3)."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2308_03310_b200 import sharding


@pytest.mark.parametrize("batch,world", [(16384, 8), (10, 3), (7, 8), (0, 2), (1, 1), (1025, 2)])
def test_bounds_partition_the_batch(batch, world):
    b = sharding.all_bounds(batch, world)
    assert b[0][0] == 0 and b[-1][1] == batch
    assert all(b[g][1] == b[g + 1][0] for g in range(world - 1))          # contiguous, disjoint
    sizes = [hi - lo for lo, hi in b]
    assert max(sizes) - min(sizes) <= 1 and sorted(sizes, reverse=True) == sizes


def test_bounds_reject_bad_arguments():
    with pytest.raises(ValueError):
        sharding.shard_bounds(8, 2, 2)
    with pytest.raises(ValueError):
        sharding.shard_bounds(-1, 2, 0)


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    return port


def _worker(rank, world, port, batch, out):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        rng = np.random.Generator(np.random.Philox(key=99))
        full = torch.from_numpy(rng.standard_normal((batch, 3, 5)))       # same on every rank
        mine = sharding.local_slice(full, world, rank)
        lo, hi = sharding.shard_bounds(batch, world, rank)
        assert mine.shape[0] == hi - lo and mine.data_ptr() == full[lo:hi].data_ptr()   # a view
        result = 2.0 * mine + 1.0                                          # stand-in for the rank's call
        got = sharding.gather_batch(result, batch)
        assert torch.equal(got, 2.0 * full + 1.0)
        t = sharding.max_over_ranks(1.0 + rank)
        assert t == float(world)
        if rank == 0:
            out.put("ok")
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("batch", [9, 64])
def test_world_size_2_gloo_gather(batch):
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, batch, out)) for r in range(2)]
    for p in procs:
        p.start()
    for p in procs:
        p.join(120)
    assert all(p.exitcode == 0 for p in procs)
    assert out.get(timeout=5) == "ok"
