"""Multi-GPU host logic on CPU: world_size-2 gloo.  The path shards by spectra with no data-path collective
(PAPER.md:27), so what needs covering is the partition and the max-over-ranks / sum-over-ranks reductions bench.py uses."""
import os
import socket

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_1812_02647_b200.shard import max_over_ranks_ms, shard_bounds, sum_over_ranks


def test_shard_bounds_partition_the_batch():
    for batch in (0, 1, 7, 8, 4096, 4097):
        for world in (1, 2, 3, 8):
            cuts = [shard_bounds(batch, world, r) for r in range(world)]
            assert cuts[0][0] == 0 and cuts[-1][1] == batch
            for a, b in zip(cuts, cuts[1:]):
                assert a[1] == b[0]
            sizes = [hi - lo for lo, hi in cuts]
            assert max(sizes) - min(sizes) <= 1
    with pytest.raises(ValueError):
        shard_bounds(4, 2, 2)


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    return port


def _worker(rank, world, port, batch, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    lo, hi = shard_bounds(batch, world, rank)
    # each rank "processes" its slice: no exchange of data, only the timing/throughput reductions
    x = torch.arange(batch, dtype=torch.float64)[lo:hi]
    local_ms = 10.0 + 5.0 * rank
    t = max_over_ranks_ms(local_ms, dist)
    units = sum_over_ranks(float(hi - lo), dist)
    chk = sum_over_ranks(float(x.sum()), dist)
    dist.barrier()
    if rank == 0:
        out.put((t, units, chk))
    dist.destroy_process_group()


def test_world_size_two_gloo_reductions():
    ctx = mp.get_context("spawn")
    q = ctx.SimpleQueue()
    port, batch = _free_port(), 4097
    procs = [ctx.Process(target=_worker, args=(r, 2, port, batch, q)) for r in range(2)]
    for p in procs:
        p.start()
    for p in procs:
        p.join(120)
        assert p.exitcode == 0
    t, units, chk = q.get()
    assert t == 15.0 and units == batch and chk == batch * (batch - 1) / 2


def test_reductions_are_identity_without_a_process_group():
    assert max_over_ranks_ms(3.5, dist) == 3.5 and sum_over_ranks(7.0, dist) == 7.0
