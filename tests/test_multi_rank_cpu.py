"""World-size-2 test of the N>1 plumbing on CPU (gloo): disjoint weak-scaling shards of the seeded
stream, max-over-ranks timing, whole-job throughput.  The data path itself has no collective
(segments are independent), so this is all the multi-rank logic there is."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2603_29785_b200 import dist_utils, inputs


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        batch = 3
        first, n = dist_utils.shard_segments(rank, world, batch)
        x = inputs.make_batch("cfg5", batch=n, first_segment=first)
        # pretend rank 1 was slower
        ms = dist_utils.max_over_ranks([10.0 + 5.0 * rank, 2.0 - rank])
        checksum = torch.tensor([float(np.abs(x).sum())], dtype=torch.float64)
        gathered = [torch.zeros(1, dtype=torch.float64) for _ in range(world)]
        dist.all_gather(gathered, checksum)
        if rank == 0:
            out.put((first, ms, [float(g) for g in gathered]))
    finally:
        dist.destroy_process_group()


def test_world_size_2_gloo():
    world = 2
    port = _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    for p in procs:
        p.join(timeout=120)
        assert p.exitcode == 0
    first, ms, sums = q.get(timeout=10)
    assert first == 0
    assert ms == [15.0, 2.0]                     # element-wise max over ranks
    # the two ranks drew different segments of the same seeded stream
    x0 = inputs.make_batch("cfg5", batch=3, first_segment=0)
    x1 = inputs.make_batch("cfg5", batch=3, first_segment=3)
    assert sums[0] == pytest.approx(float(np.abs(x0).sum())) and sums[1] == pytest.approx(float(np.abs(x1).sum()))
    assert abs(sums[0] - sums[1]) > 1e-6
    # whole-job throughput counts every rank's units against the slowest time
    assert dist_utils.aggregate_throughput(2, 3, 4096, 15.0) == pytest.approx(2 * 3 * 4096 / 15e-3)


def test_shards_are_disjoint_and_cover():
    world, batch = 4, 5
    seen = []
    for r in range(world):
        first, n = dist_utils.shard_segments(r, world, batch)
        seen += list(range(first, first + n))
    assert seen == list(range(world * batch))


def test_single_process_max_is_identity():
    assert dist_utils.max_over_ranks([1.5, 2.5]) == [1.5, 2.5]
