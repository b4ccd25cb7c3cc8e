"""N > 1 host logic on CPU: members partition across ranks, result rows gather in global order, device times
reduce by max -- world_size 2 over gloo (the data path itself has no collective)."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_1308_1856_b200 import sharding, workloads as wl


def test_member_slice_partitions():
    for n in (0, 1, 7, 256, 257):
        for world in (1, 2, 3, 8):
            seen = []
            for r in range(world):
                first, cnt = sharding.member_slice(n, r, world)
                seen += list(range(first, first + cnt))
            assert seen == list(range(n))
    with pytest.raises(ValueError):
        sharding.member_slice(4, 2, 2)


def _worker(rank, world, port, n_total, q):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        first, cnt = sharding.member_slice(n_total, rank, world)
        # each rank's "result rows" are a function of the global member index only
        c = wl.config("cfg5", batch=n_total)
        e0 = np.array([p[0] for p in wl.pulses(c)])[first:first + cnt]
        rows = np.stack([e0, np.arange(first, first + cnt, dtype=np.float64)], axis=1)
        allrows = sharding.gather_rows(rows, n_total)
        tmax = sharding.max_over_ranks(1.0 + rank)
        tsum = sharding.sum_over_ranks(cnt)
        sharding.barrier()
        q.put((rank, allrows, tmax, tsum))
    finally:
        dist.destroy_process_group()


def test_gather_and_max_world2():
    n_total = 7
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, n_total, q)) for r in range(2)]
    for p in procs:
        p.start()
    got = [q.get(timeout=120) for _ in procs]
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    c = wl.config("cfg5", batch=n_total)
    e0 = np.array([p[0] for p in wl.pulses(c)])
    for rank, allrows, tmax, tsum in got:
        assert np.array_equal(allrows[:, 1], np.arange(n_total))
        assert np.array_equal(allrows[:, 0], e0)
        assert tmax == 2.0 and tsum == n_total
