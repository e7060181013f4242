"""N > 1 host logic on CPU: world_size 2, gloo backend."""
import os
import socket

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2206_12205_b200 import sharding


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, q):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    mine = sharding.series_for_rank(256, rank, world)
    # every rank times its own work; the job time is the max, the job throughput the sum of units / max
    elapsed = 1.0 + 0.5 * rank
    t_max = sharding.max_over_ranks(elapsed)
    units = sharding.sum_over_ranks(float(len(mine)))
    dist.barrier()
    q.put((rank, mine[:3], len(mine), t_max, units))
    dist.destroy_process_group()


def test_two_rank_sharding_and_reductions():
    world = 2
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    got = sorted(q.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert got[0][1] == [0, 2, 4] and got[1][1] == [1, 3, 5]
    assert got[0][2] + got[1][2] == 256
    assert got[0][3] == got[1][3] == 1.5            # max over ranks
    assert got[0][4] == got[1][4] == 256.0          # all series accounted for, none twice


def test_partition_is_a_partition():
    for world in (1, 2, 3, 8):
        seen = []
        for r in range(world):
            seen += sharding.series_for_rank(256, r, world)
        assert sorted(seen) == list(range(256))
    with pytest.raises(ValueError):
        sharding.series_for_rank(4, 2, 2)


def test_sub_batches_fit_hbm():
    # config 4: 97 x 2^21 float planes; 180 GB HBM -> at most ~187 planes resident, never all 256
    n = sharding.max_resident_series(97, 1 << 21, 4, 180 * 10**9)
    assert 100 < n < 256
    mine = sharding.series_for_rank(256, 0, 1)
    sb = sharding.sub_batches(mine, n)
    assert sum(len(b) for b in sb) == 256 and max(len(b) for b in sb) <= n and len(sb) == 2
    assert sharding.max_over_ranks(3.25) == 3.25    # identity when not distributed
