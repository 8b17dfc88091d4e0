"""N>1 host logic on CPU: world_size 2, gloo.  Walker sharding, max-over-ranks timing, aggregate value."""
import os
import socket

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2003_09468_b200 import replicas


def test_shard_walkers_partitions_exactly():
    for total in (0, 1, 7, 32, 33):
        for world in (1, 2, 3, 8):
            spans = [replicas.shard_walkers(total, r, world) for r in range(world)]
            assert spans[0][0] == 0 and spans[-1][1] == total
            for a, b in zip(spans, spans[1:]):
                assert a[1] == b[0]
            sizes = [b - a for a, b in spans]
            assert max(sizes) - min(sizes) <= 1
    with pytest.raises(ValueError):
        replicas.shard_walkers(4, 2, 2)


def _worker(rank, world, port, out):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    my_ms = 10.0 + 5.0 * rank                      # rank 1 is slower
    mx = replicas.max_over_ranks(my_ms)
    dist.barrier()
    out[rank] = (mx, replicas.aggregate_throughput(32, 10, world, mx), replicas.shard_walkers(33, rank, world))
    dist.destroy_process_group()


def test_two_rank_timing_is_max_over_ranks():
    s = socket.socket(); s.bind(("127.0.0.1", 0)); port = s.getsockname()[1]; s.close()
    mgr = mp.Manager()
    out = mgr.dict()
    mp.spawn(_worker, args=(2, port, out), nprocs=2, join=True)
    assert out[0][0] == out[1][0] == 15.0
    assert out[0][1] == pytest.approx(32 * 2 * 10 / 15e-3)
    assert out[0][2] == (0, 17) and out[1][2] == (17, 33)


def test_single_process_identity():
    assert replicas.max_over_ranks(3.5) == 3.5
