"""N>1 path: slices are sharded across ranks with no data-path collective; the only
communication is the barrier and the max-over-ranks of the device time.  Covered here with world_size 2 on
the gloo backend (CPU)."""
import os
import socket

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_1903_10088_b200 import sharding


def test_slice_ranges_partition_the_batch():
    for n in (0, 1, 5, 64, 67):
        for w in (1, 2, 3, 8):
            spans = [sharding.slice_range(r, w, n) for r in range(w)]
            assert spans[0][0] == 0 and spans[-1][1] == n
            for (a, b), (c, d) in zip(spans, spans[1:]):
                assert b == c and a <= b
            sizes = [b - a for a, b in spans]
            assert max(sizes) - min(sizes) <= 1 and sizes == sorted(sizes, reverse=True)
    with pytest.raises(ValueError):
        sharding.slice_range(2, 2, 4)


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
    lo, hi = sharding.slice_range(rank, world, 5)
    sharding.barrier()
    t = sharding.max_over_ranks(10.0 + rank)            # rank 1 is "slower"
    n = sharding.sum_over_ranks(hi - lo)
    q.put((rank, lo, hi, t, n))
    dist.destroy_process_group()


def test_world_size_2_gloo_timing_reduction():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert [(r[1], r[2]) for r in res] == [(0, 3), (3, 5)]
    assert all(r[3] == 11.0 for r in res) and all(r[4] == 5.0 for r in res)


def test_single_process_is_identity():
    assert sharding.max_over_ranks(3.5) == 3.5 and sharding.sum_over_ranks(2) == 2.0
    sharding.barrier()
