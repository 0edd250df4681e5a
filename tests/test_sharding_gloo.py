"""N>1 path on CPU: two gloo ranks shard a batch (disjoint, covering) and agree on the max-over-ranks time."""
import os
import socket

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2606_04206_b200.sharding import max_over_ranks, shard_range


def test_shard_range_covers_and_is_balanced():
    for B in (0, 1, 7, 4096, 4097):
        for W in (1, 2, 3, 8):
            spans = [shard_range(B, r, W) for r in range(W)]
            assert spans[0][0] == 0 and spans[-1][1] == B
            assert all(a[1] == b[0] for a, b in zip(spans, spans[1:]))
            sizes = [hi - lo for lo, hi in spans]
            assert max(sizes) - min(sizes) <= 1
    with pytest.raises(ValueError):
        shard_range(8, 2, 2)


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    lo, hi = shard_range(4097, rank, world)
    mine = torch.zeros(4097, dtype=torch.int32)
    mine[lo:hi] = 1
    dist.all_reduce(mine)                       # every env owned by exactly one rank
    t = max_over_ranks(10.0 + rank)             # rank-dependent "time"
    out.put((rank, bool((mine == 1).all()), t))
    dist.destroy_process_group()


def test_two_gloo_ranks_shard_and_reduce():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert [r[1] for r in res] == [True, True]
    assert [r[2] for r in res] == [11.0, 11.0]
