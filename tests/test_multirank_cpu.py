"""World-size-2 gloo test (CPU) of the N > 1 plumbing: stream partition, max-over-ranks timing,
whole-job rate.  The LOF path itself has no collective."""
import os
import socket
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, q):
    sys.path.insert(0, ROOT)
    import torch.distributed as dist
    from paper_1701_08197_b200 import sharding
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    lo, hi = sharding.stream_range(rank, world, 97)
    t = sharding.max_over_ranks(1.0 + rank)              # rank 1 is the slow one
    dist.barrier()
    q.put((rank, lo, hi, t))
    dist.destroy_process_group()


def test_two_ranks_gloo():
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    ps = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in ps:
        p.start()
    out = sorted(q.get(timeout=120) for _ in ps)
    for p in ps:
        p.join(60)
        assert p.exitcode == 0
    (r0, lo0, hi0, t0), (r1, lo1, hi1, t1) = out
    assert (lo0, hi0, lo1, hi1) == (0, 49, 49, 97)        # contiguous, disjoint, complete
    assert t0 == t1 == 2.0                                 # max over ranks on both


def test_stream_range_properties():
    sys.path.insert(0, ROOT)
    from paper_1701_08197_b200 import sharding
    for world in (1, 2, 3, 8):
        for S in (0, 1, 7, 96, 6144, 7564):
            parts = [sharding.stream_range(r, world, S) for r in range(world)]
            assert parts[0][0] == 0 and parts[-1][1] == S
            assert all(a[1] == b[0] for a, b in zip(parts, parts[1:]))
            sizes = [b - a for a, b in parts]
            assert max(sizes) - min(sizes) <= 1
    with pytest.raises(ValueError):
        sharding.stream_range(2, 2, 10)
    assert sharding.aggregate_rate(100, 10, 1000.0, 4) == 4000.0
    assert sharding.max_over_ranks(3.5) == 3.5             # no process group: identity
