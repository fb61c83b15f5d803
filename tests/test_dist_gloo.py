"""World-size-2 gloo test (CPU) of the multi-rank plumbing bench.py uses: sharding of independent
spectra, barrier, max/sum over ranks.  The FDAS path has no data-path collective."""
import os
import socket

import pytest
import torch.multiprocessing as mp


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, q):
    os.environ.update(RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE=str(world),
                      MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    from paper_1804_05335_b200 import dist
    r, lr, w = dist.init("gloo")
    lo, hi = dist.shard(64, r, w)
    dist.barrier()
    tmax = dist.max_over_ranks(1.0 + r)
    total = dist.sum_over_ranks(float(hi - lo))
    q.put((r, lo, hi, tmax, total))
    dist.finalize()


def test_two_rank_sharding_and_reductions():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(2))
    for p in procs:
        p.join(60)
        assert p.exitcode == 0
    assert res[0][1:3] == (0, 32) and res[1][1:3] == (32, 64)
    assert all(r[3] == 2.0 and r[4] == 64.0 for r in res)


def test_shard_covers_everything():
    from paper_1804_05335_b200 import dist
    for total in (1, 7, 64, 65):
        for world in (1, 2, 3, 8):
            got = []
            for r in range(world):
                lo, hi = dist.shard(total, r, world)
                got += list(range(lo, hi))
            assert got == list(range(total))
