"""N > 1 plumbing on CPU: world_size-2 gloo processes exercise unit sharding, the barrier and the
max/sum-over-ranks reductions bench.py uses (the data path itself has no collective)."""
import os
import socket

import pytest
import torch.multiprocessing as mp

from paper_2511_02328_b200 import multi


def test_shard_units_partition():
    for n in (0, 1, 2, 7, 8, 1001):
        for world in (1, 2, 3, 8):
            parts = [list(multi.shard_units(n, r, world)) for r in range(world)]
            flat = [u for p in parts for u in p]
            assert flat == list(range(n))
            assert max(map(len, parts)) - min(map(len, parts)) <= 1
    with pytest.raises(ValueError):
        multi.shard_units(4, 2, 2)


def _worker(rank, world, port, q):
    os.environ.update(RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE=str(world),
                      MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    r, lr, w = multi.init(backend="gloo")
    assert (r, w) == (rank, world)
    units = list(multi.shard_units(world, rank, world))
    multi.barrier()
    secs = 0.25 * (rank + 1)                      # rank 1 is the slow one
    rate, t = multi.job_throughput(100.0 * len(units), secs)
    q.put((rank, units, rate, t, multi.max_over_ranks(rank), multi.sum_over_ranks(1.0)))
    multi.finalize()


def test_gloo_world2_job_throughput():
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
    assert [r[1] for r in res] == [[0], [1]]                  # one observation per rank
    for _, _, rate, t, mx, sm in res:
        assert t == pytest.approx(0.5) and rate == pytest.approx(200.0 / 0.5)
        assert mx == 1.0 and sm == 2.0


def test_single_process_is_identity():
    assert multi.max_over_ranks(3.5) == 3.5 and multi.sum_over_ranks(2.0) == 2.0
    assert multi.env_world()[2] >= 1
