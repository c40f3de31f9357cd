"""world_size-2 gloo test of the N>1 path (instances sharded across ranks, no data-path
collective; only bookkeeping is reduced).  Each rank "solves" its shard with the CPU oracle standing in
for the device, so the test checks the sharding/aggregation logic, not the kernels."""
import os
import socket

import numpy as np
import pytest
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2606_16907_b200 import shard


def test_shard_range_partitions():
    for n in (0, 1, 5, 1024, 1025):
        for w in (1, 2, 3, 8):
            parts = [list(shard.shard_range(n, r, w)) for r in range(w)]
            assert sum(parts, []) == list(range(n))
            assert max(map(len, parts)) - min(map(len, parts)) <= 1
    assert list(shard.weak_seeds(4, 2)) == [8, 9, 10, 11]
    with pytest.raises(ValueError):
        shard.shard_range(4, 2, 2)


def _worker(rank, world, port, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import oracle
    import tg_inputs as gen
    n_total = 7
    mine = shard.shard_range(n_total, rank, world)
    res = [oracle.solve(gen.random_small(s, Lmax=6, Kmax=3, Pmax=2)).iter_time_us for s in mine]
    blobs = shard.gather_results(np.array(res, np.int64).tobytes())
    sums, maxes = shard.aggregate([len(mine), 10.0 * (rank + 1)], [5.0 + rank])
    q.put((rank, [np.frombuffer(b, np.int64).tolist() for b in blobs], sums, maxes))
    dist.barrier()
    dist.destroy_process_group()


def test_world_size_2_gloo():
    s = socket.socket(); s.bind(("127.0.0.1", 0)); port = s.getsockname()[1]; s.close()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    ps = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in ps:
        p.start()
    got = [q.get(timeout=120) for _ in ps]
    for p in ps:
        p.join(timeout=60)
        assert p.exitcode == 0
    import oracle
    import tg_inputs as gen
    want = [oracle.solve(gen.random_small(s, Lmax=6, Kmax=3, Pmax=2)).iter_time_us for s in range(7)]
    for rank, blobs, sums, maxes in got:
        assert sum(blobs, []) == want                 # rank order == seed order, nothing lost or duplicated
        assert sums == [7.0, 30.0] and maxes == [6.0]
