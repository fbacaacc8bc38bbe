"""World-size-2 gloo test of the multi-GPU host logic (timing reduction, frame / sector sharding)."""
import os
import socket

import torch.multiprocessing as mp

from paper_1811_11481_b200 import distributed


def _worker(rank, world, port, q):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist = distributed.init(world, rank, "gloo")
    ms, units = distributed.aggregate(dist, 10.0 + 5.0 * rank, 1000 * (rank + 1))
    q.put((rank, ms, units, distributed.shard_sectors(36, world, rank)))
    dist.barrier()
    dist.destroy_process_group()


def test_aggregate_world2_gloo():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    ps = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in ps:
        p.start()
    res = sorted(q.get(timeout=120) for _ in ps)
    for p in ps:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert res[0][1] == res[1][1] == 15.0          # max over ranks
    assert res[0][2] == res[1][2] == 3000          # whole-job units
    assert res[0][3] == (0, 18) and res[1][3] == (18, 36)


def test_single_process_passthrough():
    assert distributed.aggregate(None, 3.5, 7) == (3.5, 7)
    cover = [distributed.shard_sectors(36, 8, r) for r in range(8)]
    assert cover[0][0] == 0 and cover[-1][1] == 36 and all(a[1] == b[0] for a, b in zip(cover, cover[1:]))
