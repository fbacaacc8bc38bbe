"""World-size-2 gloo test of the multi-GPU host logic (timing reduction, frame / sector sharding, id offsets)."""
import os
import socket

import numpy as np
import torch.multiprocessing as mp

from paper_1811_11481_b200 import distributed


def _worker(rank, world, port, q):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist = distributed.init(world, rank, "gloo")
    ms, units = distributed.aggregate(dist, 10.0 + 5.0 * rank, 1000 * (rank + 1))
    # sector split of one synthetic CSR frame: 36 sectors with 10 + s clusters each; rank r "finds" 7 + 3 r tracks
    so = np.concatenate([[0], np.cumsum(10 + np.arange(36))]).astype(np.int32)
    cl = np.arange(so[-1], dtype=np.int64)
    mine, local_so, lo = distributed.shard_frame(cl, so, world, rank)
    counts = distributed.gather_counts(dist, 7 + 3 * rank)
    off = distributed.track_id_offsets(counts)
    local_assign = np.full(len(mine), -1, np.int32)
    local_assign[::5] = np.arange(len(local_assign[::5])) % (7 + 3 * rank)
    q.put((rank, ms, units, distributed.shard_sectors(36, world, rank), mine.tolist()[:2], local_so.tolist(), lo,
           counts.tolist(), off.tolist(), distributed.globalise_assignment(local_assign, off[rank]).tolist()))
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
    so = np.concatenate([[0], np.cumsum(10 + np.arange(36))])
    # rank 0 holds clusters [0, so[18]), rank 1 [so[18], so[36]); offsets re-based, sectors outside the range empty
    assert res[0][6] == 0 and res[1][6] == so[18] and res[1][4] == [int(so[18]), int(so[18]) + 1]
    assert res[0][5] == np.minimum(so, so[18]).tolist()
    assert res[1][5] == (np.maximum(so, so[18]) - so[18]).tolist()
    # both ranks see the same counts; ids of rank 1 start after rank 0's tracks; -1 stays -1
    assert res[0][7] == res[1][7] == [7, 10] and res[0][8] == res[1][8] == [0, 7]
    g0, g1 = np.array(res[0][9]), np.array(res[1][9])
    assert g0.max() == 6 and g1[g1 >= 0].min() == 7 and g1.max() == 16 and (g0[1::5] == -1).all()


def test_single_process_passthrough():
    assert distributed.aggregate(None, 3.5, 7) == (3.5, 7)
    cover = [distributed.shard_sectors(36, 8, r) for r in range(8)]
    assert cover[0][0] == 0 and cover[-1][1] == 36 and all(a[1] == b[0] for a, b in zip(cover, cover[1:]))
    assert distributed.gather_counts(None, 5).tolist() == [5]
    assert distributed.track_id_offsets([4, 0, 9]).tolist() == [0, 4, 4]
    so = np.array([0, 3, 3, 10, 12], np.int32)
    parts = [distributed.shard_frame(np.arange(12), so, 3, r) for r in range(3)]
    assert np.concatenate([p[0] for p in parts]).tolist() == list(range(12))
    for cl, lso, lo in parts:
        assert lso[0] == 0 and lso[-1] == len(cl) and (np.diff(lso) >= 0).all()


def test_cuts_inside_a_side_tells_when_the_per_rank_merger_is_incomplete():
    """The sector split exchanges no boundary segments: only cuts between the two z sides keep the
    merged tracks of the whole frame."""
    assert [distributed.cuts_inside_a_side(36, n, 18) for n in (1, 2, 3, 4, 6, 8)] == [0, 0, 2, 2, 4, 6]
    assert distributed.cuts_inside_a_side(36, 4, 9) == 0      # four rings of nine sectors: every cut on a ring boundary
    assert distributed.cuts_inside_a_side(36, 4, 0) == 0      # ring 0: nothing merges anyway
    for n in (2, 3, 4, 6, 8):                                 # brute force: a cut at sector b is harmless iff b % ring == 0
        cuts = [distributed.shard_sectors(36, n, r)[0] for r in range(1, n)]
        assert distributed.cuts_inside_a_side(36, n, 18) == sum(1 for b in cuts if b % 18)
