"""N > 1 host logic on CPU: world_size-2 (and 3) `gloo` processes shard the seeds of every partition,
take their local argmin and merge with one exchange step; the result must equal the single-process
rule (lowest RSS, ties -> lowest global seed index, R15)."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_1911_09340_b200.sharding import local_best, merge_best, shard_events, shard_partitions


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _fake_rss(S, seed):
    rng = np.random.default_rng(seed)
    rss = rng.integers(0, 50, size=S).astype(np.float64) * 0.01      # many exact ties
    return rss


PART_OFF = np.array([0, 1000, 1000, 1000 + 4097, 1000 + 4097 + 33], dtype=np.int64)   # one empty partition


def _worker(rank, world, port, q):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        rss_all = torch.from_numpy(_fake_rss(int(PART_OFF[-1]), 7))
        ranges = shard_partitions(PART_OFF, rank, world)
        # each rank only holds the RSS of its own ranges (others poisoned)
        mine = torch.full_like(rss_all, float("nan"))
        for b, e in ranges:
            mine[b:e] = rss_all[b:e]
        v, i = local_best(mine, ranges)
        gv, gi = merge_best(v, i)
        q.put((rank, ranges, gv.numpy().copy(), gi.numpy().copy()))
        dist.barrier()
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("world", [2, 3])
def test_seed_sharded_argmin_matches_single_process(world):
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = [q.get(timeout=120) for _ in range(world)]
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    rss = _fake_rss(int(PART_OFF[-1]), 7)
    P = len(PART_OFF) - 1
    exp_v = np.full(P, np.inf)
    exp_i = np.full(P, np.iinfo(np.int64).max, dtype=np.int64)
    for p in range(P):
        lo, hi = PART_OFF[p], PART_OFF[p + 1]
        if hi > lo:
            exp_i[p] = lo + int(np.argmin(rss[lo:hi]))
            exp_v[p] = rss[exp_i[p]]
    covered = np.zeros(int(PART_OFF[-1]), dtype=np.int32)
    for rank, ranges, gv, gi in res:
        np.testing.assert_array_equal(gv, exp_v)
        np.testing.assert_array_equal(gi, exp_i)
        for (b, e), p in zip(ranges, range(P)):
            assert PART_OFF[p] <= b <= e <= PART_OFF[p + 1]
            assert (b - PART_OFF[p]) % 32 == 0 or b == PART_OFF[p + 1]
            covered[b:e] += 1
    assert np.all(covered == 1)                       # a partition of the seed set: no gap, no overlap


def test_shard_helpers_single_process():
    assert shard_events(10, 1, 4) == [1, 5, 9]
    assert shard_events(2, 3, 4) == []
    with pytest.raises(ValueError):
        shard_partitions(PART_OFF, 2, 2)
    r = shard_partitions(np.array([0, 64]), 0, 4)
    assert r == [(0, 0)] or r == [(0, 32)] or r[0][1] % 32 == 0
    allr = [shard_partitions(np.array([0, 70]), k, 4)[0] for k in range(4)]
    assert allr[0][0] == 0 and allr[-1][1] == 70 and all(a[1] == b[0] for a, b in zip(allr, allr[1:]))
    v, i = local_best(torch.tensor([3.0, 1.0, 1.0, 2.0], dtype=torch.float64), [(0, 4), (2, 2)])
    assert v.tolist() == [1.0, float("inf")] and i.tolist() == [1, np.iinfo(np.int64).max]
    gv, gi = merge_best(v, i)                          # no process group: identity
    assert gv.tolist() == v.tolist() and gi.tolist() == i.tolist()
