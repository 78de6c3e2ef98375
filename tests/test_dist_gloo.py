"""CPU-only, world_size 2 over gloo: the N>1 host logic (id sharding, all-gather of decoded slices, max-over-ranks timing).

No GPU here, so each rank's slice is decoded by the ORACLE as a stand-in for its GPU (test infrastructure only); what is
under test is the partition and the collectives around the hot path, which is exactly what differs at N>1.
"""
import os
import socket
import sys
from pathlib import Path

import numpy as np
import pytest

ROOT = Path(__file__).resolve().parent.parent
sys.path.insert(0, str(ROOT))

from paper_2605_30728_b200 import sharding  # noqa: E402


@pytest.mark.parametrize("n,world", [(0, 2), (1, 2), (5, 2), (250_000, 8), (1023, 4), (7, 8)])
def test_shard_bounds_cover_exactly(n, world):
    seen = np.zeros(n, np.int32)
    sizes = []
    for r in range(world):
        lo, hi = sharding.shard_bounds(n, r, world)
        assert 0 <= lo <= hi <= n
        seen[lo:hi] += 1
        sizes.append(hi - lo)
    assert np.all(seen == 1)
    assert max(sizes) - min(sizes) <= 1


def _worker(rank, world, port, q):
    import torch
    import torch.distributed as dist
    import oracle
    from paper_2605_30728_b200 import workloads
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        w = workloads.Tiny(n_rows=1024, batch=333)               # odd batch: ranks differ by one row
        X = w.table()
        ids = w.ids(0)
        mine = sharding.shard_ids(ids, rank, world)
        ds = oracle.Dataset(X, w.group_kind, w.group_param)      # each rank: its own store replica
        local = torch.from_numpy(ds.gather_decompress(mine))
        full = sharding.all_gather_rows(local, len(ids), world)
        ok = np.array_equal(full.numpy(), oracle.gather_plain(X, ids))
        t = sharding.max_over_ranks(1.0 + rank)
        q.put((rank, ok, t))
    finally:
        dist.destroy_process_group()


def test_world2_gloo_shard_gather():
    import torch.multiprocessing as mp
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = [q.get(timeout=120) for _ in procs]
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert sorted(r[0] for r in res) == [0, 1]
    assert all(r[1] for r in res)
    assert all(r[2] == 2.0 for r in res)                         # max over ranks of (1.0, 2.0)
