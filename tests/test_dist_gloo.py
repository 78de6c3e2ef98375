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


# ---------------------------------------------------------------------------------------------------------------------
# one packed store shared by all ranks ("each GPU reads the shared pinned store over its own PCIe link")
# ---------------------------------------------------------------------------------------------------------------------
def _shared_worker(rank, world, port, name, q):
    import torch.distributed as dist
    import oracle
    from paper_2605_30728_b200 import binding as ibp, workloads
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        w = workloads.Tiny(n_rows=2048, batch=500)
        if rank == 0:                                             # ONE rank builds and exports; nobody else holds a table or a store
            X = w.table()
            h0 = ibp.ibp_build(X, w.row_bytes, w.group_kind, w.group_param, align_bytes=32, flags=ibp.IBP_FLAG_PAGEABLE_STORE)
            h0.export_shared(name, numa_policy=1)
            h0.destroy()
        dist.barrier()
        h = ibp.ibp_open_shared(name)                             # every rank: a handle that borrows the segment
        info = h.info()
        ok = info.store_kind == ibp.IBP_STORE_SHARED and info.n_rows == 2048 and info.device == -1
        # the bookkeeping a rank needs before its GPU reads the store: where its rows lie, what they cost on the link
        ids = sharding.shard_ids(w.ids(0), rank, world)
        X = w.table()                                             # regenerated only to CHECK (seeded generator), not to build
        ds = oracle.Dataset(X, w.group_kind, w.group_param)
        for r in ids[:64]:
            data, k = h.packed_row(int(r))
            want = ds.packed_row(int(r))
            ok = ok and np.array_equal(data[: want.size], want) and k == ds.k_bits(int(r) // w.group_param)
        nu, stored, alg = h.batch_link_bytes(ids)
        ok = ok and nu == len(np.unique(ids)) and alg == sum((ds.k_bits(int(r) // w.group_param) + 7) // 8 for r in np.unique(ids))
        m, b, _ = h.metadata_host(3)
        ok = ok and np.array_equal(m, ds.mask(3)) and np.array_equal(b, ds.bitval(3))
        # the oracle stands in for the rank's GPU: decode the rank's slice FROM THE SHARED SEGMENT's bytes
        local = np.stack([oracle.unpack_row(h.packed_row(int(r))[0], ds.mask(int(r) // w.group_param), ds.bitval(int(r) // w.group_param)) for r in ids])
        import torch
        full = sharding.all_gather_rows(torch.from_numpy(local), len(w.ids(0)), world)
        ok = ok and np.array_equal(full.numpy(), oracle.gather_plain(X, w.ids(0)))
        base = h.row_ptr(0)
        dist.barrier()
        h.destroy()
        q.put((rank, bool(ok), int(base != 0)))
    finally:
        dist.destroy_process_group()


def test_world2_shared_store():
    import torch.multiprocessing as mp
    from paper_2605_30728_b200 import binding as ibp
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    name = f"/ibp_test_{os.getpid()}"
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_shared_worker, args=(r, 2, port, name, q)) for r in range(2)]
    for p in procs:
        p.start()
    try:
        res = [q.get(timeout=180) for _ in procs]
        for p in procs:
            p.join(timeout=60)
            assert p.exitcode == 0
    finally:
        ibp.ibp_unlink_shared(name)
    assert sorted(r[0] for r in res) == [0, 1]
    assert all(r[1] for r in res)
    with pytest.raises(ibp.IbpError):                             # the name is gone
        ibp.ibp_open_shared(name)


def test_shared_store_argument_checks_and_thresholded_image():
    from paper_2605_30728_b200 import binding as ibp, datagen
    import oracle
    name = f"/ibp_test_t_{os.getpid()}"
    X = (datagen.random_bytes(300 * 64, 8).reshape(300, 64) & 0x3F) | 0x40
    X[7] = datagen.random_bytes(64, 9)
    for flags, cap in ((ibp.IBP_FLAG_PAGEABLE_STORE, 0), (ibp.IBP_FLAG_PAGEABLE_STORE | ibp.IBP_FLAG_SLOT_LAYOUT, 320)):
        h0 = ibp.ibp_build(X, 64, 1, 6, align_bytes=16, threshold=(4, 5), flags=flags, capacity_rows=cap)
        h0.export_shared(name)
        h = ibp.ibp_open_shared(name)
        ds = oracle.DatasetT(X, 1, 6, 4, 5)
        i0, i1 = h0.info(), h.info()
        for f in ("n_rows", "n_groups", "packed_bytes_rows", "packed_bytes_bytealigned", "n_rows_raw", "thresholded", "slot_bytes", "capacity_rows", "max_row_stride"):
            assert getattr(i0, f) == getattr(i1, f), f
        for r in range(0, 300, 7):
            data, stored, comp = h.row_info(r)
            want, wc = ds.row(r)
            assert comp == wc and np.array_equal(data, want)
        with pytest.raises(ibp.IbpError) as e:                    # read-only, and no device here anyway
            h.append_rows_device(X.ctypes.data, 1)
        assert e.value.status == 4
        h.destroy(); h0.destroy(); ds.close()
        ibp.ibp_unlink_shared(name)
    for bad in ("noslash", "/a/b", "/"):
        with pytest.raises(ibp.IbpError):
            ibp.ibp_open_shared(bad)
    ibp.ibp_unlink_shared("/ibp_never_existed")                   # removing a name that is not there is fine
