"""GPU parity of the compressed GPU software cache against the oracle.

Output bar: ibp_cache_gather_decompress == the plain gather of the original rows (oracle c1) and == the oracle codec (c2),
byte for byte, whatever the mix of hits and misses.  Structure bar: every map value has the paper's field widths (P:353,
checked through oracle.cache_value_fields), slab ranges are disjoint and inside the slab, the bytes a value points to are
the row's packed bytes as the oracle produces them, and the compressed flag equals the row's state.
"""
import numpy as np
import pytest

import oracle
from paper_2605_30728_b200 import binding as ibp
from paper_2605_30728_b200 import datagen, workloads

pytestmark = pytest.mark.gpu
torch = pytest.importorskip("torch")


def _stream():
    return torch.cuda.current_stream().cuda_stream


def _cache_gather(c, ids, rb):
    ids_d = torch.from_numpy(np.asarray(ids, np.int64)).cuda()
    out = torch.full((max(1, len(ids)), rb), 0xA5, dtype=torch.uint8, device="cuda")
    c.gather_decompress(ids_d.data_ptr(), len(ids), out.data_ptr(), _stream())
    torch.cuda.synchronize()
    return out.cpu().numpy()[: len(ids)]


def _lookup(c, ids):
    ids_d = torch.from_numpy(np.asarray(ids, np.int64)).cuda()
    ent = torch.zeros(len(ids), dtype=torch.int64, device="cuda")
    c.lookup(ids_d.data_ptr(), len(ids), ent.data_ptr(), _stream())
    torch.cuda.synchronize()
    return ent.cpu().numpy().view(np.uint64)


def _masked(n, rb, seed=5):
    return (datagen.random_bytes(n * rb, seed + rb).reshape(n, rb) & datagen.random_bytes(rb, 9)[None, :]) | 0x01


@pytest.mark.parametrize("align", [1, 4, 16, 32])
@pytest.mark.parametrize("n_slabs", [1, 3, 8])
def test_tiny_hits_and_misses(align, n_slabs):
    """configs[0] shape; a cache that holds about a third of the rows, spread over 1, 3 or 8 slabs."""
    w = workloads.Tiny()
    X = w.table()
    h = ibp.ibp_build(X, 512, 0, 64, align_bytes=align).upload_metadata(0)
    ds = oracle.Dataset(X, 0, 64)
    info = h.info()
    cap = info.packed_bytes_stored // 3
    c = ibp.Cache(h, cap, n_slabs)
    rng = np.random.default_rng(3)
    hot = rng.permutation(w.n_rows)[:3000].astype(np.int64)
    k = c.insert(hot)
    ci = c.info()
    assert 0 < k < len(hot) and ci.n_entries == k and ci.used_bytes <= ci.capacity_bytes <= cap and ci.n_slabs == n_slabs
    assert c.insert(hot[:k]) == 0                                           # already cached: nothing added
    # ---- structure of the map values
    ent = _lookup(c, np.arange(w.n_rows))
    cached = ent != np.uint64(ibp.IBP_CACHE_MISS)
    assert cached.sum() == k and set(np.flatnonzero(cached)) == set(hot[:k].tolist())   # priority order, stops when full
    spans = []
    for r in np.flatnonzero(cached):
        slab, off, comp, spare = oracle.cache_value_fields(ent[r])
        assert spare == 0 and slab < n_slabs and comp is True and off % 16 == 0
        data, kbits = h.packed_row(int(r))
        want = ds.packed_row(int(r))
        head = _row_head(h, int(r))
        got = c.read(int(ent[r]), head + want.size)
        assert np.array_equal(got[head:], want)                            # the oracle's packed bytes sit in the slab
        spans.append((slab, off, (head + data.size + 15) // 16 * 16))
    spans.sort()
    for (s0, o0, b0), (s1, o1, _) in zip(spans, spans[1:]):
        assert s0 < s1 or o0 + b0 <= o1                                     # disjoint inside a slab
    assert all(o + b <= ci.slab_bytes for _, o, b in spans)
    # ---- output, hits and misses mixed, duplicates
    for it in range(3):
        ids = w.ids(it)
        got = _cache_gather(c, ids, 512)
        assert np.array_equal(got, oracle.gather_plain(X, ids))
        assert np.array_equal(got, ds.gather_decompress(ids))
    assert np.array_equal(_cache_gather(c, hot[:k], 512), oracle.gather_plain(X, hot[:k]))        # all hits
    cold = np.flatnonzero(~cached)[:500]
    assert np.array_equal(_cache_gather(c, cold, 512), oracle.gather_plain(X, cold))              # all misses
    assert _cache_gather(c, np.empty(0, np.int64), 512).shape[0] == 0
    c.destroy(); h.destroy(); ds.close()


def _row_head(h, r):
    """offset of the packed row inside its 16-byte-aligned cover (rows start anywhere when A < 16)"""
    p0, _ = h.packed_range(0, 0)
    return (h.row_ptr(r) - p0) % 16


@pytest.mark.parametrize("kind,param,n,rb,align", [(0, 7, 50, 12, 1), (0, 64, 3000, 64, 32), (1, 5, 203, 32, 16), (0, 33, 1000, 100, 4),
                                                   (0, 128, 700, 256, 32), (0, 50, 333, 1024, 32), (0, 20, 77, 4096, 64),
                                                   (1, 6, 600, 2048, 16), (0, 9, 100, 264, 1)])
def test_ragged_shapes(kind, param, n, rb, align):
    X = _masked(n, rb)
    h = ibp.ibp_build(X, rb, kind, param, align_bytes=align).upload_metadata(0)
    c = ibp.Cache(h, max(64, h.info().packed_bytes_stored // 2), 2)
    rng = np.random.default_rng(n)
    c.insert(rng.permutation(n)[: n // 2 + 1])
    for mode in (0, 1):
        h.set_order_mode(mode).set_dedup_mode(mode)
        ids = rng.integers(0, n, 4 * n).astype(np.int64)
        assert np.array_equal(_cache_gather(c, ids, rb), oracle.gather_plain(X, ids))
    c.destroy(); h.destroy()


def test_thresholded_flag_and_output():
    """Thresholded mode keeps some rows raw: their map value carries compressed = 0 and the slab holds the raw row."""
    n, rb = 2000, 256
    rng = np.random.default_rng(1)
    X = _masked(n, rb)
    for r in rng.choice(n, n // 5, replace=False):
        X[r, rng.integers(0, rb)] ^= 0xFF
    raw_rows = rng.choice(n, 150, replace=False)
    for r in raw_rows:
        X[r] = datagen.random_bytes(rb, 1000 + int(r))
    h = ibp.ibp_build(X, rb, 0, 128, align_bytes=32, threshold=(4, 5)).upload_metadata(0)
    ds = oracle.DatasetT(X, 0, 128, 4, 5)
    c = ibp.Cache(h, h.info().packed_bytes_stored // 2, 2)
    k = c.insert(rng.permutation(n))
    assert 0 < k < n
    ent = _lookup(c, np.arange(n))
    n_raw_cached = 0
    for r in np.flatnonzero(ent != np.uint64(ibp.IBP_CACHE_MISS)):
        slab, off, comp, spare = oracle.cache_value_fields(ent[r])
        want, want_comp = ds.row(int(r))
        assert spare == 0 and comp == bool(want_comp)
        assert np.array_equal(c.read(int(ent[r]), want.size), want)
        n_raw_cached += not comp
    assert n_raw_cached > 0
    ids = rng.integers(0, n, 20000).astype(np.int64)
    got = _cache_gather(c, ids, rb)
    assert np.array_equal(got, oracle.gather_plain(X, ids)) and np.array_equal(got, ds.gather_decompress(ids))
    c.destroy(); h.destroy(); ds.close()


def test_workload_batches_with_hot_set():
    """GNN and DLRM shapes: the cache holds the hottest ids of the workload's sampler (a static cache)."""
    for w in (workloads.GNN(n_rows=200_000, batch=30_000), workloads.DLRM(rows_per_table=20_000, n_tables=4, samples=8192)):
        X = w.table()
        h = ibp.ibp_build(X, w.row_bytes, 0, w.group_param, align_bytes=32).upload_metadata(0)
        c = ibp.Cache(h, h.info().packed_bytes_stored // 10, 1)
        k = c.insert(w.hot_ids(w.n_rows // 5))
        assert k > 0
        for it in range(2):
            ids = w.ids(it)
            ent = _lookup(c, ids)
            hit = (ent != np.uint64(ibp.IBP_CACHE_MISS)).mean()
            assert hit > 0.2                                                # Zipf: a tenth of the bytes serves far more than a tenth
            assert np.array_equal(_cache_gather(c, ids, w.row_bytes), oracle.gather_plain(X, ids))
        c.destroy(); h.destroy()


def test_argument_errors():
    X = _masked(64, 32)
    h = ibp.ibp_build(X, 32, 0, 8)
    with pytest.raises(ibp.IbpError) as e:
        ibp.Cache(h, 1024)                                                  # before upload
    assert e.value.status == 4
    h.upload_metadata(0)
    with pytest.raises(ibp.IbpError) as e:
        ibp.Cache(h, 1024, 9)                                               # 3-bit slab id
    assert e.value.status == 1
    c = ibp.Cache(h, 1024)
    with pytest.raises(ibp.IbpError) as e:
        c.insert(np.array([64], np.int64))
    assert e.value.status == 1
    c.destroy(); h.destroy()
    h = ibp.ibp_build(X, 32, 0, 8, index_span=4).upload_metadata(0)
    with pytest.raises(ibp.IbpError) as e:
        ibp.Cache(h, 1024)
    assert e.value.status == 5
    h.destroy()


# ---------------------------------------------------------------------------------------------------------------------
# slabs on several GPUs (one data slab per interconnected GPU, the slab id of a map value names the GPU)
# ---------------------------------------------------------------------------------------------------------------------
def test_create_multi_on_this_process_devices():
    """ibp_cache_create_multi: slabs placed device by device.  One GPU here, so every slab names device 0 (explicitly or as -1):
    the layout, the map values and the output must equal ibp_cache_create's; a device this process does not have is refused."""
    w = workloads.Tiny()
    X = w.table()
    h = ibp.ibp_build(X, 512, 0, 64, align_bytes=32).upload_metadata(0)
    info = h.info()
    hot = np.random.default_rng(11).permutation(w.n_rows)[:1500].astype(np.int64)
    ref = ibp.Cache(h, info.packed_bytes_stored // 2, 3)
    multi = ibp.Cache(h, info.packed_bytes_stored // 2, 3, slab_devices=[0, -1, 0])
    assert ref.insert(hot) == multi.insert(hot) > 0
    assert np.array_equal(_lookup(ref, hot), _lookup(multi, hot))          # same placement -> same 64-bit values
    ids = np.random.default_rng(12).integers(0, w.n_rows, 2000)
    assert np.array_equal(_cache_gather(multi, ids, 512), oracle.gather_plain(X, ids))
    n_dev = torch.cuda.device_count()
    with pytest.raises(ibp.IbpError):
        ibp.Cache(h, 1 << 20, 2, slab_devices=[0, n_dev])                   # no such device
    with pytest.raises(ibp.IbpError):
        ibp.Cache(h, 1 << 20, 2, slab_devices=[0, -3])
    if n_dev > 1:                                                           # a real peer slab when the box has a second GPU
        peer = ibp.Cache(h, info.packed_bytes_stored // 2, 2, slab_devices=[0, 1])
        assert peer.insert(hot) > 0
        assert np.array_equal(_cache_gather(peer, ids, 512), oracle.gather_plain(X, ids))
        peer.destroy()
    # a remote slab that was never attached holds nothing: inserts skip it, exporting it or inserting into it is a state error
    part = ibp.Cache(h, info.packed_bytes_stored // 2, 2, slab_devices=[-1, ibp.IBP_SLAB_REMOTE])
    k = part.insert(hot)
    ent = _lookup(part, hot[:k])
    assert k > 0 and all(oracle.cache_value_fields(int(e))[0] == 0 for e in ent)
    with pytest.raises(ibp.IbpError):
        part.slab_export(1)
    with pytest.raises(ibp.IbpError):
        part.insert_slab(1, hot[:4], False)
    with pytest.raises(ibp.IbpError):
        part.slab_attach(0, b"\0" * ibp.IBP_IPC_HANDLE_BYTES)               # slab 0 already has memory
    assert np.array_equal(_cache_gather(part, ids, 512), oracle.gather_plain(X, ids))
    for c in (ref, multi, part):
        c.destroy()
    h.destroy()


def _peer_slab_worker(rank, world, port, thr, q):
    """One process per GPU (both on device 0 here: the box has one): rank r owns slab r; the other slab is the peer's memory,
    mapped through a CUDA IPC handle.  Every rank inserts every slab's id list; only the owner copies bytes."""
    import os
    import torch
    import torch.distributed as dist
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        torch.cuda.set_device(0)
        w = workloads.Tiny()
        X = w.table()
        h = ibp.ibp_build(X, 512, 0, 64, align_bytes=32, threshold=thr).upload_metadata(0)
        ds = oracle.Dataset(X, 0, 64) if thr[0] == thr[1] else oracle.DatasetT(X, 0, 64, thr[0], thr[1])
        info = h.info()
        devs = [ibp.IBP_SLAB_REMOTE] * world
        devs[rank] = -1
        c = ibp.Cache(h, info.packed_bytes_stored // 2, world, slab_devices=devs)
        handles = [None] * world
        dist.all_gather_object(handles, c.slab_export(rank))
        for s in range(world):
            if s != rank:
                c.slab_attach(s, handles[s])
        hot = np.random.default_rng(21).permutation(w.n_rows)[:1600].astype(np.int64)
        lists = [hot[s::world] for s in range(world)]                       # slab s caches every world-th hot row
        counts = [c.insert_slab(s, lists[s], fill=(s == rank)) for s in range(world)]
        dist.barrier()                                                      # every slab is filled by its owner before anyone reads it
        ok = all(k == len(l) for k, l in zip(counts, lists))
        # map values: slab id = the owner's rank, on every rank
        for s in range(world):
            ent = _lookup(c, lists[s])
            ok = ok and all(oracle.cache_value_fields(int(e))[0] == s and oracle.cache_value_fields(int(e))[3] == 0 for e in ent)
            # the bytes behind a value, read from the OWNER's or the PEER's memory alike, are the oracle's packed row
            for rid, e in list(zip(lists[s], ent))[:24]:
                pr = ds.packed_row(int(rid)) if thr[0] == thr[1] else ds.row(int(rid))[0]
                head = h.row_ptr(int(rid)) % 16                            # the slab stores the row's 16-byte cover
                ok = ok and np.array_equal(c.read(int(e), head + len(pr))[head:], pr)
        ids = np.random.default_rng(22 + rank).integers(0, w.n_rows, 3000)   # hits in both slabs and misses
        ok = ok and np.array_equal(_cache_gather(c, ids, 512), oracle.gather_plain(X, ids))
        ok = ok and np.array_equal(_cache_gather(c, ids, 512), ds.gather_decompress(ids))
        dist.barrier()                                                      # nobody unmaps a slab a peer is still reading
        c.destroy()
        h.destroy()
        ds.close()
        q.put((rank, bool(ok)))
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("thr", [(1, 1), (4, 5)])
def test_peer_slabs_two_processes_one_gpu(thr):
    """P:351-357 in the one-process-per-GPU layout: two processes, each owning one slab, reading the other's through CUDA IPC."""
    import socket
    import torch.multiprocessing as mp
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_peer_slab_worker, args=(r, 2, port, thr, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = [q.get(timeout=300) for _ in procs]
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert sorted(r[0] for r in res) == [0, 1] and all(r[1] for r in res)
