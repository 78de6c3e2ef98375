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
