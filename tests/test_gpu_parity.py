"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle, element by element as raw bytes.

Bar: bit-exact (integer/byte work; floats are compared as bit patterns so NaN payloads, -0.0 and denormals count).
Sizes span several tiles (warps, CTAs, grid-stride rounds) and ragged tails; edge cases: empty batch, duplicates,
groups with no variant bit, groups with no invariant bit, multi-pass rows, every alignment unit.
"""
import numpy as np
import pytest

import oracle
from paper_2605_30728_b200 import binding as ibp
from paper_2605_30728_b200 import datagen, workloads

pytestmark = pytest.mark.gpu
torch = pytest.importorskip("torch")


def _dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def _gather(h, ids, span=1, rb=None):
    rb = rb or h.info().row_bytes
    ids_d = _dev(np.asarray(ids, np.int64))
    out = torch.full((max(1, len(ids) * span), rb), 0xA5, dtype=torch.uint8, device="cuda")
    h.gather_decompress(ids_d.data_ptr(), len(ids), out.data_ptr(), torch.cuda.current_stream().cuda_stream)
    torch.cuda.synchronize()
    return out.cpu().numpy()[: len(ids) * span]


def _resident(h, first, n):
    ptr, nbytes = h.packed_range(first, n)
    packed = _dev(h.packed_view(ptr, nbytes).copy()) if nbytes else torch.zeros(16, dtype=torch.uint8, device="cuda")
    out = torch.full((max(1, n), h.info().row_bytes), 0x5A, dtype=torch.uint8, device="cuda")
    h.decompress_resident(packed.data_ptr(), first, n, out.data_ptr(), torch.cuda.current_stream().cuda_stream)
    torch.cuda.synchronize()
    return out.cpu().numpy()[:n]


def _range(h, first, n):
    out = torch.full((max(1, n), h.info().row_bytes), 0x3C, dtype=torch.uint8, device="cuda")
    h.gather_decompress_range(first, n, out.data_ptr(), torch.cuda.current_stream().cuda_stream)
    torch.cuda.synchronize()
    return out.cpu().numpy()[:n]


def _u8(X):
    X = np.ascontiguousarray(X)
    return X.view(np.uint8).reshape(X.shape[0], -1)


# ---------------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("align", [1, 4, 16, 32, 64, 128])
@pytest.mark.parametrize("order_mode", [0, 1])
@pytest.mark.parametrize("fetch_mode", [0, 1])
def test_tiny_config_gather(align, order_mode, fetch_mode):
    """BASELINE.json configs[0] exactly: 4,096 x 128 fp32, groups of 64, 1,024 uniform ids; both fetch engines
    (cp.async through the LSU, cp.async.bulk through the TMA unit) and both processing orders."""
    w = workloads.Tiny()
    X = w.table()
    h = ibp.ibp_build(X, 512, 0, 64, align_bytes=align).upload_metadata(0).set_order_mode(order_mode).set_fetch_mode(fetch_mode)
    ds = oracle.Dataset(X, 0, 64)
    for it in range(3):
        ids = w.ids(it)
        got = _gather(h, ids)
        assert np.array_equal(got, ds.gather_decompress(ids))          # (c2) the oracle codec
        assert np.array_equal(got, oracle.gather_plain(X, ids))        # (c1) the plain definition
    h.destroy()


@pytest.mark.parametrize("kind,param,n,rb,align", [
    (0, 7, 50, 12, 1), (0, 7, 50, 12, 16), (0, 64, 3000, 64, 32), (0, 1000, 10, 8, 4), (0, 16, 40, 4, 16),
    (1, 5, 203, 32, 16), (1, 8, 64, 16, 1), (1, 3, 2, 4, 16), (0, 1, 9, 20, 8), (0, 33, 1000, 100, 32),
    (0, 128, 700, 256, 32), (0, 256, 1500, 512, 32), (0, 50, 333, 1024, 32), (0, 20, 77, 4096, 64), (1, 6, 600, 2048, 16),
    (0, 9, 100, 516, 4), (0, 9, 100, 264, 1), (0, 4, 30, 8192, 128),
])
def test_ragged_shapes_gather_and_resident(kind, param, n, rb, align):
    """Shapes the fast paths do not special-case: odd row sizes (W=1,2,4; 1..16 passes), ragged last groups, strided
    groups with a partial last matrix row, every alignment unit; gather (both orders) and resident decode."""
    X = (datagen.random_bytes(n * rb, 5 + rb).reshape(n, rb) & datagen.random_bytes(rb, 9)[None, :]) | 0x01
    h = ibp.ibp_build(X, rb, kind, param, align_bytes=align).upload_metadata(0)
    ds = oracle.Dataset(X, kind, param)
    ids = np.concatenate([(datagen.u64(777, 3) % np.uint64(n)).astype(np.int64), np.arange(n, dtype=np.int64)])
    want = ds.gather_decompress(ids)
    assert np.array_equal(want, oracle.gather_plain(X, ids))
    for fetch in (0, 1):
        h.set_fetch_mode(fetch)
        for mode in (0, 1):
            h.set_order_mode(mode)
            h.set_dedup_mode(mode ^ fetch)
            assert np.array_equal(_gather(h, ids), want)
    h.set_dedup_mode(0)
    for fetch in (0, 1):
        h.set_fetch_mode(fetch)
        for sm in (0, 1):                                               # per-row fetch kernel / TMA stream kernel
            h.set_stream_mode(sm)
            assert np.array_equal(_resident(h, 0, n), X)                # whole table from HBM
            assert np.array_equal(_range(h, 0, n), X)                   # whole table zero-copy, no id list
    if kind == 0 and n > 2 * param:
        first = param * ((n // param) // 2)
        assert np.array_equal(_resident(h, first, n - first), X[first:])
        assert np.array_equal(_resident(h, first, param), X[first:first + param])
    if kind == 1 and n > 2 * param:
        first = param * ((n // param) // 2)
        assert np.array_equal(_resident(h, first, n - first), X[first:])
    h.destroy()


def test_decode_ranges_host_destinations():
    """ibp_decode_ranges_host: several ranges of several handles into HOST buffers -- pinned and GPU-mapped (the kernels store
    straight into them, batched launches) and ordinary pageable memory (range by range through a staging buffer)."""
    mats = []
    for j, (S, n, rb) in enumerate([(8, 8 * 50, 256), (8, 8 * 31 + 3, 256), (5, 203, 256), (16, 16 * 20, 256)]):
        X = (datagen.random_bytes(n * rb, 40 + j).reshape(n, rb) & datagen.random_bytes(rb, 60 + j)[None, :]) | 0x01
        mats.append((ibp.ibp_build(X, rb, 1, S, align_bytes=16).upload_metadata(0), X))
    Xb = (datagen.random_bytes(300 * 256, 7).reshape(300, 256) & 0x3F) | 0x40
    mats.append((ibp.ibp_build(Xb, 256, 0, 64, align_bytes=16, threshold=(4, 5)).upload_metadata(0), Xb))   # a thresholded handle in the list
    total = sum(len(X) for _, X in mats)
    st = torch.cuda.current_stream().cuda_stream
    pin = ibp.PinnedBuffer(total * 256)
    for name, dest in (("pinned", pin.view(np.uint8, (total, 256))), ("pageable", np.zeros((total, 256), np.uint8))):
        dest[:] = 0xEE
        rs, off = [], 0
        for h, X in mats:
            rs.append((h, None, 0, len(X), dest[off:off + len(X)]))
            off += len(X)
        ibp.ibp_decode_ranges_host(rs, st)
        assert np.array_equal(dest, np.concatenate([X for _, X in mats])), name
    pin.free()
    for h, _ in mats:
        h.destroy()


@pytest.mark.parametrize("S,n,rb,align", [(86, 86 * 40 + 13, 256, 16), (32, 32 * 70, 256, 16), (9, 9 * 33 + 4, 512, 32), (16, 16 * 5, 64, 4),
                                           (17, 17 * 100 + 16, 128, 16), (8, 8 * 3 + 1, 256, 32), (3, 50, 512, 16), (40, 40 * 64 + 39, 128, 4)])
def test_strided_resident_tile_blocks(S, n, rb, align):
    """Resident decode of strided tables takes tile-block chunks (a CTA keeps one block of 8 column tiles, a warp one tile):
    tile counts that are not a multiple of 8, fewer tiles than consumer warps, a partial last matrix row, ranges that start
    inside the table, a tile whose rows are all identical (k = 0) and one with no invariant bit."""
    X = (datagen.random_bytes(n * rb, 11 + S).reshape(n, rb) & datagen.random_bytes(rb, 19)[None, :]) | 0x01
    X[1 % S::S] = X[1 % S]                                              # tile 1: every row the same -> nothing stored
    X[2 % S::S] = datagen.random_bytes(len(X[2 % S::S]) * rb, 23).reshape(-1, rb)   # tile 2: (almost surely) nothing invariant
    h = ibp.ibp_build(X, rb, 1, S, align_bytes=align).upload_metadata(0)
    ds = oracle.Dataset(X, 1, S)
    assert np.array_equal(_resident(h, 0, n), X)
    assert np.array_equal(ds.gather_decompress(np.arange(n)), X)
    for first, cnt in [(0, S), (0, 2 * S + 1), (S * ((n // S) // 2), n - S * ((n // S) // 2)), (S, min(n - S, 3 * S - 1))]:
        if cnt > 0 and first + cnt <= n:
            assert np.array_equal(_resident(h, first, cnt), X[first:first + cnt]), (first, cnt)
            assert np.array_equal(_range(h, first, cnt), X[first:first + cnt]), (first, cnt)
    h.configure(4, 0)                                                   # fewer CTAs than tile blocks: whole-row chunks again
    assert np.array_equal(_resident(h, 0, n), X)
    h.destroy()
    ds.close()


def test_edge_cases():
    rb = 256
    r = datagen.random_bytes(rb, 3)
    # all-identical group (k=0: nothing crosses PCIe), a group with a row and its complement (k = all bits: raw copy),
    # NaN / -0.0 / denormal patterns survive, duplicates, empty batch
    special = np.frombuffer(np.array([np.nan, -0.0, 1e-45, np.inf, -np.inf, 0.0, 1.0, -1.0] * 8, np.float32).tobytes(), np.uint8)
    X = np.stack([r] * 4 + [r, ~r, r, ~r] + [special, special ^ 1, special, special ^ 0x80])
    h = ibp.ibp_build(X, rb, 0, 4, align_bytes=16).upload_metadata(0)
    ks = [h.metadata_host(g)[2] for g in range(3)]
    assert ks[0] == 0 and ks[1] == 8 * rb
    ids = np.array([0, 3, 3, 3, 4, 5, 11, 8, 9, 10, 0, 7], np.int64)
    assert np.array_equal(_gather(h, ids), X[ids])
    assert _gather(h, np.zeros(0, np.int64)).shape[0] == 0               # n == 0 is a no-op
    assert np.array_equal(_resident(h, 0, 12), X)
    assert np.array_equal(_resident(h, 4, 4), X[4:8])
    # id validation pre-pass
    bad = _dev(np.array([0, 11, 12, -1, 5], np.int64))
    assert h.validate_ids(bad.data_ptr(), 5, torch.cuda.current_stream().cuda_stream) == 2
    # argument errors are reported, not ignored
    out = torch.zeros(16 + rb, dtype=torch.uint8, device="cuda")
    with pytest.raises(ibp.IbpError):
        h.gather_decompress(bad.data_ptr(), 1, out.data_ptr() + 1)
    with pytest.raises(ibp.IbpError):
        h.decompress_resident(out.data_ptr(), 2, 4, out.data_ptr())
    h.destroy()


@pytest.mark.parametrize("n_ids", [1, 31, 33, 4097, 100_000])
def test_gnn_shape_batches(n_ids):
    """configs[1] shape at 200k rows: dense + sparse halves and the mixed group at the boundary; batch sizes around the
    warp / CTA / grid-stride boundaries; launch configuration of bench.py (defaults)."""
    w = workloads.GNN(n_rows=200_000, batch=n_ids)
    X = w.table()
    h = ibp.ibp_build(X, 512, 0, 256, align_bytes=32).upload_metadata(0)
    ids = w.ids(0)
    assert len(np.unique(ids)) == len(ids) == n_ids
    got = _gather(h, ids)
    assert np.array_equal(got, oracle.gather_plain(X, ids))
    # the oracle codec on the groups this batch touches (groups are independent): masks, k, decode
    Xb = _u8(X)
    for g in np.unique(ids // 256)[:40]:
        rows = Xb[g * 256:(g + 1) * 256]
        mask, bitval, k = oracle.group_masks(rows)
        m, b, kk = h.metadata_host(int(g))
        assert k == kk and np.array_equal(m, mask) and np.array_equal(b, bitval)
    h.destroy()


@pytest.mark.parametrize("flags,kind", [(0, ibp.IBP_STORE_MANAGED_HOST), (ibp.IBP_FLAG_HOSTALLOC_STORE, ibp.IBP_STORE_PINNED)])
def test_dlrm_shape_duplicates(flags, kind):
    """configs[2] shape, small; both GPU-visible store kinds (managed-host default, cudaHostAlloc by flag)."""
    w = workloads.DLRM(rows_per_table=50_000, n_tables=26, samples=2048)
    X = w.table()
    h = ibp.ibp_build(X, 256, 0, 128, align_bytes=32, flags=flags).upload_metadata(0)
    assert h.info().store_kind == kind
    ids = w.ids(0)
    assert len(np.unique(ids)) < len(ids)                                 # repeats kept (reading R16)
    for dedup in (0, 1):                                                  # fetch every id / fetch distinct ids once
        h.set_dedup_mode(dedup)
        for mode in (0, 1):
            h.set_order_mode(mode)
            assert np.array_equal(_gather(h, ids), oracle.gather_plain(X, ids))
    same = np.full(5000, int(ids[7]), np.int64)                           # a batch that is one id repeated
    assert np.array_equal(_gather(h, same), oracle.gather_plain(X, same))
    h.destroy()


def test_kv_shape_spans():
    """configs[3] shape, small: one id = one page of one layer of K or V = heads*16 consecutive rows, groups of 16."""
    w = workloads.KV(layers=2, pages=64, heads=8, pages_per_layer=16)
    X = w.table()
    h = ibp.ibp_build(X, 256, 0, 16, align_bytes=16, index_span=w.index_span).upload_metadata(0)
    ds = oracle.Dataset(X, 0, 16)
    ids = w.ids(0)
    for sm in (0, 1):
        h.set_stream_mode(sm)
        got = _gather(h, ids, span=w.index_span)
        assert np.array_equal(got, ds.gather_decompress(ids, w.index_span))
        assert np.array_equal(got, oracle.gather_plain(X, ids, w.index_span))
    h.destroy()


def test_weight_shape_stream_and_resident():
    """configs[4] shape, small: strided column-tile groups; whole matrix gathered in order, and decoded from HBM."""
    for rows, cols in ((256, 512), (96, 1408)):
        w = workloads.WeightMatrix(rows, cols)
        X = w.table()
        h = ibp.ibp_build(X, 256, 1, w.group_param, align_bytes=16).upload_metadata(0)
        ds = oracle.Dataset(X, 1, w.group_param)
        ids = w.ids(0)
        got = _gather(h, ids)
        assert np.array_equal(got, ds.gather_decompress(ids))
        assert np.array_equal(got, _u8(X))
        assert np.array_equal(_resident(h, 0, w.n_rows), _u8(X))
        assert np.array_equal(_range(h, 0, w.n_rows), _u8(X))
        half = (w.mat_rows // 2) * w.group_param
        assert np.array_equal(_range(h, half, w.n_rows - half), _u8(X)[half:])
        # host destinations: pinned + mapped (the kernel stores straight into host memory) and pageable (staged)
        pin = ibp.PinnedBuffer(w.n_rows * 256)
        h.gather_decompress_range_host(0, w.n_rows, pin.view(np.uint8, (w.n_rows, 256)), torch.cuda.current_stream().cuda_stream)
        assert np.array_equal(pin.view(np.uint8, (w.n_rows, 256)), _u8(X))
        pin.free()
        pg = np.zeros((w.n_rows - half, 256), np.uint8)
        h.gather_decompress_range_host(half, w.n_rows - half, pg, torch.cuda.current_stream().cuda_stream)
        assert np.array_equal(pg, _u8(X)[half:])
        h.destroy()


@pytest.mark.parametrize("max_ctas", [0, 12, 3])
def test_decode_ranges_one_launch_per_layer(max_ctas):
    """ibp_decode_ranges: a 'layer' of matrices (strided column-tile groups with 4, 11 and 1 tile blocks, one matrix with fewer
    rows than tiles), a blocked table, a thresholded handle and an empty range in ONE call -- 11 ranges, so two batched launches
    plus per-range fall-backs -- from the host store and from packed bytes staged in HBM (tile-block chunks), whole and partial
    ranges.  Every output byte against the original rows (c1) and, per table, against the oracle codec on a sample (c2)."""
    st = torch.cuda.current_stream().cuda_stream
    specs = [("w", 96, 4096), ("w", 64, 11008), ("w", 40, 512), ("w", 3, 1408), ("b", 700, 256, 16), ("w", 33, 4096),
             ("t", 500, 256, 50), ("w", 17, 2816), ("w", 8, 4096), ("b", 90, 256, 7), ("w", 12, 11008)]
    tabs = []
    for i, sp in enumerate(specs):
        if sp[0] == "w":
            wm = workloads.WeightMatrix(sp[1], sp[2], layer=9, slot=i % 8)
            X = _u8(wm.table())
            h = ibp.ibp_build(X, 256, 1, wm.group_param, align_bytes=16).upload_metadata(0)
            unit = wm.group_param
            ds = oracle.Dataset(X, 1, wm.group_param)
        else:
            n, rb, G = sp[1], sp[2], sp[3]
            X = (datagen.random_bytes(n * rb, 70 + i).reshape(n, rb) & datagen.random_bytes(rb, 71 + i)[None, :]) | 0x04
            thr = (4, 5) if sp[0] == "t" else (1, 1)
            h = ibp.ibp_build(X, rb, 0, G, align_bytes=16, threshold=thr).upload_metadata(0)
            unit = G if sp[0] == "b" else 1
            ds = oracle.Dataset(X, 0, G) if sp[0] == "b" else oracle.DatasetT(X, 0, G, 4, 5)
        if max_ctas:
            h.configure(max_ctas, 0)
        ids = np.arange(0, X.shape[0], 5, dtype=np.int64)
        assert np.array_equal(ds.gather_decompress(ids), X[ids])
        ds.close()
        tabs.append((h, X, unit))
    for resident in (False, True):
        for partial in (False, True):
            ranges, outs, wants, keep = [], [], [], []
            for j, (h, X, unit) in enumerate(tabs):
                n = X.shape[0]
                first = (n // unit // 2) * unit if partial and n >= 2 * unit else 0
                cnt = 0 if (j == 4 and partial) else n - first                 # one empty range
                out = torch.full((max(1, cnt), X.shape[1]), 0x77, dtype=torch.uint8, device="cuda")
                packed = None
                if resident and cnt:
                    ptr, nb = h.packed_range(first, cnt)
                    buf = _dev(h.packed_view(ptr, nb).copy()) if nb else torch.zeros(16, dtype=torch.uint8, device="cuda")
                    keep.append(buf)
                    packed = buf.data_ptr()
                ranges.append((h, packed, first, cnt, out.data_ptr()))
                outs.append(out)
                wants.append(X[first:first + cnt])
            ibp.ibp_decode_ranges(ranges, st)
            torch.cuda.synchronize()
            for j, (o, want) in enumerate(zip(outs, wants)):
                assert np.array_equal(o.cpu().numpy()[: want.shape[0]], want), f"range {j} resident={resident} partial={partial}"
    with pytest.raises(ibp.IbpError):
        ibp.ibp_decode_ranges([(tabs[0][0], None, 1, 5, outs[0].data_ptr())], st)      # first_row is not a unit boundary
    for h, _, _ in tabs:
        h.destroy()


def test_fig7_sweep_shapes():
    """PAPER.md:399 microbenchmark shape: synthetic masks of chosen popcount; 256 B / 1 KB / 4 KB tensors, one group."""
    for rb, savings in ((256, 0.1), (256, 0.9), (1024, 0.5), (1024, 0.95), (4096, 0.3), (4096, 0.9)):
        w = workloads.Sweep(rb, savings, n_rows=3000)
        X = w.table()
        h = ibp.ibp_build(X, rb, 0, w.n_rows, align_bytes=32).upload_metadata(0)
        m, b, k = h.metadata_host(0)
        assert k <= 8 * rb - w.n_fixed + 0                                   # at least the chosen bits are invariant
        ids = w.ids(0)
        assert np.array_equal(_gather(h, ids), _u8(X)[ids])
        h.destroy()


def test_uncompressed_baseline_and_host_api():
    w = workloads.Tiny()
    X = w.table()
    ids = w.ids(1)
    pin = ibp.PinnedBuffer(X.nbytes)
    pin.view(np.float32, X.shape)[:] = X
    ids_d = _dev(ids)
    out = torch.zeros((len(ids), 512), dtype=torch.uint8, device="cuda")
    for order in (False, True):
        out.zero_()
        ibp.ibp_gather_uncompressed(pin.dev_ptr, 512, ids_d.data_ptr(), len(ids), out.data_ptr(),
                                    torch.cuda.current_stream().cuda_stream, n_rows=w.n_rows, locality_order=order)
        torch.cuda.synchronize()
        assert np.array_equal(out.cpu().numpy(), oracle.gather_plain(X, ids))
    # end-to-end entry point with host buffers
    h = ibp.ibp_build(X, 512, 0, 64).upload_metadata(0)
    out_h = np.zeros((len(ids), 512), np.uint8)
    h.gather_decompress_host(ids, len(ids), out_h, torch.cuda.current_stream().cuda_stream)
    assert np.array_equal(out_h, oracle.gather_plain(X, ids))
    # large batches are cut into chunks (device->host copy of one overlaps the gather of the next): 2 and 4 chunks, pinned
    # and pageable destinations, duplicates across chunk borders
    for n_big in (20_000, 70_001):
        big = np.random.default_rng(n_big).integers(0, w.n_rows, n_big).astype(np.int64)
        want = oracle.gather_plain(X, big)
        out_big = np.zeros((n_big, 512), np.uint8)
        h.gather_decompress_host(big, n_big, out_big, torch.cuda.current_stream().cuda_stream)
        assert np.array_equal(out_big, want)
        pout = ibp.PinnedBuffer(n_big * 512)
        side = torch.cuda.Stream()
        h.gather_decompress_host(big, n_big, pout.view(np.uint8, (n_big, 512)), side.cuda_stream)
        assert np.array_equal(pout.view(np.uint8, (n_big, 512)), want)
        pout.free()
    h.destroy()
    pin.free()


@pytest.mark.parametrize("rb,n_big", [(100, 90_001), (12, 700_003), (516, 70_001)])
def test_host_entry_chunks_with_odd_row_sizes(rb, n_big):
    """ibp_gather_decompress_host cuts outputs of >= 8 MB (2 chunks) / >= 32 MB (4 chunks) into chunks; with row_bytes not a
    multiple of 16 the chunk borders must fall on rows whose output offset is 16-byte aligned (a border at an arbitrary row
    made ibp_gather_decompress reject the chunk with INVALID_ARG).  Pageable destination = the staged path; ids repeat."""
    n = 5000
    X = (datagen.random_bytes(n * rb, 31 + rb).reshape(n, rb) & datagen.random_bytes(rb, 32)[None, :]) | 0x02
    h = ibp.ibp_build(X, rb, 0, 50, align_bytes=16).upload_metadata(0)
    big = np.random.default_rng(rb).integers(0, n, n_big).astype(np.int64)
    for mode in (-1, 0, 1):
        h.set_dedup_mode(mode)
        out = np.zeros((n_big, rb), np.uint8)
        h.gather_decompress_host(big, n_big, out, torch.cuda.current_stream().cuda_stream)
        assert np.array_equal(out, oracle.gather_plain(X, big))
    h.destroy()


def test_configure_limits_grid_and_streams():
    """SM-limited launch and a non-default stream give the same bytes."""
    w = workloads.Tiny()
    X = w.table()
    h = ibp.ibp_build(X, 512, 0, 64).upload_metadata(0)
    ids = w.ids(2)
    want = oracle.gather_plain(X, ids)
    s = torch.cuda.Stream()
    for ctas, warps in ((1, 1), (3, 2), (64, 8), (0, 4)):
        h.configure(ctas, warps)
        ids_d = _dev(ids)
        out = torch.zeros((len(ids), 512), dtype=torch.uint8, device="cuda")
        torch.cuda.synchronize()
        with torch.cuda.stream(s):
            h.gather_decompress(ids_d.data_ptr(), len(ids), out.data_ptr(), s.cuda_stream)
        s.synchronize()
        assert np.array_equal(out.cpu().numpy(), want)
    h.destroy()


# ---------------------------------------------------------------------------------------------------------------------
# thresholded mode (tau < 1): the paper's default codec on the CUDA path (participation bits, raw rows, per-row offsets)
# ---------------------------------------------------------------------------------------------------------------------
def _perturbed(n, rb, seed):
    """Rows with a common structure, some with chunks that break the consensus (non-participating chunks)
    and some fully random (kept raw)."""
    rng = np.random.default_rng(seed)
    keep = datagen.random_bytes(rb, 9)
    X = (datagen.random_bytes(n * rb, 5 + rb).reshape(n, rb) & keep[None, :]) | 0x01
    for r in rng.choice(n, max(1, n // 5), replace=False):
        X[r, rng.integers(0, rb)] ^= 0xFF
    for r in rng.choice(n, n // 20 + 1, replace=False):
        X[r] = datagen.random_bytes(rb, 1000 + int(r))
    return X


@pytest.mark.parametrize("align", [16, 32, 128])
@pytest.mark.parametrize("thr", [(4, 5), (7, 10), (99, 100)])
def test_T_tiny_config_gather(align, thr):
    """BASELINE.json configs[0] under the paper's thresholded codec (tau = 0.8 default)."""
    w = workloads.Tiny()
    X = w.table()
    h = ibp.ibp_build(X, 512, 0, 64, align_bytes=align, threshold=thr).upload_metadata(0)
    ds = oracle.DatasetT(X, 0, 64, *thr)
    assert h.info().n_rows_raw == ds.n_raw
    for it in range(3):
        ids = w.ids(it)
        for order_mode, dedup in ((0, 0), (1, 0), (1, 1)):
            h.set_order_mode(order_mode).set_dedup_mode(dedup)
            got = _gather(h, ids)
            assert np.array_equal(got, ds.gather_decompress(ids))          # (c2) the oracle codec
            assert np.array_equal(got, oracle.gather_plain(X, ids))        # (c1) the plain definition
    h.destroy()


@pytest.mark.parametrize("kind,param,n,rb,align,thr", [
    (0, 7, 50, 12, 16, (4, 5)), (0, 64, 3000, 64, 32, (4, 5)), (0, 1000, 10, 8, 16, (4, 5)), (0, 16, 40, 4, 16, (3, 4)),
    (1, 5, 203, 32, 16, (4, 5)), (1, 8, 64, 16, 32, (4, 5)), (0, 33, 1000, 100, 32, (7, 10)), (0, 128, 700, 256, 32, (4, 5)),
    (0, 256, 1500, 512, 32, (4, 5)), (0, 50, 333, 1024, 64, (4, 5)), (0, 20, 77, 4096, 64, (4, 5)), (1, 6, 600, 2048, 16, (9, 10)),
    (0, 9, 100, 516, 16, (4, 5)), (0, 1 << 30, 2000, 128, 32, (4, 5)), (0, 4, 30, 8192, 128, (4, 5)),
    (0, 16, 1000, 256, 16, (4, 5)), (0, 5, 333, 128, 16, (3, 4)), (0, 3, 700, 512, 16, (4, 5)), (1, 32, 2100, 256, 16, (4, 5)),
    (1, 86, 1000, 256, 16, (4, 5)), (1, 7, 500, 512, 32, (7, 10)), (1, 3, 100, 128, 16, (4, 5)), (0, 1 << 30, 3000, 512, 16, (9, 10)),
])
def test_T_ragged_shapes_gather_and_resident(kind, param, n, rb, align, thr):
    """W=1,2,4 and 1..16 passes, ragged last groups, strided groups, one global group; rows with non-participating chunks
    and raw rows; gather (orders, dedup), zero-copy range, resident decode, partial ranges starting at any row."""
    X = _perturbed(n, rb, rb + n)
    gp = min(param, n) if kind == 0 else param
    h = ibp.ibp_build(X, rb, kind, gp, align_bytes=align, threshold=thr).upload_metadata(0)
    ds = oracle.DatasetT(X, kind, gp, *thr)
    info = h.info()
    assert info.n_rows_raw == ds.n_raw and info.packed_bytes_bytealigned == ds.stored_bytes
    ids = np.concatenate([(datagen.u64(777, 3) % np.uint64(n)).astype(np.int64), np.arange(n, dtype=np.int64)])
    want = ds.gather_decompress(ids)
    assert np.array_equal(want, oracle.gather_plain(X, ids))
    for mode in (0, 1):
        h.set_order_mode(mode)
        for dd in (0, 1):
            h.set_dedup_mode(dd)
            assert np.array_equal(_gather(h, ids), want)
    for sm in (0, 1, 2):                                                    # per-row fetch kernel / TMA stream kernels (sub-warp, row-per-warp)
        h.set_stream_mode(sm)
        assert np.array_equal(_resident(h, 0, n), X)
        assert np.array_equal(_range(h, 0, n), X)
        if n > 2 * gp:
            first = gp * ((n // gp) // 2)
            assert np.array_equal(_resident(h, first, n - first), X[first:])
            assert np.array_equal(_range(h, first, gp), X[first:first + gp])
        if kind == 0 and n > 5:
            assert np.array_equal(_resident(h, 3, n - 5), X[3:n - 2])       # per-row offsets: any row starts a unit
    h.destroy()


@pytest.mark.parametrize("rb,G,n,raw_frac", [(512, 64, 1500, 1.0), (256, 16, 3000, 1.0), (512, 256, 2000, 0.6), (256, 128, 2500, 0.5), (128, 8, 900, 1.0),
                                             (512, 256, 3000, -0.7), (256, 512, 4000, -0.8)])
def test_T_chunks_larger_than_a_stage(rb, G, n, raw_frac):
    """Thresholded stream decode when most rows are kept raw: a chunk of NW pieces then exceeds one shared-memory stage
    and is loaded as sub-loads into consecutive stages; the producer and every consumer warp take that decision from the same
    two row offsets.  Contiguous ranges from the host store, resident decode, ranges starting off a group boundary, spans."""
    rng = np.random.default_rng(rb + n)
    X = _perturbed(n, rb, 3 * rb + n)
    # raw_frac < 0: the raw rows are the TAIL of the table (from |raw_frac| * n on), so the table's average stored row is small -- units
    # are sized for it -- while every unit of the tail exceeds a stage and is split
    raw = rng.random(n) < raw_frac if raw_frac >= 0 else np.arange(n) >= int(-raw_frac * n)
    X[raw] = rng.integers(0, 256, size=(int(raw.sum()), rb), dtype=np.uint8)
    h = ibp.ibp_build(X, rb, 0, G, align_bytes=16, threshold=(4, 5)).upload_metadata(0)
    ds = oracle.DatasetT(X, 0, G, 4, 5)
    assert h.info().n_rows_raw == ds.n_raw
    if G >= 64:
        assert ds.n_raw >= int(0.9 * raw.sum())                                 # random rows in a large group: nothing to gain, kept raw
    ids = np.arange(0, n, 3, dtype=np.int64)
    assert np.array_equal(ds.gather_decompress(ids), X[ids])
    ds.close()
    for sm in (1, 2):
        h.set_stream_mode(sm)
        assert np.array_equal(_resident(h, 0, n), X)
        assert np.array_equal(_range(h, 0, n), X)
        assert np.array_equal(_resident(h, 5, n - 9), X[5:n - 4])
        assert np.array_equal(_range(h, G + 3, n - G - 3), X[G + 3:])
    h.destroy()
    span = 4 * G
    hs = ibp.ibp_build(X[: n // span * span], rb, 0, G, align_bytes=16, index_span=span, threshold=(4, 5)).upload_metadata(0)
    ns = n // span
    sids = np.array([ns // 2, 0, ns - 1, ns // 2], np.int64)
    assert np.array_equal(_gather(hs, sids, span=span), oracle.gather_plain(X, sids, span))
    hs.destroy()


@pytest.mark.parametrize("rb,G,n", [(256, 16, 5000), (256, 128, 7001), (512, 256, 4099), (128, 64, 9000)])
def test_T_stream_grid_limits(rb, G, n):
    """The thresholded stream kernel's consumers follow the producer's units until the descriptor marks the CTA's last one:
    one CTA walking every chunk, a few CTAs (more chunks than CTAs, uneven shares), the default grid; split units (raw rows) and a
    ragged last piece included.  Ranges from the host store, resident decode, page spans."""
    rng = np.random.default_rng(7 * rb + n)
    X = _perturbed(n, rb, rb + n)
    raw = (np.arange(n) >= n - n // 5) | (rng.random(n) < 0.05)               # a raw tail (its units are split) and scattered raw rows
    X[raw] = rng.integers(0, 256, size=(int(raw.sum()), rb), dtype=np.uint8)
    h = ibp.ibp_build(X, rb, 0, G, align_bytes=16, threshold=(4, 5)).upload_metadata(0)
    for max_ctas in (1, 3, 0):
        h.configure(max_ctas, 0)
        assert np.array_equal(_resident(h, 0, n), X), f"resident, max_ctas={max_ctas}"
        assert np.array_equal(_range(h, 0, n), X), f"range, max_ctas={max_ctas}"
        assert np.array_equal(_resident(h, G, n - G - 1), X[G:n - 1]), f"resident off the end, max_ctas={max_ctas}"
    h.destroy()
    span = 2 * G
    ns = n // span
    hs = ibp.ibp_build(X[: ns * span], rb, 0, G, align_bytes=16, index_span=span, threshold=(4, 5)).upload_metadata(0)
    sids = rng.integers(0, ns, 37)
    for max_ctas in (1, 5, 0):
        hs.configure(max_ctas, 0)
        assert np.array_equal(_gather(hs, sids, span=span), oracle.gather_plain(X, sids, span)), f"spans, max_ctas={max_ctas}"
    hs.destroy()


def test_T_edge_cases_and_spans():
    rb = 256
    r = datagen.random_bytes(rb, 3)
    special = np.frombuffer(np.array([np.nan, -0.0, 1e-45, np.inf, -np.inf, 0.0, 1.0, -1.0] * 8, np.float32).tobytes(), np.uint8)
    # group 0: identical rows (every chunk participates, nothing but participation bits is stored);
    # group 1: rows and complements (no bit reaches T: Mask = 0, every row raw); group 2: special float patterns
    X = np.stack([r] * 4 + [r, ~r, r, ~r] + [special, special ^ 1, special, special ^ 0x80])
    h = ibp.ibp_build(X, rb, 0, 4, align_bytes=16, threshold=(3, 4)).upload_metadata(0)
    ds = oracle.DatasetT(X, 0, 4, 3, 4)
    data, stored, comp = h.row_info(0)
    assert comp and data.size == rb // 4 // 8 and stored == 16              # 64 participation bits = 8 bytes
    assert all(not h.row_info(i)[2] for i in range(4, 8))                   # kept raw
    ids = np.array([0, 3, 3, 3, 4, 5, 11, 8, 9, 10, 0, 7], np.int64)
    assert np.array_equal(_gather(h, ids), X[ids])
    assert np.array_equal(_gather(h, ids), ds.gather_decompress(ids))
    assert _gather(h, np.zeros(0, np.int64)).shape[0] == 0
    assert np.array_equal(_resident(h, 0, 12), X)
    assert np.array_equal(_resident(h, 5, 6), X[5:11])
    h.destroy()
    # index_span > 1 (KV-style page spans) in thresholded mode
    w = workloads.KV(layers=1, pages=8)
    Xk = w.table()
    hk = ibp.ibp_build(Xk, w.row_bytes, w.group_kind, w.group_param, align_bytes=16, index_span=w.index_span, threshold=(4, 5)).upload_metadata(0)
    ids = np.array([3, 0, 5, 5, 1], np.int64)
    for sm in (0, 1, 2):
        hk.set_stream_mode(sm)
        assert np.array_equal(_gather(hk, ids, span=w.index_span), oracle.gather_plain(Xk, ids, w.index_span))
    hk.destroy()


@pytest.mark.parametrize("thr,flags,cap", [((1, 1), 0, 0), ((4, 5), 0, 0), ((4, 5), ibp.IBP_FLAG_SLOT_LAYOUT, 0)])
def test_shared_store_gather(thr, flags, cap):
    """One store for all ranks: a handle exported into a POSIX shared-memory segment and opened again -- here twice
    in one process, standing in for two ranks -- is page-locked and GPU-mapped by ibp_upload_metadata and decodes the same bytes
    as the original: random gather, range, resident."""
    import os
    name = f"/ibp_gputest_{os.getpid()}"
    w = workloads.GNN(n_rows=30_000, batch=4000)
    X = _u8(w.table())
    h0 = ibp.ibp_build(X, 512, 0, 256, align_bytes=32 if not flags else 16, threshold=thr, flags=flags | ibp.IBP_FLAG_PAGEABLE_STORE, capacity_rows=cap)
    h0.export_shared(name, numa_policy=1)
    h0.destroy()                                                            # only the segment is left
    ha = ibp.ibp_open_shared(name).upload_metadata(0)
    hb = ibp.ibp_open_shared(name).upload_metadata(0)
    ibp.ibp_unlink_shared(name)                                             # the mappings keep the memory alive
    assert ha.info().store_kind == ibp.IBP_STORE_SHARED and ha.info().device == 0
    ids = w.ids(0)
    for h in (ha, hb):
        assert np.array_equal(_gather(h, ids), X[ids])
        assert np.array_equal(_range(h, 256 * 3, 5000), X[768:5768])
        assert np.array_equal(_resident(h, 0, 2048), X[:2048])
    ha.destroy()
    assert np.array_equal(_gather(hb, ids[:100]), X[ids[:100]])             # one rank leaving does not disturb the other
    hb.destroy()
    assert ibp.ibp_device_numa_node(0) >= -1


def test_link_probes():
    """The ceilings bench.py reports are measured by the library itself: sane values and argument checks."""
    sps, gbs = ibp.ibp_measure_random_read(0, 64 << 20, 128, 1)
    assert sps > 1e7 and abs(gbs - sps * 128e-9) < 1e-6 * gbs + 1e-9
    assert 5 < ibp.ibp_measure_zero_copy_read(0, 64 << 20, 1) < 200
    for bad in [(64 << 20, 100), (64 << 20, 1024), (1 << 10, 128)]:
        with pytest.raises(ibp.IbpError) as e:
            ibp.ibp_measure_random_read(0, bad[0], bad[1], 1)
        assert e.value.status == 1
