"""Guard-band checks of every entry point that writes device memory (the memcheck the suite can run everywhere).

compute-sanitizer is not available on the GPU pool these tests run on (profiles/r02_sanitizer.md), so out-of-bounds WRITES are
caught here instead: every output buffer sits between two guard bands of a known pattern, the decoded rows are compared with the
plain gather (oracle c1) and both bands must come back untouched.  Shapes are the ones the fast paths do not special-case: odd row
sizes, ragged last groups, partial matrix rows, batches that are not a multiple of any tile, thresholded rows with raw rows among
them, every kernel family (random rows with and without the pre-passes, spans, ranges, several ranges in one launch, resident
decode, the compressed cache, the uncompressed baseline, the GPU-side build and append through their results).
"""
import numpy as np
import pytest

import oracle
from paper_2605_30728_b200 import binding as ibp
from paper_2605_30728_b200 import datagen

pytestmark = pytest.mark.gpu
torch = pytest.importorskip("torch")

GUARD = 4096
PAT = 0xC3


def _stream():
    return torch.cuda.current_stream().cuda_stream


class Guarded:
    """n_bytes of device memory between two guard bands; `ptr` is 16-byte aligned"""

    def __init__(self, n_bytes, fill=0x5A):
        self.n = n_bytes
        self.buf = torch.full((GUARD + max(16, n_bytes) + GUARD,), PAT, dtype=torch.uint8, device="cuda")
        self.buf[GUARD:GUARD + n_bytes] = fill
        self.ptr = self.buf.data_ptr() + GUARD
        assert self.ptr % 16 == 0

    def check(self, rows, rb):
        torch.cuda.synchronize()
        a = self.buf.cpu().numpy()
        assert (a[:GUARD] == PAT).all(), "bytes in front of the output were overwritten"
        assert (a[GUARD + self.n:] == PAT).all(), "bytes behind the output were overwritten"
        return a[GUARD:GUARD + self.n].reshape(rows, rb) if rows else a[:0].reshape(0, rb)


def _dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def _table(n, rb, seed, raw_every=0):
    X = (datagen.random_bytes(n * rb, seed).reshape(n, rb) & datagen.random_bytes(rb, seed + 1)[None, :]) | 0x01
    if raw_every:
        for r in range(3, n, raw_every):
            X[r] = datagen.random_bytes(rb, seed + 100 + r)
    return X


SHAPES = [(0, 64, 1000, 512, 32), (0, 7, 50, 100, 16), (0, 256, 700, 128, 32), (1, 5, 203, 256, 16), (1, 86, 86 * 9 + 13, 256, 16),
          (0, 16, 16 * 37 + 5, 256, 16), (0, 3, 2, 36, 16), (0, 33, 999, 1028, 64)]


@pytest.mark.parametrize("kind,param,n,rb,align", SHAPES)
@pytest.mark.parametrize("thr", [(1, 1), (4, 5)])
def test_guard_bands_every_decode_entry_point(kind, param, n, rb, align, thr):
    X = _table(n, rb, 31 + rb + n, raw_every=17 if thr[0] != thr[1] else 0)
    h = ibp.ibp_build(X, rb, kind, param, align_bytes=align, threshold=thr).upload_metadata(0)
    rng = np.random.default_rng(n)
    # ---- random rows: plain, ordered, de-duplicated, both fetch engines; batch sizes around warp / CTA multiples
    for cnt in (1, 31, 257, 3 * n + 1):
        ids = rng.integers(0, n, cnt).astype(np.int64)
        want = oracle.gather_plain(X, ids)
        for fetch, order, dedup in ((1, 0, 0), (1, 1, 1), (0, 1, 0), (0, 0, 1)):
            h.set_fetch_mode(fetch).set_order_mode(order).set_dedup_mode(dedup)
            g = Guarded(cnt * rb)
            h.gather_decompress(_dev(ids).data_ptr(), cnt, g.ptr, _stream())
            assert np.array_equal(g.check(cnt, rb), want), (cnt, fetch, order, dedup)
    h.set_fetch_mode(1).set_order_mode(-1).set_dedup_mode(-1)
    # ---- contiguous ranges from the host store and from HBM, through both the stream kernels and the per-row kernel
    unit = param
    starts = [0] if n < 2 * unit else [0, unit * ((n // unit) // 2)]
    for first in starts:
        for cnt in {n - first, min(n - first, unit), min(n - first, 2 * unit + 1)}:
            want = X[first:first + cnt]
            ptr, nbytes = h.packed_range(first, cnt)
            packed = _dev(h.packed_view(ptr, nbytes).copy()) if nbytes else torch.zeros(16, dtype=torch.uint8, device="cuda")
            for sm in (1, 0, 2):
                h.set_stream_mode(sm)
                g = Guarded(cnt * rb)
                h.gather_decompress_range(first, cnt, g.ptr, _stream())
                assert np.array_equal(g.check(cnt, rb), want), ("range", first, cnt, sm)
                g = Guarded(cnt * rb)
                h.decompress_resident(packed.data_ptr(), first, cnt, g.ptr, _stream())
                assert np.array_equal(g.check(cnt, rb), want), ("resident", first, cnt, sm)
            h.set_stream_mode(1)
            # the same range twice in one launch list, each into its own guarded buffer (ibp_decode_ranges)
            ga, gb = Guarded(cnt * rb), Guarded(cnt * rb)
            ibp.ibp_decode_ranges([(h, packed.data_ptr(), first, cnt, ga.ptr), (h, None, first, cnt, gb.ptr)], _stream())
            assert np.array_equal(ga.check(cnt, rb), want) and np.array_equal(gb.check(cnt, rb), want)
    # ---- the compressed cache in front of the store: hits and misses
    c = ibp.Cache(h, max(256, h.info().packed_bytes_stored // 2), 2)
    c.insert(rng.permutation(n)[: n // 2 + 1])
    ids = rng.integers(0, n, 2 * n + 3).astype(np.int64)
    g = Guarded(len(ids) * rb)
    c.gather_decompress(_dev(ids).data_ptr(), len(ids), g.ptr, _stream())
    assert np.array_equal(g.check(len(ids), rb), oracle.gather_plain(X, ids))
    c.destroy()
    h.destroy()


@pytest.mark.parametrize("G,span,n_spans,rb,thr", [(16, 64, 40, 256, (1, 1)), (16, 64, 40, 256, (4, 5)), (8, 24, 33, 512, (1, 1)), (32, 32, 17, 128, (4, 5))])
def test_guard_bands_span_gather(G, span, n_spans, rb, thr):
    n = span * n_spans
    X = _table(n, rb, 77 + rb, raw_every=29 if thr[0] != thr[1] else 0)
    h = ibp.ibp_build(X, rb, 0, G, align_bytes=16, index_span=span, threshold=thr).upload_metadata(0)
    rng = np.random.default_rng(5)
    for cnt in (1, 7, n_spans + 3):
        ids = rng.integers(0, n_spans, cnt).astype(np.int64)
        for sm in (1, 0):
            h.set_stream_mode(sm)
            g = Guarded(cnt * span * rb)
            h.gather_decompress(_dev(ids).data_ptr(), cnt, g.ptr, _stream())
            assert np.array_equal(g.check(cnt * span, rb), oracle.gather_plain(X, ids, span)), (cnt, sm)
    h.destroy()


def test_guard_bands_uncompressed_baseline():
    n, rb = 3001, 112
    X = datagen.random_bytes(n * rb, 3).reshape(n, rb)
    buf = ibp.PinnedBuffer(X.nbytes)
    buf.view(np.uint8, X.shape)[:] = X
    ids = np.random.default_rng(1).integers(0, n, 4099).astype(np.int64)
    for order in (False, True):
        g = Guarded(len(ids) * rb)
        ibp.ibp_gather_uncompressed(buf.dev_ptr, rb, _dev(ids).data_ptr(), len(ids), g.ptr, _stream(), n_rows=n, locality_order=order)
        assert np.array_equal(g.check(len(ids), rb), X[ids])
    buf.free()


@pytest.mark.parametrize("thr", [(1, 1), (4, 5)])
def test_guard_bands_gpu_build_source(thr):
    """ibp_build_device reads the rows from a guarded device buffer and writes only its own store: the source and its bands stay
    as they were, and the store decodes to the rows."""
    n, rb, G = 1234, 256, 64
    X = _table(n, rb, 91, raw_every=13 if thr[0] != thr[1] else 0)
    g = Guarded(n * rb)
    g.buf[GUARD:GUARD + n * rb] = _dev(X.reshape(-1))
    h = ibp.ibp_build_device(g.ptr, n, rb, 0, G, align_bytes=16, threshold=thr)
    assert np.array_equal(g.check(n, rb), X)
    out = Guarded(n * rb)
    h.gather_decompress_range(0, n, out.ptr, _stream())
    assert np.array_equal(out.check(n, rb), X)
    h.destroy()
