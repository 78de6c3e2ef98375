"""CPU-only: the library's host compressor (ibp_build, S0/S0') against the independent oracle.

The library keeps the canonical bit order, so Mask, Bitval, k_g AND the packed bytes of every row must equal the
oracle's, and the oracle's unpacker must decode the library's store back to the original rows.
"""
import numpy as np
import pytest

import oracle
from paper_2605_30728_b200 import binding as ibp
from paper_2605_30728_b200 import datagen, workloads


def _check_against_oracle(X, kind, param, align, span=1, rows_to_check=None, build=None):
    """build: optional callable (Xb, rb, kind, param, align, span) -> Handle, for the GPU-side compressor's parity tests."""
    Xb = np.ascontiguousarray(X).view(np.uint8).reshape(X.shape[0], -1)
    n, rb = Xb.shape
    if build is None:
        h = ibp.ibp_build(Xb, rb, kind, param, align_bytes=align, index_span=span, flags=ibp.IBP_FLAG_PAGEABLE_STORE)
    else:
        h = build(Xb, rb, kind, param, align, span)
    ds = oracle.Dataset(Xb, kind, param)
    info = h.info()
    assert info.n_groups == ds.n_groups
    assert info.metadata_bytes == ds.metadata_bytes == 2 * rb * ds.n_groups       # fixed size per group
    assert info.packed_bytes_bytealigned == ds.packed_bytes                        # sum of ceil(k/8)
    assert info.packed_bytes_rows >= info.packed_bytes_bytealigned
    assert info.packed_bytes_stored >= info.packed_bytes_rows
    for g in range(ds.n_groups):
        m, b, k = h.metadata_host(g)
        assert k == ds.k_bits(g)
        assert np.array_equal(m, ds.mask(g)) and np.array_equal(b, ds.bitval(g))
    A = info.align_bytes
    rows = range(n) if rows_to_check is None else rows_to_check
    for r in rows:
        g = r // param if kind == 0 else r % param
        data, k = h.packed_row(r)
        want = ds.packed_row(r)
        assert k == ds.k_bits(g)
        assert data.size == -(-want.size // A) * A                                 # stride = roundup(ceil(k/8), A)
        assert np.array_equal(data[: want.size], want)                             # canonical packed bytes
        assert not data[want.size:].any()                                          # zero padding
        assert np.array_equal(oracle.unpack_row(data, ds.mask(g), ds.bitval(g)), Xb[r])
    # whole-range accessor: contiguous, starts at row 0, covers every row
    ptr, nbytes = h.packed_range(0, n)
    assert nbytes >= info.packed_bytes_rows and nbytes % 16 == 0
    h.destroy()
    ds.close()


@pytest.mark.parametrize("align", [1, 4, 16, 32, 128])
def test_tiny_blocked(align):
    _check_against_oracle(workloads.Tiny(n_rows=512).table(), 0, 64, align)


@pytest.mark.parametrize("kind,param,n,rb", [(0, 7, 50, 12), (0, 64, 1000, 64), (0, 1000, 10, 8), (1, 5, 203, 32),
                                             (1, 8, 64, 16), (1, 3, 2, 4), (0, 1, 9, 20), (0, 16, 40, 4)])
def test_small_shapes_ragged(kind, param, n, rb):
    X = (datagen.random_bytes(n * rb, 5).reshape(n, rb) & 0x5A) | 0x21
    _check_against_oracle(X, kind, param, 16)
    _check_against_oracle(X, kind, param, 1)


def test_workload_shapes():
    g = workloads.GNN(n_rows=4096)
    _check_against_oracle(g.table(), 0, 256, 32, rows_to_check=range(0, 4096, 37))
    d = workloads.DLRM(rows_per_table=1024, n_tables=2)
    _check_against_oracle(d.table(), 0, 128, 32, rows_to_check=range(0, 2048, 17))
    kv = workloads.KV(layers=1, pages=4, heads=4)
    _check_against_oracle(kv.table(), 0, 16, 16, span=64, rows_to_check=range(0, kv.n_rows, 5))
    w = workloads.WeightMatrix(128, 512)
    _check_against_oracle(w.table(), 1, 4, 16, rows_to_check=range(0, w.n_rows, 3))


def test_degenerate_groups():
    rb = 64
    r = datagen.random_bytes(rb, 3)
    same = np.repeat(r[None, :], 10, axis=0)                     # k = 0: nothing stored
    h = ibp.ibp_build(same, rb, 0, 10, flags=ibp.IBP_FLAG_PAGEABLE_STORE)
    m, b, k = h.metadata_host(0)
    assert k == 0 and np.all(m == 0xFF) and np.array_equal(b, r)
    assert h.info().packed_bytes_rows == 0
    h.destroy()
    both = np.stack([r, ~r])                                     # no invariant bit: packed == raw (reading R13)
    h = ibp.ibp_build(both, rb, 0, 2, align_bytes=1, flags=ibp.IBP_FLAG_PAGEABLE_STORE)
    m, b, k = h.metadata_host(0)
    assert k == 8 * rb and not m.any() and not b.any()
    for i in range(2):
        data, _ = h.packed_row(i)
        assert np.array_equal(data, both[i])
    h.destroy()


def test_soft_pext_fallback_matches(monkeypatch):
    """63/64-bit fill edge cases of the word-wise packer: masks that make the accumulator wrap at every offset."""
    rb = 64
    for seed in range(40):
        rng = np.random.default_rng(seed)
        keep = rng.integers(0, 256, rb, dtype=np.uint8) | (0xFF if seed % 5 == 0 else 0)
        base = datagen.random_bytes(rb, 100 + seed) & ~keep
        rows = (datagen.random_bytes(8 * rb, 200 + seed).reshape(8, rb) & keep) | base
        rows[0] = base
        rows[1] = base | keep
        _check_against_oracle(rows, 0, 8, 1)


def test_argument_errors():
    X = np.zeros((8, 16), np.uint8)
    with pytest.raises(ibp.IbpError) as e:
        ibp.ibp_build(X.reshape(-1)[:126].reshape(9, 14), 14, 0, 4)
    assert e.value.status == 1                                   # row_bytes not a multiple of 4 (reading R11)
    with pytest.raises(ibp.IbpError) as e:
        ibp.ibp_build(X, 16, 0, 4, threshold=(1, 2))
    assert e.value.status == 1                                   # tau must exceed 1/2 (reading R3)
    with pytest.raises(ibp.IbpError) as e:
        ibp.ibp_build(X, 16, 0, 4, threshold=(4, 5), align_bytes=4)
    assert e.value.status == 1                                   # thresholded rows start on 16-byte units
    with pytest.raises(ibp.IbpError) as e:
        ibp.ibp_build(X, 16, 0, 4, align_bytes=48)
    assert e.value.status == 1
    with pytest.raises(ibp.IbpError) as e:
        ibp.ibp_build(X, 16, 1, 4, index_span=2)
    assert e.value.status == 1
    h = ibp.ibp_build(X, 16, 0, 4, flags=ibp.IBP_FLAG_PAGEABLE_STORE)
    with pytest.raises(ibp.IbpError) as e:
        h.packed_range(2, 4)                                     # must start a layout unit
    assert e.value.status == 1
    with pytest.raises(ibp.IbpError) as e:
        h.gather_decompress(0, 1, 0)                             # before upload: BAD_STATE, never a silent fallback
    assert e.value.status == 4
    h.destroy()


def test_batch_link_bytes():
    w = workloads.Tiny(n_rows=256)
    X = w.table()
    h = ibp.ibp_build(X, 512, 0, 64, align_bytes=32, flags=ibp.IBP_FLAG_PAGEABLE_STORE)
    ids = np.array([0, 5, 5, 70, 255, 0], np.int64)
    nu, stored, ba = h.batch_link_bytes(ids)
    assert nu == 4
    want_s = want_b = 0
    for r in (0, 5, 70, 255):
        data, k = h.packed_row(r)
        want_s += data.size
        want_b += (k + 7) // 8
    assert (stored, ba) == (want_s, want_b)
    h.destroy()


# ---------------------------------------------------------------------------------------------------------------------
# thresholded mode (tau < 1; the paper's default codec): the library's compressor against oracle.DatasetT
# ---------------------------------------------------------------------------------------------------------------------
def _check_T_against_oracle(X, kind, param, thr, align=32, rows_to_check=None, build=None):
    Xb = np.ascontiguousarray(X).view(np.uint8).reshape(X.shape[0], -1)
    n, rb = Xb.shape
    if build is None:
        h = ibp.ibp_build(Xb, rb, kind, param, align_bytes=align, flags=ibp.IBP_FLAG_PAGEABLE_STORE, threshold=thr)
    else:
        h = build(Xb, rb, kind, param, align, thr)
    ds = oracle.DatasetT(Xb, kind, param, thr[0], thr[1])
    info = h.info()
    assert info.thresholded == 1 and (info.threshold_num, info.threshold_den) == thr
    assert info.n_groups == ds.n_groups
    assert info.metadata_bytes == ds.metadata_bytes
    assert info.n_rows_raw == ds.n_raw
    assert info.packed_bytes_bytealigned == ds.stored_bytes                 # sum of the byte-aligned row sizes
    assert info.rowflag_bytes == 4 * (-(-n // 32))                          # one bit per row, in 32-bit words
    for g in range(ds.n_groups):
        m, b, k = h.metadata_host(g)
        assert np.array_equal(m, ds.mask(g)) and np.array_equal(b, ds.bitval(g))
        assert k == 8 * rb - int(np.unpackbits(ds.mask(g)).sum())
    A = info.align_bytes
    total = 0
    for r in (range(n) if rows_to_check is None else rows_to_check):
        data, stored, comp = h.row_info(r)
        want, want_comp = ds.row(r)
        assert comp == want_comp
        assert np.array_equal(data, want)                                   # canonical bytes: participation bits, payloads
        assert stored == -(-want.size // A) * A
        total += stored
    if rows_to_check is None:
        assert total == info.packed_bytes_rows
        ptr, nbytes = h.packed_range(0, n)
        assert nbytes == total
        nu, st, ba = h.batch_link_bytes(np.arange(n, dtype=np.int64))
        assert (nu, st, ba) == (n, total, ds.stored_bytes)
    h.destroy()
    ds.close()


def test_T_golden_worked_example_rows_padded_to_4_bytes():
    """The hand-worked example of tests/golden/worked_example_thresholded.txt uses 1-byte chunks; the library fixes 4-byte
    chunks (reading R10), so the same five tensors are checked through the oracle at CS=4 here and the fixture itself
    in test_oracle_pins.py."""
    rows = np.array([[0xB4, 0x0F, 0xB4, 0x0F], [0xA6, 0x0F, 0xA6, 0x0F], [0xB5, 0x0F, 0xB5, 0x0F], [0xA4, 0x1F, 0xA4, 0x1F],
                     [0x36, 0x0E, 0x36, 0x0E]] * 3, np.uint8)
    _check_T_against_oracle(rows, 0, 5, (4, 5), align=16)


@pytest.mark.parametrize("kind,param,n,rb,thr", [(0, 64, 1000, 64, (4, 5)), (0, 7, 50, 12, (4, 5)), (0, 256, 700, 512, (7, 10)),
                                                 (1, 5, 203, 32, (4, 5)), (1, 6, 600, 256, (9, 10)), (0, 1 << 30, 900, 128, (4, 5)),
                                                 (0, 300, 1000, 8, (4, 5)), (0, 16, 100, 2048, (3, 4))])
def test_T_shapes_against_oracle(kind, param, n, rb, thr):
    rng = np.random.default_rng(rb + n)
    keep = datagen.random_bytes(rb, 9)
    X = (datagen.random_bytes(n * rb, 5 + rb).reshape(n, rb) & keep[None, :]) | 0x01
    # rows that break the consensus in some chunks (non-participating chunks) and some that break all (raw rows)
    for r in rng.choice(n, n // 5, replace=False):
        X[r, rng.integers(0, rb)] ^= 0xFF
    for r in rng.choice(n, n // 20 + 1, replace=False):
        X[r] = datagen.random_bytes(rb, 1000 + int(r))
    _check_T_against_oracle(X, kind, min(param, n) if kind == 0 else param, thr)


def test_T_workload_shapes():
    w = workloads.GNN(n_rows=4096)
    X = np.concatenate([w.rows(0, 1024), w.rows(3000, 1024)])
    _check_T_against_oracle(X, 0, 256, (4, 5))
    _check_T_against_oracle(X, 0, 1 << 20, (4, 5), rows_to_check=range(0, 2048, 7))   # one global Mask/Bitval
    t = workloads.Tiny(n_rows=512).table()
    _check_T_against_oracle(t, 0, 64, (4, 5), align=16)


def test_gnn_interleaved_variant_recipe_and_ratio():
    """Reading R15's secondary workload: row types drawn per row (about 70/30), any row range regenerates alone, and the host
    build of a table whose groups all mix both types keeps almost none of the sparse rows' compressibility (SURVEY 8(d):
    "the sparse rows lose their 4.6x")."""
    w = workloads.GNN(n_rows=8192, batch=64, interleaved=True)
    X = w.table()
    assert np.array_equal(w.rows(3000, 77).view(np.uint32), X[3000:3077].view(np.uint32))
    sparse = ((X == 0) | (X == 1)).all(axis=1)
    assert 0.25 < sparse.mean() < 0.35
    mixed = ibp.ibp_build(X, 512, 0, 256, align_bytes=1, flags=ibp.IBP_FLAG_PAGEABLE_STORE)
    typed = ibp.ibp_build(workloads.GNN(n_rows=8192, batch=64).table(), 512, 0, 256, align_bytes=1, flags=ibp.IBP_FLAG_PAGEABLE_STORE)
    r_mixed = X.nbytes / mixed.info().packed_bytes_bytealigned
    r_typed = X.nbytes / typed.info().packed_bytes_bytealigned
    assert r_mixed < r_typed and r_mixed < 1.9
    mixed.destroy()
    typed.destroy()


# ---------------------------------------------------------------------------------------------------------------------
# slot layout (PAPER.md:361 in-place storage) built by the host compressor
# ---------------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("kind,param,n,rb,align,cap", [(0, 1 << 20, 300, 64, 16, 400), (1, 6, 90, 32, 16, 0), (0, 16, 100, 256, 32, 112), (1, 4, 40, 516, 16, 64)])
def test_slot_layout_host_build(kind, param, n, rb, align, cap):
    """IBP_FLAG_SLOT_LAYOUT: row r lies at r * roundup(row_bytes, A); its first `size` bytes are the oracle's stored bytes of
    that row, the rest of the slot and every unused slot are zero; one size byte per slot, no offsets."""
    X = (datagen.random_bytes(n * rb, 400 + rb).reshape(n, rb) & datagen.random_bytes(rb, 401)[None, :]) | 0x08
    X[::7, 1] ^= 0x33
    X[5] = datagen.random_bytes(rb, 402)
    gp = min(param, max(cap, n)) if kind == 0 and param >= (1 << 20) else param
    h = ibp.ibp_build(X, rb, kind, gp, align_bytes=align, threshold=(4, 5), capacity_rows=cap,
                      flags=ibp.IBP_FLAG_PAGEABLE_STORE | ibp.IBP_FLAG_SLOT_LAYOUT)
    ds = oracle.DatasetT(X, kind, gp, 4, 5)
    info = h.info()
    slot = -(-rb // align) * align
    capacity = cap or n
    assert info.slot_bytes == slot and info.capacity_rows == capacity and info.rowsize_bytes == capacity and info.rowoffset_bytes == 0
    assert info.packed_bytes_stored >= capacity * slot and info.packed_bytes_bytealigned == ds.stored_bytes
    assert info.n_rows_raw == ds.n_raw
    base = h.row_ptr(0)
    img = ds.slot_image(capacity, slot)
    ptr, nb = h.packed_range(0, n)
    assert ptr == base and nb == n * slot
    got = h.packed_view(base, capacity * slot).reshape(capacity, slot)
    assert np.array_equal(got, img)                                             # every slot byte, used or not
    for r in (0, 5, n - 1):
        data, stored, comp = h.row_info(r)
        want, want_comp = ds.row(r)
        assert comp == want_comp and np.array_equal(data, want)
        assert stored == -(-want.size // align) * align and h.row_ptr(r) == base + r * slot
    h.destroy()
    ds.close()


def test_slot_layout_argument_checks():
    X = datagen.random_bytes(64 * 32, 1).reshape(64, 32)
    with pytest.raises(ibp.IbpError) as e:                                      # strict rows of a group all have one size: no slots
        ibp.ibp_build(X, 32, 0, 16, flags=ibp.IBP_FLAG_PAGEABLE_STORE | ibp.IBP_FLAG_SLOT_LAYOUT)
    assert e.value.status == 1
    with pytest.raises(ibp.IbpError) as e:
        ibp.ibp_build(X, 32, 0, 16, threshold=(4, 5), capacity_rows=10, flags=ibp.IBP_FLAG_PAGEABLE_STORE | ibp.IBP_FLAG_SLOT_LAYOUT)
    assert e.value.status == 1
    # the parameter struct of version 0.3 (no capacity_rows) is still accepted
    import ctypes as C
    p = ibp.ibp_build_params(C.sizeof(ibp.ibp_build_params) - 8, 32, 64, 0, 16, 1, 1, 16, 1, ibp.IBP_FLAG_PAGEABLE_STORE, 0, 0)
    hp = C.c_void_p()
    assert ibp.lib().ibp_build(X.ctypes.data, C.byref(p), C.byref(hp)) == 0
    h = ibp.Handle(hp)
    assert h.info().n_rows == 64
    h.destroy()
    h = ibp.ibp_build(X, 32, 0, 1 << 20, threshold=(4, 5), capacity_rows=100, flags=ibp.IBP_FLAG_PAGEABLE_STORE | ibp.IBP_FLAG_SLOT_LAYOUT)
    with pytest.raises(ibp.IbpError) as e:                                      # append needs the GPU (no CPU fallback)
        h.append_rows_device(X.ctypes.data, 4)
    assert e.value.status == 4
    h.destroy()
