"""GPU parity of the appendable slot-layout store (SURVEY 8(f) NEXT #1/#2; PAPER.md:361 in-place slots, :363 per-row bitmask,
:511-513 online KV compression: masks from the prompt tokens, decode-time K/V compressed under them as they are produced).

After every append the CUDA path is compared with (c1) the plain gather of the concatenated table and with (c2) the oracle:
oracle.DatasetT.append gives the stored bytes, the size and the compressed-bit of every appended row, which must equal what
ibp_append_rows_device wrote into the slots of the host store; Mask/Bitval must not change.
"""
import numpy as np
import pytest

import oracle
from paper_2605_30728_b200 import binding as ibp
from paper_2605_30728_b200 import datagen, workloads

pytestmark = pytest.mark.gpu
torch = pytest.importorskip("torch")

SLOT = ibp.IBP_FLAG_SLOT_LAYOUT


def _st():
    return torch.cuda.current_stream().cuda_stream


def _dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def _gather(h, ids, span=1):
    rb = h.info().row_bytes
    ids_d = _dev(np.asarray(ids, np.int64))
    out = torch.full((max(1, len(ids) * span), rb), 0xA5, dtype=torch.uint8, device="cuda")
    h.gather_decompress(ids_d.data_ptr(), len(ids), out.data_ptr(), _st())
    torch.cuda.synchronize()
    return out.cpu().numpy()[: len(ids) * span]


def _range(h, first, n):
    out = torch.full((max(1, n), h.info().row_bytes), 0x3C, dtype=torch.uint8, device="cuda")
    h.gather_decompress_range(first, n, out.data_ptr(), _st())
    torch.cuda.synchronize()
    return out.cpu().numpy()[:n]


def _resident(h, first, n):
    ptr, nbytes = h.packed_range(first, n)
    packed = _dev(h.packed_view(ptr, nbytes).copy())
    out = torch.full((max(1, n), h.info().row_bytes), 0x5A, dtype=torch.uint8, device="cuda")
    h.decompress_resident(packed.data_ptr(), first, n, out.data_ptr(), _st())
    torch.cuda.synchronize()
    return out.cpu().numpy()[:n]


def _table(n, rb, seed):
    X = (datagen.random_bytes(n * rb, seed).reshape(n, rb) & datagen.random_bytes(rb, seed + 1)[None, :]) | 0x10
    rng = np.random.default_rng(seed)
    for r in rng.choice(n, max(1, n // 4), replace=False):
        X[r, rng.integers(0, rb)] ^= 0x5A                                   # chunks that break the consensus
    for r in rng.choice(n, n // 15 + 1, replace=False):
        X[r] = datagen.random_bytes(rb, 5000 + int(r))                       # rows kept raw
    return X


def _check_rows(h, ds, X, rows):
    for r in rows:
        data, stored, comp = h.row_info(int(r))
        want, want_comp = ds.row(int(r))
        assert comp == want_comp and np.array_equal(data, want), f"row {r}"


@pytest.mark.parametrize("builder", ["host", "device"])
@pytest.mark.parametrize("kind,param,n0,rb,align,steps", [
    (0, 1 << 20, 1000, 256, 16, [1, 31, 33, 500, 7]),        # one global Mask/Bitval, appends that straddle flag words
    (1, 24, 240, 512, 32, [24, 48, 5, 19, 240]),             # strided: 24 planes, a token appends one row per plane (online KV)
    (0, 1 << 20, 64, 128, 16, [64, 64]),
    (1, 7, 70, 100, 16, [3, 4, 70]),                         # W = 1 rows
    (0, 1 << 20, 300, 1024, 64, [10, 100]),                  # two passes per row
])
def test_append_then_gather(builder, kind, param, n0, rb, align, steps):
    total = n0 + sum(steps)
    cap = total + 13
    X = _table(total, rb, 77 + rb + n0)
    if builder == "host":
        h = ibp.ibp_build(X[:n0], rb, kind, param, align_bytes=align, threshold=(4, 5), capacity_rows=cap, flags=SLOT).upload_metadata(0)
    else:
        h = ibp.ibp_build_device(_dev(X[:n0]).data_ptr(), n0, rb, kind, param, align_bytes=align, threshold=(4, 5), capacity_rows=cap, flags=SLOT)
    ds = oracle.DatasetT(X[:n0], kind, param, 4, 5)
    masks = [h.metadata_host(g) for g in range(ds.n_groups)]
    for g, (m, b, _) in enumerate(masks):
        assert np.array_equal(m, ds.mask(g)) and np.array_equal(b, ds.bitval(g))
    _check_rows(h, ds, X, range(0, n0, 7))
    n = n0
    rng = np.random.default_rng(n0)
    for k in steps:
        new = _dev(X[n:n + k])
        h.append_rows_device(new.data_ptr(), k, _st())
        ds.append(X[n:n + k])
        n += k
        info = h.info()
        assert info.n_rows == n and info.n_rows_raw == ds.n_raw and info.packed_bytes_bytealigned == ds.stored_bytes
        _check_rows(h, ds, X, range(n - k, n))                               # the bytes the kernel wrote into the slots
        ids = np.concatenate([np.arange(n - k, n), rng.integers(0, n, 300), np.arange(0, n, 11)]).astype(np.int64)
        got = _gather(h, ids)
        assert np.array_equal(got, oracle.gather_plain(X[:n], ids))          # (c1)
        assert np.array_equal(got[:k], ds.gather_decompress(ids[:k]))        # (c2)
    for g, (m, b, _) in enumerate(masks):                                    # the metadata never changes
        m2, b2, _ = h.metadata_host(g)
        assert np.array_equal(m, m2) and np.array_equal(b, b2)
    # every slot byte: the oracle's in-place image
    slot = h.info().slot_bytes
    img = h.packed_view(h.row_ptr(0), cap * slot).reshape(cap, slot)
    assert np.array_equal(img, ds.slot_image(cap, slot))
    # contiguous runs over slots: zero-copy range, resident decode, both dedup/order settings of the random gather
    unit = param if kind == 1 else 1
    first = (n // 3) // unit * unit
    assert np.array_equal(_range(h, first, n - first), X[first:n])
    assert np.array_equal(_resident(h, 0, n), X[:n])
    ids = rng.integers(0, n, 5000).astype(np.int64)
    for order, dd in ((0, 0), (1, 1)):
        h.set_order_mode(order).set_dedup_mode(dd)
        assert np.array_equal(_gather(h, ids), X[ids])
    # no room left for this many rows
    with pytest.raises(ibp.IbpError) as e:
        h.append_rows_device(_dev(X[:14]).data_ptr(), 14, _st())
    assert e.value.status == 5 and h.info().n_rows == n
    h.destroy()
    ds.close()


def test_append_argument_checks():
    X = _table(200, 64, 5)
    d = _dev(X)
    h = ibp.ibp_build(X[:100], 64, 0, 16, align_bytes=16, threshold=(4, 5), capacity_rows=200, flags=SLOT).upload_metadata(0)
    with pytest.raises(ibp.IbpError) as e:                                   # blocked groups of 16: row 112 would start a group without masks
        h.append_rows_device(d.data_ptr(), 20, _st())
    assert e.value.status == 5
    h.append_rows_device(d.data_ptr() + 100 * 64, 12, _st())                 # ... but the last group (rows 96..111) can be filled
    assert h.info().n_rows == 112
    assert np.array_equal(_gather(h, np.arange(112)), X[:112])
    h.destroy()
    hd = ibp.ibp_build(X[:100], 64, 0, 1 << 20, align_bytes=16, threshold=(4, 5)).upload_metadata(0)
    with pytest.raises(ibp.IbpError) as e:                                   # dense layout: immutable
        hd.append_rows_device(d.data_ptr(), 4, _st())
    assert e.value.status == 4
    hd.destroy()
    hs = ibp.ibp_build(X[:3], 64, 1, 8, align_bytes=16, threshold=(4, 5), capacity_rows=64, flags=SLOT).upload_metadata(0)
    with pytest.raises(ibp.IbpError) as e:                                   # strided: only 3 of the 8 groups have metadata
        hs.append_rows_device(d.data_ptr(), 8, _st())
    assert e.value.status == 5
    hs.destroy()


def test_online_kv_shape():
    """P:511-513 in small: K/V planes (layer, k|v, head) as strided groups, masks from the prompt tokens, decode tokens appended
    one at a time (one row per plane), then a 'page' of 16 tokens fetched as one contiguous range."""
    layers, heads, hd = 2, 4, 128
    planes = layers * 2 * heads
    prompt, decode = 48, 40
    rngX = workloads.KV(layers=1, pages=8, heads=planes // 2)                # bf16 N(0,1) / N(0,0.5) rows, any source of KV-like rows
    X = rngX.rows(0, (prompt + decode) * planes).view(np.uint8).reshape(-1, 256)
    h = ibp.ibp_build_device(_dev(X[: prompt * planes]).data_ptr(), prompt * planes, 256, 1, planes, align_bytes=16, threshold=(4, 5),
                             capacity_rows=(prompt + decode) * planes, flags=SLOT)
    ds = oracle.DatasetT(X[: prompt * planes], 1, planes, 4, 5)
    n = prompt * planes
    for t in range(decode):
        tok = _dev(X[n:n + planes])
        h.append_rows_device(tok.data_ptr(), planes, _st())
        ds.append(X[n:n + planes])
        n += planes
    _check_rows(h, ds, X, range(prompt * planes, n, 13))
    page = 16 * planes
    for first_tok in (0, 32, 64):                                            # prompt page, a page straddling prompt and decode, a decode page
        got = _range(h, first_tok * planes, page)
        assert np.array_equal(got, X[first_tok * planes: first_tok * planes + page])
    ids = np.random.default_rng(0).integers(0, n, 4000).astype(np.int64)
    assert np.array_equal(_gather(h, ids), X[ids])
    assert np.array_equal(_gather(h, ids[:512]), ds.gather_decompress(ids[:512]))
    h.destroy()
    ds.close()
