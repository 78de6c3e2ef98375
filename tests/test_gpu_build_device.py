"""GPU parity of the GPU-side compressor (ibp_build_device) against the CPU oracle.

Bar: bit-exact.  The kernels keep the oracle's canonical bit order, so Mask, Bitval, k_g, the per-row sizes / raw flags and
the packed bytes of every row must equal the oracle's (oracle.Dataset / oracle.DatasetT, written from PAPER.md:229-241 and
Fig. 3), and a gather through the handle must return the original rows.  Shapes cover both group kinds, every alignment
unit, multi-pass rows, ragged last groups, groups cut into slices (few groups of many rows: the merge kernel), one global
Mask/Bitval, source rows in HBM and in mapped host memory (the paper's zero-copy compressor).
"""
import os
import sys

import numpy as np
import pytest

sys.path.insert(0, os.path.dirname(os.path.abspath(__file__)))

import oracle
from paper_2605_30728_b200 import binding as ibp
from paper_2605_30728_b200 import datagen, workloads
from test_host_build import _check_against_oracle, _check_T_against_oracle

pytestmark = pytest.mark.gpu
torch = pytest.importorskip("torch")


def _stream():
    return torch.cuda.current_stream().cuda_stream


def _build_strict(Xb, rb, kind, param, align, span):
    xd = torch.from_numpy(np.ascontiguousarray(Xb)).cuda()
    h = ibp.ibp_build_device(xd.data_ptr(), Xb.shape[0], rb, kind, param, align_bytes=align, index_span=span, stream=_stream())
    torch.cuda.synchronize()
    return h


def _build_T(Xb, rb, kind, param, align, thr):
    xd = torch.from_numpy(np.ascontiguousarray(Xb)).cuda()
    h = ibp.ibp_build_device(xd.data_ptr(), Xb.shape[0], rb, kind, param, align_bytes=align, threshold=thr, stream=_stream())
    torch.cuda.synchronize()
    return h


def _masked_rows(n, rb, seed=5):
    return (datagen.random_bytes(n * rb, seed + rb).reshape(n, rb) & datagen.random_bytes(rb, 9)[None, :]) | 0x01


@pytest.mark.parametrize("align", [1, 4, 16, 32, 128])
def test_tiny_blocked(align):
    _check_against_oracle(workloads.Tiny(n_rows=512).table(), 0, 64, align, build=_build_strict)


@pytest.mark.parametrize("kind,param,n,rb,align", [
    (0, 7, 50, 12, 1), (0, 7, 50, 12, 16), (0, 64, 3000, 64, 32), (0, 1000, 10, 8, 4), (0, 16, 40, 4, 16),
    (1, 5, 203, 32, 16), (1, 8, 64, 16, 1), (1, 3, 2, 4, 16), (0, 1, 9, 20, 8), (0, 33, 1000, 100, 32),
    (0, 128, 700, 256, 32), (0, 256, 1500, 512, 32), (0, 50, 333, 1024, 32), (0, 20, 77, 4096, 64), (1, 6, 600, 2048, 16),
    (0, 9, 100, 516, 4), (0, 9, 100, 264, 1), (0, 4, 30, 8192, 128), (0, 5000, 20000, 64, 32), (1, 3, 30000, 128, 16),
    (0, 1 << 30, 70000, 32, 32), (0, 4, 12, 65536, 32),
])
def test_strict_shapes(kind, param, n, rb, align):
    """Odd row sizes (W = 1, 2, 4; 1..16 passes), ragged last groups, strided groups with a partial last matrix row, groups
    large enough to be cut into slices (5000 and 10000 rows per group, and one group of all 70000 rows)."""
    _check_against_oracle(_masked_rows(n, rb), kind, min(param, n) if kind == 0 else param, align, build=_build_strict,
                          rows_to_check=None if n <= 3000 else range(0, n, 97))


def test_strict_workload_shapes_and_host_build_bytes():
    """The configs' shapes; the whole store equals the host compressor's byte for byte (padding and gaps included)."""
    cases = [(workloads.GNN(n_rows=4096), 32, 1), (workloads.DLRM(rows_per_table=1024, n_tables=2), 32, 1),
             (workloads.KV(layers=1, pages=4, heads=4), 16, 64), (workloads.WeightMatrix(128, 512), 16, 1)]
    for w, align, span in cases:
        X = w.table()
        _check_against_oracle(X, w.group_kind, w.group_param, align, span=span, build=_build_strict,
                              rows_to_check=range(0, w.n_rows, 13))
        Xb = np.ascontiguousarray(X).view(np.uint8).reshape(w.n_rows, -1)
        hd = _build_strict(Xb, w.row_bytes, w.group_kind, w.group_param, align, span)
        hh = ibp.ibp_build(Xb, w.row_bytes, w.group_kind, w.group_param, align_bytes=align, index_span=span,
                           flags=ibp.IBP_FLAG_PAGEABLE_STORE)
        (pd, nd), (ph, nh) = hd.packed_range(0, w.n_rows), hh.packed_range(0, w.n_rows)
        assert nd == nh and np.array_equal(hd.packed_view(pd, nd), hh.packed_view(ph, nh))
        assert hd.info().packed_bytes_stored == hh.info().packed_bytes_stored
        # the handle is ready to use: gather through it
        ids = np.random.default_rng(1).integers(0, w.n_rows // span, 500).astype(np.int64)
        ids_d = torch.from_numpy(ids).cuda()
        out = torch.zeros((len(ids) * span, w.row_bytes), dtype=torch.uint8, device="cuda")
        hd.gather_decompress(ids_d.data_ptr(), len(ids), out.data_ptr(), _stream())
        torch.cuda.synchronize()
        assert np.array_equal(out.cpu().numpy(), oracle.gather_plain(X, ids, span))
        hd.destroy(); hh.destroy()


def test_degenerate_groups():
    rb = 64
    r = datagen.random_bytes(rb, 3)
    same = np.repeat(r[None, :], 10, axis=0)                      # k = 0: nothing stored (reading R12)
    h = _build_strict(same, rb, 0, 10, 32, 1)
    m, b, k = h.metadata_host(0)
    assert k == 0 and np.all(m == 0xFF) and np.array_equal(b, r)
    assert h.info().packed_bytes_rows == 0
    h.destroy()
    both = np.stack([r, ~r])                                      # no invariant bit: packed == raw (reading R13)
    h = _build_strict(both, rb, 0, 2, 1, 1)
    m, b, k = h.metadata_host(0)
    assert k == 8 * rb and not m.any() and not b.any()
    for i in range(2):
        data, _ = h.packed_row(i)
        assert np.array_equal(data, both[i])
    h.destroy()


def test_source_rows_in_mapped_host_memory():
    """the compressor reads the tensors zero-copy from CPU memory."""
    w = workloads.Tiny(n_rows=1024)
    X = w.table()
    buf = ibp.PinnedBuffer(X.nbytes)
    buf.view(X.dtype, X.shape)[:] = X
    h = ibp.ibp_build_device(buf.dev_ptr, w.n_rows, 512, 0, 64, align_bytes=32, stream=_stream())
    ds = oracle.Dataset(X, 0, 64)
    for r in range(0, 1024, 11):
        data, k = h.packed_row(r)
        want = ds.packed_row(r)
        assert np.array_equal(data[: want.size], want)
    h.destroy(); ds.close(); buf.free()


# --------------------------------------------------------------------------------------------------------- thresholded
@pytest.mark.parametrize("kind,param,n,rb,thr", [(0, 64, 1000, 64, (4, 5)), (0, 7, 50, 12, (4, 5)), (0, 256, 700, 512, (7, 10)),
                                                 (1, 5, 203, 32, (4, 5)), (1, 6, 600, 256, (9, 10)), (0, 1 << 30, 900, 128, (4, 5)),
                                                 (0, 300, 1000, 8, (4, 5)), (0, 16, 100, 2048, (3, 4)), (0, 600, 3000, 64, (4, 5)),
                                                 (0, 1 << 30, 70000, 32, (4, 5)), (1, 3, 30000, 128, (3, 4)),
                                                 (0, 4, 12, 65536, (3, 4))])
def test_T_shapes(kind, param, n, rb, thr):
    rng = np.random.default_rng(rb + n)
    X = _masked_rows(n, rb)
    for r in rng.choice(n, n // 5, replace=False):                # non-participating chunks
        X[r, rng.integers(0, rb)] ^= 0xFF
    for r in rng.choice(n, n // 20 + 1, replace=False):           # raw rows
        X[r] = datagen.random_bytes(rb, 1000 + int(r))
    _check_T_against_oracle(X, kind, min(param, n) if kind == 0 else param, thr, build=_build_T,
                            rows_to_check=None if n <= 3000 else range(0, n, 97))


def test_T_golden_worked_example():
    rows = np.array([[0xB4, 0x0F, 0xB4, 0x0F], [0xA6, 0x0F, 0xA6, 0x0F], [0xB5, 0x0F, 0xB5, 0x0F], [0xA4, 0x1F, 0xA4, 0x1F],
                     [0x36, 0x0E, 0x36, 0x0E]] * 3, np.uint8)
    _check_T_against_oracle(rows, 0, 5, (4, 5), align=16, build=_build_T)


def test_T_workload_shapes_and_gather():
    w = workloads.GNN(n_rows=4096)
    X = np.concatenate([w.rows(0, 1024), w.rows(3000, 1024)])
    _check_T_against_oracle(X, 0, 256, (4, 5), build=_build_T)
    _check_T_against_oracle(X, 0, 1 << 20, (4, 5), rows_to_check=range(0, 2048, 7), build=_build_T)   # one global Mask/Bitval
    Xb = np.ascontiguousarray(X).view(np.uint8).reshape(X.shape[0], -1)
    h = _build_T(Xb, 512, 0, 256, 32, (4, 5))
    ids = np.random.default_rng(2).integers(0, X.shape[0], 3000).astype(np.int64)
    ids_d = torch.from_numpy(ids).cuda()
    out = torch.zeros((len(ids), 512), dtype=torch.uint8, device="cuda")
    h.gather_decompress(ids_d.data_ptr(), len(ids), out.data_ptr(), _stream())
    torch.cuda.synchronize()
    assert np.array_equal(out.cpu().numpy(), oracle.gather_plain(X, ids))
    h.destroy()


def test_argument_errors():
    x = torch.zeros((8, 16), dtype=torch.uint8, device="cuda")
    with pytest.raises(ibp.IbpError) as e:
        ibp.ibp_build_device(x.data_ptr(), 8, 16, 0, 4, flags=ibp.IBP_FLAG_PAGEABLE_STORE)
    assert e.value.status == 1
    with pytest.raises(ibp.IbpError) as e:
        ibp.ibp_build_device(x.data_ptr(), 8, 14, 0, 4)
    assert e.value.status == 1
    with pytest.raises(ibp.IbpError) as e:
        ibp.ibp_build_device(x.data_ptr() + 4, 7, 16, 0, 4)
    assert e.value.status == 1
