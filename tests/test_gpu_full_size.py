"""GPU parity at BASELINE.json's FULL sizes (configs[1..4]), in the launch configuration bench.py times (library defaults).

Every output row of a batch is compared, as raw bytes, with the plain definition out[i] = X[ids[i]] (oracle c1: a numpy
gather of the original table), and the oracle codec (c2) is run on sampled groups the batch touches: Mask, Bitval, k must
equal the library's, and the oracle's unpacker must decode the library's packed bytes of sampled rows to the original.
"""
import numpy as np
import pytest

import oracle
from paper_2605_30728_b200 import binding as ibp
from paper_2605_30728_b200 import workloads

pytestmark = pytest.mark.gpu
torch = pytest.importorskip("torch")


def _u8(X):
    return X.view(np.uint8).reshape(X.shape[0], -1)


def _check_codec_on_groups(h, X, group_ids, G, strided_S=None):
    Xb = _u8(X)
    for g in group_ids:
        rows = Xb[g::strided_S] if strided_S else Xb[g * G:(g + 1) * G]
        mask, bitval, k = oracle.group_masks(rows)
        m, b, kk = h.metadata_host(int(g))
        assert kk == k and np.array_equal(m, mask) and np.array_equal(b, bitval)
        r = int(g) if strided_S else int(g) * G + (int(g) % rows.shape[0])
        data, _ = h.packed_row(r)
        want, _ = oracle.pack_row(Xb[r], mask)
        assert np.array_equal(data[: want.size], want)
        assert np.array_equal(oracle.unpack_row(data, mask, bitval), Xb[r])


def _gather(h, ids, n_out_rows, rb):
    st = torch.cuda.current_stream().cuda_stream
    ids_d = torch.from_numpy(ids).cuda()
    out = torch.empty((n_out_rows, rb), dtype=torch.uint8, device="cuda")
    h.gather_decompress(ids_d.data_ptr(), len(ids), out.data_ptr(), st)
    torch.cuda.synchronize()
    return out.cpu().numpy()


def test_full_gnn():
    w = workloads.GNN()
    X = w.table()
    h = ibp.ibp_build(X, 512, 0, 256, align_bytes=32).upload_metadata(0)
    info = h.info()
    assert info.n_groups == 39063 and info.metadata_bytes == 39063 * 1024
    for it in (0, 1):
        ids = w.ids(it)
        assert len(ids) == 250_000 == len(np.unique(ids))
        got = _gather(h, ids, len(ids), 512)
        assert np.array_equal(got, oracle.gather_plain(X, ids))
    touched = np.unique(w.ids(0) // 256)
    _check_codec_on_groups(h, X, list(touched[:12]) + list(touched[-12:]) + [27343, 39062], 256)   # incl. the mixed and the short group
    h.destroy()


def test_full_dlrm():
    w = workloads.DLRM()
    X = w.table()
    h = ibp.ibp_build(X, 256, 0, 128, align_bytes=32).upload_metadata(0)
    assert h.info().n_groups == 406_250
    ids = w.ids(0)
    assert len(ids) == 16_384 * 26 and len(np.unique(ids)) < len(ids)
    got = _gather(h, ids, len(ids), 256)
    assert np.array_equal(got, oracle.gather_plain(X, ids))
    touched = np.unique(ids // 128)
    _check_codec_on_groups(h, X, list(touched[:10]) + list(touched[-10:]), 128)
    h.destroy()


def test_full_kv():
    w = workloads.KV()
    assert w.n_rows == 67_108_864 and w.index_span == 512 and w.batch_ids == 4096
    X = w.table()
    h = ibp.ibp_build(X, 256, 0, 16, align_bytes=16, index_span=512).upload_metadata(0)
    assert h.info().n_groups == 4_194_304
    ids = w.ids(0)
    got = _gather(h, ids, len(ids) * 512, 256)
    assert np.array_equal(got, oracle.gather_plain(X, ids, 512))
    first_rows = ids[:6] * 512
    _check_codec_on_groups(h, X, [int(r // 16) + j for r in first_rows for j in (0, 31)], 16)
    # a staged page range decoded from HBM
    st = torch.cuda.current_stream().cuda_stream
    first, n = int(ids[3]) * 512, 4 * 512
    ptr, nbytes = h.packed_range(first, n)
    packed = torch.from_numpy(h.packed_view(ptr, nbytes).copy()).cuda()
    out = torch.empty((n, 256), dtype=torch.uint8, device="cuda")
    h.decompress_resident(packed.data_ptr(), first, n, out.data_ptr(), st)
    torch.cuda.synchronize()
    assert np.array_equal(out.cpu().numpy(), _u8(X)[first:first + n])
    h.destroy()


@pytest.mark.parametrize("layer", [0, 31])
def test_full_weight_layer(layer):
    """One whole 7B-shaped decoder layer (7 matrices, 405 MB) streamed in order, zero-copy and staged+resident."""
    st = torch.cuda.current_stream().cuda_stream
    for w in workloads.weight_layer(layer):
        X = w.table()
        h = ibp.ibp_build(X, 256, 1, w.group_param, align_bytes=16).upload_metadata(0)
        out = torch.empty((w.n_rows, 256), dtype=torch.uint8, device="cuda")
        h.gather_decompress_range(0, w.n_rows, out.data_ptr(), st)
        torch.cuda.synchronize()
        assert np.array_equal(out.cpu().numpy(), _u8(X))
        ptr, nbytes = h.packed_range(0, w.n_rows)
        packed = torch.from_numpy(h.packed_view(ptr, nbytes).copy()).cuda()
        out.zero_()
        h.decompress_resident(packed.data_ptr(), 0, w.n_rows, out.data_ptr(), st)
        torch.cuda.synchronize()
        assert np.array_equal(out.cpu().numpy(), _u8(X))
        _check_codec_on_groups(h, X, [0, w.group_param - 1], None, strided_S=w.group_param)
        h.destroy()


def _check_T_codec_on_groups(h, X, group_ids, G, thr):
    """Oracle (c2, thresholded) on sampled groups: Mask/Bitval from counters with T = ceil(tau N_g), and the stored form of
    every row of the group (flag, size, canonical bytes)."""
    Xb = _u8(X)
    for g in group_ids:
        rows = Xb[g * G:(g + 1) * G]
        T = -(-rows.shape[0] * thr[0] // thr[1])
        mask, bitval, _ = oracle.group_masks(rows, T=T)
        m, b, _ = h.metadata_host(int(g))
        assert np.array_equal(m, mask) and np.array_equal(b, bitval)
        for j in range(0, rows.shape[0], 37):
            want, comp = oracle.compress_row_T(rows[j], mask, bitval, 4)
            data, _, flag = h.row_info(int(g) * G + j)
            assert flag == comp and np.array_equal(data, want)
            assert np.array_equal(oracle.decompress_row_T(data, flag, mask, bitval, 4), rows[j])


def test_full_gnn_thresholded():
    """configs[1] at full size under the paper's default codec (tau = 0.8 per group)."""
    w = workloads.GNN()
    X = w.table()
    h = ibp.ibp_build(X, 512, 0, 256, align_bytes=32, threshold=(4, 5)).upload_metadata(0)
    info = h.info()
    assert info.thresholded == 1 and info.n_groups == 39063 and info.rowflag_bytes == 4 * 312_500
    assert info.packed_bytes_bytealigned < X.nbytes
    for it in (0, 1):
        ids = w.ids(it)
        got = _gather(h, ids, len(ids), 512)
        assert np.array_equal(got, oracle.gather_plain(X, ids))
    touched = np.unique(w.ids(0) // 256)
    _check_T_codec_on_groups(h, X, list(touched[:6]) + list(touched[-6:]) + [27343, 39062], 256, (4, 5))
    h.destroy()


def test_full_dlrm_thresholded():
    w = workloads.DLRM()
    X = w.table()
    h = ibp.ibp_build(X, 256, 0, 128, align_bytes=32, threshold=(4, 5)).upload_metadata(0)
    ids = w.ids(0)
    got = _gather(h, ids, len(ids), 256)
    assert np.array_equal(got, oracle.gather_plain(X, ids))
    touched = np.unique(ids // 128)
    _check_T_codec_on_groups(h, X, list(touched[:5]) + list(touched[-5:]), 128, (4, 5))
    h.destroy()


def test_kv_thresholded_spans_and_resident():
    """configs[3]'s shape (8 of the 32 layers: 4.3 GB) under the paper's default codec: page spans through the thresholded
    stream kernel (expand form: 16-row groups of bf16 pairs have words with four runs of variant bits; four rows decoded side by
    side), a staged page range from HBM, sampled groups against the oracle codec."""
    w = workloads.KV(layers=8)
    X = w.table()
    h = ibp.ibp_build(X, 256, 0, 16, align_bytes=16, index_span=512, threshold=(4, 5)).upload_metadata(0)
    assert h.info().thresholded == 1
    ids = w.ids(0)
    got = _gather(h, ids, len(ids) * 512, 256)
    assert np.array_equal(got, oracle.gather_plain(X, ids, 512))
    first_rows = ids[:4] * 512
    _check_T_codec_on_groups(h, X, [int(r // 16) + j for r in first_rows for j in (0, 31)], 16, (4, 5))
    st = torch.cuda.current_stream().cuda_stream
    first, n = int(ids[5]) * 512, 6 * 512
    ptr, nbytes = h.packed_range(first, n)
    packed = torch.from_numpy(h.packed_view(ptr, nbytes).copy()).cuda()
    out = torch.empty((n, 256), dtype=torch.uint8, device="cuda")
    h.decompress_resident(packed.data_ptr(), first, n, out.data_ptr(), st)
    torch.cuda.synchronize()
    assert np.array_equal(out.cpu().numpy(), _u8(X)[first:first + n])
    h.destroy()


def test_weight_matrix_thresholded_stream_and_resident():
    """One 4096 x 11008 bf16 matrix of configs[4] (86 column tiles as strided groups) under tau = 0.8: whole-matrix range gather
    from the host store and resident decode, both through the thresholded stream kernel's strided branch."""
    w = workloads.WeightMatrix(rows=4096, cols=11008)
    X = w.table()
    n = w.n_rows
    h = ibp.ibp_build(X, 256, 1, w.group_param, align_bytes=16, threshold=(4, 5)).upload_metadata(0)
    st = torch.cuda.current_stream().cuda_stream
    out = torch.empty((n, 256), dtype=torch.uint8, device="cuda")
    h.gather_decompress_range(0, n, out.data_ptr(), st)
    torch.cuda.synchronize()
    assert np.array_equal(out.cpu().numpy(), _u8(X))
    ptr, nbytes = h.packed_range(0, n)
    packed = torch.from_numpy(h.packed_view(ptr, nbytes).copy()).cuda()
    out.zero_()
    h.decompress_resident(packed.data_ptr(), 0, n, out.data_ptr(), st)
    torch.cuda.synchronize()
    assert np.array_equal(out.cpu().numpy(), _u8(X))
    h.destroy()
