"""GPU: ibp_gather_decompress_noalloc (scratch in a file-scope device array, no cudaMalloc) against the existing path.

Collected last on purpose (the suite runs with pytest -x).  Bar: bit-exact, as in every parity test here -- the entry point
decodes the same rows with the same kernel; only the workspace of the locality-order pre-pass differs.  Two calls in a row
share the array (the second starts from the first call's leftovers), with different batch sizes and tables.
"""
import numpy as np
import pytest

import oracle
from paper_2605_30728_b200 import binding as ibp
from paper_2605_30728_b200 import workloads

pytestmark = pytest.mark.gpu
torch = pytest.importorskip("torch")


def _call(fn, ids, rb, fill):
    ids_d = torch.from_numpy(np.ascontiguousarray(ids, dtype=np.int64)).cuda()
    out = torch.full((max(1, len(ids)), rb), fill, dtype=torch.uint8, device="cuda")
    fn(ids_d.data_ptr(), len(ids), out.data_ptr(), torch.cuda.current_stream().cuda_stream)
    torch.cuda.synchronize()
    return out.cpu().numpy()[: len(ids)]


def _table(n, words, seed):
    rng = np.random.default_rng(seed)
    X = (rng.standard_normal((n, words)) * 16).round().astype(np.float32) / 256      # quantised floats: invariant bits exist
    X[rng.random(n) < 0.3] = 0.0
    return X.view(np.uint8).reshape(n, -1)


@pytest.mark.parametrize("threshold", [(1, 1), (4, 5)])
def test_noalloc_two_calls_in_a_row_match_existing_path(threshold):
    Xb = _table(60000, 64, 7)                                                     # 256-byte rows, groups of 128
    h = ibp.ibp_build(Xb, 256, 0, 128, threshold=threshold).upload_metadata(0)
    rng = np.random.default_rng(11)
    # first call: a large batch with repeats (fills the counters and the order list); second: smaller, other ids
    for k, n in enumerate([50001, 1237]):
        ids = rng.integers(0, Xb.shape[0], n)
        want = _call(h.gather_decompress, ids, 256, 0xA5)
        got = _call(h.gather_decompress_noalloc, ids, 256, 0x5A)
        assert np.array_equal(got, want), f"call {k}: no-alloc gather differs from ibp_gather_decompress"
        assert np.array_equal(got, oracle.gather_plain(Xb, ids)), f"call {k}: differs from the plain gather"
    h.destroy()


def test_noalloc_two_tables_share_the_array():
    """Two handles with different bucket shapes, back to back on one stream without a synchronisation in between."""
    w = workloads.Tiny()
    Xa = np.ascontiguousarray(w.table()).view(np.uint8).reshape(w.n_rows, -1)
    Xb = _table(200000, 32, 3)
    ha = ibp.ibp_build(Xa, w.row_bytes, w.group_kind, w.group_param).upload_metadata(0)
    hb = ibp.ibp_build(Xb, 128, 0, 64).upload_metadata(0)
    rng = np.random.default_rng(5)
    ia, ib = rng.integers(0, Xa.shape[0], 1024), rng.integers(0, Xb.shape[0], 70000)
    st = torch.cuda.current_stream().cuda_stream
    ia_d, ib_d = torch.from_numpy(ia).cuda(), torch.from_numpy(ib).cuda()
    oa = torch.zeros((len(ia), w.row_bytes), dtype=torch.uint8, device="cuda")
    ob = torch.zeros((len(ib), 128), dtype=torch.uint8, device="cuda")
    hb.gather_decompress_noalloc(ib_d.data_ptr(), len(ib), ob.data_ptr(), st)
    ha.gather_decompress_noalloc(ia_d.data_ptr(), len(ia), oa.data_ptr(), st)
    hb.gather_decompress_noalloc(ib_d.data_ptr(), len(ib), ob.data_ptr(), st)
    torch.cuda.synchronize()
    assert np.array_equal(oa.cpu().numpy(), _call(ha.gather_decompress, ia, w.row_bytes, 1))
    assert np.array_equal(ob.cpu().numpy(), _call(hb.gather_decompress, ib, 128, 1))
    assert np.array_equal(ob.cpu().numpy(), oracle.gather_plain(Xb, ib))
    ha.destroy()
    hb.destroy()


def test_noalloc_allocates_nothing_and_rejects_oversize():
    Xb = _table(4096, 32, 1)
    h = ibp.ibp_build(Xb, 128, 0, 64).upload_metadata(0)
    ids = np.arange(4096)[::-1].copy()
    _call(h.gather_decompress_noalloc, ids, 128, 0)                              # first call: symbol address looked up
    ids_d = torch.from_numpy(ids).cuda()
    out = torch.zeros((len(ids), 128), dtype=torch.uint8, device="cuda")
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    for _ in range(3):
        h.gather_decompress_noalloc(ids_d.data_ptr(), len(ids), out.data_ptr(), torch.cuda.current_stream().cuda_stream)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free0, "device memory in use changed across no-alloc calls"
    assert np.array_equal(out.cpu().numpy(), Xb[ids])
    with pytest.raises(ibp.IbpError) as e:                                       # beyond the fixed array: rejected before any launch
        h.gather_decompress_noalloc(ids_d.data_ptr(), ibp.IBP_NOALLOC_MAX_IDS + 1, out.data_ptr(), None)
    assert e.value.status == ibp.IBP_ERR_INVALID_ARG and "IBP_NOALLOC_MAX_IDS" in str(e.value)
    h.gather_decompress_noalloc(ids_d.data_ptr(), 0, out.data_ptr(), None)       # n == 0: no-op
    h.destroy()
