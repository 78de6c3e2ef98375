"""GPU parity of the mask-quality tools (csrc/ibp_analysis.cu) against oracle/mask_tools.py.

Bar: bit-exact (integer work): per-bit counters, Mask/Bitval for any tau, per-row compressed
sizes for chunk sizes 1/2/4/8 B (Fig. 3 lines 1-19), masks built from a sample and evaluated on all rows
(P:403-405), and the bit-similarity k-means (assignments, centroids and cost of every iteration).  Shapes span
several warp runs (96 rows), several 32-word passes, ragged last groups and rows whose length is not a multiple of 8 bytes.
"""
import numpy as np
import pytest

import oracle
from oracle import mask_tools as mt
from paper_2605_30728_b200 import binding as ibp
from paper_2605_30728_b200 import datagen, workloads

pytestmark = pytest.mark.gpu
torch = pytest.importorskip("torch")


def _st():
    return torch.cuda.current_stream().cuda_stream


def _rows(n, rb, seed, keep=0.6):
    """Random bytes under a random byte mask, with a few bits forced: some bits invariant, some nearly, some free."""
    rng = np.random.default_rng(seed)
    X = datagen.random_bytes(n * rb, seed).reshape(n, rb) & rng.integers(0, 256, rb, dtype=np.uint8)[None, :]
    noisy = rng.random((n, rb)) < 0.03
    X = np.where(noisy, X ^ np.uint8(0x10), X)
    X[:, : max(1, int(rb * (1 - keep)) // 4 * 4)] |= 0x81
    return np.ascontiguousarray(X.astype(np.uint8))


def _group_map(kind, param, n, n_groups, seed):
    if kind == ibp.IBP_GROUP_BLOCKED:
        return np.arange(n) // param
    if kind == ibp.IBP_GROUP_STRIDED:
        return np.arange(n) % param
    return np.random.default_rng(seed).integers(0, n_groups, n)


def _desc(kind, param, n, rb, grp):
    if kind == ibp.IBP_GROUP_MAP:
        gd = torch.from_numpy(grp.astype(np.uint32)).cuda()
        return ibp.table_desc(n, rb, kind, 0, int(grp.max()) + 1, gd.data_ptr()), gd
    return ibp.table_desc(n, rb, kind, param), None


def _gpu_counts(xd, t, ng, rb, ids=None):
    counts = torch.zeros((ng, 8 * rb), dtype=torch.int32, device="cuda")
    gn = torch.zeros(ng, dtype=torch.int32, device="cuda")
    idd = None if ids is None else torch.from_numpy(np.asarray(ids, np.int64)).cuda()
    ibp.ibp_bit_counts_device(xd.data_ptr(), t, None if idd is None else idd.data_ptr(), 0 if ids is None else len(ids),
                              counts.data_ptr(), gn.data_ptr(), _st())
    torch.cuda.synchronize()
    return counts, gn


SHAPES = [
    (0, 64, 1000, 512), (0, 256, 700, 512), (0, 7, 50, 12), (0, 1 << 30, 3000, 256), (0, 100, 1000, 20),
    (1, 5, 1003, 32), (1, 86, 2000, 256), (1, 3, 2, 4), (2, 13, 900, 64), (2, 300, 2000, 128), (0, 33, 400, 1028),
]


@pytest.mark.parametrize("kind,param,n,rb", SHAPES)
def test_counters_masks_sizes(kind, param, n, rb):
    X = _rows(n, rb, 11 + rb)
    grp = _group_map(kind, param, n, param, 3)
    t, keep = _desc(kind, param, n, rb, grp)
    ng = ibp.ibp_table_groups(t)
    assert ng == int(grp.max()) + 1
    xd = torch.from_numpy(X).cuda()
    counts, gn = _gpu_counts(xd, t, ng, rb)
    oc, on = mt.bit_counters(X, grp, ng)
    assert np.array_equal(gn.cpu().numpy().astype(np.uint64), on)
    assert np.array_equal(counts.cpu().numpy().astype(np.uint64), oc)
    for tau in [(1, 1), (4, 5), (7, 10)]:
        mask = torch.zeros((ng, rb), dtype=torch.uint8, device="cuda")
        bitval = torch.zeros((ng, rb), dtype=torch.uint8, device="cuda")
        kb = torch.zeros(ng, dtype=torch.int32, device="cuda")
        ibp.ibp_masks_from_counts_device(counts.data_ptr(), gn.data_ptr(), ng, rb, tau[0], tau[1], mask.data_ptr(), bitval.data_ptr(),
                                         kb.data_ptr(), _st())
        torch.cuda.synchronize()
        om, ob = mt.masks_from_counters(oc, on, *tau)
        assert np.array_equal(mask.cpu().numpy(), om) and np.array_equal(bitval.cpu().numpy(), ob)
        assert np.array_equal(kb.cpu().numpy(), 8 * rb - np.unpackbits(om, axis=1).sum(axis=1))
        for cs in (1, 2, 4, 8):
            if rb % cs:
                continue
            sizes = torch.zeros(n, dtype=torch.int32, device="cuda")
            totals = torch.zeros(2, dtype=torch.int64, device="cuda")
            ibp.ibp_compressed_size_device(xd.data_ptr(), t, mask.data_ptr(), bitval.data_ptr(), cs, sizes.data_ptr(), totals.data_ptr(), _st())
            torch.cuda.synchronize()
            osz, oraw = mt.compressed_sizes(X, grp, om, ob, cs)
            assert np.array_equal(sizes.cpu().numpy().astype(np.uint32), osz)
            assert totals.cpu().tolist() == [int(osz.astype(np.uint64).sum()), int(oraw.sum())]


@pytest.mark.parametrize("kind,param,n,rb", [(0, 1 << 30, 2000, 128), (0, 50, 1000, 64), (2, 9, 1500, 32)])
def test_sampled_counters(kind, param, n, rb):
    """counters over a listed sample only (sorted, unsorted, with repeats, empty groups)."""
    X = _rows(n, rb, 5)
    grp = _group_map(kind, param, n, param, 4)
    t, keep = _desc(kind, param, n, rb, grp)
    ng = ibp.ibp_table_groups(t)
    xd = torch.from_numpy(X).cuda()
    rng = np.random.default_rng(8)
    for ids in [np.sort(rng.choice(n, n // 10, replace=False)), rng.integers(0, n, 333), np.array([7, 7, 7, n - 1]), np.arange(97)]:
        counts, gn = _gpu_counts(xd, t, ng, rb, ids)
        oc, on = mt.bit_counters(X, grp, ng, ids)
        assert np.array_equal(gn.cpu().numpy().astype(np.uint64), on)
        assert np.array_equal(counts.cpu().numpy().astype(np.uint64), oc)


def test_sweep_matches_oracle_and_sampling_generalises():
    """One counting pass, every (tau, CS): totals equal the oracle's loops; masks from a 10 % sample evaluated on all rows."""
    n, rb = 3000, 128
    X = _rows(n, rb, 21)
    grp = np.zeros(n, int)
    t = ibp.table_desc(n, rb, ibp.IBP_GROUP_BLOCKED, 1 << 30)
    xd = torch.from_numpy(X).cuda()
    taus, css = [(7, 10), (4, 5), (9, 10), (1, 1)], [1, 2, 4, 8]
    sample = np.sort(np.random.default_rng(3).choice(n, n // 10, replace=False))
    sd = torch.from_numpy(sample.astype(np.int64)).cuda()
    for ids, idd in [(None, None), (sample, sd)]:
        tot, raw = ibp.ibp_mask_sweep_device(xd.data_ptr(), t, None if idd is None else idd.data_ptr(), 0 if ids is None else len(ids),
                                             taus, css, _st())
        oc, on = mt.bit_counters(X, grp, 1, ids)
        for i, tau in enumerate(taus):
            om, ob = mt.masks_from_counters(oc, on, *tau)
            for j, cs in enumerate(css):
                osz, oraw = mt.compressed_sizes(X, grp, om, ob, cs)
                assert tot[i, j] == int(osz.astype(np.uint64).sum()) and raw[i, j] == int(oraw.sum())


def test_sweep_agrees_with_the_thresholded_build():
    """At the build's own settings (per-group tau = 4/5, 4-byte chunks) the sweep's total is the byte-aligned size of the
    store ibp_build packs (itself equal to the oracle codec's): 200k rows of the GNN table around the dense/sparse edge."""
    w = workloads.GNN()
    first, n = 6_899_968, 200_000                               # a group boundary (multiple of 256) before the 7M edge
    X = w.rows(first, n)
    Xb = np.ascontiguousarray(X).view(np.uint8).reshape(n, -1)
    h = ibp.ibp_build(Xb, 512, 0, 256, align_bytes=16, threshold=(4, 5), flags=ibp.IBP_FLAG_PAGEABLE_STORE)
    info = h.info()
    t = ibp.table_desc(n, 512, ibp.IBP_GROUP_BLOCKED, 256)
    xd = torch.from_numpy(Xb).cuda()
    tot, raw = ibp.ibp_mask_sweep_device(xd.data_ptr(), t, None, 0, [(4, 5)], [4], _st())
    assert int(tot[0, 0]) == info.packed_bytes_bytealigned and int(raw[0, 0]) == info.n_rows_raw
    h.destroy()


@pytest.mark.parametrize("n,rb,k,iters", [(300, 64, 7, 3), (1000, 32, 5, 4), (257, 516, 3, 2), (500, 128, 33, 2)])
def test_kmeans_matches_oracle(n, rb, k, iters):
    X = _rows(n, rb, 31 + k)
    X[5] = X[0]
    init = np.random.default_rng(k).choice(n, k, replace=False)
    init[:2] = [0, 5]                                          # two identical centroids: exact distance ties
    xd = torch.from_numpy(X).cuda()
    idd = torch.from_numpy(init.astype(np.int64)).cuda()
    oa, ocent, ocost = mt.kmeans_bits(X, init, iters)
    for it in range(1, iters + 1):                             # every iteration count: assignment of iteration it-1
        assign = torch.zeros(n, dtype=torch.int32, device="cuda")
        cent = torch.zeros((k, rb), dtype=torch.uint8, device="cuda")
        cost = torch.zeros(it, dtype=torch.int64, device="cuda")
        ibp.ibp_kmeans_bits_device(xd.data_ptr(), n, rb, k, idd.data_ptr(), it, assign.data_ptr(), cent.data_ptr(), cost.data_ptr(), _st())
        torch.cuda.synchronize()
        assert np.array_equal(assign.cpu().numpy().astype(np.uint32), oa[it - 1])
        assert cost.cpu().tolist() == ocost[:it]
    assert np.array_equal(cent.cpu().numpy(), ocent)


def test_kmeans_planted_clusters_and_net_savings():
    """Planted prototypes with 2 % flips: the partition is recovered (unique answer), and clustering raises the net space
    saved over one global mask once metadata is charged."""
    rng = np.random.default_rng(7)
    rb, per, k = 256, 500, 8
    protos = rng.integers(0, 256, (k, rb), dtype=np.uint8)
    truth = np.repeat(np.arange(k), per)
    flips = np.packbits(rng.random((k * per, 8 * rb)) < 0.02, axis=1, bitorder="little")
    X = protos[truth] ^ flips
    perm = rng.permutation(k * per)
    X, truth = np.ascontiguousarray(X[perm]), truth[perm]
    n = len(X)
    init = np.array([int(np.flatnonzero(truth == c)[0]) for c in range(k)])
    xd = torch.from_numpy(X).cuda()
    idd = torch.from_numpy(init.astype(np.int64)).cuda()
    assign = torch.zeros(n, dtype=torch.int32, device="cuda")
    cent = torch.zeros((k, rb), dtype=torch.uint8, device="cuda")
    ibp.ibp_kmeans_bits_device(xd.data_ptr(), n, rb, k, idd.data_ptr(), 3, assign.data_ptr(), cent.data_ptr(), None, _st())
    torch.cuda.synchronize()
    assert np.array_equal(assign.cpu().numpy(), truth)
    assert np.array_equal(cent.cpu().numpy(), protos)
    one = ibp.table_desc(n, rb, ibp.IBP_GROUP_BLOCKED, 1 << 30)
    clus = ibp.table_desc(n, rb, ibp.IBP_GROUP_MAP, 0, k, assign.data_ptr())
    t1, _ = ibp.ibp_mask_sweep_device(xd.data_ptr(), one, None, 0, [(4, 5)], [4], _st())
    tk, _ = ibp.ibp_mask_sweep_device(xd.data_ptr(), clus, None, 0, [(4, 5)], [4], _st())
    net1 = 1 - (int(t1[0, 0]) + 2 * rb) / (n * rb)
    netk = 1 - (int(tk[0, 0]) + 2 * rb * k) / (n * rb)
    assert abs(netk - mt.net_space_saved(X[:400], truth[:400], k, 4, 5, 4)) < 0.05   # same regime as the oracle on a slice
    assert netk > net1 + 0.3


def test_bad_arguments():
    X = torch.zeros((8, 16), dtype=torch.uint8, device="cuda")
    t = ibp.table_desc(8, 16, ibp.IBP_GROUP_BLOCKED, 4)
    with pytest.raises(ibp.IbpError) as e:
        ibp.ibp_mask_sweep_device(X.data_ptr(), t, None, 0, [(1, 2)], [4], _st())          # tau <= 1/2 (R3)
    assert e.value.status == 1
    with pytest.raises(ibp.IbpError):
        ibp.ibp_mask_sweep_device(X.data_ptr(), t, None, 0, [(4, 5)], [3], _st())          # chunk size
    with pytest.raises(ibp.IbpError):
        ibp.ibp_mask_sweep_device(X.data_ptr(), ibp.table_desc(8, 18, 0, 4), None, 0, [(4, 5)], [4], _st())
    with pytest.raises(ibp.IbpError):
        ibp.ibp_table_groups(ibp.table_desc(8, 16, ibp.IBP_GROUP_MAP, 0, 0, None))


def test_order_by_group_is_a_grouped_permutation():
    """Several correct answers exist (the order inside a group is unspecified): check what is unique -- a permutation, groups in
    ascending order, the group offsets -- incl. empty groups."""
    n, k = 50_000, 37
    grp = np.random.default_rng(2).integers(0, k, n).astype(np.uint32)
    grp[grp == 5] = 6                                          # an empty group
    gd = torch.from_numpy(grp).cuda()
    order = torch.zeros(n, dtype=torch.int64, device="cuda")
    start = torch.zeros(k + 1, dtype=torch.int32, device="cuda")
    ibp.ibp_order_by_group_device(gd.data_ptr(), n, k, order.data_ptr(), start.data_ptr(), _st())
    torch.cuda.synchronize()
    o = order.cpu().numpy()
    assert np.array_equal(np.sort(o), np.arange(n))
    assert np.all(np.diff(grp[o].astype(np.int64)) >= 0)
    assert np.array_equal(start.cpu().numpy().astype(np.int64), np.concatenate([[0], np.cumsum(np.bincount(grp, minlength=k))]))


def test_clustered_store_through_reordering():
    """Clustered compression end to end with positional groups: k-means on the interleaved GNN variant (reading R15),
    rows reordered so that clusters are runs of consecutive rows, blocked groups of 256 over the reordered table, ids mapped
    through the inverse permutation.  The gather returns the original rows (plain definition), and the reordered table
    compresses better than the table in its original order."""
    w = workloads.GNN(n_rows=32_768, batch=4096, interleaved=True)
    X = w.table()
    Xb = np.ascontiguousarray(X).view(np.uint8).reshape(w.n_rows, -1)
    n, rb = Xb.shape
    sparse = ((X == 0) | (X == 1)).all(axis=1)
    init = np.array([int(np.flatnonzero(~sparse)[0]), int(np.flatnonzero(sparse)[0])], np.int64)
    xd = torch.from_numpy(Xb).cuda()
    idd = torch.from_numpy(init).cuda()
    assign = torch.zeros(n, dtype=torch.int32, device="cuda")
    cent = torch.zeros((2, rb), dtype=torch.uint8, device="cuda")
    ibp.ibp_kmeans_bits_device(xd.data_ptr(), n, rb, 2, idd.data_ptr(), 3, assign.data_ptr(), cent.data_ptr(), None, _st())
    order = torch.zeros(n, dtype=torch.int64, device="cuda")
    ibp.ibp_order_by_group_device(assign.data_ptr(), n, 2, order.data_ptr(), None, _st())
    torch.cuda.synchronize()
    assert np.array_equal(assign.cpu().numpy().astype(bool), sparse)             # the two row types are the two clusters
    o = order.cpu().numpy()
    inv = np.empty(n, np.int64)
    inv[o] = np.arange(n)
    h0 = ibp.ibp_build(Xb, rb, 0, 256, align_bytes=32, flags=ibp.IBP_FLAG_PAGEABLE_STORE)
    h1 = ibp.ibp_build(np.ascontiguousarray(Xb[o]), rb, 0, 256, align_bytes=32).upload_metadata(0)
    r0 = Xb.nbytes / h0.info().packed_bytes_rows
    r1 = Xb.nbytes / h1.info().packed_bytes_rows
    assert r1 > 1.1 * r0, (r0, r1)
    ids = w.ids(0)
    ids_d = torch.from_numpy(inv[ids]).cuda()
    out = torch.zeros((len(ids), rb), dtype=torch.uint8, device="cuda")
    h1.gather_decompress(ids_d.data_ptr(), len(ids), out.data_ptr(), _st())
    torch.cuda.synchronize()
    assert np.array_equal(out.cpu().numpy(), oracle.gather_plain(Xb, ids))
    h0.destroy()
    h1.destroy()
