"""Pins for oracle/mask_tools.py: checked against brute force with Python integers, closed forms and
the values the paper prints, never against itself.  Each test names the mistake it would catch.  CPU only."""
import numpy as np
import pytest

import oracle
from oracle import mask_tools as mt


def _rows_as_ints(Xb):
    return [int.from_bytes(bytes(r), "little") for r in Xb]


def _rand_rows(rng, n, rb, p_one=0.5):
    bits = (rng.random((n, 8 * rb)) < p_one).astype(np.uint8)
    return np.packbits(bits, axis=1, bitorder="little")


def test_counters_brute_force_python_ints():
    """P:229.  A wrong bit order, a wrong group index or a dropped row fails: counters re-derived with int bit tests."""
    rng = np.random.default_rng(1)
    X = _rand_rows(rng, 37, 12, 0.3)
    grp = rng.integers(0, 5, 37)
    counts, n = mt.bit_counters(X, grp, 5)
    ints = _rows_as_ints(X)
    for g in range(5):
        members = [ints[r] for r in range(37) if grp[r] == g]
        assert n[g] == len(members)
        for p in range(96):
            assert counts[g, p] == sum((v >> p) & 1 for v in members)
    assert int(counts.sum()) == sum(v.bit_count() for v in ints)


def test_counters_full_enumeration_closed_form():
    """All 2^k values on k chosen bit positions, constant elsewhere: every chosen counter is 2^(k-1), the others 0 or N."""
    k, rb = 6, 8
    pos = [3, 9, 17, 30, 41, 63]
    const = 0x00F0_0000_0F00_0000 & ~sum(1 << p for p in pos)
    rows = []
    for j in range(1 << k):
        v = const
        for b, p in enumerate(pos):
            v |= ((j >> b) & 1) << p
        rows.append(np.frombuffer(v.to_bytes(rb, "little"), np.uint8))
    X = np.stack(rows)
    counts, n = mt.bit_counters(X, np.zeros(len(X), int), 1)
    assert n[0] == 64
    for p in range(64):
        want = 32 if p in pos else (64 if (const >> p) & 1 else 0)
        assert counts[0, p] == want


def test_counters_on_a_sample_counts_only_the_sample():
    """P:403-405.  Counting rows outside the sample, or counting a repeated id once, fails."""
    rng = np.random.default_rng(2)
    X = _rand_rows(rng, 50, 4)
    ids = np.array([3, 3, 10, 49])
    counts, n = mt.bit_counters(X, np.zeros(50, int), 1, sample_ids=ids)
    ints = _rows_as_ints(X)
    assert n[0] == 4
    for p in range(32):
        assert counts[0, p] == sum((ints[r] >> p) & 1 for r in ids)


def test_masks_tau_1_is_and_or_form():
    """T = N: Mask = ~(AND xor OR), Bitval = AND (SURVEY 8(c) independent closed form).  > instead of >= fails."""
    rng = np.random.default_rng(3)
    X = _rand_rows(rng, 20, 16, 0.5)
    X[:, :6] = X[0, :6]                              # six invariant bytes
    counts, n = mt.bit_counters(X, np.zeros(20, int), 1)
    mask, bitval = mt.masks_from_counters(counts, n, 1, 1)
    a = np.bitwise_and.reduce(X, axis=0)
    o = np.bitwise_or.reduce(X, axis=0)
    assert np.array_equal(mask[0], np.bitwise_not(a ^ o))
    assert np.array_equal(bitval[0], a)


def test_masks_threshold_boundaries():
    """P:231 with R2: N = 5, tau = 4/5 -> T = 4: counts 4 and 5 -> invariant 1, counts 0 and 1 -> invariant 0, 2 and 3 variant
    (the paper's Fig. 2 caption has T = 4, N = 5).  An off-by-one in either comparison, or floor instead of ceil
    for T, fails (tau = 7/10 of N = 5 -> T = 4, not 3)."""
    counts = np.array([[0, 1, 2, 3, 4, 5, 0, 0]], np.uint64)
    n = np.array([5], np.uint64)
    for tau in [(4, 5), (7, 10)]:
        mask, bitval = mt.masks_from_counters(counts, n, *tau)
        assert mask[0, 0] == 0b11110011
        assert bitval[0, 0] == 0b00110000
    assert mt.threshold_of(10, 7, 10) == 7 and mt.threshold_of(3, 4, 5) == 3 and mt.threshold_of(2400000, 4, 5) == 1920000
    mask, _ = mt.masks_from_counters(counts, np.array([0], np.uint64), 4, 5)
    assert mask[0, 0] == 0                           # nothing counted -> nothing invariant


@pytest.mark.parametrize("cs,overhead", [(1, 0.125), (2, 0.0625), (4, 0.03125), (8, 0.015625)])
def test_participation_overhead_matches_the_paper(cs, overhead):
    """P:527 prints 12.5 % for 1-byte chunks and 1.6 % for 8-byte chunks: with every bit invariant and every chunk
    matching, a row shrinks to exactly its participation bits = row_bytes/CS bits.  Chunk count in bytes instead of
    bits, or a missing participation term, fails."""
    rb = 512
    X = np.tile(np.arange(rb, dtype=np.uint8)[None, :], (9, 1))
    counts, n = mt.bit_counters(X, np.zeros(9, int), 1)
    mask, bitval = mt.masks_from_counters(counts, n, 4, 5)
    sizes, raw = mt.compressed_sizes(X, np.zeros(9, int), mask, bitval, cs)
    assert not raw.any()
    assert np.all(sizes == int(rb * overhead))
    assert round(100 * overhead, 1) in (12.5, 6.2, 3.1, 1.6)


def test_sizes_brute_force_python_ints():
    """Fig. 3 lines 1-19 re-derived with integer arithmetic on Python ints for every chunk size."""
    rng = np.random.default_rng(4)
    rb = 16
    X = _rand_rows(rng, 40, rb, 0.5)
    X[:, 4:12] = X[0, 4:12]
    X[7, 5] ^= 0x10                                  # one row breaks one chunk
    grp = np.arange(40) % 2
    counts, n = mt.bit_counters(X, grp, 2)
    mask, bitval = mt.masks_from_counters(counts, n, 4, 5)
    ints = _rows_as_ints(X)
    for cs in (1, 2, 4, 8):
        sizes, raw = mt.compressed_sizes(X, grp, mask, bitval, cs)
        for r in range(40):
            M = int.from_bytes(bytes(mask[grp[r]]), "little")
            B = int.from_bytes(bytes(bitval[grp[r]]), "little")
            saved = 0
            for c in range(rb // cs):
                cm = ((1 << (8 * cs)) - 1) << (8 * cs * c)
                if (ints[r] & M & cm) == (B & cm):
                    saved += (M & cm).bit_count()
            diff = saved - rb // cs
            bs = diff // 8 if diff > 0 else 0
            assert sizes[r] == (rb - bs if bs > 0 else rb)
            assert raw[r] == (bs <= 0)


def test_sizes_agree_with_the_dataset_oracle():
    """The per-row sizes must be the sizes the thresholded dataset codec (pinned by the hand-worked fixtures) stores."""
    rng = np.random.default_rng(5)
    X = _rand_rows(rng, 96, 32, 0.5)
    X[:, 8:24] = X[0, 8:24]
    ds = oracle.DatasetT(X, oracle.BLOCKED, 32, 4, 5, 4)
    grp = np.arange(96) // 32
    counts, n = mt.bit_counters(X, grp, 3)
    mask, bitval = mt.masks_from_counters(counts, n, 4, 5)
    sizes, raw = mt.compressed_sizes(X, grp, mask, bitval, 4)
    for g in range(3):
        assert np.array_equal(mask[g], ds.mask(g)) and np.array_equal(bitval[g], ds.bitval(g))
    for r in range(96):
        data, comp = ds.row(r)
        assert len(data) == sizes[r] and comp == (not raw[r])
    ds.close()


def test_kmeans_assignment_brute_force_and_monotone_cost():
    """P:542 / R25.  Assignment = argmin Hamming distance (int xor + bit_count), lowest index on ties; the Lloyd cost never
    increases.  A distance on values instead of bits, a minority centroid or a last-index tie-break fails."""
    rng = np.random.default_rng(6)
    X = _rand_rows(rng, 60, 8, 0.5)
    X[10] = X[0]                                     # exact tie between centroids 0 and 1 below
    init = np.array([0, 10, 20, 30])
    assign, cent, costs = mt.kmeans_bits(X, init, 4)
    ints = _rows_as_ints(X)
    c0 = [ints[i] for i in init]
    for r in range(60):
        d = [(ints[r] ^ c).bit_count() for c in c0]
        assert assign[0][r] == d.index(min(d))
    assert assign[0][0] == 0 and assign[0][10] == 0
    assert all(costs[i + 1] <= costs[i] for i in range(len(costs) - 1))
    # centroid = strict majority, tie -> 0
    members = [ints[r] for r in range(60) if assign[-1][r] == 2]
    if members:
        want = 0
        for p in range(64):
            if 2 * sum((v >> p) & 1 for v in members) > len(members):
                want |= 1 << p
        assert int.from_bytes(bytes(cent[2]), "little") == want


def test_kmeans_recovers_planted_clusters():
    """Four far-apart prototypes with 2 % bit flips: one Lloyd step from one member of each recovers the partition and the
    centroids equal the prototypes' majority; clustered net savings beat the single-cluster savings."""
    rng = np.random.default_rng(7)
    rb, per = 32, 64
    protos = _rand_rows(rng, 4, rb, 0.5)
    truth = np.repeat(np.arange(4), per)
    flips = _rand_rows(rng, 4 * per, rb, 0.02)
    X = protos[truth] ^ flips
    perm = rng.permutation(4 * per)
    X, truth = X[perm], truth[perm]
    init = np.array([int(np.flatnonzero(truth == c)[0]) for c in range(4)])
    assign, cent, costs = mt.kmeans_bits(X, init, 3)
    assert np.array_equal(assign[-1], truth)
    assert np.array_equal(cent, protos)
    one = mt.net_space_saved(X, np.zeros(len(X), int), 1, 4, 5, 4)
    four = mt.net_space_saved(X, assign[-1], 4, 4, 5, 4)
    assert four > one and four > 0.3


def test_net_space_saved_counts_metadata():
    """identical rows, one cluster: saved = 1 - (n * rb/32 + 2 rb) / (n rb) at CS = 4."""
    rb, n = 64, 100
    X = np.tile(np.arange(rb, dtype=np.uint8)[None, :], (n, 1))
    got = mt.net_space_saved(X, np.zeros(n, int), 1, 4, 5, 4)
    assert abs(got - (1 - (n * rb // 32 + 2 * rb) / (n * rb))) < 1e-12
    # an empty second cluster costs no metadata
    assert mt.net_space_saved(X, np.zeros(n, int), 2, 4, 5, 4) == got
