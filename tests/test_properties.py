"""CPU-only property tests (hypothesis): random shapes and bit patterns against what the mathematics fixes.

The oracle is pinned here by Python-integer brute force written independently of it (bits as Python ints, no numpy bit tricks shared
with oracle/), and the library's host compressor by the oracle.  Sizes are tiny so every case runs in milliseconds; the value is in
the shapes nobody thought of: odd row widths, one-row groups, strided tables shorter than their stride, thresholds at the edge of
the allowed range, rows that are all zero or all one, chunks that stop participating because of one flipped bit.
"""
import numpy as np
import pytest

hypothesis = pytest.importorskip("hypothesis")
from hypothesis import HealthCheck, given, settings, strategies as st

import oracle
from paper_2605_30728_b200 import binding as ibp

SET = dict(max_examples=60, deadline=None, suppress_health_check=[HealthCheck.too_slow, HealthCheck.data_too_large])


def _as_int(row):
    """row bytes -> Python int with bit p of the row at bit p (bit p = bit p mod 8 of byte p div 8: little endian)"""
    return int.from_bytes(bytes(row), "little")


def _table(draw, n, rb):
    """rows with structure: a random invariant pattern under a random mask, random elsewhere, plus a few disturbed rows"""
    rng = np.random.default_rng(draw(st.integers(0, 2**32 - 1)))
    density = draw(st.sampled_from([0.0, 0.2, 0.5, 0.9, 1.0]))
    keep = (rng.random((1, rb * 8)) < density)
    base = rng.integers(0, 2, (1, rb * 8), dtype=np.uint8)
    bits = np.where(keep, base, rng.integers(0, 2, (n, rb * 8), dtype=np.uint8))
    for _ in range(draw(st.integers(0, 3))):                                  # rows that break the pattern
        r = int(rng.integers(0, n))
        kind = draw(st.sampled_from(["flip", "zero", "one", "random"]))
        if kind == "flip":
            bits[r, int(rng.integers(0, rb * 8))] ^= 1
        elif kind == "zero":
            bits[r] = 0
        elif kind == "one":
            bits[r] = 1
        else:
            bits[r] = rng.integers(0, 2, rb * 8, dtype=np.uint8)
    return np.packbits(bits.astype(np.uint8), axis=1, bitorder="little")


def _groups(kind, param, n):
    if kind == 0:
        return [list(range(g * param, min(n, (g + 1) * param))) for g in range(-(-n // param))]
    return [list(range(g, n, param)) for g in range(min(param, n))]


@st.composite
def _case(draw, thresholded):
    rb = 4 * draw(st.integers(1, 6))
    n = draw(st.integers(1, 40))
    kind = draw(st.sampled_from([0, 1]))
    param = draw(st.integers(1, 12))
    X = _table(draw, n, rb)
    thr = draw(st.sampled_from([(4, 5), (3, 4), (2, 3), (9, 10), (51, 100)])) if thresholded else (1, 1)
    return X, kind, param, thr


@settings(**SET)
@given(_case(False))
def test_strict_masks_sizes_and_round_trip(case):
    """P:229-231 with T = N; Mask = bits on which ALL rows of the group agree, Bitval = their values, packed row j =
    the other bits in ascending position, LSB first, ceil(k/8) bytes; decoding gives the row back."""
    X, kind, param, _ = case
    n, rb = X.shape
    ds = oracle.Dataset(X, kind, param)
    groups = _groups(kind, param, n)
    assert ds.n_groups == len(groups)
    for g, members in enumerate(groups):
        ints = [_as_int(X[r]) for r in members]
        a = o = ints[0]
        for v in ints[1:]:
            a &= v
            o |= v
        full = (1 << (8 * rb)) - 1
        mask = ~(a ^ o) & full                                               # agree everywhere: AND == OR
        assert _as_int(ds.mask(g)) == mask and _as_int(ds.bitval(g)) == (a & mask)
        k = 8 * rb - bin(mask).count("1")
        assert ds.k_bits(g) == k
        positions = [p for p in range(8 * rb) if not (mask >> p) & 1]
        for r, v in zip(members, ints):
            want = sum(((v >> p) & 1) << i for i, p in enumerate(positions))
            got = ds.packed_row(r)
            assert got.size == (k + 7) // 8 and _as_int(got) == want
    ids = np.arange(n)[::-1].copy()
    assert np.array_equal(ds.gather_decompress(ids), X[ids])
    ds.close()


@settings(**SET)
@given(_case(True))
def test_thresholded_masks_sizes_and_round_trip(case):
    """P:231 (reading R2: count >= T / count <= N - T, T = ceil(tau N)); Fig. 3: participation, bitsSaved, size; P:303 raw rows."""
    X, kind, param, (tn, td) = case
    n, rb = X.shape
    ds = oracle.DatasetT(X, kind, param, tn, td)
    for g, members in enumerate(_groups(kind, param, n)):
        N = len(members)
        T = -(-tn * N // td)
        ints = [_as_int(X[r]) for r in members]
        mask = bit = 0
        for p in range(8 * rb):
            c1 = sum((v >> p) & 1 for v in ints)
            if c1 >= T:
                mask |= 1 << p
                bit |= 1 << p
            elif c1 <= N - T:
                mask |= 1 << p
        assert ds.threshold(g) == T
        assert _as_int(ds.mask(g)) == mask and _as_int(ds.bitval(g)) == bit
        for r, v in zip(members, ints):
            saved = 0
            for c in range(rb // 4):
                cm, cb, cv = (mask >> (32 * c)) & 0xFFFFFFFF, (bit >> (32 * c)) & 0xFFFFFFFF, (v >> (32 * c)) & 0xFFFFFFFF
                if cv & cm == cb:
                    saved += bin(cm).count("1")
            bytes_saved = (saved - rb // 4) // 8 if saved - rb // 4 > 0 else 0
            data, comp = ds.row(r)
            assert comp == (bytes_saved > 0) and data.size == rb - bytes_saved
            assert np.array_equal(oracle.decompress_row_T(data, comp, ds.mask(g), ds.bitval(g)), X[r])
    ids = np.arange(n)
    assert np.array_equal(ds.gather_decompress(ids), X)
    ds.close()


@settings(**SET)
@given(_case(False), st.sampled_from([1, 4, 16, 32, 64]))
def test_host_build_equals_oracle_strict(case, align):
    X, kind, param, _ = case
    n, rb = X.shape
    h = ibp.ibp_build(X, rb, kind, param, align_bytes=align, flags=ibp.IBP_FLAG_PAGEABLE_STORE)
    ds = oracle.Dataset(X, kind, param)
    info = h.info()
    assert info.n_groups == ds.n_groups and info.packed_bytes_bytealigned == ds.packed_bytes
    for g in range(ds.n_groups):
        m, b, k = h.metadata_host(g)
        assert k == ds.k_bits(g) and np.array_equal(m, ds.mask(g)) and np.array_equal(b, ds.bitval(g))
    for r in range(n):
        data, _k = h.packed_row(r)
        want = ds.packed_row(r)
        assert data.size == -(-want.size // align) * align and np.array_equal(data[: want.size], want) and not data[want.size:].any()
    h.destroy()
    ds.close()


@settings(**SET)
@given(_case(True), st.sampled_from([16, 32, 128]), st.booleans())
def test_host_build_equals_oracle_thresholded(case, align, slots):
    X, kind, param, thr = case
    n, rb = X.shape
    flags = ibp.IBP_FLAG_PAGEABLE_STORE | (ibp.IBP_FLAG_SLOT_LAYOUT if slots else 0)
    h = ibp.ibp_build(X, rb, kind, param, align_bytes=align, flags=flags, threshold=thr)
    ds = oracle.DatasetT(X, kind, param, thr[0], thr[1])
    info = h.info()
    assert info.thresholded == 1 and info.n_groups == ds.n_groups
    n_raw = 0
    for r in range(n):
        data, stored, comp = h.row_info(r)
        want, want_comp = ds.row(r)
        assert comp == bool(want_comp) and np.array_equal(data, want)
        assert stored == -(-want.size // align) * align
        n_raw += not comp
    assert info.n_rows_raw == n_raw
    if slots:
        slot = -(-rb // align) * align
        assert info.slot_bytes == slot and info.packed_bytes_stored >= n * slot
    h.destroy()
    ds.close()
