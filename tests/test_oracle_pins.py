"""Pins for the CPU oracle (oracle/): checks against what the paper and the mathematics fix, never against itself.

Each test names the plausible mistake it would catch.  All CPU-only.
"""
from pathlib import Path

import numpy as np
import pytest

import oracle
from paper_2605_30728_b200 import datagen, workloads

GOLDEN = Path(__file__).parent / "golden"


def _fixture(name):
    out = {}
    for line in (GOLDEN / name).read_text().splitlines():
        if line.startswith("#") or "=" not in line:
            continue
        k, v = line.split("=", 1)
        out[k.strip()] = v.split()
    return out


def _hex(tokens):
    return [np.frombuffer(bytes.fromhex(t), dtype=np.uint8) for t in tokens]


def _bits(a):
    return np.unpackbits(np.ascontiguousarray(a, np.uint8), axis=-1, bitorder="little")


# ---------------------------------------------------------------------------------------------------------------------
# hand-worked fixtures
# ---------------------------------------------------------------------------------------------------------------------
def test_golden_strict_worked_example():
    """PAPER.md:229-231 with T=N; a swapped Mask/Bitval, a wrong bit order or MSB-first packing fails here."""
    fx = _fixture("worked_example_strict.txt")
    rows = np.stack(_hex(fx["rows"]))
    mask, bitval, k, counters = oracle.group_masks(rows, return_counters=True)
    assert counters.tolist() == [int(c) for c in fx["counters"]]
    assert mask.tobytes().hex().upper() == fx["mask"][0]
    assert bitval.tobytes().hex().upper() == fx["bitval"][0]
    assert k == int(fx["k_bits"][0])
    for r, want in zip(rows, fx["packed"]):
        p, kk = oracle.pack_row(r, mask)
        assert kk == k and p.tobytes().hex().upper() == want
        assert np.array_equal(oracle.unpack_row(p, mask, bitval), r)


def test_golden_thresholded_worked_example():
    """PAPER.md:231 (>=T / <=N-T, reading R2), :237, :262-271; catches strict '>' comparisons, a missing
    participation-bit charge and a wrong raw fallback."""
    fx = _fixture("worked_example_thresholded.txt")
    rows = np.stack(_hex(fx["rows"]))
    T, cs = int(fx["threshold"][0]), int(fx["chunk_bytes"][0])
    mask, bitval, _ = oracle.group_masks(rows, T=T)
    assert mask.tobytes().hex().upper() == fx["mask"][0]
    assert bitval.tobytes().hex().upper() == fx["bitval"][0]
    for r, flag, want in zip(rows, fx["compressed"], fx["stored"]):
        data, comp = oracle.compress_row_T(r, mask, bitval, cs)
        assert comp == bool(int(flag))
        assert data.tobytes().hex().upper() == want
        assert np.array_equal(oracle.decompress_row_T(data, comp, mask, bitval, cs), r)


def test_golden_thresholded_mixed_chunks():
    """A compressed tensor holding a non-participating chunk: payload order and widths."""
    fx = _fixture("worked_example_mixed_chunks.txt")
    mask, bitval, row = _hex(fx["mask"])[0], _hex(fx["bitval"])[0], _hex(fx["row"])[0]
    data, comp = oracle.compress_row_T(row, mask, bitval, int(fx["chunk_bytes"][0]))
    assert comp and data.tobytes().hex().upper() == fx["stored"][0]
    assert np.array_equal(oracle.decompress_row_T(data, comp, mask, bitval, 1), row)


# ---------------------------------------------------------------------------------------------------------------------
# Mask / Bitval
# ---------------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("n,rb,seed", [(1, 4, 1), (2, 8, 2), (5, 12, 3), (17, 16, 4), (64, 32, 5)])
def test_masks_brute_force_tiny_groups(n, rb, seed):
    """Brute force over all rows, bit by bit, in Python (BASELINE.json north_star): a bit is invariant iff the set of
    values it takes over the group has one element."""
    rng = np.random.default_rng(seed)
    # low-entropy rows so that some bits really are invariant
    rows = (rng.integers(0, 256, (n, rb), dtype=np.uint8) & rng.integers(0, 256, (1, rb), dtype=np.uint8)) | \
        rng.integers(0, 256, (1, rb), dtype=np.uint8) & np.uint8(0x11)
    mask, bitval, k = oracle.group_masks(rows)
    B = _bits(rows)
    want_mask = np.zeros(8 * rb, np.uint8)
    want_val = np.zeros(8 * rb, np.uint8)
    for p in range(8 * rb):
        seen = set(int(B[r, p]) for r in range(n))
        if len(seen) == 1:
            want_mask[p] = 1
            want_val[p] = seen.pop()
    assert np.array_equal(_bits(mask), want_mask)
    assert np.array_equal(_bits(bitval), want_val)
    assert k == 8 * rb - int(want_mask.sum())


@pytest.mark.parametrize("name", ["tiny", "gnn_dense", "gnn_sparse", "dlrm", "kv", "weights"])
def test_masks_closed_form_and_invariants(name):
    """Independent closed form: Bitval = AND of rows, Mask = NOT(OR xor AND) (SURVEY 8(c) pins); and the paper's own
    invariants: Chunk AND Mask == Bitval for every row, Bitval is 0 wherever Mask is 0."""
    rows = _sample_group(name)
    R = rows.view(np.uint8).reshape(rows.shape[0], -1)
    mask, bitval, k = oracle.group_masks(R)
    a = np.bitwise_and.reduce(R, axis=0)
    o = np.bitwise_or.reduce(R, axis=0)
    assert np.array_equal(bitval, a & ~(o ^ a))
    assert np.array_equal(mask, ~(o ^ a))
    assert np.all((R & mask) == bitval)
    assert not np.any(bitval & ~mask)
    assert k == 8 * R.shape[1] - int(_bits(mask).sum())


def _sample_group(name):
    if name == "tiny":
        return workloads.Tiny().rows(128, 64)
    if name == "gnn_dense":
        return workloads.GNN(n_rows=10_000).rows(512, 256)
    if name == "gnn_sparse":
        return workloads.GNN(n_rows=10_000).rows(7168, 256)
    if name == "dlrm":
        return workloads.DLRM(rows_per_table=4096, n_tables=2).rows(4096 + 256, 128)
    if name == "kv":
        return workloads.KV(layers=1, pages=4).rows(16 * 5, 16)
    if name == "weights":
        w = workloads.WeightMatrix(256, 512)
        return w.table()[3::4]                      # column tile 3 over all matrix rows
    raise KeyError(name)


def test_special_groups():
    """Degenerate groups (readings R12, R13): one row / identical rows -> Mask all ones, k=0; a row and its complement
    -> Mask all zeros, Bitval all zeros, k = all bits."""
    rb = 24
    r = datagen.random_bytes(rb, 11)
    for rows in (r[None, :], np.repeat(r[None, :], 7, axis=0)):
        mask, bitval, k = oracle.group_masks(rows)
        assert k == 0 and np.all(mask == 0xFF) and np.array_equal(bitval, r)
        p, kk = oracle.pack_row(r, mask)
        assert kk == 0 and p.size == 0
        assert np.array_equal(oracle.unpack_row(p, mask, bitval), r)       # decode == broadcast of Bitval
    mask, bitval, k = oracle.group_masks(np.stack([r, ~r]))
    assert k == 8 * rb and not mask.any() and not bitval.any()
    p, _ = oracle.pack_row(r, mask)
    assert np.array_equal(p, r)                                              # all-variant group: pack == memcpy
    assert np.array_equal(oracle.unpack_row(p, mask, bitval), r)


# ---------------------------------------------------------------------------------------------------------------------
# pack / unpack
# ---------------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("k,positions_seed", [(1, 0), (3, 1), (5, 2), (9, 3), (11, 4)])
def test_canonical_bit_order(k, positions_seed):
    """The 2^k rows that take every value on k chosen bit positions (constant elsewhere): Mask = NOT(those positions),
    k_g = k, and row number j packs to the integer j, LSB-first (reading R4).  Catches descending walks, MSB-first
    streams and byte-swapped output."""
    rb = 8
    rng = np.random.default_rng(positions_seed)
    pos = np.sort(rng.choice(8 * rb, size=k, replace=False))
    const = _bits(datagen.random_bytes(rb, 5 + positions_seed))
    B = np.repeat(const[None, :], 1 << k, axis=0)
    for j in range(1 << k):
        for t, p in enumerate(pos):
            B[j, p] = (j >> t) & 1
    rows = np.packbits(B, axis=1, bitorder="little")
    mask, bitval, kk = oracle.group_masks(rows)
    assert kk == k
    want_mask = np.ones(8 * rb, np.uint8)
    want_mask[pos] = 0
    assert np.array_equal(_bits(mask), want_mask)
    for j in range(1 << k):
        p, _ = oracle.pack_row(rows[j], mask)
        assert p.size == (k + 7) // 8
        assert int.from_bytes(p.tobytes(), "little") == j


@pytest.mark.parametrize("rb", [4, 12, 64, 256, 512])
def test_round_trip_random_masks_every_popcount(rb):
    """unpack(pack(x)) == x on uniformly random bit patterns, for random masks of every popcount 0..8*rb (sampled above
    64 bytes) (BASELINE.json north_star; losslessness P:11).  The rows satisfy row AND Mask == Bitval."""
    nbits = 8 * rb
    pops = range(nbits + 1) if rb <= 12 else sorted(set(np.linspace(0, nbits, 41).astype(int).tolist() + [1, nbits - 1]))
    rng = np.random.default_rng(rb)
    for pc in pops:
        mbits = np.zeros(nbits, np.uint8)
        mbits[rng.choice(nbits, size=pc, replace=False)] = 1
        mask = np.packbits(mbits, bitorder="little")
        bitval = datagen.random_bytes(rb, 1000 + pc) & mask
        row = (datagen.random_bytes(rb, 2000 + pc) & ~mask) | bitval
        p, k = oracle.pack_row(row, mask)
        assert k == nbits - pc and p.size == (k + 7) // 8                  # packed size == variant-bit count
        if k % 8:
            assert p[-1] >> (k % 8) == 0                                   # zero padding of the last byte
        assert np.array_equal(oracle.unpack_row(p, mask, bitval), row)
        # the packed stream is the variant bits in ascending order (a plain numpy compress of the bit vector)
        assert np.array_equal(_bits(p)[:k], _bits(row)[mbits == 0])


# ---------------------------------------------------------------------------------------------------------------------
# dataset level
# ---------------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("kind,param,n_rows,rb", [(0, 64, 1000, 64), (0, 7, 50, 12), (1, 5, 203, 32), (1, 8, 64, 16), (0, 1000, 10, 8)])
def test_dataset_equals_plain_gather(kind, param, n_rows, rb):
    """(c2) against (c1): gather-decompress == out[i] = X[ids[i]] byte for byte, with a ragged last group; sizes:
    packed = sum ceil(k_g/8) over rows, <= raw; metadata = 2*row_bytes per group."""
    X = (datagen.random_bytes(n_rows * rb, 77).reshape(n_rows, rb) & 0x3C) | 0x41
    ds = oracle.Dataset(X, kind, param)
    ids = (datagen.u64(500, 3) % np.uint64(n_rows)).astype(np.int64)
    assert np.array_equal(ds.gather_decompress(ids), oracle.gather_plain(X, ids))
    want_groups = -(-n_rows // param) if kind == 0 else min(param, n_rows)
    assert ds.n_groups == want_groups
    assert ds.metadata_bytes == 2 * rb * want_groups
    total = 0
    for r in range(n_rows):
        g = r // param if kind == 0 else r % param
        pr = ds.packed_row(r)
        assert pr.size == (ds.k_bits(g) + 7) // 8                          # equal for every row of a group
        total += pr.size
    assert total == ds.packed_bytes <= X.nbytes
    with pytest.raises(IndexError):
        ds.gather_decompress(np.array([n_rows], np.int64))


def _brute_masks(rows_u8, T=None):
    """Mask/Bitval of exactly these rows from Python integers: per bit position, count the rows with the bit set
     and compare with T and N - T (reading R2); nothing of oracle/ is called."""
    n, rb = rows_u8.shape
    T = n if T is None else T
    ints = [int.from_bytes(r.tobytes(), "little") for r in rows_u8]
    mask = bitval = 0
    for p in range(8 * rb):
        c1 = sum((v >> p) & 1 for v in ints)
        if c1 >= T:
            mask |= 1 << p
            bitval |= 1 << p
        elif c1 <= n - T:
            mask |= 1 << p
    to = lambda v: np.frombuffer(v.to_bytes(rb, "little"), np.uint8)
    return to(mask), to(bitval)


@pytest.mark.parametrize("kind,param,n_rows,rb", [(1, 5, 203, 8), (1, 8, 64, 4), (1, 3, 2, 4), (1, 86, 615, 8), (0, 7, 50, 8),
                                                   (0, 256, 700, 4), (0, 64, 64, 8), (0, 1000, 10, 8)])
def test_dataset_group_partition(kind, param, n_rows, rb):
    """SURVEY 8(c) strict step 1 / PAPER.md:542 (one Mask/Bitval per cluster): group g of a Dataset holds EXACTLY the rows
    X[g*G:(g+1)*G] (blocked; ragged last group) or X[g::S] (strided; n % S != 0, n < S).  A partition that takes a
    superset (or a subset) of a group's rows stays lossless and keeps n_groups, so only a direct comparison of every
    group's Mask/Bitval with masks computed from exactly those rows catches it: brute force over Python integers and the
    AND/OR closed form  Bitval = AND rows, Mask = ~(AND ^ OR)."""
    X = (datagen.random_bytes(n_rows * rb, 4242 + rb + param).reshape(n_rows, rb) & datagen.random_bytes(rb, 11)[None, :]) | 0x10
    X[:: 3] ^= (datagen.random_bytes(rb, 12) & 0x0F)[None, :]           # bits shared by SOME rows only: a wrong partition changes the masks
    ds = oracle.Dataset(X, kind, param)
    dt1 = oracle.DatasetT(X, kind, param, 1, 1)
    dt = oracle.DatasetT(X, kind, param, 4, 5)
    n_groups = -(-n_rows // param) if kind == 0 else min(param, n_rows)
    assert ds.n_groups == dt.n_groups == n_groups
    seen = np.zeros(n_rows, np.int64)
    for g in range(n_groups):
        members = np.arange(g * param, min((g + 1) * param, n_rows)) if kind == 0 else np.arange(g, n_rows, param)
        seen[members] += 1
        rows = X[members]
        a, o = np.bitwise_and.reduce(rows, axis=0), np.bitwise_or.reduce(rows, axis=0)
        want_mask, want_bitval = _brute_masks(rows)
        assert np.array_equal(want_mask, ~(a ^ o)) and np.array_equal(want_bitval, a)      # the two independent forms agree
        assert np.array_equal(ds.mask(g), want_mask), f"group {g}: Mask is not that of its own rows"
        assert np.array_equal(ds.bitval(g), want_bitval)
        assert ds.k_bits(g) == 8 * rb - int(np.unpackbits(want_mask).sum())
        assert np.array_equal(dt1.mask(g), want_mask) and np.array_equal(dt1.bitval(g), want_bitval)
        T = -(-len(members) * 4 // 5)
        assert dt.threshold(g) == T
        tm, tb = _brute_masks(rows, T)
        assert np.array_equal(dt.mask(g), tm) and np.array_equal(dt.bitval(g), tb)
    assert np.all(seen == 1)                                             # the groups partition the rows


def test_dataset_index_span():
    X = workloads.KV(layers=1, pages=4, heads=2).table()
    ds = oracle.Dataset(X, 0, 16)
    ids = np.array([3, 0, 7, 3], np.int64)
    out = ds.gather_decompress(ids, index_span=32)
    assert np.array_equal(out, oracle.gather_plain(X, ids, 32))
    assert np.array_equal(out[:32], X.view(np.uint8).reshape(X.shape[0], -1)[96:128])


def test_tiny_analytic_lower_bound():
    """Tiny (multiples of 2^-6, |x| <= 8): the low 15 mantissa bits of every fp32 element are zero, so every group has
    popcount(Mask) >= 15*128 (SURVEY 8(c) analytic bounds); DLRM: low 16 bits zero and exponent MSB zero -> >= 17*64;
    bf16 N(0,0.02) weights: exponent top bits are 011 -> >= 3*128."""
    X = workloads.Tiny().table()
    ds = oracle.Dataset(X, 0, 64)
    for g in range(ds.n_groups):
        m = ds.mask(g).view(np.uint32)
        assert np.all(m & 0x7FFF == 0x7FFF)
        assert 8 * 512 - ds.k_bits(g) >= 15 * 128
    d = workloads.DLRM(rows_per_table=1024, n_tables=1)
    ds = oracle.Dataset(d.table(), 0, 128)
    for g in range(ds.n_groups):
        assert np.all(ds.mask(g).view(np.uint32) & 0x4000FFFF == 0x4000FFFF)
        assert np.all(ds.bitval(g).view(np.uint32) & 0x4000FFFF == 0)
    w = workloads.WeightMatrix(512, 256)
    ds = oracle.Dataset(w.table(), 1, 2)
    for g in range(ds.n_groups):
        assert np.all(ds.mask(g).view(np.uint16) & 0x7000 == 0x7000)
        assert np.all(ds.bitval(g).view(np.uint16) & 0x7000 == 0x3000)


# ---------------------------------------------------------------------------------------------------------------------
# thresholded mode (specified in 8(c))
# ---------------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("cs,want_pct", [(1, 12.5), (8, 1.5625)])
def test_participation_overhead_closed_form(cs, want_pct):
    """one participation bit per chunk = 12.5 % at 1-byte chunks, '1.6 %' (1.5625 %) at 8-byte chunks.
    With every bit invariant and matching, stored size == exactly the participation bits."""
    rb = 512
    mask = np.full(rb, 0xFF, np.uint8)
    bitval = datagen.random_bytes(rb, 9)
    data, comp = oracle.compress_row_T(bitval, mask, bitval, cs)
    assert comp and data.size == rb // cs // 8
    assert 100.0 * data.size / rb == want_pct


def test_bitmask_size_closed_form():
    """bitmask = dataset / (tensor * 8): 512 GB of 1 KB tensors -> 64 MB (one flag bit per tensor)."""
    assert (512 * 2 ** 30) // (1024 * 8) == 64 * 2 ** 20


@pytest.mark.parametrize("cs", [1, 2, 4, 8])
def test_thresholded_round_trip_and_bounds(cs):
    """Round trip; compressed <= raw for every row; at T=N every chunk participates and the payload after the
    participation bits equals the strict payload."""
    w = workloads.GNN(n_rows=4096)
    rows = np.concatenate([w.rows(0, 200), w.rows(3000, 56)])
    R = rows.view(np.uint8).reshape(rows.shape[0], -1)
    rb = R.shape[1]
    for T in (int(0.8 * len(R)), len(R)):
        mask, bitval, _ = oracle.group_masks(R, T=T)
        n_comp = 0
        for r in R[::5]:
            data, comp = oracle.compress_row_T(r, mask, bitval, cs)
            assert data.size <= rb
            assert comp or data.size == rb
            n_comp += comp
            assert np.array_equal(oracle.decompress_row_T(data, comp, mask, bitval, cs), r)
            if T == len(R) and comp:
                nch = rb // cs
                bits = _bits(data)
                assert np.all(bits[:nch] == 1)
                strict, k = oracle.pack_row(r, mask)
                assert np.array_equal(bits[nch:nch + k], _bits(strict)[:k])
        assert n_comp > 0


# ---------------------------------------------------------------------------------------------------------------------
# thresholded mode at dataset level (oracle.DatasetT): Mask/Bitval per group with T = ceil(tau N_g), per-row flags, store
# ---------------------------------------------------------------------------------------------------------------------
def test_datasetT_golden_worked_example():
    """The hand-worked five-tensor example (tests/golden/worked_example_thresholded.txt; T=4, N=5 as in the caption of
    Fig. 2) run as a one-group dataset with tau = 4/5: flags, sizes, stored bytes, the per-row bitmask
    (PAPER.md:363, 1 = compressed) and the decoded rows.  Catches a wrong T rounding, swapped flag polarity, a store
    that is not in row order."""
    fx = _fixture("worked_example_thresholded.txt")
    rows = np.stack(_hex(fx["rows"]))
    ds = oracle.DatasetT(rows, oracle.BLOCKED, 5, 4, 5, chunk_bytes=1)
    assert ds.n_groups == 1 and ds.threshold(0) == 4
    assert ds.mask(0).tobytes().hex().upper() == fx["mask"][0]
    assert ds.bitval(0).tobytes().hex().upper() == fx["bitval"][0]
    flags = [int(f) for f in fx["compressed"]]
    for r in range(5):
        data, comp = ds.row(r)
        assert comp == bool(flags[r]) and data.tobytes().hex().upper() == fx["stored"][r]
    assert ds.stored_bytes == sum(len(t) // 2 for t in fx["stored"]) == 8
    assert ds.n_raw == 3 and ds.rowflag_bytes == 1
    assert np.array_equal(ds.gather_decompress(np.array([4, 0, 2, 1, 3, 0])), rows[[4, 0, 2, 1, 3, 0]])


@pytest.mark.parametrize("n,num,den,want", [(5, 4, 5, 4), (256, 4, 5, 205), (128, 4, 5, 103), (64, 7, 10, 45), (100, 1, 1, 100), (3, 4, 5, 3)])
def test_datasetT_threshold_rounding(n, num, den, want):
    """T = ceil(tau N): 'at least T/N = 80 %' and Fig. 2's T=4 for N=5; a floor would give 204/102/44/2."""
    rows = datagen.random_bytes(n * 8, 3).reshape(n, 8)
    ds = oracle.DatasetT(rows, oracle.BLOCKED, n, num, den)
    assert ds.threshold(0) == want


@pytest.mark.parametrize("kind,param,n_rows,num,den", [(0, 64, 1000, 4, 5), (0, 256, 700, 7, 10), (1, 6, 600, 4, 5), (0, 1 << 30, 500, 9, 10), (0, 16, 333, 1, 1)])
def test_datasetT_equals_plain_gather_and_invariants(kind, param, n_rows, num, den):
    """Losslessness at dataset level for blocked, strided and global (one group) scopes; the compressed
    dataset never exceeds the raw one; one flag bit per row; raw rows are stored verbatim; the stored size
    of a compressed row is row_bytes - floor((bitsSaved - chunks)/8) recomputed word-wise in numpy (Fig. 3 lines 13-18)."""
    w = workloads.GNN(n_rows=4096)
    X = np.concatenate([w.rows(0, n_rows // 2), w.rows(3000, n_rows - n_rows // 2)])
    Xb = X.view(np.uint8).reshape(n_rows, -1)
    rb = Xb.shape[1]
    ds = oracle.DatasetT(X, kind, min(param, n_rows) if kind == 0 else param, num, den)
    assert ds.n_groups == (-(-n_rows // min(param, n_rows)) if kind == 0 else param)
    assert ds.rowflag_bytes == -(-n_rows // 8)
    assert ds.stored_bytes <= Xb.nbytes
    ids = (datagen.u64(400, 5) % np.uint64(n_rows)).astype(np.int64)
    assert np.array_equal(ds.gather_decompress(ids), Xb[ids])
    total, n_raw = 0, 0
    W = Xb.view("<u4")
    for r in range(n_rows):
        g = r // min(param, n_rows) if kind == 0 else r % param
        M, B = ds.mask(g).view("<u4"), ds.bitval(g).view("<u4")
        part = (W[r] & M) == B
        saved = int(sum(bin(int(m)).count("1") for m in M[part])) - rb // 4
        size = rb - saved // 8 if saved >= 8 else rb
        data, comp = ds.row(r)
        assert data.size == size and comp == (size < rb)
        if not comp:
            assert np.array_equal(data, Xb[r])
            n_raw += 1
        total += size
    assert total == ds.stored_bytes and n_raw == ds.n_raw


def test_datasetT_tau_one_equals_strict_masks():
    """At tau = 1 the thresholded masks are the strict ones (>= N / <= 0): equal to oracle.Dataset group by group."""
    w = workloads.Tiny()
    X = w.rows(0, 512)
    a, b = oracle.Dataset(X, oracle.BLOCKED, 64), oracle.DatasetT(X, oracle.BLOCKED, 64, 1, 1)
    for g in range(a.n_groups):
        assert np.array_equal(a.mask(g), b.mask(g)) and np.array_equal(a.bitval(g), b.bitval(g))
    assert b.n_raw == 0


def test_datasetT_rejects_tau_at_most_half():
    """R3: T must exceed N/2 or a bit could be invariant-1 and invariant-0 at once (PAPER.md:231-233 sweeps 0.7..1)."""
    rows = datagen.random_bytes(64, 1).reshape(8, 8)
    with pytest.raises(ValueError):
        oracle.DatasetT(rows, oracle.BLOCKED, 8, 1, 2)


# ---------------------------------------------------------------------------------------------------------------------
# compressed GPU cache: the 64-bit map value
# ---------------------------------------------------------------------------------------------------------------------
def test_cache_value_widths_from_the_paper():
    """3-bit slab id ("up to 8 GPU slabs"), 40-bit offset ("up to 1 TB"), 1 flag bit, "20 spare bits" of 64."""
    assert oracle.CACHE_SLAB_BITS + oracle.CACHE_OFFSET_BITS + oracle.CACHE_FLAG_BITS + oracle.CACHE_SPARE_BITS == 64
    assert 1 << oracle.CACHE_SLAB_BITS == 8 and 1 << oracle.CACHE_OFFSET_BITS == 1 << 40 == 1024 ** 4
    top = oracle.cache_value(7, (1 << 40) - 1, True)
    assert top == (1 << 44) - 1 and top >> 44 == 0                       # the 20 spare bits stay zero
    for slab, off, comp in [(0, 0, False), (0, 0, True), (5, 123456789, True), (7, 1 << 39, False)]:
        assert oracle.cache_value_fields(oracle.cache_value(slab, off, comp)) == (slab, off, comp, 0)
    # the fields do not overlap: flipping one changes only that field
    a = oracle.cache_value(1, 16, True)
    assert oracle.cache_value_fields(a ^ (1 << 43)) == (1, 16, False, 0)
    assert oracle.cache_value_fields(a ^ (1 << 40)) == (0, 16, True, 0)
    with pytest.raises(ValueError):
        oracle.cache_value(8, 0, True)
    with pytest.raises(ValueError):
        oracle.cache_value(0, 1 << 40, True)


# ---------------------------------------------------------------------------------------------------------------------
# online append and the in-place slot layout
# ---------------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("kind,param,n0,n_new,rb", [(1, 6, 60, 45, 32), (0, 1 << 20, 200, 77, 64), (0, 16, 40, 8, 16), (0, 16, 40, 30, 16), (1, 4, 4, 9, 8)])
def test_append_under_existing_masks(kind, param, n0, n_new, rb):
    """Appended rows are compressed under the Mask/Bitval built from the first n0 rows: the metadata does not change, an
    appended row's stored bytes are exactly compress_row_T(row, mask_g, bitval_g) (itself pinned by the hand-worked fixtures),
    and gathering from the grown dataset equals the plain gather of the concatenated table (losslessness).  A mistake in
    the group of an appended row (id taken relative to the batch instead of the table) fails the stored-bytes check."""
    n = n0 + n_new
    X = (datagen.random_bytes(n * rb, 900 + rb).reshape(n, rb) & datagen.random_bytes(rb, 901)[None, :]) | 0x20
    X[n0 + 3] = datagen.random_bytes(rb, 902)                               # an appended row that does not match: kept raw or mostly non-participating
    X[::5, 0] ^= 0x0F
    gp = min(param, n0) if kind == 0 and param < (1 << 20) else param
    ds = oracle.DatasetT(X[:n0], kind, gp, 4, 5)
    masks = [(ds.mask(g).copy(), ds.bitval(g).copy()) for g in range(ds.n_groups)]
    n_groups = ds.n_groups
    fit = (-n0) % gp if (kind == 0 and gp < (1 << 20)) else n_new           # blocked groups: room left in the last built group
    if n_new > fit:
        with pytest.raises(ValueError):                                     # rows beyond the last built group have no metadata
            ds.append(X[n0:])
        assert ds.n_rows == n0                                              # ... and nothing was appended
    ds.append(X[n0:n0 + min(fit, n_new)])
    n = n0 + min(fit, n_new)
    assert ds.n_rows == n and ds.n_groups == n_groups
    for g, (m, b) in enumerate(masks):
        assert np.array_equal(ds.mask(g), m) and np.array_equal(ds.bitval(g), b)
    total = 0
    for r in range(n):
        g = r // gp if kind == 0 else r % gp
        want, want_comp = oracle.compress_row_T(X[r], masks[g][0], masks[g][1])
        got, comp = ds.row(r)
        assert comp == want_comp and np.array_equal(got, want), f"row {r}"
        total += want.size
    assert ds.stored_bytes == total
    ids = np.concatenate([np.arange(n, dtype=np.int64), (datagen.u64(300, 5) % np.uint64(n)).astype(np.int64)])
    assert np.array_equal(ds.gather_decompress(ids), oracle.gather_plain(X[:n], ids))
    # the in-place image keeps every row in its original slot: capacity x row_bytes bytes whatever the ratio, the first
    # `size` bytes of a slot are the compressed row, the rest is zero
    cap = n + 10
    img = ds.slot_image(cap)
    assert img.shape == (cap, rb) and img.nbytes == cap * rb
    for r in (0, n0 - 1, n - 1):
        data, _ = ds.row(r)
        assert np.array_equal(img[r, : data.size], data) and not img[r, data.size:].any()
    assert not img[n:].any()
