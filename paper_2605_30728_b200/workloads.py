"""Synthetic workloads with the shapes of BASELINE.json `configs[0..4]` plus the PAPER.md:399 (Fig. 7) sweep.

Inputs only: value distributions, table shapes, group maps and id batches.  No IBP arithmetic lives here; both the
oracle tests and the CUDA path consume these arrays.  The recipe (and the readings R15-R21 of BASELINE.json it
follows) is restated in DESIGN.md section 4.  These tables stand in for the paper's
datasets (GNN features P:430-439, Criteo-trained DLRM tables, OPT/Gemma KV and weights P:387-391),
none of which is available.

Seeds: base 20260530; config seed = base + config index; batch seed = config seed * 1000 + iteration.
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

from . import datagen

BASE_SEED = 20260530
BLOCKED, STRIDED = 0, 1


def _zipf_cdf(n: int, alpha: float) -> np.ndarray:
    w = np.arange(1, n + 1, dtype=np.float64) ** (-alpha)
    c = np.cumsum(w)
    return c / c[-1]


def _uniform01(n: int, seed: int) -> np.ndarray:
    return (datagen.u64(n, seed) >> np.uint64(11)).astype(np.float64) * (1.0 / (1 << 53))


@dataclass
class Workload:
    """One table + its group map + a batch sampler.  `table()` returns a 2-D array [n_rows, row_elems]."""
    name: str
    index: int
    n_rows: int
    row_bytes: int
    dtype: str                      # "f32" or "bf16" (bf16 tables are uint16 bit patterns)
    group_kind: int
    group_param: int
    index_span: int = 1
    align_bytes: int = 32           # packed-row alignment unit A used by default for this workload
    batch_ids: int = 0              # ids per batch (each id selects index_span rows)
    ids_unique: bool = False        # the batch sampler guarantees distinct ids (lets the caller switch de-duplication off)
    note: str = ""
    _cache: dict = field(default_factory=dict, repr=False)

    @property
    def seed(self) -> int:
        return BASE_SEED + self.index

    @property
    def row_elems(self) -> int:
        return self.row_bytes // (4 if self.dtype == "f32" else 2)

    @property
    def np_dtype(self):
        return np.float32 if self.dtype == "f32" else np.uint16

    @property
    def batch_rows(self) -> int:
        return self.batch_ids * self.index_span

    # ---- table -------------------------------------------------------------------------------------------
    def table(self, out: np.ndarray | None = None) -> np.ndarray:
        if out is None:
            out = np.empty((self.n_rows, self.row_elems), dtype=self.np_dtype)
        self.fill_rows(0, self.n_rows, out)
        return out

    def rows(self, first: int, count: int) -> np.ndarray:
        """Regenerate rows [first, first+count) alone (element streams are counter-based)."""
        out = np.empty((count, self.row_elems), dtype=self.np_dtype)
        self.fill_rows(first, count, out)
        return out

    def fill_rows(self, first: int, count: int, out: np.ndarray) -> None:
        raise NotImplementedError

    # ---- ids ---------------------------------------------------------------------------------------------
    def ids(self, iteration: int) -> np.ndarray:
        raise NotImplementedError

    def batch_seed(self, iteration: int) -> int:
        return self.seed * 1000 + iteration


# ------------------------------------------------------------------------------------------------- config 0
class Tiny(Workload):
    """configs[0]: 4,096 x 128 fp32, N(0,1) rounded to 2^-6, clipped to [-8,8]; groups of 64; 1,024 uniform ids."""

    def __init__(self, n_rows=4096, batch=1024):
        super().__init__("tiny", 0, n_rows, 512, "f32", BLOCKED, 64, 1, 32, batch)

    def fill_rows(self, first, count, out):
        e = self.row_elems
        datagen.normal_f32(count * e, self.seed, first * e, 1.0, 2.0 ** -6, 8.0, out=out.reshape(-1))

    def ids(self, iteration):
        return (datagen.u64(self.batch_ids, self.batch_seed(iteration)) % np.uint64(self.n_rows)).astype(np.int64)


# ------------------------------------------------------------------------------------------------- config 1
class GNN(Workload):
    """configs[1]: 10M x 128 fp32; ids < 70%: N(0,1) in 2^-8 steps; the rest sparse 0.0/1.0 with 2% density (R15:
    contiguous by type); groups of 256; 250k UNIQUE ids per batch, Zipf(0.9) through a seeded permutation (R16, R21)."""

    def __init__(self, n_rows=10_000_000, batch=250_000, interleaved=False):
        super().__init__("gnn", 1, n_rows, 512, "f32", BLOCKED, 256, 1, 32, batch, ids_unique=True)
        self.n_dense = (n_rows * 7) // 10
        self.interleaved = interleaved       # R15's secondary variant: row type drawn per row (70/30), every group mixes both

    def fill_rows(self, first, count, out):
        e = self.row_elems
        flat = out.reshape(-1)
        if self.interleaved:
            sparse = (datagen.u64(count, self.seed + 4242, first) % np.uint64(10)) >= np.uint64(7)
            datagen.normal_f32(count * e, self.seed, first * e, 1.0, 2.0 ** -8, 0.0, out=flat)
            sp = datagen.bernoulli_f32(count * e, self.seed + 7777, first * e, 0.02).reshape(count, e)
            out.reshape(count, e)[sparse] = sp[sparse]
            return
        nd = max(0, min(first + count, self.n_dense) - first)          # dense rows in this range
        if nd:
            datagen.normal_f32(nd * e, self.seed, first * e, 1.0, 2.0 ** -8, 0.0, out=flat[: nd * e])
        if count - nd:
            datagen.bernoulli_f32((count - nd) * e, self.seed + 7777, (first + nd) * e, 0.02, out=flat[nd * e:])

    def _sampler(self):
        if "cdf" not in self._cache:
            self._cache["cdf"] = _zipf_cdf(self.n_rows, 0.9)
            self._cache["perm"] = np.random.Generator(np.random.PCG64(self.seed)).permutation(self.n_rows)
        return self._cache["cdf"], self._cache["perm"]

    def hot_ids(self, k):
        """The k ids of highest sampling probability (Zipf rank order): what a static cache would hold."""
        return self._sampler()[1][:k].astype(np.int64)

    def ids(self, iteration):
        cdf, perm = self._sampler()
        want = min(self.batch_ids, self.n_rows)
        got = np.empty(0, dtype=np.int64)
        rnd = 0
        while got.size < want:
            u = _uniform01(2 * want, self.batch_seed(iteration) + 104729 * rnd)
            cand = perm[np.searchsorted(cdf, u, side="left").clip(0, self.n_rows - 1)]
            allc = np.concatenate([got, cand])
            _, first_idx = np.unique(allc, return_index=True)
            got = allc[np.sort(first_idx)]                                # first-occurrence order
            rnd += 1
        return got[:want].astype(np.int64)


# ------------------------------------------------------------------------------------------------- config 2
class DLRM(Workload):
    """configs[2]: 26 tables x 2M x 64 fp32 (global id = table*rows_per_table + row), U(-0.05,0.05) snapped to 2^-12;
    groups of 128; batch = 16,384 samples x 26 lookups, Zipf(1.05) per table, repeats kept, sample-major order."""

    def __init__(self, rows_per_table=2_000_000, n_tables=26, samples=16_384, hot_order=False):
        super().__init__("dlrm", 2, rows_per_table * n_tables, 256, "f32", BLOCKED, 128, 1, 32, samples * n_tables)
        self.rows_per_table, self.n_tables, self.samples = rows_per_table, n_tables, samples
        # hot_order: the store is laid out by sampling rank (what a frequency-ordered build gives, e.g. through
        # ibp_build_params.row_slot_host): slot = rank * n_tables + table, so the rows a Zipf batch touches most lie in
        # one small region of the store.  The entries are i.i.d., so the table content is the same generator either way.
        self.hot_order = hot_order

    def fill_rows(self, first, count, out):
        e = self.row_elems
        datagen.uniform_f32(count * e, self.seed, first * e, -0.05, 0.05, 2.0 ** -12, out=out.reshape(-1))

    def _sampler(self):
        if "cdf" not in self._cache:
            self._cache["cdf"] = _zipf_cdf(self.rows_per_table, 1.05)
            self._cache["perm"] = np.random.Generator(np.random.PCG64(self.seed)).permutation(self.rows_per_table)
        return self._cache["cdf"], self._cache["perm"]

    def hot_ids(self, k):
        """The k ids of highest sampling probability: rank-major over the tables (every table has the same rank law)."""
        _, perm = self._sampler()
        n, per = self.rows_per_table, -(-k // self.n_tables)
        t = np.arange(self.n_tables, dtype=np.int64)[None, :]
        row = (perm[:per, None] + t * 104729) % n
        return (t * n + row).reshape(-1)[:k].astype(np.int64)

    def ids(self, iteration):
        cdf, perm = self._sampler()
        n = self.rows_per_table
        u = _uniform01(self.samples * self.n_tables, self.batch_seed(iteration)).reshape(self.samples, self.n_tables)
        rank = np.searchsorted(cdf, u, side="left").clip(0, n - 1)
        t = np.arange(self.n_tables, dtype=np.int64)[None, :]
        if self.hot_order:
            return (rank.astype(np.int64) * self.n_tables + t).reshape(-1).astype(np.int64)
        row = (perm[rank] + t * 104729) % n                                # a different hot set per table
        return (t * n + row).reshape(-1).astype(np.int64)


# ------------------------------------------------------------------------------------------------- config 3
class KV(Workload):
    """configs[3]: bf16 K/V of a 32-layer, 32-head, head_dim 128 decoder, 16-token pages, 8 x 4,096 tokens (R18):
    store order [layer][k|v][page][head][token][128]; row = one token's head vector (256 B); group = the 16 rows of
    one (layer, k|v, page, head); one id = one page of one layer of K or of V = 512 consecutive rows.
    K ~ N(0,1), V ~ N(0, std 0.5) (R17).  A step fetches 64 distinct random pages per layer, K and V."""

    def __init__(self, layers=32, pages=2048, heads=32, page_tokens=16, pages_per_layer=64):
        self.layers, self.pages, self.heads, self.page_tokens = layers, pages, heads, page_tokens
        self.pages_per_layer = min(pages_per_layer, pages)
        span = heads * page_tokens
        super().__init__("kv", 3, layers * 2 * pages * span, 256, "bf16", BLOCKED, page_tokens, span, 16,
                         layers * 2 * self.pages_per_layer)

    def fill_rows(self, first, count, out):
        e = self.row_elems
        rows_per_plane = self.pages * self.index_span                      # rows of one (layer, k|v)
        flat = out.reshape(-1)
        r = first
        while r < first + count:
            plane = r // rows_per_plane
            end = min(first + count, (plane + 1) * rows_per_plane)
            sigma = 1.0 if plane % 2 == 0 else 0.5
            datagen.normal_bf16((end - r) * e, self.seed, r * e, sigma, out=flat[(r - first) * e:(end - first) * e])
            r = end

    def ids(self, iteration):
        out = np.empty((self.layers, self.pages_per_layer, 2), dtype=np.int64)
        for layer in range(self.layers):
            h = datagen.u64(self.pages, self.batch_seed(iteration) * 64 + layer)
            pages = np.argsort(h, kind="stable")[: self.pages_per_layer]   # distinct random pages
            for kv in (0, 1):
                out[layer, :, kv] = (layer * 2 + kv) * self.pages + pages
        return out.reshape(-1)


# ------------------------------------------------------------------------------------------------- config 4
class WeightMatrix(Workload):
    """configs[4], one matrix (R19): rows x cols bf16, N(0, 0.02); codec row = 128 consecutive bf16 of one matrix row;
    id = r*(cols/128) + t; group = column tile t over all matrix rows (strided, S = cols/128).  Streamed whole."""

    def __init__(self, rows=4096, cols=4096, layer=0, slot=0):
        assert cols % 128 == 0
        S = cols // 128
        super().__init__(f"w{rows}x{cols}", 4, rows * S, 256, "bf16", STRIDED, S, 1, 16, rows * S)
        self.mat_rows, self.mat_cols, self.layer, self.slot = rows, cols, layer, slot

    @property
    def seed(self):
        return BASE_SEED + 4 + 1000 * (self.layer * 8 + self.slot + 1)

    def fill_rows(self, first, count, out):
        e = self.row_elems
        datagen.normal_bf16(count * e, self.seed, first * e, 0.02, out=out.reshape(-1))

    def ids(self, iteration):
        return np.arange(self.n_rows, dtype=np.int64)


def weight_layer(layer: int, hidden=4096, ffn=11008):
    """The 7 matrices of one 7B-shaped decoder layer: 4 x (hidden x hidden) attention + 3 x (hidden x ffn) MLP."""
    return [WeightMatrix(hidden, hidden, layer, s) for s in range(4)] + [WeightMatrix(hidden, ffn, layer, 4 + s) for s in range(3)]


# ------------------------------------------------------------------------------------------------- Fig. 7 sweep
class Sweep(Workload):
    """synthetic Mask with a chosen popcount -> chosen space savings; 100,000 tensors of 256 B / 1 KB /
    4 KB with uniformly random variant bits; one global group; every row fetched once in random order."""

    def __init__(self, row_bytes=1024, savings=0.5, n_rows=100_000):
        super().__init__(f"sweep{row_bytes}_{int(round(savings * 100))}", 5, n_rows, row_bytes, "f32", BLOCKED, n_rows, 1, 32, n_rows)
        nbits = 8 * row_bytes
        n_fixed = int(round(savings * nbits))
        order = np.argsort(datagen.u64(nbits, self.seed + 17), kind="stable")
        bits = np.zeros(nbits, np.uint8)
        bits[order[:n_fixed]] = 1
        self.fixed = np.packbits(bits, bitorder="little")
        self.pattern = datagen.random_bytes(row_bytes, self.seed + 18)
        self.n_fixed = n_fixed

    def fill_rows(self, first, count, out):
        datagen.rows_with_fixed_bits(count, self.fixed, self.pattern, self.seed, first,
                                     out=out.view(np.uint8).reshape(-1))

    def ids(self, iteration):
        return np.argsort(datagen.u64(self.n_rows, self.batch_seed(iteration)), kind="stable").astype(np.int64)


def by_name(name: str, **kw) -> Workload:
    return {"tiny": Tiny, "gnn": GNN, "dlrm": DLRM, "kv": KV, "weights": WeightMatrix, "sweep": Sweep}[name](**kw)
