"""TEST INFRASTRUCTURE ONLY: ctypes loader for the CPU oracle (oracle/ibp_oracle.cpp).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import this package.
It imports nothing from paper_2605_30728_b200 (the CUDA path) and the CUDA path imports nothing from here.

Two oracles live here:
  (c1) gather_plain      -- the plain definition of the result: out[i] = X[ids[i]] (IBP is lossless)
  (c2) the IBP codec     -- ibp_oracle.cpp, bit by bit from PAPER.md sections 4.1-4.3
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
_SRC = _HERE / "ibp_oracle.cpp"
_SO = _HERE / "libibp_oracle.so"
_lib = None


def build(force: bool = False) -> Path:
    if force or not _SO.exists() or _SO.stat().st_mtime < _SRC.stat().st_mtime:
        tmp = _SO.with_suffix(f".so.tmp{os.getpid()}")      # per process: concurrent first-time builds (spawned test workers) do not collide
        r = subprocess.run(["g++", "-O1", "-std=c++17", "-shared", "-fPIC", str(_SRC), "-o", str(tmp)],
                           capture_output=True, text=True)
        if r.returncode != 0:
            raise RuntimeError("oracle build failed:\n" + r.stderr)
        os.replace(tmp, _SO)
    return _SO


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(str(build()))
        vp, u64, u32, i64 = C.c_void_p, C.c_uint64, C.c_uint32, C.c_int64
        L.ibp_oracle_group_masks_T.argtypes = [vp, u64, u64, u32, u64, vp, vp, vp]
        L.ibp_oracle_group_masks_T.restype = u32
        L.ibp_oracle_group_masks.argtypes = [vp, u64, u64, u32, vp, vp]
        L.ibp_oracle_group_masks.restype = u32
        L.ibp_oracle_pack_row.argtypes = [vp, vp, u32, vp]
        L.ibp_oracle_pack_row.restype = u32
        L.ibp_oracle_unpack_row.argtypes = [vp, vp, vp, u32, vp]
        L.ibp_oracle_unpack_row.restype = None
        L.ibp_oracle_compress_size_T.argtypes = [vp, vp, vp, u32, u32, C.POINTER(C.c_int)]
        L.ibp_oracle_compress_size_T.restype = u32
        L.ibp_oracle_compress_row_T.argtypes = [vp, vp, vp, u32, u32, vp, C.POINTER(C.c_int)]
        L.ibp_oracle_compress_row_T.restype = u32
        L.ibp_oracle_decompress_row_T.argtypes = [vp, C.c_int, vp, vp, u32, u32, vp]
        L.ibp_oracle_decompress_row_T.restype = None
        L.ibp_oracle_build.argtypes = [vp, u64, u32, u32, u32]
        L.ibp_oracle_build.restype = vp
        L.ibp_oracle_destroy.argtypes = [vp]
        L.ibp_oracle_destroy.restype = None
        for name in ("n_groups", "packed_bytes", "metadata_bytes"):
            f = getattr(L, "ibp_oracle_" + name)
            f.argtypes, f.restype = [vp], u64
        L.ibp_oracle_mask.argtypes = [vp, u64]
        L.ibp_oracle_mask.restype = vp
        L.ibp_oracle_bitval.argtypes = [vp, u64]
        L.ibp_oracle_bitval.restype = vp
        L.ibp_oracle_k_bits.argtypes = [vp, u64]
        L.ibp_oracle_k_bits.restype = u32
        L.ibp_oracle_packed_row.argtypes = [vp, u64, C.POINTER(u64)]
        L.ibp_oracle_packed_row.restype = vp
        L.ibp_oracle_gather_decompress.argtypes = [vp, vp, i64, u32, vp]
        L.ibp_oracle_gather_decompress.restype = C.c_int
        L.ibp_oracle_build_T.argtypes = [vp, u64, u32, u32, u32, u32, u32, u32]
        L.ibp_oracle_build_T.restype = vp
        L.ibp_oracle_destroy_T.argtypes = [vp]
        L.ibp_oracle_destroy_T.restype = None
        for name in ("n_groups", "n_raw", "stored_bytes", "rowflag_bytes"):
            f = getattr(L, "ibp_oracle_T_" + name)
            f.argtypes, f.restype = [vp], u64
        L.ibp_oracle_T_threshold.argtypes = [vp, u64]
        L.ibp_oracle_T_threshold.restype = u64
        L.ibp_oracle_T_mask.argtypes = [vp, u64]
        L.ibp_oracle_T_mask.restype = vp
        L.ibp_oracle_T_bitval.argtypes = [vp, u64]
        L.ibp_oracle_T_bitval.restype = vp
        L.ibp_oracle_T_row.argtypes = [vp, u64, C.POINTER(u64), C.POINTER(C.c_int)]
        L.ibp_oracle_T_row.restype = vp
        L.ibp_oracle_T_append.argtypes = [vp, vp, u64]
        L.ibp_oracle_T_append.restype = C.c_int
        L.ibp_oracle_T_n_rows.argtypes = [vp]
        L.ibp_oracle_T_n_rows.restype = u64
        L.ibp_oracle_gather_decompress_T.argtypes = [vp, vp, i64, u32, vp]
        L.ibp_oracle_gather_decompress_T.restype = C.c_int
        _lib = L
    return _lib


def _u8(a):
    a = np.ascontiguousarray(a)
    return a.view(np.uint8).reshape(a.shape[0], -1) if a.ndim >= 2 else a.view(np.uint8)


# ---------------------------------------------------------------------------------------------------- (c1)
def gather_plain(X, ids, index_span: int = 1):
    """Plain definition of the hot path's result: rows ids[i]*span .. +span-1 of X, as raw bytes."""
    Xb = _u8(X)
    ids = np.asarray(ids, dtype=np.int64)
    if index_span == 1:
        return Xb[ids]
    rows = (ids[:, None] * index_span + np.arange(index_span, dtype=np.int64)[None, :]).reshape(-1)
    return Xb[rows]


# ---------------------------------------------------------------------------------------------------- (c2) rows
def group_masks(rows, T=None, return_counters=False):
    """Mask/Bitval/k of one group of rows (2-D uint8 view).  T=None -> strict (T=N)."""
    R = _u8(rows)
    n, rb = R.shape
    mask = np.zeros(rb, np.uint8)
    bitval = np.zeros(rb, np.uint8)
    counters = np.zeros(8 * rb, np.uint64)
    k = lib().ibp_oracle_group_masks_T(R.ctypes.data, n, rb, rb, n if T is None else int(T), mask.ctypes.data,
                                       bitval.ctypes.data, counters.ctypes.data)
    return (mask, bitval, int(k), counters) if return_counters else (mask, bitval, int(k))


def pack_row(row, mask):
    r = _u8(np.asarray(row).reshape(1, -1))[0]
    rb = r.size
    out = np.zeros(rb + 1, np.uint8)
    k = lib().ibp_oracle_pack_row(r.ctypes.data, np.ascontiguousarray(mask).ctypes.data, rb, out.ctypes.data)
    return out[: (k + 7) // 8].copy(), int(k)


def unpack_row(packed, mask, bitval):
    mask = np.ascontiguousarray(mask, np.uint8)
    bitval = np.ascontiguousarray(bitval, np.uint8)
    rb = mask.size
    p = np.ascontiguousarray(packed, np.uint8)
    buf = np.zeros(max(rb, p.size) + 8, np.uint8)      # input may carry alignment padding; only ceil(k/8) bytes are read
    buf[: p.size] = p
    out = np.zeros(rb, np.uint8)
    lib().ibp_oracle_unpack_row(buf.ctypes.data, mask.ctypes.data, bitval.ctypes.data, rb, out.ctypes.data)
    return out


def compress_row_T(row, mask, bitval, chunk_bytes=4):
    r = _u8(np.asarray(row).reshape(1, -1))[0]
    rb = r.size
    out = np.zeros(rb, np.uint8)
    flag = C.c_int(0)
    size = lib().ibp_oracle_compress_row_T(r.ctypes.data, np.ascontiguousarray(mask).ctypes.data,
                                           np.ascontiguousarray(bitval).ctypes.data, rb, chunk_bytes, out.ctypes.data,
                                           C.byref(flag))
    return out[:size].copy(), bool(flag.value)


def decompress_row_T(data, is_compressed, mask, bitval, chunk_bytes=4):
    mask = np.ascontiguousarray(mask, np.uint8)
    rb = mask.size
    buf = np.zeros(rb + 8, np.uint8)
    d = np.ascontiguousarray(data, np.uint8)
    buf[: d.size] = d
    out = np.zeros(rb, np.uint8)
    lib().ibp_oracle_decompress_row_T(buf.ctypes.data, int(is_compressed), mask.ctypes.data,
                                      np.ascontiguousarray(bitval, np.uint8).ctypes.data, rb, chunk_bytes, out.ctypes.data)
    return out


# ---------------------------------------------------------------------------------------------------- (c2) dataset
BLOCKED, STRIDED = 0, 1


class Dataset:
    """Strict group-mode IBP over a whole table (SURVEY 8(c2) steps 1-7, Appendix A canonical store)."""

    def __init__(self, X, group_kind: int, group_param: int):
        Xb = _u8(X)
        self.n_rows, self.row_bytes = Xb.shape
        self._h = lib().ibp_oracle_build(Xb.ctypes.data, self.n_rows, self.row_bytes, group_kind, group_param)
        if not self._h:
            raise ValueError("ibp_oracle_build rejected its arguments")
        self.n_groups = int(lib().ibp_oracle_n_groups(self._h))
        self.packed_bytes = int(lib().ibp_oracle_packed_bytes(self._h))
        self.metadata_bytes = int(lib().ibp_oracle_metadata_bytes(self._h))

    def mask(self, g):
        return np.ctypeslib.as_array(C.cast(lib().ibp_oracle_mask(self._h, g), C.POINTER(C.c_uint8)), (self.row_bytes,)).copy()

    def bitval(self, g):
        return np.ctypeslib.as_array(C.cast(lib().ibp_oracle_bitval(self._h, g), C.POINTER(C.c_uint8)), (self.row_bytes,)).copy()

    def k_bits(self, g):
        return int(lib().ibp_oracle_k_bits(self._h, g))

    def packed_row(self, row_id):
        n = C.c_uint64(0)
        p = lib().ibp_oracle_packed_row(self._h, row_id, C.byref(n))
        if n.value == 0:
            return np.zeros(0, np.uint8)
        return np.ctypeslib.as_array(C.cast(p, C.POINTER(C.c_uint8)), (n.value,)).copy()

    def gather_decompress(self, ids, index_span: int = 1):
        ids = np.ascontiguousarray(ids, dtype=np.int64)
        out = np.zeros((ids.size * index_span, self.row_bytes), np.uint8)
        bad = lib().ibp_oracle_gather_decompress(self._h, ids.ctypes.data, ids.size, index_span, out.ctypes.data)
        if bad:
            raise IndexError("row id out of range")
        return out

    def close(self):
        if self._h:
            lib().ibp_oracle_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


class DatasetT:
    """Thresholded (paper-default) IBP over a whole table: Mask/Bitval per group with T = ceil(tau N_g), participation
    bits, raw rows and the per-row bitmask (SURVEY 8(c2) thresholded steps 1-7)."""

    def __init__(self, X, group_kind: int, group_param: int, thr_num: int = 4, thr_den: int = 5, chunk_bytes: int = 4):
        Xb = _u8(X)
        self.n_rows, self.row_bytes = Xb.shape
        self._h = lib().ibp_oracle_build_T(Xb.ctypes.data, self.n_rows, self.row_bytes, group_kind, group_param, thr_num, thr_den, chunk_bytes)
        if not self._h:
            raise ValueError("ibp_oracle_build_T rejected its arguments")
        self.n_groups = int(lib().ibp_oracle_T_n_groups(self._h))
        self.n_raw = int(lib().ibp_oracle_T_n_raw(self._h))
        self.stored_bytes = int(lib().ibp_oracle_T_stored_bytes(self._h))
        self.rowflag_bytes = int(lib().ibp_oracle_T_rowflag_bytes(self._h))
        self.metadata_bytes = 2 * self.row_bytes * self.n_groups

    def threshold(self, g):
        return int(lib().ibp_oracle_T_threshold(self._h, g))

    def mask(self, g):
        return np.ctypeslib.as_array(C.cast(lib().ibp_oracle_T_mask(self._h, g), C.POINTER(C.c_uint8)), (self.row_bytes,)).copy()

    def bitval(self, g):
        return np.ctypeslib.as_array(C.cast(lib().ibp_oracle_T_bitval(self._h, g), C.POINTER(C.c_uint8)), (self.row_bytes,)).copy()

    def row(self, row_id):
        """(stored bytes of the row, is_compressed)"""
        n, f = C.c_uint64(0), C.c_int(0)
        p = lib().ibp_oracle_T_row(self._h, row_id, C.byref(n), C.byref(f))
        data = np.ctypeslib.as_array(C.cast(p, C.POINTER(C.c_uint8)), (n.value,)).copy() if n.value else np.zeros(0, np.uint8)
        return data, bool(f.value)

    def append(self, rows):
        """rows produced after the build are compressed under the existing Mask/Bitval of their group."""
        R = _u8(np.asarray(rows).reshape(-1, self.row_bytes) if np.asarray(rows).ndim < 2 else rows)
        if R.shape[1] != self.row_bytes:
            raise ValueError("row size mismatch")
        if lib().ibp_oracle_T_append(self._h, R.ctypes.data, R.shape[0]):
            raise ValueError("an appended row falls in a group that has no Mask/Bitval")
        self.n_rows = int(lib().ibp_oracle_T_n_rows(self._h))
        self.n_raw = int(lib().ibp_oracle_T_n_raw(self._h))
        self.stored_bytes = int(lib().ibp_oracle_T_stored_bytes(self._h))
        self.rowflag_bytes = int(lib().ibp_oracle_T_rowflag_bytes(self._h))

    def slot_image(self, capacity_rows: int, slot_bytes: int = 0):
        """PAPER.md:361 in-place storage: "each tensor occupies its original slot and only the first compressed_size bytes are
        read": row r at r*slot_bytes (slot_bytes = row_bytes unless an alignment unit rounds it up), zero beyond its size."""
        slot = slot_bytes or self.row_bytes
        img = np.zeros((capacity_rows, slot), np.uint8)
        for r in range(self.n_rows):
            data, _ = self.row(r)
            img[r, : data.size] = data
        return img

    def gather_decompress(self, ids, index_span: int = 1):
        ids = np.ascontiguousarray(ids, dtype=np.int64)
        out = np.zeros((ids.size * index_span, self.row_bytes), np.uint8)
        if lib().ibp_oracle_gather_decompress_T(self._h, ids.ctypes.data, ids.size, index_span, out.ctypes.data):
            raise IndexError("row id out of range")
        return out

    def close(self):
        if self._h:
            lib().ibp_oracle_destroy_T(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


# ---------------------------------------------------------------------------------------------------- cache map value
# "the hashmap now maps an ID to a 3-bit data slab ID, a 40-bit offset, and a bit indicating whether the tensor
# is in compressed form or not ... We have 20 spare bits".  The paper gives the widths, not the positions; reading R22
# (DESIGN.md): offset in bits 0..39, slab id in bits 40..42, compressed flag in bit 43, bits 44..63 zero.
CACHE_OFFSET_BITS, CACHE_SLAB_BITS, CACHE_FLAG_BITS, CACHE_SPARE_BITS = 40, 3, 1, 20


def cache_value(slab: int, offset: int, compressed: bool) -> int:
    if not (0 <= slab < (1 << CACHE_SLAB_BITS)) or not (0 <= offset < (1 << CACHE_OFFSET_BITS)):
        raise ValueError("slab id needs 3 bits, offset 40 bits (PAPER.md:353)")
    return offset | (slab << CACHE_OFFSET_BITS) | (int(bool(compressed)) << (CACHE_OFFSET_BITS + CACHE_SLAB_BITS))


def cache_value_fields(value: int):
    """-> (slab, offset, compressed, spare)"""
    value = int(value)
    return ((value >> CACHE_OFFSET_BITS) & ((1 << CACHE_SLAB_BITS) - 1), value & ((1 << CACHE_OFFSET_BITS) - 1),
            bool((value >> (CACHE_OFFSET_BITS + CACHE_SLAB_BITS)) & 1), value >> (CACHE_OFFSET_BITS + CACHE_SLAB_BITS + CACHE_FLAG_BITS))
