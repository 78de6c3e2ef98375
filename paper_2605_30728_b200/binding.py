"""Thin ctypes binding of libibp.so (include/ibp.h): same names, argument marshalling only.

Every step of the hot path runs inside the library's CUDA kernels; this module never computes anything and there is
no CPU fallback: if libibp.so cannot be built/loaded, or a call fails, an exception is raised.
PyTorch (optional here) supplies device memory and streams: pass `tensor.data_ptr()` and
`torch.cuda.current_stream().cuda_stream`.
"""
from __future__ import annotations

import ctypes as C

import numpy as np

from ._build import build_library

IBP_OK = 0
IBP_ERR_INVALID_ARG, IBP_ERR_OUT_OF_MEMORY, IBP_ERR_CUDA, IBP_ERR_BAD_STATE, IBP_ERR_UNSUPPORTED = 1, 2, 3, 4, 5
STATUS = {0: "IBP_OK", 1: "IBP_ERR_INVALID_ARG", 2: "IBP_ERR_OUT_OF_MEMORY", 3: "IBP_ERR_CUDA", 4: "IBP_ERR_BAD_STATE",
          5: "IBP_ERR_UNSUPPORTED"}
IBP_GROUP_BLOCKED, IBP_GROUP_STRIDED, IBP_GROUP_MAP = 0, 1, 2
IBP_FLAG_PAGEABLE_STORE = 1
IBP_FLAG_HOSTALLOC_STORE = 2
IBP_FLAG_SLOT_LAYOUT = 4
IBP_STORE_PAGEABLE, IBP_STORE_PINNED, IBP_STORE_MANAGED_HOST, IBP_STORE_SHARED = 0, 1, 2, 3


class IbpError(RuntimeError):
    def __init__(self, status, msg):
        super().__init__(f"{STATUS.get(status, status)}: {msg}")
        self.status = status


class ibp_build_params(C.Structure):
    _fields_ = [("struct_size", C.c_uint32), ("row_bytes", C.c_uint32), ("n_rows", C.c_uint64),
                ("group_kind", C.c_uint32), ("group_param", C.c_uint32), ("threshold_num", C.c_uint32),
                ("threshold_den", C.c_uint32), ("align_bytes", C.c_uint32), ("index_span", C.c_uint32),
                ("flags", C.c_uint32), ("n_threads", C.c_uint32), ("capacity_rows", C.c_uint64)]


class ibp_info(C.Structure):
    _fields_ = [("n_rows", C.c_uint64), ("n_groups", C.c_uint64), ("packed_bytes_stored", C.c_uint64),
                ("packed_bytes_rows", C.c_uint64), ("packed_bytes_bytealigned", C.c_uint64),
                ("metadata_bytes", C.c_uint64), ("aux_bytes", C.c_uint64), ("row_bytes", C.c_uint32),
                ("align_bytes", C.c_uint32), ("index_span", C.c_uint32), ("group_kind", C.c_uint32),
                ("group_param", C.c_uint32), ("max_row_stride", C.c_uint32), ("device", C.c_int32),
                ("store_kind", C.c_uint32), ("thresholded", C.c_uint32), ("threshold_num", C.c_uint32),
                ("threshold_den", C.c_uint32), ("reserved0", C.c_uint32), ("n_rows_raw", C.c_uint64),
                ("rowflag_bytes", C.c_uint64), ("rowoffset_bytes", C.c_uint64), ("capacity_rows", C.c_uint64),
                ("rowsize_bytes", C.c_uint64), ("slot_bytes", C.c_uint32), ("reserved1", C.c_uint32)]


class ibp_build_stats(C.Structure):
    _fields_ = [("mask_ms", C.c_double), ("size_ms", C.c_double), ("scan_ms", C.c_double), ("pack_ms", C.c_double),
                ("total_ms", C.c_double), ("raw_bytes", C.c_uint64), ("store_bytes", C.c_uint64),
                ("slices_per_group", C.c_uint32), ("reserved", C.c_uint32)]


class ibp_cache_info(C.Structure):
    _fields_ = [("capacity_bytes", C.c_uint64), ("used_bytes", C.c_uint64), ("n_entries", C.c_uint64), ("max_entries", C.c_uint64),
                ("map_bytes", C.c_uint64), ("n_slabs", C.c_uint32), ("reserved", C.c_uint32), ("slab_bytes", C.c_uint64)]


class ibp_range_desc(C.Structure):
    _fields_ = [("handle", C.c_void_p), ("packed_dev", C.c_void_p), ("first_row", C.c_int64), ("n_rows", C.c_int64), ("out_dev", C.c_void_p)]


class ibp_table_desc(C.Structure):
    _fields_ = [("struct_size", C.c_uint32), ("row_bytes", C.c_uint32), ("n_rows", C.c_uint64), ("group_kind", C.c_uint32),
                ("group_param", C.c_uint32), ("n_groups", C.c_uint64), ("row_group_dev", C.c_void_p)]


IBP_CACHE_MISS = 0xFFFFFFFFFFFFFFFF
IBP_NOALLOC_MAX_IDS = 1 << 20
IBP_MEM_MANAGED_HOST, IBP_MEM_HOSTALLOC, IBP_MEM_MALLOC_REGISTERED, IBP_MEM_THP_REGISTERED, IBP_MEM_HUGETLB_2M_REGISTERED = range(5)
IBP_SLAB_REMOTE = -2
IBP_IPC_HANDLE_BYTES = 64

# name -> (restype, argtypes); every symbol include/ibp.h declares (tests/test_abi.py checks the two lists agree)
_vp, _i64, _u64, _u32, _int = C.c_void_p, C.c_int64, C.c_uint64, C.c_uint32, C.c_int
SIGNATURES = {
    "ibp_build": (_int, [_vp, C.POINTER(ibp_build_params), C.POINTER(_vp)]),
    "ibp_build_device": (_int, [_vp, C.POINTER(ibp_build_params), _int, _vp, C.POINTER(_vp)]),
    "ibp_append_rows_device": (_int, [_vp, _vp, _i64, _vp]),
    "ibp_get_build_stats": (_int, [_vp, C.POINTER(ibp_build_stats)]),
    "ibp_upload_metadata": (_int, [_vp, _int, _vp]),
    "ibp_gather_decompress": (_int, [_vp, _vp, _i64, _vp, _vp]),
    "ibp_gather_decompress_host": (_int, [_vp, _vp, _i64, _vp, _vp]),
    "ibp_gather_decompress_noalloc": (_int, [_vp, _vp, _i64, _vp, _vp]),
    "ibp_decompress_resident": (_int, [_vp, _vp, _i64, _i64, _vp, _vp]),
    "ibp_gather_decompress_range": (_int, [_vp, _i64, _i64, _vp, _vp]),
    "ibp_gather_decompress_range_host": (_int, [_vp, _i64, _i64, _vp, _vp]),
    "ibp_decode_ranges": (_int, [C.POINTER(ibp_range_desc), _u32, _vp]),
    "ibp_decode_ranges_host": (_int, [C.POINTER(ibp_range_desc), _u32, _vp]),
    "ibp_packed_range": (_int, [_vp, _i64, _i64, C.POINTER(_vp), C.POINTER(_u64)]),
    "ibp_store_device_ptr": (_int, [_vp, C.POINTER(_vp)]),
    "ibp_packed_row": (_int, [_vp, _i64, C.POINTER(_vp), C.POINTER(_u32), C.POINTER(_u32)]),
    "ibp_row_info": (_int, [_vp, _i64, C.POINTER(_vp), C.POINTER(_u32), C.POINTER(_u32), C.POINTER(_int)]),
    "ibp_get_metadata_host": (_int, [_vp, _i64, C.POINTER(_vp), C.POINTER(_vp), C.POINTER(_u32)]),
    "ibp_get_info": (_int, [_vp, C.POINTER(ibp_info)]),
    "ibp_configure": (_int, [_vp, _u32, _u32]),
    "ibp_validate_ids": (_int, [_vp, _vp, _i64, C.POINTER(_i64), _vp]),
    "ibp_batch_link_bytes": (_int, [_vp, _vp, _i64, C.POINTER(_u64), C.POINTER(_u64), C.POINTER(_u64)]),
    "ibp_cache_create": (_int, [_vp, _u64, _u32, _u64, _vp, C.POINTER(_vp)]),
    "ibp_cache_insert": (_int, [_vp, _vp, _i64, _vp, C.POINTER(_i64)]),
    "ibp_cache_create_multi": (_int, [_vp, _u64, _u32, _vp, _u64, _vp, C.POINTER(_vp)]),
    "ibp_cache_slab_export": (_int, [_vp, _u32, _vp]),
    "ibp_cache_slab_attach": (_int, [_vp, _u32, _vp]),
    "ibp_cache_insert_slab": (_int, [_vp, _u32, _vp, _i64, _int, _vp, C.POINTER(_i64)]),
    "ibp_cache_gather_decompress": (_int, [_vp, _vp, _i64, _vp, _vp]),
    "ibp_cache_lookup": (_int, [_vp, _vp, _i64, _vp, _vp]),
    "ibp_cache_read": (_int, [_vp, _u64, _u32, _vp]),
    "ibp_cache_get_info": (_int, [_vp, C.POINTER(ibp_cache_info)]),
    "ibp_cache_destroy": (None, [_vp]),
    "ibp_export_shared": (_int, [_vp, C.c_char_p, _int]),
    "ibp_open_shared": (_int, [C.c_char_p, C.POINTER(_vp)]),
    "ibp_unlink_shared": (_int, [C.c_char_p]),
    "ibp_device_numa_node": (_int, [_int, C.POINTER(_int)]),
    "ibp_destroy": (None, [_vp]),
    "ibp_last_error": (C.c_char_p, []),
    "ibp_version": (C.c_char_p, []),
    "ibp_gather_uncompressed": (_int, [_vp, _u32, _vp, _i64, _vp, _vp]),
    "ibp_gather_uncompressed_ex": (_int, [_vp, _u32, _u64, _vp, _i64, _vp, _int, _vp]),
    "ibp_set_order_mode": (_int, [_vp, _int]),
    "ibp_set_fetch_mode": (_int, [_vp, _int]),
    "ibp_set_stream_mode": (_int, [_vp, _int]),
    "ibp_set_dedup_mode": (_int, [_vp, _int]),
    "ibp_set_rows_in_flight": (_int, [_vp, _int]),
    "ibp_host_alloc": (_int, [C.c_size_t, C.POINTER(_vp), C.POINTER(_vp)]),
    "ibp_host_free": (_int, [_vp]),
    "ibp_host_alloc_managed": (_int, [C.c_size_t, _int, C.POINTER(_vp)]),
    "ibp_host_free_managed": (_int, [_vp]),
    "ibp_measure_h2d": (_int, [_int, C.c_size_t, _int, C.POINTER(C.c_double)]),
    "ibp_measure_zero_copy_read": (_int, [_int, C.c_size_t, _int, C.POINTER(C.c_double)]),
    "ibp_measure_d2h": (_int, [_int, C.c_size_t, _int, C.POINTER(C.c_double)]),
    "ibp_measure_random_read": (_int, [_int, C.c_size_t, _u32, _int, C.POINTER(C.c_double), C.POINTER(C.c_double)]),
    "ibp_measure_random_read_kind": (_int, [_int, C.c_size_t, _u32, _int, _int, C.POINTER(C.c_double), C.POINTER(C.c_double)]),
    "ibp_table_groups": (_int, [C.POINTER(ibp_table_desc), C.POINTER(_u64)]),
    "ibp_bit_counts_device": (_int, [_vp, C.POINTER(ibp_table_desc), _vp, _i64, _vp, _vp, _vp]),
    "ibp_masks_from_counts_device": (_int, [_vp, _vp, _u64, _u32, _u32, _u32, _vp, _vp, _vp, _vp]),
    "ibp_compressed_size_device": (_int, [_vp, C.POINTER(ibp_table_desc), _vp, _vp, _u32, _vp, _vp, _vp]),
    "ibp_mask_sweep_device": (_int, [_vp, C.POINTER(ibp_table_desc), _vp, _i64, _vp, _u32, _vp, _u32, _vp, _vp, _vp]),
    "ibp_kmeans_bits_device": (_int, [_vp, _u64, _u32, _u32, _vp, _u32, _vp, _vp, _vp, _vp]),
    "ibp_order_by_group_device": (_int, [_vp, _u64, _u32, _vp, _vp, _vp]),
}

_lib = None


def lib():
    """Load (building if stale) the CUDA library.  Raises if nvcc or the sources are missing: no fallback."""
    global _lib
    if _lib is None:
        L = C.CDLL(str(build_library()))
        for name, (res, args) in SIGNATURES.items():
            f = getattr(L, name)
            f.restype, f.argtypes = res, args
        _lib = L
    return _lib


def _check(status):
    if status != IBP_OK:
        raise IbpError(status, lib().ibp_last_error().decode())


def _ptr(x):
    """numpy array -> address; int -> itself (device pointer); None -> NULL."""
    if x is None:
        return None
    if isinstance(x, np.ndarray):
        return x.ctypes.data
    return int(x)


class Handle:
    """Owns an ibp_handle*.  Methods mirror the C entry points one to one."""

    def __init__(self, ptr):
        self._h = ptr

    def upload_metadata(self, device=0, stream=None):
        _check(lib().ibp_upload_metadata(self._h, device, stream))
        return self

    def gather_decompress(self, row_ids_dev, n, out_dev, stream=None):
        _check(lib().ibp_gather_decompress(self._h, _ptr(row_ids_dev), n, _ptr(out_dev), stream))

    def gather_decompress_noalloc(self, row_ids_dev, n, out_dev, stream=None):
        _check(lib().ibp_gather_decompress_noalloc(self._h, _ptr(row_ids_dev), n, _ptr(out_dev), stream))

    def gather_decompress_host(self, row_ids_host, n, out_host, stream=None):
        _check(lib().ibp_gather_decompress_host(self._h, _ptr(row_ids_host), n, _ptr(out_host), stream))

    def decompress_resident(self, packed_dev, first_row, n_rows, out_dev, stream=None):
        _check(lib().ibp_decompress_resident(self._h, _ptr(packed_dev), first_row, n_rows, _ptr(out_dev), stream))

    def gather_decompress_range(self, first_row, n_rows, out_dev, stream=None):
        _check(lib().ibp_gather_decompress_range(self._h, first_row, n_rows, _ptr(out_dev), stream))

    def gather_decompress_range_host(self, first_row, n_rows, out_host, stream=None):
        _check(lib().ibp_gather_decompress_range_host(self._h, first_row, n_rows, _ptr(out_host), stream))

    def append_rows_device(self, rows_dev, n_new, stream=None):
        _check(lib().ibp_append_rows_device(self._h, _ptr(rows_dev), n_new, stream))
        return self

    def packed_range(self, first_row, n_rows):
        p, nb = _vp(), _u64()
        _check(lib().ibp_packed_range(self._h, first_row, n_rows, C.byref(p), C.byref(nb)))
        return p.value, nb.value

    def packed_row(self, row):
        """(bytes of the stored packed row incl. alignment padding, k_bits)"""
        p, st, k = _vp(), _u32(), _u32()
        _check(lib().ibp_packed_row(self._h, row, C.byref(p), C.byref(st), C.byref(k)))
        data = np.ctypeslib.as_array(C.cast(p.value, C.POINTER(C.c_uint8)), (st.value,)).copy() if st.value else np.zeros(0, np.uint8)
        return data, k.value

    def store_device_ptr(self) -> int:
        p = _vp()
        _check(lib().ibp_store_device_ptr(self._h, C.byref(p)))
        return p.value

    def row_ptr(self, row) -> int:
        """host address of the packed row inside the store"""
        p = _vp()
        _check(lib().ibp_row_info(self._h, row, C.byref(p), None, None, None))
        return p.value or 0

    def row_info(self, row):
        """(the row's byte-aligned stored bytes, bytes occupied incl. padding, is_compressed)"""
        p, st, sz, fl = _vp(), _u32(), _u32(), _int()
        _check(lib().ibp_row_info(self._h, row, C.byref(p), C.byref(st), C.byref(sz), C.byref(fl)))
        data = np.ctypeslib.as_array(C.cast(p.value, C.POINTER(C.c_uint8)), (sz.value,)).copy() if sz.value else np.zeros(0, np.uint8)
        return data, st.value, bool(fl.value)

    def packed_view(self, host_ptr, nbytes):
        return np.ctypeslib.as_array(C.cast(host_ptr, C.POINTER(C.c_uint8)), (nbytes,))

    def metadata_host(self, group):
        m, b, k = _vp(), _vp(), _u32()
        _check(lib().ibp_get_metadata_host(self._h, group, C.byref(m), C.byref(b), C.byref(k)))
        rb = self.info().row_bytes
        mask = np.ctypeslib.as_array(C.cast(m.value, C.POINTER(C.c_uint8)), (rb,)).copy()
        bitval = np.ctypeslib.as_array(C.cast(b.value, C.POINTER(C.c_uint8)), (rb,)).copy()
        return mask, bitval, k.value

    def info(self):
        out = ibp_info()
        _check(lib().ibp_get_info(self._h, C.byref(out)))
        return out

    def build_stats(self):
        st = ibp_build_stats()
        _check(lib().ibp_get_build_stats(self._h, C.byref(st)))
        return st

    def configure(self, max_ctas=0, warps_per_cta=0):
        _check(lib().ibp_configure(self._h, max_ctas, warps_per_cta))
        return self

    def set_order_mode(self, mode):
        _check(lib().ibp_set_order_mode(self._h, mode))
        return self

    def set_fetch_mode(self, mode):
        _check(lib().ibp_set_fetch_mode(self._h, mode))
        return self

    def set_dedup_mode(self, mode):
        _check(lib().ibp_set_dedup_mode(self._h, mode))
        return self

    def set_stream_mode(self, mode):
        _check(lib().ibp_set_stream_mode(self._h, mode))
        return self

    def set_rows_in_flight(self, n):
        _check(lib().ibp_set_rows_in_flight(self._h, n))
        return self

    def validate_ids(self, row_ids_dev, n, stream=None):
        bad = _i64()
        _check(lib().ibp_validate_ids(self._h, _ptr(row_ids_dev), n, C.byref(bad), stream))
        return bad.value

    def batch_link_bytes(self, row_ids_host):
        ids = np.ascontiguousarray(row_ids_host, dtype=np.int64)
        nu, st, ba = _u64(), _u64(), _u64()
        _check(lib().ibp_batch_link_bytes(self._h, ids.ctypes.data, ids.size, C.byref(nu), C.byref(st), C.byref(ba)))
        return nu.value, st.value, ba.value

    def export_shared(self, shm_name: str, numa_policy: int = 0):
        _check(lib().ibp_export_shared(self._h, shm_name.encode(), numa_policy))
        return self

    def destroy(self):
        if self._h:
            lib().ibp_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass


def ibp_open_shared(shm_name: str) -> Handle:
    h = _vp()
    _check(lib().ibp_open_shared(shm_name.encode(), C.byref(h)))
    return Handle(h)


def ibp_unlink_shared(shm_name: str):
    _check(lib().ibp_unlink_shared(shm_name.encode()))


def ibp_device_numa_node(device: int = 0) -> int:
    n = _int(-1)
    _check(lib().ibp_device_numa_node(device, C.byref(n)))
    return n.value


class Cache:
    """Owns an ibp_cache* (compressed GPU software cache).  Keeps its Handle alive."""

    def __init__(self, handle: Handle, capacity_bytes: int, n_slabs: int = 1, max_entries: int = 0, stream=None, slab_devices=None):
        """slab_devices (ibp_cache_create_multi): per slab a CUDA device, -1 = the handle's, IBP_SLAB_REMOTE = a peer process's."""
        c = _vp()
        if slab_devices is None:
            _check(lib().ibp_cache_create(handle._h, capacity_bytes, n_slabs, max_entries, stream, C.byref(c)))
        else:
            devs = np.ascontiguousarray(slab_devices, dtype=np.int32)
            assert devs.size == n_slabs
            _check(lib().ibp_cache_create_multi(handle._h, capacity_bytes, n_slabs, devs.ctypes.data, max_entries, stream, C.byref(c)))
        self._c, self.handle = c, handle

    def slab_export(self, slab: int) -> bytes:
        buf = C.create_string_buffer(IBP_IPC_HANDLE_BYTES)
        _check(lib().ibp_cache_slab_export(self._c, slab, buf))
        return buf.raw

    def slab_attach(self, slab: int, ipc_handle: bytes):
        assert len(ipc_handle) == IBP_IPC_HANDLE_BYTES
        _check(lib().ibp_cache_slab_attach(self._c, slab, C.create_string_buffer(ipc_handle, IBP_IPC_HANDLE_BYTES)))

    def insert_slab(self, slab: int, row_ids_host, fill: bool, stream=None) -> int:
        ids = np.ascontiguousarray(row_ids_host, dtype=np.int64)
        k = _i64()
        _check(lib().ibp_cache_insert_slab(self._c, slab, ids.ctypes.data, ids.size, 1 if fill else 0, stream, C.byref(k)))
        return k.value

    def insert(self, row_ids_host, stream=None) -> int:
        ids = np.ascontiguousarray(row_ids_host, dtype=np.int64)
        k = _i64()
        _check(lib().ibp_cache_insert(self._c, ids.ctypes.data, ids.size, stream, C.byref(k)))
        return k.value

    def gather_decompress(self, row_ids_dev, n, out_dev, stream=None):
        _check(lib().ibp_cache_gather_decompress(self._c, _ptr(row_ids_dev), n, _ptr(out_dev), stream))

    def lookup(self, row_ids_dev, n, entries_dev, stream=None):
        _check(lib().ibp_cache_lookup(self._c, _ptr(row_ids_dev), n, _ptr(entries_dev), stream))

    def read(self, entry: int, nbytes: int) -> np.ndarray:
        out = np.empty(nbytes, np.uint8)
        _check(lib().ibp_cache_read(self._c, entry, nbytes, out.ctypes.data))
        return out

    def info(self):
        ci = ibp_cache_info()
        _check(lib().ibp_cache_get_info(self._c, C.byref(ci)))
        return ci

    def destroy(self):
        if self._c:
            lib().ibp_cache_destroy(self._c)
            self._c = None

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass


def ibp_build(rows_host: np.ndarray, row_bytes: int, group_kind: int, group_param: int, align_bytes: int = 0,
              index_span: int = 1, flags: int = 0, n_threads: int = 0, threshold=(1, 1), capacity_rows: int = 0) -> Handle:
    rows = np.ascontiguousarray(rows_host)
    assert rows.nbytes % row_bytes == 0
    p = ibp_build_params(C.sizeof(ibp_build_params), row_bytes, rows.nbytes // row_bytes, group_kind, group_param,
                         threshold[0], threshold[1], align_bytes, index_span, flags, n_threads, capacity_rows)
    h = _vp()
    _check(lib().ibp_build(rows.ctypes.data, C.byref(p), C.byref(h)))
    return Handle(h)


def ibp_build_device(rows_dev, n_rows: int, row_bytes: int, group_kind: int, group_param: int, align_bytes: int = 0,
                     index_span: int = 1, flags: int = 0, threshold=(1, 1), device: int = 0, stream=None, capacity_rows: int = 0) -> Handle:
    """rows_dev: address of n_rows x row_bytes bytes the device can read (HBM or mapped host memory)."""
    p = ibp_build_params(C.sizeof(ibp_build_params), row_bytes, n_rows, group_kind, group_param,
                         threshold[0], threshold[1], align_bytes, index_span, flags, 0, capacity_rows)
    h = _vp()
    _check(lib().ibp_build_device(_ptr(rows_dev), C.byref(p), device, stream, C.byref(h)))
    return Handle(h)


def ibp_decode_ranges(ranges, stream=None):
    """ranges: [(Handle, packed_dev or None, first_row, n_rows, out_dev), ...] -> one launch per group of up to 8 compatible ranges."""
    arr = (ibp_range_desc * len(ranges))()
    for a, (h, packed, first, n, out) in zip(arr, ranges):
        a.handle, a.packed_dev, a.first_row, a.n_rows, a.out_dev = h._h.value if hasattr(h._h, "value") else h._h, _ptr(packed), first, n, _ptr(out)
    _check(lib().ibp_decode_ranges(arr, len(ranges), stream))


def ibp_decode_ranges_host(ranges, stream=None):
    """ranges: [(Handle, packed_dev or None, first_row, n_rows, out_host: numpy array or address), ...]; synchronises the stream."""
    arr = (ibp_range_desc * len(ranges))()
    for a, (h, packed, first, n, out) in zip(arr, ranges):
        a.handle, a.packed_dev, a.first_row, a.n_rows, a.out_dev = h._h.value if hasattr(h._h, "value") else h._h, _ptr(packed), first, n, _ptr(out)
    _check(lib().ibp_decode_ranges_host(arr, len(ranges), stream))


def ibp_gather_uncompressed(rows_mapped, row_bytes, row_ids_dev, n, out_dev, stream=None, n_rows=0, locality_order=False):
    if locality_order:
        _check(lib().ibp_gather_uncompressed_ex(_ptr(rows_mapped), row_bytes, n_rows, _ptr(row_ids_dev), n, _ptr(out_dev), 1, stream))
    else:
        _check(lib().ibp_gather_uncompressed(_ptr(rows_mapped), row_bytes, _ptr(row_ids_dev), n, _ptr(out_dev), stream))


class PinnedBuffer:
    """GPU-visible host memory viewed as a numpy array: pinned (ibp_host_alloc) or managed-host (ibp_host_alloc_managed)."""

    def __init__(self, nbytes, managed=False, device=0):
        hp, dp = _vp(), _vp()
        self.managed = managed
        if managed:
            _check(lib().ibp_host_alloc_managed(nbytes, device, C.byref(hp)))
            dp = hp
        else:
            _check(lib().ibp_host_alloc(nbytes, C.byref(hp), C.byref(dp)))
        self.host_ptr, self.dev_ptr, self.nbytes = hp.value, dp.value, nbytes
        self.array = np.ctypeslib.as_array(C.cast(hp.value, C.POINTER(C.c_uint8)), (nbytes,))

    def view(self, dtype, shape=None):
        a = self.array.view(dtype)
        return a.reshape(shape) if shape is not None else a

    def free(self):
        if self.host_ptr:
            self.array = None
            _check(lib().ibp_host_free_managed(self.host_ptr) if self.managed else lib().ibp_host_free(self.host_ptr))
            self.host_ptr = None

    def __del__(self):
        try:
            self.free()
        except Exception:
            pass


def ibp_measure_h2d(device=0, nbytes=1 << 30, reps=10) -> float:
    g = C.c_double()
    _check(lib().ibp_measure_h2d(device, nbytes, reps, C.byref(g)))
    return g.value


def ibp_measure_zero_copy_read(device=0, nbytes=1 << 30, reps=5) -> float:
    g = C.c_double()
    _check(lib().ibp_measure_zero_copy_read(device, nbytes, reps, C.byref(g)))
    return g.value


def ibp_measure_d2h(device=0, nbytes=1 << 30, reps=10) -> float:
    g = C.c_double()
    _check(lib().ibp_measure_d2h(device, nbytes, reps, C.byref(g)))
    return g.value


def ibp_measure_random_read(device=0, footprint_bytes=4 << 30, span_bytes=128, reps=3):
    """(spans per second, GB/s) of random span-aligned zero-copy reads from managed host-resident memory."""
    r, g = C.c_double(), C.c_double()
    _check(lib().ibp_measure_random_read(device, footprint_bytes, span_bytes, reps, C.byref(r), C.byref(g)))
    return r.value, g.value


def ibp_measure_random_read_kind(device: int, footprint_bytes: int, span_bytes: int, memory_kind: int, reps: int = 3):
    """(spans per second, GB/s) of random span reads over host memory of the given IBP_MEM_* kind"""
    a, b = C.c_double(), C.c_double()
    _check(lib().ibp_measure_random_read_kind(device, footprint_bytes, span_bytes, memory_kind, reps, C.byref(a), C.byref(b)))
    return a.value, b.value


# ---- mask-quality tools: marshalling only, the work is in csrc/ibp_analysis.cu
def table_desc(n_rows, row_bytes, group_kind, group_param=0, n_groups=0, row_group_dev=None) -> ibp_table_desc:
    return ibp_table_desc(C.sizeof(ibp_table_desc), row_bytes, n_rows, group_kind, group_param, n_groups, _ptr(row_group_dev))


def ibp_table_groups(t: ibp_table_desc) -> int:
    n = _u64()
    _check(lib().ibp_table_groups(C.byref(t), C.byref(n)))
    return n.value


def ibp_bit_counts_device(rows_dev, t, sample_ids_dev, n_sample, counts_dev, group_n_dev, stream=None):
    _check(lib().ibp_bit_counts_device(_ptr(rows_dev), C.byref(t), _ptr(sample_ids_dev), n_sample, _ptr(counts_dev), _ptr(group_n_dev), stream))


def ibp_masks_from_counts_device(counts_dev, group_n_dev, n_groups, row_bytes, tau_num, tau_den, mask_dev, bitval_dev, kbits_dev=None,
                                 stream=None):
    _check(lib().ibp_masks_from_counts_device(_ptr(counts_dev), _ptr(group_n_dev), n_groups, row_bytes, tau_num, tau_den, _ptr(mask_dev),
                                              _ptr(bitval_dev), _ptr(kbits_dev), stream))


def ibp_compressed_size_device(rows_dev, t, mask_dev, bitval_dev, chunk_bytes, sizes_dev, totals_dev, stream=None):
    _check(lib().ibp_compressed_size_device(_ptr(rows_dev), C.byref(t), _ptr(mask_dev), _ptr(bitval_dev), chunk_bytes, _ptr(sizes_dev),
                                            _ptr(totals_dev), stream))


def ibp_mask_sweep_device(rows_dev, t, sample_ids_dev, n_sample, taus, chunk_bytes, stream=None):
    """taus: [(num, den), ...]; chunk_bytes: [1|2|4|8, ...] -> (total_bytes[n_tau][n_cs], raw_rows[n_tau][n_cs]) as numpy uint64."""
    ta = np.ascontiguousarray(np.asarray(taus, dtype=np.uint32).reshape(-1, 2))
    cs = np.ascontiguousarray(np.asarray(chunk_bytes, dtype=np.uint32))
    tot = np.zeros((len(ta), len(cs)), np.uint64)
    raw = np.zeros((len(ta), len(cs)), np.uint64)
    _check(lib().ibp_mask_sweep_device(_ptr(rows_dev), C.byref(t), _ptr(sample_ids_dev), n_sample, ta.ctypes.data, len(ta), cs.ctypes.data,
                                       len(cs), tot.ctypes.data, raw.ctypes.data, stream))
    return tot, raw


def ibp_kmeans_bits_device(rows_dev, n_rows, row_bytes, k, init_ids_dev, iters, assign_dev, centroids_dev, cost_dev=None, stream=None):
    _check(lib().ibp_kmeans_bits_device(_ptr(rows_dev), n_rows, row_bytes, k, _ptr(init_ids_dev), iters, _ptr(assign_dev),
                                        _ptr(centroids_dev), _ptr(cost_dev), stream))


def ibp_order_by_group_device(row_group_dev, n_rows, n_groups, order_dev, group_start_dev=None, stream=None):
    _check(lib().ibp_order_by_group_device(_ptr(row_group_dev), n_rows, n_groups, _ptr(order_dev), _ptr(group_start_dev), stream))


def ibp_version() -> str:
    return lib().ibp_version().decode()
