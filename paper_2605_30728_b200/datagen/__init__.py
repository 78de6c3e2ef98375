"""Seeded synthetic inputs (ctypes binding of ibp_datagen.c) -- shared by tests of the oracle and of the CUDA path.

Holds none of IBP's arithmetic.  Every element is a pure function of (seed, index), so any sub-range of a
multi-GB table can be regenerated alone.
"""
from __future__ import annotations

import ctypes as C

import numpy as np

from .._build import build_datagen

_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(str(build_datagen()))
        u64, f32, vp = C.c_uint64, C.c_float, C.c_void_p
        L.ibp_gen_normal_f32.argtypes = [vp, u64, u64, u64, f32, f32, f32]
        L.ibp_gen_uniform_f32.argtypes = [vp, u64, u64, u64, f32, f32, f32]
        L.ibp_gen_bernoulli_f32.argtypes = [vp, u64, u64, u64, f32]
        L.ibp_gen_normal_bf16.argtypes = [vp, u64, u64, u64, f32]
        L.ibp_gen_random_bytes.argtypes = [vp, u64, u64, u64]
        L.ibp_gen_rows_with_fixed_bits.argtypes = [vp, u64, C.c_uint32, vp, vp, u64, u64]
        L.ibp_gen_u64.argtypes = [vp, u64, u64, u64]
        for f in (L.ibp_gen_normal_f32, L.ibp_gen_uniform_f32, L.ibp_gen_bernoulli_f32, L.ibp_gen_normal_bf16,
                  L.ibp_gen_random_bytes, L.ibp_gen_rows_with_fixed_bits, L.ibp_gen_u64):
            f.restype = None
        _lib = L
    return _lib


def _out(out, n, dtype):
    if out is None:
        out = np.empty(n, dtype=dtype)
    assert out.dtype == dtype and out.size == n and out.flags.c_contiguous
    return out


def normal_f32(n, seed, first=0, sigma=1.0, step=0.0, clip=0.0, out=None):
    out = _out(out, n, np.float32)
    lib().ibp_gen_normal_f32(out.ctypes.data, n, seed, first, sigma, step, clip)
    return out


def uniform_f32(n, seed, first=0, lo=0.0, hi=1.0, step=0.0, out=None):
    out = _out(out, n, np.float32)
    lib().ibp_gen_uniform_f32(out.ctypes.data, n, seed, first, lo, hi, step)
    return out


def bernoulli_f32(n, seed, first=0, p=0.5, out=None):
    out = _out(out, n, np.float32)
    lib().ibp_gen_bernoulli_f32(out.ctypes.data, n, seed, first, p)
    return out


def normal_bf16(n, seed, first=0, sigma=1.0, out=None):
    """bf16 bit patterns as uint16 (round-to-nearest-even from fp32)."""
    out = _out(out, n, np.uint16)
    lib().ibp_gen_normal_bf16(out.ctypes.data, n, seed, first, sigma)
    return out


def random_bytes(n, seed, first=0, out=None):
    out = _out(out, n, np.uint8)
    lib().ibp_gen_random_bytes(out.ctypes.data, n, seed, first)
    return out


def rows_with_fixed_bits(n_rows, fixed, pattern, seed, first_row=0, out=None):
    """Rows equal to `pattern` where `fixed` has 1 bits, fair coins elsewhere (PAPER.md:399 sweep shape)."""
    fixed = np.ascontiguousarray(fixed, dtype=np.uint8)
    pattern = np.ascontiguousarray(pattern, dtype=np.uint8)
    rb = fixed.size
    assert pattern.size == rb
    out = _out(out, n_rows * rb, np.uint8)
    lib().ibp_gen_rows_with_fixed_bits(out.ctypes.data, n_rows, rb, fixed.ctypes.data, pattern.ctypes.data, seed, first_row)
    return out.reshape(n_rows, rb)


def u64(n, seed, first=0):
    out = np.empty(n, dtype=np.uint64)
    lib().ibp_gen_u64(out.ctypes.data, n, seed, first)
    return out
