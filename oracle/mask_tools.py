"""TEST INFRASTRUCTURE ONLY: CPU oracle of IBP's mask-quality tools.

Plain numpy, one paper step per function, no blocking or fusion.  Only tests/ and bench.py's cpu_baseline leg may import
this module; it imports nothing from paper_2605_30728_b200.

What the paper defines (PAPER.md line numbers):
  bit_counters          "A counter is allocated for each bit across input tensors ... For each set bit in each input tensor,
                         we increment the corresponding counter"; on a sample of the rows for "Dataset Sampling"
                         (Mask and Bitval from a fraction of the data, ratio evaluated on the entire dataset).
  masks_from_counters   Mask/Bitval from the counters and T = ceil(tau N) (reading R2: count >= T, count <= N - T).
                         The tau sweep of P:233 ("a sweep over T values from 0.7N to N") re-thresholds the same counters.
  compressed_sizes      getCompressSize (Fig. 3 lines 1-19 = P:243-271) per row under a given Mask/Bitval and chunk size
                         CS in {1, 2, 4, 8} bytes (Fig. 13), via the row-codec oracle ibp_oracle_compress_size_T.
  kmeans_bits           "We modify k-means to use tensor bit-similarity for distances instead of absolute values".
                         Reading R25: distance = Hamming distance between a row and a centroid bit vector;
                         centroid bit = strict majority of its cluster's rows (ties -> 0: the minimiser of the summed Hamming
                         distance, lowest value on a tie); assignment ties -> lowest cluster index; an empty cluster keeps
                         its centroid; initial centroids are rows whose ids the caller passes in.
  net_space_saved       "space savings due to compression minus metadata overhead for additional Mask and Bitval":
                         1 - (sum of compressed row sizes + 2 * row_bytes * clusters) / (n_rows * row_bytes).

Parity unpinned: the READING R25 of "bit-similarity k-means" (P:542 is one sentence, the paper prints no worked example): the
pins below check this implementation of the reading, not that the authors' code takes the same distance and tie rules; and every
number of Fig. 13 / Table 5 / Fig. 15, which needs the paper's datasets.

Pins (tests/test_oracle_mask_tools.py): brute force with Python integers on tiny inputs; the closed form of the counters
of a full enumeration (2^(k-1)); tau = 1 == the AND/OR form; the participation overheads the paper prints (12.5 % at
CS = 1 B, 1.6 % at CS = 8 B); Lloyd monotonicity; exact recovery of planted clusters.
"""
from __future__ import annotations

import ctypes as C

import numpy as np

from . import _u8, lib


def bit_counters(X, row_group, n_groups, sample_ids=None):
    """counts[g, p] = number of (sampled) rows r with row_group[r] == g whose bit p is set; n[g] = rows counted."""
    Xb = _u8(X)
    n_rows, rb = Xb.shape
    row_group = np.asarray(row_group, dtype=np.int64)
    ids = np.arange(n_rows, dtype=np.int64) if sample_ids is None else np.asarray(sample_ids, dtype=np.int64)
    counts = np.zeros((n_groups, 8 * rb), np.uint64)
    n = np.zeros(n_groups, np.uint64)
    for r in ids:                                   # one row at a time, as P:229 states it
        bits = np.unpackbits(Xb[r], bitorder="little")
        counts[row_group[r]] += bits
        n[row_group[r]] += 1
    return counts, n


def threshold_of(N, tau_num, tau_den):
    """T = ceil(tau * N) in integers."""
    return (int(N) * int(tau_num) + int(tau_den) - 1) // int(tau_den)


def masks_from_counters(counts, n, tau_num, tau_den):
    """Mask/Bitval per group (R2).  A group with no counted row has no invariant bit (Mask = 0)."""
    n_groups, nbits = counts.shape
    mask = np.zeros((n_groups, nbits // 8), np.uint8)
    bitval = np.zeros((n_groups, nbits // 8), np.uint8)
    for g in range(n_groups):
        N = int(n[g])
        if N == 0:
            continue
        T = threshold_of(N, tau_num, tau_den)
        assert 2 * T > N, "tau must exceed 1/2 (R3)"
        one = counts[g] >= T
        zero = counts[g] <= N - T
        mask[g] = np.packbits(one | zero, bitorder="little")
        bitval[g] = np.packbits(one, bitorder="little")
    return mask, bitval


def compressed_sizes(X, row_group, mask, bitval, chunk_bytes=4):
    """Per row: stored size in bytes and raw flag under its group's Mask/Bitval (Fig. 3 lines 1-19)."""
    Xb = _u8(X)
    n_rows, rb = Xb.shape
    row_group = np.asarray(row_group, dtype=np.int64)
    mask = np.ascontiguousarray(mask, np.uint8)
    bitval = np.ascontiguousarray(bitval, np.uint8)
    sizes = np.zeros(n_rows, np.uint32)
    raw = np.zeros(n_rows, bool)
    L = lib()
    flag = C.c_int(0)
    for r in range(n_rows):
        g = int(row_group[r])
        sizes[r] = L.ibp_oracle_compress_size_T(Xb[r].ctypes.data, mask[g].ctypes.data, bitval[g].ctypes.data, rb, chunk_bytes,
                                                C.byref(flag))
        raw[r] = not flag.value
    return sizes, raw


def hamming(a, b):
    """Number of differing bits of two byte vectors."""
    return int(np.unpackbits(np.bitwise_xor(a, b)).sum())


def kmeans_bits(X, init_ids, iters):
    """Lloyd's k-means with Hamming distance (R25).  Returns (assign per iteration [iters][n_rows], centroids after
    the last update [k][row_bytes], cost per iteration = summed distance of each row to its assigned centroid)."""
    Xb = _u8(X)
    n_rows, rb = Xb.shape
    cent = Xb[np.asarray(init_ids, dtype=np.int64)].copy()
    k = cent.shape[0]
    assigns, costs = [], []
    for _ in range(iters):
        a = np.zeros(n_rows, np.uint32)
        cost = 0
        for r in range(n_rows):
            d = np.unpackbits(np.bitwise_xor(cent, Xb[r][None, :]), axis=1).sum(axis=1)
            a[r] = int(np.argmin(d))                # first minimum = lowest cluster index on a tie
            cost += int(d[a[r]])
        counts, n = bit_counters(Xb, a, k)
        for c in range(k):
            if n[c] == 0:
                continue                            # empty cluster keeps its centroid
            cent[c] = np.packbits(2 * counts[c] > n[c], bitorder="little")
        assigns.append(a)
        costs.append(cost)
    return np.stack(assigns), cent, costs


def net_space_saved(X, row_group, n_groups, tau_num, tau_den, chunk_bytes=4):
    """(bytes saved by compression - bytes of the groups' Mask and Bitval) / raw bytes.  Empty groups cost nothing."""
    Xb = _u8(X)
    n_rows, rb = Xb.shape
    counts, n = bit_counters(Xb, row_group, n_groups)
    mask, bitval = masks_from_counters(counts, n, tau_num, tau_den)
    sizes, _ = compressed_sizes(Xb, row_group, mask, bitval, chunk_bytes)
    meta = 2 * rb * int((n > 0).sum())
    return 1.0 - (int(sizes.astype(np.uint64).sum()) + meta) / float(n_rows * rb)
