// ibp_analysis.cu -- mask-quality tools of libibp.so (sm_100a): SURVEY 8(f) NEXT #4.
//
//   ibp_count_kernel      P:229  per-bit counters of the listed rows.  A warp takes a run of up to 1016 list positions; lane l
//                                owns W consecutive words of the row (one vector load per row); the 32 counters of a word are
//                                BIT-SLICED over 10 planes held in registers (plane j = bit j of the 32 running counts); eight
//                                rows are loaded at a time and enter four by four through two carry-save adders (lop3 xor3 /
//                                maj3) and a carry ripple;
//                                planes are unpacked and added to the global counters with atomicAdd only when the run's
//                                group changes or the run ends.
//   ibp_masks_kernel      P:231  Mask/Bitval from the counters for T = ceil(tau N_g): re-run per tau of the sweep.
//   ibp_csize_kernel      Fig. 3 lines 1-19  getCompressSize per row for chunk sizes 1/2/4/8 bytes: warp per row,
//                                lane per 8-byte unit, byte-wise match flags by SIMD-in-register tests, warp sum.
//   ibp_assign_kernel     P:542  k-means assignment with the Hamming distance: thread per row, the row's words transposed in
//                                shared memory (conflict-free), centroid words read warp-uniformly, four centroids per pass.
//   ibp_majority_kernel          centroid update: bit = strict majority of the cluster's counters (counted by
//                                ibp_count_kernel over the rows ordered by cluster: counting sort in three small kernels).
// Integer arithmetic only; results do not depend on the launch shape (sums of integers).  Checked against
// oracle/mask_tools.py in tests/test_gpu_mask_tools.py.
#include <algorithm>
#include <cstdint>
#include <cstdio>
#include <cstring>
#include <vector>

#include "ibp_devutil.cuh"

namespace {

struct TableDev {
    const uint32_t* rows;
    uint64_t n_rows, n_groups;
    uint32_t nw;                 // words per row
    uint32_t kind, param;
    const uint32_t* row_group;   // MAP
    const int64_t* list;         // listed rows, or nullptr = all
    uint64_t n_list;             // list length (virtual length for "all")
    uint64_t q_strided;          // STRIDED without a list: ceil(n_rows / S) (group-major virtual order)
};

__device__ __forceinline__ uint64_t table_group(const TableDev& T, uint64_t row) {
    return T.kind == IBP_GROUP_MAP ? (uint64_t)__ldg(T.row_group + row) : T.kind == IBP_GROUP_BLOCKED ? row / T.param : row % T.param;
}
// list position -> row id (or ~0 when the virtual position holds no row)
__device__ __forceinline__ uint64_t table_item(const TableDev& T, uint64_t pos) {
    if (T.list) return (uint64_t)__ldg(T.list + pos);
    if (T.kind == IBP_GROUP_STRIDED) {          // walk a tile's rows consecutively: pos = g*Q + j -> row j*S + g
        const uint64_t g = pos / T.q_strided, j = pos - g * T.q_strided, row = j * T.param + g;
        return row < T.n_rows ? row : ~0ull;
    }
    return pos;
}

constexpr int COUNT_NP = 10;               // planes: a run adds at most 2^10 - 1 rows to a counter before it is flushed
constexpr uint32_t COUNT_RUN_MAX = 1016;   // multiple of 8 below 2^10
constexpr uint32_t COUNT_RUN_MIN = 96;

__device__ __forceinline__ uint32_t axor3(uint32_t a, uint32_t b, uint32_t c) {
    uint32_t d;
    asm("lop3.b32 %0, %1, %2, %3, 0x96;" : "=r"(d) : "r"(a), "r"(b), "r"(c));
    return d;
}
__device__ __forceinline__ uint32_t amaj3(uint32_t a, uint32_t b, uint32_t c) {
    uint32_t d;
    asm("lop3.b32 %0, %1, %2, %3, 0xE8;" : "=r"(d) : "r"(a), "r"(b), "r"(c));
    return d;
}

template <int NP>
__device__ __forceinline__ void flush_planes(uint32_t* pl, uint32_t* dst /* 32 counters of this word */) {
    uint32_t any = 0;
#pragma unroll
    for (int p = 0; p < NP; ++p) any |= pl[p];
    while (any) {
        const int b = __ffs(any) - 1;
        any &= any - 1;
        uint32_t c = 0;
#pragma unroll
        for (int p = 0; p < NP; ++p) c |= ((pl[p] >> b) & 1u) << p;
        atomicAdd(dst + b, c);
    }
#pragma unroll
    for (int p = 0; p < NP; ++p) pl[p] = 0;
}

// A warp takes a run of `run_len` list positions; lane l owns W consecutive words of each 32*W-word pass (one vector load per
// row).  Positions are taken four at a time: when the four rows belong to the run's current group (the common case: sorted
// lists, blocked groups, one global group) they enter through two carry-save adders; otherwise one by one with a flush at
// every group change.
template <int W>
__global__ void __launch_bounds__(256) ibp_count_kernel(const TableDev T, uint32_t run_len, uint32_t* __restrict__ counts, uint32_t* __restrict__ group_n) {
    const int lane = threadIdx.x & 31, wpc = blockDim.x >> 5;
    const uint64_t n_runs = (T.n_list + run_len - 1) / run_len;
    const uint32_t n_pass = (T.nw + 32 * W - 1) / (32 * W);
    const uint64_t nbits = 32ull * T.nw;
    for (uint64_t run = (uint64_t)blockIdx.x * wpc + (threadIdx.x >> 5); run < n_runs; run += (uint64_t)gridDim.x * wpc) {
        const uint64_t p0 = run * run_len, p1 = min(T.n_list, p0 + run_len);
        for (uint32_t pass = 0; pass < n_pass; ++pass) {
            const uint32_t w0 = (pass * 32u + lane) * W;
            const bool active = w0 < T.nw;
            uint32_t pl[COUNT_NP][W];
#pragma unroll
            for (int p = 0; p < COUNT_NP; ++p)
#pragma unroll
                for (int q = 0; q < W; ++q) pl[p][q] = 0;
            uint64_t cur_g = ~0ull;
            uint32_t cur_n = 0;
            auto flush = [&]() {
                if (cur_g == ~0ull) return;
                if (active) {
#pragma unroll
                    for (int q = 0; q < W; ++q) {
                        uint32_t col[COUNT_NP];
#pragma unroll
                        for (int p = 0; p < COUNT_NP; ++p) col[p] = pl[p][q];
                        flush_planes<COUNT_NP>(col, counts + cur_g * nbits + 32ull * (w0 + q));
#pragma unroll
                        for (int p = 0; p < COUNT_NP; ++p) pl[p][q] = 0;
                    }
                }
                if (pass == 0 && lane == 0) atomicAdd(group_n + cur_g, cur_n);
            };
            auto add4 = [&](uint64_t r0, uint64_t r1, uint64_t r2, uint64_t r3) {
                uint32_t x0[W], x1[W], x2[W], x3[W];
                VecIO<W>::ld(T.rows + r0 * T.nw + w0, x0);
                VecIO<W>::ld(T.rows + r1 * T.nw + w0, x1);
                VecIO<W>::ld(T.rows + r2 * T.nw + w0, x2);
                VecIO<W>::ld(T.rows + r3 * T.nw + w0, x3);
#pragma unroll
                for (int q = 0; q < W; ++q) {
                    const uint32_t s1 = axor3(pl[0][q], x0[q], x1[q]), c1 = amaj3(pl[0][q], x0[q], x1[q]);
                    const uint32_t s2 = axor3(s1, x2[q], x3[q]), c2 = amaj3(s1, x2[q], x3[q]);
                    pl[0][q] = s2;
                    uint32_t c = amaj3(pl[1][q], c1, c2);
                    pl[1][q] = axor3(pl[1][q], c1, c2);
#pragma unroll
                    for (int p = 2; p < COUNT_NP; ++p) { const uint32_t t = pl[p][q]; pl[p][q] = t ^ c; c &= t; }
                }
            };
            // eight rows in flight (the kernel is latency-bound at the occupancy its plane registers allow)
            auto add8 = [&](uint64_t r0, uint64_t step) {
                uint32_t x[8][W];
#pragma unroll
                for (int i = 0; i < 8; ++i) VecIO<W>::ld(T.rows + (r0 + i * step) * T.nw + w0, x[i]);
#pragma unroll
                for (int h = 0; h < 2; ++h) {
#pragma unroll
                    for (int q = 0; q < W; ++q) {
                        const uint32_t s1 = axor3(pl[0][q], x[4 * h][q], x[4 * h + 1][q]), c1 = amaj3(pl[0][q], x[4 * h][q], x[4 * h + 1][q]);
                        const uint32_t s2 = axor3(s1, x[4 * h + 2][q], x[4 * h + 3][q]), c2 = amaj3(s1, x[4 * h + 2][q], x[4 * h + 3][q]);
                        pl[0][q] = s2;
                        uint32_t c = amaj3(pl[1][q], c1, c2);
                        pl[1][q] = axor3(pl[1][q], c1, c2);
#pragma unroll
                        for (int p = 2; p < COUNT_NP; ++p) { const uint32_t t = pl[p][q]; pl[p][q] = t ^ c; c &= t; }
                    }
                }
            };
            auto add1 = [&](uint64_t r0) {
                uint32_t x[W];
                VecIO<W>::ld(T.rows + r0 * T.nw + w0, x);
#pragma unroll
                for (int q = 0; q < W; ++q) {
                    uint32_t c = x[q];
#pragma unroll
                    for (int p = 0; p < COUNT_NP; ++p) { const uint32_t t = pl[p][q]; pl[p][q] = t ^ c; c &= t; }
                }
            };
            uint64_t pos = p0;
            if (!T.list && T.kind != IBP_GROUP_MAP) {
                // every row, blocked or strided groups: segments of one group with row ids in arithmetic progression
                while (pos < p1) {
                    uint64_t g, seg_end, row, step;
                    if (T.kind == IBP_GROUP_BLOCKED) {
                        g = pos / T.param; seg_end = min(p1, (g + 1) * (uint64_t)T.param); row = pos; step = 1;
                    } else {
                        g = pos / T.q_strided;
                        const uint64_t j = pos - g * T.q_strided, cnt = (T.n_rows - g + T.param - 1) / T.param;
                        if (j >= cnt) { pos = (g + 1) * T.q_strided; continue; }
                        seg_end = min(p1, g * T.q_strided + cnt); row = j * T.param + g; step = T.param;
                    }
                    const uint64_t n_seg = seg_end - pos;
                    cur_g = g; cur_n = (uint32_t)n_seg;
                    if (active) {
                        uint64_t i = 0;
                        for (; i + 8 <= n_seg; i += 8, row += 8 * step) add8(row, step);
                        for (; i + 4 <= n_seg; i += 4, row += 4 * step) add4(row, row + step, row + 2 * step, row + 3 * step);
                        for (; i < n_seg; ++i, row += step) add1(row);
                    }
                    flush();
                    cur_g = ~0ull;
                    pos = seg_end;
                }
            } else {
                while (pos < p1) {
                    uint64_t r[4], g[4];
                    const int m = (int)min((uint64_t)4, p1 - pos);
#pragma unroll
                    for (int i = 0; i < 4; ++i) {
                        r[i] = i < m ? table_item(T, pos + i) : ~0ull;
                        g[i] = r[i] != ~0ull ? table_group(T, r[i]) : ~0ull;
                    }
                    if (cur_g == ~0ull && g[0] != ~0ull) { cur_g = g[0]; cur_n = 0; }
                    if (m == 4 && g[0] == cur_g && g[1] == cur_g && g[2] == cur_g && g[3] == cur_g) {
                        cur_n += 4;
                        if (active) add4(r[0], r[1], r[2], r[3]);
                    } else {
                        for (int i = 0; i < m; ++i) {
                            if (r[i] == ~0ull) continue;
                            if (g[i] != cur_g) { flush(); cur_g = g[i]; cur_n = 0; }
                            cur_n += 1;
                            if (active) add1(r[i]);
                        }
                    }
                    pos += m;
                }
            }
            flush();
        }
    }
}

// one thread per (group, word)
__global__ void __launch_bounds__(256) ibp_masks_kernel(const uint32_t* __restrict__ counts, const uint32_t* __restrict__ group_n,
                                                        uint64_t n_groups, uint32_t nw, uint32_t tau_num, uint32_t tau_den,
                                                        uint32_t* __restrict__ mask, uint32_t* __restrict__ bitval, uint32_t* __restrict__ kbits) {
    const uint64_t cell = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (cell >= n_groups * nw) return;
    const uint64_t g = cell / nw;
    const uint64_t N = group_n[g];
    uint32_t mk = 0, bv = 0;
    if (N) {
        const uint64_t T = (N * tau_num + tau_den - 1) / tau_den;
        const uint32_t* c = counts + cell * 32ull;
#pragma unroll 8
        for (int b = 0; b < 32; ++b) {
            const uint64_t v = c[b];
            const uint32_t ge = v >= T, le = v <= N - T;
            mk |= (ge | le) << b;
            bv |= ge << b;
        }
    }
    mask[cell] = mk;
    bitval[cell] = bv;
    if (kbits) atomicAdd(kbits + g, (uint32_t)__popc(~mk));
}

// ------------------------------------------------------------------------------------------------ getCompressSize
template <int CS>
__device__ __forceinline__ uint32_t saved_bits_unit(uint32_t dlo, uint32_t mlo, uint32_t dhi, uint32_t mhi) {
    uint32_t s = 0;
    if (CS == 8) {
        if ((dlo | dhi) == 0) s = __popc(mlo) + __popc(mhi);
    } else if (CS == 4) {
        if (dlo == 0) s += __popc(mlo);
        if (dhi == 0) s += __popc(mhi);
    } else if (CS == 2) {
#pragma unroll
        for (int h = 0; h < 2; ++h) {
            const uint32_t sel = 0xFFFFu << (16 * h);
            if ((dlo & sel) == 0) s += __popc(mlo & sel);
            if ((dhi & sel) == 0) s += __popc(mhi & sel);
        }
    } else {
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const uint32_t sel = 0xFFu << (8 * j);
            if ((dlo & sel) == 0) s += __popc(mlo & sel);
            if ((dhi & sel) == 0) s += __popc(mhi & sel);
        }
    }
    return s;
}

// One warp per row (grid-stride).  Lane l owns the 8-byte units l, l+32, ...  A missing high word (row_bytes % 8 == 4, CS <= 4)
// enters as d = 1, m = 0: it never matches and saves nothing.
template <int CS>
__global__ void __launch_bounds__(256) ibp_csize_kernel(const TableDev T, const uint32_t* __restrict__ mask, const uint32_t* __restrict__ bitval,
                                                        uint32_t* __restrict__ sizes, unsigned long long* __restrict__ totals) {
    const int lane = threadIdx.x & 31, wpc = blockDim.x >> 5;
    const uint32_t row_bytes = 4u * T.nw, n_units = (T.nw + 1) / 2, n_chunks = row_bytes / CS;
    unsigned long long sum_sizes = 0, sum_raw = 0;
    for (uint64_t row = (uint64_t)blockIdx.x * wpc + (threadIdx.x >> 5); row < T.n_rows; row += (uint64_t)gridDim.x * wpc) {
        const uint64_t g = table_group(T, row);
        const uint32_t* x = T.rows + row * T.nw;
        const uint32_t* m = mask + g * T.nw;
        const uint32_t* b = bitval + g * T.nw;
        uint32_t saved = 0;
        for (uint32_t u = lane; u < n_units; u += 32) {
            const uint32_t w = 2 * u;
            uint32_t mlo = __ldg(m + w), dlo = (__ldg(x + w) & mlo) ^ __ldg(b + w), mhi = 0, dhi = 1;
            if (w + 1 < T.nw) { mhi = __ldg(m + w + 1); dhi = (__ldg(x + w + 1) & mhi) ^ __ldg(b + w + 1); }
            saved += saved_bits_unit<CS>(dlo, mlo, dhi, mhi);
        }
#pragma unroll
        for (int d = 16; d; d >>= 1) saved += __shfl_xor_sync(0xFFFFFFFFu, saved, d);
        const int diff = (int)saved - (int)n_chunks;                       // Fig. 3 line 13: bitsSaved - participation bits
        const uint32_t bytes_saved = diff > 0 ? (uint32_t)diff / 8u : 0u;  // floor (R9); <= 0 -> raw
        const uint32_t size = bytes_saved ? row_bytes - bytes_saved : row_bytes;
        if (lane == 0) {
            if (sizes) sizes[row] = size;
            sum_sizes += size;
            sum_raw += bytes_saved ? 0 : 1;
        }
    }
    if (lane == 0 && (sum_sizes | sum_raw)) {
        atomicAdd(totals, sum_sizes);
        atomicAdd(totals + 1, sum_raw);
    }
}

// Fast variant for rows that are a multiple of 8 bytes (8-byte aligned base): a warp takes FOUR consecutive rows per step, all
// their loads are issued before the first use, Mask/Bitval are loaded once when the four rows share a group, and the four
// sums are reduced together.
template <int CS>
__global__ void __launch_bounds__(256) ibp_csize4_kernel(const TableDev T, const uint32_t* __restrict__ mask, const uint32_t* __restrict__ bitval,
                                                         uint32_t* __restrict__ sizes, unsigned long long* __restrict__ totals) {
    const int lane = threadIdx.x & 31, wpc = blockDim.x >> 5;
    const uint32_t row_bytes = 4u * T.nw, n_units = T.nw / 2, n_chunks = row_bytes / CS;
    const uint64_t n_batches = (T.n_rows + 3) / 4;
    unsigned long long sum_sizes = 0, sum_raw = 0;
    for (uint64_t bt = (uint64_t)blockIdx.x * wpc + (threadIdx.x >> 5); bt < n_batches; bt += (uint64_t)gridDim.x * wpc) {
        const uint64_t row0 = bt * 4;
        const int m = (int)min((uint64_t)4, T.n_rows - row0);
        uint64_t g[4];
        bool same;
        if (T.kind == IBP_GROUP_BLOCKED) {      // one division per step: the four rows usually lie in one group
            g[0] = row0 / T.param;
            same = row0 + 3 < (g[0] + 1) * (uint64_t)T.param;
#pragma unroll
            for (int i = 1; i < 4; ++i) g[i] = same ? g[0] : (row0 + (i < m ? i : 0)) / T.param;
        } else {
#pragma unroll
            for (int i = 0; i < 4; ++i) g[i] = table_group(T, row0 + (i < m ? i : 0));
            same = g[0] == g[1] && g[0] == g[2] && g[0] == g[3];
        }
        uint32_t saved[4] = {0, 0, 0, 0};
        for (uint32_t u = lane; u < n_units; u += 32) {
            uint2 x[4];
#pragma unroll
            for (int i = 0; i < 4; ++i) x[i] = __ldg((const uint2*)(T.rows + (row0 + (i < m ? i : 0)) * T.nw) + u);
            if (same) {
                const uint2 mm = __ldg((const uint2*)(mask + g[0] * T.nw) + u), bb = __ldg((const uint2*)(bitval + g[0] * T.nw) + u);
#pragma unroll
                for (int i = 0; i < 4; ++i) saved[i] += saved_bits_unit<CS>((x[i].x & mm.x) ^ bb.x, mm.x, (x[i].y & mm.y) ^ bb.y, mm.y);
            } else {
#pragma unroll
                for (int i = 0; i < 4; ++i) {
                    const uint2 mm = __ldg((const uint2*)(mask + g[i] * T.nw) + u), bb = __ldg((const uint2*)(bitval + g[i] * T.nw) + u);
                    saved[i] += saved_bits_unit<CS>((x[i].x & mm.x) ^ bb.x, mm.x, (x[i].y & mm.y) ^ bb.y, mm.y);
                }
            }
        }
#pragma unroll
        for (int d = 16; d; d >>= 1) {
#pragma unroll
            for (int i = 0; i < 4; ++i) saved[i] += __shfl_xor_sync(0xFFFFFFFFu, saved[i], d);
        }
        if (lane < m) {
            const uint32_t sv = lane == 0 ? saved[0] : lane == 1 ? saved[1] : lane == 2 ? saved[2] : saved[3];
            const int diff = (int)sv - (int)n_chunks;
            const uint32_t bytes_saved = diff > 0 ? (uint32_t)diff / 8u : 0u;
            const uint32_t size = bytes_saved ? row_bytes - bytes_saved : row_bytes;
            if (sizes) sizes[row0 + lane] = size;
            sum_sizes += size;
            sum_raw += bytes_saved ? 0 : 1;
        }
    }
#pragma unroll
    for (int d = 2; d; d >>= 1) {     // lanes 0..3 hold the partial sums
        sum_sizes += __shfl_xor_sync(0xFFFFFFFFu, sum_sizes, d);
        sum_raw += __shfl_xor_sync(0xFFFFFFFFu, sum_raw, d);
    }
    if (lane == 0 && (sum_sizes | sum_raw)) {
        atomicAdd(totals, sum_sizes);
        atomicAdd(totals + 1, sum_raw);
    }
}

// ------------------------------------------------------------------------------------------------ k-means (R25)
// Thread per row.  smem: the CTA's rows, word-major (xs[w * blockDim.x + tid]).  Centroid words are read warp-uniformly.
__global__ void ibp_assign_kernel(const uint32_t* __restrict__ rows, uint64_t n_rows, uint32_t nw, const uint32_t* __restrict__ cent, uint32_t k,
                                  uint32_t* __restrict__ assign, unsigned long long* __restrict__ cost) {
    extern __shared__ uint32_t xs[];
    const uint32_t nt = blockDim.x, tid = threadIdx.x;
    const uint64_t row0 = (uint64_t)blockIdx.x * nt;
    const uint32_t rows_here = (uint32_t)min((uint64_t)nt, n_rows - row0);
    // coalesced load of rows_here x nw words, transposed into smem
    for (uint32_t i = tid; i < rows_here * nw; i += nt) {
        const uint32_t r = i / nw, w = i - r * nw;
        xs[w * nt + r] = __ldg(rows + (row0 + r) * nw + w);
    }
    __syncthreads();
    uint32_t best = 0xFFFFFFFFu, best_c = 0;
    if (tid < rows_here) {
        uint32_t c = 0;
        for (; c + 4 <= k; c += 4) {
            const uint32_t* c0 = cent + (uint64_t)c * nw;
            uint32_t d0 = 0, d1 = 0, d2 = 0, d3 = 0;
            for (uint32_t w = 0; w < nw; ++w) {
                const uint32_t x = xs[w * nt + tid];
                d0 += __popc(x ^ __ldg(c0 + w));
                d1 += __popc(x ^ __ldg(c0 + nw + w));
                d2 += __popc(x ^ __ldg(c0 + 2 * nw + w));
                d3 += __popc(x ^ __ldg(c0 + 3 * nw + w));
            }
            if (d0 < best) { best = d0; best_c = c; }            // strict <: the lowest index wins a tie
            if (d1 < best) { best = d1; best_c = c + 1; }
            if (d2 < best) { best = d2; best_c = c + 2; }
            if (d3 < best) { best = d3; best_c = c + 3; }
        }
        for (; c < k; ++c) {
            const uint32_t* c0 = cent + (uint64_t)c * nw;
            uint32_t d0 = 0;
            for (uint32_t w = 0; w < nw; ++w) d0 += __popc(xs[w * nt + tid] ^ __ldg(c0 + w));
            if (d0 < best) { best = d0; best_c = c; }
        }
        assign[row0 + tid] = best_c;
    }
    if (cost) {
        unsigned long long v = tid < rows_here ? best : 0ull;
#pragma unroll
        for (int d = 16; d; d >>= 1) v += __shfl_xor_sync(0xFFFFFFFFu, v, d);
        if ((tid & 31) == 0 && v) atomicAdd(cost, v);
    }
}

__global__ void ibp_gather_rows_kernel(const uint32_t* __restrict__ rows, uint32_t nw, const int64_t* __restrict__ ids, uint32_t k, uint32_t* __restrict__ out) {
    const uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= (uint64_t)k * nw) return;
    const uint32_t c = (uint32_t)(i / nw), w = (uint32_t)(i - (uint64_t)c * nw);
    out[i] = __ldg(rows + (uint64_t)__ldg(ids + c) * nw + w);
}

// counting sort of the rows by cluster: histogram, exclusive scan (one CTA), scatter (order inside a cluster is arbitrary:
// only sums over a cluster are taken afterwards)
__global__ void ibp_cluster_hist(const uint32_t* __restrict__ assign, uint64_t n, uint32_t* __restrict__ hist) {
    for (uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (uint64_t)gridDim.x * blockDim.x) atomicAdd(hist + assign[i], 1u);
}
__global__ void __launch_bounds__(1024) ibp_cluster_scan(const uint32_t* __restrict__ hist, uint32_t k, uint32_t* __restrict__ cursor) {
    __shared__ uint32_t part[1024];
    const uint32_t per = (k + 1023) / 1024, lo = threadIdx.x * per, hi = min(k, lo + per);
    uint32_t s = 0;
    for (uint32_t i = lo; i < hi; ++i) s += hist[i];
    part[threadIdx.x] = s;
    __syncthreads();
    if (threadIdx.x == 0) { uint32_t run = 0; for (int i = 0; i < 1024; ++i) { const uint32_t t = part[i]; part[i] = run; run += t; } }
    __syncthreads();
    uint32_t run = part[threadIdx.x];
    for (uint32_t i = lo; i < hi; ++i) { cursor[i] = run; run += hist[i]; }
}
__global__ void ibp_cluster_scatter(const uint32_t* __restrict__ assign, uint64_t n, uint32_t* __restrict__ cursor, int64_t* __restrict__ order) {
    for (uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (uint64_t)gridDim.x * blockDim.x)
        order[atomicAdd(cursor + assign[i], 1u)] = (int64_t)i;
}
// centroid bit = 1 iff 2*count > n (strict majority; tie -> 0); empty cluster: unchanged.  One thread per (cluster, word).
__global__ void ibp_majority_kernel(const uint32_t* __restrict__ counts, const uint32_t* __restrict__ group_n, uint32_t k, uint32_t nw, uint32_t* __restrict__ cent) {
    const uint64_t cell = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (cell >= (uint64_t)k * nw) return;
    const uint32_t n = group_n[cell / nw];
    if (!n) return;
    const uint32_t* c = counts + cell * 32ull;
    uint32_t v = 0;
#pragma unroll 8
    for (int b = 0; b < 32; ++b) v |= (uint32_t)(2ull * c[b] > n) << b;
    cent[cell] = v;
}

}  // namespace

// ------------------------------------------------------------------------------------------------ C ABI
static ibp_status check_table(const ibp_table_desc* t, const void* rows_dev, const char* who, TableDev* out) {
    if (!t || !rows_dev) { ibp_set_error("%s: null argument", who); return IBP_ERR_INVALID_ARG; }
    if (t->struct_size != sizeof(ibp_table_desc)) { ibp_set_error("%s: ibp_table_desc.struct_size mismatch", who); return IBP_ERR_INVALID_ARG; }
    if (t->row_bytes == 0 || t->row_bytes % 4 || t->row_bytes > 65536) { ibp_set_error("%s: row_bytes must be a multiple of 4 in 4..65536", who); return IBP_ERR_INVALID_ARG; }
    if (t->n_rows == 0) { ibp_set_error("%s: n_rows == 0", who); return IBP_ERR_INVALID_ARG; }
    uint64_t ng = 0;
    if (t->group_kind == IBP_GROUP_MAP) {
        if (!t->row_group_dev || t->n_groups == 0) { ibp_set_error("%s: IBP_GROUP_MAP needs row_group_dev and n_groups", who); return IBP_ERR_INVALID_ARG; }
        ng = t->n_groups;
    } else if (t->group_kind == IBP_GROUP_BLOCKED || t->group_kind == IBP_GROUP_STRIDED) {
        if (t->group_param == 0) { ibp_set_error("%s: group_param == 0", who); return IBP_ERR_INVALID_ARG; }
        ng = t->group_kind == IBP_GROUP_BLOCKED ? (t->n_rows + t->group_param - 1) / t->group_param : std::min<uint64_t>(t->group_param, t->n_rows);
        if (t->n_groups && t->n_groups != ng) { ibp_set_error("%s: n_groups does not match the group rule", who); return IBP_ERR_INVALID_ARG; }
    } else { ibp_set_error("%s: bad group_kind", who); return IBP_ERR_INVALID_ARG; }
    if (out) {
        TableDev T{};
        T.rows = (const uint32_t*)rows_dev; T.n_rows = t->n_rows; T.n_groups = ng; T.nw = t->row_bytes / 4;
        T.kind = t->group_kind; T.param = t->group_param ? t->group_param : 1; T.row_group = t->row_group_dev;
        T.list = nullptr; T.n_list = t->n_rows; T.q_strided = 0;
        *out = T;
    }
    return IBP_OK;
}

static int analysis_grid(uint64_t work_warps) {
    const int sms = ibp_sm_count_current();
    const uint64_t ctas = (work_warps + 7) / 8;
    return (int)std::max<uint64_t>(1, std::min<uint64_t>(ctas, (uint64_t)sms * 8));
}

extern "C" ibp_status ibp_table_groups(const ibp_table_desc* t, uint64_t* n_groups) {
    TableDev T;
    if (!n_groups) { ibp_set_error("ibp_table_groups: null argument"); return IBP_ERR_INVALID_ARG; }
    ibp_status s = check_table(t, (const void*)1, "ibp_table_groups", &T);
    if (s != IBP_OK) return s;
    *n_groups = T.n_groups;
    return IBP_OK;
}

static ibp_status launch_counts(TableDev T, const int64_t* sample_ids_dev, int64_t n_sample, uint32_t* counts_dev, uint32_t* group_n_dev, cudaStream_t st) {
    if (sample_ids_dev) { T.list = sample_ids_dev; T.n_list = (uint64_t)n_sample; }
    else if (T.kind == IBP_GROUP_STRIDED) { T.q_strided = (T.n_rows + T.param - 1) / T.param; T.n_list = T.q_strided * std::min<uint64_t>(T.param, T.n_rows); }
    if (T.n_list == 0) return IBP_OK;
    // run length: enough runs to fill the machine (8 warps x 8 CTAs per SM), each as long as the planes allow, so that the
    // atomic flushes (32 per word per run and group) stay rare
    const int grid_full = analysis_grid(~0ull >> 8);
    uint64_t run = ((T.n_list + (uint64_t)grid_full * 8 - 1) / ((uint64_t)grid_full * 8) + 7) / 8 * 8;   // ceil: no second, partial round of runs
    run = std::max<uint64_t>(COUNT_RUN_MIN, std::min<uint64_t>(COUNT_RUN_MAX, run));
    const uint64_t n_runs = (T.n_list + run - 1) / run;
    const int grid = analysis_grid(n_runs);
    const bool a16 = (uintptr_t)T.rows % 16 == 0, a8 = (uintptr_t)T.rows % 8 == 0;
    if (T.nw % 4 == 0 && a16) ibp_count_kernel<4><<<grid, 256, 0, st>>>(T, (uint32_t)run, counts_dev, group_n_dev);
    else if (T.nw % 2 == 0 && a8) ibp_count_kernel<2><<<grid, 256, 0, st>>>(T, (uint32_t)run, counts_dev, group_n_dev);
    else ibp_count_kernel<1><<<grid, 256, 0, st>>>(T, (uint32_t)run, counts_dev, group_n_dev);
    IBP_CUDA(cudaGetLastError());
    return IBP_OK;
}

extern "C" ibp_status ibp_bit_counts_device(const void* rows_dev, const ibp_table_desc* t, const int64_t* sample_ids_dev, int64_t n_sample,
                                            uint32_t* counts_dev, uint32_t* group_n_dev, void* cuda_stream) {
    TableDev T;
    ibp_status s = check_table(t, rows_dev, "ibp_bit_counts_device", &T);
    if (s != IBP_OK) return s;
    if (!counts_dev || !group_n_dev) { ibp_set_error("ibp_bit_counts_device: null output"); return IBP_ERR_INVALID_ARG; }
    if (sample_ids_dev && n_sample < 0) { ibp_set_error("ibp_bit_counts_device: n_sample < 0"); return IBP_ERR_INVALID_ARG; }
    return launch_counts(T, sample_ids_dev, n_sample, counts_dev, group_n_dev, (cudaStream_t)cuda_stream);
}

static ibp_status check_tau(uint32_t num, uint32_t den, const char* who) {
    if (den == 0 || num > den || 2ull * num <= den) { ibp_set_error("%s: tau = %u/%u is outside (1/2, 1]", who, num, den); return IBP_ERR_INVALID_ARG; }
    return IBP_OK;
}

extern "C" ibp_status ibp_masks_from_counts_device(const uint32_t* counts_dev, const uint32_t* group_n_dev, uint64_t n_groups, uint32_t row_bytes,
                                                   uint32_t tau_num, uint32_t tau_den, void* mask_dev, void* bitval_dev, uint32_t* kbits_dev,
                                                   void* cuda_stream) {
    if (!counts_dev || !group_n_dev || !mask_dev || !bitval_dev || n_groups == 0 || row_bytes == 0 || row_bytes % 4) {
        ibp_set_error("ibp_masks_from_counts_device: bad argument"); return IBP_ERR_INVALID_ARG;
    }
    ibp_status s = check_tau(tau_num, tau_den, "ibp_masks_from_counts_device");
    if (s != IBP_OK) return s;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const uint32_t nw = row_bytes / 4;
    if (kbits_dev) IBP_CUDA(cudaMemsetAsync(kbits_dev, 0, n_groups * 4, st));
    const uint64_t cells = n_groups * nw;
    ibp_masks_kernel<<<(unsigned)((cells + 255) / 256), 256, 0, st>>>(counts_dev, group_n_dev, n_groups, nw, tau_num, tau_den, (uint32_t*)mask_dev,
                                                                       (uint32_t*)bitval_dev, kbits_dev);
    IBP_CUDA(cudaGetLastError());
    return IBP_OK;
}

static ibp_status launch_csize(const TableDev& T, const void* mask_dev, const void* bitval_dev, uint32_t cs, uint32_t* sizes_dev, uint64_t* totals_dev,
                               cudaStream_t st) {
    const uint32_t* m = (const uint32_t*)mask_dev; const uint32_t* b = (const uint32_t*)bitval_dev;
    unsigned long long* tot = (unsigned long long*)totals_dev;
    const bool fast = T.nw % 2 == 0 && ((uintptr_t)T.rows | (uintptr_t)m | (uintptr_t)b) % 8 == 0;
    const int grid = analysis_grid(fast ? (T.n_rows + 3) / 4 : T.n_rows);
#define IBP_CSIZE(CS_) \
    do { if (fast) ibp_csize4_kernel<CS_><<<grid, 256, 0, st>>>(T, m, b, sizes_dev, tot); else ibp_csize_kernel<CS_><<<grid, 256, 0, st>>>(T, m, b, sizes_dev, tot); } while (0)
    switch (cs) {
        case 1: IBP_CSIZE(1); break;
        case 2: IBP_CSIZE(2); break;
        case 4: IBP_CSIZE(4); break;
        default: IBP_CSIZE(8); break;
    }
#undef IBP_CSIZE
    IBP_CUDA(cudaGetLastError());
    return IBP_OK;
}

static ibp_status check_cs(uint32_t cs, uint32_t row_bytes, const char* who) {
    if ((cs != 1 && cs != 2 && cs != 4 && cs != 8) || row_bytes % cs) { ibp_set_error("%s: chunk_bytes must be 1, 2, 4 or 8 and divide row_bytes", who); return IBP_ERR_INVALID_ARG; }
    return IBP_OK;
}

extern "C" ibp_status ibp_compressed_size_device(const void* rows_dev, const ibp_table_desc* t, const void* mask_dev, const void* bitval_dev,
                                                 uint32_t chunk_bytes, uint32_t* sizes_dev, uint64_t* totals_dev, void* cuda_stream) {
    TableDev T;
    ibp_status s = check_table(t, rows_dev, "ibp_compressed_size_device", &T);
    if (s != IBP_OK) return s;
    if (!mask_dev || !bitval_dev || !totals_dev) { ibp_set_error("ibp_compressed_size_device: null argument"); return IBP_ERR_INVALID_ARG; }
    s = check_cs(chunk_bytes, t->row_bytes, "ibp_compressed_size_device");
    if (s != IBP_OK) return s;
    return launch_csize(T, mask_dev, bitval_dev, chunk_bytes, sizes_dev, totals_dev, (cudaStream_t)cuda_stream);
}

extern "C" ibp_status ibp_mask_sweep_device(const void* rows_dev, const ibp_table_desc* t, const int64_t* sample_ids_dev, int64_t n_sample,
                                            const uint32_t* taus_host, uint32_t n_tau, const uint32_t* chunk_bytes_host, uint32_t n_cs,
                                            uint64_t* total_bytes_host, uint64_t* raw_rows_host, void* cuda_stream) {
    TableDev T;
    ibp_status s = check_table(t, rows_dev, "ibp_mask_sweep_device", &T);
    if (s != IBP_OK) return s;
    if (!taus_host || !chunk_bytes_host || !total_bytes_host || !raw_rows_host || n_tau == 0 || n_cs == 0) {
        ibp_set_error("ibp_mask_sweep_device: null or empty argument"); return IBP_ERR_INVALID_ARG;
    }
    for (uint32_t i = 0; i < n_tau; ++i) if ((s = check_tau(taus_host[2 * i], taus_host[2 * i + 1], "ibp_mask_sweep_device")) != IBP_OK) return s;
    for (uint32_t j = 0; j < n_cs; ++j) if ((s = check_cs(chunk_bytes_host[j], t->row_bytes, "ibp_mask_sweep_device")) != IBP_OK) return s;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const uint64_t ng = T.n_groups, meta_bytes = ng * (uint64_t)t->row_bytes, n_cells = (uint64_t)n_tau * n_cs;
    uint32_t *counts = nullptr, *gn = nullptr; uint8_t *mask = nullptr, *bitval = nullptr; uint64_t* totals = nullptr;
    IBP_CUDA(cudaMallocAsync((void**)&counts, ng * 32ull * T.nw * 4, st));
    IBP_CUDA(cudaMallocAsync((void**)&gn, ng * 4, st));
    IBP_CUDA(cudaMallocAsync((void**)&mask, meta_bytes, st));
    IBP_CUDA(cudaMallocAsync((void**)&bitval, meta_bytes, st));
    IBP_CUDA(cudaMallocAsync((void**)&totals, n_cells * 16, st));
    IBP_CUDA(cudaMemsetAsync(counts, 0, ng * 32ull * T.nw * 4, st));
    IBP_CUDA(cudaMemsetAsync(gn, 0, ng * 4, st));
    IBP_CUDA(cudaMemsetAsync(totals, 0, n_cells * 16, st));
    s = launch_counts(T, sample_ids_dev, n_sample, counts, gn, st);                               // one counting pass
    for (uint32_t i = 0; s == IBP_OK && i < n_tau; ++i) {                                         // re-threshold per tau
        s = ibp_masks_from_counts_device(counts, gn, ng, t->row_bytes, taus_host[2 * i], taus_host[2 * i + 1], mask, bitval, nullptr, st);
        for (uint32_t j = 0; s == IBP_OK && j < n_cs; ++j)                                        // sizes of ALL rows per chunk size
            s = launch_csize(T, mask, bitval, chunk_bytes_host[j], nullptr, totals + 2 * ((uint64_t)i * n_cs + j), st);
    }
    std::vector<uint64_t> host(2 * n_cells);
    if (s == IBP_OK) {
        IBP_CUDA(cudaMemcpyAsync(host.data(), totals, n_cells * 16, cudaMemcpyDeviceToHost, st));
        IBP_CUDA(cudaStreamSynchronize(st));
        for (uint64_t c = 0; c < n_cells; ++c) { total_bytes_host[c] = host[2 * c]; raw_rows_host[c] = host[2 * c + 1]; }
    }
    cudaFreeAsync(counts, st); cudaFreeAsync(gn, st); cudaFreeAsync(mask, st); cudaFreeAsync(bitval, st); cudaFreeAsync(totals, st);
    return s;
}

extern "C" ibp_status ibp_kmeans_bits_device(const void* rows_dev, uint64_t n_rows, uint32_t row_bytes, uint32_t k, const int64_t* init_ids_dev,
                                             uint32_t iters, uint32_t* assign_dev, void* centroids_dev, uint64_t* cost_dev, void* cuda_stream) {
    if (!rows_dev || !init_ids_dev || !assign_dev || !centroids_dev || n_rows == 0 || k == 0 || iters == 0) {
        ibp_set_error("ibp_kmeans_bits_device: null or empty argument"); return IBP_ERR_INVALID_ARG;
    }
    if (row_bytes == 0 || row_bytes % 4 || row_bytes > 4096) { ibp_set_error("ibp_kmeans_bits_device: row_bytes must be a multiple of 4 in 4..4096"); return IBP_ERR_INVALID_ARG; }
    if (n_rows > 0xFFFFFFFFull) { ibp_set_error("ibp_kmeans_bits_device: n_rows too large"); return IBP_ERR_INVALID_ARG; }
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const uint32_t nw = row_bytes / 4;
    const uint32_t* rows = (const uint32_t*)rows_dev;
    uint32_t* cent = (uint32_t*)centroids_dev;
    // assignment CTA: as many rows (threads) as fit ~160 KB of shared memory, 32..256
    uint32_t nt = std::min<uint32_t>(256, (160u * 1024u / row_bytes) / 32u * 32u);
    if (nt < 32) nt = 32;
    const size_t smem = (size_t)nt * row_bytes;
    static unsigned long long optin_done = 0;
    if (smem > 48 * 1024) IBP_CUDA(ibp_optin_max_smem(ibp_assign_kernel, &optin_done));
    uint32_t *counts = nullptr, *gn = nullptr, *hist = nullptr, *cursor = nullptr; int64_t* order = nullptr;
    IBP_CUDA(cudaMallocAsync((void**)&counts, (uint64_t)k * 32ull * nw * 4, st));
    IBP_CUDA(cudaMallocAsync((void**)&gn, (uint64_t)k * 4, st));
    IBP_CUDA(cudaMallocAsync((void**)&hist, (uint64_t)k * 4, st));
    IBP_CUDA(cudaMallocAsync((void**)&cursor, (uint64_t)k * 4, st));
    IBP_CUDA(cudaMallocAsync((void**)&order, n_rows * 8, st));
    if (cost_dev) IBP_CUDA(cudaMemsetAsync(cost_dev, 0, (uint64_t)iters * 8, st));
    ibp_gather_rows_kernel<<<(unsigned)(((uint64_t)k * nw + 255) / 256), 256, 0, st>>>(rows, nw, init_ids_dev, k, cent);
    IBP_CUDA(cudaGetLastError());
    TableDev T{};
    T.rows = rows; T.n_rows = n_rows; T.n_groups = k; T.nw = nw; T.kind = IBP_GROUP_MAP; T.param = 1; T.row_group = assign_dev;
    const int grid_n = analysis_grid((n_rows + 31) / 32);
    ibp_status s = IBP_OK;
    for (uint32_t it = 0; it < iters && s == IBP_OK; ++it) {
        ibp_assign_kernel<<<(unsigned)((n_rows + nt - 1) / nt), nt, smem, st>>>(rows, n_rows, nw, cent, k, assign_dev,
                                                                               cost_dev ? (unsigned long long*)cost_dev + it : nullptr);
        IBP_CUDA(cudaGetLastError());
        IBP_CUDA(cudaMemsetAsync(hist, 0, (uint64_t)k * 4, st));
        IBP_CUDA(cudaMemsetAsync(counts, 0, (uint64_t)k * 32ull * nw * 4, st));
        IBP_CUDA(cudaMemsetAsync(gn, 0, (uint64_t)k * 4, st));
        ibp_cluster_hist<<<grid_n, 256, 0, st>>>(assign_dev, n_rows, hist);
        ibp_cluster_scan<<<1, 1024, 0, st>>>(hist, k, cursor);
        ibp_cluster_scatter<<<grid_n, 256, 0, st>>>(assign_dev, n_rows, cursor, order);
        IBP_CUDA(cudaGetLastError());
        s = launch_counts(T, order, (int64_t)n_rows, counts, gn, st);
        if (s != IBP_OK) break;
        ibp_majority_kernel<<<(unsigned)(((uint64_t)k * nw + 255) / 256), 256, 0, st>>>(counts, gn, k, nw, cent);
        IBP_CUDA(cudaGetLastError());
    }
    cudaFreeAsync(counts, st); cudaFreeAsync(gn, st); cudaFreeAsync(hist, st); cudaFreeAsync(cursor, st); cudaFreeAsync(order, st);
    return s;
}

extern "C" ibp_status ibp_order_by_group_device(const uint32_t* row_group_dev, uint64_t n_rows, uint32_t n_groups, int64_t* order_dev,
                                                uint32_t* group_start_dev, void* cuda_stream) {
    if (!row_group_dev || !order_dev || n_rows == 0 || n_groups == 0 || n_rows > 0xFFFFFFFFull) {
        ibp_set_error("ibp_order_by_group_device: null or empty argument (at most 2^32 - 1 rows)"); return IBP_ERR_INVALID_ARG;
    }
    cudaStream_t st = (cudaStream_t)cuda_stream;
    uint32_t *hist = nullptr, *cursor = nullptr;
    IBP_CUDA(cudaMallocAsync((void**)&hist, (uint64_t)n_groups * 4, st));
    IBP_CUDA(cudaMallocAsync((void**)&cursor, (uint64_t)n_groups * 4, st));
    IBP_CUDA(cudaMemsetAsync(hist, 0, (uint64_t)n_groups * 4, st));
    const int grid = analysis_grid((n_rows + 31) / 32);
    ibp_cluster_hist<<<grid, 256, 0, st>>>(row_group_dev, n_rows, hist);
    ibp_cluster_scan<<<1, 1024, 0, st>>>(hist, n_groups, cursor);
    IBP_CUDA(cudaGetLastError());
    if (group_start_dev) {
        const uint32_t last = (uint32_t)n_rows;
        IBP_CUDA(cudaMemcpyAsync(group_start_dev, cursor, (uint64_t)n_groups * 4, cudaMemcpyDeviceToDevice, st));
        IBP_CUDA(cudaMemcpyAsync(group_start_dev + n_groups, &last, 4, cudaMemcpyHostToDevice, st));
        IBP_CUDA(cudaStreamSynchronize(st));      // `last` lives on this stack frame
    }
    ibp_cluster_scatter<<<grid, 256, 0, st>>>(row_group_dev, n_rows, cursor, order_dev);
    IBP_CUDA(cudaGetLastError());
    cudaFreeAsync(hist, st); cudaFreeAsync(cursor, st);
    return IBP_OK;
}
