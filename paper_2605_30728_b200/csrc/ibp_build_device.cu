// ibp_build_device.cu -- the GPU-side compressor of libibp.so (sm_100a): ibp_build_device.
//
// The paper's compressor runs on the GPU over zero-copy tensors (PAPER.md:227-229 preprocessing "performed on the GPU", P:239
// "tensors are partitioned among GPU warps", Fig. 3 = P:243-299 getCompressSize / compress) and writes the
// compressed rows in place into CPU memory.  Here:
//   ibp_mask_kernel     S0   per group: AND/OR reduction (strict, T = N) or bit-sliced per-bit counters (thresholded)
//                            held in registers -- each lane owns W 32-bit words of the row, plane j of a word holds bit j of
//                            its 32 running counters -- then Mask/Bitval by a bit-sliced comparison with T and N - T.
//                            Groups with many rows are cut into slices (one warp each) whose accumulators are merged by
//                            ibp_mask_merge_kernel; no atomics, results do not depend on the launch shape.
//   ibp_pack_kernel     S0'  strict: a warp packs runs of rows of one group; per 32-bit word a 5-stage parallel-suffix bit
//                            compress (Hacker's Delight 7-4) with move masks hoisted per group, OR-ed into a per-warp shared-
//                            memory row image at the word's bit offset (exclusive scan of the kept-bit counts),
//                            then written to the store (host memory, over PCIe) with wide stores.
//   ibp_size_kernel     S0'  thresholded: participation of every 4-byte chunk, bitsSaved, size or raw (Fig. 3 lines 1-19)
//   ibp_scan_*               exclusive scan of the row sizes -> row offsets (16-byte units)
//   ibp_pack_t_kernel   S0'  thresholded: [participation bits][payloads] per row (Fig. 3 lines 21-33), raw rows copied
// The result is bit-identical to ibp_build's (same Mask/Bitval/k, same packed bytes): both are checked against the oracle.
#include <algorithm>
#include <chrono>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <vector>

#include "ibp_devutil.cuh"

namespace {

__device__ __forceinline__ uint32_t xor3(uint32_t a, uint32_t b, uint32_t c) {
    uint32_t d;
    asm("lop3.b32 %0, %1, %2, %3, 0x96;" : "=r"(d) : "r"(a), "r"(b), "r"(c));
    return d;
}
__device__ __forceinline__ uint32_t maj3(uint32_t a, uint32_t b, uint32_t c) {
    uint32_t d;
    asm("lop3.b32 %0, %1, %2, %3, 0xE8;" : "=r"(d) : "r"(a), "r"(b), "r"(c));
    return d;
}

// bit b of the result = 1 iff the bit-sliced counter b (planes pl[0..NP), LSB plane first) is >= T
template <int NP>
__device__ __forceinline__ uint32_t sliced_ge(const uint32_t* pl, uint64_t T) {
    if (NP < 64 && (T >> NP)) return 0u;
    uint32_t gt = 0, eq = 0xFFFFFFFFu;
#pragma unroll
    for (int j = NP - 1; j >= 0; --j) {
        const uint32_t tj = ((T >> j) & 1ull) ? 0xFFFFFFFFu : 0u;
        gt |= eq & pl[j] & ~tj;
        eq &= ~(pl[j] ^ tj);
    }
    return gt | eq;
}
// ... is <= L
template <int NP>
__device__ __forceinline__ uint32_t sliced_le(const uint32_t* pl, uint64_t L) {
    if (NP < 64 && (L >> NP)) return 0xFFFFFFFFu;
    uint32_t lt = 0, eq = 0xFFFFFFFFu;
#pragma unroll
    for (int j = NP - 1; j >= 0; --j) {
        const uint32_t tj = ((L >> j) & 1ull) ? 0xFFFFFFFFu : 0u;
        lt |= eq & ~pl[j] & tj;
        eq &= ~(pl[j] ^ tj);
    }
    return lt | eq;
}

struct BuildParams {
    const uint32_t* rows;
    uint64_t n_rows, n_groups;
    uint32_t nw, n_pass;
    uint32_t group_param, group_shift, strided;
    uint32_t ns;                 // slices per group
    uint64_t rows_per_slice;
    uint32_t thr_num, thr_den;
    uint32_t* meta;              // per group: Mask words, Bitval words
    uint32_t* kbits;             // per group: popcount(~Mask)
    uint32_t* scratch;           // ns > 1: per (group, slice) accumulators
};

__device__ __forceinline__ uint64_t group_count(const BuildParams& P, uint64_t g) {
    if (P.strided) return (P.n_rows - g + P.group_param - 1) / P.group_param;
    const uint64_t first = g * P.group_param;
    return min((uint64_t)P.group_param, P.n_rows - first);
}
__device__ __forceinline__ uint64_t group_row(const BuildParams& P, uint64_t g, uint64_t j) {
    return P.strided ? j * P.group_param + g : g * P.group_param + j;
}
__device__ __forceinline__ uint64_t threshold_of(uint64_t N, uint32_t num, uint32_t den) { return (N * num + den - 1) / den; }

// ------------------------------------------------------------------------------------------------ S0: masks
// One warp per (group, slice).  TM = thresholded (bit-sliced counters, NP planes: a slice has at most 2^NP - 1 rows).
template <int W, bool TM, int NP>
__global__ void __launch_bounds__(256) ibp_mask_kernel(const BuildParams P) {
    const int lane = threadIdx.x & 31, wpc = blockDim.x >> 5;
    const uint64_t n_units = P.n_groups * P.ns;
    for (uint64_t u = (uint64_t)blockIdx.x * wpc + (threadIdx.x >> 5); u < n_units; u += (uint64_t)gridDim.x * wpc) {
        const uint64_t g = u / P.ns;
        const uint32_t s = (uint32_t)(u - g * P.ns);
        const uint64_t N = group_count(P, g);
        const uint64_t j0 = min(N, (uint64_t)s * P.rows_per_slice), j1 = min(N, j0 + P.rows_per_slice);
        uint32_t k_total = 0;
        for (uint32_t pass = 0; pass < P.n_pass; ++pass) {
            const uint32_t w0 = (pass * 32u + lane) * W;
            const bool active = w0 < P.nw;
            uint32_t a[W], o[W], pl[TM ? NP : 1][W];
#pragma unroll
            for (int q = 0; q < W; ++q) {
                a[q] = 0xFFFFFFFFu; o[q] = 0;
#pragma unroll
                for (int j = 0; j < (TM ? NP : 1); ++j) pl[j][q] = 0;
            }
            if (active) {
                const uint32_t* base = P.rows + w0;
                uint64_t j = j0;
                for (; j + 4 <= j1; j += 4) {
                    uint32_t x0[W], x1[W], x2[W], x3[W];
                    VecIO<W>::ld(base + group_row(P, g, j) * P.nw, x0);
                    VecIO<W>::ld(base + group_row(P, g, j + 1) * P.nw, x1);
                    VecIO<W>::ld(base + group_row(P, g, j + 2) * P.nw, x2);
                    VecIO<W>::ld(base + group_row(P, g, j + 3) * P.nw, x3);
#pragma unroll
                    for (int q = 0; q < W; ++q) {
                        if (!TM) {
                            a[q] &= x0[q] & x1[q] & x2[q] & x3[q];
                            o[q] |= x0[q] | x1[q] | x2[q] | x3[q];
                        } else {
                            // carry-save adders: four rows enter plane 0, two carries enter plane 1, one carry ripples on
                            const uint32_t s1 = xor3(pl[0][q], x0[q], x1[q]), c1 = maj3(pl[0][q], x0[q], x1[q]);
                            const uint32_t s2 = xor3(s1, x2[q], x3[q]), c2 = maj3(s1, x2[q], x3[q]);
                            pl[0][q] = s2;
                            uint32_t c = maj3(pl[1][q], c1, c2);
                            pl[1][q] = xor3(pl[1][q], c1, c2);
#pragma unroll
                            for (int p = 2; p < NP; ++p) { const uint32_t t = pl[p][q]; pl[p][q] = t ^ c; c &= t; }
                        }
                    }
                }
                for (; j < j1; ++j) {
                    uint32_t x[W];
                    VecIO<W>::ld(base + group_row(P, g, j) * P.nw, x);
#pragma unroll
                    for (int q = 0; q < W; ++q) {
                        if (!TM) { a[q] &= x[q]; o[q] |= x[q]; }
                        else {
                            uint32_t c = x[q];
#pragma unroll
                            for (int p = 0; p < NP; ++p) { const uint32_t t = pl[p][q]; pl[p][q] = t ^ c; c &= t; }
                        }
                    }
                }
            }
            if (P.ns == 1) {
                uint32_t mk[W], bv[W];
                const uint64_t T = TM ? threshold_of(N, P.thr_num, P.thr_den) : 0;
#pragma unroll
                for (int q = 0; q < W; ++q) {
                    if (!TM) {
                        mk[q] = ~(a[q] ^ o[q]);
                        bv[q] = a[q] & mk[q];
                    } else {
                        uint32_t col[NP];
#pragma unroll
                        for (int p = 0; p < NP; ++p) col[p] = pl[p][q];
                        const uint32_t ge = sliced_ge<NP>(col, T), le = sliced_le<NP>(col, N - T);
                        mk[q] = ge | le;
                        bv[q] = ge;
                    }
                    if (active) k_total += __popc(~mk[q]);
                }
                if (active) {
                    uint32_t* gm = P.meta + g * 2ull * P.nw;
                    VecIO<W>::st_keep((uint8_t*)(gm + w0), mk);
                    VecIO<W>::st_keep((uint8_t*)(gm + P.nw + w0), bv);
                }
            } else if (active) {
                if (!TM) {
                    VecIO<W>::st_keep((uint8_t*)(P.scratch + (u * 2ull) * P.nw + w0), a);
                    VecIO<W>::st_keep((uint8_t*)(P.scratch + (u * 2ull + 1) * P.nw + w0), o);
                } else {
#pragma unroll
                    for (int p = 0; p < NP; ++p) {
                        uint32_t col[W];
#pragma unroll
                        for (int q = 0; q < W; ++q) col[q] = pl[p][q];
                        VecIO<W>::st_keep((uint8_t*)(P.scratch + (u * (uint64_t)NP + p) * P.nw + w0), col);
                    }
                }
            }
        }
        if (P.ns == 1) {
#pragma unroll
            for (int d = 16; d; d >>= 1) k_total += __shfl_xor_sync(0xFFFFFFFFu, k_total, d);
            if (lane == 0) P.kbits[g] = k_total;
        }
    }
}

// Merge of the slices of a group: one thread per (group, word).  kbits must be zero on entry.
template <bool TM, int NP>
__global__ void ibp_mask_merge_kernel(const BuildParams P) {
    const uint64_t i = blockIdx.x * (uint64_t)blockDim.x + threadIdx.x;
    if (i >= P.n_groups * P.nw) return;
    const uint64_t g = i / P.nw;
    const uint32_t w = (uint32_t)(i - g * P.nw);
    const uint64_t N = group_count(P, g);
    uint32_t mk, bv;
    if (!TM) {
        uint32_t a = 0xFFFFFFFFu, o = 0;
        for (uint32_t s = 0; s < P.ns; ++s) {
            const uint64_t u = g * P.ns + s;
            a &= P.scratch[(u * 2ull) * P.nw + w];
            o |= P.scratch[(u * 2ull + 1) * P.nw + w];
        }
        mk = ~(a ^ o);
        bv = a & mk;
    } else {
        uint32_t acc[32];
#pragma unroll
        for (int p = 0; p < 32; ++p) acc[p] = 0;
        for (uint32_t s = 0; s < P.ns; ++s) {
            const uint64_t u = g * P.ns + s;
            uint32_t c = 0;
#pragma unroll
            for (int p = 0; p < NP; ++p) {
                const uint32_t q = P.scratch[(u * (uint64_t)NP + p) * P.nw + w];
                const uint32_t t = acc[p];
                acc[p] = xor3(t, q, c);
                c = maj3(t, q, c);
            }
#pragma unroll
            for (int p = NP; p < 32; ++p) { const uint32_t t = acc[p]; acc[p] = t ^ c; c &= t; }
        }
        const uint64_t T = threshold_of(N, P.thr_num, P.thr_den);
        const uint32_t ge = sliced_ge<32>(acc, T), le = sliced_le<32>(acc, N - T);
        mk = ge | le;
        bv = ge;
    }
    P.meta[g * 2ull * P.nw + w] = mk;
    P.meta[g * 2ull * P.nw + P.nw + w] = bv;
    atomicAdd(&P.kbits[g], (uint32_t)__popc(~mk));
}

// ------------------------------------------------------------------------------------------------ S0': pack
// the five move masks of the parallel-suffix compress/expand for the kept positions nv (Hacker's Delight 7-4)
__device__ __forceinline__ void suffix_masks(uint32_t nv, uint32_t mv[5]) {
    uint32_t m = nv, mk = ~nv << 1;
#pragma unroll
    for (int i = 0; i < 5; ++i) {
        uint32_t mp = mk ^ (mk << 1);
        mp ^= mp << 2;
        mp ^= mp << 4;
        mp ^= mp << 8;
        mp ^= mp << 16;
        const uint32_t v = mp & m;
        mv[i] = v;
        m = (m ^ v) | (v >> (1 << i));
        mk &= ~mp;
    }
}
// the bits of x at the set positions of nv, moved to the low end in order ("the matching bits are removed")
__device__ __forceinline__ uint32_t compress_bits(uint32_t x, uint32_t nv, const uint32_t mv[5]) {
    x &= nv;
#pragma unroll
    for (int i = 0; i < 5; ++i) {
        const uint32_t t = x & mv[i];
        x = (x ^ t) | (t >> (1 << i));
    }
    return x;
}
// OR the low k bits of c into the LSB-first bit image `img` (shared memory) at bit offset `bit` (P:292-295 insertBits)
__device__ __forceinline__ void insert_bits(uint32_t* img, uint32_t bit, uint32_t c, uint32_t k) {
    if (!k) return;
    const uint32_t wq = bit >> 5, sh = bit & 31u;
    atomicOr(img + wq, c << sh);
    if (sh + k > 32u) atomicOr(img + wq + 1, c >> (32u - sh));
}

struct PackParams {
    const uint32_t* rows;
    const uint32_t* meta;
    const IbpGroupEntry* gtab;
    uint8_t* store;              // device-visible address of the packed store
    uint64_t n_rows, n_units, row_stride_strided;
    uint32_t nw, n_pass, group_param, group_shift, strided, align_bytes;
    uint32_t slot_bytes;         // per-warp shared-memory row image
    uint32_t rows_per_unit;      // bulk variant: consecutive rows packed into one image and stored with one bulk copy
    // thresholded
    const uint32_t* row_off;     // 16-byte units
    uint32_t* row_off_out;       // size kernel: units per row (scanned afterwards)
    uint32_t* row_flag;
    unsigned long long* sum_size;
};

// warp-cooperative copy of nbytes from the shared row image to the store; `align` = guaranteed alignment of dst and nbytes
__device__ __forceinline__ void image_to_store(const uint8_t* img, uint8_t* dst, uint32_t nbytes, uint32_t align, int lane) {
    if (align >= 16) {
        for (uint32_t v = lane; v < nbytes / 16; v += 32) ((uint4*)dst)[v] = ((const uint4*)img)[v];
    } else if (align >= 4) {
        for (uint32_t v = lane; v < nbytes / 4; v += 32) ((uint32_t*)dst)[v] = ((const uint32_t*)img)[v];
    } else {
        for (uint32_t v = lane; v < nbytes; v += 32) dst[v] = img[v];
    }
}

// Strict mode.  Unit = 16 consecutive rows (blocked) or 16 matrix rows of one column tile (strided): the metadata, the bit
// offsets and the compress masks of the group stay in registers while consecutive rows share the group (single-pass rows).
template <int W>
__global__ void __launch_bounds__(256) ibp_pack_kernel(const PackParams P) {
    extern __shared__ __align__(16) uint8_t smem[];
    const int lane = threadIdx.x & 31, wib = threadIdx.x >> 5, wpc = blockDim.x >> 5;
    uint32_t* img = (uint32_t*)(smem + (size_t)wib * P.slot_bytes);
    const uint64_t S = P.group_param;
    uint64_t prep_g = ~0ull;
    uint32_t prep_pass = ~0u;
    uint32_t m[W], ex[W], kq[W], mv[W][5], tot = 0;
    IbpGroupEntry e{0, 0, 0};

    auto prepare = [&](uint64_t g, uint32_t pass) {
        const uint32_t w0 = (pass * 32u + lane) * W;
        if (w0 < P.nw) VecIO<W>::ld(P.meta + g * 2ull * P.nw + w0, m);
        else {
#pragma unroll
            for (int q = 0; q < W; ++q) m[q] = 0xFFFFFFFFu;
        }
        uint32_t t = 0;
#pragma unroll
        for (int q = 0; q < W; ++q) { kq[q] = __popc(~m[q]); ex[q] = t; t += kq[q]; }
        const uint32_t incl = warp_inclusive_scan(t, lane);
#pragma unroll
        for (int q = 0; q < W; ++q) {
            ex[q] += incl - t;
            if (q > 0 && m[q] == m[q - 1]) {
#pragma unroll
                for (int i = 0; i < 5; ++i) mv[q][i] = mv[q - 1][i];
            } else {
                suffix_masks(~m[q], mv[q]);
            }
        }
        tot = __shfl_sync(0xFFFFFFFFu, incl, 31);
        if (g != prep_g) e = P.gtab[g];
        prep_g = g; prep_pass = pass;
    };

    for (uint64_t u = (uint64_t)blockIdx.x * wpc + wib; u < P.n_units; u += (uint64_t)gridDim.x * wpc) {
        uint64_t id0, id_step;
        uint32_t nrows;
        if (!P.strided) {
            id0 = u * 16; id_step = 1;
            nrows = (uint32_t)min((uint64_t)16, P.n_rows - id0);
        } else {
            const uint64_t rb = u / S, t = u - rb * S;
            id0 = rb * 16 * S + t; id_step = S;
            const uint64_t n_mrows_t = t < P.n_rows ? (P.n_rows - t + S - 1) / S : 0;   // rows of tile t
            nrows = rb * 16 < n_mrows_t ? (uint32_t)min((uint64_t)16, n_mrows_t - rb * 16) : 0u;
        }
        for (uint32_t j = 0; j < nrows; ++j) {
            const uint64_t id = id0 + j * id_step;
            const uint64_t g = P.strided ? id % S : group_of_u(P.group_param, P.group_shift, id);
            // zero the row image (the previous row's copy-out is complete: __syncwarp below)
            for (uint32_t v = lane; v < P.slot_bytes / 16; v += 32) ((uint4*)img)[v] = make_uint4(0, 0, 0, 0);
            __syncwarp();
            uint32_t carry = 0;
            for (uint32_t pass = 0; pass < P.n_pass; ++pass) {
                if (g != prep_g || pass != prep_pass) prepare(g, pass);
                const uint32_t w0 = (pass * 32u + lane) * W;
                if (w0 < P.nw) {
                    uint32_t x[W];
                    VecIO<W>::ld(P.rows + id * P.nw + w0, x);
#pragma unroll
                    for (int q = 0; q < W; ++q) insert_bits(img, carry + ex[q], compress_bits(x[q], ~m[q], mv[q]), kq[q]);
                }
                carry += tot;
            }
            __syncwarp();
            if (e.stride) {
                const uint64_t off = P.strided ? (id / S) * P.row_stride_strided + e.base : e.base + (id - g * S) * (uint64_t)e.stride;
                image_to_store((const uint8_t*)img, P.store + off, e.stride, P.align_bytes, lane);
            }
            __syncwarp();
        }
    }
}

// Strict mode, blocked groups, A >= 16: the packed rows of consecutive rows of one group are contiguous in the store, so a warp
// packs a whole unit (rows_per_unit rows) into one shared-memory image and hands it to the bulk-copy engine as ONE
// cp.async.bulk shared -> global store per run of rows of a group (PCIe sees long contiguous writes instead of one short
// write per lane); two images per warp, so the store of unit i overlaps the packing of unit i+1.
template <int W>
__global__ void __launch_bounds__(256) ibp_pack_bulk_kernel(const PackParams P) {
    extern __shared__ __align__(128) uint8_t smem[];
    const int lane = threadIdx.x & 31, wib = threadIdx.x >> 5, wpc = blockDim.x >> 5;
    uint8_t* img2 = smem + (size_t)wib * 2 * P.slot_bytes;
    const uint64_t S = P.group_param;
    uint64_t prep_g = ~0ull;
    uint32_t prep_pass = ~0u;
    uint32_t m[W], ex[W], kq[W], mv[W][5], tot = 0;
    IbpGroupEntry e{0, 0, 0};

    auto prepare = [&](uint64_t g, uint32_t pass) {
        const uint32_t w0 = (pass * 32u + lane) * W;
        if (w0 < P.nw) VecIO<W>::ld(P.meta + g * 2ull * P.nw + w0, m);
        else {
#pragma unroll
            for (int q = 0; q < W; ++q) m[q] = 0xFFFFFFFFu;
        }
        uint32_t t = 0;
#pragma unroll
        for (int q = 0; q < W; ++q) { kq[q] = __popc(~m[q]); ex[q] = t; t += kq[q]; }
        const uint32_t incl = warp_inclusive_scan(t, lane);
#pragma unroll
        for (int q = 0; q < W; ++q) {
            ex[q] += incl - t;
            if (q > 0 && m[q] == m[q - 1]) {
#pragma unroll
                for (int i = 0; i < 5; ++i) mv[q][i] = mv[q - 1][i];
            } else {
                suffix_masks(~m[q], mv[q]);
            }
        }
        tot = __shfl_sync(0xFFFFFFFFu, incl, 31);
        if (g != prep_g) e = P.gtab[g];
        prep_g = g; prep_pass = pass;
    };
    // shared -> global bulk store of [src, src+bytes) (generic-proxy writes made visible to the async proxy first)
    auto flush = [&](const uint8_t* src, uint64_t dst_off, uint32_t bytes) {
        if (!bytes) return;
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        __syncwarp();
        if (lane == 0)
            asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;"
                         ::"l"(P.store + dst_off), "r"((uint32_t)__cvta_generic_to_shared(src)), "r"(bytes) : "memory");
    };

    uint32_t it = 0;
    for (uint64_t u = (uint64_t)blockIdx.x * wpc + wib; u < P.n_units; u += (uint64_t)gridDim.x * wpc, ++it) {
        const uint64_t id0 = u * P.rows_per_unit;
        const uint32_t nrows = (uint32_t)min((uint64_t)P.rows_per_unit, P.n_rows - id0);
        uint8_t* img = img2 + (size_t)(it & 1u) * P.slot_bytes;
        if (lane == 0) asm volatile("cp.async.bulk.wait_group.read 1;" ::: "memory");   // the store that last used this image has read it
        __syncwarp();
        for (uint32_t v = lane; v < P.slot_bytes / 16; v += 32) ((uint4*)img)[v] = make_uint4(0, 0, 0, 0);
        __syncwarp();
        uint32_t pos = 0, run_start = 0;
        uint64_t run_dst = 0, run_g = ~0ull;
        for (uint32_t j = 0; j < nrows; ++j) {
            const uint64_t id = id0 + j;
            const uint64_t g = group_of_u(P.group_param, P.group_shift, id);
            uint32_t carry = 0;
            for (uint32_t pass = 0; pass < P.n_pass; ++pass) {
                if (g != prep_g || pass != prep_pass) prepare(g, pass);
                if (pass == 0 && g != run_g) {                       // a new run of rows of one group starts here
                    flush(img + run_start, run_dst, pos - run_start);
                    run_start = pos; run_g = g;
                    run_dst = e.base + (id - g * S) * (uint64_t)e.stride;
                }
                const uint32_t w0 = (pass * 32u + lane) * W;
                if (w0 < P.nw) {
                    uint32_t x[W];
                    VecIO<W>::ld(P.rows + id * P.nw + w0, x);
#pragma unroll
                    for (int q = 0; q < W; ++q) insert_bits((uint32_t*)(img + pos), carry + ex[q], compress_bits(x[q], ~m[q], mv[q]), kq[q]);
                }
                carry += tot;
            }
            pos += e.stride;
        }
        flush(img + run_start, run_dst, pos - run_start);
        if (lane == 0) asm volatile("cp.async.bulk.commit_group;" ::: "memory");
    }
    if (lane == 0) asm volatile("cp.async.bulk.wait_group 0;" ::: "memory");
    __syncwarp();
}

// Thresholded mode, pass 1 (Fig. 3 lines 1-19 = P:244-271): unit = 32 consecutive rows (one word of the per-row bitmask).
template <int W>
__global__ void __launch_bounds__(256) ibp_size_kernel(const PackParams P) {
    const int lane = threadIdx.x & 31, wpc = blockDim.x >> 5;
    const uint64_t S = P.group_param;
    unsigned long long local_sum = 0;
    for (uint64_t u = (uint64_t)blockIdx.x * wpc + (threadIdx.x >> 5); u < P.n_units; u += (uint64_t)gridDim.x * wpc) {
        const uint64_t id0 = u * 32;
        const uint32_t nrows = (uint32_t)min((uint64_t)32, P.n_rows - id0);
        uint32_t flags = 0;
        for (uint32_t j = 0; j < nrows; ++j) {
            const uint64_t id = id0 + j;
            const uint64_t g = P.strided ? id % S : group_of_u(P.group_param, P.group_shift, id);
            uint32_t saved = 0;
            for (uint32_t pass = 0; pass < P.n_pass; ++pass) {
                const uint32_t w0 = (pass * 32u + lane) * W;
                if (w0 < P.nw) {
                    uint32_t m[W], b[W], x[W];
                    VecIO<W>::ld(P.meta + g * 2ull * P.nw + w0, m);
                    VecIO<W>::ld(P.meta + g * 2ull * P.nw + P.nw + w0, b);
                    VecIO<W>::ld(P.rows + id * P.nw + w0, x);
#pragma unroll
                    for (int q = 0; q < W; ++q) saved += ((x[q] & m[q]) == b[q]) ? __popc(m[q]) : 0u;
                }
            }
#pragma unroll
            for (int d = 16; d; d >>= 1) saved += __shfl_xor_sync(0xFFFFFFFFu, saved, d);
            const int64_t net = (int64_t)saved - (int64_t)P.nw;                                          // minus participation bits
            const uint32_t bytes_saved = net >= 8 ? (uint32_t)(net / 8) : 0u;                            // floor
            const uint32_t size = 4u * P.nw - bytes_saved;
            if (bytes_saved) flags |= 1u << j;                                                           // else stored raw
            if (lane == 0) {
                P.row_off_out[id] = (size + P.align_bytes - 1) / P.align_bytes * (P.align_bytes / 16);
                local_sum += size;
            }
        }
        if (lane == 0) P.row_flag[u] = flags;
    }
    if (lane == 0 && local_sum) atomicAdd(P.sum_size, local_sum);
}

// Thresholded mode, pass 2 (Fig. 3 lines 21-33 = P:275-298).  Rows lie in id order in the store, so a warp packs a unit of
// rows_per_unit consecutive rows into one shared-memory image (row r at 16*(row_off[r] - row_off[first])) and stores the
// whole unit with one cp.async.bulk shared -> global copy; two images per warp overlap the store with the next unit.
template <int W>
__global__ void __launch_bounds__(256) ibp_pack_t_kernel(const PackParams P) {
    extern __shared__ __align__(128) uint8_t smem[];
    const int lane = threadIdx.x & 31, wib = threadIdx.x >> 5, wpc = blockDim.x >> 5;
    uint8_t* img2 = smem + (size_t)wib * 2 * P.slot_bytes;
    const uint64_t S = P.group_param;
    uint32_t it = 0;
    for (uint64_t u = (uint64_t)blockIdx.x * wpc + wib; u < P.n_units; u += (uint64_t)gridDim.x * wpc, ++it) {
        const uint64_t id0 = u * P.rows_per_unit;
        const uint32_t nrows = (uint32_t)min((uint64_t)P.rows_per_unit, P.n_rows - id0);
        uint8_t* ubuf = img2 + (size_t)(it & 1u) * P.slot_bytes;
        if (lane == 0) asm volatile("cp.async.bulk.wait_group.read 1;" ::: "memory");
        __syncwarp();
        const uint32_t off0 = P.row_off[id0], off_end = P.row_off[id0 + nrows];
        const uint32_t unit_bytes = (off_end - off0) * 16u;
        for (uint32_t v = lane; v < unit_bytes / 16 + 1; v += 32) ((uint4*)ubuf)[v] = make_uint4(0, 0, 0, 0);
        __syncwarp();
        for (uint32_t j = 0; j < nrows; ++j) {
            const uint64_t id = id0 + j;
            const uint64_t g = P.strided ? id % S : group_of_u(P.group_param, P.group_shift, id);
            uint32_t* img = (uint32_t*)(ubuf + 16ull * (P.row_off[id] - off0));
            const bool compressed = (P.row_flag[id >> 5] >> (id & 31u)) & 1u;
            if (!compressed) {                                           // kept raw
                for (uint32_t w = lane; w < P.nw; w += 32) img[w] = P.rows[id * P.nw + w];
                continue;
            }
            uint32_t carry = P.nw;                                       // payloads follow the participation bits (R8)
            for (uint32_t pass = 0; pass < P.n_pass; ++pass) {
                const uint32_t w0 = (pass * 32u + lane) * W;
                const bool active = w0 < P.nw;
                uint32_t m[W], b[W], x[W], kq[W], part = 0, t = 0;
                if (active) {
                    VecIO<W>::ld(P.meta + g * 2ull * P.nw + w0, m);
                    VecIO<W>::ld(P.meta + g * 2ull * P.nw + P.nw + w0, b);
                    VecIO<W>::ld(P.rows + id * P.nw + w0, x);
                }
#pragma unroll
                for (int q = 0; q < W; ++q) {
                    const bool p = active && (x[q] & m[q]) == b[q];
                    part |= (uint32_t)p << q;
                    kq[q] = active ? (p ? __popc(~m[q]) : 32u) : 0u;
                    t += kq[q];
                }
                const uint32_t incl = warp_inclusive_scan(t, lane);
                uint32_t bit = carry + incl - t;
                if (active) {
                    if (part) atomicOr(img + (w0 >> 5), part << (w0 & 31u));                 // W divides 32: one word
#pragma unroll
                    for (int q = 0; q < W; ++q) {
                        uint32_t c = x[q];
                        if ((part >> q) & 1u) { uint32_t mv[5]; suffix_masks(~m[q], mv); c = compress_bits(x[q], ~m[q], mv); }
                        if (kq[q] == 32u) {                                                   // two plain halves (no shift by 32)
                            const uint32_t wq = bit >> 5, sh = bit & 31u;
                            atomicOr(img + wq, c << sh);
                            if (sh) atomicOr(img + wq + 1, c >> (32u - sh));
                        } else {
                            insert_bits(img, bit, c, kq[q]);
                        }
                        bit += kq[q];
                    }
                }
                carry += __shfl_sync(0xFFFFFFFFu, incl, 31);
            }
        }
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        __syncwarp();
        if (lane == 0) {
            if (unit_bytes)
                asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;"
                             ::"l"(P.store + 16ull * off0), "r"((uint32_t)__cvta_generic_to_shared(ubuf)), "r"(unit_bytes) : "memory");
            asm volatile("cp.async.bulk.commit_group;" ::: "memory");
        }
    }
    if (lane == 0) asm volatile("cp.async.bulk.wait_group 0;" ::: "memory");
    __syncwarp();
}

// Online append, slot layout: one warp per NEW row.  The row is compressed under the existing Mask/Bitval of
// its group -- getCompressSize (Fig. 3 lines 1-19) and compress (lines 21-33) in one visit -- into a shared-memory image and
// written to its own slot of the host store; the size byte and the bit of the per-row bitmask are set in GPU memory.
struct AppendParams {
    const uint32_t* rows;        // n_new rows
    const uint32_t* meta;
    uint8_t* store;
    uint8_t* row_size;
    uint32_t* row_flag;
    unsigned long long* sums;    // [0] += byte-aligned sizes, [1] += stored bytes incl. padding, [2] += rows kept raw
    uint64_t first_id, n_new;
    uint32_t nw, n_pass, group_param, group_shift, strided, align_bytes, slot_bytes, img_bytes;
};

template <int W>
__global__ void __launch_bounds__(256) ibp_append_kernel(const AppendParams P) {
    extern __shared__ __align__(128) uint8_t smem[];
    const int lane = threadIdx.x & 31, wib = threadIdx.x >> 5, wpc = blockDim.x >> 5;
    uint32_t* img = (uint32_t*)(smem + (size_t)wib * P.img_bytes);
    const uint64_t S = P.group_param;
    for (uint64_t j = (uint64_t)blockIdx.x * wpc + wib; j < P.n_new; j += (uint64_t)gridDim.x * wpc) {
        const uint64_t id = P.first_id + j;
        const uint64_t g = P.strided ? id % S : group_of_u(P.group_param, P.group_shift, id);
        const uint32_t* x_row = P.rows + j * P.nw;
        const uint32_t* gm = P.meta + g * 2ull * P.nw;
        // ---- size
        uint32_t saved = 0;
        for (uint32_t pass = 0; pass < P.n_pass; ++pass) {
            const uint32_t w0 = (pass * 32u + lane) * W;
            if (w0 < P.nw) {
                uint32_t m[W], b[W], x[W];
                VecIO<W>::ld(gm + w0, m);
                VecIO<W>::ld(gm + P.nw + w0, b);
                VecIO<W>::ld(x_row + w0, x);
#pragma unroll
                for (int q = 0; q < W; ++q) saved += ((x[q] & m[q]) == b[q]) ? __popc(m[q]) : 0u;
            }
        }
#pragma unroll
        for (int d = 16; d; d >>= 1) saved += __shfl_xor_sync(0xFFFFFFFFu, saved, d);
        const int64_t net = (int64_t)saved - (int64_t)P.nw;                       // minus the participation bits
        const uint32_t bytes_saved = net >= 8 ? (uint32_t)(net / 8) : 0u;         // floor
        const uint32_t size = 4u * P.nw - bytes_saved;
        const bool compressed = bytes_saved != 0;                                  // else stored raw
        const uint32_t stored = (size + P.align_bytes - 1) / P.align_bytes * P.align_bytes;
        // ---- image
        for (uint32_t v = lane; v < stored / 16 + 1; v += 32) ((uint4*)img)[v] = make_uint4(0, 0, 0, 0);
        __syncwarp();
        if (!compressed) {
            for (uint32_t w = lane; w < P.nw; w += 32) img[w] = x_row[w];
        } else {
            uint32_t carry = P.nw;                                                // payloads follow the participation bits (R8)
            for (uint32_t pass = 0; pass < P.n_pass; ++pass) {
                const uint32_t w0 = (pass * 32u + lane) * W;
                const bool active = w0 < P.nw;
                uint32_t m[W], b[W], x[W], kq[W], part = 0, t = 0;
                if (active) {
                    VecIO<W>::ld(gm + w0, m);
                    VecIO<W>::ld(gm + P.nw + w0, b);
                    VecIO<W>::ld(x_row + w0, x);
                }
#pragma unroll
                for (int q = 0; q < W; ++q) {
                    const bool pq = active && (x[q] & m[q]) == b[q];
                    part |= (uint32_t)pq << q;
                    kq[q] = active ? (pq ? __popc(~m[q]) : 32u) : 0u;
                    t += kq[q];
                }
                const uint32_t incl = warp_inclusive_scan(t, lane);
                uint32_t bit = carry + incl - t;
                if (active) {
                    if (part) atomicOr(img + (w0 >> 5), part << (w0 & 31u));       // W divides 32: one word
#pragma unroll
                    for (int q = 0; q < W; ++q) {
                        uint32_t c = x[q];
                        if ((part >> q) & 1u) { uint32_t mv[5]; suffix_masks(~m[q], mv); c = compress_bits(x[q], ~m[q], mv); }
                        if (kq[q] == 32u) {
                            const uint32_t wq = bit >> 5, sh = bit & 31u;
                            atomicOr(img + wq, c << sh);
                            if (sh) atomicOr(img + wq + 1, c >> (32u - sh));
                        } else {
                            insert_bits(img, bit, c, kq[q]);
                        }
                        bit += kq[q];
                    }
                }
                carry += __shfl_sync(0xFFFFFFFFu, incl, 31);
            }
        }
        __syncwarp();
        // the whole slot is rewritten (zeros beyond the row), so a slot can be reused
        uint8_t* dst = P.store + id * (uint64_t)P.slot_bytes;
        for (uint32_t v = lane; v < P.slot_bytes / 16; v += 32) {
            const uint4 t4 = v < stored / 16 ? ((const uint4*)img)[v] : make_uint4(0, 0, 0, 0);
            ((uint4*)dst)[v] = t4;
        }
        if (lane == 0) {
            P.row_size[id] = (uint8_t)(stored / 16);
            if (compressed) atomicOr(P.row_flag + (id >> 5), 1u << (id & 31u));
            else atomicAnd(P.row_flag + (id >> 5), ~(1u << (id & 31u)));
            atomicAdd(P.sums + 0, (unsigned long long)size);
            atomicAdd(P.sums + 1, (unsigned long long)stored);
            if (!compressed) atomicAdd(P.sums + 2, 1ull);
        }
        __syncwarp();
    }
}

// Slot layout in ibp_build_device: the size kernel's per-row units become the size bytes, and the offsets the pack kernel
// walks are the fixed shifts r * slot16 (a temporary array: the handle keeps no offsets in this layout).
__global__ void ibp_slot_layout_kernel(uint32_t* __restrict__ units_to_off, uint64_t n, uint32_t slot16, uint8_t* __restrict__ row_size,
                                       unsigned long long* __restrict__ stored_units) {
    unsigned long long local = 0;
    for (uint64_t r = blockIdx.x * (uint64_t)blockDim.x + threadIdx.x; r <= n; r += (uint64_t)gridDim.x * blockDim.x) {
        if (r < n) { const uint32_t u = units_to_off[r]; row_size[r] = (uint8_t)u; local += u; }
        units_to_off[r] = (uint32_t)(r * slot16);
    }
    if (local) atomicAdd(stored_units, local);
}

// ------------------------------------------------------------------------------------------------ exclusive scan (u32 -> u32)
// 4096 items per block of 1024 threads; totals in 64 bits so that an overflow of the 32-bit offsets is detected.
__global__ void __launch_bounds__(1024) ibp_scan_sums(const uint32_t* __restrict__ in, uint64_t n, unsigned long long* __restrict__ bsum) {
    __shared__ unsigned long long ws[32];
    const uint64_t i0 = (uint64_t)blockIdx.x * 4096 + threadIdx.x * 4ull;
    unsigned long long s = 0;
#pragma unroll
    for (int k = 0; k < 4; ++k) if (i0 + k < n) s += in[i0 + k];
#pragma unroll
    for (int d = 16; d; d >>= 1) s += __shfl_xor_sync(0xFFFFFFFFu, s, d);
    if ((threadIdx.x & 31) == 0) ws[threadIdx.x >> 5] = s;
    __syncthreads();
    if (threadIdx.x < 32) {
        s = ws[threadIdx.x];
#pragma unroll
        for (int d = 16; d; d >>= 1) s += __shfl_xor_sync(0xFFFFFFFFu, s, d);
        if (threadIdx.x == 0) bsum[blockIdx.x] = s;
    }
}
// exclusive scan of bsum[0..nblk) in place by one block; bsum[nblk] = total
__global__ void __launch_bounds__(1024) ibp_scan_bsums(unsigned long long* bsum, uint64_t nblk) {
    __shared__ unsigned long long ws[32];
    __shared__ unsigned long long run_s;
    if (threadIdx.x == 0) run_s = 0;
    __syncthreads();
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    for (uint64_t base = 0; base < nblk; base += 1024) {
        const uint64_t i = base + threadIdx.x;
        const unsigned long long v = i < nblk ? bsum[i] : 0ull;
        unsigned long long incl = v;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) { const unsigned long long t = __shfl_up_sync(0xFFFFFFFFu, incl, d); if (lane >= d) incl += t; }
        if (lane == 31) ws[wid] = incl;
        __syncthreads();
        if (wid == 0) {
            unsigned long long w = ws[lane], wi = w;
#pragma unroll
            for (int d = 1; d < 32; d <<= 1) { const unsigned long long t = __shfl_up_sync(0xFFFFFFFFu, wi, d); if (lane >= d) wi += t; }
            ws[lane] = wi - w;
        }
        __syncthreads();
        const unsigned long long run = run_s;
        if (i < nblk) bsum[i] = run + ws[wid] + incl - v;
        __syncthreads();
        if (threadIdx.x == 1023) run_s = run + ws[31] + incl;
        __syncthreads();
    }
    if (threadIdx.x == 0) bsum[nblk] = run_s;
}
// in place: data[i] = exclusive prefix; data[n] = total (low 32 bits)
__global__ void __launch_bounds__(1024) ibp_scan_apply(uint32_t* data, uint64_t n, const unsigned long long* __restrict__ bsum) {
    __shared__ uint32_t ws[32];
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    const uint64_t i0 = (uint64_t)blockIdx.x * 4096 + threadIdx.x * 4ull;
    uint32_t v[4], s = 0;
#pragma unroll
    for (int k = 0; k < 4; ++k) { v[k] = i0 + k < n ? data[i0 + k] : 0u; s += v[k]; }
    const uint32_t incl = warp_inclusive_scan(s, lane);
    if (lane == 31) ws[wid] = incl;
    __syncthreads();
    if (wid == 0) { const uint32_t w = ws[lane]; ws[lane] = warp_inclusive_scan(w, lane) - w; }
    __syncthreads();
    uint32_t e = (uint32_t)bsum[blockIdx.x] + ws[wid] + incl - s;
#pragma unroll
    for (int k = 0; k < 4; ++k) { if (i0 + k < n) data[i0 + k] = e; e += v[k]; }
    if (blockIdx.x == gridDim.x - 1 && threadIdx.x == 0) data[n] = (uint32_t)bsum[gridDim.x];
}

int pick_W(uint32_t row_bytes) {
    if (row_bytes % 16 == 0 && row_bytes >= 512) return 4;
    if (row_bytes % 8 == 0 && row_bytes >= 256) return 2;
    return 1;
}

template <int W>
ibp_status launch_masks(const BuildParams& P, bool tm, int np, int grid, cudaStream_t st) {
    if (!tm) ibp_mask_kernel<W, false, 1><<<grid, 256, 0, st>>>(P);
    else if (np == 9) ibp_mask_kernel<W, true, 9><<<grid, 256, 0, st>>>(P);
    else ibp_mask_kernel<W, true, 16><<<grid, 256, 0, st>>>(P);
    IBP_CUDA(cudaGetLastError());
    if (P.ns > 1) {
        const uint64_t cells = P.n_groups * P.nw;
        const unsigned blocks = (unsigned)((cells + 127) / 128);
        if (!tm) ibp_mask_merge_kernel<false, 1><<<blocks, 128, 0, st>>>(P);
        else if (np == 9) ibp_mask_merge_kernel<true, 9><<<blocks, 128, 0, st>>>(P);
        else ibp_mask_merge_kernel<true, 16><<<blocks, 128, 0, st>>>(P);
        IBP_CUDA(cudaGetLastError());
    }
    return IBP_OK;
}

struct Timer {                        // CUDA events on the stream around a phase of the build
    cudaEvent_t a = nullptr, b = nullptr;
    cudaStream_t st;
    explicit Timer(cudaStream_t s) : st(s) { cudaEventCreate(&a); cudaEventCreate(&b); }
    ~Timer() { if (a) cudaEventDestroy(a); if (b) cudaEventDestroy(b); }
    void start() { cudaEventRecord(a, st); }
    void stop() { cudaEventRecord(b, st); }
    double ms() { float t = 0; if (cudaEventSynchronize(b) != cudaSuccess || cudaEventElapsedTime(&t, a, b) != cudaSuccess) { (void)cudaGetLastError(); return 0; } return t; }
};

struct DevBuf {                       // frees device scratch on every exit path
    void* p = nullptr;
    ~DevBuf() { if (p) cudaFree(p); }
};

}  // namespace

extern "C" ibp_status ibp_build_device(const void* rows_dev, const ibp_build_params* params, int device, void* cuda_stream,
                                       ibp_handle** out_handle) {
    if (!rows_dev || !params || !out_handle) { ibp_set_error("ibp_build_device: null argument"); return IBP_ERR_INVALID_ARG; }
    if ((uintptr_t)rows_dev & 15u) { ibp_set_error("ibp_build_device: rows_dev must be 16-byte aligned"); return IBP_ERR_INVALID_ARG; }
    if (params->struct_size == sizeof(ibp_build_params) && (params->flags & IBP_FLAG_PAGEABLE_STORE)) {
        ibp_set_error("ibp_build_device: the GPU writes the packed store in place; a pageable store is not GPU-visible");
        return IBP_ERR_INVALID_ARG;
    }
    int ndev = 0;
    IBP_CUDA(cudaGetDeviceCount(&ndev));
    if (device < 0 || device >= ndev) { ibp_set_error("ibp_build_device: no CUDA device %d", device); return IBP_ERR_CUDA; }
    cudaDeviceProp prop;
    IBP_CUDA(cudaGetDeviceProperties(&prop, device));
    if (prop.major != 10) { ibp_set_error("ibp_build_device: device %d is sm_%d%d; this library is built for sm_100a only", device, prop.major, prop.minor); return IBP_ERR_UNSUPPORTED; }
    IBP_CUDA(cudaSetDevice(device));
    const auto t_begin = std::chrono::steady_clock::now();
    ibp_handle* h = nullptr;
    ibp_status rc = ibp_prepare_handle(params, "ibp_build_device", &h);
    if (rc != IBP_OK) return rc;
    struct Guard { ibp_handle* h; ~Guard() { if (h) ibp_destroy(h); } } guard{h};

    const ibp_build_params& p = h->p;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const uint32_t nw = h->n_words;
    const uint64_t ng = h->n_groups, n = p.n_rows;
    const int W = pick_W(p.row_bytes);
    const int sms = prop.multiProcessorCount;
    const uint64_t Nmax = p.group_kind == IBP_GROUP_BLOCKED ? std::min<uint64_t>(p.group_param, n) : (n + p.group_param - 1) / p.group_param;
    if (Nmax > 0xFFFFFFFFull) { ibp_set_error("ibp_build_device: groups of more than 2^32-1 rows are not supported"); return IBP_ERR_UNSUPPORTED; }

    BuildParams B;
    memset(&B, 0, sizeof B);
    B.rows = (const uint32_t*)rows_dev;
    B.n_rows = n; B.n_groups = ng; B.nw = nw;
    B.n_pass = (nw + 32 * W - 1) / (32 * W);
    B.group_param = p.group_param;
    B.group_shift = 0xFFFFFFFFu;
    if ((p.group_param & (p.group_param - 1)) == 0) { uint32_t s = 0; while ((1u << s) < p.group_param) ++s; B.group_shift = s; }
    B.strided = p.group_kind == IBP_GROUP_STRIDED;
    B.thr_num = p.threshold_num; B.thr_den = p.threshold_den;
    // slices: enough warps to fill the GPU when there are few groups; a slice never exceeds 65535 rows (16 counter planes)
    const uint64_t target_units = (uint64_t)sms * 32;
    uint64_t ns = 1;
    if (ng < target_units) ns = std::min<uint64_t>((target_units + ng - 1) / ng, (Nmax + 63) / 64);
    ns = std::max<uint64_t>(ns, (Nmax + 65534) / 65535);
    ns = std::max<uint64_t>(ns, 1);
    B.rows_per_slice = (Nmax + ns - 1) / ns;
    B.ns = (uint32_t)((Nmax + B.rows_per_slice - 1) / B.rows_per_slice);
    const int np = B.rows_per_slice <= 511 ? 9 : 16;

    IBP_CUDA(cudaMalloc((void**)&h->meta_dev, ng * 2ull * nw * 4));
    DevBuf kbits, scratch;
    IBP_CUDA(cudaMalloc(&kbits.p, ng * 4));
    B.meta = h->meta_dev;
    B.kbits = (uint32_t*)kbits.p;
    if (B.ns > 1) {
        const uint64_t per_unit = (uint64_t)(h->thresholded ? np : 2) * nw * 4;
        if (cudaMalloc(&scratch.p, ng * B.ns * per_unit) != cudaSuccess) {
            (void)cudaGetLastError();
            ibp_set_error("ibp_build_device: out of device memory (slice accumulators, %llu bytes)", (unsigned long long)(ng * B.ns * per_unit));
            return IBP_ERR_OUT_OF_MEMORY;
        }
        B.scratch = (uint32_t*)scratch.p;
        IBP_CUDA(cudaMemsetAsync(kbits.p, 0, ng * 4, st));
    }
    const int grid_masks = (int)std::min<uint64_t>((ng * B.ns + 7) / 8, (uint64_t)sms * 8);
    Timer t_mask(st), t_size(st), t_scan(st), t_pack(st);
    t_mask.start();
    switch (W) {
        case 4: rc = launch_masks<4>(B, h->thresholded, np, grid_masks, st); break;
        case 2: rc = launch_masks<2>(B, h->thresholded, np, grid_masks, st); break;
        default: rc = launch_masks<1>(B, h->thresholded, np, grid_masks, st); break;
    }
    t_mask.stop();
    if (rc != IBP_OK) return rc;

    // host copies of the metadata (accessors, layout)
    std::vector<uint32_t> kb;
    try { kb.resize(ng); } catch (...) { ibp_set_error("ibp_build_device: out of memory"); return IBP_ERR_OUT_OF_MEMORY; }
    IBP_CUDA(cudaMemcpyAsync(kb.data(), kbits.p, ng * 4, cudaMemcpyDeviceToHost, st));
    IBP_CUDA(cudaMemcpyAsync(h->meta.data(), h->meta_dev, ng * 2ull * nw * 4, cudaMemcpyDeviceToHost, st));
    IBP_CUDA(cudaStreamSynchronize(st));
    for (uint64_t g = 0; g < ng; ++g) h->gtab[g].k_bits = kb[g];
    const int nthreads = p.n_threads ? (int)p.n_threads : 0;

    PackParams K;
    memset(&K, 0, sizeof K);
    K.rows = B.rows; K.meta = h->meta_dev;
    K.n_rows = n; K.nw = nw; K.n_pass = B.n_pass;
    K.group_param = p.group_param; K.group_shift = B.group_shift; K.strided = B.strided;
    K.align_bytes = p.align_bytes;
    int wpc = 8;

    if (!h->thresholded) {
        ibp_layout_strict(h);
        rc = ibp_alloc_store(h, nthreads);
        if (rc != IBP_OK) return rc;
        rc = ibp_attach_device(h, device, cuda_stream);
        if (rc != IBP_OK) return rc;
        if (!h->store_dev) { ibp_set_error("ibp_build_device: the packed store is not GPU-visible"); return IBP_ERR_BAD_STATE; }
        K.gtab = h->gtab_dev;
        K.store = h->store_dev;
        K.row_stride_strided = h->row_stride_strided;
        const bool bulk = !B.strided && p.align_bytes >= 16 && h->max_stride > 0 && h->max_stride <= 12288;
        size_t smem;
        if (bulk) {
            K.rows_per_unit = (uint32_t)std::max<uint64_t>(1, std::min<uint64_t>(16, 12288 / h->max_stride));
            K.slot_bytes = (K.rows_per_unit * h->max_stride + 16u + 127u) / 128u * 128u;
            K.n_units = (n + K.rows_per_unit - 1) / K.rows_per_unit;
            while (wpc > 1 && (size_t)wpc * 2 * K.slot_bytes > 200 * 1024) wpc >>= 1;
            smem = (size_t)wpc * 2 * K.slot_bytes;
        } else {
            K.slot_bytes = (h->max_stride + 15u) / 16u * 16u + 16u;
            K.n_units = B.strided ? ((((n + p.group_param - 1) / p.group_param) + 15) / 16) * (uint64_t)p.group_param : (n + 15) / 16;
            while (wpc > 1 && (size_t)wpc * K.slot_bytes > 200 * 1024) wpc >>= 1;
            smem = (size_t)wpc * K.slot_bytes;
        }
        if (smem > 200 * 1024) { ibp_set_error("ibp_build_device: packed rows of %u bytes do not fit the shared-memory row images", h->max_stride); return IBP_ERR_UNSUPPORTED; }
        const int grid = (int)std::min<uint64_t>((K.n_units + wpc - 1) / wpc, (uint64_t)sms * (bulk ? 2 : 8));
#define IBP_PACK(KERN_, W_)                                                                                                  \
    do {                                                                                                                     \
        static unsigned long long optin_done = 0;                                                                            \
        if (smem > 48 * 1024) IBP_CUDA(ibp_optin_max_smem(KERN_<W_>, &optin_done));                                          \
        KERN_<W_><<<grid, wpc * 32, smem, st>>>(K);                                                                          \
    } while (0)
        t_pack.start();
        if (h->max_stride && bulk) {
            switch (W) { case 4: IBP_PACK(ibp_pack_bulk_kernel, 4); break; case 2: IBP_PACK(ibp_pack_bulk_kernel, 2); break; default: IBP_PACK(ibp_pack_bulk_kernel, 1); break; }
        } else if (h->max_stride) {
            switch (W) { case 4: IBP_PACK(ibp_pack_kernel, 4); break; case 2: IBP_PACK(ibp_pack_kernel, 2); break; default: IBP_PACK(ibp_pack_kernel, 1); break; }
        }
#undef IBP_PACK
        t_pack.stop();
        IBP_CUDA(cudaGetLastError());
        IBP_CUDA(cudaStreamSynchronize(st));
    } else {
        // pass 1: sizes and flags; scan -> row offsets
        const uint64_t n_flag_words = (n + 31) / 32;
        IBP_CUDA(cudaMalloc((void**)&h->row_off_dev, (n + 1) * 4 + 64));   // slack: the stream kernels copy 16-byte covers
        {
            const uint64_t words = h->slot_layout ? (h->capacity_rows + 31) / 32 : n_flag_words;
            IBP_CUDA(cudaMalloc((void**)&h->row_flag_dev, words * 4 + 64));
            IBP_CUDA(cudaMemsetAsync(h->row_flag_dev, 0, words * 4, st));
        }
        const uint64_t nblk = (n + 4095) / 4096;
        DevBuf aux;
        IBP_CUDA(cudaMalloc(&aux.p, (nblk + 2) * 8));
        unsigned long long* bsum = (unsigned long long*)aux.p;
        unsigned long long* sum_size = bsum + nblk + 1;
        IBP_CUDA(cudaMemsetAsync(sum_size, 0, 8, st));
        K.row_off_out = h->row_off_dev;
        K.row_flag = h->row_flag_dev;
        K.sum_size = sum_size;
        K.n_units = n_flag_words;
        const int grid1 = (int)std::min<uint64_t>((K.n_units + wpc - 1) / wpc, (uint64_t)sms * 8);
        t_size.start();
        switch (W) {
            case 4: ibp_size_kernel<4><<<grid1, wpc * 32, 0, st>>>(K); break;
            case 2: ibp_size_kernel<2><<<grid1, wpc * 32, 0, st>>>(K); break;
            default: ibp_size_kernel<1><<<grid1, wpc * 32, 0, st>>>(K); break;
        }
        t_size.stop();
        IBP_CUDA(cudaGetLastError());
        unsigned long long totals[2] = {0, 0};   // [0] = stored bytes of the rows in 16-byte units, [1] = sum of the byte-aligned row sizes
        t_scan.start();
        if (h->slot_layout) {
            const uint64_t cap = h->capacity_rows;
            if (h->slot_bytes / 16 > 255) { ibp_set_error("ibp_build_device: slot layout needs row_bytes <= 4080"); return IBP_ERR_UNSUPPORTED; }
            IBP_CUDA(cudaMalloc((void**)&h->row_size_dev, std::max<uint64_t>(cap, 16)));
            IBP_CUDA(cudaMemsetAsync(h->row_size_dev, 0, std::max<uint64_t>(cap, 16), st));
            IBP_CUDA(cudaMemsetAsync(bsum + nblk, 0, 8, st));
            ibp_slot_layout_kernel<<<(unsigned)std::min<uint64_t>((n + 256) / 256, (uint64_t)sms * 8), 256, 0, st>>>(h->row_off_dev, n, h->slot_bytes / 16, h->row_size_dev, bsum + nblk);
        } else {
            ibp_scan_sums<<<(unsigned)nblk, 1024, 0, st>>>(h->row_off_dev, n, bsum);
            ibp_scan_bsums<<<1, 1024, 0, st>>>(bsum, nblk);
            ibp_scan_apply<<<(unsigned)nblk, 1024, 0, st>>>(h->row_off_dev, n, bsum);
        }
        t_scan.stop();
        IBP_CUDA(cudaGetLastError());
        IBP_CUDA(cudaMemcpyAsync(totals, bsum + nblk, 16, cudaMemcpyDeviceToHost, st));
        const uint64_t n_flag_alloc = h->slot_layout ? (h->capacity_rows + 31) / 32 : n_flag_words;
        try {
            if (h->slot_layout) h->row_size.assign(h->capacity_rows, 0); else h->row_off.resize(n + 1);
            h->row_flag.assign(n_flag_alloc, 0u);
        } catch (...) { ibp_set_error("ibp_build_device: out of memory (row offsets)"); return IBP_ERR_OUT_OF_MEMORY; }
        IBP_CUDA(cudaMemcpyAsync(h->row_flag.data(), h->row_flag_dev, n_flag_words * 4, cudaMemcpyDeviceToHost, st));
        IBP_CUDA(cudaStreamSynchronize(st));
        if (!h->slot_layout && totals[0] > 0xFFFFFFFFull) { ibp_set_error("ibp_build_device: thresholded store exceeds 64 GiB (4-byte row offsets in 16-byte units)"); return IBP_ERR_UNSUPPORTED; }
        if (h->slot_layout) IBP_CUDA(cudaMemcpyAsync(h->row_size.data(), h->row_size_dev, n, cudaMemcpyDeviceToHost, st));
        else IBP_CUDA(cudaMemcpyAsync(h->row_off.data(), h->row_off_dev, (n + 1) * 4, cudaMemcpyDeviceToHost, st));
        uint64_t n_comp = 0;
        for (uint64_t i = 0; i < n_flag_words; ++i) n_comp += (uint64_t)__builtin_popcount(h->row_flag[i]);
        h->n_rows_raw = n - n_comp;
        h->packed_bytes_bytealigned = totals[1];
        h->packed_bytes_rows = totals[0] * 16;
        h->store_used = h->slot_layout ? h->capacity_rows * (uint64_t)h->slot_bytes : totals[0] * 16;
        h->store_bytes = (h->store_used + 64 + 4095) / 4096 * 4096;
        h->max_stride = (p.row_bytes + p.align_bytes - 1) / p.align_bytes * p.align_bytes;
        rc = ibp_alloc_store(h, nthreads);
        if (rc != IBP_OK) return rc;
        rc = ibp_attach_device(h, device, cuda_stream);
        if (rc != IBP_OK) return rc;
        if (!h->store_dev) { ibp_set_error("ibp_build_device: the packed store is not GPU-visible"); return IBP_ERR_BAD_STATE; }
        K.store = h->store_dev;
        K.row_off = h->row_off_dev;
        K.rows_per_unit = (uint32_t)std::max<uint64_t>(1, std::min<uint64_t>(16, 12288 / h->max_stride));
        K.slot_bytes = (K.rows_per_unit * h->max_stride + 16u + 127u) / 128u * 128u;
        K.n_units = (n + K.rows_per_unit - 1) / K.rows_per_unit;
        while (wpc > 1 && (size_t)wpc * 2 * K.slot_bytes > 200 * 1024) wpc >>= 1;
        const size_t smem = (size_t)wpc * 2 * K.slot_bytes;
        if (smem > 200 * 1024) { ibp_set_error("ibp_build_device: rows of %u bytes do not fit the shared-memory row images", p.row_bytes); return IBP_ERR_UNSUPPORTED; }
        const int grid2 = (int)std::min<uint64_t>((K.n_units + wpc - 1) / wpc, (uint64_t)sms * 2);
#define IBP_PACK_T(W_)                                                                                                         \
    do {                                                                                                                       \
        static unsigned long long optin_done = 0;                                                                              \
        if (smem > 48 * 1024) IBP_CUDA(ibp_optin_max_smem(ibp_pack_t_kernel<W_>, &optin_done));                                \
        ibp_pack_t_kernel<W_><<<grid2, wpc * 32, smem, st>>>(K);                                                               \
    } while (0)
        t_pack.start();
        switch (W) { case 4: IBP_PACK_T(4); break; case 2: IBP_PACK_T(2); break; default: IBP_PACK_T(1); break; }
#undef IBP_PACK_T
        t_pack.stop();
        IBP_CUDA(cudaGetLastError());
        IBP_CUDA(cudaStreamSynchronize(st));
        if (h->slot_layout) { cudaFree(h->row_off_dev); h->row_off_dev = nullptr; }   // the fixed shift needs no table
    }
    h->built_on_device = true;
    ibp_build_stats& S = h->build_stats;
    S.mask_ms = t_mask.ms();
    S.pack_ms = t_pack.ms();
    if (h->thresholded) { S.size_ms = t_size.ms(); S.scan_ms = t_scan.ms(); }
    S.raw_bytes = n * (uint64_t)p.row_bytes;
    S.store_bytes = h->packed_bytes_rows;
    S.slices_per_group = B.ns;
    S.total_ms = std::chrono::duration<double, std::milli>(std::chrono::steady_clock::now() - t_begin).count();
    guard.h = nullptr;
    *out_handle = h;
    return IBP_OK;
}

extern "C" ibp_status ibp_append_rows_device(ibp_handle* h, const void* rows_dev, int64_t n_new, void* cuda_stream) {
    if (!h) { ibp_set_error("ibp_append_rows_device: null handle"); return IBP_ERR_INVALID_ARG; }
    if (!h->slot_layout) { ibp_set_error("ibp_append_rows_device: the handle was not built with IBP_FLAG_SLOT_LAYOUT (a dense store cannot grow in place)"); return IBP_ERR_BAD_STATE; }
    if (h->store_kind == IBP_STORE_SHARED) { ibp_set_error("ibp_append_rows_device: a shared store (ibp_open_shared) is read-only"); return IBP_ERR_BAD_STATE; }
    if (h->device < 0 || !h->meta_dev || !h->store_dev) { ibp_set_error("ibp_append_rows_device: call ibp_upload_metadata first (GPU-visible store)"); return IBP_ERR_BAD_STATE; }
    if (n_new == 0) return IBP_OK;
    if (n_new < 0 || !rows_dev || ((uintptr_t)rows_dev & 15u)) { ibp_set_error("ibp_append_rows_device: bad argument (n_new < 0, null or unaligned rows_dev)"); return IBP_ERR_INVALID_ARG; }
    ibp_build_params& p = h->p;
    const uint64_t first = p.n_rows, last = first + (uint64_t)n_new - 1;
    if (last >= h->capacity_rows) { ibp_set_error("ibp_append_rows_device: %lld rows do not fit (%llu of %llu slots used)", (long long)n_new, (unsigned long long)first, (unsigned long long)h->capacity_rows); return IBP_ERR_UNSUPPORTED; }
    if ((uint64_t)n_new % p.index_span) { ibp_set_error("ibp_append_rows_device: n_new must be a multiple of index_span"); return IBP_ERR_INVALID_ARG; }
    const uint64_t g_last = p.group_kind == IBP_GROUP_BLOCKED ? last / p.group_param : std::min<uint64_t>(last, (uint64_t)p.group_param - 1);
    const uint64_t g_need = p.group_kind == IBP_GROUP_BLOCKED ? g_last : (first + (uint64_t)n_new >= p.group_param ? (uint64_t)p.group_param - 1 : last);
    if (std::max(g_last, g_need) >= h->n_groups) {
        ibp_set_error("ibp_append_rows_device: a new row falls in group %llu, which has no Mask/Bitval (%llu groups were built)", (unsigned long long)std::max(g_last, g_need), (unsigned long long)h->n_groups);
        return IBP_ERR_UNSUPPORTED;
    }
    IBP_CUDA(cudaSetDevice(h->device));
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const int W = pick_W(p.row_bytes);
    AppendParams A;
    memset(&A, 0, sizeof A);
    A.rows = (const uint32_t*)rows_dev; A.meta = h->meta_dev; A.store = h->store_dev;
    A.row_size = h->row_size_dev; A.row_flag = h->row_flag_dev;
    A.first_id = first; A.n_new = (uint64_t)n_new;
    A.nw = h->n_words; A.n_pass = (h->n_words + 32 * W - 1) / (32 * W);
    A.group_param = p.group_param; A.group_shift = 0xFFFFFFFFu;
    if ((p.group_param & (p.group_param - 1)) == 0) { uint32_t sft = 0; while ((1u << sft) < p.group_param) ++sft; A.group_shift = sft; }
    A.strided = p.group_kind == IBP_GROUP_STRIDED;
    A.align_bytes = p.align_bytes; A.slot_bytes = h->slot_bytes;
    A.img_bytes = (h->slot_bytes + 32u + 127u) / 128u * 128u;
    int wpc = 8;
    while (wpc > 1 && (size_t)wpc * A.img_bytes > 200 * 1024) wpc >>= 1;
    const size_t smem = (size_t)wpc * A.img_bytes;
    DevBuf sums;
    IBP_CUDA(cudaMalloc(&sums.p, 24));
    IBP_CUDA(cudaMemsetAsync(sums.p, 0, 24, st));
    A.sums = (unsigned long long*)sums.p;
    const int grid = (int)std::min<uint64_t>(((uint64_t)n_new + wpc - 1) / wpc, (uint64_t)h->sm_count * 4);
#define IBP_APPEND(W_)                                                                              \
    do {                                                                                            \
        static unsigned long long optin_done = 0;                                                   \
        if (smem > 48 * 1024) IBP_CUDA(ibp_optin_max_smem(ibp_append_kernel<W_>, &optin_done));     \
        ibp_append_kernel<W_><<<grid, wpc * 32, smem, st>>>(A);                                     \
    } while (0)
    switch (W) { case 4: IBP_APPEND(4); break; case 2: IBP_APPEND(2); break; default: IBP_APPEND(1); break; }
#undef IBP_APPEND
    IBP_CUDA(cudaGetLastError());
    // host mirrors: sizes and flag words of the new rows, totals
    unsigned long long tot[3] = {0, 0, 0};
    const uint64_t w_lo = first >> 5, w_hi = last >> 5;
    IBP_CUDA(cudaMemcpyAsync(tot, sums.p, 24, cudaMemcpyDeviceToHost, st));
    IBP_CUDA(cudaMemcpyAsync(h->row_size.data() + first, h->row_size_dev + first, (size_t)n_new, cudaMemcpyDeviceToHost, st));
    IBP_CUDA(cudaMemcpyAsync(h->row_flag.data() + w_lo, h->row_flag_dev + w_lo, (size_t)(w_hi - w_lo + 1) * 4, cudaMemcpyDeviceToHost, st));
    IBP_CUDA(cudaStreamSynchronize(st));
    p.n_rows += (uint64_t)n_new;
    h->packed_bytes_bytealigned += tot[0];
    h->packed_bytes_rows += tot[1];
    h->n_rows_raw += tot[2];
    return IBP_OK;
}

extern "C" ibp_status ibp_get_build_stats(const ibp_handle* h, ibp_build_stats* out) {
    if (!h || !out) { ibp_set_error("ibp_get_build_stats: null argument"); return IBP_ERR_INVALID_ARG; }
    if (!h->built_on_device) { ibp_set_error("ibp_get_build_stats: the handle was built by ibp_build (host)"); return IBP_ERR_BAD_STATE; }
    *out = h->build_stats;
    return IBP_OK;
}
