// ibp_device.cu -- CUDA side of libibp.so (sm_100a): the fused gather-and-decompress kernels and their launchers.
//
// One kernel family decodes "units" of rows, one warp per unit ("each tensor being decompressed by a
// separate warp"), in three modes:
//   MODE_ROWS    random row ids, one row per unit (GNN / DLRM gathers), optionally in a locality order
//   MODE_SPANS   runs of consecutive rows of blocked groups (KV pages, resident ranges): R rows per unit
//   MODE_STRIDED whole strided tables streamed in order (weight matrices): unit = R matrix rows of one column tile
// Per row (S1..S6 of SURVEY.md section 8a):
//   S1 locate   group entry -> source address in the packed store (pinned host memory, or HBM for resident decode)
//   S3 fetch    16-byte cp.async copies of the 16-byte-aligned cover of the packed row into a per-warp shared-memory
//               ring (P:213 workspace, P:333 aligned transfers, P:213/[75] asynchronous copies), NST rows in flight
//   S2 metadata Mask/Bitval words of the group: W consecutive 32-bit words per lane, vector loads from HBM/L2,
//               kept in registers while consecutive rows stay in the same group
//   S4 offsets  k_i = popc(~Mask_i), exclusive warp scan (shuffles) -> start bit of every word (P:319 steps 2-3)
//   S5 expand   funnel-shift the k_i bits out of shared memory, deposit them at the Mask=0 positions, OR Bitval
//   S6 store    one 16/8/4-byte streaming store per lane: 512/256/128 contiguous bytes per warp instruction
#include <cuda_runtime.h>
#include <sys/mman.h>

#include <cerrno>

#include <algorithm>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <type_traits>
#include <vector>

#include "ibp_internal.h"

#include "ibp_devutil.cuh"

enum { MODE_ROWS = 0, MODE_SPANS = 1, MODE_STRIDED = 2 };

struct DecodeParams {
    const uint8_t* store;          // device-visible packed bytes; row at store + offset(id) - bias
    uint64_t bias;
    const uint32_t* meta;          // per group: Mask words, Bitval words
    const IbpGroupEntry* gtab;
    const int64_t* ids;            // MODE_ROWS / MODE_SPANS gather; nullptr for ranges
    const int32_t* order;          // MODE_ROWS: optional processing order
    uint8_t* out;
    int64_t n;                     // ids (gather) or rows (range)
    int64_t first_row;             // ranges
    int64_t n_units;
    const uint32_t* n_units_dev;   // MODE_ROWS with de-duplication: number of work-list entries, known only on the device
    uint64_t row_stride_strided;
    uint32_t row_bytes, n_words, n_pass;
    uint32_t group_param, group_shift;   // group_shift >= 0 when group_param is a power of two, else 0xFFFFFFFF
    uint32_t span;                 // rows per id (gather) or rows of the range
    uint32_t rows_per_unit, units_per_span;
    uint32_t slot_bytes;
    uint32_t strided;              // group kind of the handle (MODE_ROWS serves both kinds)
    uint32_t occ_cap;              // host side only: CTAs per SM for random-row gathers (0 = 2)
    const uint32_t* row_off;       // thresholded mode: per-row offsets (16-byte units), n_rows + 1 entries
    const uint32_t* row_flag;      // thresholded mode: bit r = 1 iff row r is compressed
    const uint8_t* row_size;       // slot layout: stored size of row r in 16-byte units; the row lies at r * slot16 * 16
    uint32_t slot16;               // slot layout: slot size in 16-byte units; 0 = dense rows addressed through row_off
    uint32_t keep_l2;              // write the rows with the default cache policy (a later pass re-reads them) instead of streaming
    // compressed GPU cache in front of the store (CACHE instantiations only)
    const uint64_t* cmap;          // hash map slots {id + 1, value}; value = offset:40 | slab:3 | compressed:1
    uint32_t cmap_mask;
    const uint8_t* slab[8];
};

// ------------------------------------------------------------------------------------------------ device helpers
__device__ __forceinline__ void cp_async16(uint32_t smem_addr, const void* gptr) {
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(smem_addr), "l"(gptr) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

// Deposit the low popc(nv) bits of x at the set positions of nv, lowest first, one run of contiguous positions per
// iteration (float data has 1-3 runs per 32-bit word).  S5 "re-insert the removed bits" (P:211, P:319 step 5).
__device__ __forceinline__ uint32_t deposit_runs(uint32_t x, uint32_t nv) {
    uint32_t r = 0;
    while (nv) {
        const uint32_t low = nv & (0u - nv);     // lowest set bit = start of the lowest run
        const uint32_t t = nv + low;             // clears the run, carries into the bit above it
        const uint32_t run = nv & ~t;            // the run itself
        r |= (x * low) & run;                    // x << start, clipped to the run
        x >>= __popc(run);
        nv &= t;
    }
    return r;
}

__device__ __forceinline__ uint64_t group_of(const DecodeParams& P, uint64_t id, bool strided) {
    if (strided) return id % P.group_param;
    return P.group_shift != 0xFFFFFFFFu ? (id >> P.group_shift) : (id / P.group_param);
}

// ------------------------------------------------------------------------------------------------ the kernel
// FETCH selects the engine that moves the packed row into shared memory:
//   FETCH_LSU  16-byte cp.async per lane (Ampere-style asynchronous copy, the paper's [75]) through the load/store unit
//   FETCH_TMA  one cp.async.bulk per row issued by lane 0, completion on an mbarrier (Hopper/Blackwell bulk-copy engine)
// The L1TEX path returns loads in issue order per SM, so on the LSU path every fast HBM load of the kernel (ids, group
// table, Mask/Bitval) queues behind other warps' multi-microsecond PCIe reads; the TMA path keeps the slow reads out of
// that queue (profiles/r01_*).
enum { FETCH_LSU = 0, FETCH_TMA = 1 };

__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
    uint32_t ok = 0;
    while (!ok) {
        asm volatile(
            "{\n\t.reg .pred p;\n\t"
            "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
            "selp.u32 %0, 1, 0, p;\n\t}"
            : "=r"(ok) : "r"(bar), "r"(parity) : "memory");
    }
}
__device__ __forceinline__ void bulk_g2s(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(dst), "l"(src), "r"(bytes), "r"(bar) : "memory");
}

#include "ibp_stream.cuh"
#include "ibp_stream_t.cuh"

// TM = thresholded mode (the paper's default codec): the row's location and length come from the per-row
// offset table, the per-row bitmask says whether it is stored raw, the first n_words bits of a compressed row are
// the participation bits (one per 4-byte chunk), and a chunk contributes 32 - popc(Mask_i) bits if it participates, else 32
// (reading R7) -- so the exclusive scan of step 3 runs per row instead of per group.
// CACHE = the compressed GPU cache sits in front of the store: S1 probes the hash map; a hit fetches the same
// 16-byte-aligned cover from the row's slab in HBM instead of the host store, everything after the fetch is unchanged.
template <int W, int NST, int MODE, int FETCH, bool TM, bool CACHE = false>
__global__ void __launch_bounds__(256) ibp_decode_kernel(const DecodeParams P) {
    extern __shared__ __align__(128) uint8_t smem[];
    const int lane = threadIdx.x & 31, wib = threadIdx.x >> 5, wpc = blockDim.x >> 5;
    uint8_t* ring = smem + (size_t)wib * NST * P.slot_bytes;
    const uint32_t ring_s = (uint32_t)__cvta_generic_to_shared(ring);
    const uint32_t bars_s = (uint32_t)__cvta_generic_to_shared(smem + (size_t)wpc * NST * P.slot_bytes) + wib * NST * 8;
    const bool STRIDED = MODE == MODE_STRIDED || (MODE == MODE_ROWS && P.strided);

    if (FETCH == FETCH_TMA) {
        if (lane == 0) {
#pragma unroll
            for (int s = 0; s < NST; ++s) mbar_init(bars_s + s * 8, 1);
            asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        }
        __syncwarp();
    }

    // register-resident metadata of the current group (valid for single-pass rows)
    uint64_t meta_g = ~0ull;
    uint32_t m[W], b[W], kk[W], excl = 0;

    // group-entry caches: one for the fetch side, one for the decode side
    uint64_t fg = ~0ull, dg = ~0ull;
    IbpGroupEntry fe{0, 0, 0}, de{0, 0, 0};
    uint32_t seq_f = 0, seq_d = 0;   // rows fetched / decoded so far by this warp: ring slot = seq % NST

    // MODE_ROWS: the warp's whole share of the batch is ONE unit whose rows are the positions gw, gw+NWT, gw+2*NWT, ...
    // of the (locality-ordered) list, so that the NST rows it keeps in flight, together with the other warps', form
    // one contiguous window of the list.  Other modes: units of consecutive rows, grid-stride over units.
    const int64_t gw = (int64_t)blockIdx.x * wpc + wib, NWT = (int64_t)gridDim.x * wpc;
    const int64_t n_total = (MODE == MODE_ROWS && P.n_units_dev) ? (int64_t)*P.n_units_dev : P.n_units;
    const int64_t n_units = MODE == MODE_ROWS ? (gw < n_total ? gw + 1 : 0) : n_total;
    for (int64_t u = gw; u < n_units; u += NWT) {
        // ---- unit -> rows
        int64_t id0 = 0, out0 = 0;
        uint32_t nrows, id_step = 0, out_step = 0;
        if (MODE == MODE_ROWS) {
            nrows = (uint32_t)((n_total - gw + NWT - 1) / NWT);
        } else if (MODE == MODE_SPANS) {
            const int64_t si = u / P.units_per_span;
            const uint32_t c = (uint32_t)(u - si * P.units_per_span);
            const int64_t base_id = P.ids ? P.ids[si] * (int64_t)P.span : P.first_row;
            id0 = base_id + (int64_t)c * P.rows_per_unit;
            out0 = si * (int64_t)P.span + (int64_t)c * P.rows_per_unit;
            nrows = min(P.rows_per_unit, P.span - c * P.rows_per_unit);
            id_step = 1; out_step = 1;
        } else {
            const int64_t rb = u / P.group_param;
            const uint32_t t = (uint32_t)(u - rb * P.group_param);
            const int64_t r0 = rb * P.rows_per_unit;
            id0 = P.first_row + r0 * P.group_param + t;
            out0 = r0 * P.group_param + t;
            const int64_t left = (P.n - out0 + P.group_param - 1) / P.group_param;   // rows of this tile still in range
            nrows = left < (int64_t)P.rows_per_unit ? (left > 0 ? (uint32_t)left : 0u) : P.rows_per_unit;
            id_step = P.group_param; out_step = P.group_param;
        }
        // row j of the unit -> (row id, output row)
        auto locate = [&](uint32_t j, uint64_t& id, int64_t& orow_idx) {
            if (MODE == MODE_ROWS) {
                const int64_t pos = gw + (int64_t)j * NWT;
                const int64_t i = P.order ? (int64_t)P.order[pos] : pos;
                id = (uint64_t)P.ids[i];
                orow_idx = i;
            } else {
                id = (uint64_t)(id0 + (int64_t)j * id_step);
                orow_idx = out0 + (int64_t)j * out_step;
            }
        };

        // ---- S1 + S3: fetch row j of the unit into the next ring slot
        auto fetch = [&](uint32_t j) {
            uint64_t id; int64_t oi_unused;
            locate(j, id, oi_unused);
            const uint8_t* a0;
            uint32_t nvec;
            if (TM) {
                if (P.slot16) {                                               // in-place slots: a fixed shift, only the first `size` bytes are read
                    a0 = P.store + (16ull * P.slot16 * id - P.bias);
                    nvec = P.row_size[id];
                } else {
                    const uint32_t o0 = __ldg(P.row_off + id), o1 = __ldg(P.row_off + id + 1);
                    a0 = P.store + (16ull * o0 - P.bias);                     // rows start on 16-byte boundaries
                    nvec = o1 - o0;
                }
            } else {
                const uint64_t g = group_of(P, id, STRIDED);
                if (g != fg) { fg = g; fe = P.gtab[g]; }
                const uint64_t off = STRIDED ? (id / P.group_param) * P.row_stride_strided + fe.base
                                             : fe.base + (id - g * P.group_param) * (uint64_t)fe.stride;
                const uint8_t* src = P.store + (off - P.bias);
                const uint32_t head = (uint32_t)((uintptr_t)src & 15u);
                a0 = src - head;                                              // 16-byte aligned cover
                // what is fetched: the row's bytes rounded up to whole 32-byte sectors, never more than its stride (A >= 64 pads rows to
                // lines for alignment, and that padding need not cross the link)
                const uint32_t fb = min(fe.stride, (((fe.k_bits + 7u) >> 3) + 31u) & ~31u);
                nvec = fb ? (head + fb + 15u) >> 4 : 0u;
            }
            if (CACHE) {
                const uint64_t ent = ibp_cache_find(P.cmap, P.cmap_mask, id);
                if (ent != IBP_CACHE_MISS_DEV) a0 = P.slab[(ent >> 40) & 7ull] + (ent & ((1ull << 40) - 1));
            }
            const uint32_t slot = seq_f % NST;
            const uint32_t dst = ring_s + slot * P.slot_bytes;
            if (FETCH == FETCH_TMA) {
                if (lane == 0) {
                    mbar_expect_tx(bars_s + slot * 8, nvec * 16);
                    if (nvec) bulk_g2s(dst, a0, nvec * 16, bars_s + slot * 8);
                }
            } else {
                for (uint32_t v = lane; v < nvec; v += 32) cp_async16(dst + v * 16, a0 + (size_t)v * 16);
            }
            ++seq_f;
        };

#pragma unroll
        for (int s = 0; s < NST - 1; ++s) {
            if ((uint32_t)s < nrows) fetch(s);
            if (FETCH == FETCH_LSU) cp_async_commit();
        }
        for (uint32_t j = 0; j < nrows; ++j) {
            if (j + NST - 1 < nrows) fetch(j + NST - 1);
            if (FETCH == FETCH_LSU) cp_async_commit();

            // ---- locate again for the decode side (cached)
            uint64_t id; int64_t out_idx;
            locate(j, id, out_idx);
            const uint64_t g = group_of(P, id, STRIDED);
            uint32_t head_bits = 0;
            bool compressed = true;
            if (TM) {
                compressed = (__ldg(P.row_flag + (id >> 5)) >> (id & 31u)) & 1u;
                head_bits = P.n_words;                                        // payloads follow the participation bits (R8)
            } else {
                if (g != dg) { dg = g; de = P.gtab[g]; }
                const uint64_t off = STRIDED ? (id / P.group_param) * P.row_stride_strided + de.base
                                             : de.base + (id - g * P.group_param) * (uint64_t)de.stride;
                head_bits = (uint32_t)(((uintptr_t)(P.store + (off - P.bias))) & 15u) * 8u;
            }
            const uint32_t dslot = seq_d % NST;
            const uint32_t* slot = (const uint32_t*)(ring + (size_t)dslot * P.slot_bytes);
            uint8_t* orow = P.out + (uint64_t)out_idx * P.row_bytes;
            const uint32_t* gm = P.meta + g * 2ull * P.n_words;

            bool waited = false;
            uint32_t carry = 0;
            for (uint32_t pass = 0; pass < P.n_pass; ++pass) {
                const uint32_t w0 = (pass * 32u + lane) * W;
                const bool active = w0 < P.n_words;
                // ---- S2 + S4: metadata words and bit offsets (skipped while the group stays the same)
                uint32_t tot;
                if (P.n_pass > 1 || g != meta_g) {
                    if (active) { VecIO<W>::ld(gm + w0, m); VecIO<W>::ld(gm + P.n_words + w0, b); }
                    else {
#pragma unroll
                        for (int q = 0; q < W; ++q) { m[q] = 0xFFFFFFFFu; b[q] = 0; }
                    }
                    if (!TM) {
                        uint32_t t = 0;
#pragma unroll
                        for (int q = 0; q < W; ++q) { kk[q] = __popc(~m[q]); t += kk[q]; }
                        const uint32_t incl = warp_inclusive_scan(t, lane);
                        excl = incl - t;
                        tot = __shfl_sync(0xFFFFFFFFu, incl, 31);
                    }
                    meta_g = g;
                } else {
                    tot = 0;   // single pass: carry is not used again
                }
                if (!waited) {
                    if (FETCH == FETCH_TMA) mbar_wait(bars_s + dslot * 8, (seq_d / NST) & 1u);
                    else { cp_async_wait<NST - 1>(); __syncwarp(); }
                    waited = true;
                }
                uint32_t part = 0xFFFFFFFFu;   // bit c = chunk c of this lane participates
                if (TM) {
                    if (!compressed) {         // the row was kept raw -- copy it through
                        if (active) {
                            uint32_t o[W];
#pragma unroll
                            for (int c = 0; c < W; ++c) o[c] = slot[w0 + c];
                            VecIO<W>::st(orow + (size_t)w0 * 4, o);
                        }
                        continue;
                    }
                    // S4 per row: participation bits of the lane's W chunks (W divides 32: they sit in one word), kept-bit
                    // counts, exclusive scan
                    part = active ? slot[w0 >> 5] >> (w0 & 31u) : 0u;
                    uint32_t t = 0;
#pragma unroll
                    for (int q = 0; q < W; ++q) { kk[q] = active ? (((part >> q) & 1u) ? __popc(~m[q]) : 32u) : 0u; t += kk[q]; }
                    const uint32_t incl = warp_inclusive_scan(t, lane);
                    excl = incl - t;
                    tot = __shfl_sync(0xFFFFFFFFu, incl, 31);
                }
                // ---- S5: extract + deposit + OR
                uint32_t q = head_bits + carry + excl;
                uint32_t o[W];
#pragma unroll
                for (int c = 0; c < W; ++c) {
                    uint32_t word = b[c];
                    if (kk[c]) {
                        const uint32_t wq = q >> 5;
                        const uint32_t x = __funnelshift_r(slot[wq], slot[wq + 1], q & 31u);
                        if (TM && !((part >> c) & 1u)) word = x;              // non-participating chunk: all 32 bits
                        else word |= deposit_runs(x, ~m[c]);
                        q += kk[c];
                    }
                    o[c] = word;
                }
                // ---- S6
                if (active) {
                    if (MODE == MODE_ROWS && P.keep_l2) VecIO<W>::st_keep(orow + (size_t)w0 * 4, o);
                    else VecIO<W>::st(orow + (size_t)w0 * 4, o);
                }
                carry += tot;
            }
            ++seq_d;
            __syncwarp();   // every lane is done with the slot before a later fetch overwrites it
        }
        if (FETCH == FETCH_LSU) cp_async_wait<0>();
    }
}

// ------------------------------------------------------------------------------------------------ ordering pre-pass
// Random gathers over a multi-GB host store are bound by address translation, not by the link, unless the rows in
// flight are close in the store (measured: DESIGN.md section 6).  A counting sort by coarse store region gives the
// kernel a processing order with that locality; out[] positions are unchanged.
// `list` (optional) restricts the pass to the batch positions list[0..*n_dev) (the representatives after de-duplication).
__global__ void ibp_bucket_hist(const int64_t* __restrict__ ids, const int32_t* __restrict__ list, const uint32_t* __restrict__ n_dev,
                                int64_t n, uint32_t shift, uint32_t nb, uint32_t* __restrict__ cnt) {
    if (n_dev) n = *n_dev;
    for (int64_t j = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; j < n; j += (int64_t)gridDim.x * blockDim.x) {
        const int64_t i = list ? list[j] : j;
        const uint64_t bk = (uint64_t)ids[i] >> shift;
        atomicAdd(&cnt[bk < nb ? bk : nb - 1], 1u);
    }
}
// Exclusive scan in place, one CTA of 1024 threads.  cnt has nb_pad entries (a multiple of 4096, zero beyond nb): warp w owns
// the contiguous segment [w*nb_pad/32, (w+1)*nb_pad/32), lanes read consecutive uint4 (coalesced), two passes (segment
// totals, then the scan proper with the next vector prefetched).
__global__ void __launch_bounds__(1024) ibp_bucket_scan(uint32_t* cnt, uint32_t nb_pad) {
    __shared__ uint32_t wsum[32];
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    const uint32_t per_warp = nb_pad / 32, iters = per_warp / 128;
    uint4* seg = (uint4*)(cnt + (size_t)wid * per_warp) + lane;
    uint32_t s = 0;
    for (uint32_t it = 0; it < iters; ++it) { const uint4 v = seg[it * 32]; s += v.x + v.y + v.z + v.w; }
#pragma unroll
    for (int d = 16; d; d >>= 1) s += __shfl_xor_sync(0xFFFFFFFFu, s, d);
    if (lane == 0) wsum[wid] = s;
    __syncthreads();
    if (wid == 0) { const uint32_t v = wsum[lane]; wsum[lane] = warp_inclusive_scan(v, lane) - v; }
    __syncthreads();
    uint32_t run = wsum[wid];
    uint4 v = iters ? seg[0] : make_uint4(0, 0, 0, 0);
    for (uint32_t it = 0; it < iters; ++it) {
        const uint4 nxt = it + 1 < iters ? seg[(it + 1) * 32] : make_uint4(0, 0, 0, 0);
        const uint32_t t = v.x + v.y + v.z + v.w;
        const uint32_t incl = warp_inclusive_scan(t, lane);
        uint32_t e = run + incl - t;
        uint4 o;
        o.x = e; e += v.x; o.y = e; e += v.y; o.z = e; e += v.z; o.w = e;
        seg[it * 32] = o;
        run += __shfl_sync(0xFFFFFFFFu, incl, 31);
        v = nxt;
    }
}
__global__ void ibp_bucket_scatter(const int64_t* __restrict__ ids, const int32_t* __restrict__ list, const uint32_t* __restrict__ n_dev,
                                   int64_t n, uint32_t shift, uint32_t nb, uint32_t* __restrict__ cursor, int32_t* __restrict__ order) {
    if (n_dev) n = *n_dev;
    for (int64_t j = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; j < n; j += (int64_t)gridDim.x * blockDim.x) {
        const int64_t i = list ? list[j] : j;
        const uint64_t bk = (uint64_t)ids[i] >> shift;
        const uint32_t pos = atomicAdd(&cursor[bk < nb ? bk : nb - 1], 1u);
        order[pos] = (int32_t)i;
    }
}

// shift such that one bucket covers about `target` bytes of the store, and at most 2^20 buckets
static void bucket_shape(uint64_t n_rows, uint64_t store_bytes, uint64_t target, uint32_t* shift, uint32_t* nb) {
    const double bytes_per_row = (double)std::max<uint64_t>(store_bytes, 1) / (double)std::max<uint64_t>(n_rows, 1);
    uint32_t s = 0;
    while (s < 40 && (double)(1ull << s) * bytes_per_row < (double)target) ++s;
    while (((n_rows - 1) >> s) + 1 > (1u << 18)) ++s;
    *shift = s;
    *nb = (uint32_t)(((n_rows - 1) >> s) + 1);
}

// ------------------------------------------------------------------------------------------------ de-duplication
// Skewed batches (DLRM lookups, Zipf) repeat ids; a repeated row need not cross PCIe twice.  Pass 1 claims one
// representative position per distinct id in an open-addressing table (64-bit entries: id in the high word, the winner's
// batch position in the low word; one CAS per id, none when the id is already there) and appends the winners to a work
// list.  The decode kernel then runs over the work list only, and pass 3 copies each representative's decoded row
// (HBM -> HBM) to the positions of its repeats.  Output is identical to the plain path.
__global__ void ibp_dedup_insert(const int64_t* __restrict__ ids, int64_t n, unsigned long long* __restrict__ table, uint32_t mask,
                                 int32_t* __restrict__ rep, int32_t* __restrict__ uniq, uint32_t* __restrict__ n_uniq,
                                 uint32_t* __restrict__ cnt, uint32_t shift, uint32_t nb) {
    const int lane = threadIdx.x & 31;
    // warp-uniform trip count, so that the winners of a warp can claim their work-list slots with ONE atomicAdd on the shared
    // counter (a batch has ~10^5 winners: one same-address atomic each was the longest chain of this kernel)
    for (int64_t base = (blockIdx.x * (int64_t)blockDim.x + threadIdx.x) - lane; base < n; base += (int64_t)gridDim.x * blockDim.x) {
        const int64_t i = base + lane;
        bool won = false;
        if (i < n) {
            const uint64_t key = (uint64_t)ids[i];
            uint32_t slot = (uint32_t)((key * 0x9E3779B97F4A7C15ull) >> 32) & mask;
            const unsigned long long mine = ((key + 1) << 32) | (uint32_t)i;     // 0 = empty slot
            int32_t r;
            for (;;) {
                unsigned long long cur = table[slot];
                if (cur == 0ull) cur = atomicCAS(&table[slot], 0ull, mine);
                if (cur == 0ull) {
                    r = (int32_t)i;
                    won = true;
                    if (cnt) { const uint64_t bk = key >> shift; atomicAdd(&cnt[bk < nb ? bk : nb - 1], 1u); }   // locality histogram
                    break;
                }
                if ((cur >> 32) == key + 1) { r = (int32_t)(uint32_t)cur; break; }
                slot = (slot + 1) & mask;
            }
            rep[i] = r;
        }
        const uint32_t winners = __ballot_sync(0xFFFFFFFFu, won);
        if (winners) {
            uint32_t first = 0;
            if (lane == __ffs(winners) - 1) first = atomicAdd(n_uniq, (uint32_t)__popc(winners));
            first = __shfl_sync(0xFFFFFFFFu, first, __ffs(winners) - 1);
            if (won) uniq[first + __popc(winners & ((1u << lane) - 1u))] = (int32_t)i;
        }
    }
}
// LPR lanes per row (a power of two, 16 bytes per lane and trip): a 256-byte row keeps half a warp busy, so a warp copies two.
template <int LPR>
__global__ void ibp_dedup_copy(const int32_t* __restrict__ rep, int64_t n, uint32_t row_bytes, uint8_t* __restrict__ out) {
    constexpr int RPW = 32 / LPR;
    const int lane = threadIdx.x & 31, sub = lane / LPR, sl = lane % LPR, wpc = blockDim.x >> 5;
    for (int64_t i = ((int64_t)blockIdx.x * wpc + (threadIdx.x >> 5)) * RPW + sub; i < n; i += (int64_t)gridDim.x * wpc * RPW) {
        const int32_t r = rep[i];
        if (r == (int32_t)i) continue;
        const uint4* src = (const uint4*)(out + (uint64_t)r * row_bytes);
        uint4* dst = (uint4*)(out + (uint64_t)i * row_bytes);
        if (row_bytes % 16 == 0) {
            for (uint32_t v = sl; v < row_bytes / 16; v += LPR) {
                const uint4 t = src[v];
                asm volatile("st.global.cs.v4.b32 [%0], {%1,%2,%3,%4};" ::"l"(dst + v), "r"(t.x), "r"(t.y), "r"(t.z), "r"(t.w) : "memory");
            }
        } else {
            for (uint32_t v = sl; v < row_bytes / 4; v += LPR) ((uint32_t*)dst)[v] = ((const uint32_t*)src)[v];
        }
    }
}

// Pre-passes of a random gather, in one workspace and one memset: de-duplication (optional), then the locality order
// (optional) of the surviving positions.  Outputs: list/n_list = processing order (device pointers into the workspace; n_list
// is nullptr when the count is n), rep = representative position of every id (dedup only).  The caller frees ws on the stream.
struct RowPrepass {
    void* ws = nullptr;
    int32_t* rep = nullptr;
    const int32_t* list = nullptr;
    const uint32_t* n_list = nullptr;
};

static ibp_status rows_prepass(const int64_t* ids_dev, int64_t n, bool dedup, bool order, uint64_t n_ids_space, uint64_t store_bytes,
                               int sm_count, cudaStream_t st, RowPrepass* R) {
    uint32_t shift = 0, nb = 0, nb_pad = 0, cap = 0;
    if (order) {
        bucket_shape(n_ids_space, store_bytes, 256ull << 10, &shift, &nb);   // about 256 KB of the store per bucket
        nb_pad = (nb + 4095u) / 4096u * 4096u;
    }
    if (dedup) { cap = 1024; while ((uint64_t)cap < 2ull * (uint64_t)n) cap <<= 1; }
    const size_t cnt_bytes = (size_t)nb_pad * 4, tab_bytes = (size_t)cap * 8, idx_bytes = ((size_t)n * 4 + 255) / 256 * 256;
    const size_t zero_bytes = 256 + cnt_bytes + tab_bytes;
    uint8_t* ws = nullptr;
    IBP_CUDA(cudaMallocAsync((void**)&ws, zero_bytes + (dedup ? 2 : 0) * idx_bytes + (order ? idx_bytes : 0), st));
    R->ws = ws;
    IBP_CUDA(cudaMemsetAsync(ws, 0, zero_bytes, st));
    uint32_t* n_uniq = (uint32_t*)ws;
    uint32_t* cnt = order ? (uint32_t*)(ws + 256) : nullptr;
    unsigned long long* table = (unsigned long long*)(ws + 256 + cnt_bytes);
    uint8_t* idx = ws + zero_bytes;
    const int thr = 256, blocks = (int)std::min<int64_t>((n + thr - 1) / thr, (int64_t)sm_count * 8);
    const int32_t* list = nullptr;
    const uint32_t* n_list = nullptr;
    if (dedup) {
        R->rep = (int32_t*)idx;
        int32_t* uniq = (int32_t*)(idx + idx_bytes);
        idx += 2 * idx_bytes;
        ibp_dedup_insert<<<blocks, thr, 0, st>>>(ids_dev, n, table, cap - 1, R->rep, uniq, n_uniq, cnt, shift, nb);
        list = uniq; n_list = n_uniq;
    }
    if (order) {
        int32_t* ord = (int32_t*)idx;
        if (!dedup) ibp_bucket_hist<<<blocks, thr, 0, st>>>(ids_dev, nullptr, nullptr, n, shift, nb, cnt);
        ibp_bucket_scan<<<1, 1024, 0, st>>>(cnt, nb_pad);
        ibp_bucket_scatter<<<blocks, thr, 0, st>>>(ids_dev, list, n_list, n, shift, nb, cnt, ord);
        list = ord;
    }
    IBP_CUDA(cudaGetLastError());
    R->list = list;
    R->n_list = n_list;
    return IBP_OK;
}

static ibp_status make_order(const int64_t* ids_dev, int64_t n, uint64_t n_ids_space, uint64_t store_bytes, cudaStream_t st,
                             int32_t** order_out, void** ws_out) {
    RowPrepass R;
    ibp_status s = rows_prepass(ids_dev, n, false, true, n_ids_space, store_bytes, ibp_sm_count_current(), st, &R);
    *order_out = (int32_t*)R.list;
    *ws_out = R.ws;
    return s;
}

// ------------------------------------------------------------------------------------------------ launch
// The grid is persistent: at most as many CTAs as are resident at once, so that the units in flight form one contiguous
// window of the (locality-ordered) unit list; a larger grid with a grid-stride loop would interleave far-apart windows.
template <int W, int NST, int MODE, int FETCH, bool TM = false, bool CACHE = false>
static ibp_status launch_one(const DecodeParams& P, int64_t blocks_needed, int64_t max_ctas, int sm_count, int wpc, size_t smem, cudaStream_t st) {
    auto kern = ibp_decode_kernel<W, NST, MODE, FETCH, TM, CACHE>;
    static unsigned long long smem_optin_done = 0;
    if (smem > 48 * 1024) IBP_CUDA(ibp_optin_max_smem(kern, &smem_optin_done));
    int occ = 0;
    IBP_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kern, wpc * 32, smem));
    // random rows: at most 2 CTAs per SM (1 for rows of a line or more, see gather_rows) keep enough reads in flight for the link;
    // more only widens the window of store pages touched at once (measured: DLRM 0.716 -> 0.685 ms, GNN 1.388 -> 1.375 ms per batch)
    if (MODE == MODE_ROWS) occ = std::min(occ, P.occ_cap ? (int)P.occ_cap : 2);
    int64_t blocks = std::min<int64_t>(blocks_needed, (int64_t)std::max(occ, 1) * sm_count);
    if (max_ctas) blocks = std::min<int64_t>(blocks, max_ctas);
    kern<<<(int)blocks, wpc * 32, smem, st>>>(P);
    IBP_CUDA(cudaGetLastError());
    return IBP_OK;
}

static int pick_W(uint32_t row_bytes) {
    if (row_bytes % 16 == 0 && row_bytes >= 512) return 4;
    if (row_bytes % 8 == 0 && row_bytes >= 256) return 2;
    return 1;
}

static ibp_status launch_decode(ibp_handle* h, DecodeParams& P, int mode, cudaStream_t st) {
    if (P.n_units <= 0) return IBP_OK;
    const int W = pick_W(h->p.row_bytes);
    // Rows in flight.  A locality-ordered gather of line-sized rows is fastest with about 415 KB of packed bytes in flight over the
    // whole GPU, spread over as many warps as one CTA per SM offers -- less starves the link, more only queues behind it (measured,
    // two repetitions each on one box: GNN, 252-byte rows on average, 100 CTAs x 8 warps x 2 rows = 1,600 rows: 1.348 ms, against
    // 1.363 with 1,184 rows, 1.372 with 2,368 and 1.41 with 4,736; thresholded GNN, 213 bytes, 125 CTAs x 2 = 2,000 rows: 1.295 ms
    // against 1.321 with 2,368; DLRM, 128 bytes, 100 CTAs x 4 = 3,200 rows: 0.626 ms against 0.632 with 2,368 and 0.637 with
    // 4,736).  So: rows = 415 KB / average stored row; rows per warp = the smallest of 1, 2, 4 that fits them into one CTA per SM;
    // CTAs = rows / (warps per CTA x rows per warp).  Unordered gathers, small rows and host outputs keep two rows per warp.
    int nst = 4;
    int wpc = h->warps_per_cta ? (int)h->warps_per_cta : 8;
    int64_t auto_ctas = 0;
    if (mode == MODE_ROWS) {
        nst = h->rows_in_flight ? h->rows_in_flight : 2;
        if (P.occ_cap == 1 && P.order && !h->rows_in_flight) {
            const uint64_t avg = std::max<uint64_t>(1, h->packed_bytes_rows / std::max<uint64_t>(1, h->p.n_rows));
            const uint64_t rows = std::max<uint64_t>(1, 415000ull / avg), max_warps = (uint64_t)h->sm_count * (uint64_t)wpc;
            nst = 1;
            while (nst < 4 && rows / (uint64_t)nst > max_warps) nst *= 2;
            auto_ctas = (int64_t)std::max<uint64_t>(1, (rows / (uint64_t)nst + (uint64_t)wpc - 1) / (uint64_t)wpc);
        }
    }
    P.n_pass = (h->n_words + 32 * W - 1) / (32 * W);
    P.slot_bytes = ((h->max_stride + 15u) / 16u) * 16u + 48u;   // 16-byte head + tail cover + one spare word
    P.slot_bytes = (P.slot_bytes + 127u) / 128u * 128u;
    while (wpc > 1 && (size_t)wpc * nst * (P.slot_bytes + 8) > 200 * 1024) wpc >>= 1;
    const int64_t max_ctas = h->max_ctas ? (int64_t)h->max_ctas : auto_ctas;
    const size_t smem = (size_t)wpc * nst * (P.slot_bytes + 8);   // rings + one mbarrier per slot
    const int fetch = h->fetch_mode;
    if (smem > 220 * 1024) { ibp_set_error("packed rows of %u bytes do not fit the shared-memory ring", h->max_stride); return IBP_ERR_UNSUPPORTED; }
    const int64_t blocks = (P.n_units + wpc - 1) / wpc;
#define IBP_LAUNCH(W_, NST_, MODE_)                                                                                   \
    if (MODE_ == MODE_ROWS && P.cmap) {                                                                                \
        if (h->thresholded) return launch_one<W_, NST_, MODE_ROWS, FETCH_TMA, true, true>(P, blocks, max_ctas, h->sm_count, wpc, smem, st); \
        return launch_one<W_, NST_, MODE_ROWS, FETCH_TMA, false, true>(P, blocks, max_ctas, h->sm_count, wpc, smem, st); \
    }                                                                                                                  \
    if (h->thresholded) return launch_one<W_, NST_, MODE_, FETCH_TMA, true>(P, blocks, max_ctas, h->sm_count, wpc, smem, st); \
    return fetch == FETCH_TMA ? launch_one<W_, NST_, MODE_, FETCH_TMA>(P, blocks, max_ctas, h->sm_count, wpc, smem, st) \
                              : launch_one<W_, NST_, MODE_, FETCH_LSU>(P, blocks, max_ctas, h->sm_count, wpc, smem, st)
#define IBP_BY_W(NST_, MODE_)                        \
    switch (W) {                                     \
        case 4: IBP_LAUNCH(4, NST_, MODE_);          \
        case 2: IBP_LAUNCH(2, NST_, MODE_);          \
        default: IBP_LAUNCH(1, NST_, MODE_);         \
    }
    if (mode == MODE_ROWS) {
        if (nst == 1) { IBP_BY_W(1, MODE_ROWS) }
        if (nst == 2) { IBP_BY_W(2, MODE_ROWS) }
        IBP_BY_W(4, MODE_ROWS)
    }
    if (mode == MODE_SPANS) { IBP_BY_W(4, MODE_SPANS) }
    IBP_BY_W(4, MODE_STRIDED)
#undef IBP_BY_W
#undef IBP_LAUNCH
}

static void fill_common(const ibp_handle* h, DecodeParams& P) {
    memset(&P, 0, sizeof P);
    P.meta = h->meta_dev;
    P.gtab = h->gtab_dev;
    P.row_stride_strided = h->row_stride_strided;
    P.row_bytes = h->p.row_bytes;
    P.n_words = h->n_words;
    P.group_param = h->p.group_param;
    P.strided = h->p.group_kind == IBP_GROUP_STRIDED;
    P.group_shift = 0xFFFFFFFFu;
    if ((h->p.group_param & (h->p.group_param - 1)) == 0) { uint32_t s = 0; while ((1u << s) < h->p.group_param) ++s; P.group_shift = s; }
    P.row_off = h->row_off_dev;
    P.row_flag = h->row_flag_dev;
    P.row_size = h->row_size_dev;
    P.slot16 = h->slot_layout ? h->slot_bytes / 16 : 0;
}

// ------------------------------------------------------------------------------------------------ stream launch
// Contiguous runs of rows (spans of blocked groups, whole ranges of either kind) through the TMA producer/consumer
// pipeline of ibp_stream.cuh.  `packed` is the device-visible address of byte `bias` of the packed store.
template <int W, int NS, int NSEG, bool STAGED = false>
static ibp_status launch_stream_one(const StreamBatch<NSEG>& B, int64_t total_chunks, uint32_t grid_multiple, int64_t max_ctas, int sm_count,
                                    size_t smem, cudaStream_t st, uint32_t grid_min = 1) {
    constexpr int NW = 8;
    auto kern = ibp_stream_kernel<W, NS, NW, NSEG, STAGED>;
    static unsigned long long smem_optin_done = 0;
    if (smem > 48 * 1024) IBP_CUDA(ibp_optin_max_smem(kern, &smem_optin_done));
    int occ = 0;
    IBP_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kern, (NW + 1) * 32, smem));
    int64_t blocks = std::min<int64_t>(total_chunks, (int64_t)std::max(occ, 1) * sm_count);
    if (max_ctas) blocks = std::min<int64_t>(blocks, max_ctas);
    if (grid_multiple > 1) blocks = std::max<int64_t>(grid_multiple, blocks / grid_multiple * grid_multiple);   // one tile block per CTA
    blocks = std::max<int64_t>(blocks, grid_min);                                                               // every tile block has a CTA
    kern<<<(int)blocks, (NW + 1) * 32, smem, st>>>(B);
    IBP_CUDA(cudaGetLastError());
    return IBP_OK;
}

// Chunk geometry of one contiguous run (or of n_spans spans) for the stream kernel.  `allow_tile_blocks`: resident decode of a
// strided table may use tile-block chunks when the grid will have at least one CTA per tile block.
static void stream_geometry(const ibp_handle* h, const uint8_t* packed, uint64_t bias, const int64_t* ids_dev, int64_t n_spans,
                            int64_t first_row, int64_t span_rows, void* out_dev, bool allow_tile_blocks, StreamParams& P, bool allow_staged = false) {
    const int W = pick_W(h->p.row_bytes);
    const uint32_t NW = 8;
    memset(&P, 0, sizeof P);
    P.store = packed; P.bias = bias;
    P.meta = h->meta_dev; P.mvtab = h->mvtab_dev; P.gtab = h->gtab_dev;
    P.ids = ids_dev; P.out = (uint8_t*)out_dev;
    P.first_row = first_row; P.span_rows = span_rows;
    P.row_stride_strided = h->row_stride_strided;
    P.row_bytes = h->p.row_bytes; P.n_words = h->n_words;
    P.n_pass = (h->n_words + 32 * W - 1) / (32 * W);
    P.group_param = h->p.group_param;
    P.group_shift = 0xFFFFFFFFu;
    if ((h->p.group_param & (h->p.group_param - 1)) == 0) { uint32_t sft = 0; while ((1u << sft) < h->p.group_param) ++sft; P.group_shift = sft; }
    P.strided = h->p.group_kind == IBP_GROUP_STRIDED;
    P.fast_rows = h->p.align_bytes >= 4 && ((uintptr_t)packed & 3u) == 0;
    const uint64_t G = h->p.group_param;
    uint64_t need;                                   // bytes one stage must hold
    if (!P.strided) {
        // piece = rows one warp decodes with the group's Mask/Bitval, offsets and expand masks in registers: the longer, the
        // better that set-up amortises (DLRM, 128-byte packed rows: 16 -> 64 rows per piece = 0.57 -> 0.78 of the HBM peak),
        // as long as a chunk still holds one piece per consumer warp and two stages fit (GNN, 320-byte rows: stays at 16)
        const uint64_t stride = std::max<uint32_t>(h->max_stride, 16u);
        uint32_t Umax = 16;
        uint64_t capb = 48ull * 1024;
        for (uint32_t u = 32; u <= 64; u <<= 1)
            if (G >= u && G % u == 0 && (uint64_t)NW * u * stride <= 64ull * 1024) { Umax = u; capb = 64ull * 1024; }
        uint32_t U = (uint32_t)std::min<uint64_t>(G, Umax);
        if (G % U) U = Umax;
        uint64_t rc = std::min<uint64_t>((uint64_t)NW * U, capb / stride);
        rc = std::max<uint64_t>(rc, 1);
        if (rc >= U) rc = rc / U * U; else U = (uint32_t)rc;
        rc = (uint64_t)std::min<int64_t>((int64_t)rc, span_rows);
        P.rows_per_chunk = (uint32_t)rc;
        P.piece_rows = U;
        need = rc * h->max_stride + (rc / G + 2) * 128 + 64;
        P.chunks_per_span = (uint32_t)((span_rows + (int64_t)rc - 1) / (int64_t)rc);
        // staged metadata (ibp_stream.cuh): [descriptor 32 B][group entries][Mask/Bitval of the chunk's groups] in front of the bytes
        const uint64_t groups_max = rc < 2 ? 1 : (rc - 2) / G + 2;
        const uint64_t meta_off = (32 + groups_max * 16 + 127) / 128 * 128, aux = meta_off + groups_max * 2 * h->p.row_bytes;
        // Only for small groups (at least eight per chunk: KV pages of 16 rows), where every piece needs a fresh Mask/Bitval and the
        // consumers' dependent global loads were the top stall (resident KV 0.80 -> 0.83 of the HBM peak); with groups of 128 / 256
        // rows a warp keeps its prepared group across pieces and the extra stage traffic costs more than it saves (measured: GNN
        // 0.87 -> 0.84, DLRM 0.84 -> 0.81), so those keep the consumer-side loads.
        if (P.n_pass == 1 && P.fast_rows && h->p.row_bytes % 16 == 0 && aux <= 12ull * 1024 && G * 8 <= rc && allow_staged) {
            P.aux_bytes = (uint32_t)((aux + 127) / 128 * 128);
            P.aux_meta_off = (uint32_t)meta_off;
            need += P.aux_bytes;
        }
    } else if (allow_tile_blocks && P.n_pass == 1 && P.fast_rows && !ids_dev && n_spans == 1) {
        // resident decode of a strided table: tile-block chunks (ibp_stream.cuh).  A whole-row chunk holds only 2-7 matrix rows
        // of the 7B shapes, so every warp would re-prepare a tile (Mask/Bitval, offsets, expand masks) for a handful of rows;
        // here a CTA keeps one block of NW tiles for all its chunks and prepares once.  The source is HBM, so the shorter
        // contiguous reads (one block of one matrix row per bulk copy) cost nothing; the host-store path keeps whole rows.
        const uint64_t n_tiles = h->n_groups;                      // min(S, rows): the group table ends there
        const uint32_t n_tb = (uint32_t)((n_tiles + NW - 1) / NW);
        P.n_tiles = (uint32_t)n_tiles;
        uint64_t max_len = 0;
        for (uint32_t tb = 0; tb < n_tb; ++tb) {
            const IbpGroupEntry& e0 = h->gtab[(uint64_t)tb * NW];
            const IbpGroupEntry& e1 = h->gtab[std::min<uint64_t>(n_tiles, (uint64_t)tb * NW + NW) - 1];
            max_len = std::max<uint64_t>(max_len, e1.base + e1.stride - e0.base);
        }
        const uint64_t pitch = (max_len + 31 + 15) / 16 * 16;
        const int64_t n_mrows = (span_rows + (int64_t)G - 1) / (int64_t)G;
        uint64_t rc = std::max<uint64_t>(1, std::min<uint64_t>(32, (48ull * 1024) / pitch));
        rc = (uint64_t)std::min<int64_t>((int64_t)rc, n_mrows);
        P.rows_per_chunk = (uint32_t)rc;
        P.piece_rows = (uint32_t)rc;
        P.n_tile_blocks = n_tb;
        P.tb_pitch = (uint32_t)pitch;
        need = rc * pitch + 64;
        P.chunks_per_span = (uint32_t)(((n_mrows + (int64_t)rc - 1) / (int64_t)rc) * n_tb);
    } else {
        const uint64_t rs = h->row_stride_strided;
        const uint64_t cap = rs > 8192 ? 64ull * 1024 : 48ull * 1024;
        uint64_t rc = std::max<uint64_t>(1, (cap - 64) / std::max<uint64_t>(rs, 16));
        const int64_t n_mrows = (span_rows + (int64_t)G - 1) / (int64_t)G;
        rc = (uint64_t)std::min<int64_t>((int64_t)rc, n_mrows);
        P.rows_per_chunk = (uint32_t)rc;
        P.piece_rows = (uint32_t)rc;
        need = rc * rs + 64;
        P.chunks_per_span = (uint32_t)((n_mrows + (int64_t)rc - 1) / (int64_t)rc);
    }
    P.stage_bytes = (uint32_t)((need + 127) / 128 * 128);
    P.n_chunks = n_spans * (int64_t)P.chunks_per_span;
}

// Grid limit of a contiguous-run launch.  A stream that reads the HOST store is bound by the link, which 24 CTAs already saturate
// (measured: a weight layer 62.77 GB/s with 24, 48, 64, 96 CTAs or the full persistent grid; KV spans 63.2 with 32, 64 or all), so
// unless ibp_configure says otherwise it takes 48 CTAs and leaves the other SMs to whoever consumes the rows ("We reserved
// only 64 SMs for decompression"): overlapped with a GEMM on the previous layer, 8 layers take 68.6 ms instead of 102.5 ms with the
// full grid (ideal 64.5).  Resident decode (HBM source) is bound by HBM and the integer pipe and keeps the whole GPU.
static inline int64_t stream_ctas(const ibp_handle* h, bool hbm_source) {
    return h->max_ctas ? (int64_t)h->max_ctas : (hbm_source ? 0 : 48);
}

static ibp_status launch_stream(ibp_handle* h, const uint8_t* packed, uint64_t bias, const int64_t* ids_dev, int64_t n_spans,
                                int64_t first_row, int64_t span_rows, void* out_dev, cudaStream_t st, bool resident = false) {
    if (n_spans <= 0 || span_rows <= 0) return IBP_OK;
    const int64_t max_ctas = stream_ctas(h, resident);
    const int W = pick_W(h->p.row_bytes);
    StreamBatch<1> B;
    memset(&B, 0, sizeof B);
    StreamParams& P = B.seg[0];
    const bool tile_ok = resident && (!h->max_ctas || h->max_ctas >= (h->n_groups + 7) / 8);
    stream_geometry(h, packed, bias, ids_dev, n_spans, first_row, span_rows, out_dev, tile_ok, P, true);
    B.n_seg = 1;
    B.stage_bytes = P.stage_bytes;
    const int ns = P.stage_bytes > 40 * 1024 ? 2 : 3;
    const size_t smem = (size_t)ns * P.stage_bytes + (size_t)ns * 16;
    if (smem > 220 * 1024) { ibp_set_error("packed rows of %u bytes do not fit the shared-memory stages", h->max_stride); return IBP_ERR_UNSUPPORTED; }
#define IBP_STREAM(W_)                                                                                             \
    if (P.aux_bytes)                                                                                               \
        return ns == 2 ? launch_stream_one<W_, 2, 1, true>(B, P.n_chunks, P.n_tile_blocks, max_ctas, h->sm_count, smem, st) \
                       : launch_stream_one<W_, 3, 1, true>(B, P.n_chunks, P.n_tile_blocks, max_ctas, h->sm_count, smem, st); \
    return ns == 2 ? launch_stream_one<W_, 2, 1>(B, P.n_chunks, P.n_tile_blocks, max_ctas, h->sm_count, smem, st) \
                   : launch_stream_one<W_, 3, 1>(B, P.n_chunks, P.n_tile_blocks, max_ctas, h->sm_count, smem, st)
    switch (W) {
        case 4: IBP_STREAM(4);
        case 2: IBP_STREAM(2);
        default: IBP_STREAM(1);
    }
#undef IBP_STREAM
}

// Thresholded-mode contiguous runs through ibp_stream_t_kernel.  Returns IBP_ERR_UNSUPPORTED (without setting an error
// the caller would report) when the shape does not fit: the caller then uses the per-row kernel.
template <int W, int NS, bool RUNS>
static ibp_status launch_stream_t_one(const StreamTParams& P, int64_t max_ctas, int sm_count, size_t smem, cudaStream_t st) {
    constexpr int NW = 8;
    auto kern = ibp_stream_t_kernel<W, NS, NW, RUNS>;
    static unsigned long long smem_optin_done = 0;
    if (smem > 48 * 1024) IBP_CUDA(ibp_optin_max_smem(kern, &smem_optin_done));
    int occ = 0;
    IBP_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kern, (NW + 1) * 32, smem));
    int64_t blocks = std::min<int64_t>(P.n_chunks, (int64_t)std::max(occ, 1) * sm_count);
    if (max_ctas) blocks = std::min<int64_t>(blocks, max_ctas);
    kern<<<(int)blocks, (NW + 1) * 32, smem, st>>>(P);
    IBP_CUDA(cudaGetLastError());
    return IBP_OK;
}

template <int LPR, int NS, int NR>
static ibp_status launch_stream_t2_one(const StreamTParams& P, int64_t max_ctas, int sm_count, size_t smem, cudaStream_t st) {
    constexpr int NW = 8;
    auto kern = ibp_stream_t2_kernel<LPR, NS, NW, NR>;
    static unsigned long long smem_optin_done = 0;
    if (smem > 48 * 1024) IBP_CUDA(ibp_optin_max_smem(kern, &smem_optin_done));
    int occ = 0;
    IBP_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kern, (NW + 1) * 32, smem));
    int64_t blocks = std::min<int64_t>(P.n_chunks, (int64_t)std::max(occ, 1) * sm_count);
    if (max_ctas) blocks = std::min<int64_t>(blocks, max_ctas);
    kern<<<(int)blocks, (NW + 1) * 32, smem, st>>>(P);
    IBP_CUDA(cudaGetLastError());
    return IBP_OK;
}

static bool stream_t_fits(const ibp_handle* h) {
    const int W = pick_W(h->p.row_bytes);
    if ((h->n_words + 32 * W - 1) / (32 * W) != 1) return false;                       // single-pass rows only
    if (h->p.group_kind == IBP_GROUP_STRIDED && (uint64_t)h->p.group_param * h->max_stride + 64 > 96ull * 1024) return false;
    return true;
}

static ibp_status launch_stream_t(ibp_handle* h, const uint8_t* packed, uint64_t bias, const int64_t* ids_dev, int64_t n_spans,
                                  int64_t first_row, int64_t span_rows, void* out_dev, cudaStream_t st, bool resident = false) {
    if (n_spans <= 0 || span_rows <= 0) return IBP_OK;
    const int64_t max_ctas = stream_ctas(h, resident);
    const int W = pick_W(h->p.row_bytes);
    const uint32_t NW = 8;
    StreamTParams P;
    memset(&P, 0, sizeof P);
    P.store = packed; P.bias = bias;
    P.meta = h->meta_dev; P.row_off = h->row_off_dev; P.row_flag = h->row_flag_dev;
    P.ids = ids_dev; P.out = (uint8_t*)out_dev;
    P.first_row = first_row; P.span_rows = span_rows;
    P.row_bytes = h->p.row_bytes; P.n_words = h->n_words;
    P.group_param = h->p.group_param;
    P.group_shift = 0xFFFFFFFFu;
    if ((h->p.group_param & (h->p.group_param - 1)) == 0) { uint32_t sft = 0; while ((1u << sft) < h->p.group_param) ++sft; P.group_shift = sft; }
    P.strided = h->p.group_kind == IBP_GROUP_STRIDED;
    const uint64_t stride = h->max_stride;                                             // a raw row: the largest stored row
    uint64_t per;                                                                      // consecutive rows per chunk
    // rows of 128 / 256 / 512 bytes (every BASELINE workload): the sub-warp kernel (ibp_stream_t.cuh, ibp_stream_t2_kernel)
    const uint32_t lpr = h->p.row_bytes % 16 == 0 ? h->p.row_bytes / 16 : 0;
    bool t2 = (lpr == 8 || lpr == 16 || lpr == 32) && h->t2_mode && !P.strided && h->p.n_rows <= 0xFFFFFFFFull;   // (32-bit row ids on its consumer side)
    if (t2) {
        // A unit (= chunk, = stage) is NW pieces, one per consumer warp; a stage holds the unit's packed bytes plus an aux region:
        // descriptor, row-offset cover, row-flag cover, Mask/Bitval of the groups the unit touches (ibp_stream_t.cuh).  Two stages
        // per CTA, three CTAs per SM: 38,144 bytes per stage.  The piece is the largest of 32 / 16 / 8 rows whose unit fits a stage
        // even when every row is stored raw, so that no chunk is ever split (256-byte rows: 16, 512-byte rows: 8); only if even
        // 8-row pieces do not fit is a chunk above a stage loaded as sub-units of split_rows rows.
        const uint64_t STAGE = 38144;
        const uint64_t G = h->p.group_param;
        auto layout = [&](uint32_t U_, uint64_t& rc_, uint64_t& cap_) {     // aux layout and data capacity of a unit of NW pieces of U_ rows
            rc_ = (uint64_t)std::min<int64_t>((int64_t)NW * U_, span_rows);
            const uint64_t off_max = ((rc_ + 1 + 3 + 3 + 3) & ~3ull) * 4, flag_max = ((rc_ / 32 + 2 + 3 + 3) & ~3ull) * 4 + 16;
            const uint64_t groups_max = rc_ < 2 ? 1 : (rc_ - 2) / G + 2, meta_max = groups_max * 2 * h->p.row_bytes;
            P.aux_flag_off = (uint32_t)(32 + off_max);                        // [descriptor 32 B][row offsets][row flags][Mask/Bitval]
            const uint64_t meta_off = (P.aux_flag_off + flag_max + 127) / 128 * 128;
            const bool stage_meta = meta_max <= 8192;                        // small groups (a Mask/Bitval pair per row or two) stay in global memory
            P.aux_meta_off = stage_meta ? (uint32_t)meta_off : 0u;
            P.aux_bytes = (uint32_t)(stage_meta ? meta_off + meta_max : meta_off);
            cap_ = STAGE - P.aux_bytes;
        };
        uint32_t U = lpr == 32 ? 16u : 32u;
        uint64_t rc = 0, data_cap = 0;
        for (;; U >>= 1) {                                                   // worst case: every row raw
            layout(U, rc, data_cap);
            if (rc * stride + 64 <= data_cap || U <= 8) break;
        }
        // Larger pieces when the rows the table actually stores are well below the raw size (GNN: 289 of 512 bytes): a unit sized
        // for the table's AVERAGE stored row with 10 % to spare amortises the per-piece work over more rows; the rare unit that
        // exceeds a stage is split.  Only when groups are long against the piece (a piece that straddles a group boundary takes the
        // slower run-by-run path) or the piece divides / is a multiple of the group.
        {
            const uint64_t avg = std::max<uint64_t>(16, (h->packed_bytes_rows + h->p.n_rows - 1) / std::max<uint64_t>(1, h->p.n_rows));
            const uint32_t gran = 2u * (32u / lpr);                          // two passes of 32/LPR rows
            for (uint32_t Ut = 32u / gran * gran; Ut > U; Ut -= gran) {
                if (!(G >= 8ull * Ut || G % Ut == 0 || Ut % G == 0)) continue;
                uint64_t rct, capt;
                layout(Ut, rct, capt);
                if (rct < (uint64_t)NW * Ut) continue;                       // short spans: keep the worst-case size
                const uint64_t split_rows = ((capt - 64) / stride) / Ut * Ut;
                if (rct * avg * 11 / 10 + 64 <= capt && split_rows >= Ut) { U = Ut; break; }
            }
            layout(U, rc, data_cap);
        }
        P.rows_per_chunk = (uint32_t)rc;
        P.piece_rows = U;
        P.stage_bytes = (uint32_t)STAGE;
        per = rc;
        if (rc * stride + 64 <= data_cap) {
            P.nsplit = 1;
        } else {
            const uint64_t split_rows = ((data_cap - 64) / stride) / U * U;
            if (split_rows == 0) t2 = false;
            else {
                P.split_rows = (uint32_t)split_rows;
                P.nsplit = (uint32_t)((rc + split_rows - 1) / split_rows);
            }
        }
    }
    if (t2) {
    } else if (!P.strided) {
        uint32_t U = 16;
        uint64_t rc = std::min<uint64_t>((uint64_t)NW * U, (48ull * 1024) / stride);
        rc = std::max<uint64_t>(rc, 1);
        if (rc < (uint64_t)NW * U) U = (uint32_t)std::max<uint64_t>(1, rc / NW);   // one piece per consumer warp (GNN: 96 rows = 8 x 12, not 6 x 16)
        if (rc >= U) rc = rc / U * U;
        rc = (uint64_t)std::min<int64_t>((int64_t)rc, span_rows);
        P.rows_per_chunk = (uint32_t)rc;
        P.piece_rows = (uint32_t)std::min<uint64_t>(U, rc);
        per = rc;
    } else {
        const uint64_t S = h->p.group_param, rs = S * stride;
        uint64_t rc = std::max<uint64_t>(1, std::min<uint64_t>(32, (48ull * 1024) / rs));
        const int64_t n_mrows = (span_rows + (int64_t)S - 1) / (int64_t)S;
        rc = (uint64_t)std::min<int64_t>((int64_t)rc, n_mrows);
        P.rows_per_chunk = (uint32_t)rc;
        P.piece_rows = (uint32_t)rc;
        per = rc * S;
    }
    if (!t2) P.stage_bytes = (uint32_t)((per * stride + 64 + 127) / 128 * 128);
    P.chunks_per_span = (uint32_t)((span_rows + (int64_t)per - 1) / (int64_t)per);
    P.n_chunks = n_spans * (int64_t)P.chunks_per_span;
    const int ns = (P.stage_bytes > 40 * 1024 || t2) ? 2 : 3;
    const size_t smem = (size_t)ns * P.stage_bytes + (size_t)ns * 16;
    if (smem > 220 * 1024) { ibp_set_error("thresholded rows of %u bytes do not fit the shared-memory stages", h->max_stride); return IBP_ERR_UNSUPPORTED; }
    if (t2) {
        const int nr = (h->max_runs >= 1 && h->max_runs <= 4) ? h->max_runs : 0;      // bf16 pairs: mantissa + sign per half = 4 runs
#define IBP_T2_NR(LPR_, NS_)                                                                              \
        switch (nr) {                                                                                     \
            case 1: return launch_stream_t2_one<LPR_, NS_, 1>(P, max_ctas, h->sm_count, smem, st);     \
            case 2: return launch_stream_t2_one<LPR_, NS_, 2>(P, max_ctas, h->sm_count, smem, st);     \
            case 3: return launch_stream_t2_one<LPR_, NS_, 3>(P, max_ctas, h->sm_count, smem, st);     \
            case 4: return launch_stream_t2_one<LPR_, NS_, 4>(P, max_ctas, h->sm_count, smem, st);     \
            default: return launch_stream_t2_one<LPR_, NS_, 0>(P, max_ctas, h->sm_count, smem, st);    \
        }
#define IBP_T2(LPR_) { IBP_T2_NR(LPR_, 2) }                                                            /* t2: always two stages */
        if (lpr == 32) { IBP_T2(32) }
        if (lpr == 16) { IBP_T2(16) }
        IBP_T2(8)
#undef IBP_T2
#undef IBP_T2_NR
    }
    const bool runs = h->max_runs >= 0 && h->max_runs <= 3;
#define IBP_STREAM_T(W_)                                                                                         \
    if (runs) return ns == 2 ? launch_stream_t_one<W_, 2, true>(P, max_ctas, h->sm_count, smem, st)           \
                             : launch_stream_t_one<W_, 3, true>(P, max_ctas, h->sm_count, smem, st);          \
    return ns == 2 ? launch_stream_t_one<W_, 2, false>(P, max_ctas, h->sm_count, smem, st)                    \
                   : launch_stream_t_one<W_, 3, false>(P, max_ctas, h->sm_count, smem, st)
    switch (W) {
        case 4: IBP_STREAM_T(4);
        case 2: IBP_STREAM_T(2);
        default: IBP_STREAM_T(1);
    }
#undef IBP_STREAM_T
}

static ibp_status check_ready(const ibp_handle* h, const char* who) {
    if (!h) { ibp_set_error("%s: null handle", who); return IBP_ERR_INVALID_ARG; }
    if (h->device < 0 || !h->meta_dev) { ibp_set_error("%s: call ibp_upload_metadata first", who); return IBP_ERR_BAD_STATE; }
    return IBP_OK;
}

// ------------------------------------------------------------------------------------------------ C ABI
ibp_status ibp_attach_device(ibp_handle* h, int device, void* cuda_stream) {
    int ndev = 0;
    IBP_CUDA(cudaGetDeviceCount(&ndev));
    if (device < 0 || device >= ndev) { ibp_set_error("ibp_upload_metadata: no CUDA device %d", device); return IBP_ERR_CUDA; }
    cudaDeviceProp prop;
    IBP_CUDA(cudaGetDeviceProperties(&prop, device));
    if (prop.major != 10) { ibp_set_error("ibp_upload_metadata: device %d is sm_%d%d; this library is built for sm_100a only", device, prop.major, prop.minor); return IBP_ERR_UNSUPPORTED; }
    IBP_CUDA(cudaSetDevice(device));
    if (h->device == device) return IBP_OK;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    if (!h->meta_dev) {
        IBP_CUDA(cudaMalloc((void**)&h->meta_dev, h->meta.size() * 4));
        IBP_CUDA(cudaMemcpyAsync(h->meta_dev, h->meta.data(), h->meta.size() * 4, cudaMemcpyHostToDevice, st));
    }
    if (!h->gtab_dev) {
        IBP_CUDA(cudaMalloc((void**)&h->gtab_dev, h->gtab.size() * sizeof(IbpGroupEntry)));
        IBP_CUDA(cudaMemcpyAsync(h->gtab_dev, h->gtab.data(), h->gtab.size() * sizeof(IbpGroupEntry), cudaMemcpyHostToDevice, st));
    }
    if (h->slot_layout && !h->row_size_dev) {
        IBP_CUDA(cudaMalloc((void**)&h->row_size_dev, std::max<size_t>(h->row_size.size(), 16)));
        IBP_CUDA(cudaMemcpyAsync(h->row_size_dev, h->row_size.data(), h->row_size.size(), cudaMemcpyHostToDevice, st));
    }
    if (h->thresholded && !h->slot_layout && !h->row_off_dev) {
        IBP_CUDA(cudaMalloc((void**)&h->row_off_dev, h->row_off.size() * 4 + 64));   // slack: the stream kernels copy 16-byte covers
        IBP_CUDA(cudaMemcpyAsync(h->row_off_dev, h->row_off.data(), h->row_off.size() * 4, cudaMemcpyHostToDevice, st));
    }
    if (h->thresholded && !h->row_flag_dev) {
        IBP_CUDA(cudaMalloc((void**)&h->row_flag_dev, h->row_flag.size() * 4 + 64));
        IBP_CUDA(cudaMemcpyAsync(h->row_flag_dev, h->row_flag.data(), h->row_flag.size() * 4, cudaMemcpyHostToDevice, st));
    }
    // expand move masks per (group, word) when the table has few groups (strided column tiles, small tables): 20 B per word
    if (!h->thresholded && !h->mvtab_dev && h->n_groups * (uint64_t)h->n_words * 20ull <= (8ull << 20)) {
        const uint64_t cells = h->n_groups * (uint64_t)h->n_words;
        IBP_CUDA(cudaMalloc((void**)&h->mvtab_dev, cells * 20));
        ibp_build_mvtab<<<(unsigned)((cells + 255) / 256), 256, 0, st>>>(h->meta_dev, h->n_words, h->n_groups, h->mvtab_dev);
        IBP_CUDA(cudaGetLastError());
    }
    IBP_CUDA(cudaStreamSynchronize(st));
    if (h->max_runs < 0) {
        // most runs of variant bits in any Mask word: at most three everywhere lets the thresholded stream kernel re-insert bits
        // run by run (2 operations per run) instead of through the five-stage expand
        int mr = 0;
        const int64_t ng = (int64_t)h->n_groups;
        const uint32_t nw = h->n_words;
#pragma omp parallel for reduction(max : mr) schedule(static)
        for (int64_t g = 0; g < ng; ++g) {
            const uint32_t* mk = &h->meta[(uint64_t)g * 2 * nw];
            for (uint32_t w = 0; w < nw; ++w) {
                const uint32_t nv = ~mk[w];
                mr = std::max(mr, __builtin_popcount(nv & ~(nv << 1)));
            }
        }
        h->max_runs = mr;
    }
    h->sm_count = prop.multiProcessorCount;
    if (h->store_kind == IBP_STORE_PINNED && !h->store_dev) {
        void* dptr = nullptr;
        IBP_CUDA(cudaHostGetDevicePointer(&dptr, h->store, 0));
        h->store_dev = (uint8_t*)dptr;
    }
    if (h->store_kind == IBP_STORE_SHARED && !h->store_dev) {
        // the shared segment: page-lock and map it for THIS process; every rank does the same with the same physical pages
        if (!h->shm_registered) {
            IBP_CUDA(cudaHostRegister(h->store, h->store_bytes, cudaHostRegisterMapped | cudaHostRegisterPortable));
            h->shm_registered = true;
        }
        void* dptr = nullptr;
        IBP_CUDA(cudaHostGetDevicePointer(&dptr, h->store, 0));
        h->store_dev = (uint8_t*)dptr;
    }
    if (h->store_kind == IBP_STORE_MANAGED_HOST) {
        // direct mapping of the host-resident pages into this GPU's page tables: accesses go over PCIe, nothing migrates
        IBP_CUDA(cudaMemAdvise(h->store, h->store_bytes, cudaMemAdviseSetAccessedBy, device));
        h->store_dev = h->store;
    }
    cudaMemPool_t pool;
    if (cudaDeviceGetDefaultMemPool(&pool, device) == cudaSuccess) {   // keep the per-call workspaces cached
        uint64_t thr = ~0ull;
        cudaMemPoolSetAttribute(pool, cudaMemPoolAttrReleaseThreshold, &thr);
    }
    (void)cudaGetLastError();
    h->device = device;
    return IBP_OK;
}

extern "C" ibp_status ibp_upload_metadata(ibp_handle* h, int device, void* cuda_stream) {
    if (!h) { ibp_set_error("ibp_upload_metadata: null handle"); return IBP_ERR_INVALID_ARG; }
    if (h->device >= 0 && h->device != device) { ibp_set_error("ibp_upload_metadata: handle already lives on device %d", h->device); return IBP_ERR_INVALID_ARG; }
    return ibp_attach_device(h, device, cuda_stream);
}

// Random row gather (index_span 1): pre-passes, decode kernel, replication of repeats.  `c` = optional compressed GPU cache.
static ibp_status gather_rows(ibp_handle* h, const ibp_cache* c, const int64_t* row_ids_dev, int64_t n, void* out_dev, cudaStream_t st,
                              bool allow_dedup = true, bool host_out = false) {
    if (n > 0x7FFFFFFF) { ibp_set_error("ibp_gather_decompress: n too large"); return IBP_ERR_INVALID_ARG; }
    DecodeParams P;
    fill_common(h, P);
    P.store = h->store_dev;
    P.ids = row_ids_dev;
    P.out = (uint8_t*)out_dev;
    P.n = n;
    P.span = 1;
    P.n_units = n;
    if (c) {
        P.cmap = c->map_dev;
        P.cmap_mask = c->map_cap - 1;
        for (int s = 0; s < 8; ++s) P.slab[s] = c->slab_dev[s];
        // A cache that holds a sizeable share of the table serves most rows from HBM slabs: those are latency-bound (map probe,
        // then the bulk copy), so every resident CTA helps (DLRM, 10 % of the rows cached: 357 -> 414 GB/s; 60 %: 361 -> 520).
        // A small cache leaves the misses in charge, and for them a wider window of store pages in flight costs more than it
        // gains (DLRM, 2 %: 314 -> 280 GB/s with 4 CTAs per SM), so the cap of the uncached gather stays.
        if (c->n_entries * 12 >= h->p.n_rows) P.occ_cap = 4;
    } else if (!host_out && h->p.n_rows && h->packed_bytes_rows / h->p.n_rows >= 96 && h->p.row_bytes <= 512) {
        // Rows of about a line or more are bound by link bytes, and ONE CTA per SM (8 warps x 2 rows in flight) already keeps the
        // link busy: measured three times each, alternating, GNN 1.371 ms with 148 CTAs against 1.383 with 296, DLRM 0.6347 against
        // 0.6378 -- and half the registers and warp slots of every SM stay free for whatever runs beside the gather.  Smaller packed
        // rows are bound by rows per second, and rows of several passes (4 KB: 2-5 % slower with one CTA) by decode latency: both keep two.
        // So does a gather whose OUTPUT is host memory (the direct path of ibp_gather_decompress_host): its warps also wait on their
        // zero-copy stores, and with fewer rows in flight the end-to-end rate drops (GNN 40 -> 33 GB/s).
        P.occ_cap = 1;
    }
    const bool dedup = allow_dedup && (h->dedup_mode == 1 || (h->dedup_mode < 0 && n >= 16384)) && n >= 2 && h->p.n_rows <= 0xFFFFFFFEull;
    // automatic: large batches over large stores are processed in store-address order (address translation, DESIGN 6).
    // Essential for the 4 KB-page pinned store, a few percent for the managed-host store -- unless repeated ids are
    // fetched one by one (dedup off on a batch with repeats), where neighbours in the order collide on the same lines.
    const bool order = h->order_mode == 1 || (h->order_mode < 0 && h->store_used > (64ull << 20) && n >= 4096);
    RowPrepass R;
    ibp_status s = IBP_OK;
    if (dedup || order) {
        s = rows_prepass(row_ids_dev, n, dedup, order, h->p.n_rows, h->store_used, h->sm_count, st, &R);
        if (s != IBP_OK) return s;
    }
    P.order = R.list;
    P.n_units_dev = R.n_list;
    P.keep_l2 = dedup;                  // the replication pass re-reads the decoded rows: keep them in L2
    s = launch_decode(h, P, MODE_ROWS, st);
    if (s == IBP_OK && dedup) {
        const uint32_t rb = h->p.row_bytes;
        const int lpr = rb >= 512 ? 32 : rb >= 256 ? 16 : rb >= 128 ? 8 : 4, rpw = 32 / lpr;
        const int blocks = (int)std::min<int64_t>((n + 8 * rpw - 1) / (8 * rpw), (int64_t)h->sm_count * 8);
        switch (lpr) {
            case 32: ibp_dedup_copy<32><<<blocks, 256, 0, st>>>(R.rep, n, rb, (uint8_t*)out_dev); break;
            case 16: ibp_dedup_copy<16><<<blocks, 256, 0, st>>>(R.rep, n, rb, (uint8_t*)out_dev); break;
            case 8: ibp_dedup_copy<8><<<blocks, 256, 0, st>>>(R.rep, n, rb, (uint8_t*)out_dev); break;
            default: ibp_dedup_copy<4><<<blocks, 256, 0, st>>>(R.rep, n, rb, (uint8_t*)out_dev); break;
        }
        if (cudaGetLastError() != cudaSuccess) { ibp_set_error("ibp_dedup_copy launch failed"); s = IBP_ERR_CUDA; }
    }
    if (R.ws) IBP_CUDA(cudaFreeAsync(R.ws, st));
    return s;
}

extern "C" ibp_status ibp_cache_gather_decompress(ibp_cache* c, const int64_t* row_ids_dev, int64_t n, void* out_dev, void* cuda_stream) {
    if (!c) { ibp_set_error("ibp_cache_gather_decompress: null cache"); return IBP_ERR_INVALID_ARG; }
    ibp_status s = check_ready(c->h, "ibp_cache_gather_decompress");
    if (s != IBP_OK) return s;
    if (n == 0) return IBP_OK;
    if (n < 0 || !row_ids_dev || !out_dev || ((uintptr_t)out_dev & 15u)) { ibp_set_error("ibp_cache_gather_decompress: bad argument (null pointer, n<0, or out not 16-byte aligned)"); return IBP_ERR_INVALID_ARG; }
    return gather_rows(c->h, c, row_ids_dev, n, out_dev, (cudaStream_t)cuda_stream);
}

extern "C" ibp_status ibp_gather_decompress(ibp_handle* h, const int64_t* row_ids_dev, int64_t n, void* out_dev, void* cuda_stream) {
    ibp_status s = check_ready(h, "ibp_gather_decompress");
    if (s != IBP_OK) return s;
    if (n == 0) return IBP_OK;
    if (n < 0 || !row_ids_dev || !out_dev || ((uintptr_t)out_dev & 15u)) { ibp_set_error("ibp_gather_decompress: bad argument (null pointer, n<0, or out not 16-byte aligned)"); return IBP_ERR_INVALID_ARG; }
    if (!h->store_dev) { ibp_set_error("ibp_gather_decompress: the packed store is not GPU-mapped (pageable store)"); return IBP_ERR_BAD_STATE; }
    cudaStream_t st = (cudaStream_t)cuda_stream;
    if (h->p.index_span == 1) return gather_rows(h, nullptr, row_ids_dev, n, out_dev, st);
    DecodeParams P;
    fill_common(h, P);
    P.store = h->store_dev;
    P.ids = row_ids_dev;
    P.out = (uint8_t*)out_dev;
    P.n = n;
    P.span = h->p.index_span;
    if (h->stream_mode && h->thresholded && !h->slot_layout && stream_t_fits(h))
        return launch_stream_t(h, h->store_dev, 0, row_ids_dev, n, 0, (int64_t)h->p.index_span, out_dev, st);
    if (h->stream_mode && !h->thresholded)
        return launch_stream(h, h->store_dev, 0, row_ids_dev, n, 0, (int64_t)h->p.index_span, out_dev, st);
    // (fallback) spans of blocked groups: R consecutive rows per warp, never crossing a group needlessly
    const uint32_t G = h->p.group_param;
    P.rows_per_unit = std::min<uint32_t>(std::min<uint32_t>(G, 16u), h->p.index_span);
    if (G % P.rows_per_unit) P.rows_per_unit = std::min<uint32_t>(16u, h->p.index_span);
    P.units_per_span = (h->p.index_span + P.rows_per_unit - 1) / P.rows_per_unit;
    P.n_units = n * (int64_t)P.units_per_span;
    return launch_decode(h, P, MODE_SPANS, st);
}

// ------------------------------------------------------------------------------------------------ gather without allocation
// ibp_gather_decompress_noalloc: the random-row gather for callers that may not allocate (CUDA graph capture, serving loops).
// The locality-order pre-pass (bucket histogram, scan, scatter: the scratch-memory kernels of gather_rows) runs in a FIXED
// device array instead of a cudaMallocAsync workspace: [n counter, 256 B][bucket counters, <= 2^18 x 4 B][order, n x 4 B].
// The array lives in every GPU context that loads the library (5.25 MB per GPU until exit).  In host code its NAME is a
// host-side stand-in, not a device address, so the address is taken with cudaGetSymbolAddress once per device, with that
// device current, and passed to the kernels like any workspace pointer.
constexpr size_t NOALLOC_CNT_BYTES = (size_t)(1u << 18) * 4;                                    // bucket_shape: at most 2^18 buckets
constexpr size_t NOALLOC_ZERO_BYTES = 256 + NOALLOC_CNT_BYTES;
constexpr size_t NOALLOC_SCRATCH_BYTES = NOALLOC_ZERO_BYTES + (size_t)IBP_NOALLOC_MAX_IDS * 4;
static __device__ __align__(256) uint8_t ibp_noalloc_scratch[NOALLOC_SCRATCH_BYTES];
constexpr int NOALLOC_MAX_DEVICES = 64;
static std::mutex g_noalloc_mu;
static uint8_t* g_noalloc_ptr[NOALLOC_MAX_DEVICES];                                             // device address of the array, per device

static ibp_status noalloc_scratch_ptr(int device, uint8_t** out) {
    int cur = -1;
    IBP_CUDA(cudaGetDevice(&cur));
    if (cur != device || device < 0 || device >= NOALLOC_MAX_DEVICES) {
        ibp_set_error("ibp_gather_decompress_noalloc: the handle's device %d must be the current device (current: %d)", device, cur);
        return IBP_ERR_BAD_STATE;
    }
    std::lock_guard<std::mutex> lk(g_noalloc_mu);
    if (!g_noalloc_ptr[device]) {
        void* p = nullptr;
        const cudaError_t e = cudaGetSymbolAddress(&p, ibp_noalloc_scratch);
        if (e != cudaSuccess || !p) {
            ibp_set_error("ibp_gather_decompress_noalloc: cudaGetSymbolAddress failed: %s", cudaGetErrorString(e));
            (void)cudaGetLastError();
            return IBP_ERR_CUDA;
        }
        g_noalloc_ptr[device] = (uint8_t*)p;
    }
    *out = g_noalloc_ptr[device];
    return IBP_OK;
}

extern "C" ibp_status ibp_gather_decompress_noalloc(ibp_handle* h, const int64_t* row_ids_dev, int64_t n, void* out_dev, void* cuda_stream) {
    ibp_status s = check_ready(h, "ibp_gather_decompress_noalloc");
    if (s != IBP_OK) return s;
    if (n == 0) return IBP_OK;
    if (n < 0 || !row_ids_dev || !out_dev || ((uintptr_t)out_dev & 15u)) { ibp_set_error("ibp_gather_decompress_noalloc: bad argument (null pointer, n<0, or out not 16-byte aligned)"); return IBP_ERR_INVALID_ARG; }
    if (n > (int64_t)IBP_NOALLOC_MAX_IDS) {
        ibp_set_error("ibp_gather_decompress_noalloc: n = %lld exceeds IBP_NOALLOC_MAX_IDS = %d ids per call (the fixed scratch array); split the batch or use ibp_gather_decompress",
                      (long long)n, (int)IBP_NOALLOC_MAX_IDS);
        return IBP_ERR_INVALID_ARG;
    }
    if (h->p.index_span != 1 || h->p.n_rows == 0) { ibp_set_error("ibp_gather_decompress_noalloc: random rows only (index_span must be 1)"); return IBP_ERR_UNSUPPORTED; }
    if (!h->store_dev) { ibp_set_error("ibp_gather_decompress_noalloc: the packed store is not GPU-mapped (pageable store)"); return IBP_ERR_BAD_STATE; }
    cudaStream_t st = (cudaStream_t)cuda_stream;
    uint8_t* ws = nullptr;
    s = noalloc_scratch_ptr(h->device, &ws);
    if (s != IBP_OK) return s;
    uint32_t shift = 0, nb = 0;
    bucket_shape(h->p.n_rows, h->store_used, 256ull << 10, &shift, &nb);
    const uint32_t nb_pad = (nb + 4095u) / 4096u * 4096u;                                    // <= 2^18: fits NOALLOC_CNT_BYTES
    // the array keeps the last call's contents: the counters must start at zero (the order list is fully rewritten)
    IBP_CUDA(cudaMemsetAsync(ws, 0, 256 + (size_t)nb_pad * 4, st));
    uint32_t* cnt = (uint32_t*)(ws + 256);
    int32_t* ord = (int32_t*)(ws + NOALLOC_ZERO_BYTES);
    const int thr = 256, blocks = (int)std::min<int64_t>((n + thr - 1) / thr, (int64_t)h->sm_count * 8);
    ibp_bucket_hist<<<blocks, thr, 0, st>>>(row_ids_dev, nullptr, nullptr, n, shift, nb, cnt);
    ibp_bucket_scan<<<1, 1024, 0, st>>>(cnt, nb_pad);
    ibp_bucket_scatter<<<blocks, thr, 0, st>>>(row_ids_dev, nullptr, nullptr, n, shift, nb, cnt, ord);
    IBP_CUDA(cudaGetLastError());
    DecodeParams P;
    fill_common(h, P);
    P.store = h->store_dev;
    P.ids = row_ids_dev;
    P.out = (uint8_t*)out_dev;
    P.n = n;
    P.span = 1;
    P.n_units = n;
    P.order = ord;
    if (h->packed_bytes_rows / h->p.n_rows >= 96 && h->p.row_bytes <= 512) P.occ_cap = 1;    // the launch shape gather_rows picks for line-sized rows
    return launch_decode(h, P, MODE_ROWS, st);
}

// Rows [first_row, first_row+n_rows) in order, packed bytes at `packed` (device-visible), whose first byte is the packed
// byte of first_row.  Shared by the resident decode (packed bytes staged in HBM) and the zero-copy range gather.
static ibp_status decode_range(ibp_handle* h, const uint8_t* packed, int64_t first_row, int64_t n_rows, void* out_dev, cudaStream_t st, bool resident = false) {
    // (slot layout: consecutive rows are not contiguous in the store -- only the head of every slot is meaningful -- so runs
    // take the per-row kernel, which fetches exactly each row's bytes)
    if (h->stream_mode && h->thresholded && !h->slot_layout && stream_t_fits(h))
        return launch_stream_t(h, packed, ibp_row_offset(h, (uint64_t)first_row), nullptr, 1, first_row, n_rows, out_dev, st, resident);
    if (h->stream_mode && !h->thresholded)
        return launch_stream(h, packed, ibp_row_offset(h, (uint64_t)first_row), nullptr, 1, first_row, n_rows, out_dev, st, resident);
    DecodeParams P;
    fill_common(h, P);
    P.store = packed;
    P.bias = ibp_row_offset(h, (uint64_t)first_row);
    P.out = (uint8_t*)out_dev;
    P.n = n_rows;
    P.first_row = first_row;
    if (h->p.group_kind == IBP_GROUP_BLOCKED) {
        P.span = (uint32_t)n_rows;
        P.rows_per_unit = std::min<uint32_t>(h->p.group_param, 16u);
        if (h->p.group_param % P.rows_per_unit) P.rows_per_unit = 16u;
        P.units_per_span = (uint32_t)((n_rows + P.rows_per_unit - 1) / P.rows_per_unit);
        P.n_units = P.units_per_span;
        return launch_decode(h, P, MODE_SPANS, st);
    }
    const uint64_t S = h->p.group_param, n_mrows = ((uint64_t)n_rows + S - 1) / S;
    P.rows_per_unit = 16;
    P.n_units = (int64_t)(((n_mrows + P.rows_per_unit - 1) / P.rows_per_unit) * S);
    return launch_decode(h, P, MODE_STRIDED, st);
}

static ibp_status check_range(const ibp_handle* h, const char* who, int64_t first_row, int64_t n_rows, const void* out_dev) {
    if (!out_dev || first_row < 0 || n_rows < 0 || (uint64_t)(first_row + n_rows) > h->p.n_rows || ((uintptr_t)out_dev & 15u)) {
        ibp_set_error("%s: bad argument (range, null pointer or alignment)", who);
        return IBP_ERR_INVALID_ARG;
    }
    const bool any_row = h->thresholded && h->p.group_kind == IBP_GROUP_BLOCKED;   // per-row offsets: every row starts a unit
    if (!any_row && (uint64_t)first_row % h->p.group_param) { ibp_set_error("%s: first_row must be a multiple of %u", who, h->p.group_param); return IBP_ERR_INVALID_ARG; }
    if (n_rows > 0xFFFFFFFFll) { ibp_set_error("%s: range too long", who); return IBP_ERR_INVALID_ARG; }
    return IBP_OK;
}

extern "C" ibp_status ibp_decompress_resident(ibp_handle* h, const void* packed_dev, int64_t first_row, int64_t n_rows, void* out_dev, void* cuda_stream) {
    ibp_status s = check_ready(h, "ibp_decompress_resident");
    if (s != IBP_OK) return s;
    if (n_rows == 0) return IBP_OK;
    if (!packed_dev || ((uintptr_t)packed_dev & 15u)) { ibp_set_error("ibp_decompress_resident: packed_dev must be a 16-byte aligned device pointer"); return IBP_ERR_INVALID_ARG; }
    s = check_range(h, "ibp_decompress_resident", first_row, n_rows, out_dev);
    if (s != IBP_OK) return s;
    return decode_range(h, (const uint8_t*)packed_dev, first_row, n_rows, out_dev, (cudaStream_t)cuda_stream, true);
}

extern "C" ibp_status ibp_gather_decompress_range(ibp_handle* h, int64_t first_row, int64_t n_rows, void* out_dev, void* cuda_stream) {
    ibp_status s = check_ready(h, "ibp_gather_decompress_range");
    if (s != IBP_OK) return s;
    if (n_rows == 0) return IBP_OK;
    if (!h->store_dev) { ibp_set_error("ibp_gather_decompress_range: the packed store is not GPU-mapped (pageable store)"); return IBP_ERR_BAD_STATE; }
    s = check_range(h, "ibp_gather_decompress_range", first_row, n_rows, out_dev);
    if (s != IBP_OK) return s;
    return decode_range(h, h->store_dev + ibp_row_offset(h, (uint64_t)first_row), first_row, n_rows, out_dev, (cudaStream_t)cuda_stream);
}

// Range gather with a HOST destination (the end-to-end form of weight / block streaming): a pinned, GPU-mapped out_host is
// written by the decode kernel directly (zero-copy stores); anything else goes through a device staging buffer and one copy.
extern "C" ibp_status ibp_gather_decompress_range_host(ibp_handle* h, int64_t first_row, int64_t n_rows, void* out_host, void* cuda_stream) {
    ibp_status s = check_ready(h, "ibp_gather_decompress_range_host");
    if (s != IBP_OK) return s;
    if (n_rows == 0) return IBP_OK;
    if (!out_host) { ibp_set_error("ibp_gather_decompress_range_host: null destination"); return IBP_ERR_INVALID_ARG; }
    cudaStream_t st = (cudaStream_t)cuda_stream;
    cudaPointerAttributes attr;
    void* alias = nullptr;
    if (cudaPointerGetAttributes(&attr, out_host) == cudaSuccess && attr.type == cudaMemoryTypeHost &&
        cudaHostGetDevicePointer(&alias, out_host, 0) == cudaSuccess && alias && !((uintptr_t)alias & 15u)) {
        s = ibp_gather_decompress_range(h, first_row, n_rows, alias, cuda_stream);
        const cudaError_t es = cudaStreamSynchronize(st);
        if (s == IBP_OK && es != cudaSuccess) { ibp_set_error("ibp_gather_decompress_range_host: %s", cudaGetErrorString(es)); (void)cudaGetLastError(); s = IBP_ERR_CUDA; }
        return s;
    }
    (void)cudaGetLastError();
    if (first_row < 0 || n_rows < 0 || (uint64_t)(first_row + n_rows) > h->p.n_rows) { ibp_set_error("ibp_gather_decompress_range_host: bad range"); return IBP_ERR_INVALID_ARG; }
    const size_t bytes = (size_t)n_rows * h->p.row_bytes;
    uint8_t* buf = nullptr;
    IBP_CUDA(cudaMallocAsync((void**)&buf, bytes, st));
    s = ibp_gather_decompress_range(h, first_row, n_rows, buf, cuda_stream);
    cudaError_t e = cudaSuccess;
    if (s == IBP_OK) e = cudaMemcpyAsync(out_host, buf, bytes, cudaMemcpyDeviceToHost, st);
    cudaFreeAsync(buf, st);
    const cudaError_t e2 = cudaStreamSynchronize(st);
    if (s == IBP_OK && (e != cudaSuccess || e2 != cudaSuccess)) {
        ibp_set_error("ibp_gather_decompress_range_host: %s", cudaGetErrorString(e != cudaSuccess ? e : e2));
        (void)cudaGetLastError();
        s = IBP_ERR_CUDA;
    }
    return s;
}

// Several ranges in one launch (a decoder layer's seven matrices): consecutive ranges that the stream kernel can take
// together (strict mode, same word width, at most 8) become the segments of ONE persistent grid; anything else is decoded range
// by range.  One ramp and one tail per layer instead of one per matrix, and no launch gaps on the stream.
extern "C" ibp_status ibp_decode_ranges(const ibp_range_desc* ranges_host, uint32_t n_ranges, void* cuda_stream) {
    if (n_ranges == 0) return IBP_OK;
    if (!ranges_host) { ibp_set_error("ibp_decode_ranges: null range list"); return IBP_ERR_INVALID_ARG; }
    cudaStream_t st = (cudaStream_t)cuda_stream;
    int device = -1;
    for (uint32_t i = 0; i < n_ranges; ++i) {
        const ibp_range_desc& r = ranges_host[i];
        ibp_status s = check_ready(r.handle, "ibp_decode_ranges");
        if (s != IBP_OK) return s;
        if (device < 0) device = r.handle->device;
        if (r.handle->device != device) { ibp_set_error("ibp_decode_ranges: range %u lives on device %d, range 0 on device %d", i, r.handle->device, device); return IBP_ERR_INVALID_ARG; }
        if (r.n_rows == 0) continue;
        s = check_range(r.handle, "ibp_decode_ranges", r.first_row, r.n_rows, r.out_dev);
        if (s != IBP_OK) return s;
        if (r.packed_dev) {
            if ((uintptr_t)r.packed_dev & 15u) { ibp_set_error("ibp_decode_ranges: packed_dev of range %u is not 16-byte aligned", i); return IBP_ERR_INVALID_ARG; }
        } else if (!r.handle->store_dev) {
            ibp_set_error("ibp_decode_ranges: range %u reads the host store, which is not GPU-mapped (pageable store)", i); return IBP_ERR_BAD_STATE;
        }
    }
    auto batchable = [](const ibp_range_desc& r) { return r.n_rows > 0 && r.handle->stream_mode && !r.handle->thresholded; };
    auto source = [](const ibp_range_desc& r) {
        return r.packed_dev ? (const uint8_t*)r.packed_dev : r.handle->store_dev + ibp_row_offset(r.handle, (uint64_t)r.first_row);
    };
    uint32_t i = 0;
    while (i < n_ranges) {
        const ibp_range_desc& r0 = ranges_host[i];
        if (r0.n_rows == 0) { ++i; continue; }
        if (!batchable(r0)) {
            ibp_status s = decode_range(r0.handle, source(r0), r0.first_row, r0.n_rows, r0.out_dev, st, r0.packed_dev != nullptr);
            if (s != IBP_OK) return s;
            ++i;
            continue;
        }
        ibp_handle* h0 = r0.handle;
        const int W = pick_W(h0->p.row_bytes);
        StreamBatch<8> B;
        memset(&B, 0, sizeof B);
        int64_t total = 0;
        uint32_t n_seg = 0, grid_min = 1;
        const int64_t grid_cap = h0->max_ctas ? (int64_t)h0->max_ctas : 2ll * h0->sm_count;
        bool all_host = true;
        while (i < n_ranges && n_seg < 8) {
            const ibp_range_desc& r = ranges_host[i];
            if (r.n_rows == 0) { ++i; continue; }
            if (!batchable(r) || pick_W(r.handle->p.row_bytes) != W) break;
            StreamParams& P = B.seg[n_seg];
            const bool tile_ok = r.packed_dev != nullptr && grid_cap >= (int64_t)((r.handle->n_groups + 7) / 8);
            stream_geometry(r.handle, source(r), ibp_row_offset(r.handle, (uint64_t)r.first_row), nullptr, 1, r.first_row, r.n_rows, r.out_dev, tile_ok, P);
            B.chunk_start[n_seg] = total;
            all_host = all_host && r.packed_dev == nullptr;
            total += P.n_chunks;
            B.stage_bytes = std::max(B.stage_bytes, P.stage_bytes);
            grid_min = std::max(grid_min, P.n_tile_blocks);
            ++n_seg; ++i;
        }
        B.n_seg = n_seg;
        const int ns = B.stage_bytes > 40 * 1024 ? 2 : 3;
        const size_t smem = (size_t)ns * B.stage_bytes + (size_t)ns * 16;
        if (smem > 220 * 1024) { ibp_set_error("ibp_decode_ranges: packed rows do not fit the shared-memory stages"); return IBP_ERR_UNSUPPORTED; }
        ibp_status s;
#define IBP_STREAM_B(W_)                                                                                              \
    s = ns == 2 ? launch_stream_one<W_, 2, 8>(B, total, 1, stream_ctas(h0, !all_host), h0->sm_count, smem, st, grid_min)   \
                : launch_stream_one<W_, 3, 8>(B, total, 1, stream_ctas(h0, !all_host), h0->sm_count, smem, st, grid_min)
        switch (W) {
            case 4: IBP_STREAM_B(4); break;
            case 2: IBP_STREAM_B(2); break;
            default: IBP_STREAM_B(1); break;
        }
#undef IBP_STREAM_B
        if (s != IBP_OK) return s;
    }
    return IBP_OK;
}

// ibp_decode_ranges with HOST destinations.  When every destination is pinned, GPU-mapped memory the ranges are decoded by the
// batched launches of ibp_decode_ranges, the kernels storing straight into host memory (one launch and one synchronisation per
// layer instead of seven); otherwise range by range through ibp_gather_decompress_range_host (staging buffer + copy).
extern "C" ibp_status ibp_decode_ranges_host(const ibp_range_desc* ranges_host, uint32_t n_ranges, void* cuda_stream) {
    if (n_ranges == 0) return IBP_OK;
    if (!ranges_host) { ibp_set_error("ibp_decode_ranges_host: null range list"); return IBP_ERR_INVALID_ARG; }
    std::vector<ibp_range_desc> dev;
    try { dev.assign(ranges_host, ranges_host + n_ranges); } catch (...) { ibp_set_error("ibp_decode_ranges_host: out of memory"); return IBP_ERR_OUT_OF_MEMORY; }
    bool direct = true;
    for (uint32_t i = 0; i < n_ranges && direct; ++i) {
        if (dev[i].n_rows == 0) continue;
        if (!dev[i].out_dev) { ibp_set_error("ibp_decode_ranges_host: null destination in range %u", i); return IBP_ERR_INVALID_ARG; }
        cudaPointerAttributes attr;
        void* alias = nullptr;
        if (cudaPointerGetAttributes(&attr, dev[i].out_dev) == cudaSuccess && attr.type == cudaMemoryTypeHost &&
            cudaHostGetDevicePointer(&alias, dev[i].out_dev, 0) == cudaSuccess && alias && !((uintptr_t)alias & 15u)) dev[i].out_dev = alias;
        else direct = false;
    }
    (void)cudaGetLastError();
    if (direct) {
        ibp_status s = ibp_decode_ranges(dev.data(), n_ranges, cuda_stream);
        const cudaError_t es = cudaStreamSynchronize((cudaStream_t)cuda_stream);
        if (s == IBP_OK && es != cudaSuccess) { ibp_set_error("ibp_decode_ranges_host: %s", cudaGetErrorString(es)); (void)cudaGetLastError(); s = IBP_ERR_CUDA; }
        return s;
    }
    for (uint32_t i = 0; i < n_ranges; ++i) {
        const ibp_range_desc& r = ranges_host[i];
        if (r.n_rows == 0) continue;
        if (r.packed_dev) { ibp_set_error("ibp_decode_ranges_host: a range with packed_dev needs a pinned, GPU-mapped destination"); return IBP_ERR_UNSUPPORTED; }
        ibp_status s = ibp_gather_decompress_range_host(r.handle, r.first_row, r.n_rows, r.out_dev, cuda_stream);
        if (s != IBP_OK) return s;
    }
    return IBP_OK;
}

// Host-buffer entry point.  Large batches are cut into chunks so that the device->host copy of chunk c (copy engine, PCIe
// writes) overlaps the gather of chunk c+1 (SM-issued PCIe reads): the two directions of the link work at the same time.
extern "C" ibp_status ibp_gather_decompress_host(ibp_handle* h, const int64_t* row_ids_host, int64_t n, void* out_host, void* cuda_stream) {
    ibp_status s = check_ready(h, "ibp_gather_decompress_host");
    if (s != IBP_OK) return s;
    if (n == 0) return IBP_OK;
    if (n < 0 || !row_ids_host || !out_host) { ibp_set_error("ibp_gather_decompress_host: bad argument"); return IBP_ERR_INVALID_ARG; }
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const size_t id_bytes_row = (size_t)h->p.index_span * h->p.row_bytes;
    const size_t out_bytes = (size_t)n * id_bytes_row, id_bytes = ((size_t)n * 8 + 255) / 256 * 256;
    // Pinned, GPU-mapped destination (cudaHostAlloc / cudaHostRegister / ibp_host_alloc): the decode kernel stores the rows
    // straight into host memory (zero-copy writes), so PCIe reads of packed rows and PCIe writes of decoded rows share one
    // kernel and nothing is staged in HBM.  Every id is fetched (no de-duplication: its replication pass would read the
    // output back over the link), which costs nothing because the writes, not the reads, bound this path -- unless the batch
    // is one the library would de-duplicate (large, ids not declared distinct: DLRM): there the staged path below fetches each
    // distinct row once and wins (measured: DLRM 29 GB/s direct, 38 GB/s staged; GNN, distinct ids: 40 direct, 34 staged;
    // staging the decoded rows through shared memory into row-sized cp.async.bulk stores changed neither).
    const bool would_dedup = h->p.index_span == 1 && (h->dedup_mode == 1 || (h->dedup_mode < 0 && n >= 16384));
    if (!would_dedup) {
        cudaPointerAttributes attr;
        void* out_dev_alias = nullptr;
        if (cudaPointerGetAttributes(&attr, out_host) == cudaSuccess && attr.type == cudaMemoryTypeHost &&
            cudaHostGetDevicePointer(&out_dev_alias, out_host, 0) == cudaSuccess && out_dev_alias && !((uintptr_t)out_dev_alias & 15u) && h->store_dev) {
            int64_t* ids_d = nullptr;
            IBP_CUDA(cudaMallocAsync((void**)&ids_d, id_bytes, st));
            IBP_CUDA(cudaMemcpyAsync(ids_d, row_ids_host, (size_t)n * 8, cudaMemcpyHostToDevice, st));
            if (h->p.index_span == 1) s = gather_rows(h, nullptr, ids_d, n, out_dev_alias, st, false, true);
            else s = ibp_gather_decompress(h, ids_d, n, out_dev_alias, cuda_stream);
            cudaFreeAsync(ids_d, st);
            const cudaError_t es = cudaStreamSynchronize(st);
            if (s == IBP_OK && es != cudaSuccess) { ibp_set_error("ibp_gather_decompress_host: %s", cudaGetErrorString(es)); (void)cudaGetLastError(); s = IBP_ERR_CUDA; }
            return s;
        }
        (void)cudaGetLastError();
    }
    int n_chunks = out_bytes >= (32u << 20) ? 4 : out_bytes >= (8u << 20) ? 2 : 1;
    if (n < n_chunks) n_chunks = 1;
    uint8_t* buf = nullptr;
    IBP_CUDA(cudaMallocAsync((void**)&buf, id_bytes + out_bytes, st));
    IBP_CUDA(cudaMemcpyAsync(buf, row_ids_host, (size_t)n * 8, cudaMemcpyHostToDevice, st));
    cudaStream_t copy_st = nullptr;
    cudaEvent_t ev[5] = {nullptr, nullptr, nullptr, nullptr, nullptr};
    cudaError_t e = cudaSuccess;
    if (n_chunks > 1) {
        e = cudaStreamCreateWithFlags(&copy_st, cudaStreamNonBlocking);
        for (int c = 0; c <= n_chunks && e == cudaSuccess; ++c) e = cudaEventCreateWithFlags(&ev[c], cudaEventDisableTiming);
    }
    // chunk boundaries on multiples of `q` rows, so that every chunk's output starts 16-byte aligned inside the staging buffer
    // whatever row_bytes is (any multiple of 4 is allowed: 12, 100, 516, ...)
    int64_t q = 1;
    while ((q * (int64_t)id_bytes_row) % 16) q <<= 1;
    auto cut = [&](int c) { return c >= n_chunks ? n : (n * c / n_chunks) / q * q; };
    for (int c = 0; c < n_chunks && s == IBP_OK && e == cudaSuccess; ++c) {
        const int64_t i0 = cut(c), i1 = cut(c + 1);
        if (i1 <= i0) continue;
        uint8_t* dout = buf + id_bytes + (size_t)i0 * id_bytes_row;
        s = ibp_gather_decompress(h, (const int64_t*)buf + i0, i1 - i0, dout, cuda_stream);
        if (s != IBP_OK) break;
        cudaStream_t cs = st;
        if (n_chunks > 1) {
            e = cudaEventRecord(ev[c], st);
            if (e == cudaSuccess) e = cudaStreamWaitEvent(copy_st, ev[c], 0);
            cs = copy_st;
        }
        if (e == cudaSuccess) e = cudaMemcpyAsync((uint8_t*)out_host + (size_t)i0 * id_bytes_row, dout, (size_t)(i1 - i0) * id_bytes_row, cudaMemcpyDeviceToHost, cs);
    }
    if (n_chunks > 1 && e == cudaSuccess && copy_st) {
        e = cudaEventRecord(ev[n_chunks], copy_st);
        if (e == cudaSuccess) e = cudaStreamWaitEvent(st, ev[n_chunks], 0);
    }
    if (copy_st && (s != IBP_OK || e != cudaSuccess)) cudaStreamSynchronize(copy_st);   // nothing may still write out_host after an error return
    cudaFreeAsync(buf, st);
    const cudaError_t e2 = cudaStreamSynchronize(st);
    for (int c = 0; c < 5; ++c) if (ev[c]) cudaEventDestroy(ev[c]);
    if (copy_st) cudaStreamDestroy(copy_st);
    if (s == IBP_OK && (e != cudaSuccess || e2 != cudaSuccess)) {
        ibp_set_error("ibp_gather_decompress_host: %s", cudaGetErrorString(e != cudaSuccess ? e : e2));
        (void)cudaGetLastError();
        s = IBP_ERR_CUDA;
    }
    return s;
}

// ------------------------------------------------------------------------------------------------ id validation
__global__ void ibp_count_bad_ids(const int64_t* __restrict__ ids, int64_t n, int64_t limit, unsigned long long* bad) {
    unsigned long long c = 0;
    for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x)
        c += (ids[i] < 0 || ids[i] >= limit) ? 1ull : 0ull;
    if (c) atomicAdd(bad, c);
}
extern "C" ibp_status ibp_validate_ids(ibp_handle* h, const int64_t* row_ids_dev, int64_t n, int64_t* n_bad_host, void* cuda_stream) {
    ibp_status s = check_ready(h, "ibp_validate_ids");
    if (s != IBP_OK) return s;
    if (!n_bad_host || n < 0 || (!row_ids_dev && n > 0)) { ibp_set_error("ibp_validate_ids: bad argument"); return IBP_ERR_INVALID_ARG; }
    cudaStream_t st = (cudaStream_t)cuda_stream;
    unsigned long long* bad = nullptr;
    IBP_CUDA(cudaMallocAsync((void**)&bad, 8, st));
    IBP_CUDA(cudaMemsetAsync(bad, 0, 8, st));
    if (n > 0) ibp_count_bad_ids<<<(int)std::min<int64_t>((n + 255) / 256, (int64_t)h->sm_count * 8), 256, 0, st>>>(row_ids_dev, n, (int64_t)(h->p.n_rows / h->p.index_span), bad);
    unsigned long long hb = 0;
    IBP_CUDA(cudaMemcpyAsync(&hb, bad, 8, cudaMemcpyDeviceToHost, st));
    IBP_CUDA(cudaFreeAsync(bad, st));
    IBP_CUDA(cudaStreamSynchronize(st));
    *n_bad_host = (int64_t)hb;
    return IBP_OK;
}

// ------------------------------------------------------------------------------------------------ baseline
// Uncompressed zero-copy gather ("GPU", "GPU (Aligned)"): rows are row_bytes apart and 16-byte aligned,
// so every warp starts on an aligned boundary by construction.  One row per warp, 16-byte loads, streaming stores.
__global__ void ibp_gather_rows_kernel(const uint8_t* __restrict__ rows, uint32_t row_bytes, const int64_t* __restrict__ ids,
                                       const int32_t* __restrict__ order, int64_t n, uint8_t* __restrict__ out) {
    const int lane = threadIdx.x & 31, wpc = blockDim.x >> 5;
    for (int64_t u = (int64_t)blockIdx.x * wpc + (threadIdx.x >> 5); u < n; u += (int64_t)gridDim.x * wpc) {
        const int64_t i = order ? (int64_t)order[u] : u;
        const uint4* src = (const uint4*)(rows + (uint64_t)ids[i] * row_bytes);
        uint4* dst = (uint4*)(out + (uint64_t)i * row_bytes);
        for (uint32_t v = lane; v < row_bytes / 16; v += 32) {
            uint4 t;
            asm volatile("ld.global.nc.L1::no_allocate.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(t.x), "=r"(t.y), "=r"(t.z), "=r"(t.w) : "l"(src + v));
            asm volatile("st.global.cs.v4.b32 [%0], {%1,%2,%3,%4};" ::"l"(dst + v), "r"(t.x), "r"(t.y), "r"(t.z), "r"(t.w) : "memory");
        }
    }
}

extern "C" ibp_status ibp_gather_uncompressed_ex(const void* rows_mapped, uint32_t row_bytes, uint64_t n_rows, const int64_t* row_ids_dev,
                                                 int64_t n, void* out_dev, int locality_order, void* cuda_stream) {
    if (n == 0) return IBP_OK;
    if (!rows_mapped || !row_ids_dev || !out_dev || n < 0 || n > 0x7FFFFFFF || row_bytes == 0 || row_bytes % 16 || ((uintptr_t)rows_mapped & 15u) || ((uintptr_t)out_dev & 15u)) {
        ibp_set_error("ibp_gather_uncompressed: bad argument (row_bytes must be a multiple of 16, pointers 16-byte aligned)");
        return IBP_ERR_INVALID_ARG;
    }
    cudaStream_t st = (cudaStream_t)cuda_stream;
    int32_t* ord = nullptr;
    void* ws = nullptr;
    if (locality_order && n_rows > 0) {
        ibp_status s = make_order(row_ids_dev, n, n_rows, n_rows * (uint64_t)row_bytes, st, &ord, &ws);
        if (s != IBP_OK) return s;
    }
    const int wpc = 8;
    int occ = 0;
    IBP_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, ibp_gather_rows_kernel, wpc * 32, 0));
    const int blocks = (int)std::min<int64_t>((n + wpc - 1) / wpc, ibp_sm_count_current() * (int64_t)std::max(occ, 1));
    ibp_gather_rows_kernel<<<blocks, wpc * 32, 0, st>>>((const uint8_t*)rows_mapped, row_bytes, row_ids_dev, ord, n, (uint8_t*)out_dev);
    IBP_CUDA(cudaGetLastError());
    if (ws) IBP_CUDA(cudaFreeAsync(ws, st));
    return IBP_OK;
}
extern "C" ibp_status ibp_gather_uncompressed(const void* rows_mapped, uint32_t row_bytes, const int64_t* row_ids_dev, int64_t n,
                                              void* out_dev, void* cuda_stream) {
    return ibp_gather_uncompressed_ex(rows_mapped, row_bytes, 0, row_ids_dev, n, out_dev, 0, cuda_stream);
}

// ------------------------------------------------------------------------------------------------ pinned memory
extern "C" ibp_status ibp_host_alloc_managed(size_t nbytes, int device, void** ptr) {
    if (!ptr || nbytes == 0) { ibp_set_error("ibp_host_alloc_managed: bad argument"); return IBP_ERR_INVALID_ARG; }
    void* p = nullptr;
    IBP_CUDA(cudaMallocManaged(&p, nbytes, cudaMemAttachGlobal));
    cudaError_t e = cudaMemAdvise(p, nbytes, cudaMemAdviseSetPreferredLocation, cudaCpuDeviceId);
    if (e == cudaSuccess) e = cudaMemAdvise(p, nbytes, cudaMemAdviseSetAccessedBy, device);
    if (e != cudaSuccess) { cudaFree(p); ibp_set_error("cudaMemAdvise failed: %s", cudaGetErrorString(e)); (void)cudaGetLastError(); return IBP_ERR_CUDA; }
    *ptr = p;
    return IBP_OK;
}
extern "C" ibp_status ibp_host_free_managed(void* ptr) {
    if (!ptr) return IBP_OK;
    IBP_CUDA(cudaFree(ptr));
    return IBP_OK;
}
extern "C" ibp_status ibp_host_alloc(size_t nbytes, void** host_ptr, void** dev_ptr) {
    if (!host_ptr || nbytes == 0) { ibp_set_error("ibp_host_alloc: bad argument"); return IBP_ERR_INVALID_ARG; }
    void* p = nullptr;
    cudaError_t e = cudaHostAlloc(&p, nbytes, cudaHostAllocMapped | cudaHostAllocPortable);
    if (e != cudaSuccess) { ibp_set_error("cudaHostAlloc(%zu) failed: %s", nbytes, cudaGetErrorString(e)); (void)cudaGetLastError(); return e == cudaErrorMemoryAllocation ? IBP_ERR_OUT_OF_MEMORY : IBP_ERR_CUDA; }
    *host_ptr = p;
    if (dev_ptr) {
        void* d = nullptr;
        IBP_CUDA(cudaHostGetDevicePointer(&d, p, 0));
        *dev_ptr = d;
    }
    return IBP_OK;
}
extern "C" ibp_status ibp_host_free(void* host_ptr) {
    if (!host_ptr) return IBP_OK;
    IBP_CUDA(cudaFreeHost(host_ptr));
    return IBP_OK;
}

// ------------------------------------------------------------------------------------------------ link ceilings
__global__ void ibp_contig_read_kernel(const uint4* __restrict__ src, size_t n_vec, unsigned* sink) {
    const size_t tid = blockIdx.x * (size_t)blockDim.x + threadIdx.x, stride = (size_t)gridDim.x * blockDim.x;
    unsigned acc = 0;
    for (size_t i = tid; i < n_vec; i += stride) {
        uint4 t;
        asm volatile("ld.global.nc.L1::no_allocate.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(t.x), "=r"(t.y), "=r"(t.z), "=r"(t.w) : "l"(src + i));
        acc ^= t.x ^ t.y ^ t.z ^ t.w;
    }
    if (acc == 0x9E3779B9u) *sink = acc;   // keeps the loads alive; practically never true
}

static ibp_status measure_link(int device, size_t nbytes, int reps, double* gbps, bool zero_copy, bool d2h = false) {
    if (!gbps || nbytes < (1u << 20) || reps < 1) { ibp_set_error("ibp_measure_*: bad argument"); return IBP_ERR_INVALID_ARG; }
    IBP_CUDA(cudaSetDevice(device));
    void *hp = nullptr, *dp = nullptr, *hd = nullptr;
    unsigned* sink = nullptr;
    IBP_CUDA(cudaHostAlloc(&hp, nbytes, cudaHostAllocMapped | cudaHostAllocPortable));
    memset(hp, 0x5A, nbytes);
    cudaEvent_t a, b;
    ibp_status rc = IBP_OK;
    float best = 1e30f;
    if (cudaMalloc(&dp, zero_copy ? 256 : nbytes) != cudaSuccess || cudaMalloc((void**)&sink, 4) != cudaSuccess ||
        cudaHostGetDevicePointer(&hd, hp, 0) != cudaSuccess || cudaEventCreate(&a) != cudaSuccess || cudaEventCreate(&b) != cudaSuccess) {
        ibp_set_error("ibp_measure_*: allocation failed: %s", cudaGetErrorString(cudaGetLastError()));
        rc = IBP_ERR_CUDA;
    } else {
        for (int it = 0; it < reps + 1; ++it) {   // first iteration is a warm-up
            cudaEventRecord(a, 0);
            if (zero_copy) ibp_contig_read_kernel<<<ibp_sm_count_current() * 4, 512>>>((const uint4*)hd, nbytes / 16, sink);
            else if (d2h) cudaMemcpyAsync(hp, dp, nbytes, cudaMemcpyDeviceToHost, 0);
            else cudaMemcpyAsync(dp, hp, nbytes, cudaMemcpyHostToDevice, 0);
            cudaEventRecord(b, 0);
            if (cudaEventSynchronize(b) != cudaSuccess) { ibp_set_error("ibp_measure_*: %s", cudaGetErrorString(cudaGetLastError())); rc = IBP_ERR_CUDA; break; }
            float ms = 0;
            cudaEventElapsedTime(&ms, a, b);
            if (it) best = std::min(best, ms);
        }
        cudaEventDestroy(a);
        cudaEventDestroy(b);
    }
    if (dp) cudaFree(dp);
    if (sink) cudaFree(sink);
    cudaFreeHost(hp);
    if (rc == IBP_OK) *gbps = (double)nbytes / (best * 1e-3) * 1e-9;
    return rc;
}
extern "C" ibp_status ibp_measure_h2d(int device, size_t nbytes, int reps, double* gbps) { return measure_link(device, nbytes, reps, gbps, false); }
extern "C" ibp_status ibp_measure_zero_copy_read(int device, size_t nbytes, int reps, double* gbps) { return measure_link(device, nbytes, reps, gbps, true); }
extern "C" ibp_status ibp_measure_d2h(int device, size_t nbytes, int reps, double* gbps) { return measure_link(device, nbytes, reps, gbps, false, true); }

// Random span reads: `lanes` = span_bytes/16 consecutive lanes read one span at a hashed, span-aligned offset.
__global__ void ibp_random_read_kernel(const uint4* __restrict__ src, uint64_t n_spans_buf, uint32_t reads_per_group, uint32_t lanes, uint64_t seed,
                                       unsigned* sink) {
    const uint64_t t = blockIdx.x * (uint64_t)blockDim.x + threadIdx.x, grp = t / lanes;
    const uint32_t sub = (uint32_t)(t % lanes);
    unsigned acc = 0;
    for (uint32_t i = 0; i < reads_per_group; ++i) {
        uint64_t z = (grp * 0x100000001B3ull + i) ^ seed;
        z += 0x9E3779B97F4A7C15ull; z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull; z = (z ^ (z >> 27)) * 0x94D049BB133111EBull; z ^= z >> 31;
        const uint64_t s = z % n_spans_buf;
        uint4 v;
        asm volatile("ld.global.nc.L1::no_allocate.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "l"(src + s * lanes + sub));
        acc ^= v.x ^ v.y ^ v.z ^ v.w;
    }
    if (acc == 0x9E3779B9u) *sink = acc;
}

// memory_kind: how the host buffer is obtained and mapped for the GPU (ibp.h: IBP_MEM_*).  The span rate of a large footprint is set
// by the GPU-side page size of the mapping, not by the host page size.
extern "C" ibp_status ibp_measure_random_read_kind(int device, size_t footprint_bytes, uint32_t span_bytes, int memory_kind, int reps,
                                                   double* spans_per_s, double* gbps) {
    if (!spans_per_s || !gbps || footprint_bytes < (1u << 20) || reps < 1 || span_bytes < 16 || span_bytes > 512 || span_bytes % 16 ||
        memory_kind < IBP_MEM_MANAGED_HOST || memory_kind > IBP_MEM_HUGETLB_2M_REGISTERED) {
        ibp_set_error("ibp_measure_random_read: bad argument"); return IBP_ERR_INVALID_ARG;
    }
    IBP_CUDA(cudaSetDevice(device));
    void *p = nullptr, *dptr = nullptr;
    ibp_status rc = IBP_OK;
    size_t map_bytes = 0;
    bool registered = false;
    auto release = [&]() {
        if (registered) cudaHostUnregister(p);
        if (memory_kind == IBP_MEM_MANAGED_HOST && p) ibp_host_free_managed(p);
        else if (memory_kind == IBP_MEM_HOSTALLOC && p) cudaFreeHost(p);
        else if (p && map_bytes) munmap(p, map_bytes);
        (void)cudaGetLastError();
    };
    if (memory_kind == IBP_MEM_MANAGED_HOST) {
        rc = ibp_host_alloc_managed(footprint_bytes, device, &p);
        if (rc != IBP_OK) return rc;
        dptr = p;
    } else if (memory_kind == IBP_MEM_HOSTALLOC) {
        if (cudaHostAlloc(&p, footprint_bytes, cudaHostAllocMapped | cudaHostAllocPortable) != cudaSuccess) {
            ibp_set_error("ibp_measure_random_read: cudaHostAlloc: %s", cudaGetErrorString(cudaGetLastError())); return IBP_ERR_OUT_OF_MEMORY;
        }
    } else {
        map_bytes = (footprint_bytes + (2u << 20) - 1) & ~(size_t)((2u << 20) - 1);
        int flags = MAP_PRIVATE | MAP_ANONYMOUS;
        if (memory_kind == IBP_MEM_HUGETLB_2M_REGISTERED) flags |= MAP_HUGETLB | (21 << 26 /* MAP_HUGE_SHIFT */);
        p = mmap(nullptr, map_bytes, PROT_READ | PROT_WRITE, flags, -1, 0);
        if (p == MAP_FAILED) {
            p = nullptr;
            ibp_set_error("ibp_measure_random_read: mmap of %zu bytes (kind %d) failed: %s", map_bytes, memory_kind, strerror(errno));
            return memory_kind == IBP_MEM_HUGETLB_2M_REGISTERED ? IBP_ERR_UNSUPPORTED : IBP_ERR_OUT_OF_MEMORY;   // no huge pages reserved on this machine
        }
        if (memory_kind == IBP_MEM_THP_REGISTERED) (void)madvise(p, map_bytes, MADV_HUGEPAGE);
    }
    {   // first touch on the host, in parallel (before page-locking: the pages exist when they are registered)
        const int64_t nchunk = (int64_t)((footprint_bytes + (1u << 22) - 1) >> 22);
#pragma omp parallel for schedule(static)
        for (int64_t c = 0; c < nchunk; ++c) memset((char*)p + ((size_t)c << 22), 0x5A, std::min<size_t>(1u << 22, footprint_bytes - ((size_t)c << 22)));
    }
    if (memory_kind >= IBP_MEM_MALLOC_REGISTERED) {
        if (cudaHostRegister(p, map_bytes, cudaHostRegisterMapped | cudaHostRegisterPortable) != cudaSuccess) {
            ibp_set_error("ibp_measure_random_read: cudaHostRegister: %s", cudaGetErrorString(cudaGetLastError()));
            release();
            return IBP_ERR_CUDA;
        }
        registered = true;
    }
    if (!dptr && cudaHostGetDevicePointer(&dptr, p, 0) != cudaSuccess) {
        ibp_set_error("ibp_measure_random_read: cudaHostGetDevicePointer: %s", cudaGetErrorString(cudaGetLastError()));
        release();
        return IBP_ERR_CUDA;
    }
    unsigned* sink = nullptr;
    cudaEvent_t a, b;
    float best = 1e30f;
    const uint32_t lanes = span_bytes / 16, rpg = 64;
    const int grid = ibp_sm_count_current() * 8, block = 256;
    const double n_reads = (double)((uint64_t)grid * block / lanes) * rpg;
    if (cudaMalloc((void**)&sink, 4) != cudaSuccess || cudaEventCreate(&a) != cudaSuccess || cudaEventCreate(&b) != cudaSuccess) {
        ibp_set_error("ibp_measure_random_read: allocation failed: %s", cudaGetErrorString(cudaGetLastError()));
        rc = IBP_ERR_CUDA;
    } else {
        for (int it = 0; it < reps + 1; ++it) {
            cudaEventRecord(a, 0);
            ibp_random_read_kernel<<<grid, block>>>((const uint4*)dptr, footprint_bytes / span_bytes, rpg, lanes, 0x1234u + it, sink);
            cudaEventRecord(b, 0);
            if (cudaEventSynchronize(b) != cudaSuccess) { ibp_set_error("ibp_measure_random_read: %s", cudaGetErrorString(cudaGetLastError())); rc = IBP_ERR_CUDA; break; }
            float ms = 0;
            cudaEventElapsedTime(&ms, a, b);
            if (it) best = std::min(best, ms);
        }
        cudaEventDestroy(a);
        cudaEventDestroy(b);
    }
    if (sink) cudaFree(sink);
    release();
    if (rc == IBP_OK) { *spans_per_s = n_reads / (best * 1e-3); *gbps = *spans_per_s * span_bytes * 1e-9; }
    return rc;
}

extern "C" ibp_status ibp_measure_random_read(int device, size_t footprint_bytes, uint32_t span_bytes, int reps, double* spans_per_s, double* gbps) {
    return ibp_measure_random_read_kind(device, footprint_bytes, span_bytes, IBP_MEM_MANAGED_HOST, reps, spans_per_s, gbps);
}

// 1 = de-duplicate the ids of a random gather before fetching; 0 = fetch every id (the caller knows the ids are distinct);
// -1 = automatic (default): on for batches of >= 16384 ids.
extern "C" ibp_status ibp_set_dedup_mode(ibp_handle* h, int mode) {
    if (!h || mode < -1 || mode > 1) { ibp_set_error("ibp_set_dedup_mode: bad argument"); return IBP_ERR_INVALID_ARG; }
    h->dedup_mode = mode;
    return IBP_OK;
}

// Test/tuning hook: 1 = contiguous runs through the TMA producer/consumer stream kernel (default), 0 = per-row fetch.
extern "C" ibp_status ibp_set_stream_mode(ibp_handle* h, int mode) {
    if (!h || mode < 0 || mode > 2) { ibp_set_error("ibp_set_stream_mode: bad argument"); return IBP_ERR_INVALID_ARG; }
    h->stream_mode = mode ? 1 : 0;
    h->t2_mode = mode == 2 ? 0 : 1;
    return IBP_OK;
}

// Test/tuning hook: engine for the packed-row fetch: 0 = cp.async through the LSU, 1 = cp.async.bulk (TMA) + mbarrier.
extern "C" ibp_status ibp_set_rows_in_flight(ibp_handle* h, int nst) {
    if (!h || (nst != 0 && nst != 1 && nst != 2 && nst != 4)) { ibp_set_error("ibp_set_rows_in_flight: 0 (automatic), 1, 2 or 4"); return IBP_ERR_INVALID_ARG; }
    h->rows_in_flight = nst;
    return IBP_OK;
}
extern "C" ibp_status ibp_set_fetch_mode(ibp_handle* h, int mode) {
    if (!h || mode < 0 || mode > 1) { ibp_set_error("ibp_set_fetch_mode: bad argument"); return IBP_ERR_INVALID_ARG; }
    h->fetch_mode = mode;
    return IBP_OK;
}

// Test/tuning hook: force the locality-ordered gather on (1), off (0) or automatic (-1).
extern "C" ibp_status ibp_set_order_mode(ibp_handle* h, int mode) {
    if (!h || mode < -1 || mode > 1) { ibp_set_error("ibp_set_order_mode: bad argument"); return IBP_ERR_INVALID_ARG; }
    h->order_mode = mode;
    return IBP_OK;
}
