// ibp_stream.cuh -- decode of CONTIGUOUS runs of rows (KV page spans, whole weight matrices, resident ranges).
//
// A warp-specialised TMA pipeline (the Blackwell idiom; PAPER.md:213's shared-memory workspace + asynchronous reads):
//   producer  one elected lane of the last warp: for every chunk (a run of consecutive rows = one contiguous byte
//             range of the packed store) waits for the stage to be free (empty mbarrier), arms the full mbarrier with
//             the byte count and issues large cp.async.bulk copies (<= 16 KB each) of the 16-byte-aligned cover.
//             Host store: the link sees long contiguous reads instead of one short read per row.  HBM source: same code.
//   consumers NW warps wait on the full mbarrier, decode "pieces" of the chunk (rows of one group: Mask/Bitval, bit
//             offsets and the five bit-expand move masks live in registers for the whole piece), then release the stage.
// Bit re-insertion (S5), chosen per group from its masks (warp-uniform):
//   - at most three runs of variant bits in every word (float data: mantissa run, exponent run, sign): run-wise deposit, one
//     multiply by 2^(p_j - c_j) and one lop3 and-or with the run's mask per run, starting from Bitval (2-6 ops per word);
//   - otherwise the branch-free parallel-suffix expand of Hacker's Delight 7-5 (x = (x & ~mv_i) | ((x << 2^i) & mv_i)) with 3, 4
//     or 5 stages depending on the largest move, the move masks computed once per piece or loaded from a per-group table built
//     at upload time when the table has few groups (strided column-tile tables).
// Strided tables decoded from HBM use tile-block chunks (StreamParams::n_tile_blocks): a CTA keeps one block of NW column tiles
// for all its chunks, so a consumer warp prepares its tile once.
#pragma once

struct StreamParams {
    const uint8_t* store;          // device-visible packed bytes; row at store + offset(id) - bias
    uint64_t bias;
    const uint32_t* meta;          // per group: Mask words, Bitval words
    const uint32_t* mvtab;         // optional: per group, per word: 5 expand move masks (n_words * 5), else nullptr
    const IbpGroupEntry* gtab;
    const int64_t* ids;            // span gather: one id per span; nullptr: a single range
    uint8_t* out;
    int64_t first_row;             // range mode: first row id
    int64_t span_rows;             // rows per span / rows of the range
    int64_t n_chunks;
    uint64_t row_stride_strided;
    uint32_t chunks_per_span, rows_per_chunk, piece_rows;
    uint32_t row_bytes, n_words, n_pass;
    uint32_t group_param, group_shift, strided;
    uint32_t stage_bytes;
    uint32_t fast_rows;            // packed rows start on 4-byte boundaries (A >= 4): the hoisted single-pass path applies
    // strided tables, tile-block mode (resident decode): a chunk is `rows_per_chunk` matrix rows x one block of NW column
    // tiles, and chunk c belongs to block c % n_tile_blocks -- with a grid that is a multiple of n_tile_blocks every CTA
    // keeps ONE block, so consumer warp w decodes the same tile in every chunk and prepares it once.  0 = off.
    uint32_t n_tile_blocks;
    // blocked groups, single-pass rows (round 2): the stage carries an aux region IN FRONT of the packed bytes -- a 32-byte chunk
    // descriptor written by the producer, the group-table entries and Mask/Bitval of the groups the chunk touches (bulk copies) --
    // so consumer warps read nothing from global memory.  aux_bytes = 0: off (consumers compute the geometry and load metadata
    // themselves: strided tables, multi-pass rows, chunks that touch too many groups to stage).
    uint32_t aux_bytes, aux_meta_off;
    uint32_t n_tiles;              // groups that exist: min(S, rows of the table) -- the group table has no entry beyond them
    uint32_t tb_pitch;             // bytes between the block's images of consecutive matrix rows inside a stage
};

// One launch over several independent ranges (a whole decoder layer = 7 weight matrices): the segments are walked in
// order by every CTA, the mbarrier pipeline runs on across segment borders, and a CTA takes the chunks gc = blockIdx.x (mod
// gridDim.x) of the CONCATENATED chunk list, so the load balances over the whole launch and there is one ramp and one tail per
// layer instead of one per matrix.  NSEG = 1 is the single-range kernel (segment index a compile-time constant).
template <int NSEG>
struct StreamBatch {
    StreamParams seg[NSEG];
    int64_t chunk_start[NSEG];     // first global chunk index of segment j (non-tile segments)
    uint32_t n_seg;
    uint32_t stage_bytes;          // shared-memory stage size of the launch: the largest any segment needs
};

// The five move masks of the parallel-suffix expand for deposit positions nv (set bits = positions to fill, lowest first).
__device__ __forceinline__ void expand_masks(uint32_t nv, uint32_t mv[5]) {
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
// The same with only the first nstg stages computed (nstg warp-uniform): stage i moves bits by 2^i, and a bit moves by the number of
// invariant bits below it, so a word with fewer than 2^i invariant bits has mv[i] = 0 -- exactly, not approximately.
__device__ __forceinline__ void expand_masks_n(uint32_t nv, uint32_t mv[5], int nstg) {
    uint32_t m = nv, mk = ~nv << 1;
#pragma unroll
    for (int i = 0; i < 5; ++i) {
        mv[i] = 0;
        if (i < nstg) {
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
}
// bit-select in ONE logic op: (c & a) | (~c & b)  (lop3 truth table 0xE4 for inputs a, b, c)
__device__ __forceinline__ uint32_t bitselect(uint32_t a, uint32_t b, uint32_t c) {
    uint32_t d;
    asm("lop3.b32 %0, %1, %2, %3, 0xE4;" : "=r"(d) : "r"(a), "r"(b), "r"(c));
    return d;
}
// (a & b) | c in one logic op
__device__ __forceinline__ uint32_t and_or(uint32_t a, uint32_t b, uint32_t c) {
    uint32_t d;
    asm("lop3.b32 %0, %1, %2, %3, 0xEA;" : "=r"(d) : "r"(a), "r"(b), "r"(c));
    return d;
}
// NSTG = number of low stages that can move a bit: a group whose words never move a bit by 8 or 16 positions (bf16 pairs
// with a few invariant exponent bits per half) needs 3 stages instead of 5.
template <int NSTG = 5>
__device__ __forceinline__ uint32_t expand_bits(uint32_t x, const uint32_t mv[5]) {
#pragma unroll
    for (int i = NSTG - 1; i >= 0; --i) x = bitselect(x << (1 << i), x, mv[i]);
    return x;
}

// Fills mvtab for groups [0, n_groups): one thread per (group, word).
__global__ void ibp_build_mvtab(const uint32_t* __restrict__ meta, uint32_t n_words, uint64_t n_groups, uint32_t* __restrict__ mvtab) {
    const uint64_t i = blockIdx.x * (uint64_t)blockDim.x + threadIdx.x;
    if (i >= n_groups * n_words) return;
    const uint64_t g = i / n_words, w = i - g * n_words;
    uint32_t mv[5];
    expand_masks(~meta[g * 2ull * n_words + w], mv);
#pragma unroll
    for (int k = 0; k < 5; ++k) mvtab[i * 5 + k] = mv[k];
}

template <int W> __device__ __forceinline__ void lds_words(uint32_t a, uint32_t (&v)[W]);
template <> __device__ __forceinline__ void lds_words<1>(uint32_t a, uint32_t (&v)[1]) {
    asm volatile("ld.shared.u32 %0, [%1];" : "=r"(v[0]) : "r"(a));
}
template <> __device__ __forceinline__ void lds_words<2>(uint32_t a, uint32_t (&v)[2]) {
    asm volatile("ld.shared.v2.u32 {%0,%1}, [%2];" : "=r"(v[0]), "=r"(v[1]) : "r"(a));
}
template <> __device__ __forceinline__ void lds_words<4>(uint32_t a, uint32_t (&v)[4]) {
    asm volatile("ld.shared.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]) : "r"(a));
}
// consumer-side wait with a suspend-time hint: a waiting warp stays off the issue port instead of polling
__device__ __forceinline__ void mbar_wait_hint(uint32_t bar, uint32_t parity) {
    uint32_t ok = 0;
    while (!ok) {
        asm volatile(
            "{\n\t.reg .pred p;\n\t"
            "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2, %3;\n\t"
            "selp.u32 %0, 1, 0, p;\n\t}"
            : "=r"(ok) : "r"(bar), "r"(parity), "r"(20000u) : "memory");
    }
}

// STAGED: the aux region of StreamParams::aux_bytes is in use (single-segment launches of blocked tables with small groups); a
// separate instantiation, so that the other launches keep exactly the code they had.
template <int W, int NS, int NW, int NSEG, bool STAGED = false>
__global__ void __launch_bounds__((NW + 1) * 32, 2) ibp_stream_kernel(const __grid_constant__ StreamBatch<NSEG> B) {
    extern __shared__ __align__(128) uint8_t smem[];
    const int lane = threadIdx.x & 31, wib = threadIdx.x >> 5;
    const uint32_t smem_s = (uint32_t)__cvta_generic_to_shared(smem);
    const uint32_t STAGE = B.stage_bytes;
    const uint32_t full_s = smem_s + NS * STAGE, empty_s = full_s + NS * 8;
    if (threadIdx.x == 0) {
#pragma unroll
        for (int s = 0; s < NS; ++s) { mbar_init(full_s + s * 8, 1); mbar_init(empty_s + s * 8, NW); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    const uint32_t n_seg = NSEG == 1 ? 1u : B.n_seg;
    uint32_t k = 0;                       // pipeline position: the same sequence in the producer and in every consumer warp
    // consumer state of the lane's W words (see below); lives across segments, invalidated at every segment border
    uint32_t m[W], b[W], ex[W], mv[W][6];
    uint32_t mode = 15;
    uint64_t prep_g = ~0ull;
    const uint32_t w0_fast = lane * W;

  for (uint32_t seg = 0; seg < n_seg; ++seg) {
    const StreamParams& P = B.seg[NSEG == 1 ? 0 : seg];
    const uint64_t S = P.group_param;
    // this CTA's chunks of the segment: global chunk gc = chunk_start + c belongs to CTA gc mod gridDim.x
    const int64_t c_first = NSEG == 1 ? (int64_t)blockIdx.x
                                      : (int64_t)(((int64_t)blockIdx.x - B.chunk_start[seg] % (int64_t)gridDim.x + (int64_t)gridDim.x) % (int64_t)gridDim.x);
    // tile-block mode: CTA class tb = vb mod n_tile_blocks keeps tile block tb; the class's CTAs share its row blocks round-robin
    const uint32_t vb = NSEG == 1 ? blockIdx.x : (blockIdx.x + seg * 37u) % gridDim.x;
    const uint32_t tb_c = P.n_tile_blocks ? vb % P.n_tile_blocks : 0u, tb_idx = P.n_tile_blocks ? vb / P.n_tile_blocks : 0u;
    const uint32_t tb_cls = P.n_tile_blocks ? (gridDim.x - tb_c + P.n_tile_blocks - 1u) / P.n_tile_blocks : 1u;
    const uint32_t tb_rblocks = P.n_tile_blocks ? (uint32_t)(P.n_chunks / P.n_tile_blocks) : 0u;
    prep_g = ~0ull;

    // chunk c -> first row id, rows (blocked) or matrix rows (strided), first output row, packed byte range
    auto chunk_geom = [&](int64_t c, int64_t& row0, uint32_t& nrows, int64_t& out0, uint64_t& b0, uint64_t& b1) {
        const int64_t si = !P.ids ? 0 : (P.n_chunks <= 0x7FFFFFFFll ? (int64_t)((uint32_t)c / P.chunks_per_span) : c / P.chunks_per_span);
        const int64_t cc = c - si * P.chunks_per_span;
        const int64_t span_first = P.ids ? P.ids[si] * P.span_rows : P.first_row;
        if (!P.strided) {
            const int64_t r = cc * P.rows_per_chunk;
            row0 = span_first + r;
            nrows = (uint32_t)min((int64_t)P.rows_per_chunk, P.span_rows - r);
            out0 = si * P.span_rows + r;
            const uint64_t g0 = group_of_u(P.group_param, P.group_shift, (uint64_t)row0);
            const uint64_t last = (uint64_t)row0 + nrows - 1, g1 = group_of_u(P.group_param, P.group_shift, last);
            const IbpGroupEntry e0 = P.gtab[g0];
            const IbpGroupEntry e1 = g1 == g0 ? e0 : P.gtab[g1];
            b0 = e0.base + ((uint64_t)row0 - g0 * S) * e0.stride;
            b1 = e1.base + (last - g1 * S) * e1.stride + e1.stride;
        } else {
            const int64_t n_mrows = (P.span_rows + (int64_t)S - 1) / (int64_t)S;
            const int64_t mr = cc * P.rows_per_chunk;
            nrows = (uint32_t)min((int64_t)P.rows_per_chunk, n_mrows - mr);
            row0 = span_first + mr * (int64_t)S;
            out0 = si * P.span_rows + mr * (int64_t)S;
            b0 = ((uint64_t)row0 / S) * P.row_stride_strided;
            b1 = b0 + (uint64_t)nrows * P.row_stride_strided;
        }
    };

    if (wib == NW) {
        // ------------------------------------------------------------------ producer
        if (lane != 0) { if (NSEG == 1) return; continue; }
        if (P.n_tile_blocks) {
            for (uint32_t rbk = tb_idx; rbk < tb_rblocks; rbk += tb_cls, ++k) {
                const uint32_t s = k % NS;
                mbar_wait(empty_s + s * 8, ((k / NS) & 1u) ^ 1u);
                const uint32_t tb = tb_c;
                const uint32_t t0 = tb * NW, t1 = min(P.n_tiles, t0 + NW);
                const int64_t n_mrows = (P.span_rows + (int64_t)S - 1) / (int64_t)S;
                const int64_t mr0 = (int64_t)rbk * P.rows_per_chunk;
                const uint32_t nrows = (uint32_t)min((int64_t)P.rows_per_chunk, n_mrows - mr0);
                const IbpGroupEntry e0 = P.gtab[t0], e1 = P.gtab[t1 - 1];
                const uint64_t lo = e0.base, len = e1.base + e1.stride - lo;
                const uint8_t* src = P.store + (((uint64_t)P.first_row / S + (uint64_t)mr0) * P.row_stride_strided + lo - P.bias);
                const uint32_t head = (uint32_t)((uintptr_t)src & 15u);
                const uint32_t bytes = (uint32_t)((head + len + 15u) & ~15ull);
                mbar_expect_tx(full_s + s * 8, bytes * nrows);
                const uint32_t dst = smem_s + s * STAGE;
                for (uint32_t i = 0; i < nrows; ++i)
                    bulk_g2s(dst + i * P.tb_pitch, src - head + (uint64_t)i * P.row_stride_strided, bytes, full_s + s * 8);
            }
            if (NSEG == 1) return;
            continue;
        }
        for (int64_t c = c_first; c < P.n_chunks; c += gridDim.x, ++k) {
            const uint32_t s = k % NS;
            int64_t row0, out0; uint32_t nrows; uint64_t b0, b1;
            if constexpr (!STAGED) mbar_wait(empty_s + s * 8, ((k / NS) & 1u) ^ 1u);
            chunk_geom(c, row0, nrows, out0, b0, b1);
            const uint8_t* src = P.store + (b0 - P.bias);
            const uint32_t head = (uint32_t)((uintptr_t)src & 15u);
            const uint32_t bytes = (uint32_t)((head + (b1 - b0) + 15u) & ~15ull);
            if constexpr (STAGED) mbar_wait(empty_s + s * 8, ((k / NS) & 1u) ^ 1u);   // after the geometry: its loads overlap the consumers' work
            const uint32_t dst = smem_s + s * STAGE, bar = full_s + s * 8;
            if constexpr (STAGED) {
                // staged metadata: descriptor by plain stores (made visible by the release of the arrive below), group-table entries
                // and Mask/Bitval of groups g0 .. g1 by bulk copies (consecutive groups are contiguous in GPU memory)
                const uint64_t g0 = group_of_u(P.group_param, P.group_shift, (uint64_t)row0);
                const uint64_t g1 = group_of_u(P.group_param, P.group_shift, (uint64_t)row0 + nrows - 1);
                const uint32_t ng = (uint32_t)(g1 - g0 + 1);
                asm volatile("st.shared.v4.u32 [%0], {%1,%2,%3,%4};" ::"r"(dst), "r"((uint32_t)row0), "r"((uint32_t)((uint64_t)row0 >> 32)),
                             "r"((uint32_t)out0), "r"((uint32_t)((uint64_t)out0 >> 32)) : "memory");
                asm volatile("st.shared.v4.u32 [%0], {%1,%2,%3,%4};" ::"r"(dst + 16u), "r"(nrows), "r"(head), "r"((uint32_t)b0), "r"((uint32_t)(b0 >> 32)) : "memory");
                mbar_expect_tx(bar, bytes + ng * 16u + ng * 2u * P.row_bytes);
                bulk_g2s(dst + 32u, P.gtab + g0, ng * 16u, bar);
                bulk_g2s(dst + P.aux_meta_off, P.meta + g0 * 2ull * P.n_words, ng * 2u * P.row_bytes, bar);
            } else {
                mbar_expect_tx(bar, bytes);
            }
            for (uint32_t o = 0; o < bytes; o += 16384u)
                bulk_g2s(dst + (STAGED ? P.aux_bytes : 0u) + o, src - head + o, min(16384u, bytes - o), bar);
        }
        if (NSEG == 1) return;
        continue;
    }

    // ---------------------------------------------------------------------- consumers
    // Fast path (single-pass rows whose packed bytes start on a 4-byte boundary, i.e. A >= 4): everything that depends
    // only on the group is hoisted out of the row loop -- Mask/Bitval, the word offset and shift of each of the lane's W
    // words inside a packed row, the run multipliers and masks or the expand masks -- and the row loop is: 2 ld.shared + 1
    // funnel shift + 2-12 integer ops per word, one vector store, two pointer bumps.
    // Per-group decode state of the lane's W words.  Two forms, chosen per group (warp-uniform `mode`):
    //   runs (mode 1..3): every word of the group has at most 3 runs of variant bits (float data: a mantissa run, an exponent run,
    //     the sign).  Run j takes bits [c_j, c_j+len_j) of the extracted word to positions [p_j, p_j+len_j): one multiply by
    //     2^(p_j-c_j) and one lop3 (and-or) per run -- mv[q][j] = the multiplier, mv[q][3+j] = the run's mask;
    //   expand (mode 13..15): the general 5-stage parallel-suffix expand, mv[q][0..4] = its move masks, 3/4/5 stages as needed.
    const bool fast = P.n_pass == 1 && P.fast_rows;
    const bool active_fast = w0_fast < P.n_words;

    // meta_s != 0: shared address of the group's staged [Mask][Bitval] record
    auto prepare = [&](uint64_t g, uint32_t meta_s = 0u) {   // S2 + S4 for a single-pass row of group g
        const uint32_t* gm = P.meta + g * 2ull * P.n_words;
        if (STAGED && active_fast && meta_s) { lds_words<W>(meta_s + w0_fast * 4u, m); lds_words<W>(meta_s + P.row_bytes + w0_fast * 4u, b); }
        else if (active_fast) { VecIO<W>::ld(gm + w0_fast, m); VecIO<W>::ld(gm + P.n_words + w0_fast, b); }
        else {
#pragma unroll
            for (int q = 0; q < W; ++q) { m[q] = 0xFFFFFFFFu; b[q] = 0; }
        }
        uint32_t t = 0;
#pragma unroll
        for (int q = 0; q < W; ++q) { ex[q] = t; t += __popc(~m[q]); }
        const uint32_t incl = warp_inclusive_scan(t, lane);
#pragma unroll
        for (int q = 0; q < W; ++q) ex[q] += incl - t;
        // runs of variant bits, lowest first (3 at most; `more` = a word has a fourth)
        bool more = false;
        uint32_t n_runs = 0;
#pragma unroll
        for (int q = 0; q < W; ++q) {
            uint32_t nv = ~m[q], c = 0;
#pragma unroll
            for (int j = 0; j < 3; ++j) {
                const uint32_t low = nv & (0u - nv), run = nv & ~(nv + low);     // nv == 0 -> low = run = 0
                mv[q][j] = run ? 1u << ((__ffs(low) - 1) - c) : 0u;
                mv[q][3 + j] = run;
                c += __popc(run);
                nv &= ~run;
                n_runs = max(n_runs, run ? (uint32_t)j + 1u : 0u);
            }
            more = more || nv != 0;
        }
        if (!__any_sync(0xFFFFFFFFu, more)) {
            mode = __any_sync(0xFFFFFFFFu, n_runs == 3) ? 3u : __any_sync(0xFFFFFFFFu, n_runs == 2) ? 2u : 1u;
            prep_g = g;
            return;
        }
        if (P.mvtab && active_fast) {
            const uint32_t* tv = P.mvtab + (g * P.n_words + w0_fast) * 5ull;
#pragma unroll
            for (int q = 0; q < W; ++q)
#pragma unroll
                for (int i = 0; i < 5; ++i) mv[q][i] = __ldg(tv + q * 5 + i);
        } else {
#pragma unroll
            for (int q = 0; q < W; ++q) {
                if (q > 0 && m[q] == m[q - 1]) {               // homogeneous float data: neighbouring words share a mask
#pragma unroll
                    for (int i = 0; i < 5; ++i) mv[q][i] = mv[q - 1][i];
                } else {
                    expand_masks(~m[q], mv[q]);
                }
            }
        }
        uint32_t hi8 = 0, hi16 = 0;
#pragma unroll
        for (int q = 0; q < W; ++q) { hi8 |= mv[q][3]; hi16 |= mv[q][4]; }
        mode = __any_sync(0xFFFFFFFFu, hi16 != 0) ? 15u : __any_sync(0xFFFFFFFFu, hi8 != 0) ? 14u : 13u;
        prep_g = g;
    };

    // `count` rows of the prepared group: packed row r at shared address saddr + r*sstride, output row at optr + r*ostride
    auto decode_run_n = [&](auto nstg, auto runs, uint32_t saddr, uint32_t sstride, uint8_t* optr, uint64_t ostride, uint32_t count) {
        constexpr int NSTG = decltype(nstg)::value;         // expand stages, or runs per word
        constexpr bool RUNS = decltype(runs)::value;
        uint32_t wa[W], sh[W];
#pragma unroll
        for (int q = 0; q < W; ++q) { wa[q] = saddr + (ex[q] >> 5) * 4u; sh[q] = ex[q] & 31u; }
        optr += (size_t)w0_fast * 4;
        for (uint32_t r = 0; r < count; ++r) {
            uint32_t o[W];
#pragma unroll
            for (int q = 0; q < W; ++q) {
                uint32_t lo, hi;
                asm volatile("ld.shared.u32 %0, [%2];\n\tld.shared.u32 %1, [%2+4];" : "=r"(lo), "=r"(hi) : "r"(wa[q]));
                const uint32_t x = __funnelshift_r(lo, hi, sh[q]);
                if (NSTG <= 3 && RUNS) {
                    uint32_t acc = b[q];                                        // Bitval, then each run of variant bits or-ed in
#pragma unroll
                    for (int j = 0; j < NSTG; ++j) acc = and_or(x * mv[q][j], mv[q][3 + j], acc);
                    o[q] = acc;
                } else {
                    o[q] = bitselect(b[q], expand_bits<NSTG>(x, mv[q]), m[q]);   // Bitval where Mask is 1, expanded bits elsewhere
                }
                wa[q] += sstride;
            }
            if (active_fast) VecIO<W>::st(optr, o);
            optr += ostride;
        }
    };
    auto decode_run = [&](uint32_t saddr, uint32_t sstride, uint8_t* optr, uint64_t ostride, uint32_t count) {
        using std::integral_constant;
        using std::true_type;
        using std::false_type;
        switch (mode) {
            case 1: decode_run_n(integral_constant<int, 1>{}, true_type{}, saddr, sstride, optr, ostride, count); break;
            case 2: decode_run_n(integral_constant<int, 2>{}, true_type{}, saddr, sstride, optr, ostride, count); break;
            case 3: decode_run_n(integral_constant<int, 3>{}, true_type{}, saddr, sstride, optr, ostride, count); break;
            case 13: decode_run_n(integral_constant<int, 3>{}, false_type{}, saddr, sstride, optr, ostride, count); break;
            case 14: decode_run_n(integral_constant<int, 4>{}, false_type{}, saddr, sstride, optr, ostride, count); break;
            default: decode_run_n(integral_constant<int, 5>{}, false_type{}, saddr, sstride, optr, ostride, count); break;
        }
    };

    if (P.n_tile_blocks) {
        // tile-block mode: this CTA's chunks all carry tile block tb_c; warp wib owns one tile of it
        const uint32_t tb = tb_c, t = tb * NW + wib;
        const bool has_tile = t < P.n_tiles;
        uint32_t toff = 0;
        if (has_tile) {
            const IbpGroupEntry e0 = P.gtab[tb * NW], e = P.gtab[t];
            const uint8_t* src = P.store + (((uint64_t)P.first_row / S) * P.row_stride_strided + e0.base - P.bias);
            toff = (uint32_t)((uintptr_t)src & 15u) + (uint32_t)(e.base - e0.base);   // row_stride_strided is a multiple of 16
            prepare(t);
        }
        const int64_t n_mrows = (P.span_rows + (int64_t)S - 1) / (int64_t)S;
        const int64_t tile_rows = has_tile ? (P.span_rows - (int64_t)t + (int64_t)S - 1) / (int64_t)S : 0;   // rows of tile t in range
        for (uint32_t rbk = tb_idx; rbk < tb_rblocks; rbk += tb_cls, ++k) {
            const uint32_t s = k % NS;
            const int64_t mr0 = (int64_t)rbk * P.rows_per_chunk;
            const int64_t cnt = min(min((int64_t)P.rows_per_chunk, n_mrows - mr0), tile_rows - mr0);
            mbar_wait(full_s + s * 8, (k / NS) & 1u);
            if (cnt > 0)
                decode_run(smem_s + s * STAGE + toff, P.tb_pitch, P.out + ((uint64_t)mr0 * S + t) * P.row_bytes, S * P.row_bytes, (uint32_t)cnt);
            __syncwarp();
            if (lane == 0) asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(empty_s + s * 8) : "memory");
        }
        if (NSEG == 1) return;
        continue;
    }
    if constexpr (STAGED) {
        // staged chunks (blocked groups, single-pass rows): descriptor, group entries and Mask/Bitval come out of the stage
        const uint32_t U = P.piece_rows;
        for (int64_t c = c_first; c < P.n_chunks; c += gridDim.x, ++k) {
            const uint32_t s = k % NS, stage_s = smem_s + s * STAGE;
            mbar_wait_hint(full_s + s * 8, (k / NS) & 1u);
            uint32_t d0[4], d1[4];
            lds_words<4>(stage_s, d0);
            lds_words<4>(stage_s + 16u, d1);
            const uint64_t row0 = ((uint64_t)d0[1] << 32) | d0[0], out0 = ((uint64_t)d0[3] << 32) | d0[2];
            const uint32_t nrows = d1[0], head = d1[1];
            const uint64_t b0 = ((uint64_t)d1[3] << 32) | d1[2];
            const uint64_t g0 = group_of_u(P.group_param, P.group_shift, row0);
            const uint32_t n_pieces = (nrows + U - 1) / U;
            for (uint32_t p = wib; p < n_pieces; p += NW) {
                uint32_t j = p * U;
                const uint32_t j1 = min(nrows, j + U);
                while (j < j1) {                                   // runs of rows of one group inside the piece
                    const uint64_t id = row0 + j;
                    const uint64_t g = group_of_u(P.group_param, P.group_shift, id);
                    const uint32_t run = (uint32_t)min((uint64_t)(j1 - j), (g + 1) * S - id);
                    uint32_t e[4];                                 // IbpGroupEntry {base lo, base hi, stride, k_bits}
                    lds_words<4>(stage_s + 32u + (uint32_t)(g - g0) * 16u, e);
                    const uint64_t base = ((uint64_t)e[1] << 32) | e[0];
                    const uint32_t roff = head + (uint32_t)(base + (id - g * S) * e[2] - b0);
                    if (g != prep_g) prepare(g, stage_s + P.aux_meta_off + (uint32_t)(g - g0) * 2u * P.row_bytes);
                    decode_run(stage_s + P.aux_bytes + roff, e[2], P.out + (out0 + j) * P.row_bytes, P.row_bytes, run);
                    j += run;
                }
            }
            __syncwarp();
            if (lane == 0) asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(empty_s + s * 8) : "memory");
        }
        if (NSEG == 1) return;
        continue;
    }
    for (int64_t c = c_first; c < P.n_chunks; c += gridDim.x, ++k) {
        const uint32_t s = k % NS;
        int64_t row0, out0; uint32_t nrows; uint64_t b0, b1;
        chunk_geom(c, row0, nrows, out0, b0, b1);
        const uint32_t head = (uint32_t)((uintptr_t)(P.store + (b0 - P.bias)) & 15u);
        const uint32_t* stage = (const uint32_t*)(smem + (size_t)s * STAGE);
        const uint32_t stage_s = smem_s + s * STAGE;
        bool waited = false;

        // Generic path: any number of passes, any byte alignment; metadata reloaded per pass, run-wise bit deposit.
        auto decode_row_generic = [&](uint64_t g, uint32_t roff, uint8_t* orow) {
            const uint32_t* gm = P.meta + g * 2ull * P.n_words;
            uint32_t carry = 0;
            prep_g = ~0ull;
            for (uint32_t pass = 0; pass < P.n_pass; ++pass) {
                const uint32_t w0 = (pass * 32u + lane) * W;
                const bool active = w0 < P.n_words;
                uint32_t mm[W], bb[W], kq[W];
                if (active) { VecIO<W>::ld(gm + w0, mm); VecIO<W>::ld(gm + P.n_words + w0, bb); }
                else {
#pragma unroll
                    for (int q = 0; q < W; ++q) { mm[q] = 0xFFFFFFFFu; bb[q] = 0; }
                }
                uint32_t t = 0;
#pragma unroll
                for (int q = 0; q < W; ++q) { kq[q] = __popc(~mm[q]); t += kq[q]; }
                const uint32_t incl = warp_inclusive_scan(t, lane);
                uint32_t bit = roff * 8u + carry + incl - t;
                carry += __shfl_sync(0xFFFFFFFFu, incl, 31);
                if (!waited) { mbar_wait(full_s + s * 8, (k / NS) & 1u); waited = true; }
                uint32_t o[W];
#pragma unroll
                for (int q = 0; q < W; ++q) {
                    uint32_t word = bb[q];
                    if (kq[q]) {
                        const uint32_t wq = bit >> 5;
                        word |= deposit_runs(__funnelshift_r(stage[wq], stage[wq + 1], bit), ~mm[q]);
                        bit += kq[q];
                    }
                    o[q] = word;
                }
                if (active) VecIO<W>::st(orow + (size_t)w0 * 4, o);
            }
        };

        if (!P.strided) {
            const uint32_t U = P.piece_rows, n_pieces = (nrows + U - 1) / U;
            if (fast && c + gridDim.x < P.n_chunks) {
                // warm L1/L2 with the metadata of this warp's first piece of its NEXT chunk: the loads in prepare() are
                // otherwise a dependent HBM round trip at the head of every piece
                int64_t nrow0, nout0; uint32_t nn; uint64_t nb0, nb1;
                chunk_geom(c + gridDim.x, nrow0, nn, nout0, nb0, nb1);
                if (wib * U < nn && active_fast) {
                    const uint64_t ng = group_of_u(P.group_param, P.group_shift, (uint64_t)nrow0 + wib * U);
                    const uint32_t* ngm = P.meta + ng * 2ull * P.n_words + w0_fast;
                    asm volatile("prefetch.global.L1 [%0];" ::"l"(ngm));
                    asm volatile("prefetch.global.L1 [%0];" ::"l"(ngm + P.n_words));
                    // ... and with the group-table entries its geometry starts from (two dependent loads at the head of the chunk)
                    if (lane == 0) asm volatile("prefetch.global.L1 [%0];" ::"l"(P.gtab + group_of_u(P.group_param, P.group_shift, (uint64_t)nrow0)));
                    if (lane == 1) asm volatile("prefetch.global.L1 [%0];" ::"l"(P.gtab + ng));
                }
            }
            for (uint32_t p = wib; p < n_pieces; p += NW) {
                uint32_t j = p * U;
                const uint32_t j1 = min(nrows, j + U);
                while (j < j1) {                                   // runs of rows of one group inside the piece
                    const uint64_t id = (uint64_t)row0 + j;
                    const uint64_t g = group_of_u(P.group_param, P.group_shift, id);
                    const uint32_t run = (uint32_t)min((uint64_t)(j1 - j), (g + 1) * S - id);
                    const IbpGroupEntry e = P.gtab[g];
                    const uint32_t roff = head + (uint32_t)(e.base + (id - g * S) * e.stride - b0);
                    uint8_t* orow = P.out + (uint64_t)(out0 + j) * P.row_bytes;
                    if (fast) {
                        if (g != prep_g) prepare(g);
                        if (!waited) { mbar_wait(full_s + s * 8, (k / NS) & 1u); waited = true; }
                        decode_run(stage_s + roff, e.stride, orow, P.row_bytes, run);
                    } else {
                        for (uint32_t r = 0; r < run; ++r) decode_row_generic(g, roff + r * e.stride, orow + (uint64_t)r * P.row_bytes);
                    }
                    j += run;
                }
            }
        } else {
            const int64_t id_end = P.first_row + P.span_rows;     // strided tables are decoded as ranges only
            for (uint32_t t = wib; t < (uint32_t)S; t += NW) {
                const int64_t left = (id_end - (row0 + (int64_t)t) + (int64_t)S - 1) / (int64_t)S;   // rows of tile t in range
                const uint32_t cnt = left <= 0 ? 0u : (uint32_t)min((int64_t)nrows, left);
                if (!cnt) continue;
                const IbpGroupEntry e = P.gtab[t];
                const uint32_t roff = head + (uint32_t)e.base;
                uint8_t* orow = P.out + (uint64_t)(out0 + t) * P.row_bytes;
                if (fast) {
                    if ((uint64_t)t != prep_g) prepare(t);
                    if (!waited) { mbar_wait(full_s + s * 8, (k / NS) & 1u); waited = true; }
                    decode_run(stage_s + roff, (uint32_t)P.row_stride_strided, orow, S * P.row_bytes, cnt);
                } else {
                    for (uint32_t r = 0; r < cnt; ++r)
                        decode_row_generic(t, roff + r * (uint32_t)P.row_stride_strided, orow + (uint64_t)r * S * P.row_bytes);
                }
            }
        }
        if (!waited) mbar_wait(full_s + s * 8, (k / NS) & 1u);   // a warp without a piece still has to follow the phases
        __syncwarp();
        if (lane == 0) asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(empty_s + s * 8) : "memory");
    }
  }   // segments
}
