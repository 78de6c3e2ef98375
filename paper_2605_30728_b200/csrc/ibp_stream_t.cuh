// ibp_stream_t.cuh -- thresholded-mode decode of CONTIGUOUS runs of rows (KV page spans, whole weight matrices, resident
// ranges): the TMA producer/consumer pipeline of ibp_stream.cuh for the paper's default codec.
//
// Rows of a run lie back to back in the store (id order, each padded to A), so a chunk of consecutive rows is one contiguous
// byte range [16*off[row0], 16*off[row0+n)) whatever the individual sizes: the producer lane reads the two offsets and
// issues large bulk copies; consumer warps then take "pieces" (<= 32 rows of one group), load the piece's row offsets and
// raw flags with one coalesced load each, keep Mask/Bitval/expand masks of the group in registers, and per row
//   - raw row (P:363 bit clear): copy through;
//   - every chunk participates (the common case at tau = 0.8): bit offsets are the group's, precomputed once per piece;
//   - otherwise: kept-bit counts from the row's participation bits and a 5-step shuffle scan (P:319 steps 2-3, reading R7).
// Single-pass rows only (row_bytes <= 128*W bytes); longer rows take the per-row kernel.
#pragma once

struct StreamTParams {
    const uint8_t* store;          // device-visible packed bytes; byte b of the store at store + b - bias
    uint64_t bias;
    const uint32_t* meta;          // per group: Mask words, Bitval words
    const uint32_t* row_off;       // n_rows + 1 offsets, 16-byte units
    const uint32_t* row_flag;      // bit r = 1 iff row r is compressed
    const int64_t* ids;            // span gather: one id per span; nullptr: a single range
    uint8_t* out;
    int64_t first_row;             // range mode: first row id
    int64_t span_rows;             // rows per span / rows of the range
    int64_t n_chunks;
    uint32_t chunks_per_span, rows_per_chunk, piece_rows;   // strided: rows_per_chunk counts matrix rows
    uint32_t row_bytes, n_words;
    uint32_t group_param, group_shift, strided;
    uint32_t stage_bytes;
};

// RUNS: every word of every group of the table has at most three runs of variant bits (decided once per handle on the host):
// bits are re-inserted run by run (ibp_stream.cuh) instead of through the five-stage expand.
template <int W, int NS, int NW, bool RUNS>
__global__ void __launch_bounds__((NW + 1) * 32, 2) ibp_stream_t_kernel(const StreamTParams P) {
    extern __shared__ __align__(128) uint8_t smem[];
    const int lane = threadIdx.x & 31, wib = threadIdx.x >> 5;
    const uint32_t smem_s = (uint32_t)__cvta_generic_to_shared(smem);
    const uint32_t full_s = smem_s + NS * P.stage_bytes, empty_s = full_s + NS * 8;
    if (threadIdx.x == 0) {
#pragma unroll
        for (int s = 0; s < NS; ++s) { mbar_init(full_s + s * 8, 1); mbar_init(empty_s + s * 8, NW); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    const uint64_t S = P.group_param;

    // chunk c -> first row id, number of rows (consecutive ids), first output row
    auto chunk_geom = [&](int64_t c, int64_t& row0, uint32_t& nrows, int64_t& out0) {
        const int64_t si = !P.ids ? 0 : (P.n_chunks <= 0x7FFFFFFFll ? (int64_t)((uint32_t)c / P.chunks_per_span) : c / P.chunks_per_span);
        const int64_t cc = c - si * P.chunks_per_span;
        const int64_t span_first = P.ids ? P.ids[si] * P.span_rows : P.first_row;
        const int64_t per = P.strided ? (int64_t)P.rows_per_chunk * (int64_t)S : (int64_t)P.rows_per_chunk;
        const int64_t r = cc * per;
        row0 = span_first + r;
        nrows = (uint32_t)min(per, P.span_rows - r);
        out0 = si * P.span_rows + r;
    };

    if (wib == NW) {
        // ------------------------------------------------------------------ producer
        if (lane != 0) return;
        uint32_t k = 0;
        for (int64_t c = blockIdx.x; c < P.n_chunks; c += gridDim.x, ++k) {
            const uint32_t s = k % NS;
            int64_t row0, out0; uint32_t nrows;
            chunk_geom(c, row0, nrows, out0);
            const uint32_t o0 = __ldg(P.row_off + row0), o1 = __ldg(P.row_off + row0 + nrows);
            mbar_wait(empty_s + s * 8, ((k / NS) & 1u) ^ 1u);
            const uint8_t* src = P.store + (16ull * o0 - P.bias);
            const uint32_t bytes = (o1 - o0) * 16u;
            mbar_expect_tx(full_s + s * 8, bytes);
            const uint32_t dst = smem_s + s * P.stage_bytes;
            for (uint32_t o = 0; o < bytes; o += 16384u)
                bulk_g2s(dst + o, src + o, min(16384u, bytes - o), full_s + s * 8);
        }
        return;
    }

    // ---------------------------------------------------------------------- consumers
    // mv: the group's bit re-insertion state per word: RUNS -- mv[q][j] = multiplier 2^(p_j - c_j), mv[q][3+j] = mask of run j
    // (j < 3); else the five expand move masks.
    uint32_t m[W], b[W], kq[W], ex[W], mv[W][RUNS ? 6 : 5];
    uint64_t prep_g = ~0ull;
    const uint32_t w0 = lane * W;
    const bool active = w0 < P.n_words;
    const uint32_t pmask = W == 32 ? 0xFFFFFFFFu : ((1u << W) - 1u);

    auto prepare = [&](uint64_t g) {   // S2 (+ S4 for rows whose chunks all participate) for group g
        const uint32_t* gm = P.meta + g * 2ull * P.n_words;
        if (active) { VecIO<W>::ld(gm + w0, m); VecIO<W>::ld(gm + P.n_words + w0, b); }
        else {
#pragma unroll
            for (int q = 0; q < W; ++q) { m[q] = 0xFFFFFFFFu; b[q] = 0; }
        }
        uint32_t t = 0;
#pragma unroll
        for (int q = 0; q < W; ++q) { kq[q] = __popc(~m[q]); ex[q] = t; t += kq[q]; }
        const uint32_t incl = warp_inclusive_scan(t, lane);
#pragma unroll
        for (int q = 0; q < W; ++q) ex[q] += P.n_words + incl - t;            // payloads follow the participation bits
        if constexpr (RUNS) {
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
                }
            }
        } else {
#pragma unroll
            for (int q = 0; q < W; ++q) {
                if (q > 0 && m[q] == m[q - 1]) {
#pragma unroll
                    for (int i = 0; i < 5; ++i) mv[q][i] = mv[q - 1][i];
                } else {
                    expand_masks(~m[q], mv[q]);
                }
            }
        }
        prep_g = g;
    };
    // the chunk's bits x (variant bits at bit 0 upwards) back at the Mask = 0 positions, Bitval elsewhere
    auto reinsert = [&](uint32_t x, int q) -> uint32_t {
        if constexpr (RUNS) {
            uint32_t acc = b[q];
#pragma unroll
            for (int j = 0; j < 3; ++j) acc = and_or(x * mv[q][j], mv[q][RUNS ? 3 + j : 0], acc);
            return acc;
        } else {
            return bitselect(b[q], expand_bits(x, mv[q]), m[q]);
        }
    };

    // one row of the prepared group: packed bytes at shared address saddr, `comp` = the row's bit of the bitmask
    auto decode_row = [&](uint32_t saddr, bool comp, uint8_t* orow) {
        uint32_t o[W];
        if (!comp) {                                                           // stored raw: copy through
            if (active) {
#pragma unroll
                for (int q = 0; q < W; ++q) asm volatile("ld.shared.u32 %0, [%1];" : "=r"(o[q]) : "r"(saddr + (w0 + q) * 4u));
            }
        } else {
            uint32_t part = pmask;
            if (active) { asm volatile("ld.shared.u32 %0, [%1];" : "=r"(part) : "r"(saddr + (w0 >> 5) * 4u)); part = (part >> (w0 & 31u)) & pmask; }
            const bool all_in = __all_sync(0xFFFFFFFFu, part == pmask);
            uint32_t bit[W];
            if (all_in) {
#pragma unroll
                for (int q = 0; q < W; ++q) bit[q] = ex[q];
            } else {
                uint32_t t = 0;
#pragma unroll
                for (int q = 0; q < W; ++q) { bit[q] = t; t += active ? (((part >> q) & 1u) ? kq[q] : 32u) : 0u; }
                const uint32_t incl = warp_inclusive_scan(t, lane);
#pragma unroll
                for (int q = 0; q < W; ++q) bit[q] += P.n_words + incl - t;
            }
#pragma unroll
            for (int q = 0; q < W; ++q) {
                uint32_t lo, hi;
                asm volatile("ld.shared.u32 %0, [%2];\n\tld.shared.u32 %1, [%2+4];" : "=r"(lo), "=r"(hi) : "r"(saddr + (bit[q] >> 5) * 4u));
                const uint32_t x = __funnelshift_r(lo, hi, bit[q] & 31u);
                const uint32_t e = reinsert(x, q);
                o[q] = ((part >> q) & 1u) ? e : x;                             // non-participating chunk: all 32 bits
            }
        }
        if (active) VecIO<W>::st(orow + (size_t)w0 * 4, o);
    };

    // RB compressed rows of the prepared group at once.  One row is a chain of dependent steps -- participation read, kept-bit
    // counts, the 5-step shuffle scan of P:319 step 3, the extraction loads, the expand -- of about 1,200 cycles, and with two
    // warps per scheduler nothing hides it (measured: the same 7.6 us per 96-row chunk whether the SM runs one CTA or two).
    // Written out for RB rows side by side, the chains are independent and the scheduler interleaves them.
    constexpr int RB = W == 4 ? 2 : 4;   // W = 4: four rows side by side spill under the two-CTAs-per-SM register budget
    auto decode_rows = [&](const uint32_t* saddr, uint8_t* orow) {
        uint32_t part[RB], tl[RB], incl[RB], bit[RB][W];
#pragma unroll
        for (int i = 0; i < RB; ++i) {
            part[i] = pmask;
            if (active) { asm volatile("ld.shared.u32 %0, [%1];" : "=r"(part[i]) : "r"(saddr[i] + (w0 >> 5) * 4u)); part[i] = (part[i] >> (w0 & 31u)) & pmask; }
        }
#pragma unroll
        for (int i = 0; i < RB; ++i) {
            uint32_t t = 0;
#pragma unroll
            for (int q = 0; q < W; ++q) { bit[i][q] = t; t += active ? (((part[i] >> q) & 1u) ? kq[q] : 32u) : 0u; }
            tl[i] = t; incl[i] = t;
        }
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
#pragma unroll
            for (int i = 0; i < RB; ++i) {
                const uint32_t v = __shfl_up_sync(0xFFFFFFFFu, incl[i], d);
                if (lane >= d) incl[i] += v;
            }
        }
#pragma unroll
        for (int i = 0; i < RB; ++i) {
            uint32_t o[W];
#pragma unroll
            for (int q = 0; q < W; ++q) {
                const uint32_t bq = bit[i][q] + P.n_words + incl[i] - tl[i];
                uint32_t lo, hi;
                asm volatile("ld.shared.u32 %0, [%2];\n\tld.shared.u32 %1, [%2+4];" : "=r"(lo), "=r"(hi) : "r"(saddr[i] + (bq >> 5) * 4u));
                const uint32_t x = __funnelshift_r(lo, hi, bq & 31u);
                const uint32_t e = reinsert(x, q);
                o[q] = ((part[i] >> q) & 1u) ? e : x;
            }
            if (active) VecIO<W>::st(orow + (size_t)i * P.row_bytes + (size_t)w0 * 4, o);
        }
    };
    // Row offsets and raw flags of a piece (lane r <-> row id0 + r): one coalesced load each.  The loads for a warp's FIRST
    // piece of its next chunk are issued before the current chunk is decoded, so their latency (an HBM/L2 round trip in
    // front of every piece otherwise: ncu showed long-scoreboard as the top stall) overlaps the decode.
    auto load_piece = [&](int64_t id0, uint32_t cnt, uint32_t& off_abs, uint32_t& flag) {
        off_abs = lane < cnt ? __ldg(P.row_off + id0 + lane) : 0u;
        flag = lane < cnt ? (__ldg(P.row_flag + ((id0 + lane) >> 5)) >> ((id0 + lane) & 31)) & 1u : 0u;
    };
    const uint32_t U = P.piece_rows;
    int64_t n_row0 = 0, n_out0 = 0;
    uint32_t n_nrows = 0, n_base = 0, n_off = 0, n_flag = 0;
    if ((int64_t)blockIdx.x < P.n_chunks) {
        chunk_geom(blockIdx.x, n_row0, n_nrows, n_out0);
        n_base = __ldg(P.row_off + n_row0);
        if (!P.strided && wib * U < n_nrows) load_piece(n_row0 + wib * U, min(U, n_nrows - wib * U), n_off, n_flag);
    }

    uint32_t k = 0;
    for (int64_t c = blockIdx.x; c < P.n_chunks; c += gridDim.x, ++k) {
        const uint32_t s = k % NS;
        const int64_t row0 = n_row0, out0 = n_out0;
        const uint32_t nrows = n_nrows, base_off = n_base;
        uint32_t my_off = n_off, my_flag = n_flag;
        if (c + gridDim.x < P.n_chunks) {
            chunk_geom(c + gridDim.x, n_row0, n_nrows, n_out0);
            n_base = __ldg(P.row_off + n_row0);
            if (!P.strided && wib * U < n_nrows) {
                load_piece(n_row0 + wib * U, min(U, n_nrows - wib * U), n_off, n_flag);
                if (active) {                                                  // warm L1 with that piece's Mask/Bitval
                    const uint64_t ng = group_of_u(P.group_param, P.group_shift, (uint64_t)n_row0 + wib * U);
                    const uint32_t* ngm = P.meta + ng * 2ull * P.n_words + w0;
                    asm volatile("prefetch.global.L1 [%0];" ::"l"(ngm));
                    asm volatile("prefetch.global.L1 [%0];" ::"l"(ngm + P.n_words));
                }
            }
        }
        const uint32_t stage_s = smem_s + s * P.stage_bytes;
        bool waited = false;

        if (!P.strided) {
            const uint32_t n_pieces = (nrows + U - 1) / U;
            for (uint32_t p = wib; p < n_pieces; p += NW) {
                const uint32_t j0 = p * U, cnt = min(U, nrows - j0);
                const int64_t id0 = row0 + j0;
                if (p != (uint32_t)wib) load_piece(id0, cnt, my_off, my_flag);   // later pieces of the chunk: on demand
                const uint32_t flags = __ballot_sync(0xFFFFFFFFu, my_flag);
                uint8_t* orow = P.out + (uint64_t)(out0 + j0) * P.row_bytes;
                uint32_t r = 0;
                while (r < cnt) {
                    const uint64_t g = group_of_u(P.group_param, P.group_shift, (uint64_t)(id0 + r));
                    if (g != prep_g) prepare(g);
                    if (!waited) { mbar_wait(full_s + s * 8, (k / NS) & 1u); waited = true; }
                    if (r + RB <= cnt && ((flags >> r) & ((1u << RB) - 1u)) == ((1u << RB) - 1u) &&
                        group_of_u(P.group_param, P.group_shift, (uint64_t)(id0 + r + RB - 1)) == g) {
                        uint32_t sa[RB];                                   // RB compressed rows of one group
#pragma unroll
                        for (int i = 0; i < RB; ++i) sa[i] = stage_s + (__shfl_sync(0xFFFFFFFFu, my_off, r + i) - base_off) * 16u;
                        decode_rows(sa, orow);
                        r += RB; orow += (size_t)RB * P.row_bytes;
                    } else {
                        const uint32_t roff = (__shfl_sync(0xFFFFFFFFu, my_off, r) - base_off) * 16u;
                        decode_row(stage_s + roff, (flags >> r) & 1u, orow);
                        r += 1; orow += P.row_bytes;
                    }
                }
            }
        } else {
            // nrows consecutive ids = whole matrix rows of S tiles (plus a ragged tail); warp <-> tile, lane <-> matrix row
            const uint32_t n_mr = (uint32_t)((nrows + S - 1) / S);
            for (uint32_t t = wib; t < (uint32_t)S; t += NW) {
                const uint32_t cnt = t < nrows ? (uint32_t)((nrows - t + S - 1) / S) : 0u;   // rows of tile t in this chunk
                if (!cnt) continue;
                const int64_t idl = row0 + (int64_t)t + (int64_t)lane * (int64_t)S;
                const uint32_t t_off = lane < cnt ? __ldg(P.row_off + idl) - base_off : 0u;
                const uint32_t t_flag = lane < cnt ? (__ldg(P.row_flag + (idl >> 5)) >> (idl & 31)) & 1u : 0u;
                const uint32_t flags = __ballot_sync(0xFFFFFFFFu, t_flag);
                if ((uint64_t)t != prep_g) prepare(t);
                if (!waited) { mbar_wait(full_s + s * 8, (k / NS) & 1u); waited = true; }
                for (uint32_t r = 0; r < cnt; ++r) {
                    const uint32_t roff = __shfl_sync(0xFFFFFFFFu, t_off, r) * 16u;
                    decode_row(stage_s + roff, (flags >> r) & 1u, P.out + (uint64_t)(out0 + t + (int64_t)r * (int64_t)S) * P.row_bytes);
                }
            }
            (void)n_mr; (void)my_off; (void)my_flag;
        }
        if (!waited) mbar_wait(full_s + s * 8, (k / NS) & 1u);   // a warp without a piece still has to follow the phases
        __syncwarp();
        if (lane == 0) asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(empty_s + s * 8) : "memory");
    }
}
