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
    uint32_t nsplit, split_rows;   // ibp_stream_t2_kernel: a chunk above one stage is loaded as nsplit sub-loads of split_rows rows (0/1 = never)
    // ibp_stream_t2_kernel: a stage = [packed bytes: stage_bytes - aux_bytes][aux: descriptor (32 B), row offsets, row flags, Mask/Bitval]
    uint32_t aux_bytes, aux_flag_off, aux_meta_off;   // offsets inside the aux region; aux_meta_off = 0: Mask/Bitval are not staged
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

// ------------------------------------------------------------------------------------------------------------------------
// ibp_stream_t2_kernel -- the thresholded stream decode for rows of 16*LPR bytes (LPR = 8, 16 or 32 lanes per row; W = 4
// words per lane: 128 / 256 / 512-byte rows, i.e. every BASELINE workload).  Blocked groups only (strided tables keep the
// kernel above).  Built around two measurements of the kernel above (ncu, profiles/r01_resident_ncu.md, r02_resident_ncu.md):
// the instruction count per row, and the long-scoreboard stalls of the consumer warps' own global loads.
//
// EVERYTHING a consumer warp reads comes out of shared memory.  The producer lane walks the chunks (the only place that reads
// ids and row offsets from global memory) and loads UNITS: a unit is a chunk, or -- when the chunk's stored bytes exceed a stage,
// which only happens with many raw rows -- one of its sub-ranges of split_rows rows.  For every unit it writes a 32-byte
// descriptor {first row id, first output row, rows, offset of the first row, last-unit-of-the-chunk flag, last-unit-of-the-CTA flag} into the stage and
// issues bulk copies of (1) the unit's packed bytes (contiguous: rows lie back to back), (2) the 16-byte cover of the unit's row
// offsets, (3) the cover of its row-flag words and (4) Mask/Bitval of the table groups it touches (consecutive groups
// are contiguous in GPU memory: "shared-memory staging of the metadata") -- all completing on the stage's full barrier.  The
// consumers wait for the barrier, read the descriptor and never touch global memory except to store rows: no prefetch state in
// registers, no long-scoreboard stalls, and the same code for span gathers, ranges and resident decode.
//
// Consumer side:
//   - a warp decodes 32/LPR rows per pass, one row per group of LPR lanes (256-byte rows: two at a time), so the per-row fixed
//     work (participation read, counts, scan, address set-up, store) is shared by twice or four times the data;
//   - the lane groups of a pass take rows of DIFFERENT parts of the piece (group of lanes s: rows [s*Q, (s+1)*Q)), so with small
//     groups (KV: 16 rows) one set-up -- Mask/Bitval loads, run masks or expand masks -- prepares two or four groups at once;
//   - a unit is NW pieces, one per consumer warp, so every warp works on every stage and the stages double-buffer;
//   - raw rows take the SAME code with an empty header and no participating chunk (every chunk then contributes its 32
//     bits at offset 32*c), so a pass never diverges on the row kind;
//   - the bits a lane's 4 chunks store (P:319 step 2) come from ONE dp4a: -popc(Mask) of the 4 chunks sit as signed bytes in one
//     register, the 4 participation bits are spread to bytes by a multiply, and the dot product + 128 is the lane's total;
//   - the inclusive scan over the lanes of a row (P:319 step 3) runs on two rows packed into one register (16 bits each: a row
//     stores at most 4,096 bits), each step a shuffle whose in-range predicate guards the add, and RB = 2 passes are written out
//     side by side, branch-free, so that their dependency chains interleave;
//   - chunk q of a lane is read q words past (the lane's first bit - the bits removed in front of q): one predicated subtraction
//     per chunk, the word offset an immediate of the shared-memory load;
//   - the integer ALU pipe was the binding unit (ncu: 70 % busy at half rate with the FMA pipe at 19 %), so sums, scalings and
//     flags are written as (predicated) IMAD work wherever arithmetic allows, and whole pieces take a pass body without the
//     repeat / valid handling; row ids and group numbers are 32-bit here (the launcher takes this kernel below 2^32 rows), and
//     the consumers carry no chunk counter: they follow the producer's units until the descriptor marks the CTA's last one;
//   - NR (handle level: the most runs of variant bits in any Mask word of the table): bits go back run by run with exactly NR
//     multiply + and-or pairs; NR = 0 selects the five-stage expand.
__device__ __forceinline__ void mbar_wait_relaxed(uint32_t bar, uint32_t parity) {
    // wait with a suspend-time hint: a waiting warp stays off the issue port instead of polling
    uint32_t ok = 0;
    while (!ok) {
        asm volatile(
            "{\n\t.reg .pred p;\n\t"
            "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2, %3;\n\t"
            "selp.u32 %0, 1, 0, p;\n\t}"
            : "=r"(ok) : "r"(bar), "r"(parity), "r"(20000u) : "memory");
    }
}
__device__ __forceinline__ void mbar_wait_backoff(uint32_t bar, uint32_t parity) {
    // the producer lane's wait for a free stage: a plain try_wait loop comes back every ~25 cycles and its three instructions per
    // round were 9-18 % of everything the kernel issued (ncu source counters); sleeping ~100 ns between tries costs 1 % of a unit's
    // decode time in reaction at worst, and the refill has a whole stage of decode to hide behind
    for (;;) {
        uint32_t ok;
        asm volatile(
            "{\n\t.reg .pred p;\n\t"
            "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
            "selp.u32 %0, 1, 0, p;\n\t}"
            : "=r"(ok) : "r"(bar), "r"(parity) : "memory");
        if (ok) break;
        __nanosleep(100);
    }
}
__device__ __forceinline__ uint32_t lds32(uint32_t a) {
    uint32_t v;
    asm volatile("ld.shared.u32 %0, [%1];" : "=r"(v) : "r"(a));
    return v;
}
__device__ __forceinline__ void lds128(uint32_t a, uint32_t (&v)[4]) {
    asm volatile("ld.shared.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]) : "r"(a));
}

template <int LPR, int NS, int NW, int NR>
__global__ void __launch_bounds__((NW + 1) * 32, 3) ibp_stream_t2_kernel(const StreamTParams P) {
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
    const uint32_t data_cap = P.stage_bytes - P.aux_bytes;       // stage = [packed bytes][aux]
    const uint32_t cap16 = (data_cap - 64u) / 16u;               // what one stage holds, in 16-byte units
    const uint32_t row_bytes2 = 2u * P.row_bytes;

    if (wib == NW) {
        // ------------------------------------------------------------------ producer: one lane walks the chunks
        if (lane != 0) return;
        uint32_t k = 0;
        for (int64_t c = blockIdx.x; c < P.n_chunks; c += gridDim.x) {
            const int64_t si = !P.ids ? 0 : (P.n_chunks <= 0x7FFFFFFFll ? (int64_t)((uint32_t)c / P.chunks_per_span) : c / P.chunks_per_span);
            const int64_t cc = c - si * P.chunks_per_span;
            const int64_t span_first = P.ids ? P.ids[si] * P.span_rows : P.first_row;
            const int64_t r = cc * (int64_t)P.rows_per_chunk;
            const int64_t row0 = span_first + r, out0 = si * P.span_rows + r;
            const uint32_t nrows = (uint32_t)min((int64_t)P.rows_per_chunk, P.span_rows - r);
            const uint32_t o0 = __ldg(P.row_off + row0), o1 = __ldg(P.row_off + row0 + nrows);
            const bool split = P.nsplit > 1 && o1 - o0 > cap16;
            const uint32_t step = split ? P.split_rows : nrows;
            for (uint32_t r0 = 0; r0 < nrows; r0 += step, ++k) {
                const uint32_t s = k % NS, r1 = min(nrows, r0 + step), n = r1 - r0;
                const uint32_t a0 = split ? __ldg(P.row_off + row0 + r0) : o0, a1 = split ? __ldg(P.row_off + row0 + r1) : o1;
                const int64_t first = row0 + r0;
                // covers, all 16-byte aligned at both ends: row offsets [first, first + n] from index first & ~3, flag words from
                // word (first >> 5) & ~3, Mask/Bitval of groups g0 .. g1
                const int64_t oi = first & ~3ll;
                const uint32_t off_bytes = (uint32_t)(((first + n + 1 - oi) + 3) & ~3ll) * 4u;
                const int64_t fw = (first >> 5) & ~3ll;
                const uint32_t flag_bytes = (uint32_t)(((((first + n - 1) >> 5) + 1 - fw) + 3) & ~3ll) * 4u;
                const uint64_t g0 = group_of_u(P.group_param, P.group_shift, (uint64_t)first);
                const uint64_t g1 = group_of_u(P.group_param, P.group_shift, (uint64_t)first + n - 1);
                const uint32_t meta_bytes = P.aux_meta_off ? (uint32_t)(g1 - g0 + 1) * row_bytes2 : 0u;
                const uint32_t bytes = (a1 - a0) * 16u;
                const uint32_t stage_s = smem_s + s * P.stage_bytes, aux_s = stage_s + data_cap, bar = full_s + s * 8;
                mbar_wait_backoff(empty_s + s * 8, ((k / NS) & 1u) ^ 1u);   // (a wait with a 20 us suspend hint reacts late and the refill starts late)
                asm volatile("st.shared.v4.u32 [%0], {%1,%2,%3,%4};" ::"r"(aux_s), "r"((uint32_t)first), "r"((uint32_t)((uint64_t)first >> 32)),
                             "r"((uint32_t)(out0 + r0)), "r"((uint32_t)((uint64_t)(out0 + r0) >> 32)) : "memory");
                asm volatile("st.shared.v4.u32 [%0], {%1,%2,%3,%4};" ::"r"(aux_s + 16u), "r"(n), "r"(a0), "r"(r1 == nrows ? 1u : 0u),
                             "r"(r1 == nrows && c + (int64_t)gridDim.x >= P.n_chunks ? 1u : 0u) : "memory");   // .w: the CTA's last unit
                mbar_expect_tx(bar, bytes + off_bytes + flag_bytes + meta_bytes);     // release: the descriptor is visible to whoever sees the phase complete
                bulk_g2s(aux_s + 32u, P.row_off + oi, off_bytes, bar);
                bulk_g2s(aux_s + P.aux_flag_off, P.row_flag + fw, flag_bytes, bar);
                if (meta_bytes) bulk_g2s(aux_s + P.aux_meta_off, P.meta + g0 * 2ull * P.n_words, meta_bytes, bar);
                const uint8_t* src = P.store + (16ull * a0 - P.bias);
                for (uint32_t o = 0; o < bytes; o += 16384u)
                    bulk_g2s(stage_s + o, src + o, min(16384u, bytes - o), bar);
            }
        }
        return;
    }

    // ---------------------------------------------------------------------- consumers
    constexpr int W = 4, RPP = 32 / LPR, RB = 2;
    constexpr int NMV = NR ? 2 * NR : 5;
    const uint32_t sub = (uint32_t)lane / LPR, sl = (uint32_t)lane % LPR;      // lane group (row of a pass), lane inside the row
    const uint32_t w0 = sl * W;                                                // first chunk (32-bit word) of this lane
    const uint32_t hdr_off = (w0 >> 5) * 4u, hdr_sh = w0 & 31u;                // where the lane's 4 participation bits sit
    uint32_t m[W], b[W], mv[W][NMV], kq[W], pm4 = 0, npm4 = 0;                 // kq: bits a participating chunk leaves out (popc(Mask)); pm4: popc(Mask) of the 4 chunks, one per byte; npm4: minus that, as signed bytes
    // Row ids and group numbers are 32-bit on the consumer side (the launcher takes this kernel only for tables below 2^32 rows):
    // half the registers and instructions of the per-piece bookkeeping.
    auto group_of = [&](uint32_t id) -> uint32_t { return P.group_shift != 0xFFFFFFFFu ? id >> P.group_shift : id / P.group_param; };
    uint32_t prep_g = ~0u;                                                     // per lane: lane groups may hold different groups
    bool five = true;                                                          // NR = 0: some bit of the prepared groups moves by >= 16 (warp-uniform)

    // S2 for group g: Mask/Bitval from the stage's aux region (meta_s = shared address of group g0's record), else from global memory
    auto prepare = [&](uint32_t g, uint32_t g0, uint32_t meta_s) {
        if (P.aux_meta_off) {
            const uint32_t a = meta_s + (uint32_t)(g - g0) * row_bytes2 + w0 * 4u;
            lds128(a, m);
            lds128(a + P.row_bytes, b);
        } else {
            const uint32_t* gm = P.meta + (uint64_t)g * 2ull * P.n_words;
            VecIO<W>::ld(gm + w0, m);
            VecIO<W>::ld(gm + P.n_words + w0, b);
        }
        pm4 = 0;
#pragma unroll
        for (int q = 0; q < W; ++q) { const uint32_t pc = (uint32_t)__popc(m[q]); kq[q] = pc; pm4 |= pc << (8 * q); }   // <= 32 each
        npm4 = (0x80808080u - pm4) ^ 0x80808080u;                                // per byte: -popc (no borrow crosses a byte: 0x80 - pc > 0)
        if constexpr (NR > 0) {
#pragma unroll
            for (int q = 0; q < W; ++q) {
                uint32_t nv = ~m[q], c = 0;
#pragma unroll
                for (int j = 0; j < NR; ++j) {
                    const uint32_t low = nv & (0u - nv), t = nv + low, run = nv & ~t;   // nv == 0 -> low = run = 0
                    mv[q][j] = low >> c;                                         // 2^(p_j - c_j): run j moves up by (its position - bits below it)
                    mv[q][NR + j] = run;
                    c += __popc(run);
                    nv &= t;
                }
            }
        } else {
            // five-stage expand: only the stages that can move a bit are computed (a bit moves by the number of invariant bits below
            // it, at most popc(Mask word)); warp-uniform, so the branches do not diverge
            const uint32_t pmax = __reduce_max_sync(0xFFFFFFFFu, max(max(pm4 & 0xFFu, (pm4 >> 8) & 0xFFu), max((pm4 >> 16) & 0xFFu, pm4 >> 24)));
            const int nstg = pmax >= 16u ? 5 : pmax >= 8u ? 4 : pmax >= 4u ? 3 : pmax >= 2u ? 2 : pmax >= 1u ? 1 : 0;
            five = nstg == 5;
            bool shared = false;
            if constexpr (RPP == 2) shared = __all_sync(0xFFFFFFFFu, g == __shfl_xor_sync(0xFFFFFFFFu, g, 16));
            if (shared) {
                // both half-warps hold the SAME group (pieces of one 16-row group, KV): each half derives the masks of two of the
                // lane's four words and the halves swap results -- 10 shuffles instead of two more mask derivations
                if constexpr (RPP == 2) {
                    uint32_t t0[5], t1[5];
                    expand_masks_n(~(sub ? m[2] : m[0]), t0, nstg);
                    expand_masks_n(~(sub ? m[3] : m[1]), t1, nstg);
#pragma unroll
                    for (int i = 0; i < 5; ++i) {
                        const uint32_t o0 = __shfl_xor_sync(0xFFFFFFFFu, t0[i], 16), o1 = __shfl_xor_sync(0xFFFFFFFFu, t1[i], 16);
                        mv[0][i] = sub ? o0 : t0[i]; mv[1][i] = sub ? o1 : t1[i];
                        mv[2][i] = sub ? t0[i] : o0; mv[3][i] = sub ? t1[i] : o1;
                    }
                }
            } else {
#pragma unroll
                for (int q = 0; q < W; ++q) {
                    if (q > 0 && m[q] == m[q - 1]) {
#pragma unroll
                        for (int i = 0; i < 5; ++i) mv[q][i] = mv[q - 1][i];
                    } else {
                        expand_masks_n(~m[q], mv[q], nstg);
                    }
                }
            }
        }
        prep_g = g;
    };
    auto reinsert = [&](auto nstg_c, uint32_t x, int q) -> uint32_t {
        if constexpr (NR > 0) {
            uint32_t acc = b[q];
#pragma unroll
            for (int j = 0; j < NR; ++j) acc = and_or(x * mv[q][j], mv[q][NR + j], acc);
            return acc;
        } else {
            return bitselect(b[q], expand_bits<decltype(nstg_c)::value>(x, mv[q]), m[q]);
        }
    };

    // RB passes side by side: lane group `sub` decodes row rr[i] of the piece in pass i (valid[i] = 0: the row is a repeat whose
    // result is not stored).  my_off / flags: offsets (lane i <-> row i of the piece) and compressed-bits of the piece.
    auto decode_rows_n = [&](auto nstg_c, auto full_c, const uint32_t (&rr)[RB], const uint32_t (&valid)[RB], uint32_t my_off, uint32_t flags, uint32_t base_off,
                             uint32_t stage_s, uint8_t* orow0) {
        // Per pass: the bits this lane's four chunks store (kept: kq[q] if the chunk participates, else all 32) as running sums
        // rel[q] (bits in front of chunk q inside the lane) and tot; the exclusive scan of tot over the lanes of the row (P:319 step
        // 3) gives the lane's first bit.  The integer (ALU) pipe is what binds this kernel (ncu: 70 % busy at half rate, the FMA pipe
        // 19 %), so the arithmetic is arranged for the FMA pipe: sums are predicated adds, the compressed-row flag enters as a
        // multiplier, shared-memory words are addressed by WORD index (the scaled address mode takes the shift).
        uint32_t bw[RB], part[RB], tot[RB];
#pragma unroll
        for (int i = 0; i < RB; ++i) {
            const uint32_t sa = stage_s + (__shfl_sync(0xFFFFFFFFu, my_off, rr[i]) - base_off) * 16u;
            const uint32_t comp = (flags >> rr[i]) & 1u;
            const uint32_t h = lds32(sa + hdr_off);
            part[i] = (h >> hdr_sh) & (comp * 0xFu);                           // raw row: no chunk participates ...
            const uint32_t sel = (part[i] * 0x00204081u) & 0x01010101u;        // participation bit q -> byte q = 1
            tot[i] = (uint32_t)__dp4a((int)npm4, (int)sel, 128);               // bits this lane's four chunks store: 128 - sum of popc(Mask) over its participating chunks (P:319 step 2)
            bw[i] = sa * 8u + comp * P.n_words;                                 // ... and there is no header; a BIT address
        }
        static_assert(RB == 2, "the packed scan holds two passes");
        uint32_t inc = tot[0] | (tot[1] << 16);                                // inclusive scan over the lanes of a row: <= 4,096 per row
#pragma unroll
        for (int d = 1; d < LPR; d <<= 1)
            asm volatile("{\n\t.reg .pred p;\n\t.reg .u32 v;\n\t"
                "shfl.sync.up.b32 v|p, %0, %1, %2, 0xffffffff;\n\t@p add.u32 %0, %0, v;\n\t}"
                : "+r"(inc) : "r"(d), "r"((32 - LPR) << 8));
#pragma unroll
        for (int i = 0; i < RB; ++i) {
            // t = the lane's first bit minus the bits removed in front of chunk q: chunk q sits at bit t + 32 q, i.e. q words further
            // on (an immediate in the load) with the same shift; each participating chunk takes popc(Mask) off t (a predicated add)
            uint32_t t = bw[i] + (i == 0 ? (inc & 0xFFFFu) : (inc >> 16)) - tot[i];   // plus the bits stored by the lanes in front
            uint32_t o[W];
#pragma unroll
            for (int q = 0; q < W; ++q) {
                const bool in = (part[i] & (1u << q)) != 0u;
                uint32_t lo, hi, wi;
                asm("shr.u32 %0, %1, 5;" : "=r"(wi) : "r"(t));                   // word index (kept apart from the *4: one shift on the ALU pipe, the scaling elsewhere)
                asm volatile("ld.shared.u32 %0, [%2];\n\tld.shared.u32 %1, [%2+4];" : "=r"(lo), "=r"(hi) : "r"(wi * 4u + 4u * q));
                const uint32_t x = __funnelshift_r(lo, hi, t);                 // shift = t mod 32
                const uint32_t e = reinsert(nstg_c, x, q);
                o[q] = in ? e : x;                                             // non-participating chunk: all 32 bits
                if (q + 1 < W)
                    asm("{\n\t.reg .pred p;\n\tsetp.ne.u32 p, %1, 0;\n\t@p sub.u32 %0, %0, %2;\n\t}" : "+r"(t) : "r"((uint32_t)in), "r"(kq[q]));
            }
            constexpr uint32_t ROWB = 16u * LPR;                                   // = P.row_bytes (the launcher picks LPR from it)
            uint8_t* dst = decltype(full_c)::value ? orow0 + (size_t)i * ROWB : orow0 + (size_t)rr[i] * ROWB;   // whole piece: orow0 is pass 0's row, rows are consecutive
            if constexpr (decltype(full_c)::value)                                 // ... and every pass stores
                asm volatile("st.global.cs.v4.b32 [%0], {%1,%2,%3,%4};" ::"l"(dst), "r"(o[0]), "r"(o[1]), "r"(o[2]), "r"(o[3]) : "memory");
            else
                asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.u32 p, %5, 0;\n\t@p st.global.cs.v4.b32 [%0], {%1,%2,%3,%4};\n\t}"
                             ::"l"(dst), "r"(o[0]), "r"(o[1]), "r"(o[2]), "r"(o[3]), "r"(valid[i]) : "memory");
        }
    };
    // NR = 0: two copies of the pass body, with and without the stage that moves bits by 16 (bf16 pairs with a few invariant
    // exponent bits per half never need it); the choice is per prepared group and warp-uniform
    auto decode_rows = [&](auto full_c, const uint32_t (&rr)[RB], const uint32_t (&valid)[RB], uint32_t my_off, uint32_t flags, uint32_t base_off,
                           uint32_t stage_s, uint8_t* orow0) {
        using std::integral_constant;
        if (NR > 0 || five) decode_rows_n(integral_constant<int, 5>{}, full_c, rr, valid, my_off, flags, base_off, stage_s, orow0);
        else decode_rows_n(integral_constant<int, 4>{}, full_c, rr, valid, my_off, flags, base_off, stage_s, orow0);
    };

    // One piece: rows id0 .. id0 + cnt - 1 (cnt <= 32), all inside the stage.  orow = output address of row 0 of the piece.
    const uint32_t U = P.piece_rows;
    const uint32_t Q = (U + RPP - 1) / RPP;                                    // rows of a piece per lane group
    auto decode_piece = [&](uint32_t id0, uint32_t cnt, uint32_t my_off, uint32_t flags, uint32_t base_off, uint32_t stage_s, uint8_t* orow,
                            uint32_t g0, uint32_t meta_s) {
        orow += (size_t)w0 * 4;
        const uint32_t qs = min(cnt, sub * Q), qe = min(cnt, qs + Q);
        const bool have = qs < qe;
        uint32_t glo = 0, ghi = 0;
        if (have) {
            glo = group_of(id0 + qs);
            ghi = group_of(id0 + qe - 1);
        }
        if (__all_sync(0xFFFFFFFFu, !have || glo == ghi)) {
            // every lane group's rows lie in one group of the table: one set-up per piece, possibly of several groups at once
            const uint32_t g = have ? glo : group_of(id0);
            if (__any_sync(0xFFFFFFFFu, g != prep_g)) prepare(g, g0, meta_s);
            if (cnt == RPP * Q && Q % RB == 0) {
                // a whole piece (all but the tail of a span or range): every lane group has Q rows, no pass is a repeat
                uint8_t* po = orow + (size_t)qs * (16u * LPR);
                for (uint32_t i = 0; i < Q; i += RB, po += (size_t)RB * (16u * LPR)) {
                    uint32_t rr[RB], valid[RB];
#pragma unroll
                    for (int j = 0; j < RB; ++j) { rr[j] = qs + i + j; valid[j] = 1u; }
                    decode_rows(std::true_type{}, rr, valid, my_off, flags, base_off, stage_s, po);
                }
            } else {
                const uint32_t n_it = min(Q, cnt);
                for (uint32_t i = 0; i < n_it; i += RB) {
                    uint32_t rr[RB], valid[RB];
#pragma unroll
                    for (int j = 0; j < RB; ++j) {
                        const uint32_t r = qs + i + j;
                        valid[j] = r < qe;
                        rr[j] = valid[j] ? r : (have ? qs : 0u);
                    }
                    decode_rows(std::false_type{}, rr, valid, my_off, flags, base_off, stage_s, orow);
                }
            }
        } else {
            // a table group ends inside a lane group's rows (a range that starts off a group boundary): run by run of one group
            uint32_t r = 0;
            while (r < cnt) {
                const uint32_t id = id0 + r;
                const uint32_t g = group_of(id);
                const uint32_t r_end = (uint32_t)min((uint64_t)cnt, (uint64_t)r + (((uint64_t)g + 1) * S - id));
                if (__any_sync(0xFFFFFFFFu, g != prep_g)) prepare(g, g0, meta_s);
                for (; r < r_end; r += RB * RPP) {
                    uint32_t rr[RB], valid[RB];
#pragma unroll
                    for (int j = 0; j < RB; ++j) {
                        const uint32_t x = r + (uint32_t)j * RPP + sub;
                        valid[j] = x < r_end;
                        rr[j] = valid[j] ? x : r;
                    }
                    decode_rows(std::false_type{}, rr, valid, my_off, flags, base_off, stage_s, orow);
                }
                r = r_end;
            }
        }
    };

    // The consumers follow the producer's units until the descriptor says "last unit of this CTA": no chunk counter on this side
    // (a 64-bit chunk index, then a 32-bit down-counter, were spilled under the 72-register budget, and the reload at the end of
    // every unit was 4-7 % of the stall samples).
    if ((int64_t)blockIdx.x >= P.n_chunks) return;
    uint32_t k = 0, fin;
    {
        do {                                                                   // the CTA's units, in the producer's order
            const uint32_t s = k % NS, stage_s = smem_s + s * P.stage_bytes, aux_s = stage_s + data_cap;
            mbar_wait_relaxed(full_s + s * 8, (k / NS) & 1u);
            uint32_t d0[4], d1[4];
            lds128(aux_s, d0);
            lds128(aux_s + 16u, d1);
            const uint32_t first = d0[0];                                    // (d0[1] = 0: below 2^32 rows)
            const int64_t out0 = (int64_t)(((uint64_t)d0[3] << 32) | d0[2]);
            const uint32_t n = d1[0], base_off = d1[1];
            fin = d1[3];
            const uint32_t off_s = aux_s + 32u - (first & ~3u) * 4u;                    // shared address of row_off[0] (wraps mod 2^32: only differences matter)
            const uint32_t fw = (first >> 5) & ~3u;
            const uint32_t g0 = group_of(first);
            for (uint32_t j0 = wib * U; j0 < n; j0 += NW * U) {
                const uint32_t cnt = min(U, n - j0);
                const uint32_t id0 = first + j0;
                const uint32_t my_off = (uint32_t)lane < cnt ? lds32(off_s + (id0 + (uint32_t)lane) * 4u) : 0u;
                const uint32_t fa = aux_s + P.aux_flag_off + ((id0 >> 5) - fw) * 4u;
                uint32_t flags = __funnelshift_r(lds32(fa), lds32(fa + 4u), id0 & 31u);   // bit r = flag of row id0 + r
                if (cnt < 32u) flags &= (1u << cnt) - 1u;
                decode_piece(id0, cnt, my_off, flags, base_off, stage_s, P.out + (uint64_t)(out0 + j0) * P.row_bytes, g0, aux_s + P.aux_meta_off);
            }
            __syncwarp();
            if (lane == 0) asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(empty_s + s * 8) : "memory");
            ++k;
        } while (!fin);
    }
}
