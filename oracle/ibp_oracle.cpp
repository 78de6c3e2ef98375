// ibp_oracle.cpp -- TEST INFRASTRUCTURE ONLY.  Plain, slow, single-threaded CPU oracle for Invariant Bit Packing.
//
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may build, load or call
// this file.  It shares no code, header, table or helper with the CUDA library (paper_2605_30728_b200/csrc): it is
// written from /root/reference/PAPER.md ("P:<line>") and from SURVEY.md section 8(c) ("S8c"), bit by bit, in the
// paper's order, so that a reader can check it against the text by eye.  No blocking, no word tricks, no threads.
//
// Conventions (R4): bit p of a row is bit (p mod 8) of byte (p div 8); the packed stream is
// LSB-first in the same sense.  A "row" is the paper's "tensor"; a "group" is the paper's "cluster" whose
// members are fixed runs of rows.
//
// Parity pins (tests/test_oracle_pins.py, all -m "not gpu"):
//   ibp_oracle_group_masks   : brute force over all rows in Python; closed form AND/OR; invariants P:231, P:237;
//                              hand-worked fixture tests/golden/worked_example_strict.txt
//   ibp_oracle_pack_row      : canonical-order construction (row j of the 2^k-row group packs to integer j);
//                              all-variant group == memcpy; sizes == ceil(k/8)
//   ibp_oracle_unpack_row    : round trip on random bit patterns for masks of every popcount; k=0 == Bitval broadcast
//   ibp_oracle_build/gather  : equals the plain gather out[i] = X[ids[i]] byte for byte (losslessness);
//                              the group partition (blocked with a ragged last group, strided with n % S != 0 and n < S):
//                              every group's Mask/Bitval equal those computed from exactly X[gG:(g+1)G] / X[g::S] by
//                              Python-integer brute force and by the AND/OR closed form (test_dataset_group_partition)
//   thresholded mode (T<N)   : round trip; compressed <= raw; participation overhead row_bytes/CS bits
//                              (P:527 prints 12.5% and 1.6%); at T=N payload == strict payload; hand-worked fixtures
//                              tests/golden/worked_example_thresholded.txt, worked_example_mixed_chunks.txt
//   ibp_oracle_build_T/gather: equals the plain gather byte for byte; bitmask bytes = ceil(n_rows/8); at tau=1
//                              Mask/Bitval equal the strict dataset's; T = ceil(tau N_g) against Fig. 2's T=4, N=5;
//                              hand-worked 5-row dataset fixture (sizes, flags, stored bytes)
//   ibp_oracle_T_append      : append then gather == plain gather of the concatenated table; Mask/Bitval unchanged by an append;
//                              an appended row's stored bytes == ibp_oracle_compress_row_T under the group's existing masks (the
//                              row-level function is pinned above); the in-place slot image (row r in its original slot,
//                              the first `size` bytes meaningful) has capacity x row_bytes bytes: the closed form of P:361
//   Ratios on the paper's real datasets (Tables 2, 4, 5): parity unpinned -- the datasets are not available.
//
// Build: g++ -O1 -shared -fPIC oracle/ibp_oracle.cpp -o oracle/libibp_oracle.so
#include <cstdint>
#include <cstdlib>
#include <cstring>
#include <vector>

namespace {

inline int get_bit(const uint8_t* buf, uint64_t p) { return (buf[p >> 3] >> (p & 7)) & 1; }
inline void put_bit(uint8_t* buf, uint64_t p, int v) {
    if (v) buf[p >> 3] = (uint8_t)(buf[p >> 3] | (1u << (p & 7)));
    else   buf[p >> 3] = (uint8_t)(buf[p >> 3] & ~(1u << (p & 7)));
}

}  // namespace

extern "C" {

// ---------------------------------------------------------------------------------------------------------------
// Preprocessing, P:229-231 (section 4.1), applied to one group (cluster) with threshold T.
//   "A counter is allocated for each bit ... For each set bit in each input tensor, we increment the corresponding
//    counter".  "If the value of a counter is more than T, that corresponding bit is set to 1 in the Mask and
//    Bitval ... If the value is less than N - T ... set to 1 in the Mask and to 0 in the Bitval ... Otherwise the bit
//    in Mask is 0 ... We keep these bits as 0".
// Reading R2 (S8c): the comparisons are >= T and <= N - T ("at least T/N"; Fig. 2's T=4,N=5 needs it).  The
// strict group mode of the graded path is T = N: a bit is invariant iff every row of the group agrees.
// rows: n rows of row_bytes bytes, row r at rows + r*row_stride.  counters: optional out, 8*row_bytes entries.
// Returns k = number of variant bits = 8*row_bytes - popcount(Mask).
// ---------------------------------------------------------------------------------------------------------------
uint32_t ibp_oracle_group_masks_T(const uint8_t* rows, uint64_t n, uint64_t row_stride, uint32_t row_bytes, uint64_t T,
                                  uint8_t* mask, uint8_t* bitval, uint64_t* counters) {
    const uint64_t nbits = 8ull * row_bytes;
    std::vector<uint64_t> c1(nbits, 0);
    for (uint64_t r = 0; r < n; ++r)
        for (uint64_t p = 0; p < nbits; ++p)
            if (get_bit(rows + r * row_stride, p)) c1[p] += 1;
    std::memset(mask, 0, row_bytes);
    std::memset(bitval, 0, row_bytes);
    uint32_t k = 0;
    for (uint64_t p = 0; p < nbits; ++p) {
        if (c1[p] >= T) { put_bit(mask, p, 1); put_bit(bitval, p, 1); }          // invariant, value 1
        else if (c1[p] <= n - T) { put_bit(mask, p, 1); put_bit(bitval, p, 0); } // invariant, value 0
        else { k += 1; }                                                          // variant: Mask 0, Bitval kept 0
        if (counters) counters[p] = c1[p];
    }
    return k;
}

// Strict group mode: T = N (S8c strict step 3: Mask[p]=1 iff c1==N or c1==0).
uint32_t ibp_oracle_group_masks(const uint8_t* rows, uint64_t n, uint64_t row_stride, uint32_t row_bytes,
                                uint8_t* mask, uint8_t* bitval) {
    return ibp_oracle_group_masks_T(rows, n, row_stride, row_bytes, n, mask, bitval, nullptr);
}

// ---------------------------------------------------------------------------------------------------------------
// Strict compression of one row, "the matching bits are removed", P:292-295 insertBits at the running bit
// offset; S8c strict step 5: walk p ascending, append bit p wherever Mask[p]=0, zero-pad the last byte (P:241
// "We keep all the tensors byte-aligned").  packed must hold ceil(k/8) bytes.  Returns k.
// ---------------------------------------------------------------------------------------------------------------
uint32_t ibp_oracle_pack_row(const uint8_t* row, const uint8_t* mask, uint32_t row_bytes, uint8_t* packed) {
    const uint64_t nbits = 8ull * row_bytes;
    uint64_t q = 0;
    for (uint64_t p = 0; p < nbits; ++p)
        if (!get_bit(mask, p)) q += 1;
    std::memset(packed, 0, (q + 7) / 8);
    q = 0;
    for (uint64_t p = 0; p < nbits; ++p)
        if (!get_bit(mask, p)) { put_bit(packed, q, get_bit(row, p)); q += 1; }
    return (uint32_t)q;
}

// Strict decompression of one row, "reinserting the removed bits", P:319 step 5; S8c strict step 6: start from
// Bitval, walk p ascending, every Mask[p]=0 position takes the next stream bit.
void ibp_oracle_unpack_row(const uint8_t* packed, const uint8_t* mask, const uint8_t* bitval, uint32_t row_bytes,
                           uint8_t* row_out) {
    const uint64_t nbits = 8ull * row_bytes;
    std::memcpy(row_out, bitval, row_bytes);
    uint64_t q = 0;
    for (uint64_t p = 0; p < nbits; ++p)
        if (!get_bit(mask, p)) { put_bit(row_out, p, get_bit(packed, q)); q += 1; }
}

// ---------------------------------------------------------------------------------------------------------------
// Thresholded (paper-default) row codec, S8c thresholded steps 3-7.  Chunks of CS bytes (4 in the evaluation).
//   participates(i) = (Chunk_i AND Mask_i) == Bitval_i
//   bitsSaved = sum over participating chunks of popcount(Mask_i)                        (Fig. 3 lines 5-10)
//   bytesSaved = floor((bitsSaved - row_bytes/CS) / 8); <= 0 -> stored raw               (Fig. 3 lines 13-18)
//   compressed = [participation bits, one per chunk][per chunk: variant bits if participating else all bits]
//                LSB-first, zero padded to row_bytes - bytesSaved bytes                  (R8, R9)
// Returns the stored size in bytes; *is_compressed = 0 when the row is kept raw (the per-row bitmask of P:363).
// ---------------------------------------------------------------------------------------------------------------
static int chunk_participates(const uint8_t* row, const uint8_t* mask, const uint8_t* bitval, uint32_t c, uint32_t CS) {
    for (uint32_t b = 0; b < CS; ++b)
        if ((row[c * CS + b] & mask[c * CS + b]) != bitval[c * CS + b]) return 0;
    return 1;
}

uint32_t ibp_oracle_compress_size_T(const uint8_t* row, const uint8_t* mask, const uint8_t* bitval, uint32_t row_bytes,
                                    uint32_t CS, int* is_compressed) {
    const uint32_t n_chunks = row_bytes / CS;
    int64_t bitsSaved = 0;
    for (uint32_t c = 0; c < n_chunks; ++c)
        if (chunk_participates(row, mask, bitval, c, CS))
            for (uint32_t p = 0; p < 8 * CS; ++p) bitsSaved += get_bit(mask + c * CS, p);
    const int64_t participationBits = n_chunks;
    const int64_t diff = bitsSaved - participationBits;
    const int64_t bytesSaved = diff > 0 ? diff / 8 : 0;   // floor for positive values; non-positive -> not worth it
    if (bytesSaved <= 0) { *is_compressed = 0; return row_bytes; }
    *is_compressed = 1;
    return (uint32_t)(row_bytes - bytesSaved);
}

uint32_t ibp_oracle_compress_row_T(const uint8_t* row, const uint8_t* mask, const uint8_t* bitval, uint32_t row_bytes,
                                   uint32_t CS, uint8_t* out /* row_bytes */, int* is_compressed) {
    const uint32_t size = ibp_oracle_compress_size_T(row, mask, bitval, row_bytes, CS, is_compressed);
    if (!*is_compressed) { std::memcpy(out, row, row_bytes); return row_bytes; }
    const uint32_t n_chunks = row_bytes / CS;
    std::memset(out, 0, row_bytes);
    uint64_t q = 0;
    for (uint32_t c = 0; c < n_chunks; ++c) { put_bit(out, q, chunk_participates(row, mask, bitval, c, CS)); q += 1; }
    for (uint32_t c = 0; c < n_chunks; ++c) {
        const int part = chunk_participates(row, mask, bitval, c, CS);
        for (uint32_t p = 0; p < 8 * CS; ++p) {
            if (part && get_bit(mask + c * CS, p)) continue;          // invariant bit of a matching chunk: removed
            put_bit(out, q, get_bit(row + c * CS, p)); q += 1;
        }
    }
    return size;
}

void ibp_oracle_decompress_row_T(const uint8_t* in, int is_compressed, const uint8_t* mask, const uint8_t* bitval,
                                 uint32_t row_bytes, uint32_t CS, uint8_t* row_out) {
    if (!is_compressed) { std::memcpy(row_out, in, row_bytes); return; }
    const uint32_t n_chunks = row_bytes / CS;
    uint64_t q = n_chunks;                                            // payload starts after the participation bits
    for (uint32_t c = 0; c < n_chunks; ++c) {
        const int part = get_bit(in, c);
        for (uint32_t p = 0; p < 8 * CS; ++p) {
            if (part && get_bit(mask + c * CS, p)) { put_bit(row_out + c * CS, p, get_bit(bitval + c * CS, p)); continue; }
            put_bit(row_out + c * CS, p, get_bit(in, q)); q += 1;
        }
    }
}

// ---------------------------------------------------------------------------------------------------------------
// Dataset level, strict group mode (S8c strict steps 1-7; Appendix A canonical store).
//   group_kind 0 (blocked): group g = rows [g*G, min((g+1)*G, n_rows));      g(id) = id div G
//   group_kind 1 (strided): group t = rows with id mod S == t;                g(id) = id mod S
// Canonical packed store: byte-aligned rows, densely concatenated in row-id order (for blocked groups that is group
// order then row order; for strided groups the S items of matrix row r in tile order) -- no padding anywhere.
// ---------------------------------------------------------------------------------------------------------------
struct ibp_oracle_ds {
    uint64_t n_rows = 0, n_groups = 0;
    uint32_t row_bytes = 0, group_kind = 0, group_param = 0;
    std::vector<uint8_t> mask, bitval;      // n_groups x row_bytes each
    std::vector<uint32_t> k_bits;           // per group
    std::vector<uint64_t> row_offset;       // n_rows + 1 byte offsets into packed
    std::vector<uint8_t> packed;
};

static uint64_t group_of(const ibp_oracle_ds* d, uint64_t id) {
    return d->group_kind == 0 ? id / d->group_param : id % d->group_param;
}

ibp_oracle_ds* ibp_oracle_build(const uint8_t* rows, uint64_t n_rows, uint32_t row_bytes, uint32_t group_kind,
                                uint32_t group_param) {
    if (!rows || n_rows == 0 || row_bytes == 0 || group_param == 0 || group_kind > 1) return nullptr;
    ibp_oracle_ds* d = new ibp_oracle_ds();
    d->n_rows = n_rows; d->row_bytes = row_bytes; d->group_kind = group_kind; d->group_param = group_param;
    d->n_groups = group_kind == 0 ? (n_rows + group_param - 1) / group_param : (n_rows < group_param ? n_rows : group_param);
    d->mask.assign(d->n_groups * row_bytes, 0);
    d->bitval.assign(d->n_groups * row_bytes, 0);
    d->k_bits.assign(d->n_groups, 0);
    for (uint64_t g = 0; g < d->n_groups; ++g) {
        uint64_t first, count, stride;
        if (group_kind == 0) { first = g * group_param; count = n_rows - first < group_param ? n_rows - first : group_param; stride = row_bytes; }
        else { first = g; count = (n_rows - g + group_param - 1) / group_param; stride = (uint64_t)group_param * row_bytes; }
        d->k_bits[g] = ibp_oracle_group_masks(rows + first * row_bytes, count, stride, row_bytes,
                                              &d->mask[g * row_bytes], &d->bitval[g * row_bytes]);
    }
    d->row_offset.assign(n_rows + 1, 0);
    for (uint64_t id = 0; id < n_rows; ++id)
        d->row_offset[id + 1] = d->row_offset[id] + (d->k_bits[group_of(d, id)] + 7) / 8;
    d->packed.assign(d->row_offset[n_rows] + 1, 0);
    for (uint64_t id = 0; id < n_rows; ++id)
        ibp_oracle_pack_row(rows + id * row_bytes, &d->mask[group_of(d, id) * row_bytes], row_bytes, &d->packed[d->row_offset[id]]);
    return d;
}

void ibp_oracle_destroy(ibp_oracle_ds* d) { delete d; }

uint64_t ibp_oracle_n_groups(const ibp_oracle_ds* d) { return d->n_groups; }
uint64_t ibp_oracle_packed_bytes(const ibp_oracle_ds* d) { return d->row_offset[d->n_rows]; }
uint64_t ibp_oracle_metadata_bytes(const ibp_oracle_ds* d) { return 2ull * d->row_bytes * d->n_groups; }
const uint8_t* ibp_oracle_mask(const ibp_oracle_ds* d, uint64_t g) { return &d->mask[g * d->row_bytes]; }
const uint8_t* ibp_oracle_bitval(const ibp_oracle_ds* d, uint64_t g) { return &d->bitval[g * d->row_bytes]; }
uint32_t ibp_oracle_k_bits(const ibp_oracle_ds* d, uint64_t g) { return d->k_bits[g]; }
const uint8_t* ibp_oracle_packed_row(const ibp_oracle_ds* d, uint64_t id, uint64_t* nbytes) {
    *nbytes = d->row_offset[id + 1] - d->row_offset[id];
    return &d->packed[d->row_offset[id]];
}

// S8c strict step 7 with index_span (S8b): out[(i*span + j)] = row ids[i]*span + j, for j in [0, span).
// Returns 0, or 1 if an id is out of range (nothing is written for that id).
int ibp_oracle_gather_decompress(const ibp_oracle_ds* d, const int64_t* ids, int64_t n, uint32_t index_span, uint8_t* out) {
    int bad = 0;
    for (int64_t i = 0; i < n; ++i)
        for (uint32_t j = 0; j < index_span; ++j) {
            const int64_t id = ids[i] * (int64_t)index_span + j;
            if (id < 0 || (uint64_t)id >= d->n_rows) { bad = 1; continue; }
            const uint64_t g = group_of(d, (uint64_t)id);
            ibp_oracle_unpack_row(&d->packed[d->row_offset[id]], &d->mask[g * d->row_bytes], &d->bitval[g * d->row_bytes],
                                  d->row_bytes, out + ((uint64_t)i * index_span + j) * d->row_bytes);
        }
    return bad;
}

// ---------------------------------------------------------------------------------------------------------------
// Dataset level, thresholded mode (the paper's default codec; S8c thresholded steps 1-7).
//   Scope: one Mask/Bitval per group (clustered compression); a single group spanning every row is the paper's
//   global pair ("For the entire dataset, only one Mask and Bitval is constructed").
//   T = ceil(tau * N_g) with tau = thr_num/thr_den ("T=0.8N"), per group, N_g = rows of that group.
//   Every row goes through ibp_oracle_compress_row_T: it is either compressed (participation bits + payloads) or kept
//   raw, and one bit per row records which (the bitmask of P:363; 1 = compressed).
//   Canonical store: the stored bytes of the rows, in row-id order, densely concatenated.  (The paper keeps each row in
//   its original slot; only the first `size` bytes of a slot are meaningful, so the dense form holds the same
//   information.)
// ---------------------------------------------------------------------------------------------------------------
struct ibp_oracle_ds_T {
    uint64_t n_rows = 0, n_groups = 0, n_raw = 0;
    uint32_t row_bytes = 0, group_kind = 0, group_param = 0, CS = 4;
    std::vector<uint8_t> mask, bitval;      // n_groups x row_bytes each
    std::vector<uint64_t> T;                // per group
    std::vector<uint64_t> row_offset;       // n_rows + 1 byte offsets into stored
    std::vector<uint8_t> rowflag;           // ceil(n_rows/8) bytes, bit r = 1 iff row r is compressed
    std::vector<uint8_t> stored;
};

static uint64_t group_of_T(const ibp_oracle_ds_T* d, uint64_t id) {
    return d->group_kind == 0 ? id / d->group_param : id % d->group_param;
}

ibp_oracle_ds_T* ibp_oracle_build_T(const uint8_t* rows, uint64_t n_rows, uint32_t row_bytes, uint32_t group_kind,
                                    uint32_t group_param, uint32_t thr_num, uint32_t thr_den, uint32_t CS) {
    if (!rows || n_rows == 0 || row_bytes == 0 || group_param == 0 || group_kind > 1 || CS == 0 || row_bytes % CS) return nullptr;
    if (thr_den == 0 || thr_num > thr_den || 2ull * thr_num <= thr_den) return nullptr;   // tau in (0.5, 1], R3
    ibp_oracle_ds_T* d = new ibp_oracle_ds_T();
    d->n_rows = n_rows; d->row_bytes = row_bytes; d->group_kind = group_kind; d->group_param = group_param; d->CS = CS;
    d->n_groups = group_kind == 0 ? (n_rows + group_param - 1) / group_param : (n_rows < group_param ? n_rows : group_param);
    d->mask.assign(d->n_groups * row_bytes, 0);
    d->bitval.assign(d->n_groups * row_bytes, 0);
    d->T.assign(d->n_groups, 0);
    for (uint64_t g = 0; g < d->n_groups; ++g) {
        uint64_t first, count, stride;
        if (group_kind == 0) { first = g * group_param; count = n_rows - first < group_param ? n_rows - first : group_param; stride = row_bytes; }
        else { first = g; count = (n_rows - g + group_param - 1) / group_param; stride = (uint64_t)group_param * row_bytes; }
        const uint64_t T = (count * thr_num + thr_den - 1) / thr_den;                     // ceil(tau * N_g)
        d->T[g] = T;
        ibp_oracle_group_masks_T(rows + first * row_bytes, count, stride, row_bytes, T, &d->mask[g * row_bytes], &d->bitval[g * row_bytes], nullptr);
    }
    d->row_offset.assign(n_rows + 1, 0);
    d->rowflag.assign((n_rows + 7) / 8, 0);
    std::vector<uint8_t> tmp(row_bytes);
    for (uint64_t id = 0; id < n_rows; ++id) {
        const uint64_t g = group_of_T(d, id);
        int comp = 0;
        const uint32_t size = ibp_oracle_compress_row_T(rows + id * row_bytes, &d->mask[g * row_bytes], &d->bitval[g * row_bytes], row_bytes, CS, tmp.data(), &comp);
        put_bit(d->rowflag.data(), id, comp);
        if (!comp) d->n_raw += 1;
        d->row_offset[id + 1] = d->row_offset[id] + size;
        d->stored.insert(d->stored.end(), tmp.begin(), tmp.begin() + size);
    }
    return d;
}

void ibp_oracle_destroy_T(ibp_oracle_ds_T* d) { delete d; }
uint64_t ibp_oracle_T_n_groups(const ibp_oracle_ds_T* d) { return d->n_groups; }
uint64_t ibp_oracle_T_n_raw(const ibp_oracle_ds_T* d) { return d->n_raw; }
uint64_t ibp_oracle_T_stored_bytes(const ibp_oracle_ds_T* d) { return d->row_offset[d->n_rows]; }
uint64_t ibp_oracle_T_rowflag_bytes(const ibp_oracle_ds_T* d) { return d->rowflag.size(); }
uint64_t ibp_oracle_T_threshold(const ibp_oracle_ds_T* d, uint64_t g) { return d->T[g]; }
const uint8_t* ibp_oracle_T_mask(const ibp_oracle_ds_T* d, uint64_t g) { return &d->mask[g * d->row_bytes]; }
const uint8_t* ibp_oracle_T_bitval(const ibp_oracle_ds_T* d, uint64_t g) { return &d->bitval[g * d->row_bytes]; }
const uint8_t* ibp_oracle_T_row(const ibp_oracle_ds_T* d, uint64_t id, uint64_t* nbytes, int* is_compressed) {
    *nbytes = d->row_offset[id + 1] - d->row_offset[id];
    *is_compressed = get_bit(d->rowflag.data(), id);
    return d->stored.data() + d->row_offset[id];
}

// Online append ("During the prefill phase, we sample ... to create the Mask and Bitval.  This metadata is used to
// compress the KV cache generated in the decode phase"): rows that arrive after the build are compressed under the EXISTING
// Mask/Bitval of their group -- nothing is re-counted, the metadata does not change -- and stored after the rows already there.
// A new row belongs to group id div G (blocked) or id mod S (strided) like any other; its group must already have metadata.
// Returns 0, or 1 (nothing appended) when a new row's group does not exist.
int ibp_oracle_T_append(ibp_oracle_ds_T* d, const uint8_t* rows, uint64_t n_new) {
    for (uint64_t j = 0; j < n_new; ++j)
        if (group_of_T(d, d->n_rows + j) >= d->n_groups) return 1;
    std::vector<uint8_t> tmp(d->row_bytes);
    for (uint64_t j = 0; j < n_new; ++j) {
        const uint64_t id = d->n_rows;
        const uint64_t g = group_of_T(d, id);
        int comp = 0;
        const uint32_t size = ibp_oracle_compress_row_T(rows + j * d->row_bytes, &d->mask[g * d->row_bytes], &d->bitval[g * d->row_bytes],
                                                        d->row_bytes, d->CS, tmp.data(), &comp);
        if (d->rowflag.size() * 8 < id + 1) d->rowflag.push_back(0);
        put_bit(d->rowflag.data(), id, comp);
        if (!comp) d->n_raw += 1;
        d->row_offset.push_back(d->row_offset[id] + size);
        d->stored.insert(d->stored.end(), tmp.begin(), tmp.begin() + size);
        d->n_rows += 1;
    }
    return 0;
}
uint64_t ibp_oracle_T_n_rows(const ibp_oracle_ds_T* d) { return d->n_rows; }

// Gather-decompress in thresholded mode (S8c thresholded step 7): check the per-row bit, copy or decode.
int ibp_oracle_gather_decompress_T(const ibp_oracle_ds_T* d, const int64_t* ids, int64_t n, uint32_t index_span, uint8_t* out) {
    int bad = 0;
    std::vector<uint8_t> in(d->row_bytes + 8);
    for (int64_t i = 0; i < n; ++i)
        for (uint32_t j = 0; j < index_span; ++j) {
            const int64_t id = ids[i] * (int64_t)index_span + j;
            if (id < 0 || (uint64_t)id >= d->n_rows) { bad = 1; continue; }
            const uint64_t g = group_of_T(d, (uint64_t)id);
            const uint64_t size = d->row_offset[id + 1] - d->row_offset[id];
            std::memset(in.data(), 0, in.size());
            std::memcpy(in.data(), d->stored.data() + d->row_offset[id], size);
            ibp_oracle_decompress_row_T(in.data(), get_bit(d->rowflag.data(), (uint64_t)id), &d->mask[g * d->row_bytes],
                                        &d->bitval[g * d->row_bytes], d->row_bytes, d->CS, out + ((uint64_t)i * index_span + j) * d->row_bytes);
        }
    return bad;
}

}  // extern "C"

