// ibp_host.cpp -- host side of libibp.so: the compressor (S0, S0'), the packed-store layout and the accessors.
//
// Own implementation, independent of oracle/: masks come from a word-wise AND/OR reduction (not bit counters), rows
// are packed word by word with a parallel bit extract (BMI2 pext when the CPU has it), groups in parallel (OpenMP).
// The result must agree with the oracle bit for bit: Mask, Bitval, k_g and (canonical bit order, include/ibp.h) the
// packed bytes of every row.
#include <cuda_runtime.h>
#include <immintrin.h>
#include <omp.h>
#include <sys/mman.h>

#include <algorithm>
#include <cstdarg>
#include <cstddef>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>

#include "ibp_internal.h"

// ------------------------------------------------------------------------------------------------ errors
static thread_local char g_err[512] = "";
void ibp_set_error(const char* fmt, ...) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof g_err, fmt, ap);
    va_end(ap);
}
extern "C" const char* ibp_last_error(void) { return g_err; }
extern "C" const char* ibp_version(void) { return "ibp-b200 0.4 (sm_100a; group-strict and thresholded IBP, GPU build and append, compressed multi-GPU cache, shared store, mask tools)"; }

// ------------------------------------------------------------------------------------------------ bit helpers
static inline uint64_t pext64_soft(uint64_t v, uint64_t m) {
    uint64_t r = 0;
    for (unsigned k = 0; m; m &= m - 1, ++k) r |= ((v >> __builtin_ctzll(m)) & 1ull) << k;
    return r;
}
static bool g_has_bmi2 = __builtin_cpu_supports("bmi2");
static inline uint64_t pext64(uint64_t v, uint64_t m) { return g_has_bmi2 ? _pext_u64(v, m) : pext64_soft(v, m); }

// Append the variant bits of one row (words where ~mask selects) to dst as an LSB-first stream.
// dst has at least ceil(k/8) bytes plus 8 bytes of writable slack inside the store.
static void pack_row_words(const uint32_t* row, const uint32_t* mask, uint32_t n_words, uint8_t* dst, uint32_t nbytes) {
    uint64_t acc = 0;      // pending bits, LSB-first
    unsigned fill = 0;     // number of pending bits (< 64)
    uint32_t out = 0;      // bytes written
    uint32_t i = 0;
    for (; i + 1 < n_words; i += 2) {
        uint64_t v, m;
        memcpy(&v, row + i, 8);
        memcpy(&m, mask + i, 8);
        const uint64_t nv = ~m;
        const unsigned k = (unsigned)__builtin_popcountll(nv);
        if (!k) continue;
        const uint64_t x = pext64(v, nv);
        acc |= x << fill;
        if (fill + k >= 64) {
            memcpy(dst + out, &acc, 8);
            out += 8;
            acc = fill ? (x >> (64 - fill)) : 0;   // the bits of x that did not fit
            fill = fill + k - 64;
        } else {
            fill += k;
        }
    }
    if (i < n_words) {
        const uint32_t nv = ~mask[i];
        const unsigned k = (unsigned)__builtin_popcount(nv);
        if (k) {
            const uint64_t x = pext64(row[i], nv);
            acc |= x << fill;
            if (fill + k >= 64) {
                memcpy(dst + out, &acc, 8);
                out += 8;
                acc = fill ? (x >> (64 - fill)) : 0;
                fill = fill + k - 64;
            } else {
                fill += k;
            }
        }
    }
    // flush the remaining bits byte by byte (never write past nbytes: neighbours may be packed concurrently)
    for (; out < nbytes; ++out, acc >>= 8) dst[out] = (uint8_t)acc;
}

static inline uint64_t round_up(uint64_t v, uint64_t a) { return (v + a - 1) / a * a; }

// ------------------------------------------------------------------------------------------------ packed store
// Allocates h->store (h->store_bytes bytes, already set) and zero-fills it.
ibp_status ibp_alloc_store(ibp_handle* h, int nthreads) {
    if (nthreads <= 0) nthreads = omp_get_max_threads();
    // ---- packed store in host memory that the GPU can read in place (P:239 zero-copy).  Two kinds:
    //   managed-host: cudaMallocManaged + preferred location CPU; ibp_upload_metadata adds the direct GPU mapping
    //                 (accessed-by).  The pages stay in host memory, SM loads cross PCIe, and the GPU maps them
    //                 with large pages, which is what makes random row gathers translation-friendly.  Default.
    //   pinned:       cudaHostAlloc(mapped | portable), 4 KB GPU pages.  IBP_FLAG_HOSTALLOC_STORE.
    // Without a CUDA device (or with IBP_FLAG_PAGEABLE_STORE): ordinary memory, host accessors + resident decode only.
    const ibp_build_params& p = h->p;
    bool want_gpu_visible = !(p.flags & IBP_FLAG_PAGEABLE_STORE);
    if (want_gpu_visible) {
        int ndev = 0;
        if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) { want_gpu_visible = false; (void)cudaGetLastError(); }
    }
    if (want_gpu_visible && !(p.flags & IBP_FLAG_HOSTALLOC_STORE)) {
        int dev = 0, managed = 0, concurrent = 0;
        (void)cudaGetDevice(&dev);
        (void)cudaDeviceGetAttribute(&managed, cudaDevAttrManagedMemory, dev);
        (void)cudaDeviceGetAttribute(&concurrent, cudaDevAttrConcurrentManagedAccess, dev);
        void* ptr = nullptr;
        if (managed && concurrent && cudaMallocManaged(&ptr, h->store_bytes, cudaMemAttachGlobal) == cudaSuccess) {
            if (cudaMemAdvise(ptr, h->store_bytes, cudaMemAdviseSetPreferredLocation, cudaCpuDeviceId) == cudaSuccess) {
                h->store = (uint8_t*)ptr;
                h->store_kind = IBP_STORE_MANAGED_HOST;
            } else {
                cudaFree(ptr);
            }
        }
        (void)cudaGetLastError();
    }
    if (want_gpu_visible && !h->store) {
        void* ptr = nullptr;
        cudaError_t e = cudaHostAlloc(&ptr, h->store_bytes, cudaHostAllocMapped | cudaHostAllocPortable);
        if (e != cudaSuccess) {
            (void)cudaGetLastError();
            ibp_set_error("ibp_build: cudaHostAlloc(%llu) failed: %s", (unsigned long long)h->store_bytes, cudaGetErrorString(e));
            return IBP_ERR_OUT_OF_MEMORY;
        }
        h->store = (uint8_t*)ptr;
        h->store_kind = IBP_STORE_PINNED;
        void* dptr = nullptr;
        if (cudaHostGetDevicePointer(&dptr, ptr, 0) == cudaSuccess) h->store_dev = (uint8_t*)dptr;
        else (void)cudaGetLastError();
    }
    if (!h->store) {
        void* ptr = nullptr;
        if (posix_memalign(&ptr, 4096, h->store_bytes) != 0) { ibp_set_error("ibp_build: out of memory (store)"); return IBP_ERR_OUT_OF_MEMORY; }
        h->store = (uint8_t*)ptr;
        h->store_kind = IBP_STORE_PAGEABLE;
    }

    // ---- S0': pack.  Zero first (padding bytes must be 0), then every row writes exactly ceil(k/8) bytes.
    {
        const uint64_t chunk = 1ull << 22, nchunks = (h->store_bytes + chunk - 1) / chunk;
#pragma omp parallel for schedule(static) num_threads(nthreads)
        for (int64_t c = 0; c < (int64_t)nchunks; ++c)
            memset(h->store + (uint64_t)c * chunk, 0, std::min<uint64_t>(chunk, h->store_bytes - (uint64_t)c * chunk));
    }
    return IBP_OK;
}

static ibp_status build_thresholded(ibp_handle* h, const uint32_t* rows, int nthreads);

// ------------------------------------------------------------------------------------------------ build
// Validates the build parameters (shared by ibp_build and ibp_build_device), fills in the defaults and allocates the handle with
// its host-side metadata arrays.
ibp_status ibp_prepare_handle(const ibp_build_params* params, const char* who, ibp_handle** out) {
    const size_t size_v03 = offsetof(ibp_build_params, capacity_rows);        // the struct before capacity_rows was added
    if (params->struct_size != sizeof(ibp_build_params) && params->struct_size != size_v03) {
        ibp_set_error("%s: struct_size %u is neither %zu nor %zu", who, params->struct_size, sizeof(ibp_build_params), size_v03);
        return IBP_ERR_INVALID_ARG;
    }
    ibp_build_params p;
    memset(&p, 0, sizeof p);
    memcpy(&p, params, params->struct_size);
    p.struct_size = sizeof(ibp_build_params);
    if (p.row_bytes == 0 || p.row_bytes % 4 || p.row_bytes > 65536) { ibp_set_error("%s: row_bytes %u must be a multiple of 4 in 4..65536", who, p.row_bytes); return IBP_ERR_INVALID_ARG; }
    if (p.n_rows == 0 || p.group_param == 0 || p.group_kind > 1) { ibp_set_error("%s: n_rows, group_param must be >= 1 and group_kind 0|1", who); return IBP_ERR_INVALID_ARG; }
    if (p.threshold_num == 0 && p.threshold_den == 0) p.threshold_num = p.threshold_den = 1;
    if (p.threshold_den == 0 || p.threshold_num > p.threshold_den) { ibp_set_error("%s: bad threshold", who); return IBP_ERR_INVALID_ARG; }
    const bool thresholded = p.threshold_num != p.threshold_den;
    if (thresholded && 2ull * p.threshold_num <= p.threshold_den) { ibp_set_error("%s: threshold must exceed 1/2 (a bit cannot be invariant-1 and invariant-0 at once)", who); return IBP_ERR_INVALID_ARG; }
    if (p.align_bytes == 0) p.align_bytes = 32;
    if (p.align_bytes > 128 || (p.align_bytes & (p.align_bytes - 1))) { ibp_set_error("%s: align_bytes %u must be a power of two <= 128", who, p.align_bytes); return IBP_ERR_INVALID_ARG; }
    if (thresholded && p.align_bytes < 16) { ibp_set_error("%s: thresholded mode needs align_bytes >= 16 (row offsets are kept in 16-byte units)", who); return IBP_ERR_INVALID_ARG; }
    if (p.index_span == 0) p.index_span = 1;
    if (p.n_rows % p.index_span) { ibp_set_error("%s: n_rows must be a multiple of index_span", who); return IBP_ERR_INVALID_ARG; }
    if (p.index_span > 1 && p.group_kind != IBP_GROUP_BLOCKED) { ibp_set_error("%s: index_span > 1 needs blocked groups", who); return IBP_ERR_INVALID_ARG; }
    if (p.flags & IBP_FLAG_SLOT_LAYOUT) {
        if (!thresholded) { ibp_set_error("%s: IBP_FLAG_SLOT_LAYOUT is a thresholded-mode layout (strict rows of a group all have one size: a dense store is already indexable)", who); return IBP_ERR_INVALID_ARG; }
        if (p.capacity_rows == 0) p.capacity_rows = p.n_rows;
        if (p.capacity_rows < p.n_rows) { ibp_set_error("%s: capacity_rows < n_rows", who); return IBP_ERR_INVALID_ARG; }
    } else {
        p.capacity_rows = 0;
    }

    ibp_handle* h = new (std::nothrow) ibp_handle();
    if (!h) { ibp_set_error("%s: out of memory", who); return IBP_ERR_OUT_OF_MEMORY; }
    h->p = p;
    h->n_words = p.row_bytes / 4;
    h->n_groups = p.group_kind == IBP_GROUP_BLOCKED ? (p.n_rows + p.group_param - 1) / p.group_param
                                                     : std::min<uint64_t>(p.group_param, p.n_rows);
    h->thresholded = thresholded;
    if (p.flags & IBP_FLAG_SLOT_LAYOUT) {
        h->slot_layout = true;
        h->slot_bytes = (uint32_t)((p.row_bytes + p.align_bytes - 1) / p.align_bytes * p.align_bytes);
        h->capacity_rows = p.capacity_rows;
    }
    try {
        h->meta.assign(h->n_groups * 2 * h->n_words, 0);
        h->gtab.assign(h->n_groups, IbpGroupEntry{0, 0, 0});
    } catch (...) { delete h; ibp_set_error("%s: out of memory (metadata)", who); return IBP_ERR_OUT_OF_MEMORY; }
    *out = h;
    return IBP_OK;
}

// Strict mode: from gtab[].k_bits to the store layout (strides, bases, totals); include/ibp.h "Store layout".
void ibp_layout_strict(ibp_handle* h) {
    const ibp_build_params& p = h->p;
    const uint64_t ng = h->n_groups, G = p.group_param;
    const uint64_t A = p.align_bytes, base_align = std::max<uint64_t>(A, 16);
    uint64_t cursor = 0;
    h->max_stride = 0;
    h->packed_bytes_rows = h->packed_bytes_bytealigned = 0;
    for (uint64_t g = 0; g < ng; ++g) {
        IbpGroupEntry& e = h->gtab[g];
        const uint64_t nbytes = (e.k_bits + 7) / 8;
        e.stride = (uint32_t)round_up(nbytes, A);
        h->max_stride = std::max(h->max_stride, e.stride);
        uint64_t count;
        if (p.group_kind == IBP_GROUP_BLOCKED) {
            count = std::min<uint64_t>(G, p.n_rows - g * G);
            cursor = round_up(cursor, base_align);
            e.base = cursor;
            cursor += count * e.stride;
        } else {
            count = (p.n_rows - g + G - 1) / G;
            e.base = cursor;                 // prefix inside one packed matrix row
            cursor += e.stride;
        }
        h->packed_bytes_rows += count * e.stride;
        h->packed_bytes_bytealigned += count * nbytes;
    }
    if (p.group_kind == IBP_GROUP_STRIDED) {
        h->row_stride_strided = round_up(cursor, base_align);
        cursor = h->row_stride_strided * ((p.n_rows + G - 1) / G);
    }
    h->store_used = cursor;
    h->store_bytes = round_up(cursor + 64, 4096);   // slack: 16-byte vector reads may run past the last row
}

extern "C" ibp_status ibp_build(const void* rows_host, const ibp_build_params* params, ibp_handle** out_handle) {
    if (!rows_host || !params || !out_handle) { ibp_set_error("ibp_build: null argument"); return IBP_ERR_INVALID_ARG; }
    ibp_handle* h = nullptr;
    {
        const ibp_status st = ibp_prepare_handle(params, "ibp_build", &h);
        if (st != IBP_OK) return st;
    }
    const ibp_build_params& p = h->p;
    const bool thresholded = h->thresholded;
    const uint32_t nw = h->n_words;
    const uint64_t ng = h->n_groups, G = p.group_param;
    const uint32_t* rows = (const uint32_t*)rows_host;
    const int nthreads = p.n_threads ? (int)p.n_threads : omp_get_max_threads();

    if (thresholded) {
        ibp_status st = IBP_OK;
        try { st = build_thresholded(h, rows, nthreads); }
        catch (...) { ibp_set_error("ibp_build: out of memory (thresholded build)"); st = IBP_ERR_OUT_OF_MEMORY; }
        if (st != IBP_OK) { ibp_destroy(h); return st; }
        *out_handle = h;
        return IBP_OK;
    }

    // ---- S0: Mask/Bitval per group.  AND and OR over the rows; a bit is invariant iff AND == OR there (T = N).
    if (p.group_kind == IBP_GROUP_BLOCKED) {
#pragma omp parallel for schedule(dynamic, 16) num_threads(nthreads)
        for (int64_t g = 0; g < (int64_t)ng; ++g) {
            const uint64_t first = (uint64_t)g * G, count = std::min<uint64_t>(G, p.n_rows - first);
            uint32_t* a = &h->meta[(uint64_t)g * 2 * nw];   // becomes Mask
            uint32_t* o = a + nw;                            // becomes Bitval
            memcpy(a, rows + first * nw, 4ull * nw);
            memcpy(o, rows + first * nw, 4ull * nw);
            for (uint64_t r = 1; r < count; ++r) {
                const uint32_t* x = rows + (first + r) * nw;
                for (uint32_t w = 0; w < nw; ++w) { a[w] &= x[w]; o[w] |= x[w]; }
            }
            uint32_t k = 0;
            for (uint32_t w = 0; w < nw; ++w) {
                const uint32_t mask = ~(a[w] ^ o[w]);
                const uint32_t val = a[w] & mask;
                a[w] = mask; o[w] = val;
                k += (uint32_t)__builtin_popcount(~mask);
            }
            h->gtab[g].k_bits = k;
        }
    } else {
        // strided: walk matrix rows once; per-thread AND/OR accumulators for all S tiles, combined afterwards
        const uint64_t S = ng, n_mrows = (p.n_rows + G - 1) / G;
        std::vector<uint32_t> accA((size_t)nthreads * S * nw, 0xFFFFFFFFu), accO((size_t)nthreads * S * nw, 0u);
#pragma omp parallel num_threads(nthreads)
        {
            const int t = omp_get_thread_num();
            uint32_t* A = &accA[(size_t)t * S * nw];
            uint32_t* O = &accO[(size_t)t * S * nw];
#pragma omp for schedule(static)
            for (int64_t r = 0; r < (int64_t)n_mrows; ++r) {
                const uint64_t id0 = (uint64_t)r * G, cnt = std::min<uint64_t>(G, p.n_rows - id0);
                const uint32_t* x = rows + id0 * nw;
                for (uint64_t w = 0; w < cnt * nw; ++w) { A[w] &= x[w]; O[w] |= x[w]; }
            }
        }
        for (uint64_t g = 0; g < S; ++g) {
            uint32_t* a = &h->meta[g * 2 * nw];
            uint32_t* o = a + nw;
            uint32_t k = 0;
            for (uint32_t w = 0; w < nw; ++w) {
                uint32_t A = 0xFFFFFFFFu, O = 0;
                for (int t = 0; t < nthreads; ++t) { A &= accA[((size_t)t * S + g) * nw + w]; O |= accO[((size_t)t * S + g) * nw + w]; }
                const uint32_t mask = ~(A ^ O);
                a[w] = mask; o[w] = A & mask;
                k += (uint32_t)__builtin_popcount(~mask);
            }
            h->gtab[g].k_bits = k;
        }
    }

    // ---- layout
    ibp_layout_strict(h);

    {
        const ibp_status st = ibp_alloc_store(h, nthreads);
        if (st != IBP_OK) { delete h; return st; }
    }
    if (p.group_kind == IBP_GROUP_BLOCKED) {
#pragma omp parallel for schedule(dynamic, 16) num_threads(nthreads)
        for (int64_t g = 0; g < (int64_t)ng; ++g) {
            const IbpGroupEntry& e = h->gtab[g];
            if (!e.k_bits) continue;
            const uint64_t first = (uint64_t)g * G, count = std::min<uint64_t>(G, p.n_rows - first);
            const uint32_t* mask = &h->meta[(uint64_t)g * 2 * nw];
            const uint32_t nbytes = (e.k_bits + 7) / 8;
            for (uint64_t r = 0; r < count; ++r)
                pack_row_words(rows + (first + r) * nw, mask, nw, h->store + e.base + r * e.stride, nbytes);
        }
    } else {
        const uint64_t n_mrows = (p.n_rows + G - 1) / G;
#pragma omp parallel for schedule(static) num_threads(nthreads)
        for (int64_t r = 0; r < (int64_t)n_mrows; ++r) {
            const uint64_t id0 = (uint64_t)r * G, cnt = std::min<uint64_t>(G, p.n_rows - id0);
            for (uint64_t t = 0; t < cnt; ++t) {
                const IbpGroupEntry& e = h->gtab[t];
                if (!e.k_bits) continue;
                pack_row_words(rows + (id0 + t) * nw, &h->meta[t * 2 * nw], nw,
                               h->store + (uint64_t)r * h->row_stride_strided + e.base, (e.k_bits + 7) / 8);
            }
        }
    }
    *out_handle = h;
    return IBP_OK;
}

// ------------------------------------------------------------------------------------------------ thresholded build
// The paper's default codec (Fig. 3 = P:243-299), own implementation (independent of oracle/):
//   S0  per-bit counters via bit-sliced planes (8 planes = counts up to 255 per flush), Mask/Bitval from
//       count >= T / count <= N_g - T with T = ceil(tau N_g)            (reading R2)
//   S0' per row: participation of each 4-byte chunk ((chunk & Mask) == Bitval), size = row_bytes -
//       floor((bitsSaved - chunks)/8) or raw (Fig. 3 lines 13-18), offsets, then the bit stream
//       [participation bits][payloads] written 64 bits at a time with pext
namespace {

struct BitCounter {                        // counts, for every bit position of a row of nw words, the rows that have it set
    uint32_t nw, pending = 0;
    std::vector<uint32_t> planes;          // 8 planes x nw words: plane j holds bit j of the 32 running counters of a word
    std::vector<uint32_t> cnt;             // 32 x nw totals
    explicit BitCounter(uint32_t nw_) : nw(nw_), planes(8ull * nw_, 0u), cnt(32ull * nw_, 0u) {}
    void add(const uint32_t* x) {
        uint32_t* P = planes.data();
        for (uint32_t w = 0; w < nw; ++w) {
            uint32_t c = x[w];
#pragma GCC unroll 8
            for (int j = 0; j < 8; ++j) { const uint32_t t = P[j * nw + w]; P[j * nw + w] = t ^ c; c &= t; }
        }
        if (++pending == 255) flush();
    }
    void flush() {
        for (int j = 0; j < 8; ++j)
            for (uint32_t w = 0; w < nw; ++w) {
                uint32_t v = planes[j * nw + w];
                planes[j * nw + w] = 0;
                for (; v; v &= v - 1) cnt[w * 32 + __builtin_ctz(v)] += 1u << j;
            }
        pending = 0;
    }
    void reset() { std::fill(planes.begin(), planes.end(), 0u); std::fill(cnt.begin(), cnt.end(), 0u); pending = 0; }
    void merge(BitCounter& o) { o.flush(); for (size_t i = 0; i < cnt.size(); ++i) cnt[i] += o.cnt[i]; }
};

// Mask/Bitval words of one group from its counters (P:231 with >= / <=, reading R2).  Returns popcount(~Mask).
uint32_t masks_from_counts(const uint32_t* cnt, uint32_t nw, uint64_t N, uint64_t T, uint32_t* mask, uint32_t* bitval) {
    uint32_t k = 0;
    for (uint32_t w = 0; w < nw; ++w) {
        uint32_t m = 0, b = 0;
        for (int bit = 0; bit < 32; ++bit) {
            const uint64_t c = cnt[w * 32 + bit];
            if (c >= T) { m |= 1u << bit; b |= 1u << bit; }
            else if (c <= N - T) { m |= 1u << bit; }
        }
        mask[w] = m; bitval[w] = b;
        k += (uint32_t)__builtin_popcount(~m);
    }
    return k;
}

struct BitWriter {                         // LSB-first bit stream into dst; never writes past nbytes
    uint8_t* dst; uint32_t nbytes, out = 0; uint64_t acc = 0; unsigned fill = 0;
    BitWriter(uint8_t* d, uint32_t n) : dst(d), nbytes(n) {}
    inline void put(uint64_t x, unsigned k) {          // k <= 32 bits of x (upper bits of x must be 0)
        acc |= x << fill;
        if (fill + k >= 64) {
            memcpy(dst + out, &acc, 8);
            out += 8;
            acc = fill ? (x >> (64 - fill)) : 0;
            fill = fill + k - 64;
        } else {
            fill += k;
        }
    }
    void finish() { for (; out < nbytes; ++out, acc >>= 8) dst[out] = (uint8_t)acc; }
};

// size in bytes of row x under (mask, bitval); *comp = 0 when it is kept raw (Fig. 3 lines 1-19)
inline uint32_t row_size_T(const uint32_t* x, const uint32_t* mask, const uint32_t* bitval, uint32_t nw, int* comp) {
    int64_t saved = 0;
    for (uint32_t w = 0; w < nw; ++w)
        if ((x[w] & mask[w]) == bitval[w]) saved += __builtin_popcount(mask[w]);
    const int64_t bytes_saved = (saved - (int64_t)nw) >= 8 ? (saved - (int64_t)nw) / 8 : 0;
    *comp = bytes_saved > 0;
    return (uint32_t)(4ll * nw - bytes_saved);
}

}  // namespace

static ibp_status build_thresholded(ibp_handle* h, const uint32_t* rows, int nthreads) {
    const ibp_build_params& p = h->p;
    const uint32_t nw = h->n_words;
    const uint64_t ng = h->n_groups, G = p.group_param, n = p.n_rows;
    auto thr = [&](uint64_t N) { return (N * p.threshold_num + p.threshold_den - 1) / p.threshold_den; };

    // ---- S0: counters -> Mask/Bitval
    if (p.group_kind == IBP_GROUP_BLOCKED && ng >= (uint64_t)nthreads * 4) {
#pragma omp parallel num_threads(nthreads)
        {
            BitCounter bc(nw);
#pragma omp for schedule(dynamic, 16)
            for (int64_t g = 0; g < (int64_t)ng; ++g) {
                const uint64_t first = (uint64_t)g * G, count = std::min<uint64_t>(G, n - first);
                bc.reset();
                for (uint64_t r = 0; r < count; ++r) bc.add(rows + (first + r) * nw);
                bc.flush();
                uint32_t* m = &h->meta[(uint64_t)g * 2 * nw];
                h->gtab[g].k_bits = masks_from_counts(bc.cnt.data(), nw, count, thr(count), m, m + nw);
            }
        }
    } else if (p.group_kind == IBP_GROUP_BLOCKED) {
        // few large groups (e.g. one global Mask/Bitval): split the rows of each group over the threads
        for (uint64_t g = 0; g < ng; ++g) {
            const uint64_t first = g * G, count = std::min<uint64_t>(G, n - first);
            BitCounter total(nw);
#pragma omp parallel num_threads(nthreads)
            {
                BitCounter bc(nw);
#pragma omp for schedule(static)
                for (int64_t r = 0; r < (int64_t)count; ++r) bc.add(rows + (first + (uint64_t)r) * nw);
#pragma omp critical
                total.merge(bc);
            }
            uint32_t* m = &h->meta[g * 2 * nw];
            h->gtab[g].k_bits = masks_from_counts(total.cnt.data(), nw, count, thr(count), m, m + nw);
        }
    } else {
        // strided: group t = rows with id mod S == t; every thread keeps one counter set per tile
        const uint64_t S = ng, n_mrows = (n + G - 1) / G;
        std::vector<BitCounter> total(S, BitCounter(nw));
#pragma omp parallel num_threads(nthreads)
        {
            std::vector<BitCounter> bc(S, BitCounter(nw));
#pragma omp for schedule(static)
            for (int64_t r = 0; r < (int64_t)n_mrows; ++r) {
                const uint64_t id0 = (uint64_t)r * G, cnt = std::min<uint64_t>(G, n - id0);
                for (uint64_t t = 0; t < cnt; ++t) bc[t].add(rows + (id0 + t) * nw);
            }
#pragma omp critical
            for (uint64_t t = 0; t < S; ++t) total[t].merge(bc[t]);
        }
        for (uint64_t t = 0; t < S; ++t) {
            const uint64_t count = (n - t + G - 1) / G;
            uint32_t* m = &h->meta[t * 2 * nw];
            h->gtab[t].k_bits = masks_from_counts(total[t].cnt.data(), nw, count, thr(count), m, m + nw);
        }
    }

    // ---- S0' pass 1: sizes, flags, offsets
    const uint64_t A = p.align_bytes;
    std::vector<uint32_t> size(n);
    h->row_flag.assign((n + 31) / 32, 0u);
    uint64_t n_raw = 0, bytes_aligned = 0;
#pragma omp parallel for schedule(static) num_threads(nthreads) reduction(+ : n_raw, bytes_aligned)
    for (int64_t wd = 0; wd < (int64_t)h->row_flag.size(); ++wd) {          // 32 rows per flag word: no write sharing
        uint32_t flags = 0;
        for (uint64_t r = (uint64_t)wd * 32; r < std::min<uint64_t>(n, (uint64_t)wd * 32 + 32); ++r) {
            const uint32_t* m = &h->meta[ibp_group_of(h, r) * 2 * nw];
            int comp = 0;
            size[r] = row_size_T(rows + r * nw, m, m + nw, nw, &comp);
            if (comp) flags |= 1u << (r & 31); else ++n_raw;
            bytes_aligned += size[r];
        }
        h->row_flag[wd] = flags;
    }
    h->n_rows_raw = n_raw;
    h->packed_bytes_bytealigned = bytes_aligned;
    if (h->slot_layout) {
        // P:361 in-place storage: row r keeps the slot [r*slot, (r+1)*slot); one size byte per slot (16-byte units) replaces the offsets
        const uint64_t cap = h->capacity_rows;
        if (h->slot_bytes / 16 > 255) { ibp_set_error("ibp_build: slot layout needs row_bytes <= 4080 (one size byte per row, 16-byte units)"); return IBP_ERR_UNSUPPORTED; }
        h->row_size.assign(cap, 0);
        h->row_flag.resize((cap + 31) / 32, 0u);
        uint64_t stored = 0;
        for (uint64_t r = 0; r < n; ++r) { h->row_size[r] = (uint8_t)(round_up(size[r], A) / 16); stored += 16ull * h->row_size[r]; }
        h->packed_bytes_rows = stored;
        h->store_used = cap * (uint64_t)h->slot_bytes;
        h->store_bytes = round_up(h->store_used + 64, 4096);
    } else {
    h->row_off.assign(n + 1, 0u);
    uint64_t cursor = 0;                                                    // in 16-byte units
    for (uint64_t r = 0; r < n; ++r) {
        h->row_off[r] = (uint32_t)cursor;
        cursor += round_up(size[r], A) / 16;
        if (cursor > 0xFFFFFFFFull) { ibp_set_error("ibp_build: thresholded store exceeds 64 GiB (4-byte row offsets in 16-byte units)"); return IBP_ERR_UNSUPPORTED; }
    }
    h->row_off[n] = (uint32_t)cursor;
    h->packed_bytes_rows = cursor * 16;
    h->store_used = cursor * 16;
    h->store_bytes = round_up(h->store_used + 64, 4096);
    }
    h->max_stride = (uint32_t)round_up(p.row_bytes, A);
    for (uint64_t g = 0; g < ng; ++g) { h->gtab[g].base = 0; h->gtab[g].stride = 0; }    // unused in this mode

    ibp_status st = ibp_alloc_store(h, nthreads);
    if (st != IBP_OK) return st;

    // ---- S0' pass 2: the bit streams
#pragma omp parallel for schedule(dynamic, 1024) num_threads(nthreads)
    for (int64_t r = 0; r < (int64_t)n; ++r) {
        const uint32_t* x = rows + (uint64_t)r * nw;
        uint8_t* dst = h->store + ibp_row_offset(h, (uint64_t)r);
        if (!((h->row_flag[r >> 5] >> (r & 31)) & 1u)) { memcpy(dst, x, 4ull * nw); continue; }
        const uint32_t* m = &h->meta[ibp_group_of(h, (uint64_t)r) * 2 * nw];
        const uint32_t* b = m + nw;
        BitWriter bw(dst, size[r]);
        for (uint32_t w0 = 0; w0 < nw; w0 += 32) {                           // participation bits, chunk order (R8)
            uint32_t part = 0;
            const uint32_t cnt = std::min<uint32_t>(32, nw - w0);
            for (uint32_t j = 0; j < cnt; ++j) part |= (uint32_t)((x[w0 + j] & m[w0 + j]) == b[w0 + j]) << j;
            bw.put(part, cnt);
        }
        for (uint32_t w = 0; w < nw; ++w) {
            if ((x[w] & m[w]) == b[w]) {
                const uint32_t nv = ~m[w];
                const unsigned k = (unsigned)__builtin_popcount(nv);
                if (k) bw.put(pext64(x[w], nv), k);
            } else {
                bw.put(x[w], 32);
            }
        }
        bw.finish();
    }
    return IBP_OK;
}

// ------------------------------------------------------------------------------------------------ accessors
extern "C" ibp_status ibp_get_info(const ibp_handle* h, ibp_info* out) {
    if (!h || !out) { ibp_set_error("ibp_get_info: null argument"); return IBP_ERR_INVALID_ARG; }
    memset(out, 0, sizeof *out);
    out->n_rows = h->p.n_rows;
    out->n_groups = h->n_groups;
    out->packed_bytes_stored = h->store_used;
    out->packed_bytes_rows = h->packed_bytes_rows;
    out->packed_bytes_bytealigned = h->packed_bytes_bytealigned;
    out->metadata_bytes = h->n_groups * 2ull * h->p.row_bytes;
    out->aux_bytes = h->n_groups * sizeof(IbpGroupEntry);
    out->row_bytes = h->p.row_bytes;
    out->align_bytes = h->p.align_bytes;
    out->index_span = h->p.index_span;
    out->group_kind = h->p.group_kind;
    out->group_param = h->p.group_param;
    out->max_row_stride = h->max_stride;
    out->device = h->device;
    out->store_kind = (uint32_t)h->store_kind;
    out->thresholded = h->thresholded ? 1u : 0u;
    out->threshold_num = h->p.threshold_num;
    out->threshold_den = h->p.threshold_den;
    out->n_rows_raw = h->n_rows_raw;
    out->rowflag_bytes = h->row_flag.size() * 4ull;
    out->rowoffset_bytes = h->row_off.size() * 4ull;
    out->capacity_rows = h->slot_layout ? h->capacity_rows : h->p.n_rows;
    out->rowsize_bytes = h->row_size.size();
    out->slot_bytes = h->slot_layout ? h->slot_bytes : 0;
    if (h->thresholded) out->aux_bytes = out->rowflag_bytes + out->rowoffset_bytes;
    return IBP_OK;
}

extern "C" ibp_status ibp_get_metadata_host(const ibp_handle* h, int64_t group, const void** mask, const void** bitval, uint32_t* k_bits) {
    if (!h || group < 0 || (uint64_t)group >= h->n_groups) { ibp_set_error("ibp_get_metadata_host: bad group"); return IBP_ERR_INVALID_ARG; }
    const uint32_t* m = &h->meta[(uint64_t)group * 2 * h->n_words];
    if (mask) *mask = m;
    if (bitval) *bitval = m + h->n_words;
    if (k_bits) *k_bits = h->gtab[group].k_bits;
    return IBP_OK;
}

// byte-aligned size of a thresholded row, recovered from its stored form (participation bits first)
static uint32_t row_size_from_store(const ibp_handle* h, uint64_t row) {
    if (!((h->row_flag[row >> 5] >> (row & 31)) & 1u)) return h->p.row_bytes;
    const uint32_t nw = h->n_words;
    const uint32_t* m = &h->meta[ibp_group_of(h, row) * 2 * nw];
    const uint8_t* src = h->store + ibp_row_offset(h, (uint64_t)row);
    uint64_t bits = nw;
    for (uint32_t w = 0; w < nw; ++w) bits += ((src[w >> 3] >> (w & 7)) & 1u) ? (uint32_t)__builtin_popcount(~m[w]) : 32u;
    return (uint32_t)((bits + 7) / 8);
}

extern "C" ibp_status ibp_row_info(const ibp_handle* h, int64_t row, const void** host_ptr, uint32_t* stored_bytes, uint32_t* size_bytes, int* is_compressed) {
    if (!h || row < 0 || (uint64_t)row >= h->p.n_rows) { ibp_set_error("ibp_row_info: bad row"); return IBP_ERR_INVALID_ARG; }
    if (host_ptr) *host_ptr = h->store + ibp_row_offset(h, (uint64_t)row);
    if (h->thresholded) {
        if (stored_bytes) *stored_bytes = (uint32_t)ibp_row_stored_T(h, (uint64_t)row);
        if (size_bytes) *size_bytes = row_size_from_store(h, (uint64_t)row);
        if (is_compressed) *is_compressed = (int)((h->row_flag[row >> 5] >> (row & 31)) & 1u);
    } else {
        const IbpGroupEntry& e = h->gtab[ibp_group_of(h, (uint64_t)row)];
        if (stored_bytes) *stored_bytes = e.stride;
        if (size_bytes) *size_bytes = (e.k_bits + 7) / 8;
        if (is_compressed) *is_compressed = 1;
    }
    return IBP_OK;
}

extern "C" ibp_status ibp_packed_row(const ibp_handle* h, int64_t row, const void** host_ptr, uint32_t* stride_bytes, uint32_t* k_bits) {
    if (!h || row < 0 || (uint64_t)row >= h->p.n_rows) { ibp_set_error("ibp_packed_row: bad row"); return IBP_ERR_INVALID_ARG; }
    if (h->thresholded) {
        uint32_t size = 0;
        const ibp_status s = ibp_row_info(h, row, host_ptr, stride_bytes, &size, nullptr);
        if (k_bits) *k_bits = 8u * size;
        return s;
    }
    const uint64_t g = ibp_group_of(h, (uint64_t)row);
    if (host_ptr) *host_ptr = h->store + ibp_row_offset(h, (uint64_t)row);
    if (stride_bytes) *stride_bytes = h->gtab[g].stride;
    if (k_bits) *k_bits = h->gtab[g].k_bits;
    return IBP_OK;
}

extern "C" ibp_status ibp_store_device_ptr(const ibp_handle* h, const void** dev_ptr) {
    if (!h || !dev_ptr) { ibp_set_error("ibp_store_device_ptr: null argument"); return IBP_ERR_INVALID_ARG; }
    if (h->device < 0 || !h->store_dev) { ibp_set_error("ibp_store_device_ptr: the store is not attached to a device (upload first; pageable stores never are)"); return IBP_ERR_BAD_STATE; }
    *dev_ptr = h->store_dev;
    return IBP_OK;
}

extern "C" ibp_status ibp_packed_range(const ibp_handle* h, int64_t first_row, int64_t n_rows, const void** host_ptr, uint64_t* nbytes) {
    if (!h || !host_ptr || !nbytes || first_row < 0 || n_rows < 0 || (uint64_t)(first_row + n_rows) > h->p.n_rows) {
        ibp_set_error("ibp_packed_range: bad range");
        return IBP_ERR_INVALID_ARG;
    }
    if (!(h->thresholded && h->p.group_kind == IBP_GROUP_BLOCKED) && (uint64_t)first_row % h->p.group_param) { ibp_set_error("ibp_packed_range: first_row must start a layout unit (multiple of %u)", h->p.group_param); return IBP_ERR_INVALID_ARG; }
    const uint64_t begin = (uint64_t)first_row < h->p.n_rows ? ibp_row_offset(h, (uint64_t)first_row) : h->store_used;
    uint64_t end = begin;
    if (h->thresholded) {
        end = h->slot_layout ? (uint64_t)(first_row + n_rows) * h->slot_bytes : 16ull * h->row_off[first_row + n_rows];
    } else if (n_rows > 0) {
        const uint64_t last = (uint64_t)(first_row + n_rows - 1);
        const uint64_t g = h->p.group_kind == IBP_GROUP_BLOCKED ? last / h->p.group_param : last % h->p.group_param;
        end = ibp_row_offset(h, last) + h->gtab[g].stride;
    }
    *host_ptr = h->store + begin;
    *nbytes = round_up(end - begin, 16);   // the decoder reads whole 16-byte vectors (the store has slack)
    return IBP_OK;
}

extern "C" ibp_status ibp_batch_link_bytes(const ibp_handle* h, const int64_t* ids, int64_t n, uint64_t* n_unique, uint64_t* stored, uint64_t* bytealigned) {
    if (!h || (!ids && n > 0) || n < 0) { ibp_set_error("ibp_batch_link_bytes: bad argument"); return IBP_ERR_INVALID_ARG; }
    std::vector<int64_t> v(ids, ids + n);
    std::sort(v.begin(), v.end());
    v.erase(std::unique(v.begin(), v.end()), v.end());
    uint64_t s = 0, b = 0;
    const uint64_t span = h->p.index_span;
    for (int64_t id : v) {
        if (id < 0 || (uint64_t)id * span >= h->p.n_rows) { ibp_set_error("ibp_batch_link_bytes: id out of range"); return IBP_ERR_INVALID_ARG; }
        for (uint64_t j = 0; j < span; ++j) {
            const uint64_t r = (uint64_t)id * span + j;
            if (h->thresholded) { s += ibp_row_stored_T(h, r); b += row_size_from_store(h, r); continue; }
            const uint64_t g = h->p.group_kind == IBP_GROUP_BLOCKED ? r / h->p.group_param : r % h->p.group_param;
            const uint64_t ba = (h->gtab[g].k_bits + 7) / 8;
            // a single row is fetched up to whole 32-byte sectors, never beyond its stride (padding to A >= 64 stays in host memory);
            // rows of a span are read as one contiguous run, padding included
            s += span == 1 ? std::min<uint64_t>(h->gtab[g].stride, (ba + 31) & ~31ull) : h->gtab[g].stride;
            b += ba;
            if (h->p.group_kind == IBP_GROUP_BLOCKED && span > 1) {       // whole groups inside a span: skip ahead
                const uint64_t left = std::min<uint64_t>(h->p.group_param - (r % h->p.group_param), span - j) - 1;
                s += left * h->gtab[g].stride;
                b += left * ((h->gtab[g].k_bits + 7) / 8);
                j += left;
            }
        }
    }
    if (n_unique) *n_unique = v.size();
    if (stored) *stored = s;
    if (bytealigned) *bytealigned = b;
    return IBP_OK;
}

extern "C" ibp_status ibp_configure(ibp_handle* h, uint32_t max_ctas, uint32_t warps_per_cta) {
    if (!h || warps_per_cta > 8) { ibp_set_error("ibp_configure: warps_per_cta must be 0 (default) or 1..8"); return IBP_ERR_INVALID_ARG; }
    h->max_ctas = max_ctas;
    h->warps_per_cta = warps_per_cta;
    return IBP_OK;
}

extern "C" void ibp_destroy(ibp_handle* h) {
    if (!h) return;
    if (h->meta_dev) cudaFree(h->meta_dev);
    if (h->gtab_dev) cudaFree(h->gtab_dev);
    if (h->mvtab_dev) cudaFree(h->mvtab_dev);
    if (h->row_off_dev) cudaFree(h->row_off_dev);
    if (h->row_size_dev) cudaFree(h->row_size_dev);
    if (h->row_flag_dev) cudaFree(h->row_flag_dev);
    if (h->store_kind == IBP_STORE_SHARED) {
        if (h->shm_registered) cudaHostUnregister(h->store);
        if (h->shm_base) munmap(h->shm_base, h->shm_bytes);
        h->store = nullptr;
    }
    if (h->store) {
        if (h->store_kind == IBP_STORE_PINNED) cudaFreeHost(h->store);
        else if (h->store_kind == IBP_STORE_MANAGED_HOST) cudaFree(h->store);
        else free(h->store);
    }
    (void)cudaGetLastError();
    delete h;
}
