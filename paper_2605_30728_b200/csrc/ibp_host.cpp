// ibp_host.cpp -- host side of libibp.so: the compressor (S0, S0'), the packed-store layout and the accessors.
//
// Own implementation, independent of oracle/: masks come from a word-wise AND/OR reduction (not bit counters), rows
// are packed word by word with a parallel bit extract (BMI2 pext when the CPU has it), groups in parallel (OpenMP).
// The result must agree with the oracle bit for bit: Mask, Bitval, k_g and (canonical bit order, include/ibp.h) the
// packed bytes of every row.
#include <cuda_runtime.h>
#include <immintrin.h>
#include <omp.h>

#include <algorithm>
#include <cstdarg>
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
extern "C" const char* ibp_version(void) { return "ibp-b200 0.1 (sm_100a, group-strict IBP)"; }

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

// ------------------------------------------------------------------------------------------------ build
extern "C" ibp_status ibp_build(const void* rows_host, const ibp_build_params* params, ibp_handle** out_handle) {
    if (!rows_host || !params || !out_handle) { ibp_set_error("ibp_build: null argument"); return IBP_ERR_INVALID_ARG; }
    if (params->struct_size != sizeof(ibp_build_params)) { ibp_set_error("ibp_build: struct_size %u != %zu", params->struct_size, sizeof(ibp_build_params)); return IBP_ERR_INVALID_ARG; }
    ibp_build_params p = *params;
    if (p.row_bytes == 0 || p.row_bytes % 4 || p.row_bytes > 65536) { ibp_set_error("ibp_build: row_bytes %u must be a multiple of 4 in 4..65536", p.row_bytes); return IBP_ERR_INVALID_ARG; }
    if (p.n_rows == 0 || p.group_param == 0 || p.group_kind > 1) { ibp_set_error("ibp_build: n_rows, group_param must be >= 1 and group_kind 0|1"); return IBP_ERR_INVALID_ARG; }
    if (p.threshold_num == 0 && p.threshold_den == 0) p.threshold_num = p.threshold_den = 1;
    if (p.threshold_den == 0 || p.threshold_num > p.threshold_den) { ibp_set_error("ibp_build: bad threshold"); return IBP_ERR_INVALID_ARG; }
    if (p.threshold_num != p.threshold_den) { ibp_set_error("ibp_build: thresholded mode (T<N) is not on this path"); return IBP_ERR_UNSUPPORTED; }
    if (p.align_bytes == 0) p.align_bytes = 32;
    if (p.align_bytes > 128 || (p.align_bytes & (p.align_bytes - 1))) { ibp_set_error("ibp_build: align_bytes %u must be a power of two <= 128", p.align_bytes); return IBP_ERR_INVALID_ARG; }
    if (p.index_span == 0) p.index_span = 1;
    if (p.n_rows % p.index_span) { ibp_set_error("ibp_build: n_rows must be a multiple of index_span"); return IBP_ERR_INVALID_ARG; }
    if (p.index_span > 1 && p.group_kind != IBP_GROUP_BLOCKED) { ibp_set_error("ibp_build: index_span > 1 needs blocked groups"); return IBP_ERR_INVALID_ARG; }

    ibp_handle* h = new (std::nothrow) ibp_handle();
    if (!h) { ibp_set_error("ibp_build: out of memory"); return IBP_ERR_OUT_OF_MEMORY; }
    h->p = p;
    h->n_words = p.row_bytes / 4;
    h->n_groups = p.group_kind == IBP_GROUP_BLOCKED ? (p.n_rows + p.group_param - 1) / p.group_param
                                                     : std::min<uint64_t>(p.group_param, p.n_rows);
    const uint32_t nw = h->n_words;
    const uint64_t ng = h->n_groups, G = p.group_param;
    const uint32_t* rows = (const uint32_t*)rows_host;
    const int nthreads = p.n_threads ? (int)p.n_threads : omp_get_max_threads();
    try {
        h->meta.assign(ng * 2 * nw, 0);
        h->gtab.assign(ng, IbpGroupEntry{0, 0, 0});
    } catch (...) { delete h; ibp_set_error("ibp_build: out of memory (metadata)"); return IBP_ERR_OUT_OF_MEMORY; }

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

    // ---- packed store in host memory that the GPU can read in place (P:239 zero-copy).  Two kinds:
    //   managed-host: cudaMallocManaged + preferred location CPU; ibp_upload_metadata adds the direct GPU mapping
    //                 (accessed-by).  The pages stay in host memory, SM loads cross PCIe, and the GPU maps them
    //                 with large pages, which is what makes random row gathers translation-friendly.  Default.
    //   pinned:       cudaHostAlloc(mapped | portable), 4 KB GPU pages.  IBP_FLAG_HOSTALLOC_STORE.
    // Without a CUDA device (or with IBP_FLAG_PAGEABLE_STORE): ordinary memory, host accessors + resident decode only.
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
            delete h;
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
        if (posix_memalign(&ptr, 4096, h->store_bytes) != 0) { delete h; ibp_set_error("ibp_build: out of memory (store)"); return IBP_ERR_OUT_OF_MEMORY; }
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

extern "C" ibp_status ibp_packed_row(const ibp_handle* h, int64_t row, const void** host_ptr, uint32_t* stride_bytes, uint32_t* k_bits) {
    if (!h || row < 0 || (uint64_t)row >= h->p.n_rows) { ibp_set_error("ibp_packed_row: bad row"); return IBP_ERR_INVALID_ARG; }
    const uint64_t g = h->p.group_kind == IBP_GROUP_BLOCKED ? (uint64_t)row / h->p.group_param : (uint64_t)row % h->p.group_param;
    if (host_ptr) *host_ptr = h->store + ibp_row_offset(h, (uint64_t)row);
    if (stride_bytes) *stride_bytes = h->gtab[g].stride;
    if (k_bits) *k_bits = h->gtab[g].k_bits;
    return IBP_OK;
}

extern "C" ibp_status ibp_packed_range(const ibp_handle* h, int64_t first_row, int64_t n_rows, const void** host_ptr, uint64_t* nbytes) {
    if (!h || !host_ptr || !nbytes || first_row < 0 || n_rows < 0 || (uint64_t)(first_row + n_rows) > h->p.n_rows) {
        ibp_set_error("ibp_packed_range: bad range");
        return IBP_ERR_INVALID_ARG;
    }
    if ((uint64_t)first_row % h->p.group_param) { ibp_set_error("ibp_packed_range: first_row must start a layout unit (multiple of %u)", h->p.group_param); return IBP_ERR_INVALID_ARG; }
    const uint64_t begin = (uint64_t)first_row < h->p.n_rows ? ibp_row_offset(h, (uint64_t)first_row) : h->store_used;
    uint64_t end = begin;
    if (n_rows > 0) {
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
            const uint64_t g = h->p.group_kind == IBP_GROUP_BLOCKED ? r / h->p.group_param : r % h->p.group_param;
            s += h->gtab[g].stride;
            b += (h->gtab[g].k_bits + 7) / 8;
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
    if (!h || warps_per_cta > 32) { ibp_set_error("ibp_configure: bad argument"); return IBP_ERR_INVALID_ARG; }
    h->max_ctas = max_ctas;
    h->warps_per_cta = warps_per_cta;
    return IBP_OK;
}

extern "C" void ibp_destroy(ibp_handle* h) {
    if (!h) return;
    if (h->meta_dev) cudaFree(h->meta_dev);
    if (h->gtab_dev) cudaFree(h->gtab_dev);
    if (h->mvtab_dev) cudaFree(h->mvtab_dev);
    if (h->store) {
        if (h->store_kind == IBP_STORE_PINNED) cudaFreeHost(h->store);
        else if (h->store_kind == IBP_STORE_MANAGED_HOST) cudaFree(h->store);
        else free(h->store);
    }
    (void)cudaGetLastError();
    delete h;
}
