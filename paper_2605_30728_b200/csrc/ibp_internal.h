// ibp_internal.h -- private state of libibp.so (not part of the C ABI; shares nothing with oracle/).
#pragma once
#include <cstdint>
#include <string>
#include <vector>

#include "ibp.h"

// Host array that either owns its elements or borrows them from a mapping (a shared store segment, ibp_shared.cpp): the host
// mirrors of the metadata need not be copied into every process that opens the same store.
template <typename T>
struct HostArray {
    std::vector<T> own;
    T* ptr = nullptr;
    size_t n = 0;
    void assign(size_t count, const T& v) { own.assign(count, v); ptr = own.data(); n = count; }
    void resize(size_t count, const T& v = T()) {
        if (ptr != own.data() && n) own.assign(ptr, ptr + n);     // was borrowed: take a private copy first
        own.resize(count, v); ptr = own.data(); n = count;
    }
    void borrow(T* p, size_t count) { std::vector<T>().swap(own); ptr = p; n = count; }
    T* data() { return ptr; }
    const T* data() const { return ptr; }
    size_t size() const { return n; }
    T& operator[](size_t i) { return ptr[i]; }
    const T& operator[](size_t i) const { return ptr[i]; }
};

// One entry per group, 16 bytes, mirrored in HBM.
//   blocked: packed row j of the group lies at store + base + j*stride
//   strided: tile t of matrix row r lies at store + r*row_stride_strided + base   (base = prefix_t)
struct IbpGroupEntry {
    uint64_t base;
    uint32_t stride;   // roundup(ceil(k/8), A); 0 when k == 0
    uint32_t k_bits;   // variant bits per row of this group
};

struct ibp_handle {
    ibp_build_params p{};
    uint64_t n_groups = 0;
    uint32_t n_words = 0;                  // row_bytes / 4
    uint64_t row_stride_strided = 0;       // bytes of one packed matrix row (strided groups)
    uint32_t max_stride = 0;

    // host copies
    HostArray<uint32_t> meta;              // per group: Mask words then Bitval words (2*n_words)
    HostArray<IbpGroupEntry> gtab;
    uint8_t* store = nullptr;              // packed store (pinned+mapped, or malloc)
    uint8_t* store_dev = nullptr;          // device-visible address of the store (nullptr if pageable)
    uint64_t store_bytes = 0;              // incl. slack
    uint64_t store_used = 0;
    int store_kind = IBP_STORE_PAGEABLE;   // ibp_store_kind
    // IBP_STORE_SHARED: the store and the host mirrors live in a POSIX shared-memory segment opened by ibp_open_shared
    void* shm_base = nullptr;
    uint64_t shm_bytes = 0;
    bool shm_registered = false;           // cudaHostRegister'ed by this process (ibp_attach_device)
    uint64_t packed_bytes_rows = 0, packed_bytes_bytealigned = 0;

    // thresholded mode (tau < 1): data-dependent row sizes
    bool thresholded = false;
    HostArray<uint32_t> row_off;           // n_rows + 1 offsets into the store, in 16-byte units
    HostArray<uint32_t> row_flag;          // bit r (word r/32, bit r%32) = 1 iff row r is compressed
    uint64_t n_rows_raw = 0;
    uint32_t* row_off_dev = nullptr;
    uint32_t* row_flag_dev = nullptr;
    // slot layout (IBP_FLAG_SLOT_LAYOUT): row r at r * slot_bytes, its stored size in row_size[r] (16-byte units); no row_off
    bool slot_layout = false;
    uint32_t slot_bytes = 0;
    uint64_t capacity_rows = 0;
    HostArray<uint8_t> row_size;           // capacity_rows entries
    uint8_t* row_size_dev = nullptr;

    // device copies
    int device = -1;
    uint32_t* meta_dev = nullptr;
    IbpGroupEntry* gtab_dev = nullptr;
    uint32_t* mvtab_dev = nullptr;         // optional expand move masks, 5 per (group, word)
    int max_runs = -1;                     // most runs of variant bits in any Mask word of the table (set by ibp_attach_device)

    // ibp_build_device only
    bool built_on_device = false;
    ibp_build_stats build_stats{};

    // launch configuration
    uint32_t max_ctas = 0, warps_per_cta = 0;
    int sm_count = 0;
    int order_mode = -1;                   // -1 auto, 0 off, 1 on (locality-ordered gather)
    int rows_in_flight = 0;                // random gathers: rows each warp keeps in flight (1, 2 or 4); 0 = automatic
    int dedup_mode = -1;                   // random gathers: 1 = fetch each distinct id once, replicate in HBM; -1 auto
    int stream_mode = 1;                   // contiguous runs: 1 = TMA pipeline stream kernel, 0 = per-row fetch
    int fetch_mode = 1;                    // 0 = cp.async (LSU), 1 = cp.async.bulk (TMA)
    int t2_mode = 1;                       // thresholded contiguous runs: 1 = sub-warp kernel (ibp_stream_t2_kernel), 0 = row-per-warp kernel
};

// Compressed GPU cache: slabs of packed rows + a hash map id -> 64-bit value {offset:40, slab:3, compressed:1}.
struct ibp_cache {
    ibp_handle* h = nullptr;
    uint32_t n_slabs = 0, cur_slab = 0;
    uint64_t slab_bytes = 0;
    uint8_t* slab_dev[8] = {};
    uint64_t slab_used[8] = {};
    int slab_device[8] = {-1, -1, -1, -1, -1, -1, -1, -1};   // CUDA device whose memory holds the slab; -1: none yet (a peer process's slab, not attached)
    bool slab_owned[8] = {};               // allocated by this cache (it fills it and frees it); false: a peer process's slab or nothing
    bool slab_imported[8] = {};            // opened from a CUDA IPC handle (ibp_cache_slab_attach)
    uint64_t* map_dev = nullptr;           // map_cap slots of {key = id + 1 (0 = empty), value}
    uint32_t map_cap = 0;                  // power of two
    uint64_t n_entries = 0, max_entries = 0;
    std::vector<uint64_t> present;         // host bitmap of the cached row ids
};

// error plumbing (thread local)
void ibp_set_error(const char* fmt, ...);

// shared by the host compressor (ibp_host.cpp) and the GPU compressor (ibp_build_device.cu)
ibp_status ibp_prepare_handle(const ibp_build_params* params, const char* who, ibp_handle** out);   // validate + allocate
void ibp_layout_strict(ibp_handle* h);                          // gtab[].k_bits -> strides, bases, totals
ibp_status ibp_alloc_store(ibp_handle* h, int nthreads);         // host store of h->store_bytes bytes, zero-filled
// ibp_device.cu: everything ibp_upload_metadata does; arrays that already exist on the device are kept as they are
ibp_status ibp_attach_device(ibp_handle* h, int device, void* cuda_stream);

// byte offset of packed row `id` inside the store
static inline uint64_t ibp_row_offset(const ibp_handle* h, uint64_t id) {
    if (h->slot_layout) return id * (uint64_t)h->slot_bytes;
    if (h->thresholded) return 16ull * h->row_off[id];
    if (h->p.group_kind == IBP_GROUP_BLOCKED) {
        const uint64_t g = id / h->p.group_param;
        return h->gtab[g].base + (id - g * h->p.group_param) * (uint64_t)h->gtab[g].stride;
    }
    return (id / h->p.group_param) * h->row_stride_strided + h->gtab[id % h->p.group_param].base;
}

// thresholded mode: bytes row `id` occupies in the store incl. alignment padding (what a gather moves over the link)
static inline uint64_t ibp_row_stored_T(const ibp_handle* h, uint64_t id) {
    return h->slot_layout ? 16ull * h->row_size[id] : 16ull * (h->row_off[id + 1] - h->row_off[id]);
}

// group of a row id
static inline uint64_t ibp_group_of(const ibp_handle* h, uint64_t id) {
    return h->p.group_kind == IBP_GROUP_BLOCKED ? id / h->p.group_param : id % h->p.group_param;
}
