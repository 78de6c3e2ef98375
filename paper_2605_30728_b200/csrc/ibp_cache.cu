// ibp_cache.cu -- compressed GPU software cache (Fig. 6a): data slabs + hash map; management side.
// The lookup-and-decode path is ibp_cache_gather_decompress in ibp_device.cu (the decode kernel with a map probe in S1).
#include <algorithm>
#include <cstring>
#include <new>
#include <vector>

#include "ibp_devutil.cuh"

namespace {

struct FillItem {          // one row to add: copy `bytes` from the host store at `src` to slab memory at `dst`, then map id -> entry
    uint64_t id, entry, src;
    uint32_t bytes, slab;
};

// {key, value} of a map slot published with ONE 16-byte compare-and-swap: a concurrent probe (16-byte load) sees the slot either
// empty or complete, never a key without its value.
__device__ __forceinline__ ulonglong2 cas128(void* addr, ulonglong2 cmp, ulonglong2 val) {
    ulonglong2 old;
    asm volatile("{\n\t.reg .b128 c, n, o;\n\tmov.b128 c, {%2, %3};\n\tmov.b128 n, {%4, %5};\n\t"
                 "atom.global.acq_rel.gpu.cas.b128 o, [%6], c, n;\n\tmov.b128 {%0, %1}, o;\n\t}"
                 : "=l"(old.x), "=l"(old.y) : "l"(cmp.x), "l"(cmp.y), "l"(val.x), "l"(val.y), "l"(addr) : "memory");
    return old;
}

__global__ void ibp_cache_fill_kernel(const FillItem* __restrict__ items, int64_t n, const uint8_t* __restrict__ store,
                                      uint8_t* const* __restrict__ slabs, uint64_t* __restrict__ map, uint32_t mask) {
    const int lane = threadIdx.x & 31, wpc = blockDim.x >> 5;
    for (int64_t i = (int64_t)blockIdx.x * wpc + (threadIdx.x >> 5); i < n; i += (int64_t)gridDim.x * wpc) {
        const FillItem it = items[i];
        const uint4* src = (const uint4*)(store + it.src);
        uint4* dst = (uint4*)(slabs[it.slab] + (it.entry & ((1ull << 40) - 1)));
        for (uint32_t v = lane; v < it.bytes / 16; v += 32) {
            uint4 t;
            asm volatile("ld.global.nc.L1::no_allocate.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(t.x), "=r"(t.y), "=r"(t.z), "=r"(t.w) : "l"(src + v));
            dst[v] = t;
        }
        __threadfence();    // the slab bytes (possibly in a peer GPU's memory) are visible before the entry that points at them
        __syncwarp();
        if (lane == 0) {
            uint32_t slot = ibp_cache_hash(it.id, mask);
            for (;;) {
                const ulonglong2 prev = cas128(&map[2ull * slot], make_ulonglong2(0ull, 0ull), make_ulonglong2(it.id + 1, it.entry));
                if (prev.x == 0ull || prev.x == it.id + 1) break;
                slot = (slot + 1) & mask;
            }
        }
    }
}

__global__ void ibp_cache_lookup_kernel(const uint64_t* __restrict__ map, uint32_t mask, const int64_t* __restrict__ ids, int64_t n,
                                        uint64_t* __restrict__ entries) {
    for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x)
        entries[i] = ibp_cache_find(map, mask, (uint64_t)ids[i]);
}

}  // namespace

// slab_devices: n_slabs entries (nullptr = all on the handle's device): >= 0 a CUDA device of this process, -1 the handle's device,
// IBP_SLAB_REMOTE a peer process's slab that ibp_cache_slab_attach supplies later.
static ibp_status cache_create(ibp_handle* h, uint64_t capacity_bytes, uint32_t n_slabs, const int32_t* slab_devices, uint64_t max_entries,
                               void* cuda_stream, ibp_cache** out_cache, const char* who) {
    if (!h || !out_cache || n_slabs < 1 || n_slabs > 8 || capacity_bytes == 0) { ibp_set_error("%s: bad argument (1..8 slabs, capacity > 0)", who); return IBP_ERR_INVALID_ARG; }
    if (h->device < 0 || !h->meta_dev) { ibp_set_error("%s: call ibp_upload_metadata first", who); return IBP_ERR_BAD_STATE; }
    if (!h->store_dev) { ibp_set_error("%s: the packed store is not GPU-mapped (pageable store)", who); return IBP_ERR_BAD_STATE; }
    if (h->p.index_span != 1) { ibp_set_error("%s: index_span must be 1", who); return IBP_ERR_UNSUPPORTED; }
    const uint64_t slab_bytes = capacity_bytes / n_slabs / 16 * 16;
    if (slab_bytes == 0 || slab_bytes >= (1ull << 40)) { ibp_set_error("%s: a slab must hold 16 bytes .. 1 TB (40-bit offsets, P:353)", who); return IBP_ERR_INVALID_ARG; }
    int n_dev = 0;
    if (cudaGetDeviceCount(&n_dev) != cudaSuccess) { (void)cudaGetLastError(); n_dev = 0; }
    for (uint32_t s = 0; slab_devices && s < n_slabs; ++s)
        if (slab_devices[s] < IBP_SLAB_REMOTE || slab_devices[s] >= n_dev) { ibp_set_error("%s: slab %u: no CUDA device %d in this process", who, s, slab_devices[s]); return IBP_ERR_INVALID_ARG; }
    ibp_cache* c = new (std::nothrow) ibp_cache();
    if (!c) { ibp_set_error("%s: out of memory", who); return IBP_ERR_OUT_OF_MEMORY; }
    c->h = h;
    c->n_slabs = n_slabs;
    c->slab_bytes = slab_bytes;
    c->max_entries = max_entries ? std::min<uint64_t>(max_entries, h->p.n_rows) : h->p.n_rows;
    uint64_t cap = 1024;
    while (cap < 2 * c->max_entries) cap <<= 1;
    if (cap > (1ull << 31)) { delete c; ibp_set_error("%s: too many entries for the map", who); return IBP_ERR_UNSUPPORTED; }
    c->map_cap = (uint32_t)cap;
    try { c->present.assign((h->p.n_rows + 63) / 64, 0ull); } catch (...) { delete c; ibp_set_error("%s: out of memory", who); return IBP_ERR_OUT_OF_MEMORY; }
    cudaStream_t st = (cudaStream_t)cuda_stream;
    cudaError_t e = cudaSetDevice(h->device);
    if (e == cudaSuccess) e = cudaMalloc((void**)&c->map_dev, cap * 16);
    if (e == cudaSuccess) e = cudaMemsetAsync(c->map_dev, 0, cap * 16, st);
    for (uint32_t s = 0; s < n_slabs && e == cudaSuccess; ++s) {
        const int want = slab_devices ? slab_devices[s] : -1;
        if (want == IBP_SLAB_REMOTE) continue;                              // a peer process owns it: ibp_cache_slab_attach
        const int dev = want < 0 ? h->device : want;
        if (dev != h->device) {
            // a slab in a peer GPU's memory ("a contiguous memory region per interconnected GPU"): the handle's device reads and
            // fills it over NVLink / PCIe peer access
            int can = 0;
            e = cudaDeviceCanAccessPeer(&can, h->device, dev);
            if (e == cudaSuccess && !can) {
                ibp_set_error("%s: device %d cannot access the memory of device %d (no peer access)", who, h->device, dev);
                ibp_cache_destroy(c);
                return IBP_ERR_UNSUPPORTED;
            }
            if (e == cudaSuccess) {
                e = cudaDeviceEnablePeerAccess(dev, 0);                      // current device = the handle's
                if (e == cudaErrorPeerAccessAlreadyEnabled) { (void)cudaGetLastError(); e = cudaSuccess; }
            }
            if (e == cudaSuccess) e = cudaSetDevice(dev);
        }
        if (e == cudaSuccess) e = cudaMalloc((void**)&c->slab_dev[s], slab_bytes + 64);   // slack: 16-byte covers
        if (dev != h->device) { const cudaError_t e2 = cudaSetDevice(h->device); if (e == cudaSuccess) e = e2; }
        if (e == cudaSuccess) { c->slab_device[s] = dev; c->slab_owned[s] = true; }
    }
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    if (e != cudaSuccess) {
        ibp_set_error("%s: %s", who, cudaGetErrorString(e));
        (void)cudaGetLastError();
        ibp_cache_destroy(c);
        return e == cudaErrorMemoryAllocation ? IBP_ERR_OUT_OF_MEMORY : IBP_ERR_CUDA;
    }
    *out_cache = c;
    return IBP_OK;
}

extern "C" ibp_status ibp_cache_create(ibp_handle* h, uint64_t capacity_bytes, uint32_t n_slabs, uint64_t max_entries, void* cuda_stream,
                                       ibp_cache** out_cache) {
    return cache_create(h, capacity_bytes, n_slabs, nullptr, max_entries, cuda_stream, out_cache, "ibp_cache_create");
}

extern "C" ibp_status ibp_cache_create_multi(ibp_handle* h, uint64_t capacity_bytes, uint32_t n_slabs, const int32_t* slab_devices,
                                             uint64_t max_entries, void* cuda_stream, ibp_cache** out_cache) {
    if (!slab_devices) { ibp_set_error("ibp_cache_create_multi: slab_devices is null"); return IBP_ERR_INVALID_ARG; }
    return cache_create(h, capacity_bytes, n_slabs, slab_devices, max_entries, cuda_stream, out_cache, "ibp_cache_create_multi");
}

extern "C" ibp_status ibp_cache_slab_export(const ibp_cache* c, uint32_t slab, void* ipc_handle_out) {
    static_assert(sizeof(cudaIpcMemHandle_t) == IBP_IPC_HANDLE_BYTES, "IBP_IPC_HANDLE_BYTES must be the size of a CUDA IPC memory handle");
    if (!c || !ipc_handle_out || slab >= c->n_slabs) { ibp_set_error("ibp_cache_slab_export: bad argument"); return IBP_ERR_INVALID_ARG; }
    if (!c->slab_owned[slab] || !c->slab_dev[slab]) { ibp_set_error("ibp_cache_slab_export: slab %u is not allocated by this cache", slab); return IBP_ERR_BAD_STATE; }
    cudaIpcMemHandle_t hd;
    IBP_CUDA(cudaIpcGetMemHandle(&hd, c->slab_dev[slab]));
    memcpy(ipc_handle_out, &hd, sizeof hd);
    return IBP_OK;
}

extern "C" ibp_status ibp_cache_slab_attach(ibp_cache* c, uint32_t slab, const void* ipc_handle) {
    if (!c || !ipc_handle || slab >= c->n_slabs) { ibp_set_error("ibp_cache_slab_attach: bad argument"); return IBP_ERR_INVALID_ARG; }
    if (c->slab_dev[slab]) { ibp_set_error("ibp_cache_slab_attach: slab %u already has memory (create it as IBP_SLAB_REMOTE)", slab); return IBP_ERR_BAD_STATE; }
    cudaIpcMemHandle_t hd;
    memcpy(&hd, ipc_handle, sizeof hd);
    void* ptr = nullptr;
    IBP_CUDA(cudaSetDevice(c->h->device));
    IBP_CUDA(cudaIpcOpenMemHandle(&ptr, hd, cudaIpcMemLazyEnablePeerAccess));   // a slab on another GPU: peer access is enabled on first use
    cudaPointerAttributes at;
    c->slab_device[slab] = (cudaPointerGetAttributes(&at, ptr) == cudaSuccess) ? at.device : -1;
    (void)cudaGetLastError();
    c->slab_dev[slab] = (uint8_t*)ptr;
    c->slab_imported[slab] = true;
    return IBP_OK;
}

// only_slab < 0: rows go into the slabs this cache owns, in slab order (ibp_cache_insert); only_slab >= 0: into that slab alone.
// fill = false: the map entries are added but no bytes are copied -- the slab belongs to a peer process that inserts the same ids in
// the same order (the placement is a pure function of the id list, so every process computes the same entries).
static ibp_status cache_insert(ibp_cache* c, int only_slab, bool fill, const int64_t* row_ids_host, int64_t n, void* cuda_stream, int64_t* n_inserted_host) {
    if (!c || n < 0 || (!row_ids_host && n > 0)) { ibp_set_error("ibp_cache_insert: bad argument"); return IBP_ERR_INVALID_ARG; }
    if (n_inserted_host) *n_inserted_host = 0;
    const ibp_handle* h = c->h;
    if (only_slab >= 0 && !c->slab_dev[only_slab]) { ibp_set_error("ibp_cache_insert_slab: slab %d has no memory yet (ibp_cache_slab_attach)", only_slab); return IBP_ERR_BAD_STATE; }
    if (only_slab >= 0 && fill && !c->slab_owned[only_slab]) { ibp_set_error("ibp_cache_insert_slab: slab %d belongs to a peer process, which fills it (pass fill = 0)", only_slab); return IBP_ERR_BAD_STATE; }
    // every id is validated before any state changes: an error return leaves the cache exactly as it was
    for (int64_t i = 0; i < n; ++i) {
        const int64_t sid = row_ids_host[i];
        if (sid < 0 || (uint64_t)sid >= h->p.n_rows) { ibp_set_error("ibp_cache_insert: id %lld out of range", (long long)sid); return IBP_ERR_INVALID_ARG; }
    }
    std::vector<FillItem> items;
    // bookkeeping is staged in copies and committed only after the fill kernel has succeeded; `present` is marked while the list
    // is built (it also de-duplicates ids repeated inside this call) and unmarked again on any failure
    uint64_t slab_used[8];
    memcpy(slab_used, c->slab_used, sizeof slab_used);
    uint32_t cur_slab = only_slab >= 0 ? (uint32_t)only_slab : c->cur_slab;
    const uint32_t end_slab = only_slab >= 0 ? (uint32_t)only_slab + 1 : c->n_slabs;
    auto usable = [&](uint32_t sl) { return only_slab >= 0 || c->slab_owned[sl]; };
    auto rollback = [&]() { for (const FillItem& it : items) c->present[it.id >> 6] &= ~(1ull << (it.id & 63)); };
    try {
        items.reserve((size_t)std::min<int64_t>(n, 1 << 20));
        for (int64_t i = 0; i < n; ++i) {
            const uint64_t id = (uint64_t)row_ids_host[i];
            if ((c->present[id >> 6] >> (id & 63)) & 1ull) continue;
            if (c->n_entries + items.size() >= c->max_entries) break;
            // the 16-byte-aligned cover of the packed row, exactly what the decode kernel fetches from the store
            const uint64_t off = ibp_row_offset(h, id);
            uint64_t bytes, flag = 1;
            if (h->thresholded) {
                bytes = ibp_row_stored_T(h, id);
                flag = (h->row_flag[id >> 5] >> (id & 31)) & 1u;
            } else {
                bytes = h->gtab[ibp_group_of(h, id)].stride;
            }
            const uint64_t head = off & 15ull, cover = bytes ? (head + bytes + 15ull) & ~15ull : 0ull;
            while (cur_slab < end_slab && (!usable(cur_slab) || slab_used[cur_slab] + cover > c->slab_bytes)) ++cur_slab;
            if (cur_slab >= end_slab) { cur_slab = end_slab - 1; break; }          // full: stop at the first row that does not fit
            FillItem it;
            it.id = id;
            it.slab = cur_slab;
            it.entry = slab_used[it.slab] | ((uint64_t)it.slab << 40) | (flag << 43);
            it.src = off - head;
            it.bytes = fill ? (uint32_t)cover : 0u;                                // 0: entry only (the slab's owner copies the bytes)
            items.push_back(it);
            slab_used[it.slab] += cover;
            c->present[id >> 6] |= 1ull << (id & 63);
        }
    } catch (...) {
        rollback();
        ibp_set_error("ibp_cache_insert: out of memory");
        return IBP_ERR_OUT_OF_MEMORY;
    }
    if (items.empty()) return IBP_OK;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    FillItem* items_dev = nullptr;
    uint8_t** slabs_dev = nullptr;
    cudaError_t e = cudaSetDevice(h->device);
    if (e == cudaSuccess) e = cudaMalloc((void**)&items_dev, items.size() * sizeof(FillItem));
    if (e == cudaSuccess) e = cudaMalloc((void**)&slabs_dev, 8 * sizeof(uint8_t*));
    if (e == cudaSuccess) e = cudaMemcpyAsync(items_dev, items.data(), items.size() * sizeof(FillItem), cudaMemcpyHostToDevice, st);
    if (e == cudaSuccess) e = cudaMemcpyAsync(slabs_dev, c->slab_dev, 8 * sizeof(uint8_t*), cudaMemcpyHostToDevice, st);
    if (e == cudaSuccess) {
        const int blocks = (int)std::min<size_t>((items.size() + 7) / 8, (size_t)h->sm_count * 8);
        ibp_cache_fill_kernel<<<blocks, 256, 0, st>>>(items_dev, (int64_t)items.size(), h->store_dev, slabs_dev, c->map_dev, c->map_cap - 1);
        e = cudaGetLastError();
    }
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    if (items_dev) cudaFree(items_dev);
    if (slabs_dev) cudaFree(slabs_dev);
    if (e != cudaSuccess) {
        // a failure before the launch (allocation, copies) has touched neither the slabs nor the map; a failure of the kernel itself
        // is a sticky context error after which no call on this device works anyway.  Either way nothing is committed.
        rollback();
        ibp_set_error("ibp_cache_insert: %s (the cache keeps its previous contents)", cudaGetErrorString(e));
        (void)cudaGetLastError();
        return e == cudaErrorMemoryAllocation ? IBP_ERR_OUT_OF_MEMORY : IBP_ERR_CUDA;
    }
    memcpy(c->slab_used, slab_used, sizeof slab_used);
    if (only_slab < 0) c->cur_slab = cur_slab;
    c->n_entries += items.size();
    if (n_inserted_host) *n_inserted_host = (int64_t)items.size();
    return IBP_OK;
}

extern "C" ibp_status ibp_cache_insert(ibp_cache* c, const int64_t* row_ids_host, int64_t n, void* cuda_stream, int64_t* n_inserted_host) {
    return cache_insert(c, -1, true, row_ids_host, n, cuda_stream, n_inserted_host);
}

extern "C" ibp_status ibp_cache_insert_slab(ibp_cache* c, uint32_t slab, const int64_t* row_ids_host, int64_t n, int fill, void* cuda_stream,
                                            int64_t* n_inserted_host) {
    if (!c || slab >= c->n_slabs) { ibp_set_error("ibp_cache_insert_slab: bad argument"); return IBP_ERR_INVALID_ARG; }
    return cache_insert(c, (int)slab, fill != 0, row_ids_host, n, cuda_stream, n_inserted_host);
}

extern "C" ibp_status ibp_cache_lookup(ibp_cache* c, const int64_t* row_ids_dev, int64_t n, uint64_t* entries_dev, void* cuda_stream) {
    if (!c || n < 0 || (n > 0 && (!row_ids_dev || !entries_dev))) { ibp_set_error("ibp_cache_lookup: bad argument"); return IBP_ERR_INVALID_ARG; }
    if (n == 0) return IBP_OK;
    ibp_cache_lookup_kernel<<<(int)std::min<int64_t>((n + 255) / 256, (int64_t)c->h->sm_count * 8), 256, 0, (cudaStream_t)cuda_stream>>>(c->map_dev, c->map_cap - 1, row_ids_dev, n, entries_dev);
    IBP_CUDA(cudaGetLastError());
    return IBP_OK;
}

extern "C" ibp_status ibp_cache_read(const ibp_cache* c, uint64_t entry, uint32_t nbytes, void* out_host) {
    if (!c || !out_host || entry == IBP_CACHE_MISS) { ibp_set_error("ibp_cache_read: bad argument"); return IBP_ERR_INVALID_ARG; }
    const uint64_t off = entry & ((1ull << 40) - 1), slab = (entry >> 40) & 7ull;
    if (slab >= c->n_slabs || !c->slab_dev[slab] || off + nbytes > c->slab_bytes + 64 || (entry >> 44)) { ibp_set_error("ibp_cache_read: not a valid map value"); return IBP_ERR_INVALID_ARG; }
    IBP_CUDA(cudaMemcpy(out_host, c->slab_dev[slab] + off, nbytes, cudaMemcpyDeviceToHost));
    return IBP_OK;
}

extern "C" ibp_status ibp_cache_get_info(const ibp_cache* c, ibp_cache_info* out) {
    if (!c || !out) { ibp_set_error("ibp_cache_get_info: null argument"); return IBP_ERR_INVALID_ARG; }
    memset(out, 0, sizeof *out);
    out->capacity_bytes = c->slab_bytes * c->n_slabs;
    for (uint32_t s = 0; s < c->n_slabs; ++s) out->used_bytes += c->slab_used[s];
    out->n_entries = c->n_entries;
    out->max_entries = c->max_entries;
    out->map_bytes = (uint64_t)c->map_cap * 16;
    out->n_slabs = c->n_slabs;
    out->slab_bytes = c->slab_bytes;
    return IBP_OK;
}

extern "C" void ibp_cache_destroy(ibp_cache* c) {
    if (!c) return;
    if (c->map_dev) cudaFree(c->map_dev);
    for (int s = 0; s < 8; ++s) {
        if (!c->slab_dev[s]) continue;
        if (c->slab_imported[s]) cudaIpcCloseMemHandle(c->slab_dev[s]);    // a peer process's slab: unmap, the owner frees it
        else cudaFree(c->slab_dev[s]);
    }
    (void)cudaGetLastError();
    delete c;
}
