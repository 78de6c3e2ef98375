// ibp_shared.cpp -- one packed store for all the ranks of a one-process-per-GPU job.
//
// A built handle is exported as a self-contained image into a POSIX shared-memory segment; every rank opens the segment and
// gets a handle that borrows the store and the host metadata mirrors from the mapping.  ibp_upload_metadata (ibp_device.cu)
// page-locks and GPU-maps the store for the calling process, so each GPU reads the same physical pages over its own PCIe link.
#include <cuda_runtime.h>
#include <fcntl.h>
#include <sys/mman.h>
#include <sys/stat.h>
#include <sys/syscall.h>
#include <unistd.h>

#include <cerrno>
#include <cstdio>
#include <cstring>
#include <new>

#include "ibp_internal.h"

namespace {

constexpr uint64_t SHM_MAGIC = 0x31304D4853504249ull;   // "IBPSHM01"

struct ShmHeader {
    uint64_t magic, total_bytes;
    ibp_build_params p;
    uint64_t n_groups, row_stride_strided, store_bytes, store_used, packed_bytes_rows, packed_bytes_bytealigned, n_rows_raw, capacity_rows;
    uint32_t n_words, max_stride, thresholded, slot_layout, slot_bytes;
    int32_t max_runs;
    uint64_t off_meta, n_meta, off_gtab, n_gtab, off_row_off, n_row_off, off_row_flag, n_row_flag, off_row_size, n_row_size, off_store;
    uint64_t ready;                                       // written last: a reader never sees a half-written image
};

uint64_t up(uint64_t v, uint64_t a) { return (v + a - 1) / a * a; }

bool good_name(const char* s) {
    if (!s || s[0] != '/' || !s[1]) return false;
    for (const char* c = s + 1; *c; ++c)
        if (*c == '/') return false;
    return strlen(s) < 200;
}

// mbind through the raw syscall (no libnuma in the image); best effort
void place_pages(void* base, uint64_t bytes, int numa_policy) {
#ifdef SYS_mbind
    if (numa_policy <= 0) return;
    unsigned long mask[16];
    memset(mask, 0, sizeof mask);
    int mode;
    if (numa_policy == 1) {
        mode = 3;   // MPOL_INTERLEAVE
        int nodes = 0;
        for (int k = 0; k < 1024; ++k) {
            char path[64];
            snprintf(path, sizeof path, "/sys/devices/system/node/node%d", k);
            if (access(path, F_OK) != 0) break;
            mask[k / (8 * sizeof(unsigned long))] |= 1ul << (k % (8 * sizeof(unsigned long)));
            ++nodes;
        }
        if (nodes < 2) return;
    } else {
        mode = 2;   // MPOL_BIND
        const int node = numa_policy - 2;
        if (node < 0 || node >= 1024) return;
        mask[node / (8 * sizeof(unsigned long))] |= 1ul << (node % (8 * sizeof(unsigned long)));
    }
    (void)syscall(SYS_mbind, base, (unsigned long)bytes, mode, mask, (unsigned long)(8 * sizeof mask), 0u);
#else
    (void)base; (void)bytes; (void)numa_policy;
#endif
}

}  // namespace

extern "C" ibp_status ibp_device_numa_node(int device, int* node) {
    if (!node) { ibp_set_error("ibp_device_numa_node: null argument"); return IBP_ERR_INVALID_ARG; }
    *node = -1;
    char bdf[32];
    if (cudaDeviceGetPCIBusId(bdf, sizeof bdf, device) != cudaSuccess) { (void)cudaGetLastError(); ibp_set_error("ibp_device_numa_node: no CUDA device %d", device); return IBP_ERR_CUDA; }
    for (char* c = bdf; *c; ++c) if (*c >= 'A' && *c <= 'Z') *c = (char)(*c - 'A' + 'a');
    char path[128];
    snprintf(path, sizeof path, "/sys/bus/pci/devices/%s/numa_node", bdf);
    if (FILE* f = fopen(path, "r")) {
        int v = -1;
        if (fscanf(f, "%d", &v) == 1) *node = v;
        fclose(f);
    }
    return IBP_OK;
}

extern "C" ibp_status ibp_export_shared(const ibp_handle* h, const char* shm_name, int numa_policy) {
    if (!h || !good_name(shm_name)) { ibp_set_error("ibp_export_shared: bad argument (the name must look like \"/name\")"); return IBP_ERR_INVALID_ARG; }
    if (!h->store) { ibp_set_error("ibp_export_shared: the handle has no store"); return IBP_ERR_BAD_STATE; }
    ShmHeader H;
    memset(&H, 0, sizeof H);
    H.magic = SHM_MAGIC;
    H.p = h->p;
    H.n_groups = h->n_groups; H.row_stride_strided = h->row_stride_strided;
    H.store_bytes = h->store_bytes; H.store_used = h->store_used;
    H.packed_bytes_rows = h->packed_bytes_rows; H.packed_bytes_bytealigned = h->packed_bytes_bytealigned;
    H.n_rows_raw = h->n_rows_raw; H.capacity_rows = h->capacity_rows;
    H.n_words = h->n_words; H.max_stride = h->max_stride; H.thresholded = h->thresholded; H.slot_layout = h->slot_layout; H.slot_bytes = h->slot_bytes;
    H.max_runs = h->max_runs;
    uint64_t cur = up(sizeof(ShmHeader), 4096);
    auto place = [&](uint64_t& off, uint64_t& cnt, uint64_t count, uint64_t elem) { off = cur; cnt = count; cur = up(cur + count * elem, 4096); };
    place(H.off_meta, H.n_meta, h->meta.size(), 4);
    place(H.off_gtab, H.n_gtab, h->gtab.size(), sizeof(IbpGroupEntry));
    place(H.off_row_off, H.n_row_off, h->row_off.size(), 4);
    place(H.off_row_flag, H.n_row_flag, h->row_flag.size(), 4);
    place(H.off_row_size, H.n_row_size, h->row_size.size(), 1);
    H.off_store = cur;
    cur = up(cur + h->store_bytes, 4096);
    H.total_bytes = cur;

    shm_unlink(shm_name);
    const int fd = shm_open(shm_name, O_CREAT | O_EXCL | O_RDWR, 0600);
    if (fd < 0) { ibp_set_error("ibp_export_shared: shm_open(%s) failed: %s", shm_name, strerror(errno)); return IBP_ERR_OUT_OF_MEMORY; }
    if (ftruncate(fd, (off_t)H.total_bytes) != 0) {
        ibp_set_error("ibp_export_shared: ftruncate(%llu) failed: %s", (unsigned long long)H.total_bytes, strerror(errno));
        close(fd); shm_unlink(shm_name);
        return IBP_ERR_OUT_OF_MEMORY;
    }
    void* base = mmap(nullptr, H.total_bytes, PROT_READ | PROT_WRITE, MAP_SHARED, fd, 0);
    close(fd);
    if (base == MAP_FAILED) { ibp_set_error("ibp_export_shared: mmap failed: %s", strerror(errno)); shm_unlink(shm_name); return IBP_ERR_OUT_OF_MEMORY; }
    place_pages(base, H.total_bytes, numa_policy);           // before the first touch
    uint8_t* b = (uint8_t*)base;
    auto put = [&](uint64_t off, const void* src, uint64_t nbytes) { if (nbytes) memcpy(b + off, src, nbytes); };   // an empty vector's data() may be null
    put(H.off_meta, h->meta.data(), H.n_meta * 4);
    put(H.off_gtab, h->gtab.data(), H.n_gtab * sizeof(IbpGroupEntry));
    put(H.off_row_off, h->row_off.data(), H.n_row_off * 4);
    put(H.off_row_flag, h->row_flag.data(), H.n_row_flag * 4);
    put(H.off_row_size, h->row_size.data(), H.n_row_size);
    {
        const int64_t nchunk = (int64_t)((h->store_bytes + (1u << 22) - 1) >> 22);
#pragma omp parallel for schedule(static)
        for (int64_t c = 0; c < nchunk; ++c) {
            const uint64_t o = (uint64_t)c << 22, len = h->store_bytes - o < (1u << 22) ? h->store_bytes - o : (1u << 22);
            memcpy(b + H.off_store + o, h->store + o, len);
        }
    }
    memcpy(b, &H, sizeof H);
    __atomic_store_n(&((ShmHeader*)b)->ready, 1ull, __ATOMIC_RELEASE);
    munmap(base, H.total_bytes);
    return IBP_OK;
}

extern "C" ibp_status ibp_open_shared(const char* shm_name, ibp_handle** out_handle) {
    if (!good_name(shm_name) || !out_handle) { ibp_set_error("ibp_open_shared: bad argument (the name must look like \"/name\")"); return IBP_ERR_INVALID_ARG; }
    const int fd = shm_open(shm_name, O_RDWR, 0600);
    if (fd < 0) { ibp_set_error("ibp_open_shared: shm_open(%s) failed: %s", shm_name, strerror(errno)); return IBP_ERR_INVALID_ARG; }
    struct stat sb;
    if (fstat(fd, &sb) != 0 || (uint64_t)sb.st_size < sizeof(ShmHeader)) { close(fd); ibp_set_error("ibp_open_shared: %s is not an IBP store image", shm_name); return IBP_ERR_INVALID_ARG; }
    void* base = mmap(nullptr, (size_t)sb.st_size, PROT_READ | PROT_WRITE, MAP_SHARED, fd, 0);
    close(fd);
    if (base == MAP_FAILED) { ibp_set_error("ibp_open_shared: mmap failed: %s", strerror(errno)); return IBP_ERR_OUT_OF_MEMORY; }
    const ShmHeader* H = (const ShmHeader*)base;
    const uint64_t total = (uint64_t)sb.st_size;
    auto inside = [&](uint64_t off, uint64_t bytes) { return off <= total && bytes <= total - off; };
    if (H->magic != SHM_MAGIC || __atomic_load_n(&H->ready, __ATOMIC_ACQUIRE) != 1 || H->total_bytes != total ||
        H->p.struct_size != sizeof(ibp_build_params) || !inside(H->off_meta, H->n_meta * 4) || !inside(H->off_gtab, H->n_gtab * sizeof(IbpGroupEntry)) ||
        !inside(H->off_row_off, H->n_row_off * 4) || !inside(H->off_row_flag, H->n_row_flag * 4) || !inside(H->off_row_size, H->n_row_size) ||
        !inside(H->off_store, H->store_bytes)) {
        munmap(base, total);
        ibp_set_error("ibp_open_shared: %s is not a complete IBP store image of this library version", shm_name);
        return IBP_ERR_INVALID_ARG;
    }
    ibp_handle* h = new (std::nothrow) ibp_handle();
    if (!h) { munmap(base, total); ibp_set_error("ibp_open_shared: out of memory"); return IBP_ERR_OUT_OF_MEMORY; }
    uint8_t* b = (uint8_t*)base;
    h->p = H->p;
    h->n_groups = H->n_groups; h->n_words = H->n_words; h->row_stride_strided = H->row_stride_strided; h->max_stride = H->max_stride;
    h->store_bytes = H->store_bytes; h->store_used = H->store_used;
    h->packed_bytes_rows = H->packed_bytes_rows; h->packed_bytes_bytealigned = H->packed_bytes_bytealigned;
    h->thresholded = H->thresholded != 0; h->n_rows_raw = H->n_rows_raw;
    h->slot_layout = H->slot_layout != 0; h->slot_bytes = H->slot_bytes; h->capacity_rows = H->capacity_rows;
    h->max_runs = H->max_runs;
    h->meta.borrow((uint32_t*)(b + H->off_meta), H->n_meta);
    h->gtab.borrow((IbpGroupEntry*)(b + H->off_gtab), H->n_gtab);
    h->row_off.borrow((uint32_t*)(b + H->off_row_off), H->n_row_off);
    h->row_flag.borrow((uint32_t*)(b + H->off_row_flag), H->n_row_flag);
    h->row_size.borrow(b + H->off_row_size, H->n_row_size);
    h->store = b + H->off_store;
    h->store_kind = IBP_STORE_SHARED;
    h->shm_base = base;
    h->shm_bytes = total;
    *out_handle = h;
    return IBP_OK;
}

extern "C" ibp_status ibp_unlink_shared(const char* shm_name) {
    if (!good_name(shm_name)) { ibp_set_error("ibp_unlink_shared: bad name"); return IBP_ERR_INVALID_ARG; }
    if (shm_unlink(shm_name) != 0 && errno != ENOENT) { ibp_set_error("ibp_unlink_shared: %s", strerror(errno)); return IBP_ERR_INVALID_ARG; }
    return IBP_OK;
}
