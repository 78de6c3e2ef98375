/*
 * ibp.h -- C ABI of the B200-native Invariant Bit Packing library (libibp.so).
 *
 * What it is: the data-parallel hot path of IBP ("Reducing the GPU Memory Bottleneck with Lossless Compression for
 * ML", arxiv/paper_2605_30728; cited below as P:<line> of PAPER.md): a fused gather-and-decompress of indexed
 * compressed rows.  Rows ("tensors" in the paper) are compressed once on the host by removing the bits that are
 * identical across each group of rows, and kept in pinned, GPU-mapped host memory.  A CUDA kernel then
 * reads requested rows zero-copy over PCIe, re-inserts the invariant bits from per-group Mask/Bitval
 * metadata held in GPU memory, and writes the original rows into an HBM tensor.
 *
 * Two modes, selected by ibp_build_params.threshold_num/den (= tau = T/N):
 *   strict (tau = 1, the default): the paper's clustered compression with clusters that are fixed runs of
 *     rows and T = N_group: a bit is invariant iff every row of the group agrees, so every row of a group has the same
 *     packed length and there are no participation bits and no per-row raw flag.
 *   thresholded (1/2 < tau < 1; the paper's default codec, tau = 0.8): a bit is invariant when at least T = ceil(tau N_g)
 *     rows of the group agree; every 4-byte chunk of a row carries a participation bit saying whether it
 *     matches Bitval under Mask; rows that would not shrink by a whole byte are kept raw and flagged in a
 *     one-bit-per-row bitmask held in GPU memory.  A single group spanning all rows (blocked, group_param
 *     >= n_rows) is the paper's one global Mask/Bitval.  Row sizes depend on the data, so the library keeps a
 *     4-byte offset per row in GPU memory (16-byte units) over a dense store instead of the paper's fixed in-place
 *     slots: same bytes cross PCIe, less host memory, contiguous spans stay contiguous.
 *
 * Conventions
 *   - Bit p of a row is bit (p mod 8) of byte (p div 8).  Mask bit 1 = invariant; Bitval holds the invariant values
 *     and is 0 where Mask is 0.
 *   - A packed row is the row's bits at the Mask=0 positions, ascending p, LSB-first, zero padded to ceil(k/8)
 *     bytes and then to `align_bytes` (the alignment unit A).  This is the oracle's canonical order.
 *   - Thresholded mode: a compressed row is [participation bits, one per 4-byte chunk, chunk order][per chunk: its bits
 *     at the Mask=0 positions if it participates, else all 32 bits], LSB-first, zero padded to
 *     row_bytes - floor((bitsSaved - chunks)/8) bytes (Fig. 3 = P:243-299) and then to A; a raw row is the row.
 *     Rows lie in id order, each starting on a multiple of A (A >= 16 in this mode); with IBP_FLAG_SLOT_LAYOUT row r starts
 *     at r * roundup(row_bytes, A) instead (the paper's in-place slots).
 *   - Store layout.  Blocked groups: groups in order, each group's base aligned to max(A,16); rows of a group at
 *     base + j*stride_g.  Strided groups: matrix row r (= id div S) at r*rowstride, tile t at prefix_t inside it.
 *   - Pointers are named *_host (CPU addressable), *_dev (GPU addressable on the handle's device).
 *   - Streams are passed as void* (a cudaStream_t); NULL = the legacy default stream.
 *   - Every function returns ibp_status; 0 = success.  No C++ exception crosses this boundary.  ibp_last_error()
 *     returns a thread-local message for the last failing call.
 *   - There is no CPU fallback: ibp_build is host code by design (the compressor); every other step
 *     needs a CUDA device of compute capability 10.0 and fails with IBP_ERR_CUDA without one.
 *
 * Ownership: the caller owns rows_host, row_ids_dev, out_dev, packed_dev and the stream.  The handle owns all it
 * allocates (packed store, metadata copies on host and device) until ibp_destroy, which the caller may only call
 * after synchronising every stream that used the handle.
 * Thread safety: concurrent gather/decompress calls on one handle are allowed; build/upload/configure/destroy are not.
 */
#ifndef IBP_H
#define IBP_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct ibp_handle ibp_handle;

typedef enum {
    IBP_OK = 0,
    IBP_ERR_INVALID_ARG = 1,
    IBP_ERR_OUT_OF_MEMORY = 2,
    IBP_ERR_CUDA = 3,
    IBP_ERR_BAD_STATE = 4,   /* e.g. gather before ibp_upload_metadata */
    IBP_ERR_UNSUPPORTED = 5  /* e.g. a thresholded store above 64 GiB, a device that is not sm_100 */
} ibp_status;

typedef enum {
    IBP_GROUP_BLOCKED = 0, /* group(id) = id div group_param : runs of consecutive rows                    */
    IBP_GROUP_STRIDED = 1  /* group(id) = id mod group_param : column tiles of a row-major matrix (S tiles) */
} ibp_group_kind;

enum {
    IBP_FLAG_PAGEABLE_STORE = 1u,  /* keep the packed store in ordinary memory: no zero-copy gather (CPU-only tests)  */
    IBP_FLAG_HOSTALLOC_STORE = 2u, /* use cudaHostAlloc pinned memory instead of the default managed-host allocation  */
    IBP_FLAG_SLOT_LAYOUT = 4u      /* thresholded mode only: the paper's in-place storage -- row r keeps a fixed slot of
                                      roundup(row_bytes, A) bytes at r * slot, only its first `size` bytes are meaningful and
                                      read; one byte per row in GPU memory holds the size (16-byte units) instead of a 4-byte
                                      offset.  Host memory is not saved (the paper accepts that); in exchange a row can be
                                      (re)written in place, so the store is APPENDABLE: ibp_append_rows_device            */
};

typedef enum {
    IBP_STORE_PAGEABLE = 0,     /* ordinary host memory; the GPU cannot read it in place                              */
    IBP_STORE_PINNED = 1,       /* cudaHostAlloc(mapped|portable): page-locked, 4 KB GPU pages                        */
    IBP_STORE_MANAGED_HOST = 2, /* cudaMallocManaged, preferred location CPU, accessed-by GPU: host-resident, read in
                                   place over PCIe, mapped by the GPU with large pages        */
    IBP_STORE_SHARED = 3        /* a POSIX shared-memory segment (ibp_export_shared / ibp_open_shared), page-locked and
                                   GPU-mapped by every process that uploads it: ONE copy of the store in host RAM for all
                                   the ranks of a one-process-per-GPU job                                            */
} ibp_store_kind;

typedef struct {
    uint32_t struct_size;   /* = sizeof(ibp_build_params), for ABI growth                                        */
    uint32_t row_bytes;     /* bytes per row; multiple of 4 (the paper's 4-byte chunk), 4 .. 65536        */
    uint64_t n_rows;
    uint32_t group_kind;    /* ibp_group_kind                                                                    */
    uint32_t group_param;   /* G (blocked) or S (strided); >= 1                                                  */
    uint32_t threshold_num; /* tau = T/N as a fraction: 1/1 (or 0/0) = strict; 1/2 < tau < 1 = thresholded, e.g. 4/5   */
    uint32_t threshold_den;
    uint32_t align_bytes;   /* packed-row alignment unit A: power of two in 1..128 (16..128 thresholded); 0 = 32 */
    uint32_t index_span;    /* consecutive rows selected by one id in ibp_gather_decompress; 0 = 1               */
    uint32_t flags;         /* IBP_FLAG_*                                                                        */
    uint32_t n_threads;     /* host threads for the build; 0 = all                                               */
    uint64_t capacity_rows; /* IBP_FLAG_SLOT_LAYOUT: rows the store has slots for (>= n_rows; 0 = n_rows): the room
                               ibp_append_rows_device can fill.  Ignored otherwise.  (struct_size without this field -- the
                               layout of version 0.3 -- is accepted and means 0.)                                        */
} ibp_build_params;

typedef struct {
    uint64_t n_rows, n_groups;
    uint64_t packed_bytes_stored;      /* size of the packed store incl. alignment padding                       */
    uint64_t packed_bytes_rows;        /* sum over rows of the row stride roundup(ceil(k_g/8), A)                */
    uint64_t packed_bytes_bytealigned; /* sum over rows of ceil(k_g/8): the oracle's canonical size      */
    uint64_t metadata_bytes;           /* 2*row_bytes per group: Mask + Bitval                    */
    uint64_t aux_bytes;                /* per-group table (base offset, stride, k): 16 B per group               */
    uint32_t row_bytes, align_bytes, index_span, group_kind, group_param;
    uint32_t max_row_stride;           /* largest packed-row stride in bytes                                     */
    int32_t  device;                   /* device holding the metadata, -1 before ibp_upload_metadata             */
    uint32_t store_kind;               /* ibp_store_kind                                                         */
    uint32_t thresholded;              /* 0 = strict, 1 = thresholded mode                                       */
    uint32_t threshold_num, threshold_den;
    uint32_t reserved0;
    uint64_t n_rows_raw;               /* thresholded: rows kept uncompressed                            */
    uint64_t rowflag_bytes;            /* thresholded: per-row bitmask, 4*ceil(n_rows/32) bytes          */
    uint64_t rowoffset_bytes;          /* thresholded: per-row offsets, 4*(n_rows+1) bytes (0 with the slot layout) */
    uint64_t capacity_rows;            /* slot layout: rows the store has slots for; else n_rows                 */
    uint64_t rowsize_bytes;            /* slot layout: per-row sizes, 1 byte per slot; else 0                    */
    uint32_t slot_bytes;               /* slot layout: bytes per slot = roundup(row_bytes, A); else 0            */
    uint32_t reserved1;
} ibp_info;

/* -- S0, S0': host-side compressor (P:229-231 masks with T=N per group; P:237-241, P:275-298 packing). ---------------
 * rows_host: n_rows x row_bytes, row-major, borrowed for the duration of the call.  Synchronous, multi-threaded,
 * CPU only.  The handle allocates its own packed store in host memory the GPU reads in place (ibp_store_kind:
 * managed-host by default, cudaHostAlloc with IBP_FLAG_HOSTALLOC_STORE) when a CUDA device is present and
 * IBP_FLAG_PAGEABLE_STORE is not set, else ordinary memory (then only ibp_decompress_resident and the host
 * accessors work).  Thresholded mode: per-bit counters, T = ceil(tau N_g), participation bits, raw rows.
 * Errors: INVALID_ARG (null pointers, row_bytes not a multiple of 4, bad A, tau <= 1/2 or > 1, span not compatible
 * with the groups), UNSUPPORTED (thresholded store above 64 GiB), OUT_OF_MEMORY.                                   */
ibp_status ibp_build(const void* rows_host, const ibp_build_params* params, ibp_handle** out_handle);

/* -- GPU-side compressor (P:227-229 preprocessing "performed on the GPU", P:239 tensors partitioned
 * among warps, Fig. 3 = P:243-299; the way to build masks online, e.g. per-prefill KV masks).
 * rows_dev: n_rows x row_bytes, row-major, 16-byte aligned, readable by `device`: HBM, or pinned / managed host memory
 * read zero-copy.  Same parameters, modes and result as ibp_build -- identical Mask/Bitval/k_g and identical
 * packed bytes -- but S0 (AND/OR reduction or bit-sliced per-bit counters) and S0' (sizes, offsets, bit packing) run in
 * CUDA kernels, and the packed rows are written in place into the host store over PCIe.  The returned handle is
 * already attached to `device` (no ibp_upload_metadata needed; calling it is a no-op).  Host work that remains: the
 * store allocation, the prefix sum over per-group sizes (strict), copies of the metadata for the host accessors.
 * Synchronises the stream.  Errors as ibp_build, plus INVALID_ARG for IBP_FLAG_PAGEABLE_STORE, CUDA/UNSUPPORTED for a
 * missing or non-sm_100 device, UNSUPPORTED for groups of more than 2^32-1 rows.                                    */
ibp_status ibp_build_device(const void* rows_dev, const ibp_build_params* params, int device, void* cuda_stream,
                            ibp_handle** out_handle);

/* -- Online append ("we sample the KV cache generated from the prompt tokens to create the Mask
 * and Bitval.  This metadata is used to compress the KV cache generated in the decode phase").  The handle must use the slot
 * layout (IBP_FLAG_SLOT_LAYOUT) and have room: n_rows + n_new <= capacity_rows.  rows_dev: n_new x row_bytes on the handle's
 * device (HBM or mapped host memory), 16-byte aligned.  New row j gets id n_rows + j and is compressed by a CUDA kernel under the
 * EXISTING Mask/Bitval of its group (id div G, or id mod S) -- the metadata never changes -- and written into its slot of the host
 * store over PCIe; its size byte and its bit of the per-row bitmask are set in GPU memory.  The group must already have metadata:
 * strided groups need n_rows >= S at build time, blocked groups can only fill their last group (one group spanning all rows,
 * group_param >= capacity_rows, is the paper's single global Mask/Bitval and takes any number of rows).  Synchronises the stream;
 * the host mirrors (ibp_row_info, ibp_get_info) are updated.  Not concurrent with gathers that touch the new rows or with
 * another append.  index_span must be 1 or divide n_new.  Errors: BAD_STATE (no slot layout, before upload), INVALID_ARG,
 * UNSUPPORTED (no room, a group without metadata).                                                                     */
ibp_status ibp_append_rows_device(ibp_handle* h, const void* rows_dev, int64_t n_new, void* cuda_stream);

/* Where the time of an ibp_build_device call went (CUDA events on the stream around each kernel; total = wall clock of the
 * call including the host-side store allocation and copies).  BAD_STATE for a handle built by ibp_build.              */
typedef struct {
    double mask_ms;      /* ibp_mask_kernel (+ slice merge): reads every row once                                    */
    double size_ms;      /* thresholded: ibp_size_kernel (reads every row once); 0 in strict mode                    */
    double scan_ms;      /* thresholded: row-offset scan; 0 in strict mode                                            */
    double pack_ms;      /* ibp_pack_kernel / ibp_pack_t_kernel: reads every row once, writes the packed store       */
    double total_ms;
    uint64_t raw_bytes;  /* n_rows * row_bytes                                                                        */
    uint64_t store_bytes;/* packed bytes written to the store (rows incl. alignment padding)                          */
    uint32_t slices_per_group, reserved;
} ibp_build_stats;
ibp_status ibp_get_build_stats(const ibp_handle* h, ibp_build_stats* out);

/* -- S0'': copy Mask/Bitval and the group table to HBM on `device` ("stored in GPU memory").  Idempotent for the
 * same device; INVALID_ARG for a second device.  Synchronises the stream before returning.                         */
ibp_status ibp_upload_metadata(ibp_handle* h, int device, void* cuda_stream);

/* -- S1-S6: the hot path.  For i in [0,n), j in [0,index_span):
 *      out_dev[(i*index_span + j)*row_bytes ...] = original row  row_ids_dev[i]*index_span + j.
 * row_ids_dev: n int64 on the device.  out_dev: n*index_span*row_bytes bytes on the device, 16-byte aligned.
 * Asynchronous on the stream.  Duplicate ids allowed.  n == 0 is a no-op.  Ids are not validated (out of range =
 * undefined behaviour), see ibp_validate_ids.  BAD_STATE before upload or with a pageable store.                   */
ibp_status ibp_gather_decompress(ibp_handle* h, const int64_t* row_ids_dev, int64_t n, void* out_dev, void* cuda_stream);

/* The same gather of random rows (index_span 1) for callers that may not allocate: code under CUDA graph capture, serving
 * loops, harnesses that forbid cudaMalloc.  ibp_gather_decompress takes the workspace of its locality-order pre-pass (bucket
 * counters + the processing order of the batch) from cudaMallocAsync; this entry point keeps that scratch in a file-scope
 * device array of the library instead and calls no cudaMalloc / cudaMallocAsync / cudaFree nor any allocating routine.
 *   - Limit: n <= IBP_NOALLOC_MAX_IDS ids per call; a larger n is rejected with IBP_ERR_INVALID_ARG and a message (split the
 *     batch).  The array is 256 B + 1 MiB of counters + 4 B per id = 5.25 MB, and every GPU that loads the library holds it
 *     until the process exits.
 *   - Same arguments, layout and result as ibp_gather_decompress, bit for bit (the pre-pass only changes the order in which rows
 *     are fetched; repeated ids are each fetched, there is no de-duplication and no compressed cache on this path).
 *   - The handle's device must be the CURRENT device of the calling thread (BAD_STATE otherwise).  The array's device address is
 *     looked up once per device on the first call there (cudaGetSymbolAddress): make that first call outside stream capture.
 *   - Every call on a device shares the one array, which keeps the last call's contents; the call clears its counters on the
 *     stream first.  Two calls that OVERLAP on the GPU (different streams, or threads, without an ordering between them) race on
 *     the array and give undefined output: keep calls on one stream or order them with events.
 * Asynchronous on the stream.  UNSUPPORTED with index_span > 1; BAD_STATE before upload or with a pageable store.        */
#define IBP_NOALLOC_MAX_IDS (1 << 20)
ibp_status ibp_gather_decompress_noalloc(ibp_handle* h, const int64_t* row_ids_dev, int64_t n, void* out_dev, void* cuda_stream);

/* Same result with HOST buffers: row_ids_host (n int64) is copied to the device, the gather runs, and the rows are
 * copied back into out_host, all on the stream, which is synchronised before returning.  The end-to-end entry point
 * bench.py times.  The buffers should be pinned for full copy speed; pageable memory works.
 * Paths: a batch the library would de-duplicate (ibp_set_dedup_mode: mode 1, or automatic and n >= 16384) is gathered into a
 * device staging buffer -- every distinct row crosses PCIe once -- and copied out in chunks; any other batch whose out_host is
 * pinned and GPU-mapped is decoded straight into out_host by the kernel (nothing staged; every id is fetched, which is what
 * the handle's de-duplication setting asks for in that case).  There is no host entry point for the compressed GPU cache:
 * a cached gather is ibp_cache_gather_decompress with device buffers.                                              */
ibp_status ibp_gather_decompress_host(ibp_handle* h, const int64_t* row_ids_host, int64_t n, void* out_host, void* cuda_stream);

/* -- S8: decode rows [first_row, first_row+n_rows) whose packed bytes the caller already staged in device memory
 * exactly as they lie in the host store (ibp_packed_range gives the source range; e.g. cudaMemcpyAsync, or a
 * compressed GPU cache slab).  first_row must start a layout unit: a multiple of G (blocked) or of S
 * (strided); in thresholded mode with blocked groups every row starts a unit.  packed_dev must be 16-byte aligned.
 * Asynchronous on the stream.                                                                                      */
ibp_status ibp_decompress_resident(ibp_handle* h, const void* packed_dev, int64_t first_row, int64_t n_rows,
                                   void* out_dev, void* cuda_stream);

/* Zero-copy gather of the contiguous rows [first_row, first_row+n_rows) straight from the host store (whole weight
 * matrices / layers streamed in order): same unit rule as above, no id list.  out_dev[j*row_bytes ...] = row
 * first_row + j.  Asynchronous on the stream.                                                                      */
ibp_status ibp_gather_decompress_range(ibp_handle* h, int64_t first_row, int64_t n_rows, void* out_dev, void* cuda_stream);

/* ibp_gather_decompress_range with a HOST destination: out_host receives n_rows*row_bytes bytes.  A pinned, GPU-mapped
 * destination (cudaHostAlloc / cudaHostRegister / ibp_host_alloc) is written by the decode kernel directly; any other memory
 * goes through a device staging buffer and one copy.  Synchronises the stream before returning.                          */
ibp_status ibp_gather_decompress_range_host(ibp_handle* h, int64_t first_row, int64_t n_rows, void* out_host, void* cuda_stream);

/* Several contiguous ranges decoded by ONE kernel launch (whole decoder layers streamed in order: a 7B-shaped layer is
 * seven matrices = seven handles).  Range i: rows [first_row, first_row+n_rows) of `handle` (same unit rule as
 * ibp_decompress_resident) go to out_dev; packed_dev != NULL: the packed bytes of exactly that range staged in device memory
 * (as ibp_decompress_resident); packed_dev == NULL: read zero-copy from the handle's host store (as
 * ibp_gather_decompress_range).  ranges_host is read during the call only.  Consecutive ranges of strict-mode handles with the
 * same row width are walked by one persistent grid, at most 8 per launch (more ranges = more launches); thresholded handles and
 * handles with ibp_set_stream_mode(0) are decoded range by range.  The launch shape (ibp_configure) is that of the first handle
 * of each launch.  All handles must live on one device.  Asynchronous on the stream.  Output is identical to the per-range
 * calls.  Errors: INVALID_ARG (null pointers, ranges, alignment, mixed devices), BAD_STATE (before upload; host-store range of
 * a pageable store), UNSUPPORTED (rows too long for the shared-memory stages).                                             */
typedef struct {
    ibp_handle* handle;
    const void* packed_dev;
    int64_t first_row, n_rows;
    void* out_dev;
} ibp_range_desc;
ibp_status ibp_decode_ranges(const ibp_range_desc* ranges_host, uint32_t n_ranges, void* cuda_stream);

/* The same with HOST destinations: the out_dev field of every range holds a HOST pointer that receives n_rows*row_bytes bytes.
 * When all destinations are pinned, GPU-mapped memory (cudaHostAlloc / cudaHostRegister / ibp_host_alloc) the decode kernels store
 * into them directly, with the batching of ibp_decode_ranges (a 7-matrix layer: one launch); otherwise every range goes through
 * ibp_gather_decompress_range_host (device staging buffer + copy; packed_dev ranges then are UNSUPPORTED).  Synchronises the
 * stream before returning.  Errors as ibp_decode_ranges.                                                                     */
ibp_status ibp_decode_ranges_host(const ibp_range_desc* ranges_host, uint32_t n_ranges, void* cuda_stream);

/* Byte range of the packed store that holds rows [first_row, first_row+n_rows) (same unit rule as above).         */
ibp_status ibp_packed_range(const ibp_handle* h, int64_t first_row, int64_t n_rows, const void** host_ptr, uint64_t* nbytes);

/* Device-visible address of byte 0 of the packed store (what the decode kernels read; for mock-transfer baselines that move
 * packed bytes without decoding).  BAD_STATE before ibp_upload_metadata or with a pageable store.               */
ibp_status ibp_store_device_ptr(const ibp_handle* h, const void** dev_ptr);

/* Location of one packed row inside the store (host pointer, stride bytes, variant bits k).  For cross-checks.
 * Thresholded mode: stride = stored bytes incl. padding, k_bits = 8 * the row's byte-aligned size.                 */
ibp_status ibp_packed_row(const ibp_handle* h, int64_t row, const void** host_ptr, uint32_t* stride_bytes, uint32_t* k_bits);

/* Both modes: where a row lies (host pointer), the bytes it occupies incl. alignment padding, its byte-aligned size
 * (strict: ceil(k_g/8); thresholded: row_bytes - bytesSaved, or row_bytes when raw) and whether it is compressed
 * (strict: always 1; thresholded: the row's bit of the bitmask).  Any out pointer may be NULL.               */
ibp_status ibp_row_info(const ibp_handle* h, int64_t row, const void** host_ptr, uint32_t* stored_bytes, uint32_t* size_bytes,
                        int* is_compressed);

/* Host copies of one group's metadata: Mask and Bitval (row_bytes each) and k_g = 8*row_bytes - popcount(Mask).  For
 * oracle cross-checks.                                                                                              */
ibp_status ibp_get_metadata_host(const ibp_handle* h, int64_t group, const void** mask, const void** bitval, uint32_t* k_bits);

ibp_status ibp_get_info(const ibp_handle* h, ibp_info* out);

/* Launch shape of the decode kernels: max_ctas limits the grid, so that a consumer kernel can share the GPU ("We
 * reserved only 64 SMs for decompression"); 0 = library default: resident decode fills the GPU; contiguous runs read from the
 * HOST store (span gathers, ibp_gather_decompress_range, host ranges of ibp_decode_ranges) are bound by the link and take 48
 * CTAs; locality-ordered random gathers of line-sized rows take the grid that keeps about 415 KB of packed bytes in flight
 * (about 100 CTAs) -- the same or better throughput, and the other SMs stay free for the consumer of the rows; warps_per_cta of the random-row kernel: 0 = default
 * (8), else 1..8 (the kernel is compiled for CTAs of at most 256 threads); INVALID_ARG above 8.                     */
ibp_status ibp_configure(ibp_handle* h, uint32_t max_ctas, uint32_t warps_per_cta);

/* Debug pre-pass: *n_bad_host = number of ids outside [0, n_rows/index_span).  Synchronises the stream.           */
ibp_status ibp_validate_ids(ibp_handle* h, const int64_t* row_ids_dev, int64_t n, int64_t* n_bad_host, void* cuda_stream);

/* Sum over the DISTINCT ids of a batch of the packed bytes one id moves over PCIe (index_span rows each): the
 * algorithmic link traffic of one ibp_gather_decompress call.  stored = what the kernels fetch: each row with its alignment
 * padding (a single row: up to whole 32-byte sectors, at most its stride; rows of a span: the whole contiguous run),
 * bytealigned = ceil(k/8) per row.  Host-side helper for roofline accounting; ids on the host.                      */
ibp_status ibp_batch_link_bytes(const ibp_handle* h, const int64_t* row_ids_host, int64_t n, uint64_t* n_unique,
                                uint64_t* stored, uint64_t* bytealigned);

/* -- Compressed GPU software cache (Fig. 6a).  A static cache of packed rows in GPU memory:
 * "data slabs" (one contiguous region each, up to 8: the 3-bit slab id) hold the rows exactly as they lie in the host store,
 * and a hash map in GPU memory maps a row id to ONE 64-bit value (reading R22 for the bit positions):
 *      bits  0..39  byte offset inside the slab (40 bits, 1 TB)
 *      bits 40..42  slab id (3 bits)
 *      bit  43      1 = the row is stored compressed, 0 = raw (thresholded mode keeps some rows raw; strict: always 1)
 *      bits 44..63  spare, zero
 * ibp_cache_gather_decompress is ibp_gather_decompress with one extra step in S1: the id is looked up in the map; a hit
 * reads the packed row from its slab (HBM), a miss reads it from the host store over PCIe; S2-S6 are the same kernel code,
 * so the output is identical.  index_span must be 1.  The cache borrows the handle, which must outlive it.             */
typedef struct ibp_cache ibp_cache;
#define IBP_CACHE_MISS 0xFFFFFFFFFFFFFFFFull
typedef struct {
    uint64_t capacity_bytes, used_bytes;   /* all slabs together                                                        */
    uint64_t n_entries, max_entries;
    uint64_t map_bytes;                    /* hash map in GPU memory: 16 bytes per slot, >= 2 slots per possible entry  */
    uint32_t n_slabs, reserved;
    uint64_t slab_bytes;                   /* capacity of one slab                                                      */
} ibp_cache_info;
/* capacity_bytes is split evenly over n_slabs (1..8) slabs on the handle's device; max_entries bounds the map (0 = n_rows).
 * BAD_STATE before ibp_upload_metadata / with a pageable store; UNSUPPORTED when index_span != 1.                       */
ibp_status ibp_cache_create(ibp_handle* h, uint64_t capacity_bytes, uint32_t n_slabs, uint64_t max_entries, void* cuda_stream,
                            ibp_cache** out_cache);
/* Static fill: for every id of row_ids_host (n int64 on the HOST, in priority order) that is not cached yet, copies its packed
 * row from the host store into the current slab (a CUDA kernel reading zero-copy) and adds the map entry; stops at the first
 * row that does not fit.  *n_inserted_host (optional) = rows added.  Synchronises the stream.  All ids are validated before
 * anything changes: INVALID_ARG for an id out of range, OUT_OF_MEMORY and CUDA errors leave the cache exactly as it was.
 * An insert may run while gathers on other streams use the cache: the slab bytes are written first and a map slot {key, value}
 * is published with one 16-byte compare-and-swap, so a concurrent gather sees a row either as cached or as not cached (then
 * it reads the host store) -- the output is the same.  Two inserts on one cache must not overlap.  Only slabs this cache
 * allocated are filled (a peer process's slab is filled by its owner: ibp_cache_insert_slab below).                        */
ibp_status ibp_cache_insert(ibp_cache* c, const int64_t* row_ids_host, int64_t n, void* cuda_stream, int64_t* n_inserted_host);

/* -- Slabs on several GPUs ("we allocate a contiguous memory region per interconnected GPU, which we call a data slab; e.g.,
 * an 8-GPU system would have 8 separate data slabs.  Together, these slabs make up the data store"; "using the data slab ID,
 * we identify which GPU slab the required tensor is on").  The slab id of a map value names the GPU whose memory holds the row; the
 * decode kernel of the handle's device reads a hit from that slab -- its own HBM, or a peer GPU's memory over NVLink -- with the same
 * bulk copy, so S2-S6 and the output do not change.
 *
 * One process driving several GPUs: ibp_cache_create_multi is ibp_cache_create with slab s allocated on CUDA device
 * slab_devices[s] (-1 = the handle's device); peer access from the handle's device is enabled (UNSUPPORTED when the two devices
 * cannot reach each other, INVALID_ARG for a device this process does not have).  ibp_cache_insert then fills the slabs in order,
 * writing peer slabs over the interconnect.
 *
 * One process per GPU (the layout of this library's multi-GPU runs): every rank creates its cache with its own slab
 * local and the others marked IBP_SLAB_REMOTE, publishes its slab with ibp_cache_slab_export (a CUDA IPC memory handle,
 * IBP_IPC_HANDLE_BYTES bytes, sent to the peers by any host channel), and maps the peers' slabs with ibp_cache_slab_attach.  Rows
 * are then placed slab by slab with ibp_cache_insert_slab: EVERY rank calls it for EVERY slab with the same id list -- the placement
 * (offsets in insertion order, 16-byte covers) is a function of the list alone, so all ranks build identical map entries -- and
 * passes fill = 1 only for the slab it owns (it copies the packed rows from the host store into it); fill = 0 adds the entries
 * without touching the slab.  After all ranks have returned (the call synchronises the stream; the ranks then meet at a host
 * barrier) every rank's gathers hit any slab.  Errors: BAD_STATE (exporting a slab this cache did not allocate, attaching over a
 * slab that has memory, inserting into a slab with no memory, fill = 1 on a peer's slab), INVALID_ARG, CUDA.                   */
#define IBP_SLAB_REMOTE (-2)
#define IBP_IPC_HANDLE_BYTES 64
ibp_status ibp_cache_create_multi(ibp_handle* h, uint64_t capacity_bytes, uint32_t n_slabs, const int32_t* slab_devices,
                                  uint64_t max_entries, void* cuda_stream, ibp_cache** out_cache);
ibp_status ibp_cache_slab_export(const ibp_cache* c, uint32_t slab, void* ipc_handle_out);
ibp_status ibp_cache_slab_attach(ibp_cache* c, uint32_t slab, const void* ipc_handle);
ibp_status ibp_cache_insert_slab(ibp_cache* c, uint32_t slab, const int64_t* row_ids_host, int64_t n, int fill, void* cuda_stream,
                                 int64_t* n_inserted_host);
/* S1-S6 with the cache in front of the host store (see above).  Arguments as ibp_gather_decompress.                    */
ibp_status ibp_cache_gather_decompress(ibp_cache* c, const int64_t* row_ids_dev, int64_t n, void* out_dev, void* cuda_stream);
/* entries_dev[i] = the map value of row_ids_dev[i], or IBP_CACHE_MISS.  For tests and hit-rate accounting.  Asynchronous. */
ibp_status ibp_cache_lookup(ibp_cache* c, const int64_t* row_ids_dev, int64_t n, uint64_t* entries_dev, void* cuda_stream);
/* Copies nbytes of slab memory addressed by a map value (slab id + offset) to the host.  For cross-checks.  Synchronous.   */
ibp_status ibp_cache_read(const ibp_cache* c, uint64_t entry, uint32_t nbytes, void* out_host);
ibp_status ibp_cache_get_info(const ibp_cache* c, ibp_cache_info* out);
void ibp_cache_destroy(ibp_cache* c);

/* -- One store for all ranks of a one-process-per-GPU job ("each GPU reads the shared pinned store over its own
 * PCIe link").  ibp_export_shared writes a complete image of a built handle -- parameters, Mask/Bitval, group table, row
 * offsets / sizes / flags, the packed store -- into the POSIX shared-memory segment `shm_name` (created; an existing one is
 * replaced).  numa_policy places the segment's pages before they are first touched: 0 = the kernel's default (first touch:
 * the exporting thread's node), 1 = interleaved over all NUMA nodes (ranks on both sockets see the same average distance),
 * 2 + k = bound to NUMA node k (e.g. the node of the GPU that reads it; ibp_device_numa_node).  Placement is best effort: on a
 * machine without NUMA support the call still succeeds.  ibp_open_shared maps the segment in another (or the same) process and
 * returns a handle that BORROWS everything from it: no per-process copy of the store or of the host metadata mirrors.
 * ibp_upload_metadata on such a handle page-locks and GPU-maps the store for this process (cudaHostRegister) and replicates the
 * metadata on its device, after which every gather / decode entry point works as on the original.  The handle is read-only
 * (ibp_append_rows_device: BAD_STATE).  ibp_destroy unmaps; ibp_unlink_shared removes the name (the memory lives on until the
 * last process unmaps it).  Errors: INVALID_ARG (names, a segment that is not an IBP image or not complete), OUT_OF_MEMORY
 * (shm_open / ftruncate / mmap failed), CUDA (registration).                                                          */
ibp_status ibp_export_shared(const ibp_handle* h, const char* shm_name, int numa_policy);
ibp_status ibp_open_shared(const char* shm_name, ibp_handle** out_handle);
ibp_status ibp_unlink_shared(const char* shm_name);
/* NUMA node of a CUDA device's PCIe slot (sysfs), -1 if unknown.                                                       */
ibp_status ibp_device_numa_node(int device, int* node);

void ibp_destroy(ibp_handle* h);
const char* ibp_last_error(void);
const char* ibp_version(void);

/* -- Baseline in the same library so both are timed the same way ("GPU (Aligned)" zero-copy gather):
 *      out_dev[i*row_bytes ...] = rows_host_mapped[row_ids_dev[i]*row_bytes ...], uncompressed.
 * rows_host_mapped must be pinned+mapped host memory (device-visible address) or device memory; row_bytes % 16 == 0. */
ibp_status ibp_gather_uncompressed(const void* rows_mapped, uint32_t row_bytes, const int64_t* row_ids_dev, int64_t n,
                                   void* out_dev, void* cuda_stream);

/* Same gather with the locality-ordered pre-pass of ibp_gather_decompress when locality_order
 * != 0; n_rows = number of rows of the table (needed to size the buckets).                                         */
ibp_status ibp_gather_uncompressed_ex(const void* rows_mapped, uint32_t row_bytes, uint64_t n_rows, const int64_t* row_ids_dev,
                                      int64_t n, void* out_dev, int locality_order, void* cuda_stream);

/* Tuning/test hook: locality-ordered processing of random gathers: 1 = always, 0 = never, -1 = automatic (default:
 * on for stores above 64 MiB and batches of >= 4096 ids).  Results are identical either way.                         */
ibp_status ibp_set_order_mode(ibp_handle* h, int mode);

/* Tuning/test hook: engine that moves packed rows into shared memory: 1 = cp.async.bulk + mbarrier (TMA, default),
 * 0 = 16-byte cp.async through the load/store unit.  Results are identical either way.                              */
ibp_status ibp_set_fetch_mode(ibp_handle* h, int mode);

/* De-duplication of random gathers (index_span 1): 1 = every distinct id of the batch crosses PCIe once and its decoded row
 * is replicated HBM -> HBM to the positions of its repeats (skewed batches, e.g. DLRM lookups); 0 = every id is fetched
 * (for callers that know their ids are distinct, e.g. a de-duplicating GNN sampler); -1 = automatic (default): on for
 * batches of >= 16384 ids.  Output is identical either way.  Needs n_rows < 2^32 - 1, else it is ignored.          */
ibp_status ibp_set_dedup_mode(ibp_handle* h, int mode);

/* Tuning/test hook: contiguous runs (spans, ranges, resident decode): 1 = TMA producer/consumer stream kernels (default),
 * 0 = per-row fetch kernel, 2 = stream kernels with the row-per-warp form of the thresholded decode instead of the sub-warp
 * form used for 128/256/512-byte rows.  Results are identical in every mode.                                         */
ibp_status ibp_set_stream_mode(ibp_handle* h, int mode);

/* Tuning/test hook: rows each warp keeps in flight in random gathers (ring depth): 1, 2 or 4; 0 = automatic (default: two;
 * locality-ordered gathers of line-sized rows take 1, 2 or 4 and a grid chosen so that about 415 KB of packed bytes are in
 * flight on the whole GPU -- DESIGN.md section 6, P19).                                                              */
ibp_status ibp_set_rows_in_flight(ibp_handle* h, int n);

/* -- Pinned, GPU-mapped host memory for callers that are not CUDA programs (the baseline table, pinned id buffers).  */
ibp_status ibp_host_alloc(size_t nbytes, void** host_ptr, void** dev_ptr);
ibp_status ibp_host_free(void* host_ptr);
/* Host-resident managed memory with a direct mapping on `device` (the store kind IBP_STORE_MANAGED_HOST); one pointer
 * serves host and device.                                                                                           */
ibp_status ibp_host_alloc_managed(size_t nbytes, int device, void** ptr);
ibp_status ibp_host_free_managed(void* ptr);

/* -- Link ceilings measured on this machine, for the roofline (BASELINE.json: "measured cudaMemcpy H2D ceiling").
 * ibp_measure_h2d: best of `reps` cudaMemcpyAsync H2D copies of nbytes from pinned memory, in GB/s.
 * ibp_measure_zero_copy_read: best of `reps` SM-issued contiguous 16-byte zero-copy reads of nbytes, in GB/s.       */
ibp_status ibp_measure_h2d(int device, size_t nbytes, int reps, double* gbps);
ibp_status ibp_measure_zero_copy_read(int device, size_t nbytes, int reps, double* gbps);
/* ibp_measure_d2h: best of `reps` cudaMemcpyAsync D2H copies of nbytes into pinned memory (the ceiling of the GPU-side
 * compressor's store writes), in GB/s.                                                                              */
ibp_status ibp_measure_d2h(int device, size_t nbytes, int reps, double* gbps);
/* ibp_measure_random_read: SM-issued zero-copy reads of `span_bytes`-byte spans (16..512, multiple of 16) at uniformly random
 * span-aligned offsets inside a managed host-resident buffer of `footprint_bytes`; best of `reps`, in spans per second
 * and GB/s.  This is the ceiling of a random gather of small packed rows: above a few hundred MB of footprint it is set
 * by address translation on the host path, not by the link.                                   */
ibp_status ibp_measure_random_read(int device, size_t footprint_bytes, uint32_t span_bytes, int reps, double* spans_per_s,
                                   double* gbps);
/* The same probe over host memory obtained in other ways, to show what the store kind costs on a machine: the span rate of a large
 * footprint follows the GPU-side page size of the mapping (managed host-resident memory is mapped with large GPU pages; page-locked
 * memory with 4 KB ones, whatever the host page size).  UNSUPPORTED: no huge pages are reserved on this machine (HUGETLB).       */
enum {
    IBP_MEM_MANAGED_HOST = 0,          /* cudaMallocManaged, preferred location CPU, accessed-by GPU (the default store kind)      */
    IBP_MEM_HOSTALLOC = 1,             /* cudaHostAlloc mapped (IBP_FLAG_HOSTALLOC_STORE)                                          */
    IBP_MEM_MALLOC_REGISTERED = 2,     /* anonymous mmap, 4 KB pages, cudaHostRegister (what IBP_STORE_SHARED segments get)        */
    IBP_MEM_THP_REGISTERED = 3,        /* the same with madvise(MADV_HUGEPAGE) before the first touch                              */
    IBP_MEM_HUGETLB_2M_REGISTERED = 4  /* mmap(MAP_HUGETLB, 2 MB pages), cudaHostRegister                                          */
};
ibp_status ibp_measure_random_read_kind(int device, size_t footprint_bytes, uint32_t span_bytes, int memory_kind, int reps,
                                        double* spans_per_s, double* gbps);

/* -- Mask-quality tools: the paper's preprocessing counters exposed, so that Mask/Bitval can be
 * built for any threshold from one counting pass (tau sweep), from a sample of the rows, evaluated
 * under any chunk size (Fig. 13), and per cluster of a bit-similarity k-means.  All arrays named
 * *_dev live on the current device; calls are asynchronous on the stream unless stated.  Everything is integer work and
 * agrees exactly with oracle/mask_tools.py.                                                                          */
enum { IBP_GROUP_MAP = 2 }; /* group(id) = row_group_dev[id]: an explicit row -> group map (clusters)               */

typedef struct {
    uint32_t struct_size;          /* = sizeof(ibp_table_desc)                                                       */
    uint32_t row_bytes;            /* multiple of 4                                                                  */
    uint64_t n_rows;
    uint32_t group_kind;           /* IBP_GROUP_BLOCKED, IBP_GROUP_STRIDED or IBP_GROUP_MAP                          */
    uint32_t group_param;          /* G or S; ignored for MAP                                                        */
    uint64_t n_groups;             /* MAP: number of groups; BLOCKED/STRIDED: 0 or the derived count                 */
    const uint32_t* row_group_dev; /* MAP: n_rows entries, each < n_groups; else NULL                                */
} ibp_table_desc;

/* Number of groups the descriptor implies (ceil(n_rows/G), min(S, n_rows), or n_groups).                            */
ibp_status ibp_table_groups(const ibp_table_desc* t, uint64_t* n_groups);

/* P:229 "for each set bit in each input tensor, we increment the corresponding counter".
 * counts_dev[g*8*row_bytes + p] += number of listed rows of group g whose bit p is set; group_n_dev[g] += rows listed.
 * Rows listed: sample_ids_dev[0..n_sample) (repeats count twice; consecutive ids of one group are cheapest), or every
 * row when sample_ids_dev is NULL.  Both outputs are ACCUMULATED into: the caller zeroes them (cudaMemsetAsync) first. */
ibp_status ibp_bit_counts_device(const void* rows_dev, const ibp_table_desc* t, const int64_t* sample_ids_dev,
                                 int64_t n_sample, uint32_t* counts_dev, uint32_t* group_n_dev, void* cuda_stream);

/* P:231 with reading R2: T = ceil(tau N_g); Mask bit = 1 and Bitval bit = 1 where count >= T; Mask = 1, Bitval = 0 where
 * count <= N_g - T; else both 0.  A group with N_g = 0 gets Mask = 0.  mask_dev / bitval_dev: n_groups x row_bytes each;
 * kbits_dev (may be NULL): popcount(~Mask) per group.  INVALID_ARG unless 1/2 < tau <= 1.                           */
ibp_status ibp_masks_from_counts_device(const uint32_t* counts_dev, const uint32_t* group_n_dev, uint64_t n_groups,
                                        uint32_t row_bytes, uint32_t tau_num, uint32_t tau_den, void* mask_dev,
                                        void* bitval_dev, uint32_t* kbits_dev, void* cuda_stream);

/* getCompressSize (Fig. 3 lines 1-19 = P:243-271) of every row under its group's Mask/Bitval with chunks of chunk_bytes
 * in {1, 2, 4, 8} (row_bytes must be a multiple): a chunk participates iff (chunk AND Mask) == Bitval; bitsSaved = sum of
 * popcount(Mask) over participating chunks; bytesSaved = floor((bitsSaved - row_bytes/chunk_bytes)/8); <= 0 -> the row
 * stays raw.  sizes_dev (may be NULL): stored bytes per row.  totals_dev[0] += sum of the sizes, totals_dev[1] +=
 * rows kept raw (caller zeroes).                                                                                    */
ibp_status ibp_compressed_size_device(const void* rows_dev, const ibp_table_desc* t, const void* mask_dev,
                                      const void* bitval_dev, uint32_t chunk_bytes, uint32_t* sizes_dev,
                                      uint64_t* totals_dev, void* cuda_stream);

/* One counting pass, then every (tau, chunk size) pair: total_bytes_host[i*n_cs + j] and raw_rows_host[i*n_cs + j] for
 * taus_host[2i] / taus_host[2i+1] and chunk_bytes_host[j].  Masks come from the listed sample (NULL = all rows), sizes are
 * evaluated on ALL rows.  Synchronous.                                                                  */
ibp_status ibp_mask_sweep_device(const void* rows_dev, const ibp_table_desc* t, const int64_t* sample_ids_dev,
                                 int64_t n_sample, const uint32_t* taus_host, uint32_t n_tau,
                                 const uint32_t* chunk_bytes_host, uint32_t n_cs, uint64_t* total_bytes_host,
                                 uint64_t* raw_rows_host, void* cuda_stream);

/* Bit-similarity k-means (reading R25 in DESIGN.md): Lloyd iterations with the Hamming distance between a row and
 * a centroid bit vector; a centroid bit is the strict majority of its cluster's rows (tie -> 0); assignment ties go to
 * the lowest cluster index; an empty cluster keeps its centroid.  Initial centroids = rows init_ids_dev[0..k).
 * assign_dev: n_rows entries, the assignment of the LAST iteration; centroids_dev: k x row_bytes, after the last update;
 * cost_dev (may be NULL): iters entries, summed distance of every row to its assigned centroid in that iteration.
 * row_bytes <= 4096.  Allocates workspaces on the stream (stream-ordered).                                          */
ibp_status ibp_kmeans_bits_device(const void* rows_dev, uint64_t n_rows, uint32_t row_bytes, uint32_t k,
                                  const int64_t* init_ids_dev, uint32_t iters, uint32_t* assign_dev, void* centroids_dev,
                                  uint64_t* cost_dev, void* cuda_stream);

/* Rows ordered by group: a counting sort of the row ids by row_group_dev (each < n_groups).  order_dev[0..n_rows) becomes a
 * permutation of the row ids in which the rows of group 0 come first, then group 1, ...; the order inside a group is
 * unspecified.  group_start_dev (may be NULL): n_groups + 1 offsets into order_dev.  Use: reorder a table so that the clusters
 * of ibp_kmeans_bits_device become runs of consecutive rows, then build it with blocked groups -- clustered compression
 * with this library's positional groups; ids are mapped through the inverse permutation by the caller.        */
ibp_status ibp_order_by_group_device(const uint32_t* row_group_dev, uint64_t n_rows, uint32_t n_groups, int64_t* order_dev,
                                     uint32_t* group_start_dev, void* cuda_stream);

#ifdef __cplusplus
}
#endif
#endif /* IBP_H */
