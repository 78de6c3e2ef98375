// ibp_analysis.cu -- mask-quality tools of libibp.so (sm_100a): SURVEY 8(f) NEXT #4.
//
//   ibp_count_kernel      P:229  per-bit counters of the listed rows.  A warp takes a run of list positions; lane l owns the
//                                words l, l+32, ... of the row; the 32 counters of a word are BIT-SLICED over NP planes held
//                                in registers (plane j = bit j of the 32 running counts), a row enters by a ripple add of
//                                2 logic ops per plane; planes are unpacked and added to the global counters with atomicAdd
//                                only when the run's group changes or the run ends.
//   ibp_masks_kernel      P:231  Mask/Bitval from the counters for T = ceil(tau N_g): re-run per tau of the sweep.
//   ibp_csize_kernel      Fig. 3 lines 1-19  getCompressSize per row for chunk sizes 1/2/4/8 bytes: warp per row,
//                                lane per 8-byte unit, byte-wise match flags by SIMD-in-register tests, warp sum.
//   ibp_assign_kernel     P:542  k-means assignment with the Hamming distance: thread per row, the row's words transposed in
//                                shared memory (conflict-free), centroid words read warp-uniformly, four centroids per pass.
//   ibp_majority_kernel          centroid update: bit = strict majority of the cluster's counters (counted by
//                                ibp_count_kernel over the rows ordered by cluster: counting sort in three small kernels).
// Integer arithmetic only; results do not depend on the launch shape (sums of integers).  Checked against
// oracle/mask_tools.py in tests/test_gpu_mask_tools.py.
#include <algorithm>
#include <cstdio>
#include <cstring>
#include <vector>

#include "ibp_devutil.cuh"

namespace {

struct TableDev {
    const uint32_t* rows;
    uint64_t n_rows, n_groups;
    uint32_t nw;                 // words per row
    uint32_t kind, param;
    const uint32_t* row_group;   // MAP
    const int64_t* list;         // listed rows, or nullptr = all
    uint64_t n_list;             // list length (virtual length for "all")
    uint64_t q_strided;          // STRIDED without a list: ceil(n_rows / S) (group-major virtual order)
};

__device__ __forceinline__ uint64_t table_group(const TableDev& T, uint64_t row) {
    return T.kind == IBP_GROUP_MAP ? (uint64_t)__ldg(T.row_group + row) : T.kind == IBP_GROUP_BLOCKED ? row / T.param : row % T.param;
}
// list position -> row id (or ~0 when the virtual position holds no row)
__device__ __forceinline__ uint64_t table_item(const TableDev& T, uint64_t pos) {
    if (T.list) return (uint64_t)__ldg(T.list + pos);
    if (T.kind == IBP_GROUP_STRIDED) {          // walk a tile's rows consecutively: pos = g*Q + j -> row j*S + g
        const uint64_t g = pos / T.q_strided, j = pos - g * T.q_strided, row = j * T.param + g;
        return row < T.n_rows ? row : ~0ull;
    }
    return pos;
}

constexpr int COUNT_RUN = 96;   // list positions per warp run
constexpr int COUNT_NP = 7;     // planes: a run adds at most 96 < 2^7 rows to a counter before it is flushed

template <int NP>
__device__ __forceinline__ void flush_planes(uint32_t* pl, uint32_t* dst /* 32 counters of this word */) {
    uint32_t any = 0;
#pragma unroll
    for (int p = 0; p < NP; ++p) any |= pl[p];
    while (any) {
        const int b = __ffs(any) - 1;
        any &= any - 1;
        uint32_t c = 0;
#pragma unroll
        for (int p = 0; p < NP; ++p) c |= ((pl[p] >> b) & 1u) << p;
        atomicAdd(dst + b, c);
    }
#pragma unroll
    for (int p = 0; p < NP; ++p) pl[p] = 0;
}

__global__ void __launch_bounds__(256) ibp_count_kernel(const TableDev T, uint32_t* __restrict__ counts, uint32_t* __restrict__ group_n) {
    const int lane = threadIdx.x & 31, wpc = blockDim.x >> 5;
    const uint64_t n_runs = (T.n_list + COUNT_RUN - 1) / COUNT_RUN;
    const uint32_t n_pass = (T.nw + 31) / 32;
    const uint64_t nbits = 32ull * T.nw;
    for (uint64_t run = (uint64_t)blockIdx.x * wpc + (threadIdx.x >> 5); run < n_runs; run += (uint64_t)gridDim.x * wpc) {
        const uint64_t p0 = run * COUNT_RUN, p1 = min(T.n_list, p0 + COUNT_RUN);
        for (uint32_t pass = 0; pass < n_pass; ++pass) {
            const uint32_t w = pass * 32u + lane;
            const bool active = w < T.nw;
            uint32_t pl[COUNT_NP];
#pragma unroll
            for (int p = 0; p < COUNT_NP; ++p) pl[p] = 0;
            uint64_t cur_g = ~0ull;
            uint32_t cur_n = 0;
            for (uint64_t pos = p0; pos < p1; ++pos) {
                const uint64_t row = table_item(T, pos);
                if (row == ~0ull) continue;
                const uint64_t g = table_group(T, row);
                if (g != cur_g) {
                    if (cur_g != ~0ull) {
                        if (active) flush_planes<COUNT_NP>(pl, counts + cur_g * nbits + 32ull * w);
                        if (pass == 0 && lane == 0) atomicAdd(group_n + cur_g, cur_n);
                    }
                    cur_g = g; cur_n = 0;
                }
                cur_n += 1;
                if (active) {
                    uint32_t c = __ldg(T.rows + row * T.nw + w);
#pragma unroll
                    for (int p = 0; p < COUNT_NP; ++p) { const uint32_t t = pl[p]; pl[p] = t ^ c; c &= t; }
                }
            }
            if (cur_g != ~0ull) {
                if (active) flush_planes<COUNT_NP>(pl, counts + cur_g * nbits + 32ull * w);
                if (pass == 0 && lane == 0) atomicAdd(group_n + cur_g, cur_n);
            }
        }
    }
}

// one thread per (group, word)
__global__ void __launch_bounds__(256) ibp_masks_kernel(const uint32_t* __restrict__ counts, const uint32_t* __restrict__ group_n,
                                                        uint64_t n_groups, uint32_t nw, uint32_t tau_num, uint32_t tau_den,
                                                        uint32_t* __restrict__ mask, uint32_t* __restrict__ bitval, uint32_t* __restrict__ kbits) {
    const uint64_t cell = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (cell >= n_groups * nw) return;
    const uint64_t g = cell / nw;
    const uint64_t N = group_n[g];
    uint32_t mk = 0, bv = 0;
    if (N) {
        const uint64_t T = (N * tau_num + tau_den - 1) / tau_den;
        const uint32_t* c = counts + cell * 32ull;
#pragma unroll 8
        for (int b = 0; b < 32; ++b) {
            const uint64_t v = c[b];
            const uint32_t ge = v >= T, le = v <= N - T;
            mk |= (ge | le) << b;
            bv |= ge << b;
        }
    }
    mask[cell] = mk;
    bitval[cell] = bv;
    if (kbits) atomicAdd(kbits + g, (uint32_t)__popc(~mk));
}

// ------------------------------------------------------------------------------------------------ getCompressSize
template <int CS>
__device__ __forceinline__ uint32_t saved_bits_unit(uint32_t dlo, uint32_t mlo, uint32_t dhi, uint32_t mhi) {
    uint32_t s = 0;
    if (CS == 8) {
        if ((dlo | dhi) == 0) s = __popc(mlo) + __popc(mhi);
    } else if (CS == 4) {
        if (dlo == 0) s += __popc(mlo);
        if (dhi == 0) s += __popc(mhi);
    } else if (CS == 2) {
#pragma unroll
        for (int h = 0; h < 2; ++h) {
            const uint32_t sel = 0xFFFFu << (16 * h);
            if ((dlo & sel) == 0) s += __popc(mlo & sel);
            if ((dhi & sel) == 0) s += __popc(mhi & sel);
        }
    } else {
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const uint32_t sel = 0xFFu << (8 * j);
            if ((dlo & sel) == 0) s += __popc(mlo & sel);
            if ((dhi & sel) == 0) s += __popc(mhi & sel);
        }
    }
    return s;
}

// One warp per row (grid-stride).  Lane l owns the 8-byte units l, l+32, ...  A missing high word (row_bytes % 8 == 4, CS <= 4)
// enters as d = 1, m = 0: it never matches and saves nothing.
template <int CS>
__global__ void __launch_bounds__(256) ibp_csize_kernel(const TableDev T, const uint32_t* __restrict__ mask, const uint32_t* __restrict__ bitval,
                                                        uint32_t* __restrict__ sizes, unsigned long long* __restrict__ totals) {
    const int lane = threadIdx.x & 31, wpc = blockDim.x >> 5;
    const uint32_t row_bytes = 4u * T.nw, n_units = (T.nw + 1) / 2, n_chunks = row_bytes / CS;
    unsigned long long sum_sizes = 0, sum_raw = 0;
    for (uint64_t row = (uint64_t)blockIdx.x * wpc + (threadIdx.x >> 5); row < T.n_rows; row += (uint64_t)gridDim.x * wpc) {
        const uint64_t g = table_group(T, row);
        const uint32_t* x = T.rows + row * T.nw;
        const uint32_t* m = mask + g * T.nw;
        const uint32_t* b = bitval + g * T.nw;
        uint32_t saved = 0;
        for (uint32_t u = lane; u < n_units; u += 32) {
            const uint32_t w = 2 * u;
            uint32_t mlo = __ldg(m + w), dlo = (__ldg(x + w) & mlo) ^ __ldg(b + w), mhi = 0, dhi = 1;
            if (w + 1 < T.nw) { mhi = __ldg(m + w + 1); dhi = (__ldg(x + w + 1) & mhi) ^ __ldg(b + w + 1); }
            saved += saved_bits_unit<CS>(dlo, mlo, dhi, mhi);
        }
#pragma unroll
        for (int d = 16; d; d >>= 1) saved += __shfl_xor_sync(0xFFFFFFFFu, saved, d);
        const int diff = (int)saved - (int)n_chunks;                       // Fig. 3 line 13: bitsSaved - participation bits
        const uint32_t bytes_saved = diff > 0 ? (uint32_t)diff / 8u : 0u;  // floor (R9); <= 0 -> raw
        const uint32_t size = bytes_saved ? row_bytes - bytes_saved : row_bytes;
        if (lane == 0) {
            if (sizes) sizes[row] = size;
            sum_sizes += size;
            sum_raw += bytes_saved ? 0 : 1;
        }
    }
    if (lane == 0 && (sum_sizes | sum_raw)) {
        atomicAdd(totals, sum_sizes);
        atomicAdd(totals + 1, sum_raw);
    }
}

// ------------------------------------------------------------------------------------------------ k-means (R25)
// Thread per row.  smem: the CTA's rows, word-major (xs[w * blockDim.x + tid]).  Centroid words are read warp-uniformly.
__global__ void ibp_assign_kernel(const uint32_t* __restrict__ rows, uint64_t n_rows, uint32_t nw, const uint32_t* __restrict__ cent, uint32_t k,
                                  uint32_t* __restrict__ assign, unsigned long long* __restrict__ cost) {
    extern __shared__ uint32_t xs[];
    const uint32_t nt = blockDim.x, tid = threadIdx.x;
    const uint64_t row0 = (uint64_t)blockIdx.x * nt;
    const uint32_t rows_here = (uint32_t)min((uint64_t)nt, n_rows - row0);
    // coalesced load of rows_here x nw words, transposed into smem
    for (uint32_t i = tid; i < rows_here * nw; i += nt) {
        const uint32_t r = i / nw, w = i - r * nw;
        xs[w * nt + r] = __ldg(rows + (row0 + r) * nw + w);
    }
    __syncthreads();
    uint32_t best = 0xFFFFFFFFu, best_c = 0;
    if (tid < rows_here) {
        uint32_t c = 0;
        for (; c + 4 <= k; c += 4) {
            const uint32_t* c0 = cent + (uint64_t)c * nw;
            uint32_t d0 = 0, d1 = 0, d2 = 0, d3 = 0;
            for (uint32_t w = 0; w < nw; ++w) {
                const uint32_t x = xs[w * nt + tid];
                d0 += __popc(x ^ __ldg(c0 + w));
                d1 += __popc(x ^ __ldg(c0 + nw + w));
                d2 += __popc(x ^ __ldg(c0 + 2 * nw + w));
                d3 += __popc(x ^ __ldg(c0 + 3 * nw + w));
            }
            if (d0 < best) { best = d0; best_c = c; }            // strict <: the lowest index wins a tie
            if (d1 < best) { best = d1; best_c = c + 1; }
            if (d2 < best) { best = d2; best_c = c + 2; }
            if (d3 < best) { best = d3; best_c = c + 3; }
        }
        for (; c < k; ++c) {
            const uint32_t* c0 = cent + (uint64_t)c * nw;
            uint32_t d0 = 0;
            for (uint32_t w = 0; w < nw; ++w) d0 += __popc(xs[w * nt + tid] ^ __ldg(c0 + w));
            if (d0 < best) { best = d0; best_c = c; }
        }
        assign[row0 + tid] = best_c;
    }
    if (cost) {
        unsigned long long v = tid < rows_here ? best : 0ull;
#pragma unroll
        for (int d = 16; d; d >>= 1) v += __shfl_xor_sync(0xFFFFFFFFu, v, d);
        if ((tid & 31) == 0 && v) atomicAdd(cost, v);
    }
}

__global__ void ibp_gather_rows_kernel(const uint32_t* __restrict__ rows, uint32_t nw, const int64_t* __restrict__ ids, uint32_t k, uint32_t* __restrict__ out) {
    const uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= (uint64_t)k * nw) return;
    const uint32_t c = (uint32_t)(i / nw), w = (uint32_t)(i - (uint64_t)c * nw);
    out[i] = __ldg(rows + (uint64_t)__ldg(ids + c) * nw + w);
}

// counting sort of the rows by cluster: histogram, exclusive scan (one CTA), scatter (order inside a cluster is arbitrary:
// only sums over a cluster are taken afterwards)
__global__ void ibp_cluster_hist(const uint32_t* __restrict__ assign, uint64_t n, uint32_t* __restrict__ hist) {
    for (uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (uint64_t)gridDim.x * blockDim.x) atomicAdd(hist + assign[i], 1u);
}
__global__ void __launch_bounds__(1024) ibp_cluster_scan(const uint32_t* __restrict__ hist, uint32_t k, uint32_t* __restrict__ cursor) {
    __shared__ uint32_t part[1024];
    const uint32_t per = (k + 1023) / 1024, lo = threadIdx.x * per, hi = min(k, lo + per);
    uint32_t s = 0;
    for (uint32_t i = lo; i < hi; ++i) s += hist[i];
    part[threadIdx.x] = s;
    __syncthreads();
    if (threadIdx.x == 0) { uint32_t run = 0; for (int i = 0; i < 1024; ++i) { const uint32_t t = part[i]; part[i] = run; run += t; } }
    __syncthreads();
    uint32_t run = part[threadIdx.x];
    for (uint32_t i = lo; i < hi; ++i) { cursor[i] = run; run += hist[i]; }
}
__global__ void ibp_cluster_scatter(const uint32_t* __restrict__ assign, uint64_t n, uint32_t* __restrict__ cursor, int64_t* __restrict__ order) {
    for (uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (uint64_t)gridDim.x * blockDim.x)
        order[atomicAdd(cursor + assign[i], 1u)] = (int64_t)i;
}
// centroid bit = 1 iff 2*count > n (strict majority; tie -> 0); empty cluster: unchanged.  One thread per (cluster, word).
__global__ void ibp_majority_kernel(const uint32_t* __restrict__ counts, const uint32_t* __restrict__ group_n, uint32_t k, uint32_t nw, uint32_t* __restrict__ cent) {
    const uint64_t cell = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (cell >= (uint64_t)k * nw) return;
    const uint32_t n = group_n[cell / nw];
    if (!n) return;
    const uint32_t* c = counts + cell * 32ull;
    uint32_t v = 0;
#pragma unroll 8
    for (int b = 0; b < 32; ++b) v |= (uint32_t)(2ull * c[b] > n) << b;
    cent[cell] = v;
}

}  // namespace

// ------------------------------------------------------------------------------------------------ C ABI
static ibp_status check_table(const ibp_table_desc* t, const void* rows_dev, const char* who, TableDev* out) {
    if (!t || !rows_dev) { ibp_set_error("%s: null argument", who); return IBP_ERR_INVALID_ARG; }
    if (t->struct_size != sizeof(ibp_table_desc)) { ibp_set_error("%s: ibp_table_desc.struct_size mismatch", who); return IBP_ERR_INVALID_ARG; }
    if (t->row_bytes == 0 || t->row_bytes % 4 || t->row_bytes > 65536) { ibp_set_error("%s: row_bytes must be a multiple of 4 in 4..65536", who); return IBP_ERR_INVALID_ARG; }
    if (t->n_rows == 0) { ibp_set_error("%s: n_rows == 0", who); return IBP_ERR_INVALID_ARG; }
    uint64_t ng = 0;
    if (t->group_kind == IBP_GROUP_MAP) {
        if (!t->row_group_dev || t->n_groups == 0) { ibp_set_error("%s: IBP_GROUP_MAP needs row_group_dev and n_groups", who); return IBP_ERR_INVALID_ARG; }
        ng = t->n_groups;
    } else if (t->group_kind == IBP_GROUP_BLOCKED || t->group_kind == IBP_GROUP_STRIDED) {
        if (t->group_param == 0) { ibp_set_error("%s: group_param == 0", who); return IBP_ERR_INVALID_ARG; }
        ng = t->group_kind == IBP_GROUP_BLOCKED ? (t->n_rows + t->group_param - 1) / t->group_param : std::min<uint64_t>(t->group_param, t->n_rows);
        if (t->n_groups && t->n_groups != ng) { ibp_set_error("%s: n_groups does not match the group rule", who); return IBP_ERR_INVALID_ARG; }
    } else { ibp_set_error("%s: bad group_kind", who); return IBP_ERR_INVALID_ARG; }
    if (out) {
        TableDev T{};
        T.rows = (const uint32_t*)rows_dev; T.n_rows = t->n_rows; T.n_groups = ng; T.nw = t->row_bytes / 4;
        T.kind = t->group_kind; T.param = t->group_param ? t->group_param : 1; T.row_group = t->row_group_dev;
        T.list = nullptr; T.n_list = t->n_rows; T.q_strided = 0;
        *out = T;
    }
    return IBP_OK;
}

static int analysis_grid(uint64_t work_warps) {
    int dev = 0, sms = 148;
    if (cudaGetDevice(&dev) == cudaSuccess) (void)cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    (void)cudaGetLastError();
    const uint64_t ctas = (work_warps + 7) / 8;
    return (int)std::max<uint64_t>(1, std::min<uint64_t>(ctas, (uint64_t)sms * 8));
}

extern "C" ibp_status ibp_table_groups(const ibp_table_desc* t, uint64_t* n_groups) {
    TableDev T;
    if (!n_groups) { ibp_set_error("ibp_table_groups: null argument"); return IBP_ERR_INVALID_ARG; }
    ibp_status s = check_table(t, (const void*)1, "ibp_table_groups", &T);
    if (s != IBP_OK) return s;
    *n_groups = T.n_groups;
    return IBP_OK;
}

static ibp_status launch_counts(TableDev T, const int64_t* sample_ids_dev, int64_t n_sample, uint32_t* counts_dev, uint32_t* group_n_dev, cudaStream_t st) {
    if (sample_ids_dev) { T.list = sample_ids_dev; T.n_list = (uint64_t)n_sample; }
    else if (T.kind == IBP_GROUP_STRIDED) { T.q_strided = (T.n_rows + T.param - 1) / T.param; T.n_list = T.q_strided * std::min<uint64_t>(T.param, T.n_rows); }
    if (T.n_list == 0) return IBP_OK;
    const uint64_t n_runs = (T.n_list + COUNT_RUN - 1) / COUNT_RUN;
    ibp_count_kernel<<<analysis_grid(n_runs), 256, 0, st>>>(T, counts_dev, group_n_dev);
    IBP_CUDA(cudaGetLastError());
    return IBP_OK;
}

extern "C" ibp_status ibp_bit_counts_device(const void* rows_dev, const ibp_table_desc* t, const int64_t* sample_ids_dev, int64_t n_sample,
                                            uint32_t* counts_dev, uint32_t* group_n_dev, void* cuda_stream) {
    TableDev T;
    ibp_status s = check_table(t, rows_dev, "ibp_bit_counts_device", &T);
    if (s != IBP_OK) return s;
    if (!counts_dev || !group_n_dev) { ibp_set_error("ibp_bit_counts_device: null output"); return IBP_ERR_INVALID_ARG; }
    if (sample_ids_dev && n_sample < 0) { ibp_set_error("ibp_bit_counts_device: n_sample < 0"); return IBP_ERR_INVALID_ARG; }
    return launch_counts(T, sample_ids_dev, n_sample, counts_dev, group_n_dev, (cudaStream_t)cuda_stream);
}

static ibp_status check_tau(uint32_t num, uint32_t den, const char* who) {
    if (den == 0 || num > den || 2ull * num <= den) { ibp_set_error("%s: tau = %u/%u is outside (1/2, 1]", who, num, den); return IBP_ERR_INVALID_ARG; }
    return IBP_OK;
}

extern "C" ibp_status ibp_masks_from_counts_device(const uint32_t* counts_dev, const uint32_t* group_n_dev, uint64_t n_groups, uint32_t row_bytes,
                                                   uint32_t tau_num, uint32_t tau_den, void* mask_dev, void* bitval_dev, uint32_t* kbits_dev,
                                                   void* cuda_stream) {
    if (!counts_dev || !group_n_dev || !mask_dev || !bitval_dev || n_groups == 0 || row_bytes == 0 || row_bytes % 4) {
        ibp_set_error("ibp_masks_from_counts_device: bad argument"); return IBP_ERR_INVALID_ARG;
    }
    ibp_status s = check_tau(tau_num, tau_den, "ibp_masks_from_counts_device");
    if (s != IBP_OK) return s;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const uint32_t nw = row_bytes / 4;
    if (kbits_dev) IBP_CUDA(cudaMemsetAsync(kbits_dev, 0, n_groups * 4, st));
    const uint64_t cells = n_groups * nw;
    ibp_masks_kernel<<<(unsigned)((cells + 255) / 256), 256, 0, st>>>(counts_dev, group_n_dev, n_groups, nw, tau_num, tau_den, (uint32_t*)mask_dev,
                                                                       (uint32_t*)bitval_dev, kbits_dev);
    IBP_CUDA(cudaGetLastError());
    return IBP_OK;
}

static ibp_status launch_csize(const TableDev& T, const void* mask_dev, const void* bitval_dev, uint32_t cs, uint32_t* sizes_dev, uint64_t* totals_dev,
                               cudaStream_t st) {
    const int grid = analysis_grid(T.n_rows);
    const uint32_t* m = (const uint32_t*)mask_dev; const uint32_t* b = (const uint32_t*)bitval_dev;
    unsigned long long* tot = (unsigned long long*)totals_dev;
    switch (cs) {
        case 1: ibp_csize_kernel<1><<<grid, 256, 0, st>>>(T, m, b, sizes_dev, tot); break;
        case 2: ibp_csize_kernel<2><<<grid, 256, 0, st>>>(T, m, b, sizes_dev, tot); break;
        case 4: ibp_csize_kernel<4><<<grid, 256, 0, st>>>(T, m, b, sizes_dev, tot); break;
        default: ibp_csize_kernel<8><<<grid, 256, 0, st>>>(T, m, b, sizes_dev, tot); break;
    }
    IBP_CUDA(cudaGetLastError());
    return IBP_OK;
}

static ibp_status check_cs(uint32_t cs, uint32_t row_bytes, const char* who) {
    if ((cs != 1 && cs != 2 && cs != 4 && cs != 8) || row_bytes % cs) { ibp_set_error("%s: chunk_bytes must be 1, 2, 4 or 8 and divide row_bytes", who); return IBP_ERR_INVALID_ARG; }
    return IBP_OK;
}

extern "C" ibp_status ibp_compressed_size_device(const void* rows_dev, const ibp_table_desc* t, const void* mask_dev, const void* bitval_dev,
                                                 uint32_t chunk_bytes, uint32_t* sizes_dev, uint64_t* totals_dev, void* cuda_stream) {
    TableDev T;
    ibp_status s = check_table(t, rows_dev, "ibp_compressed_size_device", &T);
    if (s != IBP_OK) return s;
    if (!mask_dev || !bitval_dev || !totals_dev) { ibp_set_error("ibp_compressed_size_device: null argument"); return IBP_ERR_INVALID_ARG; }
    s = check_cs(chunk_bytes, t->row_bytes, "ibp_compressed_size_device");
    if (s != IBP_OK) return s;
    return launch_csize(T, mask_dev, bitval_dev, chunk_bytes, sizes_dev, totals_dev, (cudaStream_t)cuda_stream);
}

extern "C" ibp_status ibp_mask_sweep_device(const void* rows_dev, const ibp_table_desc* t, const int64_t* sample_ids_dev, int64_t n_sample,
                                            const uint32_t* taus_host, uint32_t n_tau, const uint32_t* chunk_bytes_host, uint32_t n_cs,
                                            uint64_t* total_bytes_host, uint64_t* raw_rows_host, void* cuda_stream) {
    TableDev T;
    ibp_status s = check_table(t, rows_dev, "ibp_mask_sweep_device", &T);
    if (s != IBP_OK) return s;
    if (!taus_host || !chunk_bytes_host || !total_bytes_host || !raw_rows_host || n_tau == 0 || n_cs == 0) {
        ibp_set_error("ibp_mask_sweep_device: null or empty argument"); return IBP_ERR_INVALID_ARG;
    }
    for (uint32_t i = 0; i < n_tau; ++i) if ((s = check_tau(taus_host[2 * i], taus_host[2 * i + 1], "ibp_mask_sweep_device")) != IBP_OK) return s;
    for (uint32_t j = 0; j < n_cs; ++j) if ((s = check_cs(chunk_bytes_host[j], t->row_bytes, "ibp_mask_sweep_device")) != IBP_OK) return s;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const uint64_t ng = T.n_groups, meta_bytes = ng * (uint64_t)t->row_bytes, n_cells = (uint64_t)n_tau * n_cs;
    uint32_t *counts = nullptr, *gn = nullptr; uint8_t *mask = nullptr, *bitval = nullptr; uint64_t* totals = nullptr;
    IBP_CUDA(cudaMallocAsync((void**)&counts, ng * 32ull * T.nw * 4, st));
    IBP_CUDA(cudaMallocAsync((void**)&gn, ng * 4, st));
    IBP_CUDA(cudaMallocAsync((void**)&mask, meta_bytes, st));
    IBP_CUDA(cudaMallocAsync((void**)&bitval, meta_bytes, st));
    IBP_CUDA(cudaMallocAsync((void**)&totals, n_cells * 16, st));
    IBP_CUDA(cudaMemsetAsync(counts, 0, ng * 32ull * T.nw * 4, st));
    IBP_CUDA(cudaMemsetAsync(gn, 0, ng * 4, st));
    IBP_CUDA(cudaMemsetAsync(totals, 0, n_cells * 16, st));
    s = launch_counts(T, sample_ids_dev, n_sample, counts, gn, st);                               // one counting pass
    for (uint32_t i = 0; s == IBP_OK && i < n_tau; ++i) {                                         // re-threshold per tau
        s = ibp_masks_from_counts_device(counts, gn, ng, t->row_bytes, taus_host[2 * i], taus_host[2 * i + 1], mask, bitval, nullptr, st);
        for (uint32_t j = 0; s == IBP_OK && j < n_cs; ++j)                                        // sizes of ALL rows per chunk size
            s = launch_csize(T, mask, bitval, chunk_bytes_host[j], nullptr, totals + 2 * ((uint64_t)i * n_cs + j), st);
    }
    std::vector<uint64_t> host(2 * n_cells);
    if (s == IBP_OK) {
        IBP_CUDA(cudaMemcpyAsync(host.data(), totals, n_cells * 16, cudaMemcpyDeviceToHost, st));
        IBP_CUDA(cudaStreamSynchronize(st));
        for (uint64_t c = 0; c < n_cells; ++c) { total_bytes_host[c] = host[2 * c]; raw_rows_host[c] = host[2 * c + 1]; }
    }
    cudaFreeAsync(counts, st); cudaFreeAsync(gn, st); cudaFreeAsync(mask, st); cudaFreeAsync(bitval, st); cudaFreeAsync(totals, st);
    return s;
}

extern "C" ibp_status ibp_kmeans_bits_device(const void* rows_dev, uint64_t n_rows, uint32_t row_bytes, uint32_t k, const int64_t* init_ids_dev,
                                             uint32_t iters, uint32_t* assign_dev, void* centroids_dev, uint64_t* cost_dev, void* cuda_stream) {
    if (!rows_dev || !init_ids_dev || !assign_dev || !centroids_dev || n_rows == 0 || k == 0 || iters == 0) {
        ibp_set_error("ibp_kmeans_bits_device: null or empty argument"); return IBP_ERR_INVALID_ARG;
    }
    if (row_bytes == 0 || row_bytes % 4 || row_bytes > 4096) { ibp_set_error("ibp_kmeans_bits_device: row_bytes must be a multiple of 4 in 4..4096"); return IBP_ERR_INVALID_ARG; }
    if (n_rows > 0xFFFFFFFFull) { ibp_set_error("ibp_kmeans_bits_device: n_rows too large"); return IBP_ERR_INVALID_ARG; }
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const uint32_t nw = row_bytes / 4;
    const uint32_t* rows = (const uint32_t*)rows_dev;
    uint32_t* cent = (uint32_t*)centroids_dev;
    // assignment CTA: as many rows (threads) as fit ~160 KB of shared memory, 32..256
    uint32_t nt = std::min<uint32_t>(256, (160u * 1024u / row_bytes) / 32u * 32u);
    if (nt < 32) nt = 32;
    const size_t smem = (size_t)nt * row_bytes;
    IBP_CUDA(cudaFuncSetAttribute(ibp_assign_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    uint32_t *counts = nullptr, *gn = nullptr, *hist = nullptr, *cursor = nullptr; int64_t* order = nullptr;
    IBP_CUDA(cudaMallocAsync((void**)&counts, (uint64_t)k * 32ull * nw * 4, st));
    IBP_CUDA(cudaMallocAsync((void**)&gn, (uint64_t)k * 4, st));
    IBP_CUDA(cudaMallocAsync((void**)&hist, (uint64_t)k * 4, st));
    IBP_CUDA(cudaMallocAsync((void**)&cursor, (uint64_t)k * 4, st));
    IBP_CUDA(cudaMallocAsync((void**)&order, n_rows * 8, st));
    if (cost_dev) IBP_CUDA(cudaMemsetAsync(cost_dev, 0, (uint64_t)iters * 8, st));
    ibp_gather_rows_kernel<<<(unsigned)(((uint64_t)k * nw + 255) / 256), 256, 0, st>>>(rows, nw, init_ids_dev, k, cent);
    IBP_CUDA(cudaGetLastError());
    TableDev T{};
    T.rows = rows; T.n_rows = n_rows; T.n_groups = k; T.nw = nw; T.kind = IBP_GROUP_MAP; T.param = 1; T.row_group = assign_dev;
    const int grid_n = analysis_grid((n_rows + 31) / 32);
    ibp_status s = IBP_OK;
    for (uint32_t it = 0; it < iters && s == IBP_OK; ++it) {
        ibp_assign_kernel<<<(unsigned)((n_rows + nt - 1) / nt), nt, smem, st>>>(rows, n_rows, nw, cent, k, assign_dev,
                                                                               cost_dev ? (unsigned long long*)cost_dev + it : nullptr);
        IBP_CUDA(cudaGetLastError());
        IBP_CUDA(cudaMemsetAsync(hist, 0, (uint64_t)k * 4, st));
        IBP_CUDA(cudaMemsetAsync(counts, 0, (uint64_t)k * 32ull * nw * 4, st));
        IBP_CUDA(cudaMemsetAsync(gn, 0, (uint64_t)k * 4, st));
        ibp_cluster_hist<<<grid_n, 256, 0, st>>>(assign_dev, n_rows, hist);
        ibp_cluster_scan<<<1, 1024, 0, st>>>(hist, k, cursor);
        ibp_cluster_scatter<<<grid_n, 256, 0, st>>>(assign_dev, n_rows, cursor, order);
        IBP_CUDA(cudaGetLastError());
        s = launch_counts(T, order, (int64_t)n_rows, counts, gn, st);
        if (s != IBP_OK) break;
        ibp_majority_kernel<<<(unsigned)(((uint64_t)k * nw + 255) / 256), 256, 0, st>>>(counts, gn, k, nw, cent);
        IBP_CUDA(cudaGetLastError());
    }
    cudaFreeAsync(counts, st); cudaFreeAsync(gn, st); cudaFreeAsync(hist, st); cudaFreeAsync(cursor, st); cudaFreeAsync(order, st);
    return s;
}
