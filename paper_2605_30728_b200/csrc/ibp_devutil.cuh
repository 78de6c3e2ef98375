// ibp_devutil.cuh -- small device/host helpers shared by the CUDA translation units of libibp.so.
#pragma once
#include <cuda_runtime.h>

#include <cstdint>

#include "ibp_internal.h"

#define IBP_CUDA(call)                                                                              \
    do {                                                                                            \
        cudaError_t e_ = (call);                                                                    \
        if (e_ != cudaSuccess) {                                                                    \
            ibp_set_error("%s failed: %s (%s:%d)", #call, cudaGetErrorString(e_), __FILE__, __LINE__); \
            (void)cudaGetLastError();                                                               \
            return IBP_ERR_CUDA;                                                                    \
        }                                                                                           \
    } while (0)

// SMs of the current device (grids are sized from this, never from a literal).  Cached per device.
static inline int ibp_sm_count_current() {
    static int cached[64] = {};
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= 64) { (void)cudaGetLastError(); return 148; }
    int n = cached[dev];
    if (n == 0) {
        if (cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || n <= 0) { (void)cudaGetLastError(); return 148; }
        cached[dev] = n;   // benign race: every thread writes the same value
    }
    return n;
}

// Opt a kernel in to the device's largest dynamic shared-memory size ONCE per (kernel, device).  The attribute is per function
// and per device for the whole process, so a per-thread "largest size seen" cache would let a second host thread lower it under
// the first one's feet; raising it to the device maximum once is order-independent.  `done` is the caller's per-kernel bitmask
// (one static per template instantiation), bit d = device d is set up.
template <typename Kern>
static inline cudaError_t ibp_optin_max_smem(Kern kern, unsigned long long* done) {
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    const unsigned long long bit = 1ull << (dev & 63);
    if (__atomic_load_n(done, __ATOMIC_ACQUIRE) & bit) return cudaSuccess;
    int optin = 0;
    e = cudaDeviceGetAttribute(&optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev);
    if (e != cudaSuccess) return e;
    cudaFuncAttributes fa;
    e = cudaFuncGetAttributes(&fa, kern);
    if (e != cudaSuccess) return e;
    e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, optin - (int)fa.sharedSizeBytes);
    if (e != cudaSuccess) return e;
    __atomic_fetch_or(done, bit, __ATOMIC_RELEASE);
    return cudaSuccess;
}

__device__ __forceinline__ uint32_t warp_inclusive_scan(uint32_t v, int lane) {
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        uint32_t t = __shfl_up_sync(0xFFFFFFFFu, v, d);
        if (lane >= d) v += t;
    }
    return v;
}

template <int W> struct VecIO;
template <> struct VecIO<1> {
    static __device__ __forceinline__ void ld(const uint32_t* p, uint32_t* v) { v[0] = __ldg(p); }
    static __device__ __forceinline__ void st(uint8_t* p, const uint32_t* v) { asm volatile("st.global.cs.b32 [%0], %1;" ::"l"(p), "r"(v[0]) : "memory"); }
    static __device__ __forceinline__ void st_keep(uint8_t* p, const uint32_t* v) { *(uint32_t*)p = v[0]; }
};
template <> struct VecIO<2> {
    static __device__ __forceinline__ void ld(const uint32_t* p, uint32_t* v) { uint2 t = __ldg((const uint2*)p); v[0] = t.x; v[1] = t.y; }
    static __device__ __forceinline__ void st(uint8_t* p, const uint32_t* v) { asm volatile("st.global.cs.v2.b32 [%0], {%1,%2};" ::"l"(p), "r"(v[0]), "r"(v[1]) : "memory"); }
    static __device__ __forceinline__ void st_keep(uint8_t* p, const uint32_t* v) { *(uint2*)p = make_uint2(v[0], v[1]); }
};
template <> struct VecIO<4> {
    static __device__ __forceinline__ void ld(const uint32_t* p, uint32_t* v) { uint4 t = __ldg((const uint4*)p); v[0] = t.x; v[1] = t.y; v[2] = t.z; v[3] = t.w; }
    static __device__ __forceinline__ void st(uint8_t* p, const uint32_t* v) { asm volatile("st.global.cs.v4.b32 [%0], {%1,%2,%3,%4};" ::"l"(p), "r"(v[0]), "r"(v[1]), "r"(v[2]), "r"(v[3]) : "memory"); }
    static __device__ __forceinline__ void st_keep(uint8_t* p, const uint32_t* v) { *(uint4*)p = make_uint4(v[0], v[1], v[2], v[3]); }
};

__device__ __forceinline__ uint64_t group_of_u(uint32_t group_param, uint32_t group_shift, uint64_t id) {
    return group_shift != 0xFFFFFFFFu ? (id >> group_shift) : (id / group_param);
}


// ---- compressed GPU cache map: open addressing, linear probing, slots of {key = id + 1, value}
#define IBP_CACHE_MISS_DEV 0xFFFFFFFFFFFFFFFFull
__device__ __forceinline__ uint32_t ibp_cache_hash(uint64_t id, uint32_t mask) {
    return (uint32_t)((id * 0x9E3779B97F4A7C15ull) >> 32) & mask;
}
__device__ __forceinline__ uint64_t ibp_cache_find(const uint64_t* __restrict__ map, uint32_t mask, uint64_t id) {
    uint32_t slot = ibp_cache_hash(id, mask);
    for (;;) {
        const ulonglong2 e = __ldg((const ulonglong2*)map + slot);
        if (e.x == id + 1) return e.y;
        if (e.x == 0ull) return IBP_CACHE_MISS_DEV;
        slot = (slot + 1) & mask;
    }
}
