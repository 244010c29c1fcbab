// common.cuh -- shared device/host helpers of the product kernels (sm_100a).
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>

#include <atomic>
#include <cstdint>
#include <cstdio>

#include "allegro_b200.h"
#include "plan.h"

namespace allegro {

// ---------------------------------------------------------------- host: errors, launch accounting
void set_error(const char* fmt, ...);
extern std::atomic<long> g_launches;

#define ALLEGRO_CHECK_ARG(cond, msg)                          \
    do {                                                      \
        if (!(cond)) {                                        \
            allegro::set_error("%s: %s", __func__, msg);      \
            return ALLEGRO_EINVAL;                            \
        }                                                     \
    } while (0)

#define ALLEGRO_CUDA(call)                                                              \
    do {                                                                                \
        cudaError_t e__ = (call);                                                       \
        if (e__ != cudaSuccess) {                                                       \
            allegro::set_error("%s: %s -> %s", __func__, #call, cudaGetErrorString(e__)); \
            return ALLEGRO_ECUDA;                                                       \
        }                                                                               \
    } while (0)

#define ALLEGRO_LAUNCHED()                    \
    do {                                      \
        allegro::g_launches.fetch_add(1);     \
        ALLEGRO_CUDA(cudaGetLastError());     \
    } while (0)

static inline bool aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }

// ---------------------------------------------------------------- device: PTX wrappers (mbarrier, bulk copy)
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t* bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ bool mbar_try_wait(uint64_t* bar, uint32_t parity) {
    uint32_t ok;
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n"
        "selp.u32 %0, 1, 0, p;\n"
        "}\n"
        : "=r"(ok)
        : "r"(smem_u32(bar)), "r"(parity)
        : "memory");
    return ok != 0;
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
    while (!mbar_try_wait(bar, parity)) {
    }
}
// 1-D bulk copy global -> shared, completion signalled on an mbarrier (SASS: UBLKCP)
__device__ __forceinline__ void bulk_load(void* dst_smem, const void* src_gmem, uint32_t bytes, uint64_t* bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_u32(dst_smem)),
                 "l"(src_gmem), "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}
// 1-D bulk copy shared -> global, tracked by the issuing thread's bulk async-group
__device__ __forceinline__ void bulk_store(void* dst_gmem, const void* src_smem, uint32_t bytes) {
    asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;" ::"l"(dst_gmem), "r"(smem_u32(src_smem)), "r"(bytes)
                 : "memory");
}
// 2-D tiled TMA copies through a tensor map (SASS: UTMALDG / UTMASTG); c0 = element index in a row, c1 = row index
__device__ __forceinline__ void tma_load_2d(void* dst_smem, const CUtensorMap* tmap, int c0, int c1, uint64_t* bar) {
    asm volatile("cp.async.bulk.tensor.2d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];" ::"r"(smem_u32(dst_smem)),
                 "l"(tmap), "r"(c0), "r"(c1), "r"(smem_u32(bar))
                 : "memory");
}
__device__ __forceinline__ void tma_store_2d(const CUtensorMap* tmap, int c0, int c1, const void* src_smem) {
    asm volatile("cp.async.bulk.tensor.2d.global.shared::cta.tile.bulk_group [%0, {%1, %2}], [%3];" ::"l"(tmap), "r"(c0), "r"(c1),
                 "r"(smem_u32(src_smem))
                 : "memory");
}
// ask the L2 to fetch a contiguous range ahead of its use (no completion to wait for; size a multiple of 16 bytes)
__device__ __forceinline__ void bulk_prefetch_l2(const void* src_gmem, uint32_t bytes) {
    asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(src_gmem), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void bulk_wait_read() {
    asm volatile("cp.async.bulk.wait_group.read %0;" ::"n"(N) : "memory");
}
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
__device__ __forceinline__ void fence_mbar_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
// named barrier over `nthreads` threads (id 1..15)
__device__ __forceinline__ void named_bar(int id, int nthreads) {
    asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(nthreads) : "memory");
}

// ---------------------------------------------------------------- device: per-thread feature rows in shared memory
// A thread owns one channel row of DV contiguous elements.  Widest vector that the row stride allows:
// 16 B when DV*sizeof(T) % 16 == 0, else 8 B (l_max = 2, fp32: stride 72 B -> LDS.64, bank-conflict free
// because 18*lane mod 32 hits 16 distinct even banks per half-warp).
template <typename T, int DV>
__device__ __forceinline__ void row_load(const T* __restrict__ p, T (&r)[DV]) {
    constexpr int RB = DV * (int)sizeof(T);
    if constexpr (RB % 16 == 0) {
        const int4* q = reinterpret_cast<const int4*>(p);
        int4 v[RB / 16];
#pragma unroll
        for (int i = 0; i < RB / 16; ++i) v[i] = q[i];
        const T* s = reinterpret_cast<const T*>(v);
#pragma unroll
        for (int i = 0; i < DV; ++i) r[i] = s[i];
    } else {
        static_assert(RB % 8 == 0, "row must be a multiple of 8 bytes");
        const int2* q = reinterpret_cast<const int2*>(p);
        int2 v[RB / 8];
#pragma unroll
        for (int i = 0; i < RB / 8; ++i) v[i] = q[i];
        const T* s = reinterpret_cast<const T*>(v);
#pragma unroll
        for (int i = 0; i < DV; ++i) r[i] = s[i];
    }
}
template <typename T, int DV>
__device__ __forceinline__ void row_store(T* __restrict__ p, const T (&r)[DV]) {
    constexpr int RB = DV * (int)sizeof(T);
    if constexpr (RB % 16 == 0) {
        int4 v[RB / 16];
        T* s = reinterpret_cast<T*>(v);
#pragma unroll
        for (int i = 0; i < DV; ++i) s[i] = r[i];
        int4* q = reinterpret_cast<int4*>(p);
#pragma unroll
        for (int i = 0; i < RB / 16; ++i) q[i] = v[i];
    } else {
        int2 v[RB / 8];
        T* s = reinterpret_cast<T*>(v);
#pragma unroll
        for (int i = 0; i < DV; ++i) s[i] = r[i];
        int2* q = reinterpret_cast<int2*>(p);
#pragma unroll
        for (int i = 0; i < RB / 8; ++i) q[i] = v[i];
    }
}

// Rows of exactly 128 bytes (l_max = 3, fp32) moved by 2-D TMA with the 128-byte swizzle: the 16-byte chunk j of row r sits at chunk
// position j ^ (r & 7) of the row's 128 bytes (tile base 1024-byte aligned).  `row` points at the row's first byte, sw = (r & 7) << 4.
// A quarter-warp's eight 128-bit accesses then hit eight different bank groups instead of one (linear rows: 8-way conflict).
template <typename T, int DV>
__device__ __forceinline__ void row_load_sw(const unsigned char* __restrict__ row, uint32_t sw, T (&r)[DV]) {
    static_assert(DV * sizeof(T) == 128, "swizzled rows are 128 bytes");
    int4 v[8];
#pragma unroll
    for (int j = 0; j < 8; ++j) v[j] = *reinterpret_cast<const int4*>(row + (((uint32_t)j << 4) ^ sw));
    const T* s = reinterpret_cast<const T*>(v);
#pragma unroll
    for (int i = 0; i < DV; ++i) r[i] = s[i];
}
template <typename T, int DV>
__device__ __forceinline__ void row_store_sw(unsigned char* __restrict__ row, uint32_t sw, const T (&r)[DV]) {
    static_assert(DV * sizeof(T) == 128, "swizzled rows are 128 bytes");
    int4 v[8];
    T* s = reinterpret_cast<T*>(v);
#pragma unroll
    for (int i = 0; i < DV; ++i) s[i] = r[i];
#pragma unroll
    for (int j = 0; j < 8; ++j) *reinterpret_cast<int4*>(row + (((uint32_t)j << 4) ^ sw)) = v[j];
}

// item it -> (centre, e0, e1); items == nullptr means one item per centre
__device__ __forceinline__ void get_item(const int* __restrict__ items, const int* __restrict__ row_ptr, long it, int& c, int& e0, int& e1) {
    if (items) {
        c = items[3 * it]; e0 = items[3 * it + 1]; e1 = items[3 * it + 2];
    } else {
        c = (int)it; e0 = row_ptr[it]; e1 = row_ptr[it + 1];
    }
}

}  // namespace allegro

namespace allegro {

// Sum the per-item partial rows of every centre in item order (A16): item `it` is the first item of its
// centre iff it == 0 or the previous item names another centre; that CTA adds the centre's partials
// sequentially, so the result is independent of scheduling.
template <typename T>
__global__ void combine_items_kernel(const int* __restrict__ items, long n_items, int rowlen, const T* __restrict__ partial,
                                     T* __restrict__ dst) {
    const long it = blockIdx.x;
    const int c = items[3 * it];
    if (it > 0 && items[3 * (it - 1)] == c) return;
    for (int idx = threadIdx.x; idx < rowlen; idx += blockDim.x) {
        T acc = T(0);
        for (long k = it; k < n_items && items[3 * k] == c; ++k) acc += partial[(size_t)k * rowlen + idx];
        dst[(size_t)c * rowlen + idx] = acc;
    }
}

__host__ __device__ static inline uint32_t align128(size_t x) { return (uint32_t)((x + 127) / 128 * 128); }

}  // namespace allegro
