// sie_common.cuh — shared device/host helpers of libsie_dfmp2.so (sm_100a only).
// PTX wrappers: FP64 tensor-core MMA (DMMA.8x8x4), mbarrier, TMA tensor loads.
#pragma once

#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>

namespace sie {

// ------------------------------------------------------------------------------------------------
// FP64 tensor core: mma.sync.m8n8k4 (the only native FP64 MMA shape on sm_100a; larger PTX shapes
// lower to sequences of DMMA.8x8x4).  Fragment ownership, lane = 4*g + t (g = lane>>2, t = lane&3):
//   A (8x4, row):  a   = A[g][t]          B (4x8, col):  b = B[t][g]
//   C/D (8x8):     c0  = C[g][2t], c1 = C[g][2t+1]
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ void dmma884(double& c0, double& c1, double a, double b) {
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                 : "+d"(c0), "+d"(c1)
                 : "d"(a), "d"(b));
}

__device__ __forceinline__ uint32_t smem_u32(const void* p) {
    return static_cast<uint32_t>(__cvta_generic_to_shared(p));
}

__device__ __forceinline__ double2 lds128(uint32_t addr) {  // 16-byte shared load from a 32-bit shared address
    double2 v;
    asm volatile("ld.shared.v2.f64 {%0,%1}, [%2];" : "=d"(v.x), "=d"(v.y) : "r"(addr));
    return v;
}

// ------------------------------------------------------------------------------------------------
// mbarrier (shared::cta, 64-bit)
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void fence_mbar_init() {
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void fence_proxy_async() {
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t* bar) {
    asm volatile("{\n\t.reg .b64 st;\n\tmbarrier.arrive.shared::cta.b64 st, [%0];\n\t}" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint64_t* bar, uint32_t bytes) {
    asm volatile("{\n\t.reg .b64 st;\n\tmbarrier.arrive.expect_tx.shared::cta.b64 st, [%0], %1;\n\t}" ::"r"(smem_u32(bar)),
                 "r"(bytes)
                 : "memory");
}
__device__ __forceinline__ bool mbar_try_wait(uint64_t* bar, uint32_t parity) {
    uint32_t ok;
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
        "selp.u32 %0, 1, 0, p;\n\t}"
        : "=r"(ok)
        : "r"(smem_u32(bar)), "r"(parity)
        : "memory");
    return ok != 0;
}
// Non-blocking test of a phase: try_wait above may SUSPEND the thread (and with it the warp at its reconvergence point)
// for a system-dependent time when the phase is not complete; test_wait returns at once.
__device__ __forceinline__ bool mbar_test_wait(uint64_t* bar, uint32_t parity) {
    uint32_t ok;
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "mbarrier.test_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
        "selp.u32 %0, 1, 0, p;\n\t}"
        : "=r"(ok)
        : "r"(smem_u32(bar)), "r"(parity)
        : "memory");
    return ok != 0;
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
    while (!mbar_try_wait(bar, parity)) {
    }
}

// ------------------------------------------------------------------------------------------------
// TMA: 3-D tiled tensor load global -> shared, completion on an mbarrier (complete_tx::bytes)
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ void tma_load_3d(void* smem_dst, const CUtensorMap* map, uint64_t* bar, int c0, int c1, int c2) {
    asm volatile(
        "cp.async.bulk.tensor.3d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];" ::"r"(
            smem_u32(smem_dst)),
        "l"(reinterpret_cast<uint64_t>(map)), "r"(c0), "r"(c1), "r"(c2), "r"(smem_u32(bar))
        : "memory");
}
// A tensor map that lives in global memory (not a __grid_constant__ kernel parameter) was written through the generic
// proxy (here: a cudaMemcpyAsync into the workspace); before the first cp.async.bulk.tensor that reads it through the
// tensormap proxy the issuing thread must acquire it, or a descriptor-cache hit may serve stale contents of that address.
__device__ __forceinline__ void tma_acquire_desc(const CUtensorMap* map) {
    asm volatile("fence.proxy.tensormap::generic.acquire.sys [%0], 128;" ::"l"(reinterpret_cast<uint64_t>(map)) : "memory");
}
__device__ __forceinline__ void tma_prefetch_desc(const CUtensorMap* map) {
    asm volatile("prefetch.tensormap [%0];" ::"l"(reinterpret_cast<uint64_t>(map)) : "memory");
}

// named barrier among a subset of warps (id 1..15), count = participating threads
__device__ __forceinline__ void named_bar_sync(int id, int nthreads) {
    asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(nthreads) : "memory");
}

// ------------------------------------------------------------------------------------------------
// host side
// ------------------------------------------------------------------------------------------------
void note_launch();                      // counts kernel launches (api.cu)
// cudaFuncSetAttribute(MaxDynamicSharedMemorySize) is a per-device setting: `done` is a per-kernel bit mask over device
// ordinals (api.cu); devices >= 64 set the attribute on every launch.  Thread-safe (atomic mask, idempotent call).
struct SmemAttrOnce {
    unsigned long long done = 0;
};
int ensure_smem_attr(const void* kernel, int bytes, SmemAttrOnce& once);
int set_cuda_error(cudaError_t e);       // records the text, returns SIE_ECUDA
int set_cuda_error_text(const char* s);  // records the text, returns SIE_ECUDA

// Encode a 3-D FP64 tensor map: dims {d0 (contiguous), d1, d2}, byte strides of d1 and d2, box {b0,b1,b2}.
// OOB elements are zero-filled.  Returns SIE_OK or SIE_ECUDA.
int make_tensor_map_3d(CUtensorMap* out, const double* base, uint64_t d0, uint64_t d1, uint64_t d2, uint64_t stride1_bytes,
                       uint64_t stride2_bytes, uint32_t b0, uint32_t b1, uint32_t b2);

static inline size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

}  // namespace sie
