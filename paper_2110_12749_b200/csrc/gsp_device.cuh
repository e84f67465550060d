// gsp_device.cuh — small device-side helpers shared by the libgsp kernels (mbarrier, bulk/TMA copies).
#pragma once

#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>

namespace gsp {

__device__ __forceinline__ uint32_t smem_u32(const void *p) {
    return (uint32_t)__cvta_generic_to_shared(p);
}

__device__ __forceinline__ void mbar_init(uint64_t *bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}

__device__ __forceinline__ void mbar_arrive(uint64_t *bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}

__device__ __forceinline__ void mbar_arrive_expect_tx(uint64_t *bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)),
                 "r"(bytes)
                 : "memory");
}

__device__ __forceinline__ bool mbar_try_wait(uint64_t *bar, uint32_t parity) {
    uint32_t done;
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n"
        "selp.u32 %0, 1, 0, p;\n"
        "}\n"
        : "=r"(done)
        : "r"(smem_u32(bar)), "r"(parity)
        : "memory");
    return done != 0;
}

__device__ __forceinline__ void mbar_wait(uint64_t *bar, uint32_t parity) {
    while (!mbar_try_wait(bar, parity)) {
    }
}

// 1-D bulk async copy global -> shared (TMA engine, SASS UBLKCP); size and both
// addresses are multiples of 16 bytes; completion is signalled on `bar` as tx bytes.
__device__ __forceinline__ void bulk_g2s(void *dst_smem, const void *src_gmem, uint32_t bytes,
                                         uint64_t *bar) {
    asm volatile(
        "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::
            "r"(smem_u32(dst_smem)),
        "l"(src_gmem), "r"(bytes), "r"(smem_u32(bar))
        : "memory");
}

__device__ __forceinline__ bool mbar_test_wait(uint64_t *bar, uint32_t parity) {
    uint32_t done;
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "mbarrier.test_wait.parity.shared::cta.b64 p, [%1], %2;\n"
        "selp.u32 %0, 1, 0, p;\n"
        "}\n"
        : "=r"(done)
        : "r"(smem_u32(bar)), "r"(parity)
        : "memory");
    return done != 0;
}


// 2-D tiled TMA load global -> shared (SASS UTMALDG): box of the tensor map at element
// coordinates {c0 (innermost), c1}; out-of-range elements are zero-filled and still counted.
__device__ __forceinline__ void tma_load_2d(void *dst_smem, const CUtensorMap *tmap, int c0, int c1,
                                            uint64_t *bar) {
    asm volatile(
        "cp.async.bulk.tensor.2d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];" ::
            "r"(smem_u32(dst_smem)),
        "l"(tmap), "r"(c0), "r"(c1), "r"(smem_u32(bar))
        : "memory");
}

// named barrier for a subset of the CTA's warps (id 1..15, nthreads a multiple of 32)
__device__ __forceinline__ void named_bar_sync(int id, int nthreads) {
    asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(nthreads) : "memory");
}

// Fold `ds` (a power of two <= 256) consecutive samples held by the 256 consecutive threads tid = 0..255 of a CTA
// (sample = block base + tid, base a multiple of 256): the thread with (tid & (ds-1)) == 0 returns the sum.
// Up to 32 samples fold with shuffles; larger ds (the DownSamp 64 / 128 rows of the paper's Tables 2-3) meet in
// `scratch` (8 entries) between two named barriers `bar` of those 256 threads.  `ds` must be CTA-uniform.
// The order of the additions is fixed (float32 results are deterministic).
template <typename T>
__device__ __forceinline__ T fold_ds256(T v, int ds, int tid, T *scratch, int bar) {
    const int w = ds < 32 ? ds : 32;
    for (int o = 1; o < w; o <<= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    if (ds > 32) {
        if ((tid & 31) == 0) scratch[tid >> 5] = v;
        named_bar_sync(bar, 256);
        if ((tid & (ds - 1)) == 0) {
            T t = scratch[tid >> 5];
            for (int q = 1; q < (ds >> 5); ++q) t += scratch[(tid >> 5) + q];
            v = t;
        }
        named_bar_sync(bar, 256);
    }
    return v;
}

// Cluster barrier that publishes the CTA's shared-memory writes to the other CTAs of the cluster with ONE
// cluster-scope fence: the CTA barrier orders every thread's writes before thread 0's fence (cumulativity),
// the arrive itself is relaxed.  (cooperative_groups' cluster.sync() makes every thread execute the fence.)
__device__ __forceinline__ void cluster_sync_publish() {
    __syncthreads();
    if (threadIdx.x == 0) asm volatile("fence.acq_rel.cluster;" ::: "memory");
    asm volatile("barrier.cluster.arrive.relaxed.aligned;" ::: "memory");
    asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory");
}

// Cluster barrier with no memory ordering (e.g. "nobody exits while its shared memory may still be read").
__device__ __forceinline__ void cluster_sync_relaxed() {
    asm volatile("barrier.cluster.arrive.relaxed.aligned;" ::: "memory");
    asm volatile("barrier.cluster.wait.aligned;" ::: "memory");
}

}  // namespace gsp
