// s2_force_common.cuh -- pieces shared by the force kernels of all three precisions:
// mbarrier / bulk-copy (TMA) primitives, the tile pipeline geometry and warp-level helpers.
#pragma once

#include "s2_internal.h"

namespace s2 {

__device__ __forceinline__ uint32_t smem_u32(const void *p)
{
    return (uint32_t)__cvta_generic_to_shared(p);
}

__device__ __forceinline__ void mbar_init(uint64_t *bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}

__device__ __forceinline__ void mbar_fence_init()
{
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}

__device__ __forceinline__ void mbar_arrive_expect_tx(uint64_t *bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes)
                 : "memory");
}

__device__ __forceinline__ void mbar_wait(uint64_t *bar, uint32_t parity)
{
    asm volatile(
        "{\n"
        ".reg .pred P1;\n"
        "WAIT_LOOP:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 P1, [%0], %1;\n"
        "@P1 bra WAIT_DONE;\n"
        "bra WAIT_LOOP;\n"
        "WAIT_DONE:\n"
        "}\n" ::"r"(smem_u32(bar)),
        "r"(parity)
        : "memory");
}

// 1-D bulk asynchronous copy global -> shared, completion counted in bytes on an mbarrier
// (cp.async.bulk; SASS UBLKCP).  dst, src 16-byte aligned, bytes a multiple of 16.
__device__ __forceinline__ void bulk_g2s(void *dst, const void *src, uint32_t bytes, uint64_t *bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                     smem_u32(dst)),
                 "l"(src), "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}

// Thread-block cluster primitives (distributed shared memory)
__device__ __forceinline__ uint32_t cluster_ctarank()
{
    uint32_t r;
    asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r));
    return r;
}
__device__ __forceinline__ void cluster_sync()
{
    asm volatile("barrier.cluster.arrive.release.aligned;\n\tbarrier.cluster.wait.acquire.aligned;" ::: "memory");
}
// fp64 load from the shared memory of CTA `rank` of this cluster, at the same offset as local address saddr
__device__ __forceinline__ double ld_dsmem_f64(uint32_t saddr, uint32_t rank)
{
    uint32_t ra;
    double v;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(ra) : "r"(saddr), "r"(rank));
    asm volatile("ld.shared::cluster.f64 %0, [%1];" : "=d"(v) : "r"(ra) : "memory");
    return v;
}

// Work decomposition of one CTA:
//   warp w -> (wi, wj) = (w / Wj, w % Wj);  lane -> (il, jl) = (lane / L, lane % L)
//   i index  = (blockIdx.x * (kWarps / Wj) + wi) * (32 / L) + il
//   slice id = blockIdx.y * Wj + wj   (the partial-record row this warp column writes)
struct Decomp {
    int lane, il, jl, wi, wj, i, slice;
    bool i_valid;
};

template <int L>
__device__ __forceinline__ Decomp decompose(int Wj, int ni)
{
    Decomp d;
    const int w = threadIdx.x >> 5;
    d.lane = threadIdx.x & 31;
    d.il = d.lane / L;
    d.jl = d.lane % L;
    d.wi = w / Wj;
    d.wj = w % Wj;
    d.i = (blockIdx.x * (kWarps / Wj) + d.wi) * (32 / L) + d.il;
    d.i_valid = d.i < ni;
    if (!d.i_valid) d.i = ni - 1;   // padding threads recompute the last i and never write
    d.slice = blockIdx.y * Wj + d.wj;
    return d;
}

__device__ __forceinline__ double shfl_xor_d(double v, int m)
{
    return __shfl_xor_sync(0xffffffffu, v, m);
}

}  // namespace s2
