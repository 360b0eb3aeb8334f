// adsc_ptx.cuh — one-line PTX wrappers shared by the stage kernels (sm_90+ features on sm_100a):
// mbarrier (split arrive / wait, transaction bytes), thread-block-cluster addressing, remote
// shared-memory stores that complete transaction bytes on the consumer's mbarrier, and the bulk
// asynchronous copy engine (TMA, 1-D form: cp.async.bulk global -> shared).
#pragma once
#include <cstdint>

namespace adsc {

__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ uint32_t cluster_rank()
{
    uint32_t r;
    asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r));
    return r;
}
__device__ __forceinline__ uint32_t map_rank(uint32_t addr, int rank)
{
    uint32_t r;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(addr), "r"(rank));
    return r;
}
__device__ __forceinline__ void mbar_init(uint32_t mb, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(mb), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t mb)
{
    asm volatile("{\n\t.reg .b64 st;\n\tmbarrier.arrive.shared::cta.b64 st, [%0];\n\t}" ::"r"(mb) : "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint32_t mb, uint32_t bytes)
{
    asm volatile("{\n\t.reg .b64 st;\n\tmbarrier.arrive.expect_tx.shared::cta.b64 st, [%0], %1;\n\t}" ::"r"(mb), "r"(bytes) : "memory");
}
template <bool CLUSTER_SCOPE>
__device__ __forceinline__ void mbar_wait(uint32_t mb, uint32_t parity)
{
    if (CLUSTER_SCOPE)
        asm volatile("{\n\t.reg .pred p;\n\tLAB_WAIT:\n\t"
                     "mbarrier.try_wait.parity.acquire.cluster.shared::cta.b64 p, [%0], %1;\n\t"
                     "@p bra DONE;\n\tbra LAB_WAIT;\n\tDONE:\n\t}" ::"r"(mb), "r"(parity) : "memory");
    else
        asm volatile("{\n\t.reg .pred p;\n\tLAB_WAIT:\n\t"
                     "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
                     "@p bra DONE;\n\tbra LAB_WAIT;\n\tDONE:\n\t}" ::"r"(mb), "r"(parity) : "memory");
}
// Remote store into a peer CTA's shared memory that completes 8 (16) transaction bytes on the peer's mbarrier.
__device__ __forceinline__ void st_async_f64(uint32_t dst_cluster, double v, uint32_t mbar_cluster)
{
    asm volatile("st.async.weak.shared::cluster.mbarrier::complete_tx::bytes.b64 [%0], %1, [%2];"
                 ::"r"(dst_cluster), "l"(__double_as_longlong(v)), "r"(mbar_cluster) : "memory");
}
__device__ __forceinline__ void st_async_f64x2(uint32_t dst_cluster, double v0, double v1, uint32_t mbar_cluster)
{
    asm volatile("st.async.weak.shared::cluster.mbarrier::complete_tx::bytes.v2.b64 [%0], {%1, %2}, [%3];"
                 ::"r"(dst_cluster), "l"(__double_as_longlong(v0)), "l"(__double_as_longlong(v1)), "r"(mbar_cluster) : "memory");
}
// Bulk asynchronous copy (TMA, 1-D): `bytes` (multiple of 16) from global to this CTA's shared memory; completion is
// signalled as transaction bytes on the mbarrier.  Source and destination 16-byte aligned.
__device__ __forceinline__ void bulk_g2s(uint32_t dst_smem, const void *src_global, uint32_t bytes, uint32_t mbar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(dst_smem), "l"(src_global), "r"(bytes), "r"(mbar) : "memory");
}
// mbarrier.arrive.expect_tx followed by the bulk copy that completes it (one thread).
__device__ __forceinline__ void bulk_g2s_arrive(uint32_t dst_smem, const void *src_global, uint32_t bytes, uint32_t mbar)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%3], %2;\n\t"
                 "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(dst_smem), "l"(src_global), "r"(bytes), "r"(mbar) : "memory");
}
// Orders this thread's earlier generic-proxy accesses to shared memory (and those a preceding warp barrier made
// cumulative) before its later async-proxy operations (bulk copies into the same buffer).
__device__ __forceinline__ void fence_proxy_async_smem()
{
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
}
// 256-bit global accesses (sm_100: LDG.E.256 / STG.E.256), 32-byte aligned.
__device__ __forceinline__ void ldg256(const double *p, double &a, double &b, double &c, double &d)
{
    // streamed once per use: no L1 allocation (the little L1 left beside 227 KB of shared memory serves the stack)
    asm volatile("ld.global.L1::no_allocate.v4.f64 {%0,%1,%2,%3}, [%4];" : "=d"(a), "=d"(b), "=d"(c), "=d"(d) : "l"(p) : "memory");
}
__device__ __forceinline__ void stg256(double *p, double a, double b, double c, double d)
{
    asm volatile("st.global.v4.f64 [%0], {%1,%2,%3,%4};" ::"l"(p), "d"(a), "d"(b), "d"(c), "d"(d) : "memory");
}

}  // namespace adsc
