// cluster.cuh -- thread-block-cluster exchange primitives (sm_100a): data and signal in ONE distributed-shared-memory
// trip.  A sender issues st.async stores that complete transaction bytes on the RECEIVER's mbarrier; the receiver arms
// the mbarrier with the byte count it expects and waits on its parity.  Measured on B200 in round 1:
// one such all-to-all among 16 CTAs costs 0.3-0.4 us, a hardware cluster barrier 0.55-0.7 us.
#pragma once
#include "common.cuh"

namespace hpsd {

__device__ __forceinline__ unsigned cx_smem_u32(const void *p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ unsigned cx_rank() {
    unsigned r;
    asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r));
    return r;
}
// address of the same shared-memory location in CTA `rank` of this cluster
__device__ __forceinline__ unsigned cx_mapa(unsigned addr, int rank) {
    unsigned remote;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(remote) : "r"(addr), "r"(rank));
    return remote;
}
__device__ __forceinline__ void cx_st_async(unsigned raddr, cplx v, unsigned rmbar) {
    asm volatile("st.async.weak.shared::cluster.mbarrier::complete_tx::bytes.v2.f64 [%0], {%1, %2}, [%3];" ::"r"(raddr), "d"(v.x), "d"(v.y), "r"(rmbar) : "memory");
}
__device__ __forceinline__ void cx_mbar_init(unsigned mbar, unsigned count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(mbar), "r"(count) : "memory");
}
__device__ __forceinline__ void cx_fence_mbar_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
// one pending arrival per phase (this arm) + the bytes the phase will receive
__device__ __forceinline__ void cx_arm(unsigned mbar, unsigned bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(mbar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void cx_wait(unsigned mbar, unsigned parity) {
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "CX_WAIT_%=:\n\t"
        "mbarrier.try_wait.parity.acquire.cluster.shared::cta.b64 p, [%0], %1;\n\t"
        "@p bra CX_DONE_%=;\n\t"
        "bra CX_WAIT_%=;\n\t"
        "CX_DONE_%=:\n\t}" ::"r"(mbar), "r"(parity) : "memory");
}
// release/acquire at CLUSTER scope (cooperative_groups' cluster.sync() fences at gpu scope)
__device__ __forceinline__ void cx_barrier() {
    asm volatile("barrier.cluster.arrive.release.aligned;\n\tbarrier.cluster.wait.acquire.aligned;" ::: "memory");
}

}  // namespace hpsd
