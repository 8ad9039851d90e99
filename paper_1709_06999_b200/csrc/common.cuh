// common.cuh — complex / node-pair types, programmatic-dependent-launch, mbarrier and TMA bulk-copy wrappers (sm_100a).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "types.h"

namespace galb {

template <typename T> struct Vec2;
template <> struct Vec2<double> { using type = double2; };
template <> struct Vec2<float> { using type = float2; };
template <typename T> using cx = typename Vec2<T>::type;

// one entry of the sampled spectrum: the node of this column (.a) and of the next one (.b)
template <typename T> struct __align__(2 * sizeof(cx<T>)) NodePair { cx<T> a, b; };
// whole-entry stores: one 256-bit store in fp64 (sm_100), 128-bit in fp32
__device__ __forceinline__ void store_pair(NodePair<double>* p, const NodePair<double>& e) {
    asm volatile("st.global.v4.f64 [%0], {%1,%2,%3,%4};" ::"l"(p), "d"(e.a.x), "d"(e.a.y), "d"(e.b.x), "d"(e.b.y) : "memory");
}
__device__ __forceinline__ void store_pair(NodePair<float>* p, const NodePair<float>& e) {
    *reinterpret_cast<float4*>(p) = make_float4(e.a.x, e.a.y, e.b.x, e.b.y);
}

// Programmatic dependent launch (sm_90+): let the next kernel of the chain start placing its CTAs, and wait
// until the kernel before this one has completed and its writes are visible.  Every kernel of a call does both
// before its first global-memory access (harmless when launched without the attribute).
__device__ __forceinline__ void pdl_wait() {
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    asm volatile("griddepcontrol.wait;" ::: "memory");
}

template <typename T> __device__ __forceinline__ cx<T> mk(T x, T y) { cx<T> r; r.x = x; r.y = y; return r; }
template <typename V> __device__ __forceinline__ V cadd(V a, V b) { a.x += b.x; a.y += b.y; return a; }
template <typename V> __device__ __forceinline__ V csub(V a, V b) { a.x -= b.x; a.y -= b.y; return a; }
template <typename V> __device__ __forceinline__ V cmul(V a, V b) {
    V r; r.x = a.x * b.x - a.y * b.y; r.y = a.x * b.y + a.y * b.x; return r;
}
template <typename V> __device__ __forceinline__ V mul_mi(V a) { V r; r.x = a.y; r.y = -a.x; return r; }  // * (-i)

// ------------------------------------------------------------------------------------------
// mbarrier + TMA bulk-copy wrappers (PTX, sm_90+/sm_100a).
// ------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint32_t mb, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(mb), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_fence_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
__device__ __forceinline__ void mbar_expect_tx(uint32_t mb, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(mb), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t mb, uint32_t parity) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE_%=;\n"
        "bra WAIT_%=;\n"
        "DONE_%=:\n"
        "}\n" ::"r"(mb), "r"(parity) : "memory");
}
// same, for a thread that expects to wait long (the producer): sleep between polls so the spin does not
// take issue slots from the warps that share its scheduler
__device__ __forceinline__ void mbar_wait_relaxed(uint32_t mb, uint32_t parity) {
    uint32_t done = 0;
    for (;;) {
        asm volatile("{ .reg .pred p; mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2; selp.u32 %0, 1, 0, p; }"
                     : "=r"(done) : "r"(mb), "r"(parity) : "memory");
        if (done) break;
        __nanosleep(200);
    }
}
__device__ __forceinline__ uint64_t l2_policy_evict_first() {
    uint64_t pol;
    asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(pol));
    return pol;
}
// global -> shared bulk copy (TMA, 1-D): 16-byte aligned addresses, size a multiple of 16 bytes.
__device__ __forceinline__ void tma_load_1d(uint32_t dst, const void* src, uint32_t bytes, uint32_t mb, uint64_t pol) {
    asm volatile(
        "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;"
        ::"r"(dst), "l"(src), "r"(bytes), "r"(mb), "l"(pol) : "memory");
}

// Ask the L2 to fetch `bytes` (a multiple of 16, 16-byte aligned) from global memory: no destination, no completion
// to wait for.  One thread prefetches what a LATER CTA of the grid will read, so that CTA's loads find it in the
// L2 (about 250 clocks) instead of in HBM (a microsecond and more under load).
__device__ __forceinline__ void l2_prefetch_bulk(const void* src, uint32_t bytes) {
    asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(src), "r"(bytes) : "memory");
}

__device__ __forceinline__ void mbar_arrive(uint32_t mb) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(mb) : "memory");
}

}  // namespace galb
