// bulk_common.cuh — mbarrier / bulk-copy (TMA engine, cp.async.bulk) primitives and shared-memory accessors shared by the
// warp-pipelined tile kernels (nasg_tile_kernels.cu: layout v1 rows; nasg_rec_kernels.cu: tile records).
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>
#include <string.h>

namespace nasg {
namespace bulk {

__device__ __forceinline__ unsigned smem_u32(const void *p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(unsigned bar, unsigned count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_init_fence()
{
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
}
__device__ __forceinline__ void mbar_expect_tx(unsigned bar, unsigned bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(unsigned bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
// One probe of the phase with this parity (the suspend-time hint lets the hardware park the thread while the data is late).
__device__ __forceinline__ bool mbar_try_wait(unsigned bar, unsigned parity)
{
    unsigned done;
    asm volatile(
        "{\n\t"
        ".reg .pred p;\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2, %3;\n\t"
        "selp.u32 %0, 1, 0, p;\n\t"
        "}" : "=r"(done) : "r"(bar), "r"(parity), "r"(0x989680u) : "memory");
    return done != 0;
}
// Wait for the phase with this parity.
__device__ __forceinline__ void mbar_wait(unsigned bar, unsigned parity)
{
    while (!mbar_try_wait(bar, parity)) {}
}
__device__ __forceinline__ bool elect_one()
{
    unsigned pred;
    asm volatile(
        "{\n\t"
        ".reg .pred p;\n\t"
        "elect.sync _|p, 0xffffffff;\n\t"
        "selp.u32 %0, 1, 0, p;\n\t"
        "}" : "=r"(pred));
    return pred != 0;
}
// SLOT REFILL PROTOCOL (a round-2 bug, found by the host-pipeline bit-identity test). A slot is refilled by the copy engine
// (async proxy) right after the lanes have read it (generic proxy). Program order + __syncwarp() is NOT enough: the async-proxy
// write is not ordered after generic-proxy reads that have been issued but not yet performed, and when the SM comes out of idle
// (low clocks) with per-lane global loads queued in front of them, the shared-memory reads of a few lanes were overtaken by the
// refill: wrong values for some lanes of ONE tile in ~40 % of cold launches with N % 16 != 0, never when warm. The PTX rule is a
// proxy fence between the two: all lanes read, __syncwarp(), then the issuing lane executes fence.proxy.async before
// mbarrier.arrive.expect_tx + cp.async.bulk. Measured cost 1.2 % (an explicit "empty" mbarrier with 32 arrivals per refill
// was also correct and cost 7 %). tests/test_rec_gpu.py::test_cold_launches_are_correct keeps the scenario covered.
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
// 1-D bulk copy global -> shared of `bytes` (multiple of 16; both addresses 16-byte aligned), completing on `bar`
__device__ __forceinline__ void bulk_g2s(unsigned dst, const void *src, unsigned bytes, unsigned bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(dst), "l"(src), "r"(bytes), "r"(bar) : "memory");
}

// shared-memory accesses by 32-bit shared-window address. Plain loads (not asm): they cannot move across the mbarrier
// wait or the __syncwarp + re-issue, which are asm volatile with a memory clobber / a barrier.
__device__ __forceinline__ float4 lds128(unsigned addr) { return *reinterpret_cast<const float4 *>(__cvta_shared_to_generic(addr)); }
__device__ __forceinline__ float lds32(unsigned addr) { return *reinterpret_cast<const float *>(__cvta_shared_to_generic(addr)); }
__device__ __forceinline__ unsigned lds8(unsigned addr) { return *reinterpret_cast<const unsigned char *>(__cvta_shared_to_generic(addr)); }
// two 64-bit values (any 8-byte type: the packed f32x2 pairs) as one 16-byte access
template <typename T8>
__device__ __forceinline__ void sts64x2(unsigned addr, T8 a, T8 b)
{
    static_assert(sizeof(T8) == 8, "8-byte type");
    unsigned long long ua, ub;
    memcpy(&ua, &a, 8); memcpy(&ub, &b, 8);
    asm volatile("st.shared.v2.b64 [%0], {%1,%2};" ::"r"(addr), "l"(ua), "l"(ub) : "memory");
}
template <typename T8>
__device__ __forceinline__ void lds64x2(unsigned addr, T8 &a, T8 &b)
{
    static_assert(sizeof(T8) == 8, "8-byte type");
    unsigned long long ua, ub;
    asm volatile("ld.shared.v2.b64 {%0,%1}, [%2];" : "=l"(ua), "=l"(ub) : "r"(addr) : "memory");   // (reads memory: must not be hoisted over the stores)
    memcpy(&a, &ua, 8); memcpy(&b, &ub, 8);
}
template <typename T8>
__device__ __forceinline__ T8 lds64(unsigned addr)
{
    static_assert(sizeof(T8) == 8, "8-byte type");
    return *reinterpret_cast<const T8 *>(__cvta_shared_to_generic(addr));
}
__device__ __forceinline__ void sts128(unsigned addr, float4 v)
{
    asm volatile("st.shared.v4.f32 [%0], {%1,%2,%3,%4};" ::"r"(addr), "f"(v.x), "f"(v.y), "f"(v.z), "f"(v.w) : "memory");
}

} // namespace bulk
} // namespace nasg
