// pipe_common.cuh — pieces shared by the persistent cp.async-pipelined kernels (NASGabor and SH):
// LDGSTS wrappers, streaming stores, the visibility-mask load and the resident-grid launch helper.
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

#include "nasg_internal.h"   // resident_grid

namespace nasg {

#ifndef NASG_PBLOCK
#define NASG_PBLOCK 256
#endif
constexpr int PBLOCK = NASG_PBLOCK;

__device__ __forceinline__ void cp_async16(void *smem, const void *gmem)
{
    const unsigned s = (unsigned)__cvta_generic_to_shared(smem);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(s), "l"(gmem) : "memory");
}
__device__ __forceinline__ void cp_async4(void *smem, const void *gmem)
{
    const unsigned s = (unsigned)__cvta_generic_to_shared(smem);
    asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(s), "l"(gmem) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N_PENDING>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N_PENDING) : "memory"); }

__device__ __forceinline__ void st_cs(float *p, float v) { __stcs(p, v); }
__device__ __forceinline__ void st_cs4(float *p, float4 v) { __stcs(reinterpret_cast<float4 *>(p), v); }

__device__ __forceinline__ unsigned load_mask(const uint8_t *vis, int64_t N, int64_t n, int C)
{
    unsigned m = 0;
    if (n < N) {
        if (!vis) return (1u << C) - 1u;
#pragma unroll 4
        for (int c = 0; c < C; ++c) m |= (vis[(int64_t)c * N + n] != 0 ? 1u : 0u) << c;
    }
    return m;
}

// Visibility mask staging (packed NASGabor kernels, SH kernels). A byte load from global memory that is consumed in the same
// iteration stalls the warp for a DRAM latency (ncu: 11% of all stall samples sat on it), and the compiler
// places the consumer wherever it likes. When vis rows are 4-byte aligned (N % 4 == 0) every fourth lane
// copies the 4 bytes of its quad with cp.async into the header slot instead, a few items ahead of use;
// the bytes are read back from shared memory after the wait + __syncwarp. Otherwise (vis == NULL or an
// unaligned N) the raw bytes are loaded one Gaussian ahead into registers.
struct RawMask { unsigned b[4]; };
__device__ __forceinline__ RawMask load_raw_mask(const uint8_t *vis, int64_t N, int64_t n, int C)
{
    RawMask m;
#pragma unroll
    for (int c = 0; c < 4; ++c) m.b[c] = (n < N) ? ((c < C) ? (vis ? vis[(int64_t)c * N + n] : 1u) : 0u) : 0u;
    return m;
}
__device__ __forceinline__ unsigned combine_mask(const RawMask &m)
{
    return (m.b[0] ? 1u : 0u) | (m.b[1] ? 2u : 0u) | (m.b[2] ? 4u : 0u) | (m.b[3] ? 8u : 0u);
}
__device__ __forceinline__ bool vis_rows_aligned(const uint8_t *vis, int64_t N)
{
    return vis != nullptr && (N & 3) == 0 && (reinterpret_cast<uintptr_t>(vis) & 3u) == 0;
}
__device__ __forceinline__ void prefetch_vis(unsigned char *vm, int hslot, int tid, const uint8_t *vis, int64_t N, int64_t gn, int C)
{
    if ((tid & 3) == 0) {
#pragma unroll
        for (int c = 0; c < 4; ++c)
            if (c < C) cp_async4(vm + (hslot * 4 + c) * PBLOCK + tid, vis + (int64_t)c * N + gn);
    }
}
__device__ __forceinline__ unsigned staged_mask(const unsigned char *vm, int hslot, int tid, int C, bool valid)
{
    unsigned m = 0;
#pragma unroll
    for (int c = 0; c < 4; ++c)
        if (c < C) m |= (vm[(hslot * 4 + c) * PBLOCK + tid] != 0 ? 1u : 0u) << c;
    return valid ? m : 0u;
}
// Sum `v` over the block (PBLOCK threads) in a fixed order and let thread 0 store it to *dst.
// All threads of the block must call; `red` is PBLOCK/32 floats of shared memory.
__device__ __forceinline__ void pipe_block_sum_store(float v, float *red, float *dst)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    __syncthreads();
    if (lane == 0) red[warp] = v;
    __syncthreads();
    if (threadIdx.x == 0) {
        float s = 0.f;
#pragma unroll
        for (int w = 0; w < PBLOCK / 32; ++w) s += red[w];
        *dst = s;
    }
}

// Resident-grid size of a persistent kernel; the occupancy query and the shared-memory opt-in are done
// once per (kernel instantiation, device) and cached (benign, idempotent state).
template <typename Kernel>
static int pipe_grid(Kernel kernel, size_t smem, int64_t N, int *cached /* [64], one per kernel instantiation */)
{
    return resident_grid(kernel, PBLOCK, smem, N, cached);
}

} // namespace nasg
