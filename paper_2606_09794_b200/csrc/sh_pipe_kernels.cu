// sh_pipe_kernels.cu — fast path of the SH degree-3 comparison kernels for C <= 4 cameras (sm_100a),
// built the same way as the NASGabor fast path (nasg_pipe_kernels.cu): persistent threads, one thread per
// Gaussian, parameters streamed through a shared-memory ring filled by cp.async (LDGSTS) ahead of use,
// gradients written once with streaming stores, no atomics.
//
// Item stream: (Gaussian i, group g), g = 0..3; group g holds the 4 basis functions j = 4g..4g+3, i.e.
// 12 planar coefficient rows = 48 B per Gaussian (a NASGabor lobe is 44 B), and always lives in ring
// slot g. The per-Gaussian header (mean, g_colors in the backward, visibility bytes) travels with
// group 0 into header slot i % 2.
//
// The SH path has almost no arithmetic, so the load/store unit is what limits it (ncu: mio_throttle):
// 51 four-byte LDGSTS per Gaussian and thread. When the rows are 16-byte aligned (N % 4 == 0, aligned
// base pointers) the four lanes of a quad therefore share the work: lane j copies rows j, j+4, j+8 of
// the group for all four Gaussians of the quad with ONE 16-byte LDGSTS each (4x fewer copy
// instructions), and the [N,3] mean / g_colors records of the quad (48 contiguous bytes) with three
// 16-byte copies. Data is then read by a lane that did not copy it, so every step is:
// wait (own copies of the item landed) -> __syncwarp (quad's copies visible; everyone is done with the
// slot about to be refilled) -> prefetch -> compute. The loop has a warp-uniform trip count for this.
// Otherwise every thread copies its own 4-byte elements (same loop).
#include "nasg_internal.h"
#include "pipe_common.cuh"
#include "sh_math.cuh"

namespace nasg {

constexpr int SH_GROUPS = 4;    // groups of 4 basis functions
constexpr int SH_DIST = 3;      // prefetch distance in groups
constexpr int SH_HR = 2;        // header slots

// ring [4][12][PBLOCK] floats, header [SH_HR][HF][PBLOCK] floats, visibility bytes [SH_HR][4][PBLOCK]
__host__ __device__ constexpr size_t sh_pipe_smem_bytes(int HF)
{
    return (size_t)PBLOCK * 4 * (SH_GROUPS * 12 + SH_HR * HF) + (size_t)SH_HR * 4 * PBLOCK;
}
static inline bool ptr_aligned16(const void *p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }

// copies of one group item: rows 12g + r, r < 12
__device__ __forceinline__ void sh_prefetch_group(float *ring, int tid, bool coop, const float *coeffs, int64_t N, int64_t n, int g)
{
    if (coop) {
        const int j = tid & 3, q0 = tid & ~3;
        const float *src = coeffs + ((int64_t)g * 12 + j) * N + (n - j);
        float *dst = ring + (g * 12 + j) * PBLOCK + q0;
#pragma unroll
        for (int r = 0; r < 3; ++r) cp_async16(dst + 4 * r * PBLOCK, src + (int64_t)4 * r * N);
    } else {
        const float *src = coeffs + (int64_t)g * 12 * N + n;
        float *dst = ring + g * 12 * PBLOCK + tid;
#pragma unroll
        for (int r = 0; r < 12; ++r) cp_async4(dst + r * PBLOCK, src + (int64_t)r * N);
    }
}
// a [N,3] record of the quad (mean or one camera's g_colors) into a 3*PBLOCK-float header area:
// cooperative: the tile's records stay interleaved (thread t reads h[3t+i]); else planar (h[i*PBLOCK+t])
__device__ __forceinline__ void sh_prefetch_rec3(float *area, int tid, bool coop, const float *src3 /* record of Gaussian n */)
{
    if (coop) {
        const int j = tid & 3;
        if (j < 3) cp_async16(area + 3 * (tid & ~3) + 4 * j, src3 - 3 * j + 4 * j);     // record base of the quad + 4j floats
    } else {
        cp_async4(area + tid, src3); cp_async4(area + PBLOCK + tid, src3 + 1); cp_async4(area + 2 * PBLOCK + tid, src3 + 2);
    }
}
__device__ __forceinline__ float sh_rec3(const float *area, int tid, bool coop, int i)
{
    return coop ? area[3 * tid + i] : area[i * PBLOCK + tid];
}

template <int CT>
__device__ __forceinline__ void sh_directions(const float *campos, int C, float mx, float my, float mz,
                                              float (&dx)[CT], float (&dy)[CT], float (&dz)[CT], float (&idist)[CT])
{
#pragma unroll
    for (int t = 0; t < CT; ++t) {
        const int c = t < C ? t : 0;
        const float ex = mx - __ldg(campos + 3 * c), ey = my - __ldg(campos + 3 * c + 1), ez = mz - __ldg(campos + 3 * c + 2);
        const float r2 = fmaf(ex, ex, fmaf(ey, ey, ez * ez));
        float inv = rsqrtf(r2);
        inv = inv * fmaf(-0.5f * r2, inv * inv, 1.5f);
        dx[t] = ex * inv; dy[t] = ey * inv; dz[t] = ez * inv; idist[t] = inv;
    }
}

// ---- forward: colors[c,n,:] = sum_j coeffs[j,:,n] Y_j(d_cn) -------------------------------------
template <int G, int CT>
__device__ __forceinline__ void sh_fwd_group(const float *slot, const float (&dx)[CT], const float (&dy)[CT],
                                             const float (&dz)[CT], float (&col)[CT][3])
{
#pragma unroll
    for (int jj = 0; jj < 4; ++jj) {
        const float k0 = slot[(jj * 3 + 0) * PBLOCK], k1 = slot[(jj * 3 + 1) * PBLOCK], k2 = slot[(jj * 3 + 2) * PBLOCK];
#pragma unroll
        for (int t = 0; t < CT; ++t) {
            float Y = 0.f, gx, gy, gz;
            if (jj == 0) sh_term<4 * G + 0>(dx[t], dy[t], dz[t], Y, gx, gy, gz);
            if (jj == 1) sh_term<4 * G + 1>(dx[t], dy[t], dz[t], Y, gx, gy, gz);
            if (jj == 2) sh_term<4 * G + 2>(dx[t], dy[t], dz[t], Y, gx, gy, gz);
            if (jj == 3) sh_term<4 * G + 3>(dx[t], dy[t], dz[t], Y, gx, gy, gz);
            col[t][0] = fmaf(k0, Y, col[t][0]); col[t][1] = fmaf(k1, Y, col[t][1]); col[t][2] = fmaf(k2, Y, col[t][2]);
        }
    }
}

template <int CT, bool COOP>
__global__ void __launch_bounds__(PBLOCK, 4) sh_fwd_pipe_kernel(ShParams p)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    constexpr int HF = 3;
    float *ring = reinterpret_cast<float *>(smem_raw);
    float *hdr = ring + SH_GROUPS * 12 * PBLOCK;
    unsigned char *vm = reinterpret_cast<unsigned char *>(hdr + SH_HR * HF * PBLOCK);
    const int tid = threadIdx.x;
    const int64_t N = p.N, stride = (int64_t)gridDim.x * PBLOCK;
    int64_t n = (int64_t)blockIdx.x * PBLOCK + tid;
    constexpr bool coop = COOP;      // rows 16-byte aligned (checked by the launcher)
    const bool vis_cp = vis_rows_aligned(p.vis, N);

    auto prefetch_item = [&](int64_t gn, int g, int hslot) {
        if (gn < N) {
            sh_prefetch_group(ring, tid, coop, p.coeffs, N, gn, g);
            if (g == 0) {
                sh_prefetch_rec3(hdr + hslot * HF * PBLOCK, tid, coop, p.means + 3 * gn);
                if (vis_cp) prefetch_vis(vm, hslot, tid, p.vis, N, gn, p.C);
            }
        }
        cp_async_commit();
    };
#pragma unroll
    for (int j = 0; j < SH_DIST; ++j) prefetch_item(n, j, 0);

    unsigned hs = 0;
    RawMask raw = {{0u, 0u, 0u, 0u}};
    if (!vis_cp) raw = load_raw_mask(p.vis, N, n, p.C);
    for (; n - (tid & 31) < N; n += stride) {       // warp-uniform trip count: lanes past N idle (mask 0, no stores)
        const bool valid = n < N;
        RawMask raw_next = {{0u, 0u, 0u, 0u}};
        if (!vis_cp) raw_next = load_raw_mask(p.vis, N, n + stride, p.C);
        unsigned mask = 0;
        float dx[CT], dy[CT], dz[CT], idist[CT], col[CT][3];
#pragma unroll
        for (int g = 0; g < SH_GROUPS; ++g) {
            cp_async_wait<SH_DIST - 1>();       // item g (own copies) landed
            __syncwarp();                       // ... and the quad's; slot (g+3)%4 is free in every lane
            prefetch_item(n + ((g + SH_DIST) / SH_GROUPS) * stride, (g + SH_DIST) % SH_GROUPS, (hs + (g + SH_DIST) / SH_GROUPS) % SH_HR);
            if (g == 0) {
                mask = vis_cp ? staged_mask(vm, hs, tid, p.C, valid) : combine_mask(raw);
                const float *h = hdr + hs * HF * PBLOCK;
                sh_directions<CT>(p.campos, p.C, sh_rec3(h, tid, coop, 0), sh_rec3(h, tid, coop, 1), sh_rec3(h, tid, coop, 2),
                                  dx, dy, dz, idist);
#pragma unroll
                for (int t = 0; t < CT; ++t) col[t][0] = col[t][1] = col[t][2] = 0.f;
            }
            if (mask != 0) {
                const float *slot = ring + g * 12 * PBLOCK + tid;
                if (g == 0) sh_fwd_group<0, CT>(slot, dx, dy, dz, col);
                if (g == 1) sh_fwd_group<1, CT>(slot, dx, dy, dz, col);
                if (g == 2) sh_fwd_group<2, CT>(slot, dx, dy, dz, col);
                if (g == 3) sh_fwd_group<3, CT>(slot, dx, dy, dz, col);
            }
        }
#pragma unroll
        for (int t = 0; t < CT; ++t) {
            if (t < p.C && valid) {
                const bool on = mask & (1u << t);
                float *o = p.colors + ((int64_t)t * N + n) * 3;
                st_cs(o, on ? col[t][0] : 0.f); st_cs(o + 1, on ? col[t][1] : 0.f); st_cs(o + 2, on ? col[t][2] : 0.f);
            }
        }
        hs = (hs + 1) % SH_HR;
        raw = raw_next;
    }
    cp_async_wait<0>();
}

// ---- backward: g_coeffs[j,:,n] = sum_c Y_j(d_c) g_col_c;  g_d = sum_j grad Y_j (coeff_j . g_col) ----
template <int G, int CT>
__device__ __forceinline__ void sh_bwd_group(const float *slot, bool live, bool valid, float *g_coeffs, int64_t N, int64_t n,
                                             const float (&dx)[CT], const float (&dy)[CT], const float (&dz)[CT],
                                             const float (&gc)[CT][3], float (&gd)[CT][3])
{
#pragma unroll
    for (int jj = 0; jj < 4; ++jj) {
        float a0 = 0.f, a1 = 0.f, a2 = 0.f;
        if (live) {
            const float k0 = slot[(jj * 3 + 0) * PBLOCK], k1 = slot[(jj * 3 + 1) * PBLOCK], k2 = slot[(jj * 3 + 2) * PBLOCK];
#pragma unroll
            for (int t = 0; t < CT; ++t) {
                float Y = 0.f, gx = 0.f, gy = 0.f, gz = 0.f;
                if (jj == 0) sh_term<4 * G + 0>(dx[t], dy[t], dz[t], Y, gx, gy, gz);
                if (jj == 1) sh_term<4 * G + 1>(dx[t], dy[t], dz[t], Y, gx, gy, gz);
                if (jj == 2) sh_term<4 * G + 2>(dx[t], dy[t], dz[t], Y, gx, gy, gz);
                if (jj == 3) sh_term<4 * G + 3>(dx[t], dy[t], dz[t], Y, gx, gy, gz);
                a0 = fmaf(gc[t][0], Y, a0); a1 = fmaf(gc[t][1], Y, a1); a2 = fmaf(gc[t][2], Y, a2);     // gc = 0 when culled
                const float s = fmaf(k0, gc[t][0], fmaf(k1, gc[t][1], k2 * gc[t][2]));
                gd[t][0] = fmaf(s, gx, gd[t][0]); gd[t][1] = fmaf(s, gy, gd[t][1]); gd[t][2] = fmaf(s, gz, gd[t][2]);
            }
        }
        if (g_coeffs && valid) {
            float *o = g_coeffs + (int64_t)((4 * G + jj) * 3) * N + n;
            st_cs(o, a0); st_cs(o + N, a1); st_cs(o + 2 * N, a2);
        }
    }
}

// CAMGRAD: also produce this block's partial of g_campos (per-thread partial over the persistent loop, kept in
// shared memory behind the staged visibility bytes; one block sum at the end of the kernel)
template <int CT, bool COOP, bool CAMGRAD>
__global__ void __launch_bounds__(PBLOCK, 2) sh_bwd_pipe_kernel(ShParams p)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    constexpr int HF = 3 + 3 * CT;
    float *ring = reinterpret_cast<float *>(smem_raw);
    float *hdr = ring + SH_GROUPS * 12 * PBLOCK;
    unsigned char *vm = reinterpret_cast<unsigned char *>(hdr + SH_HR * HF * PBLOCK);
    const int tid = threadIdx.x;
    const int C = p.C;
    const int64_t N = p.N, stride = (int64_t)gridDim.x * PBLOCK;
    int64_t n = (int64_t)blockIdx.x * PBLOCK + tid;
    constexpr bool coop = COOP;      // rows 16-byte aligned (checked by the launcher)
    const bool vis_cp = vis_rows_aligned(p.vis, N);

    auto prefetch_item = [&](int64_t gn, int g, int hslot) {
        if (gn < N) {
            sh_prefetch_group(ring, tid, coop, p.coeffs, N, gn, g);
            if (g == 0) {
                float *h = hdr + hslot * HF * PBLOCK;
                sh_prefetch_rec3(h, tid, coop, p.means + 3 * gn);
#pragma unroll
                for (int t = 0; t < CT; ++t)
                    if (t < C) sh_prefetch_rec3(h + (3 + 3 * t) * PBLOCK, tid, coop, p.g_colors + ((int64_t)t * N + gn) * 3);
                if (vis_cp) prefetch_vis(vm, hslot, tid, p.vis, N, gn, C);
            }
        }
        cp_async_commit();
    };
#pragma unroll
    for (int j = 0; j < SH_DIST; ++j) prefetch_item(n, j, 0);

    unsigned hs = 0;
    float *hc = reinterpret_cast<float *>(vm + SH_HR * 4 * PBLOCK) + tid;       // [3 CT][PBLOCK], CAMGRAD only
    if (CAMGRAD) {
#pragma unroll
        for (int i = 0; i < 3 * CT; ++i) hc[i * PBLOCK] = 0.f;
    }
    RawMask raw = {{0u, 0u, 0u, 0u}};
    if (!vis_cp) raw = load_raw_mask(p.vis, N, n, C);
    for (; n - (tid & 31) < N; n += stride) {
        const bool valid = n < N;
        RawMask raw_next = {{0u, 0u, 0u, 0u}};
        if (!vis_cp) raw_next = load_raw_mask(p.vis, N, n + stride, C);
        unsigned mask = 0;
        float dx[CT], dy[CT], dz[CT], idist[CT], gc[CT][3], gd[CT][3];
#pragma unroll
        for (int g = 0; g < SH_GROUPS; ++g) {
            cp_async_wait<SH_DIST - 1>();
            __syncwarp();
            prefetch_item(n + ((g + SH_DIST) / SH_GROUPS) * stride, (g + SH_DIST) % SH_GROUPS, (hs + (g + SH_DIST) / SH_GROUPS) % SH_HR);
            if (g == 0) {
                mask = vis_cp ? staged_mask(vm, hs, tid, C, valid) : combine_mask(raw);
                const float *h = hdr + hs * HF * PBLOCK;
                sh_directions<CT>(p.campos, C, sh_rec3(h, tid, coop, 0), sh_rec3(h, tid, coop, 1), sh_rec3(h, tid, coop, 2),
                                  dx, dy, dz, idist);
#pragma unroll
                for (int t = 0; t < CT; ++t) {
                    const bool on = mask & (1u << t);
                    const float *hg = h + (3 + 3 * t) * PBLOCK;
                    gc[t][0] = on ? sh_rec3(hg, tid, coop, 0) : 0.f;
                    gc[t][1] = on ? sh_rec3(hg, tid, coop, 1) : 0.f;
                    gc[t][2] = on ? sh_rec3(hg, tid, coop, 2) : 0.f;
                    idist[t] = on ? idist[t] : 0.f;
                    gd[t][0] = gd[t][1] = gd[t][2] = 0.f;
                }
            }
            const float *slot = ring + g * 12 * PBLOCK + tid;
            const bool live = mask != 0;
            if (g == 0) sh_bwd_group<0, CT>(slot, live, valid, p.g_coeffs, N, n, dx, dy, dz, gc, gd);
            if (g == 1) sh_bwd_group<1, CT>(slot, live, valid, p.g_coeffs, N, n, dx, dy, dz, gc, gd);
            if (g == 2) sh_bwd_group<2, CT>(slot, live, valid, p.g_coeffs, N, n, dx, dy, dz, gc, gd);
            if (g == 3) sh_bwd_group<3, CT>(slot, live, valid, p.g_coeffs, N, n, dx, dy, dz, gc, gd);
        }
        if ((p.g_means || CAMGRAD) && valid) {        // through d = Delta/|Delta|: (I - d d^T)/|Delta|; g_campos gets minus the same
            float gm0 = 0.f, gm1 = 0.f, gm2 = 0.f;
#pragma unroll
            for (int t = 0; t < CT; ++t) {
                const float dg = fmaf(dx[t], gd[t][0], fmaf(dy[t], gd[t][1], dz[t] * gd[t][2]));
                if (CAMGRAD) {
                    const float t0 = (gd[t][0] - dx[t] * dg) * idist[t], t1 = (gd[t][1] - dy[t] * dg) * idist[t],
                                t2 = (gd[t][2] - dz[t] * dg) * idist[t];
                    gm0 += t0; gm1 += t1; gm2 += t2;
                    hc[(3 * t) * PBLOCK] -= t0; hc[(3 * t + 1) * PBLOCK] -= t1; hc[(3 * t + 2) * PBLOCK] -= t2;
                } else {
                    gm0 = fmaf(gd[t][0] - dx[t] * dg, idist[t], gm0);
                    gm1 = fmaf(gd[t][1] - dy[t] * dg, idist[t], gm1);
                    gm2 = fmaf(gd[t][2] - dz[t] * dg, idist[t], gm2);
                }
            }
            if (p.g_means) {
                float *o = p.g_means + 3 * n;
                st_cs(o, gm0); st_cs(o + 1, gm1); st_cs(o + 2, gm2);
            }
        }
        hs = (hs + 1) % SH_HR;
        raw = raw_next;
    }
    cp_async_wait<0>();
    if (CAMGRAD) {                  // block partial: warp shuffle -> shared memory -> fixed-order sum (deterministic)
        __syncthreads();            // (every thread is done with the ring: reuse its first bytes)
        float *red = reinterpret_cast<float *>(smem_raw);
        for (int t = 0; t < C; ++t)
            for (int i = 0; i < 3; ++i)
                pipe_block_sum_store(hc[(3 * t + i) * PBLOCK], red, p.cam_partial + ((int64_t)blockIdx.x * C + t) * 3 + i);
    }
}

// ---- launchers --------------------------------------------------------------------------------
template <int CT>
static cudaError_t launch_sh_fwd_pipe_c(const ShParams &p, cudaStream_t st)
{
    constexpr size_t smem = sh_pipe_smem_bytes(3);
    static int cache[2][64] = {{0}};
    const bool coop = (p.N & 3) == 0 && ptr_aligned16(p.coeffs) && ptr_aligned16(p.means);
    if (coop) sh_fwd_pipe_kernel<CT, true><<<pipe_grid(sh_fwd_pipe_kernel<CT, true>, smem, p.N, cache[1]), PBLOCK, smem, st>>>(p);
    else sh_fwd_pipe_kernel<CT, false><<<pipe_grid(sh_fwd_pipe_kernel<CT, false>, smem, p.N, cache[0]), PBLOCK, smem, st>>>(p);
    return cudaGetLastError();
}
cudaError_t launch_sh_fwd_pipe(const ShParams &p, cudaStream_t st)
{
    switch (p.C) {
    case 1: return launch_sh_fwd_pipe_c<1>(p, st);
    case 2: return launch_sh_fwd_pipe_c<2>(p, st);
    case 3: return launch_sh_fwd_pipe_c<3>(p, st);
    case 4: return launch_sh_fwd_pipe_c<4>(p, st);
    default: return cudaErrorInvalidValue;
    }
}
template <int CT>
static cudaError_t launch_sh_bwd_pipe_c(const ShParams &p, cudaStream_t st, int *grid_out)
{
    const bool camgrad = p.cam_partial != nullptr;
    const size_t smem = sh_pipe_smem_bytes(3 + 3 * CT) + (camgrad ? (size_t)PBLOCK * 4 * 3 * CT : 0);
    static int cache[4][64] = {{0}};       // per (CT, cooperative copies, g_campos) instantiation and device
    const bool coop = (p.N & 3) == 0 && ptr_aligned16(p.coeffs) && ptr_aligned16(p.means) && ptr_aligned16(p.g_colors);
    int *c = cache[(coop ? 1 : 0) + (camgrad ? 2 : 0)];
    if (camgrad) {
        if (coop) sh_bwd_pipe_kernel<CT, true, true><<<pipe_grid(sh_bwd_pipe_kernel<CT, true, true>, smem, p.N, c), PBLOCK, smem, st>>>(p);
        else sh_bwd_pipe_kernel<CT, false, true><<<pipe_grid(sh_bwd_pipe_kernel<CT, false, true>, smem, p.N, c), PBLOCK, smem, st>>>(p);
    } else {
        if (coop) sh_bwd_pipe_kernel<CT, true, false><<<pipe_grid(sh_bwd_pipe_kernel<CT, true, false>, smem, p.N, c), PBLOCK, smem, st>>>(p);
        else sh_bwd_pipe_kernel<CT, false, false><<<pipe_grid(sh_bwd_pipe_kernel<CT, false, false>, smem, p.N, c), PBLOCK, smem, st>>>(p);
    }
    int dev = 0;
    cudaGetDevice(&dev);
    const int64_t need = (p.N + PBLOCK - 1) / PBLOCK;
    const int resident = c[(dev >= 0 && dev < 64) ? dev : 0];
    *grid_out = (int)(need < resident ? need : resident);       // = the grid just launched (rows of cam_partial written)
    return cudaGetLastError();
}
cudaError_t launch_sh_bwd_pipe(const ShParams &p, cudaStream_t st, int *grid_out)
{
    switch (p.C) {
    case 1: return launch_sh_bwd_pipe_c<1>(p, st, grid_out);
    case 2: return launch_sh_bwd_pipe_c<2>(p, st, grid_out);
    case 3: return launch_sh_bwd_pipe_c<3>(p, st, grid_out);
    case 4: return launch_sh_bwd_pipe_c<4>(p, st, grid_out);
    default: return cudaErrorInvalidValue;
    }
}

} // namespace nasg
