// sh_kernels.cu — comparison path: real spherical harmonics of degree 3 (eq.(5)),
// built with the same skeleton as the NASGabor kernels (one thread per Gaussian, planar coefficient
// rows [16,3,N], cameras in register tiles, gradients written once, no atomics).
// Basis convention: DESIGN.md reading R15 (j = l^2+l+m, Condon-Shortley sign kept).
#include "nasg_internal.h"
#include "sh_math.cuh"

namespace nasg {

constexpr int SH_BLOCK = 256;
constexpr int SH_CT = 4;

struct ShCams {
    float dx[SH_CT], dy[SH_CT], dz[SH_CT], idist[SH_CT];
    unsigned mask;
};

__device__ __forceinline__ void sh_load_cams(const ShParams &p, int64_t n, bool valid, int c0, float mx,
                                             float my, float mz, ShCams &cm)
{
    cm.mask = 0;
#pragma unroll
    for (int t = 0; t < SH_CT; ++t) {
        const int c = c0 + t;
        bool on = valid && c < p.C;
        if (on && p.vis) on = p.vis[(int64_t)c * p.N + n] != 0;
        if (on) {
            cm.mask |= 1u << t;
            float ex = mx - __ldg(p.campos + 3 * c), ey = my - __ldg(p.campos + 3 * c + 1),
                  ez = mz - __ldg(p.campos + 3 * c + 2);
            float r2 = fmaf(ex, ex, fmaf(ey, ey, ez * ez));
            float inv = rsqrtf(r2);
            inv = inv * fmaf(-0.5f * r2, inv * inv, 1.5f);
            cm.dx[t] = ex * inv; cm.dy[t] = ey * inv; cm.dz[t] = ez * inv; cm.idist[t] = inv;
        } else {
            cm.dx[t] = 0.f; cm.dy[t] = 0.f; cm.dz[t] = 1.f; cm.idist[t] = 0.f;
        }
    }
}

template <int J>
__device__ __forceinline__ void sh_fwd_terms(const ShParams &p, int64_t n, const ShCams &cm, float (&col)[SH_CT][3])
{
    const int64_t N = p.N;
    const float k0 = __ldg(p.coeffs + ((int64_t)J * 3 + 0) * N + n);
    const float k1 = __ldg(p.coeffs + ((int64_t)J * 3 + 1) * N + n);
    const float k2 = __ldg(p.coeffs + ((int64_t)J * 3 + 2) * N + n);
#pragma unroll
    for (int t = 0; t < SH_CT; ++t) {
        float Y, gx, gy, gz;
        sh_term<J>(cm.dx[t], cm.dy[t], cm.dz[t], Y, gx, gy, gz);
        col[t][0] = fmaf(k0, Y, col[t][0]); col[t][1] = fmaf(k1, Y, col[t][1]); col[t][2] = fmaf(k2, Y, col[t][2]);
    }
    if constexpr (J + 1 < 16) sh_fwd_terms<J + 1>(p, n, cm, col);
}

__global__ void __launch_bounds__(SH_BLOCK, 2) sh_fwd_kernel(ShParams p)
{
    const int64_t N = p.N;
    const int64_t n = (int64_t)blockIdx.x * SH_BLOCK + threadIdx.x;
    if (n >= N) return;
    const float mx = __ldg(p.means + 3 * n), my = __ldg(p.means + 3 * n + 1), mz = __ldg(p.means + 3 * n + 2);
    for (int c0 = 0; c0 < p.C; c0 += SH_CT) {
        ShCams cm;
        sh_load_cams(p, n, true, c0, mx, my, mz, cm);
        float col[SH_CT][3];
#pragma unroll
        for (int t = 0; t < SH_CT; ++t) col[t][0] = col[t][1] = col[t][2] = 0.f;
        if (cm.mask != 0) sh_fwd_terms<0>(p, n, cm, col);
#pragma unroll
        for (int t = 0; t < SH_CT; ++t) {
            const int c = c0 + t;
            if (c < p.C) {
                const bool on = cm.mask & (1u << t);
                float *o = p.colors + ((int64_t)c * N + n) * 3;
                o[0] = on ? col[t][0] : 0.f; o[1] = on ? col[t][1] : 0.f; o[2] = on ? col[t][2] : 0.f;
            }
        }
    }
}

template <int J>
__device__ __forceinline__ void sh_bwd_terms(const ShParams &p, int64_t n, bool first, const ShCams &cm,
                                             const float (&gc)[SH_CT][3], float (&gd)[SH_CT][3])
{
    const int64_t N = p.N;
    float a0 = 0.f, a1 = 0.f, a2 = 0.f;
    if (cm.mask != 0) {
        const float k0 = __ldg(p.coeffs + ((int64_t)J * 3 + 0) * N + n);
        const float k1 = __ldg(p.coeffs + ((int64_t)J * 3 + 1) * N + n);
        const float k2 = __ldg(p.coeffs + ((int64_t)J * 3 + 2) * N + n);
#pragma unroll
        for (int t = 0; t < SH_CT; ++t) {
            float Y, gx, gy, gz;
            sh_term<J>(cm.dx[t], cm.dy[t], cm.dz[t], Y, gx, gy, gz);
            a0 = fmaf(gc[t][0], Y, a0); a1 = fmaf(gc[t][1], Y, a1); a2 = fmaf(gc[t][2], Y, a2);   // gc is 0 when culled
            const float s = fmaf(k0, gc[t][0], fmaf(k1, gc[t][1], k2 * gc[t][2]));
            gd[t][0] = fmaf(s, gx, gd[t][0]); gd[t][1] = fmaf(s, gy, gd[t][1]); gd[t][2] = fmaf(s, gz, gd[t][2]);
        }
    }
    if (p.g_coeffs && (first || cm.mask != 0)) {
        float *o0 = p.g_coeffs + ((int64_t)J * 3 + 0) * N + n, *o1 = o0 + N, *o2 = o1 + N;
        if (!first) { a0 += *o0; a1 += *o1; a2 += *o2; }
        *o0 = a0; *o1 = a1; *o2 = a2;
    }
    if constexpr (J + 1 < 16) sh_bwd_terms<J + 1>(p, n, first, cm, gc, gd);
}

__device__ __forceinline__ void sh_block_sum_store(float v, float *smem, float *dst)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    __syncthreads();
    if (lane == 0) smem[warp] = v;
    __syncthreads();
    if (threadIdx.x == 0) {
        float s = 0.f;
#pragma unroll
        for (int w = 0; w < SH_BLOCK / 32; ++w) s += smem[w];
        *dst = s;
    }
}

template <bool CAMGRAD>
__global__ void __launch_bounds__(SH_BLOCK, 2) sh_bwd_kernel(ShParams p)
{
    __shared__ float red[SH_BLOCK / 32];
    const int64_t N = p.N;
    const int64_t n = (int64_t)blockIdx.x * SH_BLOCK + threadIdx.x;
    const bool valid = n < N;
    if (!CAMGRAD && !valid) return;
    float mx = 0.f, my = 0.f, mz = 0.f;
    if (valid) { mx = __ldg(p.means + 3 * n); my = __ldg(p.means + 3 * n + 1); mz = __ldg(p.means + 3 * n + 2); }
    for (int c0 = 0; c0 < p.C; c0 += SH_CT) {
        const bool first = c0 == 0;
        ShCams cm;
        sh_load_cams(p, n, valid, c0, mx, my, mz, cm);
        float gc[SH_CT][3], gd[SH_CT][3];
#pragma unroll
        for (int t = 0; t < SH_CT; ++t) {
            gd[t][0] = gd[t][1] = gd[t][2] = 0.f;
            if (cm.mask & (1u << t)) {
                const float *g = p.g_colors + ((int64_t)(c0 + t) * N + n) * 3;
                gc[t][0] = __ldg(g); gc[t][1] = __ldg(g + 1); gc[t][2] = __ldg(g + 2);
            } else {
                gc[t][0] = gc[t][1] = gc[t][2] = 0.f;
            }
        }
        if (valid) sh_bwd_terms<0>(p, n, first, cm, gc, gd);
        float gm0 = 0.f, gm1 = 0.f, gm2 = 0.f;
#pragma unroll
        for (int t = 0; t < SH_CT; ++t) {
            const float dg = fmaf(cm.dx[t], gd[t][0], fmaf(cm.dy[t], gd[t][1], cm.dz[t] * gd[t][2]));
            const float t0 = (gd[t][0] - cm.dx[t] * dg) * cm.idist[t];
            const float t1 = (gd[t][1] - cm.dy[t] * dg) * cm.idist[t];
            const float t2 = (gd[t][2] - cm.dz[t] * dg) * cm.idist[t];
            gm0 += t0; gm1 += t1; gm2 += t2;
            if (CAMGRAD) {
                const int c = c0 + t;
                if (c < p.C) {
                    float *dst = p.cam_partial + ((int64_t)blockIdx.x * p.C + c) * 3;
                    sh_block_sum_store(-t0, red, dst);
                    sh_block_sum_store(-t1, red, dst + 1);
                    sh_block_sum_store(-t2, red, dst + 2);
                }
            }
        }
        if (valid && p.g_means) {
            float *o = p.g_means + 3 * n;
            if (!first) { gm0 += o[0]; gm1 += o[1]; gm2 += o[2]; }
            o[0] = gm0; o[1] = gm1; o[2] = gm2;
        }
    }
}

cudaError_t launch_sh_fwd(const ShParams &p, cudaStream_t st)
{
    sh_fwd_kernel<<<(unsigned)((p.N + SH_BLOCK - 1) / SH_BLOCK), SH_BLOCK, 0, st>>>(p);
    return cudaGetLastError();
}
cudaError_t launch_sh_bwd(const ShParams &p, cudaStream_t st)
{
    const unsigned grid = (unsigned)((p.N + SH_BLOCK - 1) / SH_BLOCK);
    if (p.cam_partial) sh_bwd_kernel<true><<<grid, SH_BLOCK, 0, st>>>(p);
    else sh_bwd_kernel<false><<<grid, SH_BLOCK, 0, st>>>(p);
    return cudaGetLastError();
}

} // namespace nasg
