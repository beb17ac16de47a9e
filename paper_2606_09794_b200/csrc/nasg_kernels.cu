// nasg_kernels.cu — sm_100a kernels of the NASGabor path and the host-side launchers.
//
// Mapping: one thread per Gaussian, lobes unrolled per compile-time K, cameras in
// register tiles of CT (1 or 4). Parameters are structure-of-arrays: quat/shape are float4 groups
// (one 128-bit coalesced load each), amp/dc planar rows. The path is HBM-bound for K <= 4
// (algorithmic bytes in DESIGN.md §7), so nothing is saved between forward and backward: the
// backward recomputes the lobe values. Every gradient element is written once by its own thread;
// the only cross-thread term, g_campos, is a warp-shuffle -> shared-memory -> second-stage reduction.
#include "nasg_internal.h"
#include "nasg_math.cuh"

namespace nasg {

constexpr int BLOCK = 256;

__device__ __forceinline__ float4 ldg4(const float *base, int64_t idx)
{
    return __ldg(reinterpret_cast<const float4 *>(base) + idx);
}

// ---------------------------------------------------------------------------------------------
// forward: colors[c,n,:] = c0 + sum_l w_l G_l(d_cn)           eq.(6), eq.(9), eq.(10)
// ---------------------------------------------------------------------------------------------
template <int K, int CT, int MODE>
__global__ void __launch_bounds__(BLOCK, 2) nasg_fwd_kernel(FwdParams p)
{
    const int64_t N = p.N;
    const int64_t n = (int64_t)blockIdx.x * BLOCK + threadIdx.x;
    if (n >= N) return;
    const float mx = __ldg(p.means + 3 * n), my = __ldg(p.means + 3 * n + 1), mz = __ldg(p.means + 3 * n + 2);
    const float dc0 = __ldg(p.dc + n), dc1 = __ldg(p.dc + N + n), dc2 = __ldg(p.dc + 2 * N + n);

    for (int c0 = 0; c0 < p.C; c0 += CT) {
        float dx[CT], dy[CT], dz[CT], col[CT][3];
        unsigned mask = 0;
#pragma unroll
        for (int t = 0; t < CT; ++t) {
            const int c = c0 + t;
            bool on = c < p.C;
            if (on && p.vis) on = p.vis[(int64_t)c * N + n] != 0;
            if (on) {
                mask |= 1u << t;
                float ex = mx - __ldg(p.campos + 3 * c), ey = my - __ldg(p.campos + 3 * c + 1),
                      ez = mz - __ldg(p.campos + 3 * c + 2);
                float r2 = fmaf(ex, ex, fmaf(ey, ey, ez * ez));
                float inv = f_rsqrt(r2);
                inv = inv * fmaf(-0.5f * r2, inv * inv, 1.5f);        // Newton step: d accurate to 1 ulp
                dx[t] = ex * inv; dy[t] = ey * inv; dz[t] = ez * inv;
            } else {
                dx[t] = 0.f; dy[t] = 0.f; dz[t] = 1.f;
            }
            col[t][0] = dc0; col[t][1] = dc1; col[t][2] = dc2;
        }
        if (mask != 0) {
#pragma unroll
            for (int l = 0; l < K; ++l) {
                const float4 q = ldg4(p.quat, (int64_t)l * N + n);
                const float4 sp = ldg4(p.shape, (int64_t)l * N + n);
                const float w0 = __ldg(p.amp + ((int64_t)l * 3 + 0) * N + n);
                const float w1 = __ldg(p.amp + ((int64_t)l * 3 + 1) * N + n);
                const float w2 = __ldg(p.amp + ((int64_t)l * 3 + 2) * N + n);
                Lobe L; LobeBwd B;
                lobe_setup<MODE, false>(q, sp, L, B);
#pragma unroll
                for (int t = 0; t < CT; ++t) {
                    if (mask & (1u << t)) {
                        EvalTerms T;
                        const float G = lobe_eval<false, MODE != 2>(L, dx[t], dy[t], dz[t], T);
                        col[t][0] = fmaf(w0, G, col[t][0]);
                        col[t][1] = fmaf(w1, G, col[t][1]);
                        col[t][2] = fmaf(w2, G, col[t][2]);
                    }
                }
            }
        }
#pragma unroll
        for (int t = 0; t < CT; ++t) {
            const int c = c0 + t;
            if (c < p.C) {
                const bool on = mask & (1u << t);
                float *o = p.colors + ((int64_t)c * N + n) * 3;
                o[0] = on ? col[t][0] : 0.f; o[1] = on ? col[t][1] : 0.f; o[2] = on ? col[t][2] : 0.f;
            }
        }
    }
}

// ---------------------------------------------------------------------------------------------
// backward
// ---------------------------------------------------------------------------------------------
// Sum `v` over the block and let thread 0 store it to *dst. All threads of the block must call.
__device__ __forceinline__ void block_sum_store(float v, float *smem, float *dst)
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
        for (int w = 0; w < BLOCK / 32; ++w) s += smem[w];
        *dst = s;
    }
}

template <int K, int CT, int MODE, bool CAMGRAD>
__global__ void __launch_bounds__(BLOCK, 2) nasg_bwd_kernel(BwdParams p)
{
    __shared__ float red[BLOCK / 32];
    const int64_t N = p.N;
    const int64_t n = (int64_t)blockIdx.x * BLOCK + threadIdx.x;
    const bool valid = n < N;
    if (!CAMGRAD && !valid) return;
    float mx = 0.f, my = 0.f, mz = 0.f;
    if (valid) { mx = __ldg(p.means + 3 * n); my = __ldg(p.means + 3 * n + 1); mz = __ldg(p.means + 3 * n + 2); }

    for (int c0 = 0; c0 < p.C; c0 += CT) {
        const bool first = c0 == 0;         // first camera tile stores, later tiles accumulate (C > CT only)
        float dx[CT], dy[CT], dz[CT], idist[CT], gc[CT][3], gd[CT][3];
        unsigned mask = 0;
        float gdc0 = 0.f, gdc1 = 0.f, gdc2 = 0.f;
#pragma unroll
        for (int t = 0; t < CT; ++t) {
            const int c = c0 + t;
            bool on = valid && c < p.C;
            if (on && p.vis) on = p.vis[(int64_t)c * N + n] != 0;
            gd[t][0] = gd[t][1] = gd[t][2] = 0.f;
            if (on) {
                mask |= 1u << t;
                float ex = mx - __ldg(p.campos + 3 * c), ey = my - __ldg(p.campos + 3 * c + 1),
                      ez = mz - __ldg(p.campos + 3 * c + 2);
                float r2 = fmaf(ex, ex, fmaf(ey, ey, ez * ez));
                float inv = f_rsqrt(r2);
                inv = inv * fmaf(-0.5f * r2, inv * inv, 1.5f);
                dx[t] = ex * inv; dy[t] = ey * inv; dz[t] = ez * inv; idist[t] = inv;
                const float *g = p.g_colors + ((int64_t)c * N + n) * 3;
                gc[t][0] = __ldg(g); gc[t][1] = __ldg(g + 1); gc[t][2] = __ldg(g + 2);
                gdc0 += gc[t][0]; gdc1 += gc[t][1]; gdc2 += gc[t][2];
            } else {
                dx[t] = 0.f; dy[t] = 0.f; dz[t] = 1.f; idist[t] = 0.f;
                gc[t][0] = gc[t][1] = gc[t][2] = 0.f;
            }
        }
        if (valid && p.g_dc) {                                   // B5: g_c0 = sum_c vis g_col
            if (!first) { gdc0 += p.g_dc[n]; gdc1 += p.g_dc[N + n]; gdc2 += p.g_dc[2 * N + n]; }
            p.g_dc[n] = gdc0; p.g_dc[N + n] = gdc1; p.g_dc[2 * N + n] = gdc2;
        }

        if (valid && (mask != 0 || first)) {
#pragma unroll
            for (int l = 0; l < K; ++l) {
                const int64_t ln = (int64_t)l * N + n;
                float gq[4] = {0.f, 0.f, 0.f, 0.f}, gs[4] = {0.f, 0.f, 0.f, 0.f}, gw[3] = {0.f, 0.f, 0.f};
                if (mask != 0) {
                    const float4 q = ldg4(p.quat, ln);
                    const float4 sp = ldg4(p.shape, ln);
                    const float w0 = __ldg(p.amp + ((int64_t)l * 3 + 0) * N + n);
                    const float w1 = __ldg(p.amp + ((int64_t)l * 3 + 1) * N + n);
                    const float w2 = __ldg(p.amp + ((int64_t)l * 3 + 2) * N + n);
                    Lobe L; LobeBwd B;
                    lobe_setup<MODE, true>(q, sp, L, B);
                    float gX0 = 0.f, gX1 = 0.f, gX2 = 0.f, gZ0 = 0.f, gZ1 = 0.f, gZ2 = 0.f;
                    float S0 = 0.f, S1 = 0.f, S2 = 0.f, Sk = 0.f, Sp = 0.f;
#pragma unroll
                    for (int t = 0; t < CT; ++t) {
                        if (mask & (1u << t)) {
                            EvalTerms T;
                            const float G = lobe_eval<true, MODE != 2>(L, dx[t], dy[t], dz[t], T);
                            const float gG = fmaf(gc[t][0], w0, fmaf(gc[t][1], w1, gc[t][2] * w2)); // dL/dG, eq.(6)
                            gw[0] = fmaf(gc[t][0], G, gw[0]);
                            gw[1] = fmaf(gc[t][1], G, gw[1]);
                            gw[2] = fmaf(gc[t][2], G, gw[2]);
                            const float gGG = gG * G;
                            // ln(pE) = 2 lambda (kappa' - 1) + tau ln kappa, kappa' = kappa^(1+tau)
                            const float A_tau = T.Lk * fmaf(B.lam2, T.kp, 1.0f);                    // d/d tau
                            const float A_kap2 = fmaf(B.lam2 * (1.0f + T.tau), T.kp, T.tau) * T.inv_2kappa; // (d/d kappa)/2
                            const float B1 = 2.0f * gGG * A_tau * T.inv_s2;
                            const float hs = gG * T.Gh * T.sn;                                       // carrier terms, eqs.(59),(65)
                            const float gu = fmaf(B1 * L.a, T.u, -hs * B.k);                         // gG dG/du, tau_u = 2 a u / s^2 (eq.57)
                            const float gv = fmaf(B1 * T.tau, T.v, gGG * A_kap2);                    // gG dG/dv, tau_v = 2 tau v / s^2 (eq.61)
                            S0 += gGG;
                            S1 = fmaf(gGG, T.em1, S1);
                            S2 = fmaf(B1, T.uu, S2);                                                 // 2 gGG A_tau c2 (halved below)
                            Sk = fmaf(hs, T.u, Sk);
                            Sp += hs;
                            gX0 = fmaf(gu, dx[t], gX0); gX1 = fmaf(gu, dy[t], gX1); gX2 = fmaf(gu, dz[t], gX2);  // eq.(60)
                            gZ0 = fmaf(gv, dx[t], gZ0); gZ1 = fmaf(gv, dy[t], gZ1); gZ2 = fmaf(gv, dz[t], gZ2);  // eq.(64)
                            gd[t][0] = fmaf(gu, L.Xx, fmaf(gv, L.Zx, gd[t][0]));
                            gd[t][1] = fmaf(gu, L.Xy, fmaf(gv, L.Zy, gd[t][1]));
                            gd[t][2] = fmaf(gu, L.Xz, fmaf(gv, L.Zz, gd[t][2]));
                        }
                    }
                    // shape: (lambda, a) = (e^{l2}, e^{l1-l2} - 1)
                    gs[0] = fmaf(0.5f * S2, B.one_pa, -S0 * B.nA);
                    gs[1] = fmaf(B.lam2, S1, -S0 * B.nL) - gs[0];
                    gs[2] = -fmaf(S0, B.nk, Sk);
                    gs[3] = -Sp;
                    // frame: transpose Jacobian of columns X and Z of R(qhat), then qhat = q/|q|
                    const float w = B.qw, x = B.qx, y = B.qy, z = B.qz;
                    float a0 = 2.0f * (z * gX1 - y * gX2 + y * gZ0 - x * gZ1);
                    float a1 = 2.0f * (y * gX1 + z * gX2 + z * gZ0 - w * gZ1) - 4.0f * x * gZ2;
                    float a2 = 2.0f * (x * gX1 - w * gX2 + w * gZ0 + z * gZ1) - 4.0f * y * (gX0 + gZ2);
                    float a3 = 2.0f * (w * gX1 + x * gX2 + x * gZ0 + y * gZ1) - 4.0f * z * gX0;
                    const float dot = w * a0 + x * a1 + y * a2 + z * a3;
                    gq[0] = (a0 - w * dot) * B.inv_qn; gq[1] = (a1 - x * dot) * B.inv_qn;
                    gq[2] = (a2 - y * dot) * B.inv_qn; gq[3] = (a3 - z * dot) * B.inv_qn;
                }
                if (p.g_quat) {
                    float4 *o = reinterpret_cast<float4 *>(p.g_quat) + ln;
                    float4 val = make_float4(gq[0], gq[1], gq[2], gq[3]);
                    if (!first) { float4 old = *o; val.x += old.x; val.y += old.y; val.z += old.z; val.w += old.w; }
                    *o = val;
                }
                if (p.g_shape) {
                    float4 *o = reinterpret_cast<float4 *>(p.g_shape) + ln;
                    float4 val = make_float4(gs[0], gs[1], gs[2], gs[3]);
                    if (!first) { float4 old = *o; val.x += old.x; val.y += old.y; val.z += old.z; val.w += old.w; }
                    *o = val;
                }
                if (p.g_amp) {
#pragma unroll
                    for (int ch = 0; ch < 3; ++ch) {
                        float *o = p.g_amp + ((int64_t)l * 3 + ch) * N + n;
                        *o = first ? gw[ch] : *o + gw[ch];
                    }
                }
            }
        }

        // B3: through d = Delta/|Delta|:  g_m += (g_d - d (d.g_d))/|Delta|, g_campos -= same
        float gm0 = 0.f, gm1 = 0.f, gm2 = 0.f;
#pragma unroll
        for (int t = 0; t < CT; ++t) {
            const float dg = fmaf(dx[t], gd[t][0], fmaf(dy[t], gd[t][1], dz[t] * gd[t][2]));
            const float t0 = (gd[t][0] - dx[t] * dg) * idist[t];
            const float t1 = (gd[t][1] - dy[t] * dg) * idist[t];
            const float t2 = (gd[t][2] - dz[t] * dg) * idist[t];
            gm0 += t0; gm1 += t1; gm2 += t2;
            if (CAMGRAD) {
                const int c = c0 + t;
                if (c < p.C) {      // uniform across the block
                    float *dst = p.cam_partial + ((int64_t)blockIdx.x * p.C + c) * 3;
                    block_sum_store(-t0, red, dst);
                    block_sum_store(-t1, red, dst + 1);
                    block_sum_store(-t2, red, dst + 2);
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

// second stage of g_campos: out[j] = sum_b partial[b*stride + j]; one block per j, fixed order.
__global__ void __launch_bounds__(BLOCK) campos_reduce_kernel(const float *partial, int64_t nblocks,
                                                              int stride, float *out)
{
    __shared__ float sm[BLOCK];
    const int j = blockIdx.x;
    float s = 0.f;
    for (int64_t b = threadIdx.x; b < nblocks; b += BLOCK) s += partial[b * stride + j];
    sm[threadIdx.x] = s;
    __syncthreads();
    for (int o = BLOCK / 2; o > 0; o >>= 1) {
        if (threadIdx.x < o) sm[threadIdx.x] += sm[threadIdx.x + o];
        __syncthreads();
    }
    if (threadIdx.x == 0) out[j] = sm[0];
}

#ifndef NASG_HOSTSIM   // (the launchers use <<<>>>; a host-only build of the kernel bodies skips them)
// ---------------------------------------------------------------------------------------------
// launchers
// ---------------------------------------------------------------------------------------------
int64_t grid_blocks(int64_t N) { return (N + BLOCK - 1) / BLOCK; }

template <int K, int CT>
static cudaError_t launch_fwd_kc(const FwdParams &p, int mode, cudaStream_t st)
{
    const dim3 grid((unsigned)grid_blocks(p.N)), block(BLOCK);
    if (mode == 1) nasg_fwd_kernel<K, CT, 1><<<grid, block, 0, st>>>(p);
    else if (mode == 0) nasg_fwd_kernel<K, CT, 0><<<grid, block, 0, st>>>(p);
    else nasg_fwd_kernel<K, CT, 2><<<grid, block, 0, st>>>(p);
    return cudaGetLastError();
}
template <int K>
static cudaError_t launch_fwd_k(const FwdParams &p, int mode, cudaStream_t st)
{
    return p.C == 1 ? launch_fwd_kc<K, 1>(p, mode, st) : launch_fwd_kc<K, 4>(p, mode, st);
}
cudaError_t launch_nasg_fwd(const FwdParams &p, int K, int mode, cudaStream_t st)
{
    switch (K) {
    case 1: return launch_fwd_k<1>(p, mode, st);
    case 2: return launch_fwd_k<2>(p, mode, st);
    case 3: return launch_fwd_k<3>(p, mode, st);
    case 4: return launch_fwd_k<4>(p, mode, st);
    case 5: return launch_fwd_k<5>(p, mode, st);
    case 8: return launch_fwd_k<8>(p, mode, st);
    default: return cudaErrorInvalidValue;
    }
}

template <int K, int CT, bool CAMGRAD>
static cudaError_t launch_bwd_kcg(const BwdParams &p, int mode, cudaStream_t st)
{
    const dim3 grid((unsigned)grid_blocks(p.N)), block(BLOCK);
    if (mode == 1) nasg_bwd_kernel<K, CT, 1, CAMGRAD><<<grid, block, 0, st>>>(p);
    else if (mode == 0) nasg_bwd_kernel<K, CT, 0, CAMGRAD><<<grid, block, 0, st>>>(p);
    else nasg_bwd_kernel<K, CT, 2, CAMGRAD><<<grid, block, 0, st>>>(p);
    return cudaGetLastError();
}
template <int K>
static cudaError_t launch_bwd_k(const BwdParams &p, int mode, cudaStream_t st)
{
    const bool cam = p.cam_partial != nullptr;
    if (p.C == 1) return cam ? launch_bwd_kcg<K, 1, true>(p, mode, st) : launch_bwd_kcg<K, 1, false>(p, mode, st);
    return cam ? launch_bwd_kcg<K, 4, true>(p, mode, st) : launch_bwd_kcg<K, 4, false>(p, mode, st);
}
cudaError_t launch_nasg_bwd(const BwdParams &p, int K, int mode, cudaStream_t st)
{
    switch (K) {
    case 1: return launch_bwd_k<1>(p, mode, st);
    case 2: return launch_bwd_k<2>(p, mode, st);
    case 3: return launch_bwd_k<3>(p, mode, st);
    case 4: return launch_bwd_k<4>(p, mode, st);
    case 5: return launch_bwd_k<5>(p, mode, st);
    case 8: return launch_bwd_k<8>(p, mode, st);
    default: return cudaErrorInvalidValue;
    }
}

cudaError_t launch_campos_reduce(const float *partial, int64_t nblocks, int C, float *out, cudaStream_t st)
{
    campos_reduce_kernel<<<3 * C, BLOCK, 0, st>>>(partial, nblocks, 3 * C, out);
    return cudaGetLastError();
}
#endif // NASG_HOSTSIM

} // namespace nasg
