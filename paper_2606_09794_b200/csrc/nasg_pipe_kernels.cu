// nasg_pipe_kernels.cu — the fast path of the NASGabor kernels for C <= 4 cameras (sm_100a).
//
// Same arithmetic as nasg_kernels.cu (nasg_math.cuh), different data movement. The generic kernels
// load a lobe's parameters and immediately use them, so with 16 resident warps per SM (128 registers
// per thread) every warp sleeps a full DRAM latency per lobe (ncu: 45% long-scoreboard stalls,
// profiles/). Here each thread is persistent and streams its lobes through a private shared-memory
// ring filled by cp.async (LDGSTS) DIST lobes ahead of use: the bytes in flight per SM are
// DIST * 44 B * 512 threads ~ 66 KB, independent of occupancy and without spending registers.
// A thread only ever reads the ring slots it filled itself, so no block barrier is needed:
// cp.async.wait_group orders a thread's own copies.
//
// Work assignment: thread t of block b owns Gaussians n = (i * gridDim.x + b) * 256 + t, i = 0,1,...
// (coalesced across the warp: quat/shape rows are float4 groups, amp/dc rows are planar).
// Item stream of a thread: (Gaussian i, lobe l) in order; item j lives in ring slot j % RING; the
// per-Gaussian header (mean, dc or g_colors) travels with lobe 0 into header slot i % HR.
#include "nasg_internal.h"
#include "nasg_math.cuh"
#include "pipe_common.cuh"

namespace nasg {

constexpr int RING = 4;     // lobe slots per thread
constexpr int DIST = 3;     // prefetch distance in lobes

template <int K> struct PipeCfg {
    static constexpr int HR = (K <= 2) ? 4 : 2;          // header slots: ceil(DIST/K)+1 rounded to a power of 2
    static constexpr bool STATIC_SLOTS = (K % RING) == 0; // lobe l always lives in ring slot l % RING
};

// shared-memory carve-up for one block
struct Ring {
    float4 *q;      // [RING][PBLOCK]
    float4 *s;      // [RING][PBLOCK]
    float *w;       // [RING][3][PBLOCK]
    float *h;       // [HR][HF][PBLOCK]   HF = header floats
};
__host__ __device__ constexpr size_t pipe_smem_bytes(int HR, int HF)
{
    return (size_t)PBLOCK * (RING * (16 + 16 + 12) + HR * HF * 4);
}
__device__ __forceinline__ Ring carve(unsigned char *raw)
{
    Ring r;
    r.q = reinterpret_cast<float4 *>(raw);
    r.s = r.q + RING * PBLOCK;
    r.w = reinterpret_cast<float *>(r.s + RING * PBLOCK);
    r.h = r.w + RING * 3 * PBLOCK;
    return r;
}

// issue the copies of one lobe item (and nothing if the Gaussian is out of range); always commits
__device__ __forceinline__ void prefetch_lobe(const Ring &r, int slot, int tid, const float *quat, const float *shape,
                                              const float *amp, int64_t N, int64_t n, int l)
{
    if (n < N) {
        const int64_t ln = (int64_t)l * N + n;
        cp_async16(&r.q[slot * PBLOCK + tid], quat + 4 * ln);
        cp_async16(&r.s[slot * PBLOCK + tid], shape + 4 * ln);
        const float *a = amp + (int64_t)l * 3 * N + n;
        cp_async4(&r.w[(slot * 3 + 0) * PBLOCK + tid], a);
        cp_async4(&r.w[(slot * 3 + 1) * PBLOCK + tid], a + N);
        cp_async4(&r.w[(slot * 3 + 2) * PBLOCK + tid], a + 2 * N);
    }
}

// ---------------------------------------------------------------------------------------------
// forward
// ---------------------------------------------------------------------------------------------
template <int K, int CT, bool EXACT>
__global__ void __launch_bounds__(PBLOCK, CT >= 3 ? 3 : 4) nasg_fwd_pipe_kernel(FwdParams p)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    constexpr int HR = PipeCfg<K>::HR, HF = 6;
    const Ring r = carve(smem_raw);
    const int tid = threadIdx.x;
    const int64_t N = p.N, stride = (int64_t)gridDim.x * PBLOCK;
    int64_t n = (int64_t)blockIdx.x * PBLOCK + tid;

    auto prefetch_item = [&](int64_t gn, int l, int slot, int hslot) {
        prefetch_lobe(r, slot, tid, p.quat, p.shape, p.amp, N, gn, l);
        if (l == 0 && gn < N) {
            float *h = r.h + (hslot * HF) * PBLOCK + tid;
            cp_async4(h, p.means + 3 * gn); cp_async4(h + PBLOCK, p.means + 3 * gn + 1);
            cp_async4(h + 2 * PBLOCK, p.means + 3 * gn + 2);
            cp_async4(h + 3 * PBLOCK, p.dc + gn); cp_async4(h + 4 * PBLOCK, p.dc + N + gn);
            cp_async4(h + 5 * PBLOCK, p.dc + 2 * N + gn);
        }
        cp_async_commit();
    };
#pragma unroll
    for (int j = 0; j < DIST; ++j) prefetch_item(n + (j / K) * stride, j % K, j % RING, (j / K) % HR);

    unsigned sbase = 0, hs = 0;                  // ring slot of lobe 0 / header slot of the current Gaussian
    unsigned mask = load_mask(p.vis, N, n, p.C);
    for (; n < N; n += stride) {
        const unsigned mask_next = load_mask(p.vis, N, n + stride, p.C);     // lands during this Gaussian
        float dx[CT], dy[CT], dz[CT], col[CT][3];
#pragma unroll
        for (int l = 0; l < K; ++l) {
            prefetch_item(n + ((l + DIST) / K) * stride, (l + DIST) % K, ((PipeCfg<K>::STATIC_SLOTS ? 0u : sbase) + (l + DIST) % RING) % RING,
                          (hs + (l + DIST) / K) % HR);
            cp_async_wait<DIST>();
            if (l == 0) {
                const float *h = r.h + (hs * HF) * PBLOCK + tid;
                const float mx = h[0], my = h[PBLOCK], mz = h[2 * PBLOCK];
                const float dc0 = h[3 * PBLOCK], dc1 = h[4 * PBLOCK], dc2 = h[5 * PBLOCK];
#pragma unroll
                for (int t = 0; t < CT; ++t) {
                    const int c = t < p.C ? t : 0;
                    const float ex = mx - __ldg(p.campos + 3 * c), ey = my - __ldg(p.campos + 3 * c + 1),
                                ez = mz - __ldg(p.campos + 3 * c + 2);
                    const float r2 = fmaf(ex, ex, fmaf(ey, ey, ez * ez));
                    float inv = f_rsqrt(r2);
                    inv = inv * fmaf(-0.5f * r2, inv * inv, 1.5f);
                    dx[t] = ex * inv; dy[t] = ey * inv; dz[t] = ez * inv;
                    col[t][0] = dc0; col[t][1] = dc1; col[t][2] = dc2;
                }
            }
            if (mask != 0) {
                const int slot = ((PipeCfg<K>::STATIC_SLOTS ? 0u : sbase) + l) % RING;
                const float4 q = r.q[slot * PBLOCK + tid];
                const float4 sp = r.s[slot * PBLOCK + tid];
                const float w0 = r.w[(slot * 3 + 0) * PBLOCK + tid], w1 = r.w[(slot * 3 + 1) * PBLOCK + tid],
                            w2 = r.w[(slot * 3 + 2) * PBLOCK + tid];
                Lobe L; LobeBwd B;
                lobe_setup<EXACT, false>(q, sp, L, B);
#pragma unroll
                for (int t = 0; t < CT; ++t) {
                    {   // every camera slot is evaluated: culled slots carry g_colors = 0 / are zeroed at the store
                        EvalTerms T;
                        const float G = lobe_eval<false>(L, dx[t], dy[t], dz[t], T);
                        col[t][0] = fmaf(w0, G, col[t][0]);
                        col[t][1] = fmaf(w1, G, col[t][1]);
                        col[t][2] = fmaf(w2, G, col[t][2]);
                    }
                }
            }
        }
#pragma unroll
        for (int t = 0; t < CT; ++t) {
            if (t < p.C) {
                const bool on = mask & (1u << t);
                float *o = p.colors + ((int64_t)t * N + n) * 3;
                st_cs(o, on ? col[t][0] : 0.f); st_cs(o + 1, on ? col[t][1] : 0.f); st_cs(o + 2, on ? col[t][2] : 0.f);
            }
        }
        sbase = (sbase + K) % RING;
        hs = (hs + 1) % HR;
        mask = mask_next;
    }
    cp_async_wait<0>();
}

// ---------------------------------------------------------------------------------------------
// backward (no g_campos: that optional reduction stays on the generic kernel)
// ---------------------------------------------------------------------------------------------
template <int K, int CT, bool EXACT>
__global__ void __launch_bounds__(PBLOCK, 2) nasg_bwd_pipe_kernel(BwdParams p)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    constexpr int HR = PipeCfg<K>::HR, HF = 3 + 3 * CT;
    const Ring r = carve(smem_raw);
    const int tid = threadIdx.x;
    const int64_t N = p.N, stride = (int64_t)gridDim.x * PBLOCK;
    int64_t n = (int64_t)blockIdx.x * PBLOCK + tid;
    const int C = p.C;

    auto prefetch_item = [&](int64_t gn, int l, int slot, int hslot) {
        prefetch_lobe(r, slot, tid, p.quat, p.shape, p.amp, N, gn, l);
        if (l == 0 && gn < N) {
            float *h = r.h + (hslot * HF) * PBLOCK + tid;
            cp_async4(h, p.means + 3 * gn); cp_async4(h + PBLOCK, p.means + 3 * gn + 1);
            cp_async4(h + 2 * PBLOCK, p.means + 3 * gn + 2);
#pragma unroll
            for (int t = 0; t < CT; ++t) {
                if (t < C) {
                    const float *g = p.g_colors + ((int64_t)t * N + gn) * 3;
                    cp_async4(h + (3 + 3 * t) * PBLOCK, g); cp_async4(h + (4 + 3 * t) * PBLOCK, g + 1);
                    cp_async4(h + (5 + 3 * t) * PBLOCK, g + 2);
                }
            }
        }
        cp_async_commit();
    };
#pragma unroll
    for (int j = 0; j < DIST; ++j) prefetch_item(n + (j / K) * stride, j % K, j % RING, (j / K) % HR);

    unsigned sbase = 0, hs = 0;
    unsigned mask = load_mask(p.vis, N, n, C);
    for (; n < N; n += stride) {
        const unsigned mask_next = load_mask(p.vis, N, n + stride, C);
        float dx[CT], dy[CT], dz[CT], idist[CT], gc[CT][3], gd[CT][3];
#pragma unroll
        for (int l = 0; l < K; ++l) {
            prefetch_item(n + ((l + DIST) / K) * stride, (l + DIST) % K, ((PipeCfg<K>::STATIC_SLOTS ? 0u : sbase) + (l + DIST) % RING) % RING,
                          (hs + (l + DIST) / K) % HR);
            cp_async_wait<DIST>();
            if (l == 0) {
                const float *h = r.h + (hs * HF) * PBLOCK + tid;
                const float mx = h[0], my = h[PBLOCK], mz = h[2 * PBLOCK];
                float gdc0 = 0.f, gdc1 = 0.f, gdc2 = 0.f;
#pragma unroll
                for (int t = 0; t < CT; ++t) {
                    const int c = t < C ? t : 0;
                    const bool on = mask & (1u << t);
                    const float ex = mx - __ldg(p.campos + 3 * c), ey = my - __ldg(p.campos + 3 * c + 1),
                                ez = mz - __ldg(p.campos + 3 * c + 2);
                    const float r2 = fmaf(ex, ex, fmaf(ey, ey, ez * ez));
                    float inv = f_rsqrt(r2);
                    inv = inv * fmaf(-0.5f * r2, inv * inv, 1.5f);
                    dx[t] = ex * inv; dy[t] = ey * inv; dz[t] = ez * inv; idist[t] = on ? inv : 0.f;
                    gc[t][0] = on ? h[(3 + 3 * t) * PBLOCK] : 0.f;
                    gc[t][1] = on ? h[(4 + 3 * t) * PBLOCK] : 0.f;
                    gc[t][2] = on ? h[(5 + 3 * t) * PBLOCK] : 0.f;
                    gdc0 += gc[t][0]; gdc1 += gc[t][1]; gdc2 += gc[t][2];
                    gd[t][0] = gd[t][1] = gd[t][2] = 0.f;
                }
                if (p.g_dc) { st_cs(p.g_dc + n, gdc0); st_cs(p.g_dc + N + n, gdc1); st_cs(p.g_dc + 2 * N + n, gdc2); }
            }
            const int64_t ln = (int64_t)l * N + n;
            float4 gq = make_float4(0.f, 0.f, 0.f, 0.f), gs = make_float4(0.f, 0.f, 0.f, 0.f);
            float gw0 = 0.f, gw1 = 0.f, gw2 = 0.f;
            if (mask != 0) {
                const int slot = ((PipeCfg<K>::STATIC_SLOTS ? 0u : sbase) + l) % RING;
                const float4 q = r.q[slot * PBLOCK + tid];
                const float4 sp = r.s[slot * PBLOCK + tid];
                const float w0 = r.w[(slot * 3 + 0) * PBLOCK + tid], w1 = r.w[(slot * 3 + 1) * PBLOCK + tid],
                            w2 = r.w[(slot * 3 + 2) * PBLOCK + tid];
                Lobe L; LobeBwd B;
                lobe_setup<EXACT, true>(q, sp, L, B);
                float gX0 = 0.f, gX1 = 0.f, gX2 = 0.f, gZ0 = 0.f, gZ1 = 0.f, gZ2 = 0.f;
                float S0 = 0.f, S1 = 0.f, S2 = 0.f, Sk = 0.f, Sp = 0.f;
#pragma unroll
                for (int t = 0; t < CT; ++t) {
                    {   // every camera slot is evaluated: culled slots carry g_colors = 0 / are zeroed at the store
                        EvalTerms T;
                        const float G = lobe_eval<true>(L, dx[t], dy[t], dz[t], T);
                        const float gG = fmaf(gc[t][0], w0, fmaf(gc[t][1], w1, gc[t][2] * w2));   // dL/dG, eq.(6)
                        gw0 = fmaf(gc[t][0], G, gw0); gw1 = fmaf(gc[t][1], G, gw1); gw2 = fmaf(gc[t][2], G, gw2);
                        const float gGG = gG * G;
                        const float A_tau = T.Lk * fmaf(B.lam2, T.kp, 1.0f);                      // d ln(pE)/d tau
                        const float A_kap2 = fmaf(B.lam2 * (1.0f + T.tau), T.kp, T.tau) * T.inv_2kappa;  // (d ln(pE)/d kappa)/2
                        const float B1 = 2.0f * gGG * A_tau * T.inv_s2;
                        const float hs_ = gG * T.Gh * T.sn;                                       // carrier, eqs.(59),(65)
                        const float gu = fmaf(B1 * L.a, T.u, -hs_ * B.k);                         // gG dG/du (eqs.57-60)
                        const float gv = fmaf(B1 * T.tau, T.v, gGG * A_kap2);                     // gG dG/dv (eqs.61-64)
                        S0 += gGG;
                        S1 = fmaf(gGG, T.em1, S1);
                        S2 = fmaf(B1, T.uu, S2);
                        Sk = fmaf(hs_, T.u, Sk);
                        Sp += hs_;
                        gX0 = fmaf(gu, dx[t], gX0); gX1 = fmaf(gu, dy[t], gX1); gX2 = fmaf(gu, dz[t], gX2);
                        gZ0 = fmaf(gv, dx[t], gZ0); gZ1 = fmaf(gv, dy[t], gZ1); gZ2 = fmaf(gv, dz[t], gZ2);
                        gd[t][0] = fmaf(gu, L.Xx, fmaf(gv, L.Zx, gd[t][0]));
                        gd[t][1] = fmaf(gu, L.Xy, fmaf(gv, L.Zy, gd[t][1]));
                        gd[t][2] = fmaf(gu, L.Xz, fmaf(gv, L.Zz, gd[t][2]));
                    }
                }
                gs.x = fmaf(0.5f * S2, B.one_pa, -S0 * B.nA);            // (lambda, a) = (e^{l2}, e^{l1-l2} - 1)
                gs.y = fmaf(B.lam2, S1, -S0 * B.nL) - gs.x;
                gs.z = -fmaf(S0, B.nk, Sk);
                gs.w = -Sp;
                const float w = B.qw, x = B.qx, y = B.qy, z = B.qz;      // J^T of columns X, Z of R(qhat); qhat = q/|q|
                const float a0 = 2.0f * (z * gX1 - y * gX2 + y * gZ0 - x * gZ1);
                const float a1 = 2.0f * (y * gX1 + z * gX2 + z * gZ0 - w * gZ1) - 4.0f * x * gZ2;
                const float a2 = 2.0f * (x * gX1 - w * gX2 + w * gZ0 + z * gZ1) - 4.0f * y * (gX0 + gZ2);
                const float a3 = 2.0f * (w * gX1 + x * gX2 + x * gZ0 + y * gZ1) - 4.0f * z * gX0;
                const float dot = w * a0 + x * a1 + y * a2 + z * a3;
                gq.x = (a0 - w * dot) * B.inv_qn; gq.y = (a1 - x * dot) * B.inv_qn;
                gq.z = (a2 - y * dot) * B.inv_qn; gq.w = (a3 - z * dot) * B.inv_qn;
            }
            if (p.g_quat) st_cs4(p.g_quat + 4 * ln, gq);
            if (p.g_shape) st_cs4(p.g_shape + 4 * ln, gs);
            if (p.g_amp) {
                float *o = p.g_amp + (int64_t)l * 3 * N + n;
                st_cs(o, gw0); st_cs(o + N, gw1); st_cs(o + 2 * N, gw2);
            }
        }
        if (p.g_means) {        // through d = Delta/|Delta|: (I - d d^T)/|Delta|
            float gm0 = 0.f, gm1 = 0.f, gm2 = 0.f;
#pragma unroll
            for (int t = 0; t < CT; ++t) {
                const float dg = fmaf(dx[t], gd[t][0], fmaf(dy[t], gd[t][1], dz[t] * gd[t][2]));
                gm0 = fmaf(gd[t][0] - dx[t] * dg, idist[t], gm0);
                gm1 = fmaf(gd[t][1] - dy[t] * dg, idist[t], gm1);
                gm2 = fmaf(gd[t][2] - dz[t] * dg, idist[t], gm2);
            }
            float *o = p.g_means + 3 * n;
            st_cs(o, gm0); st_cs(o + 1, gm1); st_cs(o + 2, gm2);
        }
        sbase = (sbase + K) % RING;
        hs = (hs + 1) % HR;
        mask = mask_next;
    }
    cp_async_wait<0>();
}

// ---------------------------------------------------------------------------------------------
// launchers: persistent grid, 2 blocks per SM
// ---------------------------------------------------------------------------------------------
template <int K, int CT>
static cudaError_t launch_fwd_pipe_kc(const FwdParams &p, bool exact, cudaStream_t st)
{
    constexpr size_t smem = pipe_smem_bytes(PipeCfg<K>::HR, 6);
    const dim3 block(PBLOCK);
    static int cache[2][64] = {{0}};        // per (K, CT, norm mode) instantiation and device
    if (exact) nasg_fwd_pipe_kernel<K, CT, true><<<pipe_grid(nasg_fwd_pipe_kernel<K, CT, true>, smem, p.N, cache[1]), block, smem, st>>>(p);
    else nasg_fwd_pipe_kernel<K, CT, false><<<pipe_grid(nasg_fwd_pipe_kernel<K, CT, false>, smem, p.N, cache[0]), block, smem, st>>>(p);
    return cudaGetLastError();
}
template <int K>
static cudaError_t launch_fwd_pipe_k(const FwdParams &p, bool exact, cudaStream_t st)
{
    if (p.C == 1) return launch_fwd_pipe_kc<K, 1>(p, exact, st);
    if (p.C == 2) return launch_fwd_pipe_kc<K, 2>(p, exact, st);
    if (p.C == 3) return launch_fwd_pipe_kc<K, 3>(p, exact, st);
    return launch_fwd_pipe_kc<K, 4>(p, exact, st);
}
cudaError_t launch_nasg_fwd_pipe(const FwdParams &p, int K, bool exact, cudaStream_t st)
{
    switch (K) {
    case 1: return launch_fwd_pipe_k<1>(p, exact, st);
    case 2: return launch_fwd_pipe_k<2>(p, exact, st);
    case 3: return launch_fwd_pipe_k<3>(p, exact, st);
    case 4: return launch_fwd_pipe_k<4>(p, exact, st);
    case 5: return launch_fwd_pipe_k<5>(p, exact, st);
    case 8: return launch_fwd_pipe_k<8>(p, exact, st);
    default: return cudaErrorInvalidValue;
    }
}

template <int K, int CT>
static cudaError_t launch_bwd_pipe_kc(const BwdParams &p, bool exact, cudaStream_t st)
{
    constexpr size_t smem = pipe_smem_bytes(PipeCfg<K>::HR, 3 + 3 * CT);
    const dim3 block(PBLOCK);
    static int cache[2][64] = {{0}};        // per (K, CT, norm mode) instantiation and device
    if (exact) nasg_bwd_pipe_kernel<K, CT, true><<<pipe_grid(nasg_bwd_pipe_kernel<K, CT, true>, smem, p.N, cache[1]), block, smem, st>>>(p);
    else nasg_bwd_pipe_kernel<K, CT, false><<<pipe_grid(nasg_bwd_pipe_kernel<K, CT, false>, smem, p.N, cache[0]), block, smem, st>>>(p);
    return cudaGetLastError();
}
template <int K>
static cudaError_t launch_bwd_pipe_k(const BwdParams &p, bool exact, cudaStream_t st)
{
    if (p.C == 1) return launch_bwd_pipe_kc<K, 1>(p, exact, st);
    if (p.C == 2) return launch_bwd_pipe_kc<K, 2>(p, exact, st);
    if (p.C == 3) return launch_bwd_pipe_kc<K, 3>(p, exact, st);
    return launch_bwd_pipe_kc<K, 4>(p, exact, st);
}
cudaError_t launch_nasg_bwd_pipe(const BwdParams &p, int K, bool exact, cudaStream_t st)
{
    switch (K) {
    case 1: return launch_bwd_pipe_k<1>(p, exact, st);
    case 2: return launch_bwd_pipe_k<2>(p, exact, st);
    case 3: return launch_bwd_pipe_k<3>(p, exact, st);
    case 4: return launch_bwd_pipe_k<4>(p, exact, st);
    case 5: return launch_bwd_pipe_k<5>(p, exact, st);
    case 8: return launch_bwd_pipe_k<8>(p, exact, st);
    default: return cudaErrorInvalidValue;
    }
}

} // namespace nasg
