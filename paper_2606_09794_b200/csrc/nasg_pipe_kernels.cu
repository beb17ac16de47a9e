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
//
// Two families: nasg_{fwd,bwd}_pipe_kernel (C = 1: scalar arithmetic) and nasg_{fwd,bwd}_pipe2_kernel
// (C = 2..4: camera slots evaluated in pairs on packed f32x2 arithmetic, visibility bytes staged through
// shared memory with cp.async, culled slots neutralised without a branch). MODE = normaliser / carrier mode
// (include/nasg.h: 0 approximate, 1 exact eq.(10), 2 pure NASG), compiled in.
#include "nasg_internal.h"
#include "nasg_math.cuh"
#include "pipe_common.cuh"

namespace nasg {

constexpr int RING = 4;     // lobe slots per thread
constexpr int DIST = 3;     // prefetch distance in lobes

template <int K> struct PipeCfg {
    static constexpr int HR = (K == 1) ? 5 : (K <= 3) ? 3 : 2;   // header slots: Gaussians spanned by DIST lobes ahead, + 1 (K = 1, 3: + 1 more so that
                                                                 // the l == 0 prefetch never targets the slot other lanes still read their visibility bytes from)
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
// the packed kernels stage the visibility bytes of a Gaussian next to its header: [HR][4][PBLOCK] bytes
__host__ __device__ constexpr size_t pipe2_smem_bytes(int HR, int HF) { return pipe_smem_bytes(HR, HF) + (size_t)HR * 4 * PBLOCK; }

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
template <int K, int CT, int MODE>
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
                lobe_setup<MODE, false>(q, sp, L, B);
#pragma unroll
                for (int t = 0; t < CT; ++t) {
                    {   // every camera slot is evaluated: culled slots carry g_colors = 0 / are zeroed at the store
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

// forward, two cameras per packed f32x2 instruction (CT >= 2)
template <int K, int CT, int MODE>
__global__ void __launch_bounds__(PBLOCK, K <= 2 ? 2 : (CT >= 3 ? 3 : 4)) nasg_fwd_pipe2_kernel(FwdParams p)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    constexpr int HR = PipeCfg<K>::HR, HF = 6;
    const Ring r = carve(smem_raw);
    const int tid = threadIdx.x;
    const int64_t N = p.N, stride = (int64_t)gridDim.x * PBLOCK;
    int64_t n = (int64_t)blockIdx.x * PBLOCK + tid;
    unsigned char *vm = smem_raw + pipe_smem_bytes(HR, HF);
    const bool vis_cp = vis_rows_aligned(p.vis, N);

    auto prefetch_item = [&](int64_t gn, int l, int slot, int hslot) {
        prefetch_lobe(r, slot, tid, p.quat, p.shape, p.amp, N, gn, l);
        if (l == 0 && gn < N) {
            float *h = r.h + (hslot * HF) * PBLOCK + tid;
            cp_async4(h, p.means + 3 * gn); cp_async4(h + PBLOCK, p.means + 3 * gn + 1);
            cp_async4(h + 2 * PBLOCK, p.means + 3 * gn + 2);
            cp_async4(h + 3 * PBLOCK, p.dc + gn); cp_async4(h + 4 * PBLOCK, p.dc + N + gn);
            cp_async4(h + 5 * PBLOCK, p.dc + 2 * N + gn);
            if (vis_cp) prefetch_vis(vm, hslot, tid, p.vis, N, gn, p.C);
        }
        cp_async_commit();
    };
#pragma unroll
    for (int j = 0; j < DIST; ++j) prefetch_item(n + (j / K) * stride, j % K, j % RING, (j / K) % HR);

    unsigned sbase = 0, hs = 0;                  // ring slot of lobe 0 / header slot of the current Gaussian
    RawMask raw = {{0u, 0u, 0u, 0u}};
    if (!vis_cp) raw = load_raw_mask(p.vis, N, n, p.C);
    for (; n - (tid & 31) < N; n += stride) {       // warp-uniform trip count: lanes past N idle (mask 0, no stores)
        const bool valid = n < N;
        RawMask raw_next = {{0u, 0u, 0u, 0u}};
        if (!vis_cp) raw_next = load_raw_mask(p.vis, N, n + stride, p.C);
        unsigned mask = 0;
        // camera slots live in pairs (x = slot 2j, y = slot 2j+1) so that the evaluation runs on packed
        // f32x2 arithmetic; a slot beyond C repeats camera 0 and is never stored
        constexpr int NP = (CT + 1) / 2;
        float2 dx[NP], dy[NP], dz[NP], col[NP][3];
#pragma unroll
        for (int l = 0; l < K; ++l) {
            prefetch_item(n + ((l + DIST) / K) * stride, (l + DIST) % K, (sbase + (l + DIST) % RING) % RING,
                          (hs + (l + DIST) / K) % HR);
            cp_async_wait<DIST>();
            if (l == 0) {
                if (vis_cp) { __syncwarp(); mask = staged_mask(vm, hs, tid, p.C, valid); }
                else mask = combine_mask(raw);
                const float *h = r.h + (hs * HF) * PBLOCK + tid;
                const float2 mx = splat(h[0]), my = splat(h[PBLOCK]), mz = splat(h[2 * PBLOCK]);
                const float2 dc0 = splat(h[3 * PBLOCK]), dc1 = splat(h[4 * PBLOCK]), dc2 = splat(h[5 * PBLOCK]);
#pragma unroll
                for (int j = 0; j < NP; ++j) {
                    const int c0 = 2 * j < p.C ? 2 * j : 0, c1 = 2 * j + 1 < p.C ? 2 * j + 1 : 0;
                    const float2 ex = sub2(mx, make_float2(__ldg(p.campos + 3 * c0), __ldg(p.campos + 3 * c1)));
                    const float2 ey = sub2(my, make_float2(__ldg(p.campos + 3 * c0 + 1), __ldg(p.campos + 3 * c1 + 1)));
                    const float2 ez = sub2(mz, make_float2(__ldg(p.campos + 3 * c0 + 2), __ldg(p.campos + 3 * c1 + 2)));
                    const float2 r2 = fma2(ex, ex, fma2(ey, ey, mul2(ez, ez)));
                    float2 inv = make_float2(f_rsqrt(r2.x), f_rsqrt(r2.y));
                    inv = mul2(inv, fma2(mul2(splat(-0.5f), r2), mul2(inv, inv), splat(1.5f)));     // one Newton step
                    dx[j] = mul2(ex, inv); dy[j] = mul2(ey, inv); dz[j] = mul2(ez, inv);
                    col[j][0] = dc0; col[j][1] = dc1; col[j][2] = dc2;
                }
            }
            if (mask != 0) {
                const int slot = (sbase + l) % RING;
                const float4 q = r.q[slot * PBLOCK + tid];
                const float4 sp = r.s[slot * PBLOCK + tid];
                const float2 w0 = splat(r.w[(slot * 3 + 0) * PBLOCK + tid]), w1 = splat(r.w[(slot * 3 + 1) * PBLOCK + tid]),
                             w2 = splat(r.w[(slot * 3 + 2) * PBLOCK + tid]);
                Lobe L; LobeBwd B;
                lobe_setup<MODE, false>(q, sp, L, B);
#pragma unroll
                for (int j = 0; j < NP; ++j) {
                    // every camera slot is evaluated: culled slots are zeroed at the store
                    EvalTerms2 T;
                    const float2 G = lobe_eval2<false, MODE != 2>(L, dx[j], dy[j], dz[j], splat(0.f), T);
                    col[j][0] = fma2(w0, G, col[j][0]);
                    col[j][1] = fma2(w1, G, col[j][1]);
                    col[j][2] = fma2(w2, G, col[j][2]);
                }
            }
        }
#pragma unroll
        for (int t = 0; t < CT; ++t) {
            if (t < p.C && valid) {
                const bool on = mask & (1u << t);
                float *o = p.colors + ((int64_t)t * N + n) * 3;
                const float c0 = (t & 1) ? col[t / 2][0].y : col[t / 2][0].x, c1 = (t & 1) ? col[t / 2][1].y : col[t / 2][1].x,
                            c2 = (t & 1) ? col[t / 2][2].y : col[t / 2][2].x;
                st_cs(o, on ? c0 : 0.f); st_cs(o + 1, on ? c1 : 0.f); st_cs(o + 2, on ? c2 : 0.f);
            }
        }
        sbase = (sbase + K) % RING;
        hs = (hs + 1) % HR;
        raw = raw_next;
    }
    cp_async_wait<0>();
}

// ---------------------------------------------------------------------------------------------
// backward (g_campos, if asked for: per-thread partial over the thread's Gaussians -> block sum at the end)
// ---------------------------------------------------------------------------------------------
template <int K, int CT, int MODE>
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
    float cam[CT][3];                 // this thread's share of g_campos (only if p.cam_partial): summed over its Gaussians
#pragma unroll
    for (int t = 0; t < CT; ++t) cam[t][0] = cam[t][1] = cam[t][2] = 0.f;
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
                lobe_setup<MODE, true>(q, sp, L, B);
                float gX0 = 0.f, gX1 = 0.f, gX2 = 0.f, gZ0 = 0.f, gZ1 = 0.f, gZ2 = 0.f;
                float S0 = 0.f, S1 = 0.f, S2 = 0.f, Sk = 0.f, Sp = 0.f;
#pragma unroll
                for (int t = 0; t < CT; ++t) {
                    {   // every camera slot is evaluated: culled slots carry g_colors = 0 / are zeroed at the store
                        EvalTerms T;
                        const float G = lobe_eval<true, MODE != 2>(L, dx[t], dy[t], dz[t], T);
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
        if (p.g_means || p.cam_partial) {        // through d = Delta/|Delta|: (I - d d^T)/|Delta|; g_campos gets minus the same
            float gm0 = 0.f, gm1 = 0.f, gm2 = 0.f;
#pragma unroll
            for (int t = 0; t < CT; ++t) {
                const float dg = fmaf(dx[t], gd[t][0], fmaf(dy[t], gd[t][1], dz[t] * gd[t][2]));
                const float t0 = (gd[t][0] - dx[t] * dg) * idist[t], t1 = (gd[t][1] - dy[t] * dg) * idist[t],
                            t2 = (gd[t][2] - dz[t] * dg) * idist[t];
                gm0 += t0; gm1 += t1; gm2 += t2;
                cam[t][0] -= t0; cam[t][1] -= t1; cam[t][2] -= t2;
            }
            if (p.g_means) {
                float *o = p.g_means + 3 * n;
                st_cs(o, gm0); st_cs(o + 1, gm1); st_cs(o + 2, gm2);
            }
        }
        sbase = (sbase + K) % RING;
        hs = (hs + 1) % HR;
        mask = mask_next;
    }
    cp_async_wait<0>();
    if (p.cam_partial) {            // block partial of g_campos: warp shuffle -> shared memory -> fixed-order sum (deterministic)
        __syncthreads();            // (every thread is done with the ring: reuse its first bytes)
        float *red = reinterpret_cast<float *>(smem_raw);
#pragma unroll
        for (int t = 0; t < CT; ++t)
            if (t < C)
                for (int i = 0; i < 3; ++i)
                    pipe_block_sum_store(cam[t][i], red, p.cam_partial + ((int64_t)blockIdx.x * C + t) * 3 + i);
    }
}

// ---------------------------------------------------------------------------------------------
// backward, two cameras per packed f32x2 instruction (CT >= 2)
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ float hsum(float2 a) { return a.x + a.y; }

#ifndef NASG_BWD2_MINB
#define NASG_BWD2_MINB 2
#endif
// CAMGRAD: also produce this block's partial of g_campos (compile-time: the extra code would cost the common
// no-g_campos instantiation ~2 % through register allocation alone)
template <int K, int CT, int MODE, bool CAMGRAD>
__global__ void __launch_bounds__(PBLOCK, NASG_BWD2_MINB) nasg_bwd_pipe2_kernel(BwdParams p)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    constexpr int HR = PipeCfg<K>::HR, HF = 3 + 3 * CT, NP = (CT + 1) / 2;
    const Ring r = carve(smem_raw);
    const int tid = threadIdx.x;
    const int64_t N = p.N, stride = (int64_t)gridDim.x * PBLOCK;
    int64_t n = (int64_t)blockIdx.x * PBLOCK + tid;
    const int C = p.C;
    unsigned char *vm = smem_raw + pipe_smem_bytes(HR, HF);
    const bool vis_cp = vis_rows_aligned(p.vis, N);

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
            if (vis_cp) prefetch_vis(vm, hslot, tid, p.vis, N, gn, C);
        }
        cp_async_commit();
    };
#pragma unroll
    for (int j = 0; j < DIST; ++j) prefetch_item(n + (j / K) * stride, j % K, j % RING, (j / K) % HR);

    unsigned sbase = 0, hs = 0;
    // this thread's share of g_campos, 3 floats per camera slot, kept in shared memory (registers are the scarce
    // resource here); the area exists only when the launcher was asked for g_campos
    auto cam_acc = [&]() { return reinterpret_cast<float *>(vm + HR * 4 * PBLOCK) + 2 * NP * PBLOCK + tid; };
    if (CAMGRAD) {
        float *hc = cam_acc();
#pragma unroll
        for (int i = 0; i < 6 * NP; ++i) hc[i * PBLOCK] = 0.f;
    }
    RawMask raw = {{0u, 0u, 0u, 0u}};
    if (!vis_cp) raw = load_raw_mask(p.vis, N, n, C);
    for (; n - (tid & 31) < N; n += stride) {       // warp-uniform trip count: lanes past N idle (mask 0, no stores)
        const bool valid = n < N;
        RawMask raw_next = {{0u, 0u, 0u, 0u}};
        if (!vis_cp) raw_next = load_raw_mask(p.vis, N, n + stride, C);
        unsigned mask = 0;
        // camera slots in pairs (x = slot 2j, y = slot 2j+1). A culled or padding slot gets an exponent bias of
        // -1e30: its lobe value and with it every gradient contribution is exactly 0.
        float2 dx[NP], dy[NP], dz[NP], gd[NP][3];
        // per-thread scratch behind the staged visibility bytes: 1/|Delta| per camera is parked here instead of
        // in registers until the end of the Gaussian (parking the directions too costs more than it frees)
        float *hi = reinterpret_cast<float *>(vm + HR * 4 * PBLOCK) + tid;
        const float *h = r.h + (hs * HF) * PBLOCK + tid;                        // header of this Gaussian (valid after lobe 0 landed)
#pragma unroll 1
        for (int l = 0; l < K; ++l) {
            prefetch_item(n + ((l + DIST) / K) * stride, (l + DIST) % K, (sbase + l + DIST) % RING, (hs + (l + DIST) / K) % HR);
            cp_async_wait<DIST>();
            if (l == 0) {
                if (vis_cp) { __syncwarp(); mask = staged_mask(vm, hs, tid, C, valid); }
                else mask = combine_mask(raw);
                const float2 mx = splat(h[0]), my = splat(h[PBLOCK]), mz = splat(h[2 * PBLOCK]);
                float gdc0 = 0.f, gdc1 = 0.f, gdc2 = 0.f;
#pragma unroll
                for (int j = 0; j < NP; ++j) {
                    const int t0 = 2 * j, t1 = 2 * j + 1;
                    const int c0 = t0 < C ? t0 : 0, c1 = t1 < C ? t1 : 0;
                    const bool on0 = mask & (1u << t0), on1 = (t1 < CT) && (mask & (1u << t1));
                    const float2 ex = sub2(mx, make_float2(__ldg(p.campos + 3 * c0), __ldg(p.campos + 3 * c1)));
                    const float2 ey = sub2(my, make_float2(__ldg(p.campos + 3 * c0 + 1), __ldg(p.campos + 3 * c1 + 1)));
                    const float2 ez = sub2(mz, make_float2(__ldg(p.campos + 3 * c0 + 2), __ldg(p.campos + 3 * c1 + 2)));
                    const float2 r2 = fma2(ex, ex, fma2(ey, ey, mul2(ez, ez)));
                    float2 inv = make_float2(f_rsqrt(r2.x), f_rsqrt(r2.y));
                    inv = mul2(inv, fma2(mul2(splat(-0.5f), r2), mul2(inv, inv), splat(1.5f)));
                    dx[j] = mul2(ex, inv); dy[j] = mul2(ey, inv); dz[j] = mul2(ez, inv);
                    hi[t0 * PBLOCK] = inv.x; hi[t1 * PBLOCK] = inv.y;
                    // g_colors of a culled slot is never used (it may be NaN or uninitialised memory): the staged copy in this
                    // thread's private header column is zeroed once, so that the per-lobe reads below need no select
                    float *hw = r.h + (hs * HF) * PBLOCK + tid;
                    if (on0) { gdc0 += h[(3 + 3 * t0) * PBLOCK]; gdc1 += h[(4 + 3 * t0) * PBLOCK]; gdc2 += h[(5 + 3 * t0) * PBLOCK]; }
                    else { hw[(3 + 3 * t0) * PBLOCK] = 0.f; hw[(4 + 3 * t0) * PBLOCK] = 0.f; hw[(5 + 3 * t0) * PBLOCK] = 0.f; }
                    if (t1 < CT) {
                        if (on1) { gdc0 += h[(3 + 3 * t1) * PBLOCK]; gdc1 += h[(4 + 3 * t1) * PBLOCK]; gdc2 += h[(5 + 3 * t1) * PBLOCK]; }
                        else { hw[(3 + 3 * t1) * PBLOCK] = 0.f; hw[(4 + 3 * t1) * PBLOCK] = 0.f; hw[(5 + 3 * t1) * PBLOCK] = 0.f; }
                    }
                    gd[j][0] = gd[j][1] = gd[j][2] = splat(0.f);
                }
                if (p.g_dc && valid) { st_cs(p.g_dc + n, gdc0); st_cs(p.g_dc + N + n, gdc1); st_cs(p.g_dc + 2 * N + n, gdc2); }
            }
            const int64_t ln = (int64_t)l * N + n;
            float4 gq = make_float4(0.f, 0.f, 0.f, 0.f), gs = make_float4(0.f, 0.f, 0.f, 0.f);
            float gw0 = 0.f, gw1 = 0.f, gw2 = 0.f;
            if (mask != 0) {
                const int slot = (sbase + l) % RING;
                const float4 sp = r.s[slot * PBLOCK + tid];
                const float2 w0 = splat(r.w[(slot * 3 + 0) * PBLOCK + tid]), w1 = splat(r.w[(slot * 3 + 1) * PBLOCK + tid]),
                             w2 = splat(r.w[(slot * 3 + 2) * PBLOCK + tid]);
                Lobe L; LobeBwd B;
                lobe_setup<MODE, true>(r.q[slot * PBLOCK + tid], sp, L, B);
                const float2 z2 = splat(0.f);
                float2 pw0 = z2, pw1 = z2, pw2 = z2;                             // packed accumulators, halves summed below
                float2 gX0 = z2, gX1 = z2, gX2 = z2, gZ0 = z2, gZ1 = z2, gZ2 = z2;
                float2 S0 = z2, S1 = z2, S2 = z2, Sk = z2, Sp = z2;
                const float2 lam2 = splat(B.lam2), a2 = splat(L.a), nk2 = splat(-sp.z);
#pragma unroll
                for (int j = 0; j < NP; ++j) {
                    const int t0 = 2 * j, t1 = (2 * j + 1 < CT) ? 2 * j + 1 : 2 * j;
                    const float2 gc0 = make_float2(h[(3 + 3 * t0) * PBLOCK], h[(3 + 3 * t1) * PBLOCK]);     // g_colors of the pair
                    const float2 gc1 = make_float2(h[(4 + 3 * t0) * PBLOCK], h[(4 + 3 * t1) * PBLOCK]);
                    const float2 gc2 = make_float2(h[(5 + 3 * t0) * PBLOCK], h[(5 + 3 * t1) * PBLOCK]);
                    const float2 dxj = dx[j], dyj = dy[j], dzj = dz[j];
                    EvalTerms2 T;
                    const float2 bias = make_float2((mask & (1u << t0)) ? 0.f : -1e30f,
                                                    (2 * j + 1 < CT && (mask & (1u << t1))) ? 0.f : -1e30f);   // (re-derived: 4 fewer live registers)
                    const float2 G = lobe_eval2<true, MODE != 2>(L, dxj, dyj, dzj, bias, T);
                    const float2 gG = fma2(gc0, w0, fma2(gc1, w1, mul2(gc2, w2)));                      // dL/dG, eq.(6)
                    pw0 = fma2(gc0, G, pw0); pw1 = fma2(gc1, G, pw1); pw2 = fma2(gc2, G, pw2);
                    const float2 gGG = mul2(gG, G);
                    const float2 A_tau = mul2(T.Lk, fma2(lam2, T.kp, splat(1.0f)));                     // d ln(pE)/d tau
                    const float2 A_kap2 = mul2(fma2(mul2(lam2, add2(T.tau, splat(1.0f))), T.kp, T.tau), T.inv_2kappa);  // (d ln(pE)/d kappa)/2
                    const float2 B1 = mul2(mul2(add2(gGG, gGG), A_tau), T.inv_s2);
                    const float2 hs_ = mul2(mul2(gG, T.Gh), T.sn);                                      // carrier, eqs.(59),(65)
                    const float2 gu = fma2(mul2(B1, a2), T.u, mul2(hs_, nk2));                          // gG dG/du (eqs.57-60)
                    const float2 gv = fma2(mul2(B1, T.tau), T.v, mul2(gGG, A_kap2));                    // gG dG/dv (eqs.61-64)
                    S0 = add2(S0, gGG);
                    S1 = fma2(gGG, T.em1, S1);
                    S2 = fma2(B1, T.uu, S2);
                    Sk = fma2(hs_, T.u, Sk);
                    Sp = add2(Sp, hs_);
                    gX0 = fma2(gu, dxj, gX0); gX1 = fma2(gu, dyj, gX1); gX2 = fma2(gu, dzj, gX2);
                    gZ0 = fma2(gv, dxj, gZ0); gZ1 = fma2(gv, dyj, gZ1); gZ2 = fma2(gv, dzj, gZ2);
                    gd[j][0] = fma2(gu, splat(L.Xx), fma2(gv, splat(L.Zx), gd[j][0]));
                    gd[j][1] = fma2(gu, splat(L.Xy), fma2(gv, splat(L.Zy), gd[j][1]));
                    gd[j][2] = fma2(gu, splat(L.Xz), fma2(gv, splat(L.Zz), gd[j][2]));
                }
                gw0 = hsum(pw0); gw1 = hsum(pw1); gw2 = hsum(pw2);
                const float s0 = hsum(S0), s1 = hsum(S1), s2 = hsum(S2), sk = hsum(Sk), sp_ = hsum(Sp);
                const float X0 = hsum(gX0), X1 = hsum(gX1), X2 = hsum(gX2), Z0 = hsum(gZ0), Z1 = hsum(gZ1), Z2 = hsum(gZ2);
                gs.x = fmaf(0.5f * s2, L.a + 1.0f, -s0 * B.nA);          // (lambda, a) = (e^{l2}, e^{l1-l2} - 1)
                gs.y = fmaf(B.lam2, s1, -s0 * B.nL) - gs.x;
                gs.z = -fmaf(s0, B.nk, sk);
                gs.w = -sp_;
                // J^T of columns X, Z of R(qhat), qhat = q/|q| (re-normalised here: cheaper than keeping it live)
                const float4 q = r.q[slot * PBLOCK + tid];
                const float qq = q.x * q.x + q.y * q.y + q.z * q.z + q.w * q.w;
                float inv_qn = f_rsqrt(qq);
                inv_qn = inv_qn * fmaf(-0.5f * qq, inv_qn * inv_qn, 1.5f);
                const float w = q.x * inv_qn, x = q.y * inv_qn, y = q.z * inv_qn, z = q.w * inv_qn;
                const float a0 = 2.0f * (z * X1 - y * X2 + y * Z0 - x * Z1);
                const float a1 = 2.0f * (y * X1 + z * X2 + z * Z0 - w * Z1) - 4.0f * x * Z2;
                const float a2_ = 2.0f * (x * X1 - w * X2 + w * Z0 + z * Z1) - 4.0f * y * (X0 + Z2);
                const float a3 = 2.0f * (w * X1 + x * X2 + x * Z0 + y * Z1) - 4.0f * z * X0;
                const float dot = w * a0 + x * a1 + y * a2_ + z * a3;
                gq.x = (a0 - w * dot) * inv_qn; gq.y = (a1 - x * dot) * inv_qn;
                gq.z = (a2_ - y * dot) * inv_qn; gq.w = (a3 - z * dot) * inv_qn;
            }
            if (p.g_quat && valid) st_cs4(p.g_quat + 4 * ln, gq);
            if (p.g_shape && valid) st_cs4(p.g_shape + 4 * ln, gs);
            if (p.g_amp && valid) {
                float *o = p.g_amp + (int64_t)l * 3 * N + n;
                st_cs(o, gw0); st_cs(o + N, gw1); st_cs(o + 2 * N, gw2);
            }
        }
        if ((p.g_means || CAMGRAD) && valid) {    // through d = Delta/|Delta|: (I - d d^T)/|Delta|   (gd of a culled slot is exactly 0)
            float2 gm0 = splat(0.f), gm1 = splat(0.f), gm2 = splat(0.f);
#pragma unroll
            for (int j = 0; j < NP; ++j) {
                const float2 dxj = dx[j], dyj = dy[j], dzj = dz[j];
                const float2 dg = fma2(dxj, gd[j][0], fma2(dyj, gd[j][1], mul2(dzj, gd[j][2])));
                const float2 idist = make_float2(hi[(2 * j) * PBLOCK], hi[(2 * j + 1) * PBLOCK]);
                gm0 = fma2(sub2(gd[j][0], mul2(dxj, dg)), idist, gm0);
                gm1 = fma2(sub2(gd[j][1], mul2(dyj, dg)), idist, gm1);
                gm2 = fma2(sub2(gd[j][2], mul2(dzj, dg)), idist, gm2);
                if (CAMGRAD) {                                  // g_campos_c -= the same terms, per camera slot
                    const float2 t0 = mul2(sub2(gd[j][0], mul2(dxj, dg)), idist), t1 = mul2(sub2(gd[j][1], mul2(dyj, dg)), idist),
                                 t2 = mul2(sub2(gd[j][2], mul2(dzj, dg)), idist);
                    float *c0 = cam_acc() + (6 * j) * PBLOCK, *c1 = c0 + 3 * PBLOCK;
                    c0[0] -= t0.x; c0[PBLOCK] -= t1.x; c0[2 * PBLOCK] -= t2.x;
                    c1[0] -= t0.y; c1[PBLOCK] -= t1.y; c1[2 * PBLOCK] -= t2.y;
                }
            }
            if (p.g_means) {
                float *o = p.g_means + 3 * n;
                st_cs(o, hsum(gm0)); st_cs(o + 1, hsum(gm1)); st_cs(o + 2, hsum(gm2));
            }
        }
        sbase = (sbase + K) % RING;
        hs = (hs + 1) % HR;
        raw = raw_next;
    }
    cp_async_wait<0>();
    if (CAMGRAD) {                  // block partial of g_campos: warp shuffle -> shared memory -> fixed-order sum (deterministic)
        __syncthreads();            // (every thread is done with the ring: reuse its first bytes)
        float *red = reinterpret_cast<float *>(smem_raw);
        const float *hc = cam_acc();
        for (int t = 0; t < C; ++t)
            for (int i = 0; i < 3; ++i)
                pipe_block_sum_store(hc[(3 * t + i) * PBLOCK], red, p.cam_partial + ((int64_t)blockIdx.x * C + t) * 3 + i);
    }
}

// ---------------------------------------------------------------------------------------------
// launchers: persistent grid, 2 blocks per SM
// ---------------------------------------------------------------------------------------------
template <int K, int CT>
static cudaError_t launch_fwd_pipe_kc(const FwdParams &p, int mode, cudaStream_t st)
{
    constexpr size_t smem = CT >= 2 ? pipe2_smem_bytes(PipeCfg<K>::HR, 6) : pipe_smem_bytes(PipeCfg<K>::HR, 6);
    const dim3 block(PBLOCK);
    static int cache[3][64] = {{0}};        // per (K, CT, norm mode) instantiation and device
    if constexpr (CT >= 2) {
        if (mode == 1) nasg_fwd_pipe2_kernel<K, CT, 1><<<pipe_grid(nasg_fwd_pipe2_kernel<K, CT, 1>, smem, p.N, cache[1]), block, smem, st>>>(p);
        else if (mode == 0) nasg_fwd_pipe2_kernel<K, CT, 0><<<pipe_grid(nasg_fwd_pipe2_kernel<K, CT, 0>, smem, p.N, cache[0]), block, smem, st>>>(p);
        else nasg_fwd_pipe2_kernel<K, CT, 2><<<pipe_grid(nasg_fwd_pipe2_kernel<K, CT, 2>, smem, p.N, cache[2]), block, smem, st>>>(p);
    } else {
        if (mode == 1) nasg_fwd_pipe_kernel<K, CT, 1><<<pipe_grid(nasg_fwd_pipe_kernel<K, CT, 1>, smem, p.N, cache[1]), block, smem, st>>>(p);
        else if (mode == 0) nasg_fwd_pipe_kernel<K, CT, 0><<<pipe_grid(nasg_fwd_pipe_kernel<K, CT, 0>, smem, p.N, cache[0]), block, smem, st>>>(p);
        else nasg_fwd_pipe_kernel<K, CT, 2><<<pipe_grid(nasg_fwd_pipe_kernel<K, CT, 2>, smem, p.N, cache[2]), block, smem, st>>>(p);
    }
    return cudaGetLastError();
}
template <int K>
static cudaError_t launch_fwd_pipe_k(const FwdParams &p, int mode, cudaStream_t st)
{
    if (p.C == 1) return launch_fwd_pipe_kc<K, 1>(p, mode, st);
    if (p.C == 2) return launch_fwd_pipe_kc<K, 2>(p, mode, st);
    if (p.C == 3) return launch_fwd_pipe_kc<K, 3>(p, mode, st);
    return launch_fwd_pipe_kc<K, 4>(p, mode, st);
}
cudaError_t launch_nasg_fwd_pipe(const FwdParams &p, int K, int mode, cudaStream_t st)
{
    switch (K) {
    case 1: return launch_fwd_pipe_k<1>(p, mode, st);
    case 2: return launch_fwd_pipe_k<2>(p, mode, st);
    case 3: return launch_fwd_pipe_k<3>(p, mode, st);
    case 4: return launch_fwd_pipe_k<4>(p, mode, st);
    case 5: return launch_fwd_pipe_k<5>(p, mode, st);
    case 8: return launch_fwd_pipe_k<8>(p, mode, st);
    default: return cudaErrorInvalidValue;
    }
}

template <int K, int CT>
static cudaError_t launch_bwd_pipe_kc(const BwdParams &p, int mode, cudaStream_t st, int *grid_out)
{
    const bool camgrad = p.cam_partial != nullptr;       // packed kernels: + 3 floats per camera slot and thread for g_campos
    const size_t smem = CT >= 2 ? pipe2_smem_bytes(PipeCfg<K>::HR, 3 + 3 * CT) + (size_t)PBLOCK * 4 * (camgrad ? 8 : 2) * ((CT + 1) / 2)
                                : pipe_smem_bytes(PipeCfg<K>::HR, 3 + 3 * CT);
    const dim3 block(PBLOCK);
    static int cache_all[2][3][64] = {{{0}}};   // per (K, CT, g_campos, norm mode) instantiation and device
    int (*cache)[64] = cache_all[camgrad ? 1 : 0];
    if constexpr (CT >= 2) {
        if (camgrad) {
            if (mode == 1) nasg_bwd_pipe2_kernel<K, CT, 1, true><<<pipe_grid(nasg_bwd_pipe2_kernel<K, CT, 1, true>, smem, p.N, cache[1]), block, smem, st>>>(p);
            else if (mode == 0) nasg_bwd_pipe2_kernel<K, CT, 0, true><<<pipe_grid(nasg_bwd_pipe2_kernel<K, CT, 0, true>, smem, p.N, cache[0]), block, smem, st>>>(p);
            else nasg_bwd_pipe2_kernel<K, CT, 2, true><<<pipe_grid(nasg_bwd_pipe2_kernel<K, CT, 2, true>, smem, p.N, cache[2]), block, smem, st>>>(p);
        } else {
            if (mode == 1) nasg_bwd_pipe2_kernel<K, CT, 1, false><<<pipe_grid(nasg_bwd_pipe2_kernel<K, CT, 1, false>, smem, p.N, cache[1]), block, smem, st>>>(p);
            else if (mode == 0) nasg_bwd_pipe2_kernel<K, CT, 0, false><<<pipe_grid(nasg_bwd_pipe2_kernel<K, CT, 0, false>, smem, p.N, cache[0]), block, smem, st>>>(p);
            else nasg_bwd_pipe2_kernel<K, CT, 2, false><<<pipe_grid(nasg_bwd_pipe2_kernel<K, CT, 2, false>, smem, p.N, cache[2]), block, smem, st>>>(p);
        }
    } else {
        if (mode == 1) nasg_bwd_pipe_kernel<K, CT, 1><<<pipe_grid(nasg_bwd_pipe_kernel<K, CT, 1>, smem, p.N, cache[1]), block, smem, st>>>(p);
        else if (mode == 0) nasg_bwd_pipe_kernel<K, CT, 0><<<pipe_grid(nasg_bwd_pipe_kernel<K, CT, 0>, smem, p.N, cache[0]), block, smem, st>>>(p);
        else nasg_bwd_pipe_kernel<K, CT, 2><<<pipe_grid(nasg_bwd_pipe_kernel<K, CT, 2>, smem, p.N, cache[2]), block, smem, st>>>(p);
    }
    int dev = 0;
    cudaGetDevice(&dev);
    const int64_t need = (p.N + PBLOCK - 1) / PBLOCK;
    const int resident = cache[mode][(dev >= 0 && dev < 64) ? dev : 0];
    *grid_out = (int)(need < resident ? need : resident);       // = the grid just launched (blocks of cam_partial written)
    return cudaGetLastError();
}
template <int K>
static cudaError_t launch_bwd_pipe_k(const BwdParams &p, int mode, cudaStream_t st, int *grid_out)
{
    if (p.C == 1) return launch_bwd_pipe_kc<K, 1>(p, mode, st, grid_out);
    if (p.C == 2) return launch_bwd_pipe_kc<K, 2>(p, mode, st, grid_out);
    if (p.C == 3) return launch_bwd_pipe_kc<K, 3>(p, mode, st, grid_out);
    return launch_bwd_pipe_kc<K, 4>(p, mode, st, grid_out);
}
cudaError_t launch_nasg_bwd_pipe(const BwdParams &p, int K, int mode, cudaStream_t st, int *grid_out)
{
    switch (K) {
    case 1: return launch_bwd_pipe_k<1>(p, mode, st, grid_out);
    case 2: return launch_bwd_pipe_k<2>(p, mode, st, grid_out);
    case 3: return launch_bwd_pipe_k<3>(p, mode, st, grid_out);
    case 4: return launch_bwd_pipe_k<4>(p, mode, st, grid_out);
    case 5: return launch_bwd_pipe_k<5>(p, mode, st, grid_out);
    case 8: return launch_bwd_pipe_k<8>(p, mode, st, grid_out);
    default: return cudaErrorInvalidValue;
    }
}

} // namespace nasg
