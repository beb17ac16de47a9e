// nasg_tile_kernels.cu — the tile kernels of the ROW-ARRAY entry points nasg_eval_fwd / nasg_eval_bwd (sm_100a; the
// headline path is the record family of nasg_rec_kernels.cu, which this file preceded): even lobe counts (K = 2, 4, 8),
// C <= 4 cameras, N a multiple of 4 (16 with a visibility mask) and 16-byte aligned arrays. Everything else
// (odd K, C > 4, ragged N, misaligned views, g_campos, small N) runs the cp.async ring kernels of
// nasg_pipe_kernels.cu or the generic kernels of nasg_kernels.cu.
//
// Arithmetic: lobe PAIRS on packed f32x2 instructions (nasg_lp_math.cuh): set-up, evaluation and backward all issue
// one instruction for two lobes.
//
// Data movement: every WARP runs its own pipeline over "warp tiles" of 32 consecutive Gaussians (lane = Gaussian).
// The inputs of a warp tile are contiguous row segments of the structure-of-arrays layout (quat/shape rows of a
// lobe: 512 B, amp/dc rows: 128 B, means: 384 B, g_colors of a camera: 384 B, visibility bytes of a camera: 32 B),
// so ONE elected lane moves them with 1-D bulk copies (cp.async.bulk, the TMA engine) that complete on an mbarrier
// of that warp: ~4 uniform-datapath instructions per row and WARP instead of an LDGSTS plus 64-bit address
// arithmetic per row and THREAD (10 % of the ring kernels' instructions).
//   * item = (warp tile, lobe pair); a warp's items live in a ring of STAGES slots of its private shared-memory
//     region, each with a "full" mbarrier (armed with the byte count, completed by the copy engine).
//   * the warp waits for the slot, every lane copies its 22 values into registers, __syncwarp, and the elected lane
//     at once issues the copies of the item STAGES ahead into the same slot: the slot is busy only between issue
//     and read, an item is in flight for STAGES item-times (microseconds; DRAM latency is < 1 us).
//   * the per-tile header (means, dc | g_colors, visibility bytes) has its own slot(s); it is consumed at the start
//     of a tile (directions and masked g_colors go to registers / a per-lane scratch column) and re-armed for the
//     next tile at once.
// Warps never wait for each other: no __syncthreads, no atomics (a first version that shared 256-Gaussian tiles
// between the 8 warps of a block, refilled by the last warp to release a slot, lost 25 % of its time to the drift
// between warps: profiles/).
#include "bulk_common.cuh"
#include "nasg_internal.h"
#include "nasg_lp_math.cuh"
#include "pipe_common.cuh"

namespace nasg {
namespace lp {      // (the names of nasg_lp_math.cuh hide the camera-pair helpers of nasg_math.cuh in here)

#ifndef NASG_TB
#define NASG_TB 256
#endif
constexpr int TB = NASG_TB;             // threads per block = Gaussians per block tile (8 warp tiles)
constexpr int NWARP = TB / 32;
constexpr int WT = 32;                  // Gaussians per warp tile
constexpr int STAGE_BYTES = WT * (2 * 16 + 2 * 16 + 6 * 4);        // quat[2], shape[2], amp[6] rows of a lobe pair: 2816 B

using namespace bulk;          // mbarrier / bulk-copy primitives, shared-memory accessors (bulk_common.cuh)

// ---- shared-memory layout: one private region per warp ---------------------------------------------
// [ stage 0 | ... | stage S-1 ][ header 0 | ... ][ scratch (backward) ][ mbarriers ]
// stage:   quat float4 [2][32] | shape float4 [2][32] | amp float [6][32]
// header:  means float [32][3] | forward: dc float [3][32], backward: g_colors float [CT][32][3] | vis uint8 [CT][32]
// scratch (backward, per-lane columns): cam float4 [CT][32] = (dx,dy,dz,1/|Delta|) | gcm float4 [CT][32] = masked g_colors |
//          qs 2 x (f2,f2) [32] = qhat 2/|q| of the current pair
template <int CT, bool BWD> struct TileLayout {
    static constexpr int HDR_MEANS = 0;
    static constexpr int HDR_BODY = WT * 12;
    static constexpr int HDR_VIS = HDR_BODY + (BWD ? CT * WT * 12 : WT * 12);
    static constexpr int HDR_BYTES = HDR_VIS + CT * WT;
    static constexpr int SCRATCH_BYTES = BWD ? (2 * CT + 2) * WT * 16 : 0;
};
template <int CT, bool BWD> __host__ __device__ constexpr int warp_region_bytes(int stages, int hslots)
{
    return stages * STAGE_BYTES + hslots * TileLayout<CT, BWD>::HDR_BYTES + TileLayout<CT, BWD>::SCRATCH_BYTES + 64;
}
template <int CT, bool BWD> __host__ __device__ constexpr size_t tile_smem_bytes(int stages, int hslots)
{
    return (size_t)NWARP * warp_region_bytes<CT, BWD>(stages, hslots);
}

struct WarpCtx {
    unsigned stage0, hdr, scr, bars;     // shared-memory addresses (u32) inside this warp's region
    int warp;                            // warp index in the block (warp-uniform)
    int64_t N;
};
// mbarriers: full[s] at bars + 8 s (s < 4), hfull[h] at bars + 32 + 8 h (h < 4)
__device__ __forceinline__ unsigned bar_full(const WarpCtx &c, int s) { return c.bars + 8u * s; }
__device__ __forceinline__ unsigned bar_hfull(const WarpCtx &c, int h) { return c.bars + 32u + 8u * h; }
// first Gaussian of this warp's tile in the block's i-th tile
__device__ __forceinline__ int64_t warp_tile_start(const WarpCtx &c, int i)
{
    return ((int64_t)blockIdx.x + (int64_t)i * gridDim.x) * TB + c.warp * WT;
}

// copies of item m = (i-th tile, lobe pair j) of this warp into slot m % STAGES; nothing if the warp has no such tile
template <int K, int STAGES>
__device__ __forceinline__ void issue_stage(const WarpCtx &c, int m, const float *quat, const float *shape, const float *amp)
{
    constexpr int NPAIR = K / 2;
    const int i = m / NPAIR, j = m % NPAIR;
    const int64_t n0 = warp_tile_start(c, i), N = c.N;
    if (n0 >= N) return;
    const unsigned cnt = (unsigned)(N - n0 < WT ? N - n0 : WT);
    const int slot = m % STAGES;
    const unsigned bar = bar_full(c, slot), dst = c.stage0 + (unsigned)slot * STAGE_BYTES;
    fence_proxy_async();            // the lanes' reads of the slot (generic proxy) before the refill (async proxy): bulk_common.cuh
    mbar_expect_tx(bar, cnt * 88u);
#pragma unroll
    for (int h = 0; h < 2; ++h) {
        const int64_t ln = (int64_t)(2 * j + h) * N + n0;
        bulk_g2s(dst + h * WT * 16, quat + 4 * ln, cnt * 16u, bar);
        bulk_g2s(dst + (2 + h) * WT * 16, shape + 4 * ln, cnt * 16u, bar);
#pragma unroll
        for (int ch = 0; ch < 3; ++ch)
            bulk_g2s(dst + 4 * WT * 16 + (h * 3 + ch) * WT * 4, amp + (int64_t)((2 * j + h) * 3 + ch) * N + n0, cnt * 4u, bar);
    }
}
// header of this warp's part of the block's i-th tile
template <int CT, bool BWD, int HSLOTS>
__device__ __forceinline__ void issue_header(const WarpCtx &c, int i, int C, const float *means, const float *body, const uint8_t *vis)
{
    using L = TileLayout<CT, BWD>;
    const int64_t n0 = warp_tile_start(c, i), N = c.N;
    if (n0 >= N) return;
    const unsigned cnt = (unsigned)(N - n0 < WT ? N - n0 : WT);
    const int h = i % HSLOTS;
    const unsigned bar = bar_hfull(c, h), hdr = c.hdr + (unsigned)h * (unsigned)L::HDR_BYTES;
    const unsigned rows = BWD ? (unsigned)C : 1u;        // forward: dc = 3 planar rows of 4 B; backward: g_colors = C rows of 12 B
    fence_proxy_async();            // the lanes' reads of the slot (generic proxy) before the refill (async proxy): bulk_common.cuh
    mbar_expect_tx(bar, cnt * (12u + 12u * rows + (vis ? (unsigned)C : 0u)));
    bulk_g2s(hdr + L::HDR_MEANS, means + 3 * n0, cnt * 12u, bar);
    if (BWD) {
        for (int t = 0; t < C; ++t) bulk_g2s(hdr + L::HDR_BODY + t * WT * 12, body + ((int64_t)t * N + n0) * 3, cnt * 12u, bar);
    } else {
#pragma unroll
        for (int ch = 0; ch < 3; ++ch) bulk_g2s(hdr + L::HDR_BODY + ch * WT * 4, body + (int64_t)ch * N + n0, cnt * 4u, bar);
    }
    if (vis)
        for (int t = 0; t < C; ++t) bulk_g2s(hdr + L::HDR_VIS + t * WT, vis + (int64_t)t * N + n0, cnt, bar);
}

__device__ __forceinline__ void warp_init(WarpCtx &c, unsigned char *smem, int region_bytes, int stages, int hslots, int hdr_bytes, int64_t N)
{
    c.warp = __shfl_sync(0xffffffffu, (int)(threadIdx.x >> 5), 0);
    c.stage0 = smem_u32(smem) + (unsigned)c.warp * (unsigned)region_bytes;
    c.hdr = c.stage0 + (unsigned)stages * STAGE_BYTES;
    c.scr = c.hdr + (unsigned)hslots * (unsigned)hdr_bytes;
    c.bars = c.stage0 + (unsigned)region_bytes - 64u;
    c.N = N;
    if ((threadIdx.x & 31) == 0) {
        for (int s = 0; s < 4; ++s) { mbar_init(bar_full(c, s), 1); mbar_init(bar_hfull(c, s), 1); }
        mbar_init_fence();
    }
    __syncwarp();
}

// the 22 values of a lobe pair for this lane, as 11 pairs (lobe l, lobe l+1). Every value is read with its own
// 32-bit load: 128-bit loads would deliver (w,x,y,z) of ONE lobe in adjacent registers, and turning that into
// same-component pairs costs moves. The 16-byte stride makes the quat/shape loads 4-way bank conflicted: 88
// shared-memory wavefronts per pair and warp, well inside the shared-memory pipe's budget.
struct PairRegs { f2 qw, qx, qy, qz, l1, l2, k, phi, w0, w1, w2; };
__device__ __forceinline__ void load_pair(unsigned stage, int lane, PairRegs &r)
{
    const unsigned q = stage + lane * 16, sh = q + 2 * WT * 16;
    r.qw = pack(lds32(q), lds32(q + WT * 16)); r.qx = pack(lds32(q + 4), lds32(q + WT * 16 + 4));
    r.qy = pack(lds32(q + 8), lds32(q + WT * 16 + 8)); r.qz = pack(lds32(q + 12), lds32(q + WT * 16 + 12));
    r.l1 = pack(lds32(sh), lds32(sh + WT * 16)); r.l2 = pack(lds32(sh + 4), lds32(sh + WT * 16 + 4));
    r.k = pack(lds32(sh + 8), lds32(sh + WT * 16 + 8)); r.phi = pack(lds32(sh + 12), lds32(sh + WT * 16 + 12));
    const unsigned w = stage + 4 * WT * 16 + lane * 4;
    r.w0 = pack(lds32(w), lds32(w + 3 * WT * 4));
    r.w1 = pack(lds32(w + WT * 4), lds32(w + 4 * WT * 4));
    r.w2 = pack(lds32(w + 2 * WT * 4), lds32(w + 5 * WT * 4));
}

__device__ __forceinline__ void direction(float mx, float my, float mz, const float *campos, int c, float &dx, float &dy, float &dz, float &inv)
{
    const float ex = mx - __ldg(campos + 3 * c), ey = my - __ldg(campos + 3 * c + 1), ez = mz - __ldg(campos + 3 * c + 2);
    const float r2 = fmaf(ex, ex, fmaf(ey, ey, ez * ez));
    inv = f_rsqrt(r2);
    inv = inv * fmaf(-0.5f * r2, inv * inv, 1.5f);          // one Newton step
    dx = ex * inv; dy = ey * inv; dz = ez * inv;
}

#ifndef NASG_TILE_SKIP
#define NASG_TILE_SKIP 0            // 1: a camera no lane of the warp sees is skipped (branches cost the iid case ~5 %)
#endif
#ifndef NASG_TILE_FWD_STAGES
#define NASG_TILE_FWD_STAGES 3
#endif
#ifndef NASG_TILE_BWD_STAGES
#define NASG_TILE_BWD_STAGES 2
#endif
#ifndef NASG_TILE_FWD_HSLOTS
#define NASG_TILE_FWD_HSLOTS 2
#endif
#ifndef NASG_TILE_FWD_MINB
#define NASG_TILE_FWD_MINB (512 / NASG_TB)
#endif
constexpr int TILE_BWD_HSLOTS = 1;  // backward: shared memory is the limit (2 blocks of 256 threads per SM)
// The barrier block at the end of a warp's region is 64 bytes: full[4] at 0..31, hfull[4] at 32..63.
static_assert(NASG_TILE_FWD_STAGES >= 1 && NASG_TILE_FWD_STAGES <= 4 && NASG_TILE_BWD_STAGES >= 1 && NASG_TILE_BWD_STAGES <= 4 &&
              NASG_TILE_FWD_HSLOTS >= 1 && NASG_TILE_FWD_HSLOTS <= 4 && TILE_BWD_HSLOTS <= 4,
              "more than 4 stages alias the header barriers, more than 4 header slots run into the next warp's region");
constexpr int TILE_BWD_MINB = 512 / TB;

// ---------------------------------------------------------------------------------------------
// forward
// ---------------------------------------------------------------------------------------------
template <int K, int CT, int MODE>
__global__ void __launch_bounds__(TB, NASG_TILE_FWD_MINB) nasg_fwd_tile_kernel(FwdParams p)
{
    extern __shared__ __align__(128) unsigned char smem_raw[];
    constexpr int STAGES = NASG_TILE_FWD_STAGES, NPAIR = K / 2, HS = NASG_TILE_FWD_HSLOTS;
    using L = TileLayout<CT, false>;
    const int lane = threadIdx.x & 31;
    const int C = p.C;
    WarpCtx c;
    warp_init(c, smem_raw, warp_region_bytes<CT, false>(STAGES, HS), STAGES, HS, L::HDR_BYTES, p.N);
    if (elect_one()) {
#pragma unroll
        for (int h = 0; h < HS; ++h) issue_header<CT, false, HS>(c, h, C, p.means, p.dc, p.vis);
#pragma unroll
        for (int m = 0; m < STAGES; ++m) issue_stage<K, STAGES>(c, m, p.quat, p.shape, p.amp);
    }
    int m = 0, slot = 0, hslot = 0;
    unsigned par = 0, hpar = 0;
    for (int i = 0;; ++i) {
        const int64_t n0 = warp_tile_start(c, i);
        if (n0 >= p.N) break;                              // (warp-uniform) this warp has no further tile
        const int64_t n = n0 + lane;
        const bool valid = n < p.N;
        // ---- header: means, dc, visibility bytes -> registers; then the slot is re-armed for the header HS tiles ahead
        mbar_wait(bar_hfull(c, hslot), hpar);
        const unsigned hdr = c.hdr + (unsigned)hslot * (unsigned)L::HDR_BYTES;
        const float mx = lds32(hdr + L::HDR_MEANS + lane * 12), my = lds32(hdr + L::HDR_MEANS + lane * 12 + 4),
                    mz = lds32(hdr + L::HDR_MEANS + lane * 12 + 8);
        const float dc0 = lds32(hdr + L::HDR_BODY + lane * 4), dc1 = lds32(hdr + L::HDR_BODY + WT * 4 + lane * 4),
                    dc2 = lds32(hdr + L::HDR_BODY + 2 * WT * 4 + lane * 4);
        unsigned mask = 0;
#pragma unroll
        for (int t = 0; t < CT; ++t)
            if (t < C) mask |= ((p.vis ? lds8(hdr + L::HDR_VIS + t * WT + lane) : 1u) != 0 ? 1u : 0u) << t;
        mask = valid ? mask : 0u;
        __syncwarp();
        if (elect_one()) issue_header<CT, false, HS>(c, i + HS, C, p.means, p.dc, p.vis);
        if (++hslot == HS) { hslot = 0; hpar ^= 1u; }
        const unsigned wmask = NASG_TILE_SKIP ? __reduce_or_sync(0xffffffffu, mask) : 0xfu;   // cameras some lane of this warp sees
        float dx[CT], dy[CT], dz[CT];
        f2 col[CT][3];
#pragma unroll
        for (int t = 0; t < CT; ++t) {
            float inv;
            direction(mx, my, mz, p.campos, t < C ? t : 0, dx[t], dy[t], dz[t], inv);
            col[t][0] = pack(dc0, 0.f); col[t][1] = pack(dc1, 0.f); col[t][2] = pack(dc2, 0.f);
        }
        // ---- lobe pairs
#pragma unroll
        for (int j = 0; j < NPAIR; ++j) {
            mbar_wait(bar_full(c, slot), par);
            PairRegs r;
            load_pair(c.stage0 + (unsigned)slot * STAGE_BYTES, lane, r);
            __syncwarp();
            if (elect_one()) issue_stage<K, STAGES>(c, m + STAGES, p.quat, p.shape, p.amp);
            if (!NASG_TILE_SKIP || wmask != 0) {       // (warp-uniform: a warp whose Gaussians are all culled skips the arithmetic)
                LobePair Lp; LobePairGrad Gd; f2 u0, u1, u2, u3;
                lobe_pair_setup<MODE, false>(r.qw, r.qx, r.qy, r.qz, r.l1, r.l2, r.k, r.phi, Lp, Gd, u0, u1, u2, u3);
#pragma unroll
                for (int t = 0; t < CT; ++t) {
                    // a camera slot is evaluated by the whole warp (iid masks: some lane always needs it); culled slots are
                    // zeroed at the store
                    if (!NASG_TILE_SKIP || (wmask & (1u << t))) {
                        EvalPair T;
                        const f2 G = lobe_pair_eval<false, MODE != 2>(Lp, dx[t], dy[t], dz[t], T);
                        col[t][0] = fma2(r.w0, G, col[t][0]);
                        col[t][1] = fma2(r.w1, G, col[t][1]);
                        col[t][2] = fma2(r.w2, G, col[t][2]);
                    }
                }
            }
            ++m;
            if (++slot == STAGES) { slot = 0; par ^= 1u; }
        }
        if (valid) {
#pragma unroll
            for (int t = 0; t < CT; ++t) {
                if (t < C) {
                    const bool on = mask & (1u << t);
                    float *o = p.colors + ((int64_t)t * p.N + n) * 3;
                    st_cs(o, on ? lo(col[t][0]) + hi(col[t][0]) : 0.f);
                    st_cs(o + 1, on ? lo(col[t][1]) + hi(col[t][1]) : 0.f);
                    st_cs(o + 2, on ? lo(col[t][2]) + hi(col[t][2]) : 0.f);
                }
            }
        }
    }
}

// ---------------------------------------------------------------------------------------------
// backward
// ---------------------------------------------------------------------------------------------
template <int K, int CT, int MODE>
__global__ void __launch_bounds__(TB, TILE_BWD_MINB) nasg_bwd_tile_kernel(BwdParams p)
{
    extern __shared__ __align__(128) unsigned char smem_raw[];
    constexpr int STAGES = NASG_TILE_BWD_STAGES, NPAIR = K / 2, HS = TILE_BWD_HSLOTS;
    using L = TileLayout<CT, true>;
    const int lane = threadIdx.x & 31;
    const int C = p.C;
    const int64_t N = p.N;
    WarpCtx c;
    warp_init(c, smem_raw, warp_region_bytes<CT, true>(STAGES, HS), STAGES, HS, L::HDR_BYTES, N);
    const unsigned scr_cam = c.scr + lane * 16;                          // + t * WT * 16: (dx,dy,dz,1/|Delta|) of camera t
    const unsigned scr_gc = scr_cam + CT * WT * 16;                      // + t * WT * 16: masked g_colors of camera t
    const unsigned scr_qs = scr_gc + CT * WT * 16;                       // + {0, WT * 16}
    if (elect_one()) {
        issue_header<CT, true, HS>(c, 0, C, p.means, p.g_colors, p.vis);
#pragma unroll
        for (int m = 0; m < STAGES; ++m) issue_stage<K, STAGES>(c, m, p.quat, p.shape, p.amp);
    }
    int m = 0, slot = 0;
    unsigned par = 0;
    for (int i = 0;; ++i) {
        const int64_t n0 = warp_tile_start(c, i);
        if (n0 >= N) break;                                // (warp-uniform)
        const int64_t n = n0 + lane;
        const bool valid = n < N;
        // ---- header: directions and masked g_colors -> this lane's scratch column; g_dc; then the slot is re-armed
        mbar_wait(bar_hfull(c, 0), i & 1);
        unsigned mask = 0;
        {
            const float mx = lds32(c.hdr + L::HDR_MEANS + lane * 12), my = lds32(c.hdr + L::HDR_MEANS + lane * 12 + 4),
                        mz = lds32(c.hdr + L::HDR_MEANS + lane * 12 + 8);
            float gdc0 = 0.f, gdc1 = 0.f, gdc2 = 0.f;
#pragma unroll
            for (int t = 0; t < CT; ++t) {
                const bool on = valid && t < C && (p.vis ? lds8(c.hdr + L::HDR_VIS + t * WT + lane) : 1u) != 0;
                mask |= (on ? 1u : 0u) << t;
                float4 cam, gc = make_float4(0.f, 0.f, 0.f, 0.f);
                direction(mx, my, mz, p.campos, t < C ? t : 0, cam.x, cam.y, cam.z, cam.w);
                if (on) {       // g_colors of a culled pair is never read as a value (it may be NaN or uninitialised)
                    const unsigned g = c.hdr + L::HDR_BODY + t * WT * 12 + lane * 12;
                    gc.x = lds32(g); gc.y = lds32(g + 4); gc.z = lds32(g + 8);
                }
                gdc0 += gc.x; gdc1 += gc.y; gdc2 += gc.z;
                sts128(scr_cam + t * WT * 16, cam);
                sts128(scr_gc + t * WT * 16, gc);
            }
            if (p.g_dc && valid) { st_cs(p.g_dc + n, gdc0); st_cs(p.g_dc + N + n, gdc1); st_cs(p.g_dc + 2 * N + n, gdc2); }
        }
        __syncwarp();
        if (elect_one()) issue_header<CT, true, HS>(c, i + 1, C, p.means, p.g_colors, p.vis);
        const unsigned wmask = NASG_TILE_SKIP ? __reduce_or_sync(0xffffffffu, mask) : 0xfu;   // cameras some lane of this warp sees
        float gd[CT][3];
#pragma unroll
        for (int t = 0; t < CT; ++t) gd[t][0] = gd[t][1] = gd[t][2] = 0.f;
        // ---- lobe pairs
#pragma unroll 1
        for (int j = 0; j < NPAIR; ++j) {
            mbar_wait(bar_full(c, slot), par);
            PairRegs r;
            load_pair(c.stage0 + (unsigned)slot * STAGE_BYTES, lane, r);
            __syncwarp();
            if (elect_one()) issue_stage<K, STAGES>(c, m + STAGES, p.quat, p.shape, p.amp);
            float4 gq0 = make_float4(0.f, 0.f, 0.f, 0.f), gq1 = gq0, gs0 = gq0, gs1 = gq0;
            AccPair A;
            acc_zero(A);
            if (!NASG_TILE_SKIP || wmask != 0) {       // (warp-uniform; a culled Gaussian in a live warp runs on g_colors = 0: exact zeros)
                LobePair Lp; LobePairGrad Gd;
                {
                    f2 qsw, qsx, qsy, qsz;
                    lobe_pair_setup<MODE, true>(r.qw, r.qx, r.qy, r.qz, r.l1, r.l2, r.k, r.phi, Lp, Gd, qsw, qsx, qsy, qsz);
                    sts64x2(scr_qs, qsw, qsx);
                    sts64x2(scr_qs + WT * 16, qsy, qsz);
                }
#pragma unroll
                for (int t = 0; t < CT; ++t) {
                    if (!NASG_TILE_SKIP || (wmask & (1u << t))) {          // a camera no lane of the warp sees is skipped
                        const float4 cam = lds128(scr_cam + t * WT * 16);
                        const float4 gc = lds128(scr_gc + t * WT * 16);     // zero for a culled slot: every contribution vanishes
                        EvalPair T;
                        const f2 G = lobe_pair_eval<true, MODE != 2>(Lp, cam.x, cam.y, cam.z, T);
                        f2 gx = splat(0.f), gy = splat(0.f), gz = splat(0.f);
                        lobe_pair_bwd<MODE != 2>(Lp, T, G, gc.x, gc.y, gc.z, r.w0, r.w1, r.w2, A, gx, gy, gz);
                        gd[t][0] += lo(gx) + hi(gx); gd[t][1] += lo(gy) + hi(gy); gd[t][2] += lo(gz) + hi(gz);
                    }
                }
                f2 qsw, qsx, qsy, qsz;
                lds64x2(scr_qs, qsw, qsx);
                lds64x2(scr_qs + WT * 16, qsy, qsz);
                lobe_pair_finish(Lp, Gd, A, qsw, qsx, qsy, qsz, gs0, gs1, gq0, gq1);
            }
            if (valid) {
                const int64_t ln = (int64_t)(2 * j) * N + n;
                if (p.g_quat) { st_cs4(p.g_quat + 4 * ln, gq0); st_cs4(p.g_quat + 4 * (ln + N), gq1); }
                if (p.g_shape) { st_cs4(p.g_shape + 4 * ln, gs0); st_cs4(p.g_shape + 4 * (ln + N), gs1); }
                if (p.g_amp) {
                    float *o = p.g_amp + (int64_t)(2 * j) * 3 * N + n;
                    st_cs(o, lo(A.gw0)); st_cs(o + N, lo(A.gw1)); st_cs(o + 2 * N, lo(A.gw2));
                    st_cs(o + 3 * N, hi(A.gw0)); st_cs(o + 4 * N, hi(A.gw1)); st_cs(o + 5 * N, hi(A.gw2));
                }
            }
            ++m;
            if (++slot == STAGES) { slot = 0; par ^= 1u; }
        }
        if (p.g_means && valid) {        // through d = Delta/|Delta|: (I - d d^T)/|Delta|   (gd of a culled slot is exactly 0)
            float gm0 = 0.f, gm1 = 0.f, gm2 = 0.f;
#pragma unroll
            for (int t = 0; t < CT; ++t) {
                const float4 cam = lds128(scr_cam + t * WT * 16);
                const float dg = fmaf(cam.x, gd[t][0], fmaf(cam.y, gd[t][1], cam.z * gd[t][2]));
                gm0 = fmaf(gd[t][0] - cam.x * dg, cam.w, gm0);
                gm1 = fmaf(gd[t][1] - cam.y * dg, cam.w, gm1);
                gm2 = fmaf(gd[t][2] - cam.z * dg, cam.w, gm2);
            }
            float *o = p.g_means + 3 * n;
            st_cs(o, gm0); st_cs(o + 1, gm1); st_cs(o + 2, gm2);
        }
    }
}

} // namespace lp

using lp::TB;
using lp::nasg_bwd_tile_kernel;
using lp::nasg_fwd_tile_kernel;
using lp::tile_smem_bytes;

// ---------------------------------------------------------------------------------------------
// launchers: persistent grid = resident blocks (occupancy API, cached per instantiation and device)
// ---------------------------------------------------------------------------------------------
// resident-grid size of a persistent tile kernel (occupancy query and shared-memory opt-in once per instantiation and device)
template <typename Kernel>
static int tile_grid(Kernel kernel, size_t smem, int64_t N, int *cached)
{
    return resident_grid(kernel, TB, smem, N, cached);
}

bool tile_path_ok(int64_t N, int K, int C, const void *means, const void *amp, const void *planar, const void *rows, const void *vis)
{
    auto a16 = [](const void *q) { return (reinterpret_cast<uintptr_t>(q) & 15u) == 0; };
    if (K % 2 != 0 || C > 4 || (N & 3) != 0) return false;
    if (vis && ((N & 15) != 0 || !a16(vis))) return false;
    return a16(means) && a16(amp) && (!planar || a16(planar)) && (!rows || a16(rows));
}

template <int K, int CT>
static cudaError_t launch_fwd_tile_kc(const FwdParams &p, int mode, cudaStream_t st)
{
    constexpr size_t smem = tile_smem_bytes<CT, false>(NASG_TILE_FWD_STAGES, NASG_TILE_FWD_HSLOTS);
    static int cache[3][64] = {{0}};
    if (mode == 1) nasg_fwd_tile_kernel<K, CT, 1><<<tile_grid(nasg_fwd_tile_kernel<K, CT, 1>, smem, p.N, cache[1]), TB, smem, st>>>(p);
    else if (mode == 0) nasg_fwd_tile_kernel<K, CT, 0><<<tile_grid(nasg_fwd_tile_kernel<K, CT, 0>, smem, p.N, cache[0]), TB, smem, st>>>(p);
    else nasg_fwd_tile_kernel<K, CT, 2><<<tile_grid(nasg_fwd_tile_kernel<K, CT, 2>, smem, p.N, cache[2]), TB, smem, st>>>(p);
    return cudaGetLastError();
}
template <int K>
static cudaError_t launch_fwd_tile_k(const FwdParams &p, int mode, cudaStream_t st)
{
    switch (p.C) {
    case 1: return launch_fwd_tile_kc<K, 1>(p, mode, st);
    case 2: return launch_fwd_tile_kc<K, 2>(p, mode, st);
    case 3: return launch_fwd_tile_kc<K, 3>(p, mode, st);
    default: return launch_fwd_tile_kc<K, 4>(p, mode, st);
    }
}
cudaError_t launch_nasg_fwd_tile(const FwdParams &p, int K, int mode, cudaStream_t st)
{
    switch (K) {
    case 2: return launch_fwd_tile_k<2>(p, mode, st);
    case 4: return launch_fwd_tile_k<4>(p, mode, st);
    case 8: return launch_fwd_tile_k<8>(p, mode, st);
    default: return cudaErrorInvalidValue;
    }
}

template <int K, int CT>
static cudaError_t launch_bwd_tile_kc(const BwdParams &p, int mode, cudaStream_t st)
{
    constexpr size_t smem = lp::tile_smem_bytes<CT, true>(NASG_TILE_BWD_STAGES, lp::TILE_BWD_HSLOTS);
    static int cache[3][64] = {{0}};
    if (mode == 1) nasg_bwd_tile_kernel<K, CT, 1><<<tile_grid(nasg_bwd_tile_kernel<K, CT, 1>, smem, p.N, cache[1]), TB, smem, st>>>(p);
    else if (mode == 0) nasg_bwd_tile_kernel<K, CT, 0><<<tile_grid(nasg_bwd_tile_kernel<K, CT, 0>, smem, p.N, cache[0]), TB, smem, st>>>(p);
    else nasg_bwd_tile_kernel<K, CT, 2><<<tile_grid(nasg_bwd_tile_kernel<K, CT, 2>, smem, p.N, cache[2]), TB, smem, st>>>(p);
    return cudaGetLastError();
}
template <int K>
static cudaError_t launch_bwd_tile_k(const BwdParams &p, int mode, cudaStream_t st)
{
    switch (p.C) {
    case 1: return launch_bwd_tile_kc<K, 1>(p, mode, st);
    case 2: return launch_bwd_tile_kc<K, 2>(p, mode, st);
    case 3: return launch_bwd_tile_kc<K, 3>(p, mode, st);
    default: return launch_bwd_tile_kc<K, 4>(p, mode, st);
    }
}
cudaError_t launch_nasg_bwd_tile(const BwdParams &p, int K, int mode, cudaStream_t st)
{
    switch (K) {
    case 2: return launch_bwd_tile_k<2>(p, mode, st);
    case 4: return launch_bwd_tile_k<4>(p, mode, st);
    case 8: return launch_bwd_tile_k<8>(p, mode, st);
    default: return cudaErrorInvalidValue;
    }
}

} // namespace nasg
