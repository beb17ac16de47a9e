// nasg_rec_kernels.cu — NASGabor forward / backward on the TILE-RECORD parameter layout ("layout v2", include/nasg.h:
// nasg_rec_*), the headline path on sm_100a. Even lobe counts (K = 2, 4, 8), C <= 4 cameras.
//
// Why a second layout. The kernels are issue-bound, not HBM-bound (profiles/r2_*): with the structure-of-arrays rows
// of layout v1 a warp tile of 32 Gaussians is 24-29 separate row segments, and every one costs a bulk-copy instruction
// plus ~7 uniform-datapath instructions of 64-bit address arithmetic (20 % of the forward's, 17 % of the backward's
// executed instructions), the 128-bit quaternion / shape loads must be re-assembled into lobe pairs with moves, and
// every gradient store needs its own 64-bit row address. In the record layout everything a warp tile needs is ONE
// contiguous, 16-byte aligned block:
//
//   record of tile T (32 Gaussians n = 32 T + lane), floats:
//     [  0 ..  95]  means, planar:  x[32] y[32] z[32]
//     [ 96 .. 191]  dc (c0), planar: r[32] g[32] b[32]
//     [192 + 704 j + 64 c + 2 lane + h]   component c of lobe 2j+h, for lobe pair j < K/2,
//                    c = 0..10: quat w, x, y, z | log Lambda, log lambda, k, phi | amplitude r, g, b
//   (6 + 11 K floats per Gaussian: the same bytes as layout v1; lanes past N in the last record are padding.)
//
// so a lobe pair is one 2,816-byte bulk copy, its 11 operand pairs are 11 conflict-free 64-bit shared-memory loads that
// land as packed f32x2 registers (lobe l, lobe l+1) with no moves, and the gradient record (same layout) is written
// with 64-bit stores at immediate offsets from one per-lane pointer. colors / g_colors [C,N,3] and vis [C,N] keep the
// shapes the neighbouring stages (rasteriser) use.
//
// Structure (as nasg_tile_kernels.cu): persistent grid; every WARP runs its own pipeline over its tiles with bulk
// copies (cp.async.bulk, the TMA engine) issued by one elected lane and completed on mbarriers of that warp; warps
// never wait for each other (no __syncthreads, no atomics). Arithmetic: lobe pairs on packed f32x2 (nasg_lp_math.cuh).
#include <type_traits>
#include "bulk_common.cuh"
#include "nasg_internal.h"
#include "nasg_lp_math.cuh"
#include "pipe_common.cuh"

namespace nasg {
namespace lp {      // (the names of nasg_lp_math.cuh hide the camera-pair helpers of nasg_math.cuh in here)
namespace rec {

using namespace bulk;

#ifndef NASG_REC_FWD_TB
#define NASG_REC_FWD_TB 256
#endif
#ifndef NASG_REC_BWD_TB
#define NASG_REC_BWD_TB 256
#endif
#ifndef NASG_REC_FWD_MINB
#define NASG_REC_FWD_MINB 2
#endif
#ifndef NASG_REC_BWD_MINB
#define NASG_REC_BWD_MINB 2
#endif
constexpr int FWD_TB = NASG_REC_FWD_TB, BWD_TB = NASG_REC_BWD_TB;     // threads per block (warps are independent: any multiple of 32)
constexpr int WT = 32;                  // Gaussians per tile record
constexpr int HDR_FLOATS = 6 * WT;      // means + dc
constexpr int HDR_BYTES = HDR_FLOATS * 4;       // 768
// PK = parameter kind of the record: 0 = quaternion + (log Lambda, log lambda, k, phi) + amplitude: 11 components per lobe;
//      1 = the paper's own record (Table 8, Supplementary C): 3 frame angles + (lambda, a, k) + amplitude, all raw
//          (pre-activation), no phase: 9 components per lobe (3 + 9 K appearance floats)
//      2 = an isotropic function of Table 6 (MODE = 0 Spherical Gaussian, 1 Spherical Beta, 2 Spherical
//          Cauchy): axis (3, unnormalised) + raw shape value + amplitude: 7 components per lobe
//      3 = kind 0 with the quaternion and the amplitude stored as bfloat16 (fp32 arithmetic):
//          per pair 4 x 128 B (quat: one 32-bit word per lane = bf16 of lobe 2j | bf16 of lobe 2j+1 << 16), 4 x 256 B (shape,
//          fp32 pairs), 3 x 128 B (amplitude, bf16 pairs) = 1,920 B; the header and the GRADIENT record stay fp32 (kind 0)
//      4 = the Anisotropic Spherical Gaussian of Table 6: quaternion + (raw mu, raw lambda) + amplitude:
//          9 components per lobe (MODE unused: 0)
template <int PK> struct Rec {
    static constexpr int NCOMP = PK == 2 ? 7 : (PK == 1 || PK == 4) ? 9 : 11;
    static constexpr int PAIR_FLOATS = PK == 3 ? 480 : NCOMP * 2 * WT;          // 32-bit words of a pair
    static constexpr int PAIR_BYTES = PAIR_FLOATS * 4;        // 2816 | 2304 | 1792 | 1920
    static constexpr int GPK = PK == 3 ? 0 : PK;             // layout of the gradient record
    __host__ __device__ static constexpr int rec_floats(int K) { return HDR_FLOATS + (K / 2) * PAIR_FLOATS; }
};

#ifndef NASG_REC_FWD_STAGES
#define NASG_REC_FWD_STAGES 3
#endif
#ifndef NASG_REC_BWD_STAGES
#define NASG_REC_BWD_STAGES 2
#endif
#ifndef NASG_REC_FWD_HSLOTS
#define NASG_REC_FWD_HSLOTS 2
#endif
// The barrier block at the end of a warp's region is 64 bytes: full[4] at 0..31, hfull[4] at 32..63 (bar_full / bar_hfull).
static_assert(NASG_REC_FWD_STAGES >= 1 && NASG_REC_FWD_STAGES <= 4 && NASG_REC_BWD_STAGES >= 1 && NASG_REC_BWD_STAGES <= 4 &&
              NASG_REC_FWD_HSLOTS >= 1 && NASG_REC_FWD_HSLOTS <= 4,
              "more than 4 stages alias the header barriers, more than 4 header slots run into the next warp's region");

// ---- shared memory: one private region per warp ---------------------------------------------------
// [ stage 0 | ... | stage S-1 ][ header slot 0 | ... ][ scratch (backward) ][ mbarriers: full[4], hfull[4] ]
// header slot: record header (means, dc: 768 B) | backward: g_colors float [CT][32][3] | vis uint8 [CT][32]
// scratch (backward, per-lane columns): cam float4 [CT][32] = (dx,dy,dz,1/|Delta|) | gcm float4 [CT][32] = masked
//          g_colors | qs 2 x (f2,f2) [32] = qhat 2/|q| of the current pair
template <int CT, bool BWD, int PK> struct Layout {
    static constexpr int PAIR_BYTES = Rec<PK>::PAIR_BYTES;
    static constexpr int H_GC = HDR_BYTES;
    static constexpr int H_VIS = H_GC + (BWD ? CT * WT * 12 : 0);
    static constexpr int H_BYTES = H_VIS + ((CT * WT + 127) / 128) * 128;
    static constexpr int SCRATCH = BWD ? (2 * CT + (PK == 1 ? 3 : (PK == 2 || PK == 4) ? 0 : 2)) * WT * 16 : 0;     // (PK 0 and 3: 2)   // cam, gcm, parked frame terms (qs | trig | none)
    __host__ __device__ static constexpr int region(int stages, int hslots) { return stages * PAIR_BYTES + hslots * H_BYTES + SCRATCH + 64; }
};

struct Warp {                            // warp-uniform state
    unsigned stage0, hdr0, scr, bars;    // shared-memory addresses (u32) inside this warp's region
    int tile0, tstride, T;               // first tile of this warp, tiles between two of its tiles, number of tiles
    unsigned last_cnt;                   // Gaussians in the last tile (1..32)
};

// cursor of the copies that are issued ahead (all lanes keep it: warp-uniform values stay in uniform registers)
struct StageCursor { const char *src; int tile, j; };
struct HdrCursor { const char *src; const char *gc; const uint8_t *vis; int tile; };

template <int NPAIR, int PAIR_BYTES>
__device__ __forceinline__ void stage_advance(StageCursor &s, int tstride, int64_t rec_jump)
{
    s.src += PAIR_BYTES;
    if (++s.j == NPAIR) { s.j = 0; s.tile += tstride; s.src += rec_jump; }
}
// (elected lane) lobe pair under the cursor -> stage slot `dst`, completing on `bar`
template <int PAIR_BYTES>
__device__ __forceinline__ void stage_issue(const StageCursor &s, int T, unsigned dst, unsigned bar)
{
    if (s.tile < T) {
        fence_proxy_async();        // the lanes' reads of the slot (generic proxy) before the refill (async proxy): bulk_common.cuh
        mbar_expect_tx(bar, PAIR_BYTES);
        bulk_g2s(dst, s.src, PAIR_BYTES, bar);
    }
}
// (elected lane) record header (+ backward: g_colors rows; + visibility bytes) of the tile under the cursor
template <int CT, bool BWD>
__device__ __forceinline__ void hdr_issue(const HdrCursor &h, const Warp &w, unsigned dst, unsigned bar, bool bulk_rows, int64_t N)
{
    using L = Layout<CT, BWD, 0>;           // (the header slot does not depend on the parameter kind)
    if (h.tile < w.T) {
        const unsigned cnt = h.tile == w.T - 1 ? w.last_cnt : (unsigned)WT;
        unsigned bytes = HDR_BYTES;
        if (bulk_rows) bytes += (BWD ? CT * 12u * cnt : 0u) + (h.vis ? CT * cnt : 0u);
        fence_proxy_async();        // the lanes' reads of the slot (generic proxy) before the refill (async proxy): bulk_common.cuh
        mbar_expect_tx(bar, bytes);
        bulk_g2s(dst, h.src, HDR_BYTES, bar);
        if (bulk_rows) {
            if (BWD) {
                const char *g = h.gc;
#pragma unroll
                for (int t = 0; t < CT; ++t) { bulk_g2s(dst + L::H_GC + t * WT * 12, g, 12u * cnt, bar); g += N * 12; }
            }
            if (h.vis) {
                const uint8_t *v = h.vis;
#pragma unroll
                for (int t = 0; t < CT; ++t) { bulk_g2s(dst + L::H_VIS + t * WT, v, cnt, bar); v += N; }
            }
        }
    }
}
template <bool BWD>
__device__ __forceinline__ void hdr_advance(HdrCursor &h, int tstride, int rec_bytes)
{
    h.tile += tstride;
    h.src += (int64_t)tstride * rec_bytes;
    if (BWD) h.gc += (int64_t)tstride * (WT * 12);
    if (h.vis) h.vis += (int64_t)tstride * WT;
}

template <int CT, bool BWD, int PK>
__device__ __forceinline__ void warp_init(Warp &w, unsigned char *smem, int stages, int hslots, int64_t N)
{
    using L = Layout<CT, BWD, PK>;
    constexpr int NWARP = (BWD ? BWD_TB : FWD_TB) / 32;
    const int warp = __shfl_sync(0xffffffffu, (int)(threadIdx.x >> 5), 0);
    const int region = L::region(stages, hslots);
    w.stage0 = smem_u32(smem) + (unsigned)warp * (unsigned)region;
    w.hdr0 = w.stage0 + (unsigned)stages * L::PAIR_BYTES;
    w.scr = w.hdr0 + (unsigned)hslots * (unsigned)L::H_BYTES;
    w.bars = w.stage0 + (unsigned)region - 64u;
    w.T = (int)((N + WT - 1) / WT);
    w.last_cnt = (unsigned)(N - (int64_t)(w.T - 1) * WT);
    w.tile0 = (int)blockIdx.x * NWARP + warp;
    w.tstride = (int)gridDim.x * NWARP;
    if ((threadIdx.x & 31) == 0) {
        for (int s = 0; s < 8; ++s) mbar_init(w.bars + 8u * s, 1);
        mbar_init_fence();
    }
    __syncwarp();
}
__device__ __forceinline__ unsigned bar_full(const Warp &w, int s) { return w.bars + 8u * s; }
__device__ __forceinline__ unsigned bar_hfull(const Warp &w, int h) { return w.bars + 32u + 8u * h; }

// the operand pairs (lobe 2j, lobe 2j+1) of this lane: 64-bit loads, conflict-free, no re-assembly
template <int PK> struct PairRegs { f2 v[Rec<PK>::NCOMP]; };
__device__ __forceinline__ f2 bf16x2_to_f2(unsigned w)        // (bf16 lo | bf16 hi << 16) -> packed fp32 pair: exact
{
    return pack(__uint_as_float(w << 16), __uint_as_float(w & 0xffff0000u));
}
__device__ __forceinline__ unsigned lds32u(unsigned addr) { return *reinterpret_cast<const unsigned *>(__cvta_shared_to_generic(addr)); }
template <int PK>
__device__ __forceinline__ void load_pair(unsigned stage, int lane, PairRegs<PK> &r)
{
    if constexpr (PK == 3) {
        const unsigned h = stage + lane * 4, a = stage + 512 + lane * 8;
#pragma unroll
        for (int c = 0; c < 4; ++c) r.v[c] = bf16x2_to_f2(lds32u(h + 128 * c));
#pragma unroll
        for (int c = 0; c < 4; ++c) r.v[4 + c] = lds64<f2>(a + 256 * c);
#pragma unroll
        for (int c = 0; c < 3; ++c) r.v[8 + c] = bf16x2_to_f2(lds32u(h + 1536 + 128 * c));
    } else {
        const unsigned a = stage + lane * 8;
#pragma unroll
        for (int c = 0; c < Rec<PK>::NCOMP; ++c) r.v[c] = lds64<f2>(a + 256 * c);
    }
}
// set-up of the pair from its record components; w = the (activated) amplitudes
template <int PK, int MODE, bool GRAD>
__device__ __forceinline__ void setup_pair(const PairRegs<PK> &r, LobePair &Lp, LobePairGrad &Gd, f2 (&park)[6], f2 &w0, f2 &w1, f2 &w2)
{
    if constexpr (PK == 0 || PK == 3) {
        lobe_pair_setup<MODE, GRAD>(r.v[0], r.v[1], r.v[2], r.v[3], r.v[4], r.v[5], r.v[6], r.v[7], Lp, Gd, park[0], park[1], park[2], park[3]);
        w0 = r.v[8]; w1 = r.v[9]; w2 = r.v[10];
    } else if constexpr (PK == 1) {
        PaperTrig tr;
        lobe_pair_setup_paper<MODE, GRAD>(r.v[0], r.v[1], r.v[2], r.v[3], r.v[4], r.v[5], Lp, Gd, tr);
        if (GRAD) { park[0] = tr.st; park[1] = tr.cp; park[2] = tr.sp; park[3] = tr.cu; park[4] = tr.su; park[5] = tr.su; }
        w0 = tanh2(r.v[6]); w1 = tanh2(r.v[7]); w2 = tanh2(r.v[8]);
    }
}

__device__ __forceinline__ void direction(float mx, float my, float mz, const float *campos, int c, float &dx, float &dy, float &dz, float &inv)
{
    const float ex = mx - __ldg(campos + 3 * c), ey = my - __ldg(campos + 3 * c + 1), ez = mz - __ldg(campos + 3 * c + 2);
    const float r2 = fmaf(ex, ex, fmaf(ey, ey, ez * ez));
    inv = f_rsqrt(r2);
    inv = inv * fmaf(-0.5f * r2, inv * inv, 1.5f);          // one Newton step
    dx = ex * inv; dy = ey * inv; dz = ez * inv;
}
__device__ __forceinline__ void st_cs2(float *p, f2 v)
{
    unsigned long long u;
    memcpy(&u, &v, 8);
    __stcs(reinterpret_cast<unsigned long long *>(p), u);
}

// ---------------------------------------------------------------------------------------------
// forward
// ---------------------------------------------------------------------------------------------
// SKIP (NASG_HINT_COHERENT_VIS): test per warp which cameras are seen by any lane and skip the others; a separate
// instantiation, because the extra control flow costs the iid case ~5 % of the forward (measured), which never skips anything.
template <int K, int CT, int MODE, int PK, bool SKIP>
__global__ void __launch_bounds__(FWD_TB, NASG_REC_FWD_MINB) nasg_rec_fwd_kernel(RecFwdParams p)
{
    extern __shared__ __align__(128) unsigned char smem_raw[];
    constexpr int S = NASG_REC_FWD_STAGES, NPAIR = K / 2, HS = NASG_REC_FWD_HSLOTS;
    using L = Layout<CT, false, PK>;
    constexpr int PAIR_BYTES = Rec<PK>::PAIR_BYTES;
    constexpr int RECB = Rec<PK>::rec_floats(K) * 4;
    const int lane = threadIdx.x & 31;
    const int64_t N = p.N;
    const bool bulk_rows = p.bulk_rows != 0;
    Warp w;
    warp_init<CT, false, PK>(w, smem_raw, S, HS, N);
    const int64_t rec_jump = (int64_t)w.tstride * RECB - (int64_t)NPAIR * PAIR_BYTES;
    const char *params = reinterpret_cast<const char *>(p.params);
    StageCursor sc{params + (int64_t)w.tile0 * RECB + HDR_BYTES, w.tile0, 0};
    HdrCursor hc{params + (int64_t)w.tile0 * RECB, nullptr, p.vis ? p.vis + (int64_t)w.tile0 * WT : nullptr, w.tile0};
    // prologue: HS headers and S stages in flight
#pragma unroll
    for (int h = 0; h < HS; ++h) {
        if (elect_one()) hdr_issue<CT, false>(hc, w, w.hdr0 + h * L::H_BYTES, bar_hfull(w, h), bulk_rows, N);
        hdr_advance<false>(hc, w.tstride, RECB);
    }
#pragma unroll
    for (int m = 0; m < S; ++m) {
        if (elect_one()) stage_issue<PAIR_BYTES>(sc, w.T, w.stage0 + m * PAIR_BYTES, bar_full(w, m));
        stage_advance<NPAIR, PAIR_BYTES>(sc, w.tstride, rec_jump);
    }
    int slot = 0, hslot = 0;
    unsigned par = 0, hpar = 0;
    for (int tile = w.tile0; tile < w.T; tile += w.tstride) {
        const int64_t n = (int64_t)tile * WT + lane;
        const bool valid = n < N;
        // ---- header: means, dc, visibility -> registers; then the slot is re-armed for the header HS tiles ahead
        const unsigned hdr = w.hdr0 + (unsigned)hslot * (unsigned)L::H_BYTES;
        mbar_wait(bar_hfull(w, hslot), hpar);
        const float mx = lds32(hdr + lane * 4), my = lds32(hdr + 128 + lane * 4), mz = lds32(hdr + 256 + lane * 4);
        const float dc0 = lds32(hdr + 384 + lane * 4), dc1 = lds32(hdr + 512 + lane * 4), dc2 = lds32(hdr + 640 + lane * 4);
        unsigned mask = 0;
        if (p.vis) {
#pragma unroll
            for (int t = 0; t < CT; ++t) {
                const unsigned b = bulk_rows ? lds8(hdr + L::H_VIS + t * WT + lane) : (valid ? (unsigned)p.vis[(int64_t)t * N + n] : 0u);
                mask |= (b != 0 ? 1u : 0u) << t;
            }
        } else {
            mask = (1u << CT) - 1u;
        }
        mask = valid ? mask : 0u;
        // cameras that SOME lane of this warp sees: with spatially coherent visibility (frustum culling of a sorted scene) whole
        // warps lose cameras and skip their evaluations; with iid masks wmask is full and the unrolled path below runs
        constexpr unsigned FULL = (1u << CT) - 1u;
        const unsigned wmask = SKIP ? __reduce_or_sync(0xffffffffu, mask) : FULL;     // (every lane takes part: never under a per-lane condition)
        __syncwarp();
        if (elect_one()) hdr_issue<CT, false>(hc, w, hdr, bar_hfull(w, hslot), bulk_rows, N);
        hdr_advance<false>(hc, w.tstride, RECB);
        if (++hslot == HS) { hslot = 0; hpar ^= 1u; }
        float dx[CT], dy[CT], dz[CT];
        f2 col[CT][3];
#pragma unroll
        for (int t = 0; t < CT; ++t) {
            float inv;
            direction(mx, my, mz, p.campos, t, dx[t], dy[t], dz[t], inv);
            col[t][0] = pack(dc0, 0.f); col[t][1] = pack(dc1, 0.f); col[t][2] = pack(dc2, 0.f);
        }
        // ---- lobe pairs. Two copies of the loop: ALL = every camera is seen by some lane (always with iid masks): straight-line
        // code, the CT evaluations of a pair interleave and the next pair's wait / loads / set-up overlap them; otherwise cameras
        // no lane sees are skipped with warp-uniform branches, and a tile culled in every camera skips all lobe arithmetic (F0).
        auto run_pairs = [&](auto all_tag) {
            constexpr bool ALL = decltype(all_tag)::value;
#pragma unroll
            for (int j = 0; j < NPAIR; ++j) {
                const unsigned stage = w.stage0 + (unsigned)slot * PAIR_BYTES;
                mbar_wait(bar_full(w, slot), par);
                PairRegs<PK> r;
                load_pair<PK>(stage, lane, r);
                __syncwarp();
                if (elect_one()) stage_issue<PAIR_BYTES>(sc, w.T, stage, bar_full(w, slot));
                stage_advance<NPAIR, PAIR_BYTES>(sc, w.tstride, rec_jump);
                if (++slot == S) { slot = 0; par ^= 1u; }
                if constexpr (PK == 2) {           // isotropic Table-6 function MODE
                    IsoPair Ip;
                    iso_pair_setup<MODE>(r.v[0], r.v[1], r.v[2], r.v[3], Ip);
#pragma unroll
                    for (int t = 0; t < CT; ++t) {
                        f2 u0, u1;
                        const f2 G = iso_pair_eval<MODE, false>(Ip, dx[t], dy[t], dz[t], u0, u1);
                        col[t][0] = fma2(r.v[4], G, col[t][0]);
                        col[t][1] = fma2(r.v[5], G, col[t][1]);
                        col[t][2] = fma2(r.v[6], G, col[t][2]);
                    }
                } else if constexpr (PK == 4) {    // Anisotropic Spherical Gaussian
                    AsgPair Ap; f2 q0, q1, q2, q3;
                    asg_pair_setup<false>(r.v[0], r.v[1], r.v[2], r.v[3], r.v[4], r.v[5], Ap, q0, q1, q2, q3);
#pragma unroll
                    for (int t = 0; t < CT; ++t) {
                        AsgEval T;
                        const f2 G = asg_pair_eval<false>(Ap, dx[t], dy[t], dz[t], T);
                        col[t][0] = fma2(r.v[6], G, col[t][0]);
                        col[t][1] = fma2(r.v[7], G, col[t][1]);
                        col[t][2] = fma2(r.v[8], G, col[t][2]);
                    }
                } else if (ALL || wmask != 0u) {
                    LobePair Lp; LobePairGrad Gd; f2 park[6], w0, w1, w2;
                    setup_pair<PK, MODE, false>(r, Lp, Gd, park, w0, w1, w2);
#pragma unroll
                    for (int t = 0; t < CT; ++t) {
                        if (ALL || (wmask & (1u << t))) {      // culled slots of a camera some lane sees are evaluated and zeroed at the store
                            EvalPair T;
                            const f2 G = lobe_pair_eval<false, MODE != 2>(Lp, dx[t], dy[t], dz[t], T);
                            col[t][0] = fma2(w0, G, col[t][0]);
                            col[t][1] = fma2(w1, G, col[t][1]);
                            col[t][2] = fma2(w2, G, col[t][2]);
                        }
                    }
                }
            }
        };
        if (!SKIP || PK == 2 || PK == 4 || wmask == FULL) run_pairs(std::true_type{});
        else run_pairs(std::false_type{});
        if (valid) {
            float *o = p.colors + n * 3;
#pragma unroll
            for (int t = 0; t < CT; ++t) {
                const bool on = mask & (1u << t);
                st_cs(o, on ? lo(col[t][0]) + hi(col[t][0]) : 0.f);
                st_cs(o + 1, on ? lo(col[t][1]) + hi(col[t][1]) : 0.f);
                st_cs(o + 2, on ? lo(col[t][2]) + hi(col[t][2]) : 0.f);
                o += N * 3;
            }
        }
    }
}

// ---------------------------------------------------------------------------------------------
// backward
// ---------------------------------------------------------------------------------------------
template <int K, int CT, int MODE, int PK, bool SKIP>
__global__ void __launch_bounds__(BWD_TB, NASG_REC_BWD_MINB) nasg_rec_bwd_kernel(RecBwdParams p)
{
    extern __shared__ __align__(128) unsigned char smem_raw[];
    constexpr int S = NASG_REC_BWD_STAGES, NPAIR = K / 2;
    using L = Layout<CT, true, PK>;
    constexpr int PAIR_BYTES = Rec<PK>::PAIR_BYTES, RECB = Rec<PK>::rec_floats(K) * 4;
    constexpr int GPAIR_FLOATS = Rec<Rec<PK>::GPK>::PAIR_FLOATS, GRECF = Rec<Rec<PK>::GPK>::rec_floats(K);     // gradient record
    const int lane = threadIdx.x & 31;
    const int64_t N = p.N;
    const bool bulk_rows = p.bulk_rows != 0;
    Warp w;
    warp_init<CT, true, PK>(w, smem_raw, S, 1, N);
    const unsigned scr_cam = w.scr + lane * 16;                          // + t * WT * 16: (dx,dy,dz,1/|Delta|) of camera t
    const unsigned scr_gc = scr_cam + CT * WT * 16;                      // + t * WT * 16: masked g_colors of camera t
    const unsigned scr_qs = scr_gc + CT * WT * 16;                       // + {0, WT * 16[, 2 WT * 16]}: parked frame terms
    const int64_t rec_jump = (int64_t)w.tstride * RECB - (int64_t)NPAIR * PAIR_BYTES;
    const char *params = reinterpret_cast<const char *>(p.params);
    StageCursor sc{params + (int64_t)w.tile0 * RECB + HDR_BYTES, w.tile0, 0};
    HdrCursor hc{params + (int64_t)w.tile0 * RECB, reinterpret_cast<const char *>(p.g_colors) + (int64_t)w.tile0 * (WT * 12),
                 p.vis ? p.vis + (int64_t)w.tile0 * WT : nullptr, w.tile0};
    if (elect_one()) hdr_issue<CT, true>(hc, w, w.hdr0, bar_hfull(w, 0), bulk_rows, N);
    hdr_advance<true>(hc, w.tstride, RECB);
#pragma unroll
    for (int m = 0; m < S; ++m) {
        if (elect_one()) stage_issue<PAIR_BYTES>(sc, w.T, w.stage0 + m * PAIR_BYTES, bar_full(w, m));
        stage_advance<NPAIR, PAIR_BYTES>(sc, w.tstride, rec_jump);
    }
    int slot = 0;
    unsigned par = 0, hpar = 0;
    for (int tile = w.tile0; tile < w.T; tile += w.tstride) {
        const int64_t n = (int64_t)tile * WT + lane;
        const bool valid = n < N;
        float *grec = p.g_params + (int64_t)tile * GRECF + lane;         // this lane's column of the gradient record
        // ---- header: directions and masked g_colors -> this lane's scratch column; g_dc; then the slot is re-armed
        mbar_wait(bar_hfull(w, 0), hpar);
        hpar ^= 1u;
        unsigned mask = 0;
        {
            const float mx = lds32(w.hdr0 + lane * 4), my = lds32(w.hdr0 + 128 + lane * 4), mz = lds32(w.hdr0 + 256 + lane * 4);
            float gdc0 = 0.f, gdc1 = 0.f, gdc2 = 0.f;
#pragma unroll
            for (int t = 0; t < CT; ++t) {
                bool on = valid;
                if (p.vis) on = on && (bulk_rows ? lds8(w.hdr0 + L::H_VIS + t * WT + lane) : (valid ? (unsigned)p.vis[(int64_t)t * N + n] : 0u)) != 0;
                float4 cam, gc = make_float4(0.f, 0.f, 0.f, 0.f);
                direction(mx, my, mz, p.campos, t, cam.x, cam.y, cam.z, cam.w);
                mask |= (on ? 1u : 0u) << t;
                if (on) {       // g_colors of a culled pair is never read as a value (it may be NaN or uninitialised)
                    if (bulk_rows) {
                        const unsigned g = w.hdr0 + L::H_GC + t * WT * 12 + lane * 12;
                        gc.x = lds32(g); gc.y = lds32(g + 4); gc.z = lds32(g + 8);
                    } else {
                        const float *g = p.g_colors + ((int64_t)t * N + n) * 3;
                        gc.x = __ldg(g); gc.y = __ldg(g + 1); gc.z = __ldg(g + 2);
                    }
                }
                gdc0 += gc.x; gdc1 += gc.y; gdc2 += gc.z;
                sts128(scr_cam + t * WT * 16, cam);
                sts128(scr_gc + t * WT * 16, gc);
            }
            if (valid) { st_cs(grec + 96, gdc0); st_cs(grec + 128, gdc1); st_cs(grec + 160, gdc2); }
        }
        constexpr unsigned FULL = (1u << CT) - 1u;
        const unsigned wmask = SKIP ? __reduce_or_sync(0xffffffffu, mask) : FULL;     // (every lane takes part: never under a per-lane condition)     // cameras some lane of this warp sees
        __syncwarp();
        if (elect_one()) hdr_issue<CT, true>(hc, w, w.hdr0, bar_hfull(w, 0), bulk_rows, N);
        hdr_advance<true>(hc, w.tstride, RECB);
        float gd[CT][3];
#pragma unroll
        for (int t = 0; t < CT; ++t) gd[t][0] = gd[t][1] = gd[t][2] = 0.f;
        // ---- lobe pairs
        float *gpair = grec + HDR_FLOATS + lane;                        // + 704 j + 64 c: pair (lobe 2j, 2j+1) of component c
#pragma unroll 1
        for (int j = 0; j < NPAIR; ++j) {
            const unsigned stage = w.stage0 + (unsigned)slot * PAIR_BYTES;
            mbar_wait(bar_full(w, slot), par);
            PairRegs<PK> r;
            load_pair<PK>(stage, lane, r);
            __syncwarp();
            if (elect_one()) stage_issue<PAIR_BYTES>(sc, w.T, stage, bar_full(w, slot));
            stage_advance<NPAIR, PAIR_BYTES>(sc, w.tstride, rec_jump);
            if (++slot == S) { slot = 0; par ^= 1u; }
            f2 g[Rec<PK>::NCOMP];
            if constexpr (PK == 2) {           // isotropic Table-6 function MODE
                IsoPair Ip;
                iso_pair_setup<MODE>(r.v[0], r.v[1], r.v[2], r.v[3], Ip);
                const f2 w0 = r.v[4], w1 = r.v[5], w2 = r.v[6];
                f2 gw0 = splat(0.f), gw1 = gw0, gw2 = gw0, gs = gw0, gzx = gw0, gzy = gw0, gzz = gw0;
#pragma unroll
                for (int t = 0; t < CT; ++t) {
                    const float4 cam = lds128(scr_cam + t * WT * 16);
                    const float4 gc = lds128(scr_gc + t * WT * 16);     // zero for a culled slot: every contribution vanishes
                    f2 Fv, Fr;
                    const f2 F = iso_pair_eval<MODE, true>(Ip, cam.x, cam.y, cam.z, Fv, Fr);
                    const f2 c0 = splat(gc.x), c1 = splat(gc.y), c2 = splat(gc.z);
                    const f2 gF = fma2(w0, c0, fma2(w1, c1, mul2(w2, c2)));             // dL/dF, eq.(6)
                    gw0 = fma2(F, c0, gw0); gw1 = fma2(F, c1, gw1); gw2 = fma2(F, c2, gw2);
                    gs = fma2(gF, Fr, gs);
                    const f2 gv = mul2(gF, Fv);                                         // v = d . zhat
                    gzx = fma2(gv, splat(cam.x), gzx); gzy = fma2(gv, splat(cam.y), gzy); gzz = fma2(gv, splat(cam.z), gzz);
                    const f2 gx = mul2(gv, Ip.zx), gy = mul2(gv, Ip.zy), gz = mul2(gv, Ip.zz);
                    gd[t][0] += lo(gx) + hi(gx); gd[t][1] += lo(gy) + hi(gy); gd[t][2] += lo(gz) + hi(gz);
                }
                // zhat = z/|z|: (I - zhat zhat^T)/|z|
                const f2 dot = fma2(Ip.zx, gzx, fma2(Ip.zy, gzy, mul2(Ip.zz, gzz)));
                g[0] = mul2(fma2(neg2(Ip.zx), dot, gzx), Ip.inv);
                g[1] = mul2(fma2(neg2(Ip.zy), dot, gzy), Ip.inv);
                g[2] = mul2(fma2(neg2(Ip.zz), dot, gzz), Ip.inv);
                g[3] = gs; g[4] = gw0; g[5] = gw1; g[6] = gw2;
            } else if constexpr (PK == 4) {    // Anisotropic Spherical Gaussian
                AsgPair Ap; f2 q0, q1, q2, q3;
                asg_pair_setup<true>(r.v[0], r.v[1], r.v[2], r.v[3], r.v[4], r.v[5], Ap, q0, q1, q2, q3);
                const f2 w0 = r.v[6], w1 = r.v[7], w2 = r.v[8];
                AsgAcc A;
                auto cam_bwd = [&](int t, auto first) {
                    const float4 cam = lds128(scr_cam + t * WT * 16);
                    const float4 gc = lds128(scr_gc + t * WT * 16);         // zero for a culled slot: every contribution vanishes
                    AsgEval T;
                    const f2 G = asg_pair_eval<true>(Ap, cam.x, cam.y, cam.z, T);
                    f2 gx = splat(0.f), gy = splat(0.f), gz = splat(0.f);
                    asg_pair_bwd<decltype(first)::value>(Ap, T, G, gc.x, gc.y, gc.z, w0, w1, w2, A, gx, gy, gz);
                    gd[t][0] += lo(gx) + hi(gx); gd[t][1] += lo(gy) + hi(gy); gd[t][2] += lo(gz) + hi(gz);
                };
                cam_bwd(0, std::true_type{});
#pragma unroll
                for (int t = 1; t < CT; ++t) cam_bwd(t, std::false_type{});
                asg_pair_finish(Ap, A, q0, q1, q2, q3, g[4], g[5], g[0], g[1], g[2], g[3]);
                g[6] = A.gw0; g[7] = A.gw1; g[8] = A.gw2;
            } else if (SKIP && wmask == 0u) {  // (warp-uniform) a tile culled in every camera: zero gradients, no arithmetic (F0)
#pragma unroll
                for (int c = 0; c < Rec<PK>::NCOMP; ++c) g[c] = splat(0.f);
            } else {
                LobePair Lp; LobePairGrad Gd;
                f2 w0, w1, w2;
                {       // frame terms the end of the pair needs (quaternion 2/|q| | sines and cosines of the angles) are parked in shared memory
                    f2 park[6];
                    setup_pair<PK, MODE, true>(r, Lp, Gd, park, w0, w1, w2);
                    sts64x2(scr_qs, park[0], park[1]);
                    sts64x2(scr_qs + WT * 16, park[2], park[3]);
                    if constexpr (PK == 1) sts64x2(scr_qs + 2 * WT * 16, park[4], park[5]);
                }
                AccPair A;
                auto cam_bwd = [&](int t, auto first) {
                    const float4 cam = lds128(scr_cam + t * WT * 16);
                    const float4 gc = lds128(scr_gc + t * WT * 16);         // zero for a culled slot: every contribution vanishes
                    EvalPair T;
                    const f2 G = lobe_pair_eval<true, MODE != 2>(Lp, cam.x, cam.y, cam.z, T);
                    f2 gx = splat(0.f), gy = splat(0.f), gz = splat(0.f);
                    lobe_pair_bwd<MODE != 2, decltype(first)::value>(Lp, T, G, gc.x, gc.y, gc.z, w0, w1, w2, A, gx, gy, gz);
                    gd[t][0] += lo(gx) + hi(gx); gd[t][1] += lo(gy) + hi(gy); gd[t][2] += lo(gz) + hi(gz);
                };
                if (!SKIP || wmask == FULL) {      // all camera slots, unrolled (the evaluations interleave); the first initialises the accumulators
                    cam_bwd(0, std::true_type{});
#pragma unroll
                    for (int t = 1; t < CT; ++t) cam_bwd(t, std::false_type{});
                } else {                           // some camera is seen by no lane of the warp: skip it (uniform branches)
                    acc_zero(A);
#pragma unroll
                    for (int t = 0; t < CT; ++t)
                        if (wmask & (1u << t)) cam_bwd(t, std::false_type{});
                }
                f2 park[6];
                lds64x2(scr_qs, park[0], park[1]);
                lds64x2(scr_qs + WT * 16, park[2], park[3]);
                if constexpr (PK == 1) {
                    lds64x2(scr_qs + 2 * WT * 16, park[4], park[5]);
                    const PaperTrig tr{park[0], park[1], park[2], park[3], park[4]};
                    lobe_pair_finish_paper<MODE>(Lp, Gd, A, tr, w0, w1, w2, g[0], g[1], g[2], g[3], g[4], g[5], g[6], g[7], g[8]);
                } else {
                    lobe_pair_finish2(Lp, Gd, A, park[0], park[1], park[2], park[3], g[4], g[5], g[6], g[7], g[0], g[1], g[2], g[3]);
                    g[8] = A.gw0; g[9] = A.gw1; g[10] = A.gw2;
                }
            }
            if (valid) {
#pragma unroll
                for (int c = 0; c < Rec<PK>::NCOMP; ++c) st_cs2(gpair + 64 * c, g[c]);
            }
            gpair += GPAIR_FLOATS;
        }
        if (valid) {        // through d = Delta/|Delta|: (I - d d^T)/|Delta|   (gd of a culled slot is exactly 0)
            float gm0 = 0.f, gm1 = 0.f, gm2 = 0.f;
#pragma unroll
            for (int t = 0; t < CT; ++t) {
                const float4 cam = lds128(scr_cam + t * WT * 16);
                const float dg = fmaf(cam.x, gd[t][0], fmaf(cam.y, gd[t][1], cam.z * gd[t][2]));
                gm0 = fmaf(gd[t][0] - cam.x * dg, cam.w, gm0);
                gm1 = fmaf(gd[t][1] - cam.y * dg, cam.w, gm1);
                gm2 = fmaf(gd[t][2] - cam.z * dg, cam.w, gm2);
            }
            st_cs(grec, gm0); st_cs(grec + 32, gm1); st_cs(grec + 64, gm2);
        }
    }
}

// ---------------------------------------------------------------------------------------------
// layout conversion: v1 arrays <-> tile records (one thread per record lane; pure data movement)
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) rec_pack_kernel(int64_t N, int K, const float *means, const float *quat, const float *shape,
                                                        const float *amp, const float *dc, float *rec)
{
    const int64_t n = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const int64_t T = (N + WT - 1) / WT;
    if (n >= T * WT) return;
    const int lane = (int)(n & 31);
    float *r = rec + (n >> 5) * Rec<0>::rec_floats(K);
    const bool valid = n < N;
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        r[c * WT + lane] = valid ? means[3 * n + c] : 0.f;
        r[(3 + c) * WT + lane] = valid ? dc[(int64_t)c * N + n] : 0.f;
    }
    for (int l = 0; l < K; ++l) {
        float *o = r + HDR_FLOATS + (l >> 1) * Rec<0>::PAIR_FLOATS + 2 * lane + (l & 1);
        float4 q = make_float4(1.f, 0.f, 0.f, 0.f), s = make_float4(0.f, 0.f, 0.f, 0.f);
        float a0 = 0.f, a1 = 0.f, a2 = 0.f;
        if (valid) {
            q = reinterpret_cast<const float4 *>(quat)[(int64_t)l * N + n];
            s = reinterpret_cast<const float4 *>(shape)[(int64_t)l * N + n];
            a0 = amp[((int64_t)l * 3 + 0) * N + n]; a1 = amp[((int64_t)l * 3 + 1) * N + n]; a2 = amp[((int64_t)l * 3 + 2) * N + n];
        }
        o[0] = q.x; o[64] = q.y; o[128] = q.z; o[192] = q.w;
        o[256] = s.x; o[320] = s.y; o[384] = s.z; o[448] = s.w;
        o[512] = a0; o[576] = a1; o[640] = a2;
    }
}
// bf16 records (kind 3): quaternion and amplitude rounded to bfloat16 (round to nearest even). A NaN stays a NaN (sign and
// upper payload kept, quiet bit set): the rounding increment would carry a NaN with low mantissa bits set out of the
// exponent field (0x7FFFFFFF -> 0x8000 = -0.0) and a NaN parameter would be stored as a finite number.
__device__ __forceinline__ unsigned short f2bf(float x)
{
    unsigned u = __float_as_uint(x);
    if ((u & 0x7fffffffu) > 0x7f800000u) return (unsigned short)((u >> 16) | 0x40u);
    u += 0x7fffu + ((u >> 16) & 1u);
    return (unsigned short)(u >> 16);
}
__global__ void __launch_bounds__(256) rec16_pack_kernel(int64_t N, int K, const float *means, const float *quat, const float *shape,
                                                          const float *amp, const float *dc, unsigned *rec)
{
    const int64_t n = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const int64_t T = (N + WT - 1) / WT;
    if (n >= T * WT) return;
    const int lane = (int)(n & 31);
    unsigned *r = rec + (n >> 5) * Rec<3>::rec_floats(K);
    const bool valid = n < N;
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        r[c * WT + lane] = __float_as_uint(valid ? means[3 * n + c] : 0.f);
        r[(3 + c) * WT + lane] = __float_as_uint(valid ? dc[(int64_t)c * N + n] : 0.f);
    }
    for (int j = 0; j < K / 2; ++j) {
        unsigned *o = r + HDR_FLOATS + j * Rec<3>::PAIR_FLOATS;
        float4 q[2], s[2]; float a[2][3];
#pragma unroll
        for (int h = 0; h < 2; ++h) {
            const int l = 2 * j + h;
            q[h] = make_float4(1.f, 0.f, 0.f, 0.f); s[h] = make_float4(0.f, 0.f, 0.f, 0.f); a[h][0] = a[h][1] = a[h][2] = 0.f;
            if (valid) {
                q[h] = reinterpret_cast<const float4 *>(quat)[(int64_t)l * N + n];
                s[h] = reinterpret_cast<const float4 *>(shape)[(int64_t)l * N + n];
                for (int ch = 0; ch < 3; ++ch) a[h][ch] = amp[((int64_t)l * 3 + ch) * N + n];
            }
        }
        const float qv[2][4] = {{q[0].x, q[0].y, q[0].z, q[0].w}, {q[1].x, q[1].y, q[1].z, q[1].w}};
        const float sv[2][4] = {{s[0].x, s[0].y, s[0].z, s[0].w}, {s[1].x, s[1].y, s[1].z, s[1].w}};
#pragma unroll
        for (int c = 0; c < 4; ++c) {
            o[32 * c + lane] = (unsigned)f2bf(qv[0][c]) | ((unsigned)f2bf(qv[1][c]) << 16);
            o[128 + 64 * c + 2 * lane] = __float_as_uint(sv[0][c]);
            o[128 + 64 * c + 2 * lane + 1] = __float_as_uint(sv[1][c]);
        }
#pragma unroll
        for (int c = 0; c < 3; ++c) o[384 + 32 * c + lane] = (unsigned)f2bf(a[0][c]) | ((unsigned)f2bf(a[1][c]) << 16);
    }
}
__global__ void __launch_bounds__(256) rec_unpack_kernel(int64_t N, int K, const float *rec, float *means, float *quat, float *shape,
                                                          float *amp, float *dc)
{
    const int64_t n = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (n >= N) return;
    const int lane = (int)(n & 31);
    const float *r = rec + (n >> 5) * Rec<0>::rec_floats(K);
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        if (means) means[3 * n + c] = r[c * WT + lane];
        if (dc) dc[(int64_t)c * N + n] = r[(3 + c) * WT + lane];
    }
    for (int l = 0; l < K; ++l) {
        const float *o = r + HDR_FLOATS + (l >> 1) * Rec<0>::PAIR_FLOATS + 2 * lane + (l & 1);
        if (quat) reinterpret_cast<float4 *>(quat)[(int64_t)l * N + n] = make_float4(o[0], o[64], o[128], o[192]);
        if (shape) reinterpret_cast<float4 *>(shape)[(int64_t)l * N + n] = make_float4(o[256], o[320], o[384], o[448]);
        if (amp) { amp[((int64_t)l * 3 + 0) * N + n] = o[512]; amp[((int64_t)l * 3 + 1) * N + n] = o[576]; amp[((int64_t)l * 3 + 2) * N + n] = o[640]; }
    }
}

} // namespace rec
} // namespace lp
namespace rec = lp::rec;

// ---------------------------------------------------------------------------------------------
// launchers: persistent grid = resident blocks (occupancy API, cached per instantiation and device)
// ---------------------------------------------------------------------------------------------
int64_t rec_total_floats(int64_t N, int K, int pk)
{
    return ((N + rec::WT - 1) / rec::WT) * (int64_t)(pk == 4 ? rec::Rec<4>::rec_floats(K) : pk == 3 ? rec::Rec<3>::rec_floats(K) : pk == 2 ? rec::Rec<2>::rec_floats(K) : pk == 1 ? rec::Rec<1>::rec_floats(K) : rec::Rec<0>::rec_floats(K));
}

template <typename Kernel>
static int rec_grid(Kernel kernel, int TB, size_t smem, int64_t N, int *cached)
{
    return resident_grid(kernel, TB, smem, N, cached);
}

template <int K, int CT, int PK, bool SKIP>
static cudaError_t launch_rec_fwd_kc(const RecFwdParams &p, int mode, cudaStream_t st)
{
    constexpr int TB = rec::FWD_TB;
    constexpr size_t smem = (size_t)(TB / 32) * rec::Layout<CT, false, PK>::region(NASG_REC_FWD_STAGES, NASG_REC_FWD_HSLOTS);
    static int cache[3][64] = {{0}};
    using namespace rec;
    if constexpr (PK == 4) {        // one function: MODE 0 only
        nasg_rec_fwd_kernel<K, CT, 0, PK, SKIP><<<rec_grid(nasg_rec_fwd_kernel<K, CT, 0, PK, SKIP>, TB, smem, p.N, cache[0]), TB, smem, st>>>(p);
    } else if (mode == 1) nasg_rec_fwd_kernel<K, CT, 1, PK, SKIP><<<rec_grid(nasg_rec_fwd_kernel<K, CT, 1, PK, SKIP>, TB, smem, p.N, cache[1]), TB, smem, st>>>(p);
    else if (mode == 0) nasg_rec_fwd_kernel<K, CT, 0, PK, SKIP><<<rec_grid(nasg_rec_fwd_kernel<K, CT, 0, PK, SKIP>, TB, smem, p.N, cache[0]), TB, smem, st>>>(p);
    else nasg_rec_fwd_kernel<K, CT, 2, PK, SKIP><<<rec_grid(nasg_rec_fwd_kernel<K, CT, 2, PK, SKIP>, TB, smem, p.N, cache[2]), TB, smem, st>>>(p);
    return cudaGetLastError();
}
template <int K, int PK>
static cudaError_t launch_rec_fwd_k(const RecFwdParams &p, int mode_and_hint, cudaStream_t st)
{
    const int mode = mode_and_hint & 0xff;
    const bool skip = (mode_and_hint & 0x100) != 0;           // NASG_HINT_COHERENT_VIS (quaternion records with C > 1 only)
    switch (p.C) {
    case 1: return (PK == 0 && 1 > 1 && skip) ? launch_rec_fwd_kc<K, 1, PK, PK == 0 && (1 > 1)>(p, mode, st) : launch_rec_fwd_kc<K, 1, PK, false>(p, mode, st);
    case 2: return (PK == 0 && 2 > 1 && skip) ? launch_rec_fwd_kc<K, 2, PK, PK == 0 && (2 > 1)>(p, mode, st) : launch_rec_fwd_kc<K, 2, PK, false>(p, mode, st);
    case 3: return (PK == 0 && 3 > 1 && skip) ? launch_rec_fwd_kc<K, 3, PK, PK == 0 && (3 > 1)>(p, mode, st) : launch_rec_fwd_kc<K, 3, PK, false>(p, mode, st);
    case 4: return (PK == 0 && 4 > 1 && skip) ? launch_rec_fwd_kc<K, 4, PK, PK == 0 && (4 > 1)>(p, mode, st) : launch_rec_fwd_kc<K, 4, PK, false>(p, mode, st);
    default: return cudaErrorInvalidValue;
    }
}
template <int PK>
static cudaError_t launch_rec_fwd_pk(const RecFwdParams &p, int K, int mode, cudaStream_t st)
{
    switch (K) {
    case 2: return launch_rec_fwd_k<2, PK>(p, mode, st);
    case 4: return launch_rec_fwd_k<4, PK>(p, mode, st);
    case 8: return launch_rec_fwd_k<8, PK>(p, mode, st);
    default: return cudaErrorInvalidValue;
    }
}
cudaError_t launch_nasg_rec_fwd(const RecFwdParams &p, int K, int mode, int pk, cudaStream_t st)
{
    return pk == 4 ? launch_rec_fwd_pk<4>(p, K, mode, st) : pk == 3 ? launch_rec_fwd_pk<3>(p, K, mode, st) : pk == 2 ? launch_rec_fwd_pk<2>(p, K, mode, st)
                   : pk == 1 ? launch_rec_fwd_pk<1>(p, K, mode, st) : launch_rec_fwd_pk<0>(p, K, mode, st);
}

template <int K, int CT, int PK, bool SKIP>
static cudaError_t launch_rec_bwd_kc(const RecBwdParams &p, int mode, cudaStream_t st)
{
    constexpr int TB = rec::BWD_TB;
    constexpr size_t smem = (size_t)(TB / 32) * rec::Layout<CT, true, PK>::region(NASG_REC_BWD_STAGES, 1);
    static int cache[3][64] = {{0}};
    using namespace rec;
    if constexpr (PK == 4) {        // one function: MODE 0 only
        nasg_rec_bwd_kernel<K, CT, 0, PK, SKIP><<<rec_grid(nasg_rec_bwd_kernel<K, CT, 0, PK, SKIP>, TB, smem, p.N, cache[0]), TB, smem, st>>>(p);
    } else if (mode == 1) nasg_rec_bwd_kernel<K, CT, 1, PK, SKIP><<<rec_grid(nasg_rec_bwd_kernel<K, CT, 1, PK, SKIP>, TB, smem, p.N, cache[1]), TB, smem, st>>>(p);
    else if (mode == 0) nasg_rec_bwd_kernel<K, CT, 0, PK, SKIP><<<rec_grid(nasg_rec_bwd_kernel<K, CT, 0, PK, SKIP>, TB, smem, p.N, cache[0]), TB, smem, st>>>(p);
    else nasg_rec_bwd_kernel<K, CT, 2, PK, SKIP><<<rec_grid(nasg_rec_bwd_kernel<K, CT, 2, PK, SKIP>, TB, smem, p.N, cache[2]), TB, smem, st>>>(p);
    return cudaGetLastError();
}
template <int K, int PK>
static cudaError_t launch_rec_bwd_k(const RecBwdParams &p, int mode_and_hint, cudaStream_t st)
{
    const int mode = mode_and_hint & 0xff;
    const bool skip = (mode_and_hint & 0x100) != 0;           // NASG_HINT_COHERENT_VIS (quaternion records with C > 1 only)
    switch (p.C) {
    case 1: return (PK == 0 && 1 > 1 && skip) ? launch_rec_bwd_kc<K, 1, PK, PK == 0 && (1 > 1)>(p, mode, st) : launch_rec_bwd_kc<K, 1, PK, false>(p, mode, st);
    case 2: return (PK == 0 && 2 > 1 && skip) ? launch_rec_bwd_kc<K, 2, PK, PK == 0 && (2 > 1)>(p, mode, st) : launch_rec_bwd_kc<K, 2, PK, false>(p, mode, st);
    case 3: return (PK == 0 && 3 > 1 && skip) ? launch_rec_bwd_kc<K, 3, PK, PK == 0 && (3 > 1)>(p, mode, st) : launch_rec_bwd_kc<K, 3, PK, false>(p, mode, st);
    case 4: return (PK == 0 && 4 > 1 && skip) ? launch_rec_bwd_kc<K, 4, PK, PK == 0 && (4 > 1)>(p, mode, st) : launch_rec_bwd_kc<K, 4, PK, false>(p, mode, st);
    default: return cudaErrorInvalidValue;
    }
}
template <int PK>
static cudaError_t launch_rec_bwd_pk(const RecBwdParams &p, int K, int mode, cudaStream_t st)
{
    switch (K) {
    case 2: return launch_rec_bwd_k<2, PK>(p, mode, st);
    case 4: return launch_rec_bwd_k<4, PK>(p, mode, st);
    case 8: return launch_rec_bwd_k<8, PK>(p, mode, st);
    default: return cudaErrorInvalidValue;
    }
}
cudaError_t launch_nasg_rec_bwd(const RecBwdParams &p, int K, int mode, int pk, cudaStream_t st)
{
    return pk == 4 ? launch_rec_bwd_pk<4>(p, K, mode, st) : pk == 3 ? launch_rec_bwd_pk<3>(p, K, mode, st) : pk == 2 ? launch_rec_bwd_pk<2>(p, K, mode, st)
                   : pk == 1 ? launch_rec_bwd_pk<1>(p, K, mode, st) : launch_rec_bwd_pk<0>(p, K, mode, st);
}

cudaError_t launch_rec_pack(int64_t N, int K, const float *means, const float *quat, const float *shape, const float *amp, const float *dc,
                            float *rec_out, cudaStream_t st)
{
    const int64_t threads = ((N + rec::WT - 1) / rec::WT) * rec::WT;
    rec::rec_pack_kernel<<<(unsigned)((threads + 255) / 256), 256, 0, st>>>(N, K, means, quat, shape, amp, dc, rec_out);
    return cudaGetLastError();
}
cudaError_t launch_rec16_pack(int64_t N, int K, const float *means, const float *quat, const float *shape, const float *amp, const float *dc,
                              float *rec_out, cudaStream_t st)
{
    const int64_t threads = ((N + rec::WT - 1) / rec::WT) * rec::WT;
    rec::rec16_pack_kernel<<<(unsigned)((threads + 255) / 256), 256, 0, st>>>(N, K, means, quat, shape, amp, dc, reinterpret_cast<unsigned *>(rec_out));
    return cudaGetLastError();
}
cudaError_t launch_rec_unpack(int64_t N, int K, const float *rec_in, float *means, float *quat, float *shape, float *amp, float *dc,
                              cudaStream_t st)
{
    rec::rec_unpack_kernel<<<(unsigned)((N + 255) / 256), 256, 0, st>>>(N, K, rec_in, means, quat, shape, amp, dc);
    return cudaGetLastError();
}

} // namespace nasg
