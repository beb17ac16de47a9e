// nasg_math.cuh — fp32 per-lobe arithmetic of the NASGabor path (device; also compilable for the host
// so that the conditioning can be studied without a GPU).
//
// What is computed is eq.(9)/(10) of arxiv/paper_2606_09794 and its gradient
// (PAPER.md:754-861 + DESIGN.md §4); HOW it is computed is the well-conditioned fp32 form of
// DESIGN.md §5, because the literal transcription loses the 1e-5 parity bar exactly where sharp
// lobes are bright:
//   * s^2 = 1-(d.z)^2 is formed as (d.x)^2 + (d.y)^2, never by subtraction;
//   * q = (1-|v|)/2 = s^2/(2(1+|v|)) is 1-kappa on the lobe side and kappa on the far side, so neither
//     1-v nor 1+v is formed by a cancelling subtraction; log2(kappa) = log2(1-q) by series for small q;
//   * kappa^(1+tau) - 1 uses an exp2m1 series when the argument is small;
//   * exponents are kept in base 2 (one ex2 for p*E/I including the normaliser), and MUFU
//     approximations (ex2, lg2, sin, cos, rcp, rsqrt) are used only where their error is relative to
//     the exponent or otherwise bounded well inside the tolerance (DESIGN.md §5 table).
// The XU (MUFU) pipe issues 16 lanes/clk/SM on B200 (measured, profiles/), 1/8 of the FP32 rate, so
// every reciprocal that can be shared is shared: 5 MUFU per forward lobe evaluation, 6 backward.
#pragma once

#include <cuda_runtime.h>
#include <math.h>

#define NASG_HD __host__ __device__ __forceinline__

namespace nasg {

constexpr float LOG2E = 1.4426950408889634f;
constexpr float LN2 = 0.6931471805599453f;
constexpr float TWO_PI = 6.283185307179586f;
constexpr float INV_TWO_PI = 0.15915494309189535f;
constexpr float TINY = 1e-30f;

// ---------------------------------------------------------------------------------------------
// MUFU wrappers (one XU instruction each on the device)
// ---------------------------------------------------------------------------------------------
#ifdef __CUDA_ARCH__
#define NASG_MUFU(name, ptx, hostexpr)                                                             \
    NASG_HD float name(float x) { float r; asm(ptx " %0, %1;" : "=f"(r) : "f"(x)); return r; }
#else
#define NASG_MUFU(name, ptx, hostexpr) NASG_HD float name(float x) { return hostexpr; }
#endif
NASG_MUFU(f_rcp, "rcp.approx.ftz.f32", 1.0f / x)
NASG_MUFU(f_rsqrt, "rsqrt.approx.ftz.f32", 1.0f / sqrtf(x))
NASG_MUFU(f_ex2, "ex2.approx.ftz.f32", exp2f(x))
NASG_MUFU(f_lg2, "lg2.approx.ftz.f32", log2f(x))
NASG_MUFU(f_sin, "sin.approx.ftz.f32", sinf(x))
NASG_MUFU(f_cos, "cos.approx.ftz.f32", cosf(x))
#undef NASG_MUFU
NASG_HD float f_exp(float x) { return f_ex2(x * LOG2E); }
// angle given in TURNS (theta/2pi): exact reduction to [-1/2,1/2] turns, then radians in [-pi,pi]
// (round-to-nearest via the 1.5*2^23 magic constant: two FADDs on the FMA pipe instead of an FRND on the
// XU pipe; exact for |t| < 2^22)
NASG_HD float reduce_turns(float t)
{
    const float n = (t + 12582912.0f) - 12582912.0f;
    return TWO_PI * (t - n);
}

// ---------------------------------------------------------------------------------------------
// accurate small-argument helpers (base 2)
// ---------------------------------------------------------------------------------------------
// log2(kappa) where kappa = 1-q if `upper` (v > 0: q is small near the lobe axis) else kappa = q.
// Series -log2e q (1 + q/2 + ... + q^5/6) for q < 1/16 on the upper side (truncation 8e-9 relative);
// lg2.approx otherwise (absolute error 2^-22 on |log2| >= 0.093: < 3e-6 relative, and an error that is
// relative to the exponent only perturbs G by |exponent| * 3e-6, which is largest, 1e-6 of the lobe
// peak, at exponent -1).
NASG_HD float log2_kappa(float q, bool upper)
{
    float p = fmaf(q, -LOG2E / 6.0f, -LOG2E / 5.0f);
    p = fmaf(q, p, -LOG2E / 4.0f);
    p = fmaf(q, p, -LOG2E / 3.0f);
    p = fmaf(q, p, -LOG2E / 2.0f);
    p = fmaf(q, p, -LOG2E);
    const float small = q * p;
    const float big = f_lg2(upper ? 1.0f - q : q);
    return (upper && q < 0.0625f) ? small : big;
}
// 2^x - 1 for x <= 0; also returns 2^x. Series for |x| < 1/8 (truncation 7e-9 relative), ex2 otherwise.
NASG_HD float exp2m1_neg(float x, float &two_x)
{
    float p = fmaf(x, 1.3333558e-3f, 9.6181291e-3f);   // ln2^5/120, ln2^4/24
    p = fmaf(x, p, 5.5504109e-2f);                       // ln2^3/6
    p = fmaf(x, p, 0.24022651f);                         // ln2^2/2
    p = fmaf(x, p, LN2);
    const float small = x * p;
    const float e = f_ex2(x);
    const bool s = x > -0.125f;
    two_x = s ? small + 1.0f : e;
    return s ? small : e - 1.0f;
}
// g(x) = (x coth x - 1)/x^2, x > 0   (d ln sinhc(x)/dx = x g(x)). Straight-line: the caller passes
// ix ~ 1/x, e = e^{-2x} and i1e ~ 1/(1-e) (it has them anyway); series below x = 0.7, closed form above.
NASG_HD float g_fun(float x, float ix, float e, float i1e)
{
    const float x2 = x * x;
    float p = fmaf(x2, 2.1377799e-5f, -2.1164021e-4f);
    p = fmaf(x2, p, 2.1164021e-3f);
    p = fmaf(x2, p, -2.2222222e-2f);
    const float small = fmaf(x2, p, 0.33333333f);
    const float big = fmaf(ix, 1.0f - ix, 2.0f * ix * e * i1e);
    return x < 0.7f ? small : big;
}

// ---------------------------------------------------------------------------------------------
// per-lobe, camera-independent set-up
// ---------------------------------------------------------------------------------------------
struct Lobe {
    float Xx, Xy, Xz, Yx, Yy, Yz, Zx, Zy, Zz; // columns of R(q/|q|)
    float a;                                   // Lambda/lambda - 1
    float lam2e;                               // 2 lambda log2(e)
    float kt, pt;                              // k/2pi, phi/2pi (carrier angle in turns)
    float lgI;                                 // log2(1/(2 I)): normaliser and the carrier's 1/2, folded into the exponent
};
struct LobeBwd {        // extra camera-independent terms of the backward pass
    float qw, qx, qy, qz, inv_qn;  // unit quaternion and 1/|q|
    float lam2, k;                 // 2 lambda, k
    float one_pa;                  // 1 + a = Lambda/lambda
    float nA;                      // (1+a) d ln I / d a        = -1/2 + Lambda D
    float nL;                      // lambda d ln I / d lambda  = 2 lambda e^{-2 lambda}/(1-e^{-2 lambda}) - 1 + Lambda D
    float nk;                      // d ln I / d k
};

// lgI = log2(1/(2I)) for I of eq.(10) (EXACT) or of NASG (approximate); if GRAD also the
// log-derivative terms of I. D = Psi_Lambda/(1+Psi).
//
// Straight-line code: both analytic branches of Psi (k < Lambda: sinhc of a real argument; k >= Lambda:
// the continuation S(s), reading R4) are evaluated on clamped arguments and selected per lane. With iid
// lobes nearly every warp holds lanes of both kinds, so a divergent branch would execute both sides
// anyway, and it would cut the set-up into basic blocks whose dependent MUFU chains (rsqrt -> rcp -> ex2
// -> rcp ...) the scheduler cannot overlap with each other or with the quaternion frame. The only branch
// left is warp-uniform: the k >= Lambda side is skipped when no lane of the warp needs it (always in cfg4).
template <bool EXACT, bool GRAD>
NASG_HD void normaliser(float l1, float l2, float Lam, float lam, float k, float &lgI, float &nA,
                        float &nL, float &nk)
{
    const float em = f_exp(-2.0f * lam);
    // 1 - e^{-2 lambda}, epsilon = 0 (R8): by subtraction, or by its series where that would cancel
    const float x = 2.0f * lam;
    float ps = fmaf(x, -1.0f / 720.0f, 1.0f / 120.0f);
    ps = fmaf(x, ps, -1.0f / 24.0f);
    ps = fmaf(x, ps, 1.0f / 6.0f);
    ps = fmaf(x, ps, -0.5f);
    ps = fmaf(x, ps, 1.0f);
    const float one_m = lam > 0.125f ? 1.0f - em : x * ps;
    // 1/(2I) = lambda sqrt(1+a) / (2 pi (1-e^{-2 lambda}) (1+Psi));  lambda sqrt(1+a) = e^{(l1+l2)/2}
    const float lg_root = 0.5f * LOG2E * (l1 + l2);
    float dl = 0.f;
    if (GRAD) dl = x * em * f_rcp(one_m) - 1.0f;                          // lambda d ln(base)/d lambda
    if (!EXACT) {
        lgI = lg_root - f_lg2(2.0f * TWO_PI * one_m);                     // NASG: I = 2 pi (1-e^{-2 lambda})/(lambda sqrt(1+a))
        if (GRAD) { nA = -0.5f; nL = dl; nk = 0.f; }
        return;
    }
    const float s = (Lam - k) * (Lam + k);                                // Lambda^2 - k^2
    const bool real_r = s > 0.05f;
    // ---- k < Lambda:  Psi = (Lambda/r) e^{r-Lambda} (1-e^{-2r})/(1-e^{-2 Lambda}),  r-Lambda = -k^2/(Lambda+r)
    const float sm = fmaxf(s, 0.05f);
    const float ir = f_rsqrt(sm), r = sm * ir;
    const float del = k * k * f_rcp(Lam + r);                             // Lambda - r
    const float ed = f_exp(-del);                                          // e^{r - Lambda}
    const float e2r = f_exp(-2.0f * r), e2L = e2r * ed * ed;              // e^{-2 Lambda} = e^{-2r} e^{-2(Lambda-r)}
    const float i1L = f_rcp(1.0f - e2L);
    float Psi = Lam * ir * ed * (1.0f - e2r) * i1L;
    float LD = 0.f, dk = 0.f;                                             // Lambda dPsi/dLambda, dPsi/dk
    if (GRAD) {
        const float i1r = f_rcp(1.0f - e2r), iL = f_rcp(Lam);
        const float gr = g_fun(r, ir, e2r, i1r);
        // g(r) - g(Lambda): without cancellation for r >= 4, plain difference below
        const float tail = 2.0f * (ir * e2r * i1r - iL * e2L * i1L);
        const float dg_big = fmaf(del * ir * iL, 1.0f - (Lam + r) * ir * iL, tail);
        const float dg = r >= 4.0f ? dg_big : gr - g_fun(Lam, iL, e2L, i1L);
        LD = Psi * Lam * Lam * dg;                                        // = Psi Lambda^2 (g(r) - g(Lambda))
        dk = -Psi * k * gr;
    }
    // ---- k >= Lambda (or |s| tiny): S(s) = sinhc(sqrt(s)) continued to s < 0 (reading R4), S' = dS/ds
#ifdef __CUDA_ARCH__
    if (__any_sync(__activemask(), !real_r))       // (called under divergent control flow: active lanes only)
#else
    if (!real_r)
#endif
    {
        const float sc = fminf(fmaxf(s, -0.05f), 0.05f);
        const float S_ser = fmaf(sc, fmaf(sc, fmaf(sc, 1.9841270e-4f, 8.3333333e-3f), 0.16666667f), 1.0f);
        const float Sp_ser = fmaf(sc, fmaf(sc, fmaf(sc, 1.1022928e-5f, 5.9523810e-4f), 1.6666667e-2f), 0.16666667f);
        const float sn = fminf(s, -0.05f);
        const float irho = f_rsqrt(-sn), rho = -sn * irho;
        const float ang = reduce_turns(rho * INV_TWO_PI);
        const float S_trig = f_sin(ang) * irho;
        const float Sp_trig = (f_cos(ang) - S_trig) * f_rcp(2.0f * sn);
        const bool ser = s > -0.05f;
        const float S = ser ? S_ser : S_trig, Sp = ser ? Sp_ser : Sp_trig;
        const float eL = f_exp(-Lam);
        const float i1 = f_rcp(1.0f - eL * eL);
        const float ish = 2.0f * eL * i1;                                 // 1/sinh(Lambda)
        const float Psi2 = Lam * S * ish;
        Psi = real_r ? Psi : Psi2;
        if (GRAD) {
            const float coth = (1.0f + eL * eL) * i1;
            const float LD2 = Psi2 + 2.0f * Lam * Lam * Lam * Sp * ish - Psi2 * Lam * coth;
            const float dk2 = -2.0f * k * Lam * Sp * ish;
            LD = real_r ? LD : LD2;
            dk = real_r ? dk : dk2;
        }
    }
    lgI = lg_root - f_lg2(TWO_PI * one_m * (1.0f + Psi));
    if (GRAD) {
        const float i1p = f_rcp(1.0f + Psi);
        const float LamD = LD * i1p;
        nA = -0.5f + LamD;
        nL = dl + LamD;
        nk = dk * i1p;
    }
}

// MODE: 0 = NASG normaliser (approximate), 1 = eq.(10) (exact), 2 = pure NASG: no carrier (k = phi = 0 assumed,
// shape.z/.w ignored), for which both normalisers coincide (Psi(k=0) = 1)
template <int MODE, bool GRAD>
NASG_HD void lobe_setup(const float4 q, const float4 sp, Lobe &L, LobeBwd &B)
{
    const float qq = q.x * q.x + q.y * q.y + q.z * q.z + q.w * q.w;
    float inv_qn = f_rsqrt(qq);
    inv_qn = inv_qn * fmaf(-0.5f * qq, inv_qn * inv_qn, 1.5f);            // one Newton step
    const float w = q.x * inv_qn, x = q.y * inv_qn, y = q.z * inv_qn, z = q.w * inv_qn;
    const float x2 = x + x, y2 = y + y, z2 = z + z;
    L.Xx = 1.0f - fmaf(y2, y, z2 * z); L.Xy = fmaf(x2, y, z2 * w); L.Xz = fmaf(x2, z, -y2 * w);
    L.Yx = fmaf(x2, y, -z2 * w); L.Yy = 1.0f - fmaf(x2, x, z2 * z); L.Yz = fmaf(y2, z, x2 * w);
    L.Zx = fmaf(x2, z, y2 * w); L.Zy = fmaf(y2, z, -x2 * w); L.Zz = 1.0f - fmaf(x2, x, y2 * y);
    // relative errors of Lambda, lambda only scale the exponent (benign), so ex2.approx is enough
    const float lam = f_exp(sp.y);
    const float one_pa = f_exp(sp.x - sp.y);
    const float Lam = lam * one_pa;
    L.a = fmaxf(one_pa - 1.0f, 0.0f);
    L.lam2e = 2.0f * LOG2E * lam;
    L.kt = MODE == 2 ? 0.f : sp.z * INV_TWO_PI; L.pt = MODE == 2 ? 0.f : sp.w * INV_TWO_PI;
    float nA = 0.f, nL = 0.f, nk = 0.f;
    normaliser<MODE == 1, GRAD>(sp.x, sp.y, Lam, lam, sp.z, L.lgI, nA, nL, nk);
    if (GRAD) {
        B.qw = w; B.qx = x; B.qy = y; B.qz = z; B.inv_qn = inv_qn;
        B.lam2 = 2.0f * lam; B.k = sp.z;
        B.one_pa = one_pa; B.nA = nA; B.nL = nL; B.nk = nk;
    }
}

// ---------------------------------------------------------------------------------------------
// per (lobe, camera) evaluation
// ---------------------------------------------------------------------------------------------
struct EvalTerms {      // what the backward needs from the recomputed forward
    float u, v, uu, inv_s2, tau, Lk, kp, em1, inv_2kappa, Gh, sn;
};

// G = H p E / I at direction (dx,dy,dz) (eq.(9) over eq.(10)). With FULL also fills the terms the
// backward needs. MUFU count: rcp, lg2, ex2, ex2, cos (+ sin with FULL).
template <bool FULL, bool CARRIER = true>
NASG_HD float lobe_eval(const Lobe &L, float dx, float dy, float dz, EvalTerms &T)
{
    const float u = fmaf(dx, L.Xx, fmaf(dy, L.Xy, dz * L.Xz));
    const float om = fmaf(dx, L.Yx, fmaf(dy, L.Yy, dz * L.Yz));
    const float v = fmaf(dx, L.Zx, fmaf(dy, L.Zy, dz * L.Zz));
    const float uu = u * u;
    const float s2 = fmaxf(fmaf(om, om, uu), TINY);          // 1 - v^2 without cancellation
    const float w2 = fmaf(fabsf(v), 2.0f, 2.0f);             // 2 (1 + |v|)
    const float rw = f_rcp(s2 * w2);                         // one reciprocal serves 1/s^2 and 1/(1+|v|)
    const float inv_s2 = rw * w2;
    const float q = s2 * (s2 * rw);                          // (1 - |v|)/2 = s^2 / (2 (1 + |v|))
    const float tau = L.a * uu * inv_s2;                     // a (d.x)^2 / (1 - (d.z)^2)
    const bool upper = v > 0.0f;
    const float L2 = log2_kappa(q, upper);                   // log2 kappa
    const float x1 = fmaf(tau, L2, L2);                      // (1+tau) log2 kappa
    float kp;
    const float em1 = exp2m1_neg(x1, kp);                    // kappa^(1+tau) - 1, kappa^(1+tau)
    const float arg = fmaf(L.lam2e, em1, fmaf(tau, L2, L.lgI));   // log2( p E / (2 I) )
    float Gh = f_ex2(arg);
    Gh = (s2 <= TINY && !upper) ? 0.0f : Gh;                 // d = -z: G = 0 (eq.(9), third case)
    const float ang = CARRIER ? reduce_turns(fmaf(L.kt, u, L.pt)) : 0.f;     // k d.x + phi  (mod 2 pi)
    const float G = CARRIER ? fmaf(Gh, f_cos(ang), Gh) : Gh + Gh;            // (1 + cos)/2 * p E / I   (no carrier: H = 1)
    if (FULL) {
        T.u = u; T.v = v; T.uu = uu; T.inv_s2 = inv_s2; T.tau = tau; T.Lk = LN2 * L2; T.kp = kp; T.em1 = em1;
        T.inv_2kappa = upper ? 2.0f * s2 * rw : 0.5f * w2 * inv_s2;      // 1/(1+v)
        T.Gh = Gh; T.sn = CARRIER ? f_sin(ang) : 0.f;
    }
    return G;
}

// ---------------------------------------------------------------------------------------------
// packed f32x2 evaluation: TWO cameras per instruction (device only)
// ---------------------------------------------------------------------------------------------
// On sm_100a FFMA2/FMUL2/FADD2 occupy the FP32 pipe for two cycles but only ONE issue slot, and the
// scheduler fills the other slot with ALU/XU/LSU work (measured: 4 FFMA2 + 8 FMNMX issue in 8.4
// cycles, profiles/). The camera loop is issue-bound, so the same arithmetic as lobe_eval, done on a
// pair of cameras, costs ~40% fewer issue slots. Rounding is per lane and identical to the scalar form.
#ifdef __CUDACC__
__device__ __forceinline__ float2 splat(float s) { return make_float2(s, s); }
__device__ __forceinline__ float2 mul2(float2 a, float2 b) { return __fmul2_rn(a, b); }
__device__ __forceinline__ float2 add2(float2 a, float2 b) { return __fadd2_rn(a, b); }
__device__ __forceinline__ float2 fma2(float2 a, float2 b, float2 c) { return __ffma2_rn(a, b, c); }
__device__ __forceinline__ float2 sub2(float2 a, float2 b) { return __ffma2_rn(b, make_float2(-1.0f, -1.0f), a); }   // a - b, one rounding

struct EvalTerms2 {
    float2 u, v, uu, inv_s2, tau, Lk, kp, em1, inv_2kappa, Gh, sn;
};

// lobe_eval for a pair of directions (dx.x,dy.x,dz.x), (dx.y,dy.y,dz.y)
// `bias` is added to the base-2 exponent of each half: 0 for a live camera slot, -1e30 for a culled one
// (then p E / I = 0 and every gradient contribution of the slot vanishes without a select).
template <bool FULL, bool CARRIER = true>
__device__ __forceinline__ float2 lobe_eval2(const Lobe &L, float2 dx, float2 dy, float2 dz, float2 bias, EvalTerms2 &T)
{
    const float2 u = fma2(dx, splat(L.Xx), fma2(dy, splat(L.Xy), mul2(dz, splat(L.Xz))));
    const float2 om = fma2(dx, splat(L.Yx), fma2(dy, splat(L.Yy), mul2(dz, splat(L.Yz))));
    const float2 v = fma2(dx, splat(L.Zx), fma2(dy, splat(L.Zy), mul2(dz, splat(L.Zz))));
    const float2 uu = mul2(u, u);
    float2 s2 = fma2(om, om, uu);                                  // 1 - v^2 without cancellation
    s2.x = fmaxf(s2.x, TINY); s2.y = fmaxf(s2.y, TINY);
    const float2 w2 = fma2(make_float2(fabsf(v.x), fabsf(v.y)), splat(2.0f), splat(2.0f));   // 2 (1 + |v|)
    const float2 sw = mul2(s2, w2);
    const float2 rw = make_float2(f_rcp(sw.x), f_rcp(sw.y));
    const float2 inv_s2 = mul2(rw, w2);
    const float2 s2rw = mul2(s2, rw);                              // 1/(2 (1 + |v|))
    const float2 q = mul2(s2, s2rw);                               // (1 - |v|)/2
    const float2 tau = mul2(mul2(splat(L.a), uu), inv_s2);
    const bool up0 = v.x > 0.0f, up1 = v.y > 0.0f;
    // log2 kappa (log2_kappa)
    float2 p = fma2(q, splat(-LOG2E / 6.0f), splat(-LOG2E / 5.0f));
    p = fma2(q, p, splat(-LOG2E / 4.0f));
    p = fma2(q, p, splat(-LOG2E / 3.0f));
    p = fma2(q, p, splat(-LOG2E / 2.0f));
    p = fma2(q, p, splat(-LOG2E));
    const float2 lsmall = mul2(q, p);
    const float2 omq = sub2(splat(1.0f), q);
    const float big0 = f_lg2(up0 ? omq.x : q.x), big1 = f_lg2(up1 ? omq.y : q.y);
    const float2 L2 = make_float2((up0 && q.x < 0.0625f) ? lsmall.x : big0, (up1 && q.y < 0.0625f) ? lsmall.y : big1);
    const float2 x1 = fma2(tau, L2, L2);                           // (1+tau) log2 kappa
    // kappa^(1+tau) - 1 (exp2m1_neg)
    float2 pe = fma2(x1, splat(1.3333558e-3f), splat(9.6181291e-3f));
    pe = fma2(x1, pe, splat(5.5504109e-2f));
    pe = fma2(x1, pe, splat(0.24022651f));
    pe = fma2(x1, pe, splat(LN2));
    const float2 esmall = mul2(x1, pe);
    const float2 ebig = add2(make_float2(f_ex2(x1.x), f_ex2(x1.y)), splat(-1.0f));
    const float2 em1 = make_float2(x1.x > -0.125f ? esmall.x : ebig.x, x1.y > -0.125f ? esmall.y : ebig.y);
    const float2 arg = fma2(splat(L.lam2e), em1, fma2(tau, L2, add2(splat(L.lgI), bias)));   // log2( p E / (2 I) )
    float2 Gh = make_float2(f_ex2(arg.x), f_ex2(arg.y));
    Gh.x = (s2.x <= TINY && !up0) ? 0.0f : Gh.x;                   // d = -z: G = 0 (eq.(9), third case)
    Gh.y = (s2.y <= TINY && !up1) ? 0.0f : Gh.y;
    // carrier: angle in turns, exact reduction to [-1/2, 1/2] (reduce_turns); without carrier H = 1
    float2 ang = splat(0.f), G;
    if (CARRIER) {
        const float2 t = fma2(splat(L.kt), u, splat(L.pt));
        const float2 n = add2(add2(t, splat(12582912.0f)), splat(-12582912.0f));
        ang = mul2(sub2(t, n), splat(TWO_PI));
        G = fma2(Gh, make_float2(f_cos(ang.x), f_cos(ang.y)), Gh);
    } else {
        G = add2(Gh, Gh);
    }
    if (FULL) {
        T.u = u; T.v = v; T.uu = uu; T.inv_s2 = inv_s2; T.tau = tau; T.Lk = mul2(splat(LN2), L2);
        T.kp = add2(em1, splat(1.0f)); T.em1 = em1;
        const float2 hi = add2(s2rw, s2rw), lo = mul2(mul2(splat(0.5f), w2), inv_s2);   // 1/(1+v) on the lobe side / far side
        T.inv_2kappa = make_float2(up0 ? hi.x : lo.x, up1 ? hi.y : lo.y);
        T.Gh = Gh; T.sn = CARRIER ? make_float2(f_sin(ang.x), f_sin(ang.y)) : splat(0.f);
    }
    return G;
}
#endif // __CUDACC__

} // namespace nasg
