// nasg_lp_math.cuh — fp32 NASGabor arithmetic on LOBE PAIRS: the two halves of every f32x2 operand are
// lobes l and l+1 of one Gaussian (device; compiles for the host too, with scalar halves, so that the
// formulas can be checked without a GPU).
//
// What is computed: eq.(9)/(10) of arxiv/paper_2606_09794 and its gradient
// (PAPER.md:754-861 + DESIGN.md §4), in the well-conditioned fp32 form of DESIGN.md §5 (s^2 = u^2 + w^2,
// q = s^2/(2(1+|v|)), series for log2 kappa and 2^x - 1 near the lobe axis, base-2 exponents with the
// normaliser folded in). Why pairs of LOBES and not pairs of cameras (nasg_math.cuh: lobe_eval2):
//   * on sm_100a FFMA2/FMUL2/FADD2 hold the FP32 pipe for two cycles but take ONE issue slot, and the
//     kernels are issue-bound; with lobes in the halves the camera-independent set-up (quaternion frame,
//     eq.(10) and its log-derivatives: 27 % of the backward's instructions when it ran scalar) and the
//     frame/shape backward are packed as well as the evaluations, a single camera (C = 1) is packed too,
//     camera quantities (d, g_colors) enter as free scalar-broadcast operands, and the per-lobe sums over
//     cameras need no horizontal adds;
//   * the MUFU count per lobe set-up drops from 14 (21 with gradients) to 11 (13): both analytic
//     branches of Psi share their MUFU operations through argument selects, and reciprocals are shared
//     pairwise (1/x and 1/y from one rcp(x y)).
// The gradient with respect to the frame is accumulated as a rotation vector in the lobe's own frame,
//   g_theta = sum_c ( -g_v w, g_v u - g_u v, g_u w ),   (u, w, v) = (d.x, d.y, d.z),
// which follows from delta u = delta theta . (x cross d), delta v = delta theta . (z cross d) for
// R -> R (I + [delta theta]x); g_q = (2/|q|) qhat (x) (0, g_theta) is then already tangent to the unit
// sphere: no projection, no subtraction of nearly equal terms (4 accumulations instead of 6 per
// evaluation, 17 operations instead of 42 per lobe for the quaternion chain).
#pragma once

#include <cuda_runtime.h>
#include <math.h>

#include "nasg_math.cuh"      // MUFU wrappers (f_rcp, f_ex2, ...), constants

namespace nasg {
namespace lp {

// ---------------------------------------------------------------------------------------------
// f32x2 helpers. On the device a pair lives in ONE 64-bit register (an aligned register pair) for its whole
// life: the CUDA float2 intrinsics (__ffma2_rn ...) take a struct of two floats, which the compiler splits
// into scalars and re-assembles at every use — 14 % of the executed instructions of the first version of the
// tile kernels were IMAD.MOV pair assembly. Halves are taken out (lo/hi) only for the scalar-only operations
// (MUFU, compare + select, min/max, |x|) and put back with pack().
// ---------------------------------------------------------------------------------------------
#if defined(__CUDA_ARCH__) && !defined(NASG_LP_SCALAR)
typedef unsigned long long f2;
__device__ __forceinline__ f2 pack(float lo, float hi) { f2 r; asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi)); return r; }
__device__ __forceinline__ float lo(f2 v) { float a; asm("{ .reg .b32 t; mov.b64 {%0, t}, %1; }" : "=f"(a) : "l"(v)); return a; }
__device__ __forceinline__ float hi(f2 v) { float b; asm("{ .reg .b32 t; mov.b64 {t, %0}, %1; }" : "=f"(b) : "l"(v)); return b; }
__device__ __forceinline__ f2 mul2(f2 a, f2 b) { f2 r; asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b)); return r; }
__device__ __forceinline__ f2 add2(f2 a, f2 b) { f2 r; asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b)); return r; }
__device__ __forceinline__ f2 fma2(f2 a, f2 b, f2 c) { f2 r; asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c)); return r; }
#else
struct f2 { float x, y; };
NASG_HD f2 pack(float lo, float hi) { f2 r; r.x = lo; r.y = hi; return r; }
NASG_HD float lo(f2 v) { return v.x; }
NASG_HD float hi(f2 v) { return v.y; }
NASG_HD f2 mul2(f2 a, f2 b) { return pack(a.x * b.x, a.y * b.y); }
NASG_HD f2 add2(f2 a, f2 b) { return pack(a.x + b.x, a.y + b.y); }
NASG_HD f2 fma2(f2 a, f2 b, f2 c) { return pack(fmaf(a.x, b.x, c.x), fmaf(a.y, b.y, c.y)); }
#endif
NASG_HD f2 splat(float s) { return pack(s, s); }
NASG_HD f2 sub2(f2 a, f2 b) { return fma2(b, splat(-1.0f), a); }          // a - b, one rounding
NASG_HD f2 neg2(f2 a) { return pack(-lo(a), -hi(a)); }
NASG_HD f2 scl2(f2 a, float s) { return mul2(a, splat(s)); }
NASG_HD f2 abs2(f2 a) { return pack(fabsf(lo(a)), fabsf(hi(a))); }
NASG_HD f2 max2(f2 a, float m) { return pack(fmaxf(lo(a), m), fmaxf(hi(a), m)); }
NASG_HD f2 sel2(bool cx, bool cy, f2 a, f2 b) { return pack(cx ? lo(a) : lo(b), cy ? hi(a) : hi(b)); }
#define NASG_LP_MAP(name, fn) NASG_HD f2 name(f2 a) { return pack(fn(lo(a)), fn(hi(a))); }
NASG_LP_MAP(rcp2, f_rcp)
NASG_LP_MAP(rsqrt2, f_rsqrt)
NASG_LP_MAP(ex2_2, f_ex2)
NASG_LP_MAP(lg2_2, f_lg2)
NASG_LP_MAP(sin2, f_sin)
NASG_LP_MAP(cos2, f_cos)
#undef NASG_LP_MAP

// ---------------------------------------------------------------------------------------------
// camera-independent state of a lobe pair
// ---------------------------------------------------------------------------------------------
struct LobePair {
    f2 Xx, Xy, Xz, Yx, Yy, Yz, Zx, Zy, Zz;   // columns of R(q/|q|)
    f2 a;                                     // Lambda/lambda - 1
    f2 lam2e;                                 // 2 lambda log2(e)
    f2 k, phi;                                // carrier frequency and phase (radians)
    f2 lgI;                                   // log2(1/(2 I)): normaliser and the carrier's 1/2 in the exponent
};
struct LobePairGrad {   // log-derivatives of the normaliser
    f2 nA;              // (1+a) d ln I / d a        = -1/2 + Lambda D
    f2 nL;              // lambda d ln I / d lambda  = 2 lambda e^{-2 lambda}/(1-e^{-2 lambda}) - 1 + Lambda D
    f2 nk;              // d ln I / d k
};

// g(x) = (x coth x - 1)/x^2 (d ln sinhc(x)/dx = x g(x)) from x^2, 1/x, and t = e^{-2x}/(x (1-e^{-2x}));
// series below x = 0.7, closed form 1/x - 1/x^2 + 2t above.
NASG_HD f2 g_fun2(f2 x2, f2 ix, f2 t)
{
    f2 p = fma2(x2, splat(2.1377799e-5f), splat(-2.1164021e-4f));
    p = fma2(x2, p, splat(2.1164021e-3f));
    p = fma2(x2, p, splat(-2.2222222e-2f));
    const f2 small = fma2(x2, p, splat(0.33333333f));
    const f2 big = fma2(ix, sub2(splat(1.0f), ix), add2(t, t));
    return sel2(lo(x2) < 0.49f, hi(x2) < 0.49f, small, big);
}

// lgI = log2(1/(2I)) for I of eq.(10) (EXACT) or of NASG; with GRAD also the log-derivative terms.
// Straight-line: the two analytic branches of Psi (k < Lambda: sinhc of a real argument; k >= Lambda:
// the continuation S(s) = sin(rho)/rho, reading R4) share every MUFU through argument selects:
//   real (s = Lambda^2-k^2 > 0.05):  Psi = Lambda/(1-e^{-2 Lambda}) e^{r-Lambda} (1-e^{-2r})/r,  r-Lambda = -k^2/(Lambda+r)
//   else:                            Psi = Lambda/(1-e^{-2 Lambda}) e^{-Lambda}   2 S(s)
// E1 = ex2 of (r-Lambda) or of (-Lambda); e^{-2 Lambda} = E1^2 (e^{-2r} or 1). The trigonometric side
// is skipped when no active lane of the warp holds a lobe with s <= 0.05 (always in cfg4).
// lg_root = log2(lambda sqrt(1+a)).
template <bool EXACT, bool GRAD>
NASG_HD void normaliser2(f2 lg_root, f2 Lam, f2 lam, f2 k, f2 &lgI, LobePairGrad &G)
{
    const f2 x = add2(lam, lam);
    const f2 em = ex2_2(scl2(x, -LOG2E));                                   // e^{-2 lambda}
    // 1 - e^{-2 lambda}, epsilon = 0 (R8): by subtraction, or by its series where that would cancel
    f2 ps = fma2(x, splat(-1.0f / 720.0f), splat(1.0f / 120.0f));
    ps = fma2(x, ps, splat(-1.0f / 24.0f));
    ps = fma2(x, ps, splat(1.0f / 6.0f));
    ps = fma2(x, ps, splat(-0.5f));
    ps = fma2(x, ps, splat(1.0f));
    const f2 one_m = sel2(lo(lam) > 0.125f, hi(lam) > 0.125f, sub2(splat(1.0f), em), mul2(x, ps));
    // 1/(2I) = lambda sqrt(1+a) / (2 pi (1-e^{-2 lambda}) (1+Psi))
    if (!EXACT) {
        lgI = sub2(lg_root, lg2_2(scl2(one_m, 2.0f * TWO_PI)));             // NASG: I = 2 pi (1-e^{-2 lambda})/(lambda sqrt(1+a))
        if (GRAD) {
            G.nA = splat(-0.5f);
            G.nL = fma2(mul2(x, em), rcp2(one_m), splat(-1.0f));            // lambda d ln(base)/d lambda
            G.nk = splat(0.f);
        }
        return;
    }
    const f2 s = mul2(sub2(Lam, k), add2(Lam, k));                          // Lambda^2 - k^2
    const bool re0 = lo(s) > 0.05f, re1 = hi(s) > 0.05f;
    const f2 sm = max2(abs2(s), 0.05f);
    const f2 ir = rsqrt2(sm), r = mul2(sm, ir);                             // r = sqrt(|s|) (clamped)
    const f2 Lr = add2(Lam, r);
    f2 irL, iL = splat(0.f);
    if (GRAD) { const f2 R2 = rcp2(mul2(Lr, Lam)); irL = mul2(R2, Lam); iL = mul2(R2, Lr); }   // 1/(Lambda+r), 1/Lambda from one rcp
    else irL = rcp2(Lr);
    const f2 del = mul2(mul2(k, k), irL);                                   // Lambda - r  (real side)
    const f2 E1 = ex2_2(scl2(sel2(re0, re1, del, Lam), -LOG2E));            // e^{r-Lambda} | e^{-Lambda}
    const f2 e2r = ex2_2(scl2(r, -2.0f * LOG2E));                           // e^{-2r}
    const f2 e2L = mul2(mul2(E1, E1), sel2(re0, re1, e2r, splat(1.0f)));    // e^{-2 Lambda}
    const f2 om2L = sub2(splat(1.0f), e2L), om2r = sub2(splat(1.0f), e2r);
    f2 i1L, i1r = splat(0.f);
    if (GRAD) { const f2 R3 = rcp2(mul2(om2L, om2r)); i1L = mul2(R3, om2r); i1r = mul2(R3, om2L); }
    else i1L = rcp2(om2L);
    f2 Fx = mul2(ir, om2r);                                                 // (1-e^{-2r})/r
    f2 S_trig = splat(0.f), sc = splat(0.f);
    bool ser0 = false, ser1 = false;
#ifdef __CUDA_ARCH__
    const bool any_cont = __any_sync(__activemask(), !(re0 && re1));        // (called under divergent control flow: active lanes only)
#else
    const bool any_cont = !(re0 && re1);
#endif
    if (any_cont) {
        sc = pack(fminf(fmaxf(lo(s), -0.05f), 0.05f), fminf(fmaxf(hi(s), -0.05f), 0.05f));
        const f2 S_ser = fma2(sc, fma2(sc, fma2(sc, splat(1.9841270e-4f), splat(8.3333333e-3f)), splat(0.16666667f)), splat(1.0f));
        S_trig = mul2(sin2(r), ir);                                         // sin(rho)/rho, rho = sqrt(-s) <= k: no range reduction needed
        ser0 = lo(s) > -0.05f; ser1 = hi(s) > -0.05f;
        const f2 S = sel2(ser0, ser1, S_ser, S_trig);
        Fx = sel2(re0, re1, Fx, add2(S, S));
    }
    const f2 LiE = mul2(mul2(Lam, i1L), E1);
    const f2 Psi = mul2(LiE, Fx);
    const f2 opP = add2(Psi, splat(1.0f));
    const f2 P = mul2(one_m, opP);
    lgI = sub2(lg_root, lg2_2(scl2(P, TWO_PI)));
    if (GRAD) {
        const f2 R = rcp2(P);
        const f2 i1m = mul2(R, opP), i1p = mul2(R, one_m);                  // 1/(1-e^{-2 lambda}), 1/(1+Psi) from one rcp
        const f2 dl = fma2(mul2(x, em), i1m, splat(-1.0f));                 // lambda d ln(base)/d lambda
        // ---- real side: Lambda dPsi/dLambda = Psi Lambda^2 (g(r) - g(Lambda)), dPsi/dk = -Psi k g(r)
        const f2 tr = mul2(mul2(ir, e2r), i1r), tL = mul2(mul2(iL, e2L), i1L);
        const f2 gr = g_fun2(sm, ir, tr);
        // g(r) - g(Lambda) without cancellation for r >= 4, plain difference below
        const f2 iriL = mul2(ir, iL);
        const f2 tail = sub2(tr, tL);
        const f2 dg_big = fma2(mul2(del, iriL), fma2(neg2(Lr), iriL, splat(1.0f)), add2(tail, tail));
        const f2 dg_small = sub2(gr, g_fun2(mul2(Lam, Lam), iL, tL));
        const f2 dg = sel2(lo(r) >= 4.0f, hi(r) >= 4.0f, dg_big, dg_small);
        f2 LD = mul2(mul2(Psi, mul2(Lam, Lam)), dg);
        f2 dk = neg2(mul2(mul2(Psi, k), gr));
        // ---- continuation side: S' = dS/ds,  Lambda dPsi/dLambda = Psi + 2 Lambda^3 S'/sinh - Psi Lambda coth,  dPsi/dk = -2 k Lambda S'/sinh
        if (any_cont) {
            const f2 Sp_ser = fma2(sc, fma2(sc, fma2(sc, splat(1.1022928e-5f), splat(5.9523810e-4f)), splat(1.6666667e-2f)), splat(0.16666667f));
            const f2 Sp_trig = mul2(sub2(cos2(r), S_trig), scl2(mul2(ir, ir), -0.5f));   // (cos rho - S)/(2s), 1/(2s) = -1/(2 rho^2)
            const f2 Sp = sel2(ser0, ser1, Sp_ser, Sp_trig);
            const f2 M = mul2(scl2(LiE, 4.0f), Sp);                         // 2 Lambda S'/sinh(Lambda),  1/sinh = 2 e^{-Lambda}/(1-e^{-2 Lambda})
            const f2 coth = mul2(add2(e2L, splat(1.0f)), i1L);
            const f2 LD2 = fma2(mul2(Lam, Lam), M, fma2(neg2(mul2(Psi, Lam)), coth, Psi));
            const f2 dk2 = neg2(mul2(k, M));
            LD = sel2(re0, re1, LD, LD2);
            dk = sel2(re0, re1, dk, dk2);
        }
        const f2 LamD = mul2(LD, i1p);
        G.nA = add2(LamD, splat(-0.5f));
        G.nL = add2(dl, LamD);
        G.nk = mul2(dk, i1p);
    }
}

// MODE: 0 = NASG normaliser (approximate), 1 = eq.(10) (exact), 2 = pure NASG: no carrier (k = phi = 0 assumed,
// shape.z/.w ignored), for which both normalisers coincide (Psi(k=0) = 1).
// (w,x,y,z): quaternion, (l1,l2,k0,phi0): shape of lobes l and l+1, each as a pair.
// qs (GRAD only) = qhat * 2/|q| of the pair, what the quaternion chain of the backward needs.
template <int MODE, bool GRAD>
NASG_HD void lobe_pair_setup(f2 w, f2 x, f2 y, f2 z, const f2 l1, const f2 l2, const f2 k0, const f2 phi0, LobePair &L, LobePairGrad &G,
                             f2 &qsw, f2 &qsx, f2 &qsy, f2 &qsz)
{
    const f2 qq = fma2(w, w, fma2(x, x, fma2(y, y, mul2(z, z))));
    f2 inv = rsqrt2(qq);
    inv = mul2(inv, fma2(scl2(qq, -0.5f), mul2(inv, inv), splat(1.5f)));   // one Newton step
    w = mul2(w, inv); x = mul2(x, inv); y = mul2(y, inv); z = mul2(z, inv);
    const f2 x2 = add2(x, x), y2 = add2(y, y), z2 = add2(z, z);
    const f2 one = splat(1.0f);
    L.Xx = sub2(one, fma2(y2, y, mul2(z2, z))); L.Xy = fma2(x2, y, mul2(z2, w)); L.Xz = fma2(x2, z, neg2(mul2(y2, w)));
    L.Yx = fma2(x2, y, neg2(mul2(z2, w))); L.Yy = sub2(one, fma2(x2, x, mul2(z2, z))); L.Yz = fma2(y2, z, mul2(x2, w));
    L.Zx = fma2(x2, z, mul2(y2, w)); L.Zy = fma2(y2, z, neg2(mul2(x2, w))); L.Zz = sub2(one, fma2(x2, x, mul2(y2, y)));
    if (GRAD) {
        const f2 i2 = add2(inv, inv);
        qsw = mul2(w, i2); qsx = mul2(x, i2); qsy = mul2(y, i2); qsz = mul2(z, i2);
    }
    // relative errors of Lambda, lambda only scale the exponent (benign), so ex2.approx is enough
    const f2 lam = ex2_2(scl2(l2, LOG2E));
    const f2 one_pa = ex2_2(scl2(sub2(l1, l2), LOG2E));
    const f2 Lam = mul2(lam, one_pa);
    L.a = max2(sub2(one_pa, one), 0.0f);
    L.lam2e = scl2(lam, 2.0f * LOG2E);
    L.k = MODE == 2 ? splat(0.f) : k0;
    L.phi = MODE == 2 ? splat(0.f) : phi0;
    normaliser2<MODE == 1, GRAD>(scl2(add2(l1, l2), 0.5f * LOG2E), Lam, lam, k0, L.lgI, G);   // lambda sqrt(1+a) = e^{(l1+l2)/2}
}

// ---------------------------------------------------------------------------------------------
// Paper-native parameter record (Table 8, Supplementary C; include/nasg.h: nasg_paper_*): the lobe pair is
// given by RAW values: frame angles (theta, phi, tau) with cos = tanh(raw), sin = +sqrt(1 - cos^2) = sech(raw);
// lambda = exp(raw), a = exp(raw), k = 20 (tanh(raw) + 1), w = tanh(raw); no phase. [x y z] = Rz(theta) Ry(phi) Rz(tau).
// tanh and sech come from h = e^{-|raw|} directly, cos = sign (1-h^2)/(1+h^2), sin = 2h/(1+h^2): the pair (cos, sin) is a
// unit vector to fp32 rounding even when sin is tiny (sqrt(1 - cos^2) would lose it), so the frame stays orthonormal.
// ---------------------------------------------------------------------------------------------
#if defined(__CUDA_ARCH__) && !defined(NASG_LP_SCALAR)
__device__ __forceinline__ f2 copysign2(f2 mag, f2 sgn) { return (mag & 0x7fffffff7fffffffull) | (sgn & 0x8000000080000000ull); }
#else
NASG_HD f2 copysign2(f2 mag, f2 sgn) { return pack(copysignf(lo(mag), lo(sgn)), copysignf(hi(mag), hi(sgn))); }
#endif
// tanh(x) from t = e^{-2|x|}: sign(x) (1-t)/(1+t)
NASG_HD f2 tanh2(f2 x)
{
    const f2 t = ex2_2(scl2(abs2(x), -2.0f * LOG2E));
    return copysign2(mul2(sub2(splat(1.0f), t), rcp2(add2(t, splat(1.0f)))), x);
}
struct PaperTrig { f2 st, cp, sp, cu, su; };      // sin theta | cos, sin phi | cos, sin tau  (what the backward chain needs)

template <int MODE, bool GRAD>
NASG_HD void lobe_pair_setup_paper(f2 th, f2 ph, f2 ta, f2 lr, f2 ar, f2 kr, LobePair &L, LobePairGrad &G, PaperTrig &tr)
{
    f2 c[3], s[3];
    const f2 raw[3] = {th, ph, ta};
#pragma unroll
    for (int i = 0; i < 3; ++i) {
        const f2 h = ex2_2(scl2(abs2(raw[i]), -LOG2E));                     // e^{-|x|}
        const f2 t = mul2(h, h);
        const f2 r = rcp2(add2(t, splat(1.0f)));
        c[i] = copysign2(mul2(sub2(splat(1.0f), t), r), raw[i]);           // tanh(x)
        s[i] = mul2(add2(h, h), r);                                         // sech(x) = sqrt(1 - tanh^2)
    }
    const f2 ct = c[0], st = s[0], cp = c[1], sp = s[1], cu = c[2], su = s[2];
    const f2 cpcu = mul2(cp, cu), cpsu = mul2(cp, su);
    L.Xx = fma2(ct, cpcu, neg2(mul2(st, su))); L.Xy = fma2(st, cpcu, mul2(ct, su)); L.Xz = neg2(mul2(sp, cu));
    L.Yx = neg2(fma2(ct, cpsu, mul2(st, cu))); L.Yy = fma2(ct, cu, neg2(mul2(st, cpsu))); L.Yz = mul2(sp, su);
    L.Zx = mul2(ct, sp); L.Zy = mul2(st, sp); L.Zz = cp;
    if (GRAD) { tr.st = st; tr.cp = cp; tr.sp = sp; tr.cu = cu; tr.su = su; }
    const f2 lam = ex2_2(scl2(lr, LOG2E));
    const f2 a = ex2_2(scl2(ar, LOG2E));
    const f2 one_pa = add2(a, splat(1.0f));
    L.a = a;
    L.lam2e = scl2(lam, 2.0f * LOG2E);
    f2 k = splat(0.f);
    if (MODE != 2) k = fma2(tanh2(kr), splat(20.0f), splat(20.0f));        // 20 (tanh + 1)
    L.k = k;
    L.phi = splat(0.f);
    // log2(lambda sqrt(1+a)) = raw_lambda log2(e) + log2(1+a)/2
    normaliser2<MODE == 1, GRAD>(fma2(lr, splat(LOG2E), scl2(lg2_2(one_pa), 0.5f)), mul2(lam, one_pa), lam, k, L.lgI, G);
}


// ---------------------------------------------------------------------------------------------
// Isotropic spherical functions of the paper's Table 6 (include/nasg.h: nasg_iso_*), normalised:
//   KIND 0 Spherical Gaussian  F = lambda/(2 pi (1-e^{-2 lambda})) exp{lambda (v-1)}        lambda = e^raw
//   KIND 1 Spherical Beta      F = (beta+1)/(2 pi) max(v,0)^beta                             beta = e^raw
//   KIND 2 Spherical Cauchy    F = 1/(4 pi) ((1-rho^2)/(1+rho^2-2 rho v))^2                  rho = 1/(1+e^-raw)   (R19)
// v = d.zhat, zhat = z/|z|. Lobe pairs on f32x2 like the NASGabor arithmetic. 1 - v is formed without cancellation as
// h = |d - zhat|^2 / 2 (both unit vectors): every function is sharpest at v = 1, where 1 - d.zhat would lose all digits.
// ---------------------------------------------------------------------------------------------
struct IsoPair {
    f2 zx, zy, zz, inv;     // unit axis and 1/|z|
    f2 p;                   // lambda | beta | rho
    f2 q0, q1, q2;          // per-kind constants (see iso_pair_setup)
    f2 lgc;                 // log2 of the normalisation constant (SG, SB)
};
template <int KIND>
NASG_HD void iso_pair_setup(f2 x, f2 y, f2 z, f2 raw, IsoPair &P)
{
    const f2 nn = fma2(x, x, fma2(y, y, mul2(z, z)));
    f2 inv = rsqrt2(nn);
    inv = mul2(inv, fma2(scl2(nn, -0.5f), mul2(inv, inv), splat(1.5f)));   // one Newton step
    P.zx = mul2(x, inv); P.zy = mul2(y, inv); P.zz = mul2(z, inv); P.inv = inv;
    const f2 one = splat(1.0f);
    if (KIND == 0) {
        const f2 lam = ex2_2(scl2(raw, LOG2E));
        const f2 x2 = add2(lam, lam);
        const f2 em = ex2_2(scl2(x2, -LOG2E));                              // e^{-2 lambda}
        f2 ps = fma2(x2, splat(-1.0f / 720.0f), splat(1.0f / 120.0f));
        ps = fma2(x2, ps, splat(-1.0f / 24.0f)); ps = fma2(x2, ps, splat(1.0f / 6.0f));
        ps = fma2(x2, ps, splat(-0.5f)); ps = fma2(x2, ps, one);
        const f2 one_m = sel2(lo(lam) > 0.125f, hi(lam) > 0.125f, sub2(one, em), mul2(x2, ps));   // 1 - e^{-2 lambda}
        const f2 i1m = rcp2(one_m);
        P.p = lam;
        P.q0 = scl2(lam, LOG2E);                                            // lambda log2(e)
        P.q1 = fma2(neg2(mul2(x2, em)), i1m, one);                          // 1 - 2 lambda e^{-2 lambda}/(1-e^{-2 lambda}) = lambda d ln c/d lambda
        P.q2 = splat(0.f);
        P.lgc = lg2_2(mul2(scl2(lam, INV_TWO_PI), i1m));
    } else if (KIND == 1) {
        const f2 beta = ex2_2(scl2(raw, LOG2E));
        const f2 bp1 = add2(beta, one);
        P.p = beta;
        P.q0 = mul2(beta, rcp2(bp1));                                       // beta/(beta+1)
        P.q1 = scl2(beta, LN2);
        P.q2 = splat(0.f);
        P.lgc = lg2_2(scl2(bp1, INV_TWO_PI));
    } else {
        const f2 t = ex2_2(scl2(raw, -LOG2E));                              // e^{-raw}
        const f2 rho = rcp2(add2(t, one));
        const f2 omr = mul2(t, rho);                                        // 1 - rho without cancellation
        const f2 opr = add2(rho, one);
        P.p = rho;
        P.q0 = omr;
        P.q1 = mul2(omr, opr);                                              // 1 - rho^2
        P.q2 = mul2(scl2(mul2(rho, rho), -4.0f), rcp2(opr));                // -4 rho^2/(1+rho) = rho (1-rho) d ln(1-rho^2)^2/d rho
        P.lgc = splat(0.f);
    }
}
// F at direction d; with GRAD also Fv = dF/dv and Fr = dF/draw.
template <int KIND, bool GRAD>
NASG_HD f2 iso_pair_eval(const IsoPair &P, float dx, float dy, float dz, f2 &Fv, f2 &Fr)
{
    const f2 ex = sub2(splat(dx), P.zx), ey = sub2(splat(dy), P.zy), ez = sub2(splat(dz), P.zz);
    const f2 h = scl2(fma2(ex, ex, fma2(ey, ey, mul2(ez, ez))), 0.5f);      // 1 - v
    if (KIND == 0) {
        const f2 F = ex2_2(fma2(neg2(P.q0), h, P.lgc));
        if (GRAD) { Fv = mul2(P.p, F); Fr = mul2(F, fma2(neg2(P.p), h, P.q1)); }
        return F;
    } else if (KIND == 1) {
        const f2 v = sub2(splat(1.0f), h);
        const bool on0 = lo(v) > 0.0f, on1 = hi(v) > 0.0f;
        const f2 vc = max2(v, TINY);
        f2 pl = fma2(h, splat(-0.39963189f), splat(-0.47933504f));          // log2(1-h)/h on [0,1/16] (as in lobe_pair_eval)
        pl = fma2(h, pl, splat(-0.72136736f)); pl = fma2(h, pl, splat(-1.4426950f));
        const f2 L2 = sel2(lo(h) < 0.0625f, hi(h) < 0.0625f, mul2(h, pl), lg2_2(vc));
        f2 F = ex2_2(fma2(P.p, L2, P.lgc));
        F = pack(on0 ? lo(F) : 0.0f, on1 ? hi(F) : 0.0f);                   // far hemisphere: 0
        if (GRAD) { Fv = mul2(mul2(P.p, F), rcp2(vc)); Fr = mul2(F, fma2(P.q1, L2, P.q0)); }
        return F;
    } else {
        const f2 D = fma2(add2(P.p, P.p), h, mul2(P.q0, P.q0));             // (1-rho)^2 + 2 rho (1-v) = 1 + rho^2 - 2 rho v
        const f2 iD = rcp2(D);
        const f2 ratio = mul2(P.q1, iD);
        const f2 F = scl2(mul2(ratio, ratio), 0.5f * INV_TWO_PI);
        if (GRAD) {
            const f2 r4 = scl2(P.p, 4.0f);
            Fv = mul2(F, mul2(r4, iD));
            Fr = mul2(F, fma2(neg2(mul2(mul2(r4, P.q0), sub2(h, P.q0))), iD, P.q2));   // rho (1-rho) dF/drho / F
        }
        return F;
    }
}

// ---------------------------------------------------------------------------------------------
// Anisotropic Spherical Gaussian of the paper's Table 6 ([XSD*13]; include/nasg.h: nasg_asg_*):
//   G = max(d.z, 0) exp{-mu (d.x)^2 - lambda (d.y)^2},  [x y z] = R(q/|q|),  mu = e^raw0, lambda = e^raw1, no normaliser.
// Nothing cancels here (the exponent is a sum of squares of plain dot products), so the arithmetic is the direct one.
// The frame gradient is accumulated as a rotation vector in the lobe frame like the NASGabor backward's:
// with p = (u, t, v) the direction in the lobe frame and g = dL/dp, g_theta = g x p, then g_q = qs (x) (0, g_theta).
// ---------------------------------------------------------------------------------------------
struct AsgPair {
    f2 Xx, Xy, Xz, Yx, Yy, Yz, Zx, Zy, Zz;   // columns of R(q/|q|)
    f2 mu, lam;                               // bandwidths
};
struct AsgEval { f2 u, t, v, uu, tt, S; };    // what the backward needs from the recomputed forward
struct AsgAcc { f2 gw0, gw1, gw2, Sm, Sl, th0, th1, th2; };
// qs (GRAD only) = qhat * 2/|q|
template <bool GRAD>
NASG_HD void asg_pair_setup(f2 w, f2 x, f2 y, f2 z, f2 raw_mu, f2 raw_lam, AsgPair &P, f2 &qsw, f2 &qsx, f2 &qsy, f2 &qsz)
{
    const f2 qq = fma2(w, w, fma2(x, x, fma2(y, y, mul2(z, z))));
    f2 inv = rsqrt2(qq);
    inv = mul2(inv, fma2(scl2(qq, -0.5f), mul2(inv, inv), splat(1.5f)));   // one Newton step
    w = mul2(w, inv); x = mul2(x, inv); y = mul2(y, inv); z = mul2(z, inv);
    const f2 x2 = add2(x, x), y2 = add2(y, y), z2 = add2(z, z);
    const f2 one = splat(1.0f);
    P.Xx = sub2(one, fma2(y2, y, mul2(z2, z))); P.Xy = fma2(x2, y, mul2(z2, w)); P.Xz = fma2(x2, z, neg2(mul2(y2, w)));
    P.Yx = fma2(x2, y, neg2(mul2(z2, w))); P.Yy = sub2(one, fma2(x2, x, mul2(z2, z))); P.Yz = fma2(y2, z, mul2(x2, w));
    P.Zx = fma2(x2, z, mul2(y2, w)); P.Zy = fma2(y2, z, neg2(mul2(x2, w))); P.Zz = sub2(one, fma2(x2, x, mul2(y2, y)));
    if (GRAD) {
        const f2 i2 = add2(inv, inv);
        qsw = mul2(w, i2); qsx = mul2(x, i2); qsy = mul2(y, i2); qsz = mul2(z, i2);
    }
    P.mu = ex2_2(scl2(raw_mu, LOG2E));
    P.lam = ex2_2(scl2(raw_lam, LOG2E));
}
template <bool FULL>
NASG_HD f2 asg_pair_eval(const AsgPair &P, float dx, float dy, float dz, AsgEval &T)
{
    const f2 ddx = splat(dx), ddy = splat(dy), ddz = splat(dz);
    const f2 u = fma2(P.Xx, ddx, fma2(P.Xy, ddy, mul2(P.Xz, ddz)));
    const f2 t = fma2(P.Yx, ddx, fma2(P.Yy, ddy, mul2(P.Yz, ddz)));
    const f2 v = fma2(P.Zx, ddx, fma2(P.Zy, ddy, mul2(P.Zz, ddz)));
    const f2 uu = mul2(u, u), tt = mul2(t, t);
    const f2 S = ex2_2(scl2(fma2(P.mu, uu, mul2(P.lam, tt)), -LOG2E));
    if (FULL) { T.u = u; T.t = t; T.v = v; T.uu = uu; T.tt = tt; T.S = S; }
    return mul2(max2(v, 0.0f), S);
}
// Backward of one (lobe pair, camera); FIRST initialises the accumulators. Returns the pair's dL/dd in gdx, gdy, gdz.
template <bool FIRST>
NASG_HD void asg_pair_bwd(const AsgPair &P, const AsgEval &T, f2 G, float gc0, float gc1, float gc2, f2 w0, f2 w1, f2 w2,
                          AsgAcc &A, f2 &gdx, f2 &gdy, f2 &gdz)
{
    const f2 c0 = splat(gc0), c1 = splat(gc1), c2 = splat(gc2);
    const f2 gG = fma2(w0, c0, fma2(w1, c1, mul2(w2, c2)));                 // dL/dG, eq.(6)
    const f2 gGG = mul2(gG, G);
    const f2 m2 = scl2(gGG, -2.0f);
    const f2 gu = mul2(mul2(m2, P.mu), T.u);                                // gG dG/du = -2 mu u G
    const f2 gt = mul2(mul2(m2, P.lam), T.t);                               // gG dG/dt = -2 lambda t G
    const f2 gS = mul2(gG, T.S);
    const f2 gv = pack(lo(T.v) > 0.0f ? lo(gS) : 0.0f, hi(T.v) > 0.0f ? hi(gS) : 0.0f);   // gG dG/dv = S on the lobe side, 0 beyond the kink
    if (FIRST) {
        A.gw0 = mul2(G, c0); A.gw1 = mul2(G, c1); A.gw2 = mul2(G, c2);
        A.Sm = mul2(gGG, T.uu); A.Sl = mul2(gGG, T.tt);
        A.th0 = fma2(gt, T.v, mul2(neg2(gv), T.t));
        A.th1 = fma2(gv, T.u, mul2(neg2(gu), T.v));
        A.th2 = fma2(gu, T.t, mul2(neg2(gt), T.u));
    } else {
        A.gw0 = fma2(G, c0, A.gw0); A.gw1 = fma2(G, c1, A.gw1); A.gw2 = fma2(G, c2, A.gw2);
        A.Sm = fma2(gGG, T.uu, A.Sm); A.Sl = fma2(gGG, T.tt, A.Sl);
        A.th0 = fma2(gt, T.v, fma2(neg2(gv), T.t, A.th0));                  // g_theta = g x p, p = (u, t, v)
        A.th1 = fma2(gv, T.u, fma2(neg2(gu), T.v, A.th1));
        A.th2 = fma2(gu, T.t, fma2(neg2(gt), T.u, A.th2));
    }
    gdx = fma2(gu, P.Xx, fma2(gt, P.Yx, fma2(gv, P.Zx, gdx)));
    gdy = fma2(gu, P.Xy, fma2(gt, P.Yy, fma2(gv, P.Zy, gdy)));
    gdz = fma2(gu, P.Xz, fma2(gt, P.Yz, fma2(gv, P.Zz, gdz)));
}
// gradients of the raw bandwidths and of the (unnormalised) quaternion: (w, v) (x) (0, t) = ( -v.t ,  w t + v cross t )
NASG_HD void asg_pair_finish(const AsgPair &P, const AsgAcc &A, f2 qw, f2 qx, f2 qy, f2 qz, f2 &gmu, f2 &glam, f2 &gqw, f2 &gqx, f2 &gqy, f2 &gqz)
{
    gmu = mul2(neg2(P.mu), A.Sm);                                           // d/draw = mu d/dmu
    glam = mul2(neg2(P.lam), A.Sl);
    gqw = neg2(fma2(qx, A.th0, fma2(qy, A.th1, mul2(qz, A.th2))));
    gqx = fma2(qw, A.th0, fma2(qy, A.th2, mul2(neg2(qz), A.th1)));
    gqy = fma2(qw, A.th1, fma2(qz, A.th0, mul2(neg2(qx), A.th2)));
    gqz = fma2(qw, A.th2, fma2(qx, A.th1, mul2(neg2(qy), A.th0)));
}

// ---------------------------------------------------------------------------------------------
// evaluation of a lobe pair at ONE direction d (scalar-broadcast operands)
// ---------------------------------------------------------------------------------------------
struct EvalPair {       // what the backward needs from the recomputed forward
    f2 u, om, v, uu, inv_s2, tau, L2, kp, em1, inv_1pv, Gh, sn;
};

// G = H p E / I of both lobes at d (eq.(9) over eq.(10)). MUFU per half: rcp, lg2, ex2, ex2, cos (+ sin with FULL).
// The carrier angle k u + phi needs no range reduction: |k u + phi| <= k + 2 pi stays below ~4 turns for the
// supported frequencies (MUFU.SIN/COS take the angle in turns and reduce it themselves; the product by 1/2pi the
// PTX approximations insert costs 2^-24 relative of <= 4 turns: ~1.5e-6 rad).
template <bool FULL, bool CARRIER>
NASG_HD f2 lobe_pair_eval(const LobePair &L, float dx, float dy, float dz, EvalPair &T)
{
    const f2 ddx = splat(dx), ddy = splat(dy), ddz = splat(dz);
    const f2 u = fma2(L.Xx, ddx, fma2(L.Xy, ddy, mul2(L.Xz, ddz)));
    const f2 om = fma2(L.Yx, ddx, fma2(L.Yy, ddy, mul2(L.Yz, ddz)));
    const f2 v = fma2(L.Zx, ddx, fma2(L.Zy, ddy, mul2(L.Zz, ddz)));
    const f2 uu = mul2(u, u);
    const f2 s2 = max2(fma2(om, om, uu), TINY);                      // 1 - v^2 without cancellation
    const f2 w2 = fma2(abs2(v), splat(2.0f), splat(2.0f));           // 2 (1 + |v|)
    const f2 rw = rcp2(mul2(s2, w2));                                // one reciprocal serves 1/s^2 and 1/(1+|v|)
    const f2 inv_s2 = mul2(rw, w2);
    const f2 s2rw = mul2(s2, rw);                                    // 1/(2 (1 + |v|))
    const f2 q = mul2(s2, s2rw);                                     // (1 - |v|)/2
    const f2 tau = mul2(mul2(L.a, uu), inv_s2);                      // a (d.x)^2 / (1 - (d.z)^2)
    const bool up0 = lo(v) > 0.0f, up1 = hi(v) > 0.0f;
    // log2 kappa, kappa = 1-q on the lobe side (v > 0) else q: minimax cubic of log2(1-q)/q on [0,1/16] (2.7e-8 relative)
    // near the axis, lg2.approx elsewhere (absolute error 2^-22 on |log2| >= 0.093: relative to the exponent, benign)
    f2 p = fma2(q, splat(-0.39963189f), splat(-0.47933504f));
    p = fma2(q, p, splat(-0.72136736f));
    p = fma2(q, p, splat(-1.4426950f));
    const f2 lsmall = mul2(q, p);
    const f2 omq = sub2(splat(1.0f), q);
    const f2 big = lg2_2(sel2(up0, up1, omq, q));
    const f2 L2 = sel2(up0 && lo(q) < 0.0625f, up1 && hi(q) < 0.0625f, lsmall, big);
    const f2 x1 = fma2(tau, L2, L2);                                 // (1+tau) log2 kappa
    // kappa^(1+tau) - 1 = 2^x1 - 1: minimax cubic of (2^x-1)/x on [-1/8,0] (4.5e-9 relative), ex2 - 1 below
    f2 pe = fma2(x1, splat(9.2798658e-3f), splat(5.5477057e-2f));
    pe = fma2(x1, pe, splat(0.24022582f));
    pe = fma2(x1, pe, splat(0.69314718f));
    const f2 esmall = mul2(x1, pe);
    const f2 ebig = add2(ex2_2(x1), splat(-1.0f));
    const f2 em1 = sel2(lo(x1) > -0.125f, hi(x1) > -0.125f, esmall, ebig);
    const f2 arg = fma2(L.lam2e, em1, fma2(tau, L2, L.lgI));         // log2( p E / (2 I) )
    f2 Gh = ex2_2(arg);
    Gh = pack((lo(s2) <= TINY && !up0) ? 0.0f : lo(Gh), (hi(s2) <= TINY && !up1) ? 0.0f : hi(Gh));   // d = -z: G = 0 (eq.(9), third case)
    f2 ang = splat(0.f), G;
    if (CARRIER) {
#ifdef NASG_LP_REDUCE
        {   // exact reduction to [-1/2, 1/2] turns (1.5 * 2^23 magic constant), then radians
            const f2 t = fma2(scl2(L.k, INV_TWO_PI), u, scl2(L.phi, INV_TWO_PI));
            const f2 n = add2(add2(t, splat(12582912.0f)), splat(-12582912.0f));
            ang = scl2(sub2(t, n), TWO_PI);
        }
#else
        ang = fma2(L.k, u, L.phi);                                   // k d.x + phi
#endif
        G = fma2(Gh, cos2(ang), Gh);                                 // (1 + cos)/2 * p E / I
    } else {
        G = add2(Gh, Gh);                                            // no carrier: H = 1
    }
    if (FULL) {
        T.u = u; T.om = om; T.v = v; T.uu = uu; T.inv_s2 = inv_s2; T.tau = tau; T.L2 = L2;
        T.kp = add2(em1, splat(1.0f)); T.em1 = em1;
        const f2 hi = add2(s2rw, s2rw), lo = mul2(scl2(w2, 0.5f), inv_s2);   // 1/(1+v) on the lobe side / far side
        T.inv_1pv = sel2(up0, up1, hi, lo);
        T.Gh = Gh; T.sn = CARRIER ? sin2(ang) : splat(0.f);
    }
    return G;
}

// Per-lobe accumulators of the backward over the cameras of one Gaussian (all packed over the lobe pair).
struct AccPair {
    f2 gw0, gw1, gw2;        // dL/dw (eq.(6))
    f2 S0, S1, S2, Sk, Sp;   // sums that become g_shape
    f2 th0, th1, th2;        // rotation-vector gradient in the lobe frame
};
NASG_HD void acc_zero(AccPair &A)
{
    const f2 z = splat(0.f);
    A.gw0 = A.gw1 = A.gw2 = A.S0 = A.S1 = A.S2 = A.Sk = A.Sp = A.th0 = A.th1 = A.th2 = z;
}

// Backward of one (lobe pair, camera): adds to the pair's accumulators and returns the pair's contribution to
// dL/dd of this camera (gdx, gdy, gdz: halves summed by the caller when it wants to).
// gc = dL/dcolour of this camera (0 for a culled camera), w = amplitudes of the pair.
// FIRST: this is the first camera of the lobe pair: the accumulators are initialised instead of added to (no zeroing pass).
template <bool CARRIER, bool FIRST = false>
NASG_HD void lobe_pair_bwd(const LobePair &L, const EvalPair &T, f2 G, float gc0, float gc1, float gc2, f2 w0, f2 w1, f2 w2,
                           AccPair &A, f2 &gdx, f2 &gdy, f2 &gdz)
{
    const f2 c0 = splat(gc0), c1 = splat(gc1), c2 = splat(gc2);
    const f2 gG = fma2(w0, c0, fma2(w1, c1, mul2(w2, c2)));                 // dL/dG, eq.(6)
    if (FIRST) {
        A.gw0 = mul2(G, c0); A.gw1 = mul2(G, c1); A.gw2 = mul2(G, c2);
        const f2 gGG = mul2(gG, G);
        const f2 P = mul2(scl2(L.lam2e, LN2), T.kp);
        const f2 Q = add2(P, splat(1.0f));
        const f2 A_tau2 = mul2(scl2(T.L2, 2.0f * LN2), Q);
        const f2 A_kap = mul2(fma2(T.tau, Q, P), T.inv_1pv);
        const f2 B1 = mul2(mul2(gGG, A_tau2), T.inv_s2);
        f2 gu = mul2(mul2(B1, L.a), T.u);
        if (CARRIER) {
            const f2 hs = mul2(mul2(gG, T.Gh), T.sn);
            gu = fma2(neg2(hs), L.k, gu);
            A.Sk = mul2(hs, T.u);
            A.Sp = hs;
        } else {
            A.Sk = splat(0.f); A.Sp = splat(0.f);
        }
        const f2 gv = fma2(mul2(B1, T.tau), T.v, mul2(gGG, A_kap));
        A.S0 = gGG;
        A.S1 = mul2(gGG, T.em1);
        A.S2 = mul2(B1, T.uu);
        A.th0 = mul2(gv, T.om);
        A.th1 = fma2(gv, T.u, mul2(neg2(gu), T.v));
        A.th2 = mul2(gu, T.om);
        gdx = fma2(gu, L.Xx, fma2(gv, L.Zx, gdx));
        gdy = fma2(gu, L.Xy, fma2(gv, L.Zy, gdy));
        gdz = fma2(gu, L.Xz, fma2(gv, L.Zz, gdz));
        return;
    }
    A.gw0 = fma2(G, c0, A.gw0); A.gw1 = fma2(G, c1, A.gw1); A.gw2 = fma2(G, c2, A.gw2);
    const f2 gGG = mul2(gG, G);
    const f2 P = mul2(scl2(L.lam2e, LN2), T.kp);                            // 2 lambda kappa^(1+tau)
    const f2 Q = add2(P, splat(1.0f));
    const f2 A_tau2 = mul2(scl2(T.L2, 2.0f * LN2), Q);                      // 2 d ln(pE)/d tau = 2 ln kappa (1 + 2 lambda kappa')
    const f2 A_kap = mul2(fma2(T.tau, Q, P), T.inv_1pv);                    // (d ln(pE)/d kappa)/2 = (tau + 2 lambda (1+tau) kappa')/(2 kappa)
    const f2 B1 = mul2(mul2(gGG, A_tau2), T.inv_s2);
    f2 gu = mul2(mul2(B1, L.a), T.u);                                       // gG dG/du (eqs.57-60)
    if (CARRIER) {
        const f2 hs = mul2(mul2(gG, T.Gh), T.sn);                           // carrier, eqs.(59),(65)
        gu = fma2(neg2(hs), L.k, gu);
        A.Sk = fma2(hs, T.u, A.Sk);
        A.Sp = add2(A.Sp, hs);
    }
    const f2 gv = fma2(mul2(B1, T.tau), T.v, mul2(gGG, A_kap));             // gG dG/dv (eqs.61-64)
    A.S0 = add2(A.S0, gGG);
    A.S1 = fma2(gGG, T.em1, A.S1);
    A.S2 = fma2(B1, T.uu, A.S2);
    A.th0 = fma2(gv, T.om, A.th0);                                          // (sign applied at the end)
    A.th1 = fma2(gv, T.u, fma2(neg2(gu), T.v, A.th1));
    A.th2 = fma2(gu, T.om, A.th2);
    gdx = fma2(gu, L.Xx, fma2(gv, L.Zx, gdx));
    gdy = fma2(gu, L.Xy, fma2(gv, L.Zy, gdy));
    gdz = fma2(gu, L.Xz, fma2(gv, L.Zz, gdz));
}

// g_shape and g_quat of ONE lobe of the pair from the accumulators (B4): (lambda, a) = (e^{l2}, e^{l1-l2} - 1);
// g_q = qs (x) (0, g_theta) with qs = qhat 2/|q| (Hamilton product, zero scalar part on the right). Scalar on purpose:
// the results must sit in four consecutive registers for the 128-bit stores, which packed results (lobe l, lobe l+1)
// never do; 21 scalar operations per lobe cost fewer FP32-pipe cycles than 21 packed ones plus 16 moves per pair.
NASG_HD void lobe_finish(float a, float lam2e, float nA, float nL, float nk, float S0, float S1, float S2, float Sk, float Sp,
                         float th0, float th1, float th2, float qw, float qx, float qy, float qz, float4 &gs, float4 &gq)
{
    gs.x = fmaf(0.5f * S2, a + 1.0f, -S0 * nA);
    gs.y = fmaf(lam2e * LN2, S1, -S0 * nL) - gs.x;
    gs.z = -fmaf(S0, nk, Sk);
    gs.w = -Sp;
    const float t0 = -th0, t1 = th1, t2 = th2;                              // g_theta in the lobe frame
    // (w, v) (x) (0, t) = ( -v.t ,  w t + v cross t )
    gq.x = -fmaf(qx, t0, fmaf(qy, t1, qz * t2));
    gq.y = fmaf(qw, t0, fmaf(qy, t2, -qz * t1));
    gq.z = fmaf(qw, t1, fmaf(qz, t0, -qx * t2));
    gq.w = fmaf(qw, t2, fmaf(qx, t1, -qy * t0));
}
NASG_HD void lobe_pair_finish(const LobePair &L, const LobePairGrad &Gd, const AccPair &A, f2 qsw, f2 qsx, f2 qsy, f2 qsz,
                              float4 &gs0, float4 &gs1, float4 &gq0, float4 &gq1)
{
    lobe_finish(lo(L.a), lo(L.lam2e), lo(Gd.nA), lo(Gd.nL), lo(Gd.nk), lo(A.S0), lo(A.S1), lo(A.S2), lo(A.Sk), lo(A.Sp),
                lo(A.th0), lo(A.th1), lo(A.th2), lo(qsw), lo(qsx), lo(qsy), lo(qsz), gs0, gq0);
    lobe_finish(hi(L.a), hi(L.lam2e), hi(Gd.nA), hi(Gd.nL), hi(Gd.nk), hi(A.S0), hi(A.S1), hi(A.S2), hi(A.Sk), hi(A.Sp),
                hi(A.th0), hi(A.th1), hi(A.th2), hi(qsw), hi(qsx), hi(qsy), hi(qsz), gs1, gq1);
}

// The same for both lobes at once, results as pairs (lobe l, lobe l+1) per component: for the tile-record layout, whose
// gradient records hold pairs (nasg_rec_kernels.cu), the packed form needs no re-assembly: 25 packed operations per pair.
NASG_HD void lobe_pair_finish2(const LobePair &L, const LobePairGrad &Gd, const AccPair &A, f2 qw, f2 qx, f2 qy, f2 qz,
                               f2 &gl1, f2 &gl2, f2 &gk, f2 &gphi, f2 &gqw, f2 &gqx, f2 &gqy, f2 &gqz)
{
    gl1 = fma2(scl2(A.S2, 0.5f), add2(L.a, splat(1.0f)), mul2(neg2(A.S0), Gd.nA));
    gl2 = sub2(fma2(scl2(L.lam2e, LN2), A.S1, mul2(neg2(A.S0), Gd.nL)), gl1);
    gk = fma2(neg2(A.S0), Gd.nk, neg2(A.Sk));
    gphi = scl2(A.Sp, -1.0f);
    // g_theta = (-th0, th1, th2);  (w, v) (x) (0, t) = ( -v.t ,  w t + v cross t )
    gqw = fma2(qx, A.th0, neg2(fma2(qy, A.th1, mul2(qz, A.th2))));
    gqx = fma2(neg2(qw), A.th0, fma2(qy, A.th2, mul2(neg2(qz), A.th1)));
    gqy = fma2(qw, A.th1, fma2(neg2(qz), A.th0, mul2(neg2(qx), A.th2)));
    gqz = fma2(qw, A.th2, fma2(qx, A.th1, mul2(qy, A.th0)));
}

// gradients with respect to the 9 raw values of both lobes from the accumulators (eqs.(37)-(44) in rotation-vector
// form: for R = Rz(theta) Ry(phi) Rz(tau) the body-frame rotation vectors of the three angles are e3 (tau),
// (sin tau, cos tau, 0) (phi) and (-sin phi cos tau, sin phi sin tau, cos phi) (theta); d angle / d raw = -sin(angle),
// so the 1/sin of eq.(36) cancels against tanh' = sin^2), w = activated amplitudes.
template <int MODE>
NASG_HD void lobe_pair_finish_paper(const LobePair &L, const LobePairGrad &Gd, const AccPair &A, const PaperTrig &tr, f2 w0, f2 w1, f2 w2,
                                    f2 &gth, f2 &gph, f2 &gta, f2 &glr, f2 &gar, f2 &gkr, f2 &gw0, f2 &gw1, f2 &gw2)
{
    const f2 one_pa = add2(L.a, splat(1.0f));
    const f2 gl1 = fma2(scl2(A.S2, 0.5f), one_pa, mul2(neg2(A.S0), Gd.nA));            // (1+a) dL/da
    glr = fma2(scl2(L.lam2e, LN2), A.S1, mul2(neg2(A.S0), Gd.nL));                       // lambda dL/dlambda
    gar = mul2(gl1, mul2(L.a, rcp2(one_pa)));                                            // a dL/da
    if (MODE != 2) {
        const f2 gk = fma2(neg2(A.S0), Gd.nk, neg2(A.Sk));
        gkr = mul2(gk, mul2(L.k, fma2(L.k, splat(-0.05f), splat(2.0f))));                // dk/draw = 20 (1 - tanh^2) = k (2 - k/20)
    } else {
        gkr = splat(0.f);
    }
    gw0 = mul2(A.gw0, fma2(neg2(w0), w0, splat(1.0f)));
    gw1 = mul2(A.gw1, fma2(neg2(w1), w1, splat(1.0f)));
    gw2 = mul2(A.gw2, fma2(neg2(w2), w2, splat(1.0f)));
    // g_theta (rotation vector in the lobe frame) = (-th0, th1, th2)
    const f2 g_tau = A.th2;
    const f2 g_phi = fma2(tr.cu, A.th1, mul2(neg2(tr.su), A.th0));
    const f2 g_the = fma2(tr.sp, fma2(tr.su, A.th1, mul2(tr.cu, A.th0)), mul2(tr.cp, A.th2));
    gta = mul2(neg2(tr.su), g_tau);
    gph = mul2(neg2(tr.sp), g_phi);
    gth = mul2(neg2(tr.st), g_the);
}

} // namespace lp
} // namespace nasg
