// nasg_math.cuh — fp32 per-lobe arithmetic of the NASGabor path (device; also compilable for the host
// so that the conditioning can be studied without a GPU).
//
// What is computed is eq.(9)/(10) of arxiv/paper_2606_09794 and its gradient
// (PAPER.md:754-861 + DESIGN.md §4); HOW it is computed is the well-conditioned fp32 form of
// DESIGN.md §5, because the literal transcription loses the 1e-5 parity bar exactly where sharp
// lobes are bright:
//   * s^2 = 1-(d.z)^2 is formed as (d.x)^2 + (d.y)^2, never by subtraction;
//   * 1-kappa = s^2/(2(1+v)) for v > 0, ln kappa = log1p(-(1-kappa)) by polynomial when it is small;
//   * 2 lambda (kappa^(1+tau) - 1) uses an expm1 polynomial when the argument is small;
//   * MUFU approximations (ex2, lg2, sin, cos, rcp, rsqrt) only where their error is relative to the
//     exponent or otherwise bounded well inside the tolerance (DESIGN.md §5 table).
#pragma once

#include <cuda_runtime.h>
#include <math.h>

#define NASG_HD __host__ __device__ __forceinline__

namespace nasg {

// ---------------------------------------------------------------------------------------------
// MUFU wrappers (one SFU instruction each on the device)
// ---------------------------------------------------------------------------------------------
NASG_HD float f_rcp(float x)
{
#ifdef __CUDA_ARCH__
    float r; asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r;
#else
    return 1.0f / x;
#endif
}
NASG_HD float f_rsqrt(float x)
{
#ifdef __CUDA_ARCH__
    float r; asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r;
#else
    return 1.0f / sqrtf(x);
#endif
}
NASG_HD float f_sqrt(float x)
{
#ifdef __CUDA_ARCH__
    float r; asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r;
#else
    return sqrtf(x);
#endif
}
NASG_HD float f_ex2(float x)
{
#ifdef __CUDA_ARCH__
    float r; asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r;
#else
    return exp2f(x);
#endif
}
NASG_HD float f_lg2(float x)
{
#ifdef __CUDA_ARCH__
    float r; asm("lg2.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r;
#else
    return log2f(x);
#endif
}
NASG_HD float f_exp(float x) { return f_ex2(x * 1.4426950408889634f); }

// sin and cos of theta after a two-constant Cody-Waite reduction to [-pi, pi] (|theta| <~ 1e3)
NASG_HD void f_sincos(float theta, float &sn, float &cs)
{
    float n = rintf(theta * 0.15915494309189535f);
    float r = fmaf(n, -6.2831854820251465f, theta);     // 2pi hi (fp32)
    r = fmaf(n, 1.7484555e-7f, r);                      // 2pi lo: 2pi = hi - 1.7484555e-7
#ifdef __CUDA_ARCH__
    asm("sin.approx.ftz.f32 %0, %1;" : "=f"(sn) : "f"(r));
    asm("cos.approx.ftz.f32 %0, %1;" : "=f"(cs) : "f"(r));
#else
    sn = sinf(r); cs = cosf(r);
#endif
}
NASG_HD float f_cos(float theta)
{
    float n = rintf(theta * 0.15915494309189535f);
    float r = fmaf(n, -6.2831854820251465f, theta);
    r = fmaf(n, 1.7484555e-7f, r);
#ifdef __CUDA_ARCH__
    float cs; asm("cos.approx.ftz.f32 %0, %1;" : "=f"(cs) : "f"(r)); return cs;
#else
    return cosf(r);
#endif
}

// ---------------------------------------------------------------------------------------------
// accurate small-argument helpers
// ---------------------------------------------------------------------------------------------
// ln(kappa) where kappa = 1-q if `upper` (v > 0: q = 1-kappa is small near the lobe axis) else kappa = q
// (v <= 0: kappa itself is small near the antipode). Polynomial -q(1 + q/2 + ...) for q < 1/8 on the
// upper side (relative error < 1e-7), lg2 otherwise (its absolute error 2^-22 is then < 2e-6 relative).
NASG_HD float log_kappa(float q, bool upper)
{
    float p = fmaf(q, 0.11111111f, 0.125f);
    p = fmaf(q, p, 0.14285714f);
    p = fmaf(q, p, 0.16666667f);
    p = fmaf(q, p, 0.2f);
    p = fmaf(q, p, 0.25f);
    p = fmaf(q, p, 0.33333333f);
    p = fmaf(q, p, 0.5f);
    p = fmaf(q, p, 1.0f);
    float small = -q * p;
    float big = 0.6931471805599453f * f_lg2(upper ? 1.0f - q : q);
    return (upper && q < 0.125f) ? small : big;
}
// e^x - 1 for x <= 0. Polynomial for |x| < 1/8, ex2 otherwise.
NASG_HD float expm1_neg(float x)
{
    float p = fmaf(x, 1.9841270e-4f, 1.3888889e-3f);
    p = fmaf(x, p, 8.3333333e-3f);
    p = fmaf(x, p, 4.1666667e-2f);
    p = fmaf(x, p, 0.16666667f);
    p = fmaf(x, p, 0.5f);
    p = fmaf(x, p, 1.0f);
    float small = x * p;
    float big = f_exp(x) - 1.0f;
    return x > -0.125f ? small : big;
}
// g(x) = (x coth x - 1)/x^2, x > 0   (d ln sinhc(x)/dx = x g(x))
NASG_HD float g_fun(float x)
{
    if (x < 0.7f) {
        float x2 = x * x;
        float p = fmaf(x2, 2.1377799e-5f, -2.1164021e-4f);
        p = fmaf(x2, p, 2.1164021e-3f);
        p = fmaf(x2, p, -2.2222222e-2f);
        return fmaf(x2, p, 0.33333333f);
    }
    float ix = f_rcp(x);
    float e = f_exp(-2.0f * x);
    return fmaf(ix, 1.0f - ix, 2.0f * ix * e * f_rcp(1.0f - e));
}

// ---------------------------------------------------------------------------------------------
// per-lobe, camera-independent set-up
// ---------------------------------------------------------------------------------------------
struct Lobe {
    float Xx, Xy, Xz, Yx, Yy, Yz, Zx, Zy, Zz; // columns of R(q/|q|)
    float lam2;                                // 2 lambda
    float a;                                   // Lambda/lambda - 1
    float k, phi;
    float invI;                                // 1 / normalising integral
};
struct LobeBwd {        // extra camera-independent terms of the backward pass
    float qw, qx, qy, qz, inv_qn;  // unit quaternion and 1/|q|
    float one_pa;                  // 1 + a = Lambda/lambda
    float nA;                      // (1+a) d ln I / d a        = -1/2 + Lambda D
    float nL;                      // lambda d ln I / d lambda  = 2 lambda e^{-2 lambda}/(1-e^{-2 lambda}) - 1 + Lambda D
    float nk;                      // d ln I / d k
};

// Normaliser 1/I of eq.(10) (EXACT) or of NASG (approximate), and, if GRAD, the log-derivative terms.
template <bool EXACT, bool GRAD>
NASG_HD void normaliser(float l1, float l2, float Lam, float lam, float k, float &invI, float &nA,
                        float &nL, float &nk)
{
    const float INV_PI = 0.3183098861837907f;
    float em = f_exp(-2.0f * lam);
    float one_m = lam > 0.5f ? 1.0f - em : -expm1f(-2.0f * lam);
    float root = f_exp(0.5f * (l1 + l2));                   // lambda sqrt(1+a) = sqrt(lambda Lambda)
    float inv_base = root * INV_PI * f_rcp(one_m);          // 1 / (pi (1-e^{-2 lambda})/(lambda sqrt(1+a)))
    float dl = 0.f;
    if (GRAD) dl = 2.0f * lam * em * f_rcp(one_m) - 1.0f;   // lambda d ln(base)/d lambda
    if (!EXACT) {
        invI = 0.5f * inv_base;
        if (GRAD) { nA = -0.5f; nL = dl; nk = 0.f; }
        return;
    }
    float s = (Lam - k) * (Lam + k);                        // Lambda^2 - k^2
    float Psi, LD, dk;                                      // Psi, Lambda dPsi/dLambda, dPsi/dk
    if (s > 0.05f) {
        // k < Lambda:  Psi = (Lambda/r) e^{r-Lambda} (1-e^{-2r})/(1-e^{-2 Lambda}),  r-Lambda = -k^2/(Lambda+r)
        float r = f_sqrt(s);
        float ir = f_rcp(r);
        float del = k * k * f_rcp(Lam + r);                 // Lambda - r
        float e2r = f_exp(-2.0f * r), e2L = f_exp(-2.0f * Lam);
        Psi = Lam * ir * f_exp(-del) * (1.0f - e2r) * f_rcp(1.0f - e2L);
        if (GRAD) {
            float gr = g_fun(r), dg;
            if (r >= 4.0f) {
                // g(r) - g(Lambda) without cancellation
                float iL = f_rcp(Lam);
                float tail = 2.0f * (ir * e2r * f_rcp(1.0f - e2r) - iL * e2L * f_rcp(1.0f - e2L));
                dg = fmaf(del * ir * iL, 1.0f - (Lam + r) * ir * iL, tail);
            } else {
                dg = gr - g_fun(Lam);
            }
            LD = Psi * Lam * Lam * dg;                      // Lambda dPsi/dLambda = Psi Lambda^2 (g(r)-g(Lambda))
            dk = -Psi * k * gr;
        }
    } else {
        // k >= Lambda (or |s| tiny): S(s) = sinhc(sqrt(s)) continued to s < 0, S' = dS/ds
        float S, Sp;
        if (s > -0.05f) {
            S = fmaf(s, fmaf(s, fmaf(s, 1.9841270e-4f, 8.3333333e-3f), 0.16666667f), 1.0f);
            Sp = fmaf(s, fmaf(s, fmaf(s, 1.1022928e-5f, 5.9523810e-4f), 1.6666667e-2f), 0.16666667f);
        } else {
            float rho = f_sqrt(-s), sn, cs;
            f_sincos(rho, sn, cs);
            S = sn * f_rcp(rho);
            Sp = (cs - S) * f_rcp(2.0f * s);
        }
        float eL = f_exp(-Lam);
        float ish = 2.0f * eL * f_rcp(1.0f - eL * eL);      // 1/sinh(Lambda)
        Psi = Lam * S * ish;
        if (GRAD) {
            float coth = (1.0f + eL * eL) * f_rcp(1.0f - eL * eL);
            LD = Psi + 2.0f * Lam * Lam * Lam * Sp * ish - Psi * Lam * coth;
            dk = -2.0f * k * Lam * Sp * ish;
        }
    }
    float i1p = f_rcp(1.0f + Psi);
    invI = inv_base * i1p;
    if (GRAD) {
        float LamD = LD * i1p;
        nA = -0.5f + LamD;
        nL = dl + LamD;
        nk = dk * i1p;
    }
}

template <bool EXACT, bool GRAD>
NASG_HD void lobe_setup(const float4 q, const float4 sp, Lobe &L, LobeBwd &B)
{
    float inv_qn = f_rsqrt(q.x * q.x + q.y * q.y + q.z * q.z + q.w * q.w);
    // one Newton step: the frame error would otherwise be 2^-22 relative on every axis
    inv_qn = inv_qn * fmaf(-0.5f * (q.x * q.x + q.y * q.y + q.z * q.z + q.w * q.w), inv_qn * inv_qn, 1.5f);
    float w = q.x * inv_qn, x = q.y * inv_qn, y = q.z * inv_qn, z = q.w * inv_qn;
    L.Xx = 1.0f - 2.0f * (y * y + z * z); L.Xy = 2.0f * (x * y + w * z); L.Xz = 2.0f * (x * z - w * y);
    L.Yx = 2.0f * (x * y - w * z); L.Yy = 1.0f - 2.0f * (x * x + z * z); L.Yz = 2.0f * (y * z + w * x);
    L.Zx = 2.0f * (x * z + w * y); L.Zy = 2.0f * (y * z - w * x); L.Zz = 1.0f - 2.0f * (x * x + y * y);
    float Lam = expf(sp.x), lam = expf(sp.y);
    float one_pa = f_exp(sp.x - sp.y);
    L.lam2 = 2.0f * lam;
    L.a = fmaxf(one_pa - 1.0f, 0.0f);
    L.k = sp.z; L.phi = sp.w;
    float nA = 0.f, nL = 0.f, nk = 0.f;
    normaliser<EXACT, GRAD>(sp.x, sp.y, Lam, lam, sp.z, L.invI, nA, nL, nk);
    if (GRAD) {
        B.qw = w; B.qx = x; B.qy = y; B.qz = z; B.inv_qn = inv_qn;
        B.one_pa = one_pa; B.nA = nA; B.nL = nL; B.nk = nk;
    }
}

// ---------------------------------------------------------------------------------------------
// per (lobe, camera) evaluation
// ---------------------------------------------------------------------------------------------
struct EvalTerms {      // what the backward needs from the recomputed forward
    float u, v, c2, inv_s2, tau, Lk, kp, em1, inv_2kappa, Gbar, H, sn;
};

// G = H p E / I at direction (dx,dy,dz). If T != nullptr-like (FULL), also fills the terms for backward.
template <bool FULL>
NASG_HD float lobe_eval(const Lobe &L, float dx, float dy, float dz, EvalTerms &T)
{
    float u = fmaf(dx, L.Xx, fmaf(dy, L.Xy, dz * L.Xz));
    float om = fmaf(dx, L.Yx, fmaf(dy, L.Yy, dz * L.Yz));
    float v = fmaf(dx, L.Zx, fmaf(dy, L.Zy, dz * L.Zz));
    float s2 = fmaxf(fmaf(u, u, om * om), 1e-30f);          // 1 - v^2 without cancellation
    float inv_s2 = f_rcp(s2);
    float c2 = u * u * inv_s2;                               // d tau / d a, eq.(50)
    float tau = L.a * c2;
    // q = (1 - |v|)/2 = s^2/(2(1+|v|)): 1-kappa on the lobe side (v > 0), kappa itself on the far side;
    // neither 1 - v nor 1 + v is ever formed by a cancelling subtraction
    const bool upper = v > 0.0f;
    float q = fmaxf(0.5f * s2 * f_rcp(1.0f + fabsf(v)), 1e-30f);
    float Lk = log_kappa(q, upper);                          // ln kappa
    float x1 = fmaf(tau, Lk, Lk);                            // (1+tau) ln kappa
    float em1 = expm1_neg(x1);                               // kappa^(1+tau) - 1
    float arg = fmaf(L.lam2, em1, tau * Lk);                 // ln(p E)
    float Gbar = f_exp(arg) * L.invI;
    Gbar = (s2 <= 1e-30f && !upper) ? 0.0f : Gbar;           // d = -z: G = 0 (eq.(9), third case)
    float theta = fmaf(L.k, u, L.phi);
    float H;
    if (FULL) {
        float sn, cs;
        f_sincos(theta, sn, cs);
        H = fmaf(0.5f, cs, 0.5f);
        T.u = u; T.v = v; T.c2 = c2; T.inv_s2 = inv_s2; T.tau = tau; T.Lk = Lk; T.kp = em1 + 1.0f; T.em1 = em1;
        T.inv_2kappa = f_rcp(2.0f * (upper ? 1.0f - q : q));
        T.Gbar = Gbar; T.H = H; T.sn = sn;
    } else {
        H = fmaf(0.5f, f_cos(theta), 0.5f);
    }
    return Gbar * H;
}

} // namespace nasg
