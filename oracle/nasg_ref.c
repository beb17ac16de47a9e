/* ============================================================================================
 * oracle/nasg_ref.c — TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Plain, slow, fp64 CPU implementation of the per-Gaussian NASGabor colour evaluation
 * (forward + analytic backward) of arxiv/paper_2606_09794, written from the paper:
 *
 *   eq.(6)   PAPER.md:137      f_C(d) = c0 + sum_l w_l G_l(d)
 *   eq.(9)   PAPER.md:202-205  G = (1+cos(k d.x))/2 * exp{2 lambda kappa^(1+tau) - 2 lambda} * kappa^tau,
 *                              kappa = (d.z+1)/2, tau = a (d.x)^2 / (1-(d.z)^2); cases d = +-z
 *   eq.(10)  PAPER.md:209-211  integral = pi(1-e^{-2 lambda})/(lambda sqrt(1+a)) * (1+Psi),
 *                              Psi = 2 Lambda e^{-Lambda} sinhc(sqrt(Lambda^2-k^2)) / (1-e^{-2 Lambda}),
 *                              Lambda = lambda (1+a)
 *   NASG normaliser (norm_mode 0)  PAPER.md:423, 746 (eq.48): 2 pi (1-e^{-2 lambda})/(lambda sqrt(1+a))
 *   central-ray direction      PAPER.md:234: d = normalize(mean - campos), once per primitive per frame
 *   derivatives                PAPER.md:754-861 (eqs.50-65) for a, lambda, x, z, k with the NASG
 *                              normaliser; everything the paper does not give (d/mean, phase,
 *                              quaternion, the eq.(10) normaliser) is derived in DESIGN.md section 4
 *                              and pinned by finite differences (tests/test_oracle_pins.py).
 *
 * Readings of the paper (R1-R12) used here: the two log-bandwidths are
 * l1 = log Lambda, l2 = log lambda, a = Lambda/lambda - 1 (R1); "sinh" in eq.(10) is sinhc (R3);
 * sqrt(Lambda^2-k^2) is continued analytically to k > Lambda through sinhc(sqrt(s)) = sin(sqrt(-s))/sqrt(-s)
 * (R4); the phase phi enters only the carrier, never the normaliser (R5); epsilon = 0 (R8).
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
 * call this file. It shares no code, header, table or constant with the CUDA path; it has no
 * blocking, fusion or reordering beyond the formulas above. The one algebraic rearrangement is in
 * psi_terms(): e^{-Lambda} sinh(r) is written e^{r-Lambda}(1-e^{-2r})/2 because the literal product
 * overflows fp64 for Lambda > 709 (config 4 reaches Lambda = e^8); it is pinned against the literal
 * formula evaluated with 50-digit mpmath arithmetic.
 *
 * The measure-zero points d = +-z (R11) follow the paper's case split for the value; tau-dependent
 * gradient terms are defined as 0 there, which is their limit at +z. Pinned by
 * tests/test_oracle_pins.py::test_R11_* (case values of eq.(9), continuity of all seven partials at +z
 * along both meridians, the X-meridian limit 0 and the Y-meridian limit e^{-2 lambda} H/I at -z).
 * No function of this file is "parity unpinned".
 *
 * All arrays are fp64 host arrays (the harness promotes the fp32 inputs exactly). Layouts:
 *   means [N,3] quat [K,N,4] (w,x,y,z) shape [K,N,4] = (log Lambda, log lambda, k, phi)
 *   amp [K,3,N] dc [3,N] campos [C,3] vis [C,N] uint8 or NULL colors/g_colors [C,N,3]
 * ============================================================================================ */
#include <math.h>
#include <stddef.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#ifdef _OPENMP
#include <omp.h>
#endif

#define PI 3.14159265358979323846264338327950288

/* g(x) = (x coth x - 1) / x^2  (d ln sinhc(x) / dx = x g(x)) */
static double g_fun(double x)
{
    if (x < 1e-2) { double x2 = x * x; return 1.0 / 3.0 - x2 / 45.0 + 2.0 * x2 * x2 / 945.0; }
    double e = exp(-2.0 * x);
    double coth = (1.0 + e) / (1.0 - e);
    return (x * coth - 1.0) / (x * x);
}

/* Psi(Lambda,k) of eq.(10) and its two partial derivatives.
 * S(s) = sinhc(sqrt(s)) is an entire function of s = Lambda^2 - k^2 (reading R4). */
static void psi_terms(double Lam, double k, double *Psi, double *Psi_L, double *Psi_k)
{
    double s = Lam * Lam - k * k;
    if (s > 1e-4) {
        /* k < Lambda. 2 Lam e^{-Lam} sinh(r)/r / (1-e^{-2Lam}) with sinh(r) = e^r (1-e^{-2r})/2 and
         * r - Lam = -k^2/(Lam+r) (overflow-safe; identical algebraically). */
        double r = sqrt(s);
        double P = (Lam / r) * exp(-k * k / (Lam + r)) * (-expm1(-2.0 * r)) / (-expm1(-2.0 * Lam));
        /* ln Psi = ln Lam + ln sinhc(r) - ln sinh(Lam):
         *   d/dLam = 1/Lam + Lam g(r) - coth Lam = Lam (g(r) - g(Lam)),  d/dk = -k g(r). */
        double gr = g_fun(r), gL = g_fun(Lam);
        *Psi = P;
        *Psi_L = P * Lam * (gr - gL);
        *Psi_k = -P * k * gr;
    } else {
        /* k >= Lambda (or |s| tiny): S and S' = dS/ds directly; Lambda <= k here so sinh is safe
         * up to Lambda ~ 700, beyond which Psi underflows to 0 as it should. */
        double S, Sp;
        if (s > -1e-4) {
            S = 1.0 + s / 6.0 + s * s / 120.0 + s * s * s / 5040.0;
            Sp = 1.0 / 6.0 + s / 60.0 + s * s / 1680.0;
        } else {
            double rho = sqrt(-s);
            S = sin(rho) / rho;
            Sp = (cos(rho) - S) / (2.0 * s);
        }
        double ish = 1.0 / sinh(Lam);
        double P = Lam * S * ish; /* = 2 Lam e^{-Lam} S / (1 - e^{-2 Lam}) */
        *Psi = P;
        *Psi_L = P / Lam + 2.0 * Lam * Lam * Sp * ish - P / tanh(Lam);
        *Psi_k = -2.0 * k * Lam * Sp * ish;
    }
}

/* The integral I(lambda,a,k) the lobe is divided by, and d ln I / d(lambda, a, k).
 * norm_mode 1: eq.(10) literally. norm_mode 0: NASG normaliser. */
static void normaliser(double lambda, double a, double k, int norm_mode,
                       double *I, double *dlnI_dlambda, double *dlnI_da, double *dlnI_dk)
{
    double em2l = exp(-2.0 * lambda);
    double one_m = -expm1(-2.0 * lambda); /* 1 - e^{-2 lambda}, epsilon = 0 (R8) */
    double base = PI * one_m / (lambda * sqrt(1.0 + a));
    double dl = 2.0 * em2l / one_m - 1.0 / lambda;
    double da = -0.5 / (1.0 + a);
    if (norm_mode == 0) {
        *I = 2.0 * base;
        *dlnI_dlambda = dl; *dlnI_da = da; *dlnI_dk = 0.0;
        return;
    }
    double Lam = lambda * (1.0 + a), Psi, Psi_L, Psi_k;
    psi_terms(Lam, k, &Psi, &Psi_L, &Psi_k);
    *I = base * (1.0 + Psi);
    double D = Psi_L / (1.0 + Psi);
    *dlnI_dlambda = dl + (1.0 + a) * D; /* dLam/dlambda = 1+a */
    *dlnI_da = da + lambda * D;         /* dLam/da = lambda   */
    *dlnI_dk = Psi_k / (1.0 + Psi);
}

/* Value and scalar partial derivatives of one normalised lobe at (u = d.x, v = d.z).
 * out = { G, G_u, G_v, G_lambda, G_a, G_k, G_phi }  (u and v treated as independent). */
static void lobe_partials(double u, double v, double lambda, double a, double k, double phi,
                          int norm_mode, double out[7])
{
    double I, nl, na, nk;
    normaliser(lambda, a, k, norm_mode, &I, &nl, &na, &nk);
    double theta = k * u + phi;
    double H = 0.5 * (1.0 + cos(theta));
    double sn = sin(theta);
    double omv2 = 1.0 - v * v;

    if (omv2 <= 0.0 && v < 0.0) { /* d = -z: G = 0 (eq.9 third case) */
        for (int i = 0; i < 7; ++i) out[i] = 0.0;
        return;
    }
    double kappa = 0.5 * (v + 1.0);
    double c2, tau, tau_u, tau_v;
    if (omv2 <= 0.0) { /* d = +z: unnormalised value 1 (times the carrier at u = 0); tau terms := 0 (R11) */
        c2 = 0.0; tau = 0.0; tau_u = 0.0; tau_v = 0.0;
    } else {
        c2 = u * u / omv2;                 /* d tau / d a, eq.(50) */
        tau = a * c2;
        tau_u = 2.0 * a * u / omv2;        /* eq.(57) without the vector d */
        tau_v = 2.0 * a * u * u * v / (omv2 * omv2); /* eq.(61) without the vector d */
    }
    double L = log(kappa);
    double E = pow(kappa, tau);            /* eq.(47) */
    double kp = E * kappa;                 /* kappa^(1+tau) */
    double p = exp(2.0 * lambda * (kp - 1.0)); /* eq.(48) */
    double Gbar = p * E / I;               /* lobe without the carrier */
    double G = Gbar * H;

    /* ln(pE) = 2 lambda (kappa^(1+tau) - 1) + tau ln kappa */
    double A_tau = L * (1.0 + 2.0 * lambda * kp);                         /* d ln(pE)/d tau   */
    double A_kappa = (tau + 2.0 * lambda * (1.0 + tau) * kp) / kappa;     /* d ln(pE)/d kappa */

    out[0] = G;
    out[1] = G * A_tau * tau_u - Gbar * 0.5 * k * sn;       /* eqs.(58)-(60) */
    out[2] = G * (A_tau * tau_v + 0.5 * A_kappa);           /* eqs.(61)-(64), d kappa/d v = 1/2 */
    out[3] = G * (2.0 * (kp - 1.0) - nl);                   /* eqs.(54)-(56) */
    out[4] = G * (A_tau * c2 - na);                         /* eqs.(50)-(53) */
    out[5] = -Gbar * 0.5 * u * sn - G * nk;                 /* eq.(65) + normaliser term */
    out[6] = -Gbar * 0.5 * sn;
}

/* Columns X (carrier axis) and Z (lobe axis) of R(q/|q|), Hamilton convention (w,x,y,z) (R12). */
static void frame_from_quat(const double q[4], double qh[4], double *qnorm, double X[3], double Z[3])
{
    double n = sqrt(q[0] * q[0] + q[1] * q[1] + q[2] * q[2] + q[3] * q[3]);
    double w = q[0] / n, x = q[1] / n, y = q[2] / n, z = q[3] / n;
    qh[0] = w; qh[1] = x; qh[2] = y; qh[3] = z; *qnorm = n;
    X[0] = 1.0 - 2.0 * (y * y + z * z); X[1] = 2.0 * (x * y + w * z); X[2] = 2.0 * (x * z - w * y);
    Z[0] = 2.0 * (x * z + w * y); Z[1] = 2.0 * (y * z - w * x); Z[2] = 1.0 - 2.0 * (x * x + y * y);
}

/* ------------------------------------------------------------------------------------------ */
/* scalar helpers exported for the pins                                                        */
/* ------------------------------------------------------------------------------------------ */
double nasg_ref_integral(double lambda, double a, double k, int norm_mode)
{
    double I, x0, x1, x2;
    normaliser(lambda, a, k, norm_mode, &I, &x0, &x1, &x2);
    return I;
}
void nasg_ref_psi(double Lam, double k, double out[3]) { psi_terms(Lam, k, &out[0], &out[1], &out[2]); }
void nasg_ref_dlnI(double lambda, double a, double k, int norm_mode, double out[3])
{
    double I;
    normaliser(lambda, a, k, norm_mode, &I, &out[0], &out[1], &out[2]);
}
void nasg_ref_partials(double u, double v, double lambda, double a, double k, double phi,
                       int norm_mode, double out[7])
{
    lobe_partials(u, v, lambda, a, k, phi, norm_mode, out);
}
void nasg_ref_frame(const double q[4], double X[3], double Z[3])
{
    double qh[4], n;
    frame_from_quat(q, qh, &n, X, Z);
}
int nasg_ref_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
/* timing harness only (bench.py: single-thread vs all-core baseline); no effect on any result */
void nasg_ref_set_num_threads(int t)
{
#ifdef _OPENMP
    if (t > 0) omp_set_num_threads(t);
#else
    (void)t;
#endif
}

/* ------------------------------------------------------------------------------------------ */
/* forward: colors[c,n,:] = c0 + sum_l w_l G_l(d_cn); culled entries 0                          */
/* ------------------------------------------------------------------------------------------ */
int nasg_ref_fwd(int64_t N, int K, int C, const double *means, const double *quat,
                 const double *shape, const double *amp, const double *dc, const double *campos,
                 const uint8_t *vis, int norm_mode, double *colors)
{
#pragma omp parallel for schedule(static)
    for (int64_t n = 0; n < N; ++n) {
        for (int c = 0; c < C; ++c) {
            double *col = colors + ((size_t)c * N + n) * 3;
            if (vis && !vis[(size_t)c * N + n]) { col[0] = col[1] = col[2] = 0.0; continue; }
            double dx = means[3 * n] - campos[3 * c], dy = means[3 * n + 1] - campos[3 * c + 1],
                   dz = means[3 * n + 2] - campos[3 * c + 2];
            double dist = sqrt(dx * dx + dy * dy + dz * dz);
            double d[3] = { dx / dist, dy / dist, dz / dist };
            double rgb[3] = { dc[n], dc[N + n], dc[2 * N + n] };
            for (int l = 0; l < K; ++l) {
                const double *q = quat + ((size_t)l * N + n) * 4;
                const double *sp = shape + ((size_t)l * N + n) * 4;
                double qh[4], qn, X[3], Z[3], o[7];
                frame_from_quat(q, qh, &qn, X, Z);
                double Lam = exp(sp[0]), lambda = exp(sp[1]);
                double a = Lam / lambda - 1.0;
                double u = d[0] * X[0] + d[1] * X[1] + d[2] * X[2];
                double v = d[0] * Z[0] + d[1] * Z[1] + d[2] * Z[2];
                lobe_partials(u, v, lambda, a, sp[2], sp[3], norm_mode, o);
                for (int ch = 0; ch < 3; ++ch) rgb[ch] += amp[((size_t)l * 3 + ch) * N + n] * o[0];
            }
            col[0] = rgb[0]; col[1] = rgb[1]; col[2] = rgb[2];
        }
    }
    return 0;
}

/* ------------------------------------------------------------------------------------------ */
/* backward: exact gradient of sum(g_colors * colors) w.r.t. every input; any output may be NULL */
/* ------------------------------------------------------------------------------------------ */
int nasg_ref_bwd(int64_t N, int K, int C, const double *means, const double *quat,
                 const double *shape, const double *amp, const double *dc, const double *campos,
                 const uint8_t *vis, const double *g_colors, int norm_mode, double *g_means,
                 double *g_quat, double *g_shape, double *g_amp, double *g_dc, double *g_campos)
{
    (void)dc;
    if (g_campos) memset(g_campos, 0, sizeof(double) * 3 * (size_t)C);
#pragma omp parallel
    {
        double *gc_local = (double *)calloc((size_t)3 * C, sizeof(double));
#pragma omp for schedule(static)
        for (int64_t n = 0; n < N; ++n) {
            double gm[3] = { 0, 0, 0 }, gdc[3] = { 0, 0, 0 };
            for (int c = 0; c < C; ++c) {
                if (vis && !vis[(size_t)c * N + n]) continue;
                const double *gcol = g_colors + ((size_t)c * N + n) * 3;
                for (int ch = 0; ch < 3; ++ch) gdc[ch] += gcol[ch];
            }
            for (int l = 0; l < K; ++l) {
                const double *q = quat + ((size_t)l * N + n) * 4;
                const double *sp = shape + ((size_t)l * N + n) * 4;
                double qh[4], qn, X[3], Z[3];
                frame_from_quat(q, qh, &qn, X, Z);
                double Lam = exp(sp[0]), lambda = exp(sp[1]);
                double a = Lam / lambda - 1.0;
                double w[3] = { amp[((size_t)l * 3 + 0) * N + n], amp[((size_t)l * 3 + 1) * N + n],
                                amp[((size_t)l * 3 + 2) * N + n] };
                double gX[3] = { 0, 0, 0 }, gZ[3] = { 0, 0, 0 }, gw[3] = { 0, 0, 0 };
                double g_lambda = 0, g_a = 0, g_k = 0, g_phi = 0;
                for (int c = 0; c < C; ++c) {
                    if (vis && !vis[(size_t)c * N + n]) continue;
                    const double *gcol = g_colors + ((size_t)c * N + n) * 3;
                    double dx = means[3 * n] - campos[3 * c], dy = means[3 * n + 1] - campos[3 * c + 1],
                           dz = means[3 * n + 2] - campos[3 * c + 2];
                    double dist = sqrt(dx * dx + dy * dy + dz * dz);
                    double d[3] = { dx / dist, dy / dist, dz / dist };
                    double u = d[0] * X[0] + d[1] * X[1] + d[2] * X[2];
                    double v = d[0] * Z[0] + d[1] * Z[1] + d[2] * Z[2];
                    double o[7];
                    lobe_partials(u, v, lambda, a, sp[2], sp[3], norm_mode, o);
                    double gG = gcol[0] * w[0] + gcol[1] * w[1] + gcol[2] * w[2]; /* dL/dG, eq.(6) */
                    for (int ch = 0; ch < 3; ++ch) gw[ch] += gcol[ch] * o[0];
                    g_lambda += gG * o[3]; g_a += gG * o[4]; g_k += gG * o[5]; g_phi += gG * o[6];
                    double gd[3];
                    for (int i = 0; i < 3; ++i) {
                        gX[i] += gG * o[1] * d[i];                 /* dG/dx = G_u d, eq.(60) */
                        gZ[i] += gG * o[2] * d[i];                 /* dG/dz = G_v d, eq.(64) */
                        gd[i] = gG * (o[1] * X[i] + o[2] * Z[i]);  /* dG/dd */
                    }
                    /* d = Delta/|Delta|: dd/dm = (I - d d^T)/|Delta| */
                    double dg = d[0] * gd[0] + d[1] * gd[1] + d[2] * gd[2];
                    for (int i = 0; i < 3; ++i) {
                        double t = (gd[i] - d[i] * dg) / dist;
                        gm[i] += t;
                        gc_local[3 * c + i] -= t;
                    }
                }
                if (g_amp) for (int ch = 0; ch < 3; ++ch) g_amp[((size_t)l * 3 + ch) * N + n] = gw[ch];
                if (g_shape) {
                    double *gs = g_shape + ((size_t)l * N + n) * 4;
                    /* (lambda, a) = (e^{l2}, e^{l1-l2} - 1) */
                    gs[0] = g_a * (1.0 + a);
                    gs[1] = lambda * g_lambda - g_a * (1.0 + a);
                    gs[2] = g_k;
                    gs[3] = g_phi;
                }
                if (g_quat) {
                    double qw = qh[0], qx = qh[1], qy = qh[2], qz = qh[3];
                    double gq[4];
                    /* transpose Jacobian of the X and Z columns of R(qhat) */
                    gq[0] = 2.0 * (qz * gX[1] - qy * gX[2] + qy * gZ[0] - qx * gZ[1]);
                    gq[1] = 2.0 * (qy * gX[1] + qz * gX[2] + qz * gZ[0] - qw * gZ[1]) - 4.0 * qx * gZ[2];
                    gq[2] = -4.0 * qy * gX[0] + 2.0 * (qx * gX[1] - qw * gX[2] + qw * gZ[0] + qz * gZ[1])
                            - 4.0 * qy * gZ[2];
                    gq[3] = -4.0 * qz * gX[0] + 2.0 * (qw * gX[1] + qx * gX[2] + qx * gZ[0] + qy * gZ[1]);
                    /* qhat = q/|q|: dqhat/dq = (I - qhat qhat^T)/|q| */
                    double dot = qh[0] * gq[0] + qh[1] * gq[1] + qh[2] * gq[2] + qh[3] * gq[3];
                    double *o4 = g_quat + ((size_t)l * N + n) * 4;
                    for (int i = 0; i < 4; ++i) o4[i] = (gq[i] - qh[i] * dot) / qn;
                }
            }
            if (g_means) { g_means[3 * n] = gm[0]; g_means[3 * n + 1] = gm[1]; g_means[3 * n + 2] = gm[2]; }
            if (g_dc) { g_dc[n] = gdc[0]; g_dc[N + n] = gdc[1]; g_dc[2 * N + n] = gdc[2]; }
        }
        if (g_campos) {
#pragma omp critical
            for (int i = 0; i < 3 * C; ++i) g_campos[i] += gc_local[i];
        }
        free(gc_local);
    }
    return 0;
}

/* ============================================================================================
 * Paper-native parameter record: 3 + 9K floats per primitive
 * (Table 5), no phase, Table 8 activations:
 *
 *   (c_theta, c_phi, c_tau) = tanh(raw)                 cosines of the frame angles
 *   lambda = exp(raw), a = exp(raw), k = 20 (tanh(raw) + 1), w = tanh(raw)
 *   s = +sqrt(1 - c^2);  z = (c_theta s_phi, s_theta s_phi, c_phi),
 *   x = (c_theta c_phi c_tau - s_theta s_tau, s_theta c_phi c_tau + c_theta s_tau, -s_phi c_tau)
 *                                                      Supplementary C
 *   backward through the frame: eqs.(37)-(44) PAPER.md:687-720, with eq.(39) read as
 *   dz/dc_theta = (s_phi, -(c_theta/s_theta) s_phi, 0) (R6(iii): the printed eq.(39) is garbled),
 *   and ds/dc = -c/s (eq.36).
 * The DC colour c0 has no activation (the paper lists none). The lobe itself is lobe_partials()
 * above with phi = 0. Layouts: euler [K,N,3] (theta, phi, tau raw), shp [K,N,3] (lambda, a, k raw),
 * ampraw [K,3,N], dc [3,N]; gradients are with respect to the RAW (pre-activation) values.
 * ============================================================================================ */
typedef struct {
    double c[3], s[3];      /* cos / sin of theta, phi, tau */
    double X[3], Z[3];
    double lambda, a, k, w[3];
    double tk;              /* tanh(k_raw) */
} paper_lobe;

static void paper_decode(const double *eu, const double *sp, const double w_raw[3], paper_lobe *L)
{
    for (int i = 0; i < 3; ++i) { L->c[i] = tanh(eu[i]); L->s[i] = sqrt(1.0 - L->c[i] * L->c[i]); }
    const double ct = L->c[0], cp = L->c[1], cu = L->c[2], st = L->s[0], sp_ = L->s[1], su = L->s[2];
    L->Z[0] = ct * sp_; L->Z[1] = st * sp_; L->Z[2] = cp;
    L->X[0] = ct * cp * cu - st * su; L->X[1] = st * cp * cu + ct * su; L->X[2] = -sp_ * cu;
    L->lambda = exp(sp[0]); L->a = exp(sp[1]);
    L->tk = tanh(sp[2]); L->k = 20.0 * (L->tk + 1.0);
    for (int ch = 0; ch < 3; ++ch) L->w[ch] = tanh(w_raw[ch]);
}

/* exported for the pins: frame (X, Z) and its derivatives with respect to the three cosines, eqs.(38)-(44) */
void nasg_ref_paper_frame(const double eu_raw[3], double X[3], double Z[3], double dX[3][3], double dZ[3][3])
{
    paper_lobe L; double sp[3] = { 0, 0, 0 }, w[3] = { 0, 0, 0 };
    paper_decode(eu_raw, sp, w, &L);
    for (int i = 0; i < 3; ++i) { X[i] = L.X[i]; Z[i] = L.Z[i]; }
    const double ct = L.c[0], cp = L.c[1], cu = L.c[2], st = L.s[0], sp_ = L.s[1], su = L.s[2];
    /* d/dc_theta: eq.(38), eq.(39) as corrected */
    dX[0][0] = cp * cu + (ct / st) * su; dX[0][1] = -(ct / st) * cp * cu + su; dX[0][2] = 0.0;
    dZ[0][0] = sp_; dZ[0][1] = -(ct / st) * sp_; dZ[0][2] = 0.0;
    /* d/dc_phi: eqs.(41), (42) */
    dX[1][0] = ct * cu; dX[1][1] = st * cu; dX[1][2] = (cp / sp_) * cu;
    dZ[1][0] = -ct * cp / sp_; dZ[1][1] = -st * cp / sp_; dZ[1][2] = 1.0;
    /* d/dc_tau: eq.(44); z does not depend on tau */
    dX[2][0] = ct * cp + st * cu / su; dX[2][1] = st * cp - ct * cu / su; dX[2][2] = -sp_;
    dZ[2][0] = dZ[2][1] = dZ[2][2] = 0.0;
}

int nasg_ref_paper_fwd(int64_t N, int K, int C, const double *means, const double *euler, const double *shp,
                       const double *ampraw, const double *dc, const double *campos, const uint8_t *vis,
                       int norm_mode, double *colors)
{
#pragma omp parallel for schedule(static)
    for (int64_t n = 0; n < N; ++n) {
        for (int c = 0; c < C; ++c) {
            double *col = colors + ((size_t)c * N + n) * 3;
            if (vis && !vis[(size_t)c * N + n]) { col[0] = col[1] = col[2] = 0.0; continue; }
            double dx = means[3 * n] - campos[3 * c], dy = means[3 * n + 1] - campos[3 * c + 1],
                   dz = means[3 * n + 2] - campos[3 * c + 2];
            double dist = sqrt(dx * dx + dy * dy + dz * dz);
            double d[3] = { dx / dist, dy / dist, dz / dist };
            double rgb[3] = { dc[n], dc[N + n], dc[2 * N + n] };
            for (int l = 0; l < K; ++l) {
                double wr[3] = { ampraw[((size_t)l * 3 + 0) * N + n], ampraw[((size_t)l * 3 + 1) * N + n],
                                 ampraw[((size_t)l * 3 + 2) * N + n] };
                paper_lobe L; double o[7];
                paper_decode(euler + ((size_t)l * N + n) * 3, shp + ((size_t)l * N + n) * 3, wr, &L);
                double u = d[0] * L.X[0] + d[1] * L.X[1] + d[2] * L.X[2];
                double v = d[0] * L.Z[0] + d[1] * L.Z[1] + d[2] * L.Z[2];
                lobe_partials(u, v, L.lambda, L.a, L.k, 0.0, norm_mode, o);
                for (int ch = 0; ch < 3; ++ch) rgb[ch] += L.w[ch] * o[0];
            }
            col[0] = rgb[0]; col[1] = rgb[1]; col[2] = rgb[2];
        }
    }
    return 0;
}

int nasg_ref_paper_bwd(int64_t N, int K, int C, const double *means, const double *euler, const double *shp,
                       const double *ampraw, const double *dc, const double *campos, const uint8_t *vis,
                       const double *g_colors, int norm_mode, double *g_means, double *g_euler, double *g_shp,
                       double *g_ampraw, double *g_dc)
{
    (void)dc;
#pragma omp parallel for schedule(static)
    for (int64_t n = 0; n < N; ++n) {
        double gm[3] = { 0, 0, 0 }, gdc[3] = { 0, 0, 0 };
        for (int c = 0; c < C; ++c) {
            if (vis && !vis[(size_t)c * N + n]) continue;
            const double *gcol = g_colors + ((size_t)c * N + n) * 3;
            for (int ch = 0; ch < 3; ++ch) gdc[ch] += gcol[ch];
        }
        for (int l = 0; l < K; ++l) {
            const double *eu = euler + ((size_t)l * N + n) * 3;
            double wr[3] = { ampraw[((size_t)l * 3 + 0) * N + n], ampraw[((size_t)l * 3 + 1) * N + n],
                             ampraw[((size_t)l * 3 + 2) * N + n] };
            paper_lobe L;
            paper_decode(eu, shp + ((size_t)l * N + n) * 3, wr, &L);
            double gX[3] = { 0, 0, 0 }, gZ[3] = { 0, 0, 0 }, gw[3] = { 0, 0, 0 }, g_lambda = 0, g_a = 0, g_k = 0;
            for (int c = 0; c < C; ++c) {
                if (vis && !vis[(size_t)c * N + n]) continue;
                const double *gcol = g_colors + ((size_t)c * N + n) * 3;
                double dx = means[3 * n] - campos[3 * c], dy = means[3 * n + 1] - campos[3 * c + 1],
                       dz = means[3 * n + 2] - campos[3 * c + 2];
                double dist = sqrt(dx * dx + dy * dy + dz * dz);
                double d[3] = { dx / dist, dy / dist, dz / dist };
                double u = d[0] * L.X[0] + d[1] * L.X[1] + d[2] * L.X[2];
                double v = d[0] * L.Z[0] + d[1] * L.Z[1] + d[2] * L.Z[2];
                double o[7];
                lobe_partials(u, v, L.lambda, L.a, L.k, 0.0, norm_mode, o);
                double gG = gcol[0] * L.w[0] + gcol[1] * L.w[1] + gcol[2] * L.w[2];
                for (int ch = 0; ch < 3; ++ch) gw[ch] += gcol[ch] * o[0];
                g_lambda += gG * o[3]; g_a += gG * o[4]; g_k += gG * o[5];
                double gd[3];
                for (int i = 0; i < 3; ++i) {
                    gX[i] += gG * o[1] * d[i];
                    gZ[i] += gG * o[2] * d[i];
                    gd[i] = gG * (o[1] * L.X[i] + o[2] * L.Z[i]);
                }
                double dg = d[0] * gd[0] + d[1] * gd[1] + d[2] * gd[2];
                for (int i = 0; i < 3; ++i) gm[i] += (gd[i] - d[i] * dg) / dist;
            }
            /* chain rule through the cosines, eqs.(37), (40), (43), then through tanh: dc/draw = 1 - c^2 */
            double X[3], Z[3], dX[3][3], dZ[3][3];
            nasg_ref_paper_frame(eu, X, Z, dX, dZ);
            if (g_euler) {
                double *ge = g_euler + ((size_t)l * N + n) * 3;
                for (int i = 0; i < 3; ++i) {
                    double gc = 0.0;
                    for (int j = 0; j < 3; ++j) gc += gX[j] * dX[i][j] + gZ[j] * dZ[i][j];
                    ge[i] = gc * (1.0 - L.c[i] * L.c[i]);
                }
            }
            if (g_shp) {
                double *gs = g_shp + ((size_t)l * N + n) * 3;
                gs[0] = g_lambda * L.lambda;                       /* lambda = exp(raw) */
                gs[1] = g_a * L.a;                                 /* a = exp(raw)      */
                gs[2] = g_k * 20.0 * (1.0 - L.tk * L.tk);          /* k = 20 (tanh(raw) + 1) */
            }
            if (g_ampraw)
                for (int ch = 0; ch < 3; ++ch) g_ampraw[((size_t)l * 3 + ch) * N + n] = gw[ch] * (1.0 - L.w[ch] * L.w[ch]);
        }
        if (g_means) { g_means[3 * n] = gm[0]; g_means[3 * n + 1] = gm[1]; g_means[3 * n + 2] = gm[2]; }
        if (g_dc) { g_dc[n] = gdc[0]; g_dc[N + n] = gdc[1]; g_dc[2 * N + n] = gdc[2]; }
    }
    return 0;
}
