/* ============================================================================================
 * oracle/iso_ref.c — TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Plain fp64 CPU implementation of the per-Gaussian colour evaluation (forward + analytic backward) with the
 * ISOTROPIC spherical functions of the paper's Table 6, in the
 * appearance model of eq.(6):   colour = c0 + sum_l w_l c_l G_l(d . z_l),   d = normalize(mean - campos)
 * (PAPER.md:234), each multiplied by its normalisation constant c (the paper's study normalises every function,
 * PAPER.md:172-182):
 *
 *   kind 0  Spherical Gaussian   G = exp{lambda (z.d - 1)},                 c = lambda / (2 pi (1 - e^{-2 lambda}))
 *   kind 1  Spherical Beta       G = max(z.d, 0)^beta,                      c = (beta + 1) / (2 pi)
 *   kind 2  Spherical Cauchy     G = ((1 - rho^2) / (1 + rho^2 - 2 rho z.d))^2,   c = 1 / (4 pi)
 *
 * Readings (R19): Table 6 prints the Cauchy denominator as "1 - rho^2 - 2 rho z.d"; only
 * 1 + rho^2 - 2 rho z.d integrates to 4 pi (= 1/c) over the sphere, so that is what is implemented (pinned by quadrature;
 * the printed form is shown NOT to). The Beta lobe is taken as 0 on the far hemisphere (z.d <= 0), which is what
 * c = (beta+1)/(2 pi) normalises. Parameterisation: the axis is a free 3-vector z (normalised inside, gradient through
 * the normalisation); the shape parameter is stored raw: lambda = exp(raw), beta = exp(raw), rho = 1/(1 + e^{-raw}).
 * Layouts: means [N,3], axis [K,N,3], shp [K,N] (raw), amp [K,3,N], dc [3,N], campos [C,3], vis [C,N] uint8 or NULL,
 * colors / g_colors [C,N,3]. Shares no code with the CUDA path; only tests/ and bench.py's oracle legs may call it.
 * ============================================================================================ */
#include <math.h>
#include <stddef.h>
#include <stdint.h>

#define PI 3.14159265358979323846264338327950288

/* F = c G and its partial derivatives with respect to v = z.d and to the RAW shape value. out = {F, F_v, F_raw}. */
void iso_ref_lobe(int kind, double v, double raw, double out[3])
{
    if (kind == 0) {
        double lam = exp(raw);
        double one_m = -expm1(-2.0 * lam);
        double c = lam / (2.0 * PI * one_m);
        double F = c * exp(lam * (v - 1.0));
        double dlnc = 1.0 / lam - 2.0 * exp(-2.0 * lam) / one_m;        /* d ln c / d lambda */
        out[0] = F; out[1] = lam * F; out[2] = F * ((v - 1.0) + dlnc) * lam;
    } else if (kind == 1) {
        double beta = exp(raw);
        if (v <= 0.0) { out[0] = out[1] = out[2] = 0.0; return; }
        double F = (beta + 1.0) / (2.0 * PI) * pow(v, beta);
        out[0] = F; out[1] = beta * F / v; out[2] = F * (1.0 / (beta + 1.0) + log(v)) * beta;
    } else {
        double rho = 1.0 / (1.0 + exp(-raw));
        double num = 1.0 - rho * rho, D = 1.0 + rho * rho - 2.0 * rho * v;
        double F = (num / D) * (num / D) / (4.0 * PI);
        double F_rho = F * 2.0 * (-2.0 * rho / num - (2.0 * rho - 2.0 * v) / D);
        out[0] = F; out[1] = F * 4.0 * rho / D; out[2] = F_rho * rho * (1.0 - rho);
    }
}

int iso_ref_fwd(int64_t N, int K, int C, int kind, const double *means, const double *axis, const double *shp,
                const double *amp, const double *dc, const double *campos, const uint8_t *vis, double *colors)
{
#pragma omp parallel for schedule(static)
    for (int64_t n = 0; n < N; ++n) {
        for (int c = 0; c < C; ++c) {
            double *col = colors + ((size_t)c * N + n) * 3;
            if (vis && !vis[(size_t)c * N + n]) { col[0] = col[1] = col[2] = 0.0; continue; }
            double dx = means[3 * n] - campos[3 * c], dy = means[3 * n + 1] - campos[3 * c + 1], dz = means[3 * n + 2] - campos[3 * c + 2];
            double dist = sqrt(dx * dx + dy * dy + dz * dz);
            double d[3] = { dx / dist, dy / dist, dz / dist };
            double rgb[3] = { dc[n], dc[N + n], dc[2 * N + n] };
            for (int l = 0; l < K; ++l) {
                const double *z = axis + ((size_t)l * N + n) * 3;
                double zn = sqrt(z[0] * z[0] + z[1] * z[1] + z[2] * z[2]);
                double v = (d[0] * z[0] + d[1] * z[1] + d[2] * z[2]) / zn, o[3];
                iso_ref_lobe(kind, v, shp[(size_t)l * N + n], o);
                for (int ch = 0; ch < 3; ++ch) rgb[ch] += amp[((size_t)l * 3 + ch) * N + n] * o[0];
            }
            col[0] = rgb[0]; col[1] = rgb[1]; col[2] = rgb[2];
        }
    }
    return 0;
}

int iso_ref_bwd(int64_t N, int K, int C, int kind, const double *means, const double *axis, const double *shp,
                const double *amp, const double *dc, const double *campos, const uint8_t *vis, const double *g_colors,
                double *g_means, double *g_axis, double *g_shp, double *g_amp, double *g_dc)
{
    (void)dc;
#pragma omp parallel for schedule(static)
    for (int64_t n = 0; n < N; ++n) {
        double gm[3] = { 0, 0, 0 }, gdc[3] = { 0, 0, 0 };
        for (int c = 0; c < C; ++c) {
            if (vis && !vis[(size_t)c * N + n]) continue;
            for (int ch = 0; ch < 3; ++ch) gdc[ch] += g_colors[((size_t)c * N + n) * 3 + ch];
        }
        for (int l = 0; l < K; ++l) {
            const double *z = axis + ((size_t)l * N + n) * 3;
            double zn = sqrt(z[0] * z[0] + z[1] * z[1] + z[2] * z[2]);
            double zh[3] = { z[0] / zn, z[1] / zn, z[2] / zn };
            double w[3] = { amp[((size_t)l * 3 + 0) * N + n], amp[((size_t)l * 3 + 1) * N + n], amp[((size_t)l * 3 + 2) * N + n] };
            double gz[3] = { 0, 0, 0 }, gw[3] = { 0, 0, 0 }, gs = 0.0;
            for (int c = 0; c < C; ++c) {
                if (vis && !vis[(size_t)c * N + n]) continue;
                const double *gcol = g_colors + ((size_t)c * N + n) * 3;
                double dx = means[3 * n] - campos[3 * c], dy = means[3 * n + 1] - campos[3 * c + 1], dz = means[3 * n + 2] - campos[3 * c + 2];
                double dist = sqrt(dx * dx + dy * dy + dz * dz);
                double d[3] = { dx / dist, dy / dist, dz / dist };
                double v = d[0] * zh[0] + d[1] * zh[1] + d[2] * zh[2], o[3];
                iso_ref_lobe(kind, v, shp[(size_t)l * N + n], o);
                double gF = gcol[0] * w[0] + gcol[1] * w[1] + gcol[2] * w[2];      /* dL/dF, eq.(6) */
                for (int ch = 0; ch < 3; ++ch) gw[ch] += gcol[ch] * o[0];
                gs += gF * o[2];
                double gd[3];
                for (int i = 0; i < 3; ++i) { gz[i] += gF * o[1] * d[i]; gd[i] = gF * o[1] * zh[i]; }   /* v = d . zhat */
                double dg = d[0] * gd[0] + d[1] * gd[1] + d[2] * gd[2];
                for (int i = 0; i < 3; ++i) gm[i] += (gd[i] - d[i] * dg) / dist;    /* d = Delta/|Delta| */
            }
            if (g_amp) for (int ch = 0; ch < 3; ++ch) g_amp[((size_t)l * 3 + ch) * N + n] = gw[ch];
            if (g_shp) g_shp[(size_t)l * N + n] = gs;
            if (g_axis) {       /* zhat = z/|z|: (I - zhat zhat^T)/|z| */
                double dot = zh[0] * gz[0] + zh[1] * gz[1] + zh[2] * gz[2];
                for (int i = 0; i < 3; ++i) g_axis[((size_t)l * N + n) * 3 + i] = (gz[i] - zh[i] * dot) / zn;
            }
        }
        if (g_means) { g_means[3 * n] = gm[0]; g_means[3 * n + 1] = gm[1]; g_means[3 * n + 2] = gm[2]; }
        if (g_dc) { g_dc[n] = gdc[0]; g_dc[N + n] = gdc[1]; g_dc[2 * N + n] = gdc[2]; }
    }
    return 0;
}
