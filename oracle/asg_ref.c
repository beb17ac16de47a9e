/* ============================================================================================
 * oracle/asg_ref.c — TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Plain fp64 CPU implementation of the per-Gaussian colour evaluation (forward + analytic backward) with the
 * Anisotropic Spherical Gaussian of the paper's Table 6 ([XSD*13]) in the
 * appearance model of eq.(6):   colour = c0 + sum_l w_l G_l(d),   d = normalize(mean - campos),
 *
 *   G(d; x, y, z, mu, lambda) = max(d.z, 0) exp{ -mu (d.x)^2 - lambda (d.y)^2 }
 *
 * with no normalisation constant (Table 6: "Not analytical"). Parameterisation (the quaternion frame of the NASGabor
 * path, R12): [x y z] = R(q/|q|), Hamilton convention (w,x,y,z), gradient through the normalisation; the bandwidths are
 * stored raw: mu = exp(raw0), lambda = exp(raw1). At d.z = 0 the lobe has a kink: the derivative is taken as 0 there
 * (the max's far side), as on the whole far hemisphere.
 * Layouts: means [N,3], quat [K,N,4], shp [K,N,2] (raw mu, raw lambda), amp [K,3,N], dc [3,N], campos [C,3],
 * vis [C,N] uint8 or NULL, colors / g_colors [C,N,3]. Shares no code with the CUDA path; only tests/ and bench.py's
 * oracle legs may call it.
 * ============================================================================================ */
#include <math.h>
#include <stddef.h>
#include <stdint.h>

/* Columns of R(q/|q|); qh = q/|q|, *qn = |q|. */
static void asg_frame(const double q[4], double qh[4], double *qn, double X[3], double Y[3], double Z[3])
{
    double n = sqrt(q[0] * q[0] + q[1] * q[1] + q[2] * q[2] + q[3] * q[3]);
    double w = q[0] / n, x = q[1] / n, y = q[2] / n, z = q[3] / n;
    qh[0] = w; qh[1] = x; qh[2] = y; qh[3] = z; *qn = n;
    X[0] = 1.0 - 2.0 * (y * y + z * z); X[1] = 2.0 * (x * y + w * z); X[2] = 2.0 * (x * z - w * y);
    Y[0] = 2.0 * (x * y - w * z); Y[1] = 1.0 - 2.0 * (x * x + z * z); Y[2] = 2.0 * (y * z + w * x);
    Z[0] = 2.0 * (x * z + w * y); Z[1] = 2.0 * (y * z - w * x); Z[2] = 1.0 - 2.0 * (x * x + y * y);
}
void asg_ref_frame(const double q[4], double X[3], double Y[3], double Z[3])
{
    double qh[4], qn;
    asg_frame(q, qh, &qn, X, Y, Z);
}

/* G and its partial derivatives at (u, t, v) = (d.x, d.y, d.z): out = {G, G_u, G_t, G_v, G_rawmu, G_rawlambda}. */
void asg_ref_lobe(double u, double t, double v, double raw_mu, double raw_lam, double out[6])
{
    double mu = exp(raw_mu), lam = exp(raw_lam);
    if (v <= 0.0) { for (int i = 0; i < 6; ++i) out[i] = 0.0; return; }
    double S = exp(-mu * u * u - lam * t * t), G = v * S;
    out[0] = G;
    out[1] = -2.0 * mu * u * G;
    out[2] = -2.0 * lam * t * G;
    out[3] = S;
    out[4] = -mu * u * u * G;           /* d/draw = mu d/dmu */
    out[5] = -lam * t * t * G;
}

int asg_ref_fwd(int64_t N, int K, int C, const double *means, const double *quat, const double *shp, const double *amp,
                const double *dc, const double *campos, const uint8_t *vis, double *colors)
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
                double qh[4], qn, X[3], Y[3], Z[3], o[6];
                asg_frame(quat + ((size_t)l * N + n) * 4, qh, &qn, X, Y, Z);
                double u = d[0] * X[0] + d[1] * X[1] + d[2] * X[2];
                double t = d[0] * Y[0] + d[1] * Y[1] + d[2] * Y[2];
                double v = d[0] * Z[0] + d[1] * Z[1] + d[2] * Z[2];
                const double *sp = shp + ((size_t)l * N + n) * 2;
                asg_ref_lobe(u, t, v, sp[0], sp[1], o);
                for (int ch = 0; ch < 3; ++ch) rgb[ch] += amp[((size_t)l * 3 + ch) * N + n] * o[0];
            }
            col[0] = rgb[0]; col[1] = rgb[1]; col[2] = rgb[2];
        }
    }
    return 0;
}

int asg_ref_bwd(int64_t N, int K, int C, const double *means, const double *quat, const double *shp, const double *amp,
                const double *dc, const double *campos, const uint8_t *vis, const double *g_colors,
                double *g_means, double *g_quat, double *g_shp, double *g_amp, double *g_dc)
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
            double qh[4], qn, X[3], Y[3], Z[3];
            asg_frame(quat + ((size_t)l * N + n) * 4, qh, &qn, X, Y, Z);
            const double *sp = shp + ((size_t)l * N + n) * 2;
            double w[3] = { amp[((size_t)l * 3 + 0) * N + n], amp[((size_t)l * 3 + 1) * N + n], amp[((size_t)l * 3 + 2) * N + n] };
            double gX[3] = { 0, 0, 0 }, gY[3] = { 0, 0, 0 }, gZ[3] = { 0, 0, 0 }, gw[3] = { 0, 0, 0 }, gs[2] = { 0, 0 };
            for (int c = 0; c < C; ++c) {
                if (vis && !vis[(size_t)c * N + n]) continue;
                const double *gcol = g_colors + ((size_t)c * N + n) * 3;
                double dx = means[3 * n] - campos[3 * c], dy = means[3 * n + 1] - campos[3 * c + 1], dz = means[3 * n + 2] - campos[3 * c + 2];
                double dist = sqrt(dx * dx + dy * dy + dz * dz);
                double d[3] = { dx / dist, dy / dist, dz / dist };
                double u = d[0] * X[0] + d[1] * X[1] + d[2] * X[2];
                double t = d[0] * Y[0] + d[1] * Y[1] + d[2] * Y[2];
                double v = d[0] * Z[0] + d[1] * Z[1] + d[2] * Z[2], o[6];
                asg_ref_lobe(u, t, v, sp[0], sp[1], o);
                double gG = gcol[0] * w[0] + gcol[1] * w[1] + gcol[2] * w[2];      /* dL/dG, eq.(6) */
                for (int ch = 0; ch < 3; ++ch) gw[ch] += gcol[ch] * o[0];
                gs[0] += gG * o[4]; gs[1] += gG * o[5];
                double gd[3];
                for (int i = 0; i < 3; ++i) {
                    gX[i] += gG * o[1] * d[i];          /* u = d.x */
                    gY[i] += gG * o[2] * d[i];          /* t = d.y */
                    gZ[i] += gG * o[3] * d[i];          /* v = d.z */
                    gd[i] = gG * (o[1] * X[i] + o[2] * Y[i] + o[3] * Z[i]);
                }
                double dg = d[0] * gd[0] + d[1] * gd[1] + d[2] * gd[2];
                for (int i = 0; i < 3; ++i) gm[i] += (gd[i] - d[i] * dg) / dist;    /* d = Delta/|Delta| */
            }
            if (g_amp) for (int ch = 0; ch < 3; ++ch) g_amp[((size_t)l * 3 + ch) * N + n] = gw[ch];
            if (g_shp) { g_shp[((size_t)l * N + n) * 2] = gs[0]; g_shp[((size_t)l * N + n) * 2 + 1] = gs[1]; }
            if (g_quat) {
                double qw = qh[0], qx = qh[1], qy = qh[2], qz = qh[3], gq[4];
                /* transpose Jacobian of the three columns of R(qhat) (the entries written out in asg_frame) */
                gq[0] = 2.0 * (qz * gX[1] - qy * gX[2] - qz * gY[0] + qx * gY[2] + qy * gZ[0] - qx * gZ[1]);
                gq[1] = 2.0 * (qy * gX[1] + qz * gX[2] + qy * gY[0] + qw * gY[2] + qz * gZ[0] - qw * gZ[1]) - 4.0 * qx * (gY[1] + gZ[2]);
                gq[2] = 2.0 * (qx * gX[1] - qw * gX[2] + qx * gY[0] + qz * gY[2] + qw * gZ[0] + qz * gZ[1]) - 4.0 * qy * (gX[0] + gZ[2]);
                gq[3] = 2.0 * (qw * gX[1] + qx * gX[2] - qw * gY[0] + qy * gY[2] + qx * gZ[0] + qy * gZ[1]) - 4.0 * qz * (gX[0] + gY[1]);
                /* qhat = q/|q|: dqhat/dq = (I - qhat qhat^T)/|q| */
                double dot = qh[0] * gq[0] + qh[1] * gq[1] + qh[2] * gq[2] + qh[3] * gq[3];
                double *o4 = g_quat + ((size_t)l * N + n) * 4;
                for (int i = 0; i < 4; ++i) o4[i] = (gq[i] - qh[i] * dot) / qn;
            }
        }
        if (g_means) { g_means[3 * n] = gm[0]; g_means[3 * n + 1] = gm[1]; g_means[3 * n + 2] = gm[2]; }
        if (g_dc) { g_dc[n] = gdc[0]; g_dc[N + n] = gdc[1]; g_dc[2 * N + n] = gdc[2]; }
    }
    return 0;
}
