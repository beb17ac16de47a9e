/* ============================================================================================
 * oracle/sh_ref.c — TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Plain fp64 CPU implementation of the comparison path: real spherical harmonics of degree 3,
 * colour[c,n,:] = sum_{j<16} coeff[j,:,n] Y_j(d), d = normalize(mean - campos_c)
 * (eq.(5); 48 parameters per primitive), forward and analytic
 * backward. The paper gives only eq.(5); the basis convention is reading R15 of DESIGN.md: real
 * orthonormal SH, index j = l^2 + l + m, Condon-Shortley sign (-1)^{|m|} retained, written out
 * below as polynomials in the components of the unit vector d. The constants are spelled as
 * sqrt() expressions so they can be checked by eye; tests pin the basis against
 * scipy.special.sph_harm_y, the Gram matrix by quadrature, and the addition theorem.
 *
 * Same rules as nasg_ref.c: only tests/, smoke() and bench.py's CPU legs call this; no code is
 * shared with the CUDA path. Arrays are fp64 host arrays:
 *   means [N,3] coeffs [16,3,N] campos [C,3] vis [C,N] uint8 or NULL colors/g_colors [C,N,3]
 * ============================================================================================ */
#include <math.h>
#include <stddef.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#define PI 3.14159265358979323846264338327950288

/* Y[16] and the R^3 polynomial gradient dY[16][3] at the unit vector (x,y,z). */
static void sh_basis(double x, double y, double z, double Y[16], double dY[16][3])
{
    const double c0 = 0.5 * sqrt(1.0 / PI);
    const double c1 = sqrt(3.0 / (4.0 * PI));
    const double c2a = 0.5 * sqrt(15.0 / PI), c2b = 0.25 * sqrt(5.0 / PI), c2c = 0.25 * sqrt(15.0 / PI);
    const double c3a = 0.25 * sqrt(35.0 / (2.0 * PI)), c3b = 0.5 * sqrt(105.0 / PI),
                 c3c = 0.25 * sqrt(21.0 / (2.0 * PI)), c3d = 0.25 * sqrt(7.0 / PI),
                 c3e = 0.25 * sqrt(105.0 / PI);
    double xx = x * x, yy = y * y, zz = z * z;
#define SET(j, val, gx, gy, gz) do { Y[j] = (val); dY[j][0] = (gx); dY[j][1] = (gy); dY[j][2] = (gz); } while (0)
    SET(0, c0, 0.0, 0.0, 0.0);
    SET(1, -c1 * y, 0.0, -c1, 0.0);
    SET(2, c1 * z, 0.0, 0.0, c1);
    SET(3, -c1 * x, -c1, 0.0, 0.0);
    SET(4, c2a * x * y, c2a * y, c2a * x, 0.0);
    SET(5, -c2a * y * z, 0.0, -c2a * z, -c2a * y);
    SET(6, c2b * (2.0 * zz - xx - yy), -2.0 * c2b * x, -2.0 * c2b * y, 4.0 * c2b * z);
    SET(7, -c2a * x * z, -c2a * z, 0.0, -c2a * x);
    SET(8, c2c * (xx - yy), 2.0 * c2c * x, -2.0 * c2c * y, 0.0);
    SET(9, -c3a * y * (3.0 * xx - yy), -c3a * 6.0 * x * y, -c3a * (3.0 * xx - 3.0 * yy), 0.0);
    SET(10, c3b * x * y * z, c3b * y * z, c3b * x * z, c3b * x * y);
    SET(11, -c3c * y * (4.0 * zz - xx - yy), c3c * 2.0 * x * y, -c3c * (4.0 * zz - xx - 3.0 * yy),
        -c3c * 8.0 * y * z);
    SET(12, c3d * z * (2.0 * zz - 3.0 * xx - 3.0 * yy), -c3d * 6.0 * x * z, -c3d * 6.0 * y * z,
        c3d * (6.0 * zz - 3.0 * xx - 3.0 * yy));
    SET(13, -c3c * x * (4.0 * zz - xx - yy), -c3c * (4.0 * zz - 3.0 * xx - yy), c3c * 2.0 * x * y,
        -c3c * 8.0 * x * z);
    SET(14, c3e * z * (xx - yy), c3e * 2.0 * x * z, -c3e * 2.0 * y * z, c3e * (xx - yy));
    SET(15, -c3a * x * (xx - 3.0 * yy), -c3a * (3.0 * xx - 3.0 * yy), c3a * 6.0 * x * y, 0.0);
#undef SET
}

void sh_ref_basis(const double d[3], double Y[16], double dY[48])
{
    double g[16][3];
    sh_basis(d[0], d[1], d[2], Y, g);
    memcpy(dY, g, sizeof(g));
}

int sh_ref_fwd(int64_t N, int C, const double *means, const double *coeffs, const double *campos,
               const uint8_t *vis, double *colors)
{
#pragma omp parallel for schedule(static)
    for (int64_t n = 0; n < N; ++n) {
        for (int c = 0; c < C; ++c) {
            double *col = colors + ((size_t)c * N + n) * 3;
            if (vis && !vis[(size_t)c * N + n]) { col[0] = col[1] = col[2] = 0.0; continue; }
            double dx = means[3 * n] - campos[3 * c], dy = means[3 * n + 1] - campos[3 * c + 1],
                   dz = means[3 * n + 2] - campos[3 * c + 2];
            double dist = sqrt(dx * dx + dy * dy + dz * dz);
            double Y[16], dY[16][3];
            sh_basis(dx / dist, dy / dist, dz / dist, Y, dY);
            double rgb[3] = { 0, 0, 0 };
            for (int j = 0; j < 16; ++j)
                for (int ch = 0; ch < 3; ++ch) rgb[ch] += coeffs[((size_t)j * 3 + ch) * N + n] * Y[j];
            col[0] = rgb[0]; col[1] = rgb[1]; col[2] = rgb[2];
        }
    }
    return 0;
}

int sh_ref_bwd(int64_t N, int C, const double *means, const double *coeffs, const double *campos,
               const uint8_t *vis, const double *g_colors, double *g_means, double *g_coeffs,
               double *g_campos)
{
    if (g_campos) memset(g_campos, 0, sizeof(double) * 3 * (size_t)C);
#pragma omp parallel
    {
        double *gc_local = (double *)calloc((size_t)3 * C, sizeof(double));
#pragma omp for schedule(static)
        for (int64_t n = 0; n < N; ++n) {
            double gm[3] = { 0, 0, 0 };
            double gco[16][3];
            memset(gco, 0, sizeof(gco));
            for (int c = 0; c < C; ++c) {
                if (vis && !vis[(size_t)c * N + n]) continue;
                const double *gcol = g_colors + ((size_t)c * N + n) * 3;
                double dx = means[3 * n] - campos[3 * c], dy = means[3 * n + 1] - campos[3 * c + 1],
                       dz = means[3 * n + 2] - campos[3 * c + 2];
                double dist = sqrt(dx * dx + dy * dy + dz * dz);
                double d[3] = { dx / dist, dy / dist, dz / dist };
                double Y[16], dY[16][3];
                sh_basis(d[0], d[1], d[2], Y, dY);
                double gd[3] = { 0, 0, 0 };
                for (int j = 0; j < 16; ++j) {
                    double s = 0.0; /* coeff_j . g_col */
                    for (int ch = 0; ch < 3; ++ch) {
                        gco[j][ch] += gcol[ch] * Y[j];
                        s += coeffs[((size_t)j * 3 + ch) * N + n] * gcol[ch];
                    }
                    for (int i = 0; i < 3; ++i) gd[i] += s * dY[j][i];
                }
                double dg = d[0] * gd[0] + d[1] * gd[1] + d[2] * gd[2];
                for (int i = 0; i < 3; ++i) {
                    double t = (gd[i] - d[i] * dg) / dist; /* (I - d d^T)/|Delta| */
                    gm[i] += t;
                    gc_local[3 * c + i] -= t;
                }
            }
            if (g_means) { g_means[3 * n] = gm[0]; g_means[3 * n + 1] = gm[1]; g_means[3 * n + 2] = gm[2]; }
            if (g_coeffs)
                for (int j = 0; j < 16; ++j)
                    for (int ch = 0; ch < 3; ++ch) g_coeffs[((size_t)j * 3 + ch) * N + n] = gco[j][ch];
        }
        if (g_campos) {
#pragma omp critical
            for (int i = 0; i < 3 * C; ++i) g_campos[i] += gc_local[i];
        }
        free(gc_local);
    }
    return 0;
}
