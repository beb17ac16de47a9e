"""Spherical quadrature of the ORACLE's forward function (test helper, no method arithmetic).

The lobe frame is the identity quaternion (x = e1, z = e3); directions d(theta, phi) are fed to
``oracle.ref.nasg_fwd`` as Gaussians at mean = 2 d seen from campos = 0, with amp = (1,0,0), dc = 0,
so colour[...,0] is the normalised lobe value G(d). Polar variable: kappa = (1+cos theta)/2 = t^4,
Gauss-Legendre in t (the t^3 Jacobian removes the kappa^tau end-point singularity at d = -z);
azimuth: periodic trapezoid (spectrally accurate for a periodic analytic integrand).
"""
import numpy as np


def sphere_integral_of_G(ref, lam, a, k, phi, norm_mode, nt=1400, nphi=1536):
    """Integral over S^2 of the oracle's normalised lobe (== 1 if the normaliser is exact)."""
    x, w = np.polynomial.legendre.leggauss(nt)
    t = 0.5 * (x + 1.0)
    wt = 0.5 * w
    kappa = t ** 4
    v = 2.0 * kappa - 1.0                       # cos(theta)
    jac = 2.0 * 4.0 * t ** 3                    # dv = 2 dkappa = 8 t^3 dt
    s = np.sqrt(np.maximum(0.0, 1.0 - v * v))
    az = (np.arange(nphi) + 0.5) * (2.0 * np.pi / nphi)
    d = np.stack([np.outer(s, np.cos(az)), np.outer(s, np.sin(az)),
                  np.repeat(v[:, None], nphi, 1)], axis=-1).reshape(-1, 3)
    N = d.shape[0]
    inp = dict(N=N, K=1, C=1, means=2.0 * d, campos=np.zeros((1, 3)),
               quat=np.tile(np.array([1.0, 0, 0, 0]), (1, N, 1)),
               shape=np.tile(np.array([np.log(lam * (1.0 + a)), np.log(lam), k, phi]), (1, N, 1)),
               amp=np.concatenate([np.ones((1, 1, N)), np.zeros((1, 2, N))], axis=1),
               dc=np.zeros((3, N)), vis=None)
    G = ref.nasg_fwd(inp, norm_mode)[0, :, 0].reshape(nt, nphi)
    return float(((G.sum(axis=1) * (2.0 * np.pi / nphi)) * wt * jac).sum())
