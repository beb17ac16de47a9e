"""Pins of the oracle's isotropic Table-6 functions (oracle/iso_ref.c)
against what the paper and the mathematics fix (CPU only): the normalisation constants of Table 6 by quadrature, library
densities, the reduction of NASG to SG at a = 0, k = 0, and finite differences."""
import numpy as np
import pytest
import scipy.integrate
import scipy.stats

SG, SB, SC = 0, 1, 2


def _sphere_integral(f):
    """2 pi int_{-1}^{1} f(v) dv for a function of v = z.d only."""
    val, _ = scipy.integrate.quad(f, -1.0, 1.0, epsabs=1e-13, epsrel=1e-13, limit=400, points=[0.0])
    return 2.0 * np.pi * val


@pytest.mark.parametrize("kind,raws", [(SG, (-1.0, 0.0, 1.5, 3.0, 5.0)), (SB, (-1.0, 0.0, 1.5, 3.0, 5.0)), (SC, (-3.0, -0.5, 0.0, 1.0, 2.5))])
def test_table6_normalisation_constants_by_quadrature(oracle, kind, raws):
    """c G integrates to 1 over the sphere: c = lambda/(2 pi (1-e^{-2 lambda})), (beta+1)/(2 pi), 1/(4 pi) (Table 6).
    Catches a wrong constant, a missing hemisphere cut-off in SB, the wrong Cauchy denominator."""
    for raw in raws:
        assert abs(_sphere_integral(lambda v: oracle.iso_lobe(kind, v, raw)[0]) - 1.0) < 1e-9, (kind, raw)


def test_cauchy_denominator_as_printed_is_not_normalised():
    """Reading R19: Table 6 prints (1 - rho^2)/(1 - rho^2 - 2 rho z.d); with c = 1/(4 pi) that does not integrate to 1
    (it even has a pole for rho > sqrt(2) - 1), whereas 1 + rho^2 - 2 rho z.d does (the standard spherical Cauchy)."""
    rho = 0.3
    printed = lambda v: ((1 - rho ** 2) / (1 - rho ** 2 - 2 * rho * v)) ** 2 / (4 * np.pi)
    assert abs(_sphere_integral(printed) - 1.0) > 0.2


def test_sg_is_the_von_mises_fisher_density_and_nasg_at_zero_anisotropy(oracle):
    """SG x c = vMF pdf (scipy), and equals the NASGabor oracle at a = 0, k = 0 (pinned P4)."""
    z = np.array([0.0, 0.0, 1.0])
    for raw in (0.0, 1.0, 3.0):
        lam = np.exp(raw)
        for v in (-0.7, 0.1, 0.95):
            d = np.array([np.sqrt(1 - v * v), 0.0, v])
            want = scipy.stats.vonmises_fisher(z, lam).pdf(d)
            got = oracle.iso_lobe(SG, v, raw)[0]
            assert abs(got / want - 1.0) < 1e-12
            # NASG with a = 0: exp(2 lambda kappa - 2 lambda) = exp(lambda (v - 1))  (kappa = (1+v)/2)
            nasg = oracle.partials(d[0], v, lam, 0.0, 0.0, 0.0, 0)[0]
            assert abs(got / nasg - 1.0) < 1e-12


def test_sb_closed_form_and_hemisphere(oracle):
    for raw, v in ((0.0, 0.5), (1.0, 0.9), (2.0, 0.2)):
        beta = np.exp(raw)
        assert abs(oracle.iso_lobe(SB, v, raw)[0] / ((beta + 1) / (2 * np.pi) * v ** beta) - 1.0) < 1e-14
    assert (oracle.iso_lobe(SB, -0.3, 1.0) == 0).all() and (oracle.iso_lobe(SB, 0.0, 1.0) == 0).all()


@pytest.mark.parametrize("kind", [SG, SB, SC])
def test_lobe_partials_by_differences(oracle, kind):
    for raw in (-0.5, 0.7, 2.0):
        for v in (0.15, 0.6, 0.97):
            F, Fv, Fr = oracle.iso_lobe(kind, v, raw)
            h = 1e-6
            nv = (oracle.iso_lobe(kind, v + h, raw)[0] - oracle.iso_lobe(kind, v - h, raw)[0]) / (2 * h)
            nr = (oracle.iso_lobe(kind, v, raw + h)[0] - oracle.iso_lobe(kind, v, raw - h)[0]) / (2 * h)
            assert abs(nv - Fv) < 1e-7 * max(1.0, abs(Fv)) and abs(nr - Fr) < 1e-7 * max(1.0, abs(Fr)), (kind, raw, v)


def _case(N=4, K=2, C=2, seed=0):
    r = np.random.default_rng(seed)
    return dict(N=N, K=K, C=C, means=r.uniform(-1, 1, (N, 3)), axis=r.normal(0, 1, (K, N, 3)) * r.uniform(0.5, 2.0, (K, N, 1)),
                shp=r.uniform(-0.5, 2.5, (K, N)), amp=r.normal(0, 0.5, (K, 3, N)), dc=r.normal(0, 0.3, (3, N)),
                campos=4.0 * np.array([[0.3, -0.5, 0.81], [-0.6, 0.64, 0.48]])[:C], vis=(r.random((C, N)) < 0.7).astype(np.uint8),
                g_colors=r.normal(0, 1, (C, N, 3)))


@pytest.mark.parametrize("kind", [SG, SB, SC])
def test_eq6_mix_and_finite_differences_of_every_gradient(oracle, kind):
    """eq.(6) by brute force from iso_lobe; central differences of sum(g_colors * colours) for every input array, incl. the
    unnormalised axis (gradient through the normalisation: g_axis is orthogonal to the axis)."""
    inp = _case(seed=3 + kind)
    col = oracle.iso_fwd(inp, kind)
    for c in range(2):
        for n in range(4):
            if not inp["vis"][c, n]:
                assert (col[c, n] == 0).all()
                continue
            d = inp["means"][n] - inp["campos"][c]; d /= np.linalg.norm(d)
            want = inp["dc"][:, n].copy()
            for l in range(2):
                z = inp["axis"][l, n] / np.linalg.norm(inp["axis"][l, n])
                want += inp["amp"][l, :, n] * oracle.iso_lobe(kind, float(d @ z), inp["shp"][l, n])[0]
            assert np.abs(col[c, n] - want).max() < 1e-13
    g = oracle.iso_bwd(inp, kind)
    L = lambda x: float((oracle.iso_fwd(x, kind) * inp["g_colors"]).sum())
    for key, gkey in (("axis", "g_axis"), ("shp", "g_shp"), ("amp", "g_amp"), ("dc", "g_dc"), ("means", "g_means")):
        base = inp[key]
        num = np.empty_like(base)
        it = np.nditer(base, flags=["multi_index"])
        for _ in it:
            i = it.multi_index
            h = 1e-6 * max(1.0, abs(base[i]))
            p, m = base.copy(), base.copy()
            p[i] += h; m[i] -= h
            num[i] = (L(dict(inp, **{key: p})) - L(dict(inp, **{key: m}))) / (2 * h)
        assert np.abs(num - g[gkey]).max() < 3e-7 * max(np.abs(g[gkey]).max(), 1e-3), (key, np.abs(num - g[gkey]).max())
    assert np.abs((g["g_axis"] * inp["axis"]).sum(-1)).max() < 1e-12 * np.abs(g["g_axis"]).max()
