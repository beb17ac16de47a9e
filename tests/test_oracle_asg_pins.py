"""Pins of the oracle's Anisotropic Spherical Gaussian (oracle/asg_ref.c; Table 6,
PAPER.md:424) against what the paper and the mathematics fix (CPU only): the frame against a library rotation, closed
forms of the sphere integral, the pairing of (mu, x) and (lambda, y) the table prints, symmetries and finite differences.
Nothing here compares with the CUDA path."""
import numpy as np
import pytest
from scipy.spatial.transform import Rotation


def _case(N=5, K=2, C=2, seed=0, vis=True):
    r = np.random.default_rng(seed)
    return dict(N=N, K=K, C=C, means=r.uniform(-1, 1, (N, 3)), quat=r.normal(0, 1, (K, N, 4)),
                shp=r.uniform(-1.0, 3.0, (K, N, 2)), amp=r.normal(0, 0.5, (K, 3, N)), dc=r.normal(0, 0.3, (3, N)),
                campos=4.0 * np.array([[0.3, -0.5, 0.81], [-0.6, 0.64, 0.48]])[:C],
                vis=(r.random((C, N)) < 0.7).astype(np.uint8) if vis else None, g_colors=r.normal(0, 1, (C, N, 3)))


def _one_lobe(q, raw_mu, raw_lam, dirs):
    """Inputs that evaluate ONE unit-amplitude lobe at the unit directions `dirs` [N,3] (camera at the origin)."""
    N = len(dirs)
    return dict(N=N, K=1, C=1, means=np.asarray(dirs, dtype=np.float64), quat=np.tile(np.asarray(q, dtype=np.float64), (1, N, 1)),
                shp=np.tile(np.array([raw_mu, raw_lam]), (1, N, 1)), amp=np.ones((1, 3, N)), dc=np.zeros((3, N)),
                campos=np.zeros((1, 3)), vis=None)


def _sphere_integral(oracle, q, raw_mu, raw_lam, n=96):
    """int G dOmega by a Gauss-Legendre product rule in polar coordinates about the lobe's z axis (columns from the
    library rotation), the polar angle split at the equator where the lobe has its kink; one asg_fwd call."""
    R = Rotation.from_quat([q[1], q[2], q[3], q[0]]).as_matrix()
    x, w = np.polynomial.legendre.leggauss(n)
    total = 0.0
    for lo, hi in ((0.0, np.pi / 2), (np.pi / 2, np.pi)):
        th = 0.5 * (hi - lo) * x + 0.5 * (hi + lo); wt = 0.5 * (hi - lo) * w
        ph = np.pi * x + np.pi; wp = np.pi * w
        T, P = np.meshgrid(th, ph, indexing="ij")
        local = np.stack([np.sin(T) * np.cos(P), np.sin(T) * np.sin(P), np.cos(T)], axis=-1).reshape(-1, 3)
        G = oracle.asg_fwd(_one_lobe(q, raw_mu, raw_lam, local @ R.T))[0, :, 0].reshape(n, n)
        total += float((G * np.sin(T) * wt[:, None] * wp[None, :]).sum())
    return total


@pytest.mark.parametrize("q", [(1.0, 0.0, 0.0, 0.0), (0.3, -0.5, 0.2, 0.7), (-2.0, 0.4, 0.1, -0.3)])
def test_frame_is_the_library_rotation_matrix(oracle, q):
    """[x y z] = R(q/|q|), Hamilton (w,x,y,z), against scipy (which takes (x,y,z,w)); right-handed and orthonormal.
    Catches a transposed matrix, a swapped column, a sign error in any entry."""
    X, Y, Z = oracle.asg_frame(q)
    R = Rotation.from_quat([q[1], q[2], q[3], q[0]]).as_matrix()
    assert np.abs(np.stack([X, Y, Z], axis=1) - R).max() < 1e-14
    assert np.abs(np.cross(X, Y) - Z).max() < 1e-14


def test_sphere_integral_closed_form_for_equal_bandwidths(oracle):
    """mu = lambda: (d.x)^2 + (d.y)^2 = 1 - (d.z)^2, so int G = 2 pi int_0^1 v e^{-mu (1 - v^2)} dv = pi (1 - e^{-mu})/mu;
    mu -> 0 gives the clamped cosine lobe, integral pi. Catches a missing max(.,0), a wrong sign or factor in the exponent."""
    q = (0.3, -0.5, 0.2, 0.7)
    for mu in (1e-9, 0.5, 3.0, 20.0):
        want = np.pi * (-np.expm1(-mu)) / mu
        got = _sphere_integral(oracle, q, np.log(mu), np.log(mu))
        assert abs(got / want - 1.0) < 1e-10, (mu, got, want)


def test_sphere_integral_large_bandwidth_limit(oracle):
    """[XSD*13]: for large bandwidths int G -> pi / sqrt(mu lambda) (the Gaussian integral over the tangent plane); the
    relative correction is O(1/mu + 1/lambda). Catches a dropped term (one bandwidth ignored) or a missing square."""
    for mu, lam in ((400.0, 100.0), (150.0, 600.0)):
        got = _sphere_integral(oracle, (0.9, 0.1, -0.3, 0.2), np.log(mu), np.log(lam))
        assert abs(got * np.sqrt(mu * lam) / np.pi - 1.0) < 2.0 * (1.0 / mu + 1.0 / lam), (mu, lam, got)


def test_mu_goes_with_x_and_lambda_with_y(oracle):
    """Table 6: exp{-mu (d.x)^2 - lambda (d.y)^2}. On the great circle through z and x the lobe is cos(al) e^{-mu sin^2 al},
    through z and y it is cos(al) e^{-lambda sin^2 al}; the frame columns come from the library rotation."""
    q = np.array([0.3, -0.5, 0.2, 0.7])
    R = Rotation.from_quat([q[1], q[2], q[3], q[0]]).as_matrix()
    mu, lam = 7.0, 0.8
    al = np.array([-1.2, -0.4, 0.0, 0.3, 1.0])
    for axis, bw in ((0, mu), (1, lam)):
        dirs = np.cos(al)[:, None] * R[:, 2][None, :] + np.sin(al)[:, None] * R[:, axis][None, :]
        got = oracle.asg_fwd(_one_lobe(q, np.log(mu), np.log(lam), dirs))[0, :, 0]
        assert np.abs(got - np.cos(al) * np.exp(-bw * np.sin(al) ** 2)).max() < 1e-14


def test_far_hemisphere_is_zero_with_zero_gradient(oracle):
    q = np.array([1.0, 0.0, 0.0, 0.0])
    dirs = np.array([[0.6, 0.0, -0.8], [0.0, 1.0, 0.0], [0.0, -0.6, -0.8]])       # d.z < 0, = 0, < 0
    inp = _one_lobe(q, 0.3, 1.1, dirs)
    assert (oracle.asg_fwd(inp) == 0).all()
    g = oracle.asg_bwd(dict(inp, g_colors=np.ones((1, 3, 3))))
    assert (g["g_quat"] == 0).all() and (g["g_shp"] == 0).all() and (g["g_means"] == 0).all() and (g["g_amp"] == 0).all()


def test_quarter_turn_about_z_swaps_the_bandwidths(oracle):
    """Rotating the frame by 90 degrees about its own z axis maps x -> y, y -> -x: the same lobe with mu and lambda swapped."""
    inp = _case(N=30, K=2, C=2, seed=4, vis=False)
    rz = np.array([np.cos(np.pi / 4), 0.0, 0.0, np.sin(np.pi / 4)])             # (w,x,y,z): 90 degrees about e3, applied on the right
    q = inp["quat"]
    w1, x1, y1, z1 = (q[..., i] for i in range(4))
    w2, x2, y2, z2 = rz
    qr = np.stack([w1 * w2 - x1 * x2 - y1 * y2 - z1 * z2, w1 * x2 + x1 * w2 + y1 * z2 - z1 * y2,
                   w1 * y2 - x1 * z2 + y1 * w2 + z1 * x2, w1 * z2 + x1 * y2 - y1 * x2 + z1 * w2], axis=-1)
    a, b = oracle.asg_fwd(inp), oracle.asg_fwd(dict(inp, quat=qr, shp=inp["shp"][..., ::-1].copy()))
    assert np.abs(a - b).max() < 1e-13 * np.abs(a).max()


def test_rotating_the_scene_rotates_the_gradients(oracle):
    """A rigid rotation of means, cameras and frames (q -> r q) leaves the colours unchanged and rotates g_means."""
    inp = _case(N=25, K=3, C=2, seed=8)
    rot = Rotation.from_rotvec([0.4, -0.9, 0.5])
    r = rot.as_quat()[[3, 0, 1, 2]]
    q = inp["quat"]
    w1, x1, y1, z1 = r
    w2, x2, y2, z2 = (q[..., i] for i in range(4))
    rq = np.stack([w1 * w2 - x1 * x2 - y1 * y2 - z1 * z2, w1 * x2 + x1 * w2 + y1 * z2 - z1 * y2,
                   w1 * y2 - x1 * z2 + y1 * w2 + z1 * x2, w1 * z2 + x1 * y2 - y1 * x2 + z1 * w2], axis=-1)
    inp2 = dict(inp, means=rot.apply(inp["means"]), campos=rot.apply(inp["campos"]), quat=rq)
    a, b = oracle.asg_fwd(inp), oracle.asg_fwd(inp2)
    assert np.abs(a - b).max() < 1e-13 * np.abs(a).max()
    ga, gb = oracle.asg_bwd(inp), oracle.asg_bwd(inp2)
    assert np.abs(rot.apply(ga["g_means"]) - gb["g_means"]).max() < 1e-12 * np.abs(ga["g_means"]).max()
    for k in ("g_shp", "g_amp", "g_dc"):
        assert np.abs(ga[k] - gb[k]).max() < 1e-12 * np.abs(ga[k]).max(), k


def test_lobe_partials_by_differences(oracle):
    for (u, t, v) in ((0.3, -0.2, 0.93), (-0.6, 0.5, 0.62), (0.1, 0.9, 0.42)):
        for rm, rl in ((-0.5, 1.0), (2.0, 0.3)):
            o = oracle.asg_lobe(u, t, v, rm, rl)
            h = 1e-6
            num = [(oracle.asg_lobe(u + h, t, v, rm, rl)[0] - oracle.asg_lobe(u - h, t, v, rm, rl)[0]) / (2 * h),
                   (oracle.asg_lobe(u, t + h, v, rm, rl)[0] - oracle.asg_lobe(u, t - h, v, rm, rl)[0]) / (2 * h),
                   (oracle.asg_lobe(u, t, v + h, rm, rl)[0] - oracle.asg_lobe(u, t, v - h, rm, rl)[0]) / (2 * h),
                   (oracle.asg_lobe(u, t, v, rm + h, rl)[0] - oracle.asg_lobe(u, t, v, rm - h, rl)[0]) / (2 * h),
                   (oracle.asg_lobe(u, t, v, rm, rl + h)[0] - oracle.asg_lobe(u, t, v, rm, rl - h)[0]) / (2 * h)]
            assert np.abs(np.array(num) - o[1:]).max() < 1e-8 * max(1.0, np.abs(o[1:]).max())


def test_finite_differences_of_every_input(oracle):
    """Central differences of sum(g_colors * colours) with respect to means, quat (through the normalisation), shp, amp, dc
    against asg_ref_bwd. The quaternions are NOT unit: a missing (I - qhat qhat^T)/|q| fails. Directions are kept away
    from the kink at d.z = 0 by the seed (checked)."""
    inp = _case(N=4, K=2, C=2, seed=12)
    g = oracle.asg_bwd(inp)
    for l in range(2):
        for n in range(4):
            _, _, Z = oracle.asg_frame(inp["quat"][l, n])
            for c in range(2):
                d = inp["means"][n] - inp["campos"][c]
                assert abs(d @ Z) / np.linalg.norm(d) > 1e-3
    L = lambda d: float((oracle.asg_fwd(d) * inp["g_colors"]).sum())
    for key, gkey in (("quat", "g_quat"), ("shp", "g_shp"), ("amp", "g_amp"), ("dc", "g_dc"), ("means", "g_means")):
        base = inp[key]
        num = np.empty_like(base)
        it = np.nditer(base, flags=["multi_index"])
        for _ in it:
            i = it.multi_index
            h = 1e-6 * max(1.0, abs(base[i]))
            p, m = base.copy(), base.copy()
            p[i] += h; m[i] -= h
            num[i] = (L(dict(inp, **{key: p})) - L(dict(inp, **{key: m}))) / (2 * h)
        scale = np.abs(g[gkey]).max()
        assert np.abs(num - g[gkey]).max() < 2e-7 * scale, (key, np.abs(num - g[gkey]).max() / scale)
    # the gradient of a quaternion is orthogonal to it (the frame does not depend on |q|)
    assert np.abs((g["g_quat"] * inp["quat"]).sum(-1)).max() < 1e-12 * np.abs(g["g_quat"]).max()


def test_culled_pairs(oracle):
    inp = _case(N=6, K=2, C=2, seed=5)
    inp["vis"][:, 2] = 0
    inp["vis"][0, 3] = 0; inp["vis"][1, 3] = 1
    col, g = oracle.asg_fwd(inp), oracle.asg_bwd(inp)
    assert (col[:, 2] == 0).all() and (col[0, 3] == 0).all()
    assert (g["g_quat"][:, 2] == 0).all() and (g["g_means"][2] == 0).all() and (g["g_dc"][:, 2] == 0).all()
    only = oracle.asg_bwd(dict(inp, C=1, campos=inp["campos"][1:], vis=inp["vis"][1:], g_colors=inp["g_colors"][1:]))
    assert np.abs(only["g_quat"][:, 3] - g["g_quat"][:, 3]).max() == 0.0      # the culled camera contributes nothing
