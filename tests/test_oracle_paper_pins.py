"""Pins of the oracle's paper-native record functions (oracle/nasg_ref.c: nasg_ref_paper_*; SURVEY.md section 8(f)
NEXT-2) against what the paper and the mathematics fix (CPU only). Nothing here compares with the CUDA path.

The record: 3 + 9 K appearance floats per primitive (Table 5), Table 8 activations
(PAPER.md:483-491), Supplementary C frame, eqs.(37)-(44) chain rule."""
import numpy as np
import pytest
from scipy.spatial.transform import Rotation


def _case(N=5, K=2, C=2, seed=0, vis=True):
    r = np.random.default_rng(seed)
    return dict(N=N, K=K, C=C, means=r.uniform(-1, 1, (N, 3)), euler=r.uniform(-1.5, 1.5, (K, N, 3)),
                shp=np.stack([r.uniform(0, 3, (K, N)), r.uniform(-1, 2, (K, N)), r.uniform(-2, -0.3, (K, N))], axis=2),
                ampraw=r.normal(0, 0.5, (K, 3, N)), dc=r.normal(0, 0.3, (3, N)),
                campos=4.0 * np.array([[0.3, -0.5, 0.81], [-0.6, 0.64, 0.48]])[:C],
                vis=(r.random((C, N)) < 0.7).astype(np.uint8) if vis else None, g_colors=r.normal(0, 1, (C, N, 3)))


def test_parameter_count_is_3_plus_9K():
    """PAPER.md:258-260, Table 5: 12 / 21 / 39 appearance floats for K = 1 / 2 / 4."""
    from paper_2606_09794_b200 import workloads as W
    for K, want in ((1, 12), (2, 21), (4, 39)):
        assert 3 + 9 * K == want
    inp = W.make_paper(W.CONFIGS[2], 64)
    per_gaussian = sum(inp[k].size for k in ("euler", "shp", "ampraw", "dc")) // 64
    assert per_gaussian == 39 and W.paper_rec_floats(64, 4) == 64 * (3 + 39)


@pytest.mark.parametrize("raw", [(0.3, -0.2, 0.5), (-1.2, 0.9, -0.4), (0.0, 0.0, 0.0), (1.7, -1.7, 1.1)])
def test_frame_is_the_ZYZ_euler_rotation_with_nonnegative_sines(oracle, raw):
    """Supplementary C: x and z are columns 0 and 2 of Rz(theta) Ry(phi) Rz(tau) with
    cos = tanh(raw), sin = +sqrt(1 - cos^2) (angles in [0, pi]); orthonormal; y = z cross x completes a right-handed
    frame. Catches a transposed frame, a wrong sign in x, swapped angles."""
    X, Z, _, _ = oracle.paper_frame(raw)
    ang = np.arccos(np.tanh(np.asarray(raw, dtype=np.float64)))         # in [0, pi]: the sines are non-negative
    R = Rotation.from_euler("ZYZ", ang).as_matrix()
    assert np.abs(X - R[:, 0]).max() < 1e-14 and np.abs(Z - R[:, 2]).max() < 1e-14
    assert abs(X @ X - 1) < 1e-14 and abs(Z @ Z - 1) < 1e-14 and abs(X @ Z) < 1e-14
    assert np.abs(np.cross(Z, X) - R[:, 1]).max() < 1e-14
    assert Z[1] >= 0.0      # the quirk SURVEY.md notes: z is confined to the y >= 0 half-space


def test_frame_derivatives_eqs_38_to_44(oracle):
    """dX/dc, dZ/dc of eqs.(38), (39: as corrected in R6(iii)), (41), (42), (44) against numerical differentiation of
    Supplementary C's frame with respect to the COSINES (mpmath-free: central differences in fp64 on c directly)."""
    def frame_of_c(c):
        s = np.sqrt(1 - c * c)
        z = np.array([c[0] * s[1], s[0] * s[1], c[1]])
        x = np.array([c[0] * c[1] * c[2] - s[0] * s[2], s[0] * c[1] * c[2] + c[0] * s[2], -s[1] * c[2]])
        return x, z
    for raw in ((0.3, -0.2, 0.5), (-1.0, 0.8, -0.6)):
        raw = np.asarray(raw, dtype=np.float64)
        c = np.tanh(raw)
        _, _, dX, dZ = oracle.paper_frame(raw)
        for i in range(3):
            h = 1e-6
            cp, cm = c.copy(), c.copy()
            cp[i] += h; cm[i] -= h
            xp, zp = frame_of_c(cp); xm, zm = frame_of_c(cm)
            assert np.abs((xp - xm) / (2 * h) - dX[i]).max() < 1e-8, ("dX", i)
            assert np.abs((zp - zm) / (2 * h) - dZ[i]).max() < 1e-8, ("dZ", i)


@pytest.mark.parametrize("mode", [0, 1])
def test_equals_the_quaternion_oracle_on_the_equivalent_parameters(oracle, mode):
    """The paper record is a re-parameterisation: with q = quaternion of Rz Ry Rz, (log Lambda, log lambda) =
    (raw_lambda + log(1 + e^{raw_a}), raw_lambda), k = 20 (tanh + 1), phi = 0, w = tanh(raw) the quaternion oracle
    (pinned by test_oracle_pins.py) gives the same colours, and the same gradients for the shared inputs (means, dc)."""
    inp = _case(N=40, K=3, C=2, seed=3)
    ang = np.arccos(np.tanh(inp["euler"]))
    quat = Rotation.from_euler("ZYZ", ang.reshape(-1, 3)).as_quat().reshape(3, 40, 4)[..., [3, 0, 1, 2]]   # (w,x,y,z)
    lam, a = np.exp(inp["shp"][..., 0]), np.exp(inp["shp"][..., 1])
    shape = np.stack([np.log(lam * (1 + a)), np.log(lam), 20 * (np.tanh(inp["shp"][..., 2]) + 1), np.zeros_like(lam)], axis=2)
    eq = dict(inp, quat=quat, shape=shape, amp=np.tanh(inp["ampraw"]))
    a_col, b_col = oracle.paper_fwd(inp, mode), oracle.nasg_fwd(eq, mode)
    assert np.abs(a_col - b_col).max() < 1e-12 * np.abs(b_col).max()
    ga, gb = oracle.paper_bwd(inp, mode), oracle.nasg_bwd(eq, mode)
    for k in ("g_means", "g_dc"):
        assert np.abs(ga[k] - gb[k]).max() < 1e-11 * np.abs(gb[k]).max(), k
    # chain rule of the activations the two share: w = tanh(raw), k = 20 (tanh + 1), lambda / a = exp
    assert np.abs(ga["g_ampraw"] - gb["g_amp"] * (1 - np.tanh(inp["ampraw"]) ** 2)).max() < 1e-11 * np.abs(gb["g_amp"]).max()
    g_k = gb["g_shape"][..., 2] * 20 * (1 - np.tanh(inp["shp"][..., 2]) ** 2)
    assert np.abs(ga["g_shp"][..., 2] - g_k).max() < 1e-11 * np.abs(g_k).max()
    g_lam = gb["g_shape"][..., 0] + gb["g_shape"][..., 1]                        # d/dlog lambda at fixed a
    g_a = gb["g_shape"][..., 0] * a / (1 + a)                                   # d/dlog a
    assert np.abs(ga["g_shp"][..., 0] - g_lam).max() < 1e-10 * np.abs(g_lam).max()
    assert np.abs(ga["g_shp"][..., 1] - g_a).max() < 1e-10 * np.abs(g_a).max()


@pytest.mark.parametrize("mode", [0, 1])
def test_finite_differences_through_the_activations(oracle, mode):
    """Central differences of sum(g_colors * colours) with respect to every RAW input (euler, shp, ampraw, dc, means)
    against nasg_ref_paper_bwd: pins eqs.(37)-(44) + the Table 8 activation derivatives end to end. A wrong sign in
    ds/dc (eq.36), the garbled eq.(39), or a missing tanh' = 1 - c^2 fails it."""
    inp = _case(N=4, K=2, C=2, seed=11)
    g = oracle.paper_bwd(inp, mode)
    L = lambda d: float((oracle.paper_fwd(d, mode) * inp["g_colors"]).sum())
    for key, gkey in (("euler", "g_euler"), ("shp", "g_shp"), ("ampraw", "g_ampraw"), ("dc", "g_dc"), ("means", "g_means")):
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


def test_culled_pairs_and_ranges(oracle):
    """Culled (c,n): colour exactly 0, no gradient; k stays in [0, 40] and w in [-1, 1] whatever the raw value
    (Table 8 ranges): colours are finite for extreme raw inputs."""
    inp = _case(N=6, K=2, C=2, seed=5)
    inp["vis"][:, 2] = 0
    col, g = oracle.paper_fwd(inp, 1), oracle.paper_bwd(inp, 1)
    assert (col[:, 2] == 0).all() and (g["g_euler"][:, 2] == 0).all() and (g["g_means"][2] == 0).all() and (g["g_dc"][:, 2] == 0).all()
    wild = dict(inp, vis=None)
    wild["shp"] = inp["shp"].copy(); wild["shp"][..., 2] = 30.0              # k -> 40
    wild["ampraw"] = np.full_like(inp["ampraw"], -40.0)                     # w -> -1
    c2 = oracle.paper_fwd(wild, 1)
    assert np.isfinite(c2).all()
