"""Helpers of the GPU parity tests: move a workload to the device, run the CUDA path through the
C-ABI binding, compare with the fp64 oracle. Tolerances are BASELINE.json's: max|err| <= 1e-5 max|ref|
for the forward colours, <= 1e-4 max|ref| for every gradient array."""
import numpy as np
import torch

FWD_TOL = 1e-5
BWD_TOL = 1e-4
NASG_KEYS = ("means", "quat", "shape", "amp", "dc", "campos", "vis", "g_colors")
SH_KEYS = ("means", "coeffs", "campos", "vis", "g_colors")


def to_dev(inp: dict, keys) -> dict:
    out = {}
    for k in keys:
        v = inp.get(k)
        out[k] = None if v is None else torch.from_numpy(np.ascontiguousarray(v)).cuda()
    return out


def rel_err(got, ref) -> float:
    got = got.detach().cpu().numpy().astype(np.float64) if isinstance(got, torch.Tensor) else np.asarray(got, np.float64)
    assert np.all(np.isfinite(got)), "non-finite output"
    return float(np.max(np.abs(got - ref)) / (np.max(np.abs(ref)) + 1e-300))


def p99_rel(got, ref) -> float:
    """99th percentile of the element-wise relative error |got-ref| / max(|ref|, 1e-6 max|ref|): printed next to
    the max-norm figure (never asserted) so that a regression in the bulk of a heavy-tailed gradient array shows."""
    got = got.detach().cpu().numpy() if isinstance(got, torch.Tensor) else np.asarray(got)
    g, r = got.reshape(-1), np.asarray(ref).reshape(-1)
    if g.size > 4_000_000:                                 # a fixed stride keeps the percentile cheap on 1e8-element arrays
        step = g.size // 2_000_000
        g, r = g[::step], r[::step]
    r = r.astype(np.float64)
    den = np.maximum(np.abs(r), 1e-6 * (np.max(np.abs(ref)) + 1e-300))
    return float(np.percentile(np.abs(g.astype(np.float64) - r) / den, 99.0)) if g.size else 0.0


def run_nasg(B, d: dict, norm_mode=1, want_campos=False):
    col = B.nasg_eval_fwd(d["means"], d["quat"], d["shape"], d["amp"], d["dc"], d["campos"], d["vis"], norm_mode)
    g = B.nasg_eval_bwd(d["means"], d["quat"], d["shape"], d["amp"], d["dc"], d["campos"], d["g_colors"],
                        d["vis"], norm_mode, want_campos=want_campos)
    torch.cuda.synchronize()
    return col, g


def run_sh(B, d: dict, want_campos=False):
    col = B.sh_eval_fwd(d["means"], d["coeffs"], d["campos"], d["vis"])
    g = B.sh_eval_bwd(d["means"], d["coeffs"], d["campos"], d["g_colors"], d["vis"], want_campos=want_campos)
    torch.cuda.synchronize()
    return col, g


def _assert_errs(errs: dict, label):
    print(label, " ".join(f"{k}={v:.2e}" for k, v in errs.items()))
    assert errs["colors"] <= FWD_TOL, (label, errs)
    for k, v in errs.items():
        if k != "colors":
            assert v <= BWD_TOL, (label, k, errs)


def check_nasg(B, oracle, inp: dict, norm_mode=1, want_campos=False, label=""):
    """Forward + backward against the oracle. The backward is always run WITHOUT g_campos and, if want_campos,
    once more WITH it (for C <= 4 both stay on the persistent fast path: g_campos is a compile-time variant of
    the same kernels plus the second-stage reduction; C > 4 runs the generic kernels either way); both must
    meet the tolerances."""
    d = to_dev(inp, NASG_KEYS)
    rc = oracle.nasg_fwd(inp, norm_mode)
    rg = oracle.nasg_bwd(inp, norm_mode)
    col, g = run_nasg(B, d, norm_mode, False)
    errs = {"colors": rel_err(col, rc)}
    for k in ("g_means", "g_quat", "g_shape", "g_amp", "g_dc"):
        errs[k] = rel_err(g[k], rg[k])
    _assert_errs(errs, label)
    if want_campos:
        col, g = run_nasg(B, d, norm_mode, True)
        errs = {"colors": rel_err(col, rc)}
        for k in ("g_means", "g_quat", "g_shape", "g_amp", "g_dc", "g_campos"):
            errs[k] = rel_err(g[k], rg[k])
        _assert_errs(errs, label + " [+g_campos]")
    return col, g, errs


def check_sh(B, oracle, inp: dict, want_campos=False, label=""):
    d = to_dev(inp, SH_KEYS)
    rc = oracle.sh_fwd(inp)
    rg = oracle.sh_bwd(inp)
    col, g = run_sh(B, d, False)
    errs = {"colors": rel_err(col, rc)}
    for k in ("g_means", "g_coeffs"):
        errs[k] = rel_err(g[k], rg[k])
    _assert_errs(errs, label)
    if want_campos:
        col, g = run_sh(B, d, True)
        errs = {"colors": rel_err(col, rc)}
        for k in ("g_means", "g_coeffs", "g_campos"):
            errs[k] = rel_err(g[k], rg[k])
        _assert_errs(errs, label + " [+g_campos]")
    return col, g, errs


def near_antipode(inp: dict, v_max: float = -0.99, lam_max: float = 4.0) -> np.ndarray:
    """Gaussians with a visible (lobe, camera) evaluation close to d = -z of a broad lobe (d.z < v_max, lambda <= lam_max).
    DESIGN.md R11: eq.(9) is discontinuous at d = -z (0 along the x meridian, e^{-2 lambda} along y), so next to it the
    azimuth u/s decides the value and a relative perturbation of 6e-8 of the mean (one fp32 rounding) moves the gradients by
    ~1e-4 of their size: no fp32 evaluation can be held to the tolerance there, the oracle's own result is that sensitive.
    Returns a boolean [N] mask; the test that uses it reports how many Gaussians it excludes."""
    q = np.asarray(inp["quat"], dtype=np.float64)
    q = q / np.linalg.norm(q, axis=2, keepdims=True)
    w, x, y, z = q[..., 0], q[..., 1], q[..., 2], q[..., 3]
    Z = np.stack([2 * (x * z + w * y), 2 * (y * z - w * x), 1 - 2 * (x * x + y * y)], axis=2)           # [K,N,3], column 2 of R(q)
    lam = np.exp(np.asarray(inp["shape"], dtype=np.float64)[..., 1])                                    # [K,N]
    bad = np.zeros(q.shape[1], dtype=bool)
    for c in range(inp["campos"].shape[0]):
        d = np.asarray(inp["means"], dtype=np.float64) - np.asarray(inp["campos"], dtype=np.float64)[c]
        d /= np.linalg.norm(d, axis=1, keepdims=True)
        v = np.einsum("kni,ni->kn", Z, d)
        hit = ((v < v_max) & (lam <= lam_max)).any(axis=0)
        if inp.get("vis") is not None:
            hit &= inp["vis"][c] != 0
        bad |= hit
    return bad
