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


# Gaussian axis of every gradient array (quaternion records and paper records)
GAUSSIAN_AXIS = {"g_means": 0, "g_quat": 1, "g_shape": 1, "g_amp": 2, "g_dc": 1, "g_euler": 1, "g_shp": 1, "g_ampraw": 2}
ULP_SENS_LIMIT = 0.25 * BWD_TOL


def one_ulp(a: np.ndarray, rng: np.random.Generator) -> np.ndarray:
    """Every element of an fp32 array moved to a neighbouring fp32 number, up or down at random."""
    a = np.asarray(a, dtype=np.float32)
    toward = np.where(rng.random(a.shape) < 0.5, np.float32(-np.inf), np.float32(np.inf)).astype(np.float32)
    return np.nextafter(a, toward).astype(np.float32)


def oracle_ulp_sensitivity(bwd, inp: dict, float_keys, ref_grads: dict, draws: int = 3, seed: int = 2024, scale: dict = None) -> np.ndarray:
    """How far the ORACLE's own gradients of each Gaussian move when its fp32 inputs move by one unit in the last place.

    `bwd(inp) -> dict` is the fp64 oracle's backward (ref.nasg_bwd / ref.paper_bwd, norm mode bound by the caller),
    `float_keys` the fp32 input arrays to perturb (means, campos and every parameter array), `ref_grads` the oracle's
    gradients on the unperturbed inputs (`scale`: max|g| per array if `inp` is a subset of a larger set). For each of `draws` seeded draws every element of every one of those arrays
    is replaced by a neighbouring fp32 number (up or down at random) and the oracle is run again; Gaussians are
    independent, so one run yields the response of all of them. Returns [N]: per Gaussian the largest
    |g' - g| / max|g array| over all draws, gradient arrays and components, the same max-norm scale BWD_TOL is stated in.

    Why it exists (R11): eq.(9) is discontinuous at d = -z (0 along the x meridian, e^{-2 lambda} along y).
    Next to that point, for a broad and very anisotropic lobe, the azimuth decides the value, and a single rounding of
    ONE input already moves the oracle's gradient by 3e-5 .. 5e-5 of the array's maximum (tests/test_oracle_conditioning.py
    measures it). An fp32 evaluation, with a dozen roundings on the way to d.x, d.y, d.z, cannot be held to 1e-4 there by
    any implementation. The parity tests that meet such Gaussians leave out exactly those whose response exceeds
    ULP_SENS_LIMIT = 0.25 BWD_TOL, report how many they are, and bound their deviation by a multiple of this response."""
    rng = np.random.default_rng(seed)
    N = int(inp["N"])
    if scale is None:
        scale = {k: float(np.abs(v).max()) + 1e-300 for k, v in ref_grads.items() if k in GAUSSIAN_AXIS}
    sens = np.zeros(N)
    for _ in range(draws):
        moved = dict(inp)
        for k in float_keys:
            moved[k] = one_ulp(inp[k], rng)
        g = bwd(moved)
        for k, sc in scale.items():
            diff = np.abs(g[k] - ref_grads[k])
            axes = tuple(i for i in range(diff.ndim) if i != GAUSSIAN_AXIS[k])
            np.maximum(sens, diff.max(axis=axes) / sc, out=sens)
    return sens


def split_by_conditioning(got: dict, ref_grads: dict, sens: np.ndarray, pairs) -> dict:
    """Max-norm errors of every gradient array over the well-conditioned Gaussians (sens <= ULP_SENS_LIMIT), and for the
    others the largest ratio of a Gaussian's own deviation to its own oracle response. `pairs`: (oracle key, got key)."""
    keep = sens <= ULP_SENS_LIMIT
    out = {"excluded": int((~keep).sum()), "worst_ratio": 0.0}
    for gk, pk in pairs:
        a = got[pk].detach().cpu().numpy() if isinstance(got[pk], torch.Tensor) else np.asarray(got[pk])
        b = ref_grads[gk]
        assert np.all(np.isfinite(a)), gk
        ax = GAUSSIAN_AXIS[gk]
        per_n = np.abs(a - b).max(axis=tuple(i for i in range(b.ndim) if i != ax)) / (np.abs(b).max() + 1e-300)    # [N]
        out[gk] = float(per_n[keep].max())
        out[gk + "(all)"] = float(per_n.max())
        if (~keep).any():
            out["worst_ratio"] = max(out["worst_ratio"], float((per_n[~keep] / sens[~keep]).max()))
    return out
