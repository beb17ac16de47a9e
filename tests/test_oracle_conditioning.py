"""The conditioning of eq.(9) next to d = -z, measured on the fp64 oracle itself (CPU only; R11).

Two full-size GPU parity tests (test_rec16_full_size_every_element, test_paper_unmirrored_cameras) leave a handful of
Gaussians out of the 1e-4 max-norm check. This file is the evidence that they may: for the Gaussian that first showed the
problem, ONE rounding of ONE fp32 input moves the oracle's own gradient by a quarter to a half of the whole tolerance, so no
fp32 evaluation (a dozen roundings on the way to d.x, d.y, d.z) can be held to 1e-4 there; and the selector the GPU tests
use (gpu_util.oracle_ulp_sensitivity, the oracle's response to a one-ulp move of every input) picks that Gaussian and
almost nothing else."""
import numpy as np
import pytest

from gpu_util import BWD_TOL, ULP_SENS_LIMIT, oracle_ulp_sensitivity

N_BAD = 1_266_176          # cfg2, bf16-rounded quaternion / amplitude: a broad, very anisotropic lobe seen from next to its antipode
FLOAT_KEYS = ("means", "campos", "quat", "shape", "amp", "dc")


@pytest.fixture(scope="module")
def W():
    from paper_2606_09794_b200 import workloads
    return workloads


@pytest.fixture(scope="module")
def full(oracle, W):
    inp = W.make(2, None)
    inp = dict(inp, quat=W.to_bf16(inp["quat"]), amp=W.to_bf16(inp["amp"]))
    rg = oracle.nasg_bwd(inp, 1)                                   # the whole of cfg2 once: the max-norm scale of every array
    scale = {k: float(np.abs(v).max()) for k, v in rg.items() if k != "g_campos"}
    return inp, scale


def test_the_ill_conditioned_gaussian_sits_next_to_an_antipode(W, full):
    inp, _ = full
    one = W.take(inp, [N_BAD])
    q = one["quat"][:, 0].astype(np.float64)
    q /= np.linalg.norm(q, axis=1, keepdims=True)
    w, x, y, z = q.T
    Z = np.stack([2 * (x * z + w * y), 2 * (y * z - w * x), 1 - 2 * (x * x + y * y)], axis=1)         # lobe axes [K,3]
    d = one["means"][0].astype(np.float64) - inp["campos"].astype(np.float64)                          # [C,3]
    d /= np.linalg.norm(d, axis=1, keepdims=True)
    v = Z @ d.T                                                                                        # d.z per (lobe, camera)
    lam = np.exp(one["shape"][:, 0, 1].astype(np.float64))
    a = np.exp(one["shape"][:, 0, 0].astype(np.float64)) / lam - 1.0
    seen = one["vis"][:, 0] != 0
    hit = (v < -0.999) & seen[None, :] & (lam < 2.0)[:, None] & (a > 100.0)[:, None]
    assert hit.any(), (v, lam, a)                                  # d.z = -0.99945, lambda = 1.08, a = 116


def test_one_rounding_of_one_input_uses_up_a_quarter_of_the_tolerance(oracle, W, full):
    """Gaussian N_BAD: the largest change of the oracle's g_means (relative to max|g_means| of the whole array) when a single
    element of a single input array moves to the next fp32 number. Measured: 7.8e-6 (a mean component), 3.1e-5 (a campos
    component), 4.8e-5 (a quaternion component) -- against BWD_TOL = 1e-4 for the whole evaluation."""
    inp, scale = full
    one = W.take(inp, [N_BAD])
    base = oracle.nasg_bwd(one, 1)["g_means"]
    assert np.abs(base).max() > 0.5 * scale["g_means"]             # and its gradient is among the largest of the array (0.80 of the max)
    worst = {}
    for key in ("means", "campos", "quat"):
        worst[key] = 0.0
        for idx in np.ndindex(one[key].shape):
            for toward in (np.float32(np.inf), np.float32(-np.inf)):
                moved = dict(one)
                moved[key] = one[key].copy()
                moved[key][idx] = np.nextafter(moved[key][idx], toward)
                worst[key] = max(worst[key], float(np.abs(oracle.nasg_bwd(moved, 1)["g_means"] - base).max()) / scale["g_means"])
    print("one-ulp responses of g_means at n = %d:" % N_BAD, worst)
    assert worst["means"] >= 5e-6 and worst["campos"] >= 0.25 * BWD_TOL and worst["quat"] >= 0.3 * BWD_TOL, worst
    assert max(worst.values()) <= BWD_TOL                         # (one rounding alone does not break the tolerance; a dozen do)


def test_the_selector_finds_it_and_little_else(oracle, W, full):
    """gpu_util.oracle_ulp_sensitivity on the first 30,000 Gaussians of cfg2 plus N_BAD, in the max-norm scale of the full
    arrays: N_BAD responds with 1e-4 .. 2e-4 depending on the draw (the tolerance itself or twice it) and is selected; of the 30,000 ordinary Gaussians at most
    3 are (full N: 6 of 3,000,000), and their median response is below 1e-8."""
    inp, scale = full
    idx = np.concatenate([np.arange(30_000), [N_BAD]])
    sub = W.take(inp, idx)
    bwd = lambda x: oracle.nasg_bwd(x, 1)
    sens = oracle_ulp_sensitivity(bwd, sub, FLOAT_KEYS, bwd(sub), draws=3, scale=scale)
    print("response of N_BAD %.2e; ordinary Gaussians: median %.1e, max %.1e, selected %d" %
          (sens[-1], np.median(sens[:-1]), sens[:-1].max(), int((sens[:-1] > ULP_SENS_LIMIT).sum())))
    assert sens[-1] > 2 * ULP_SENS_LIMIT
    assert (sens[:-1] > ULP_SENS_LIMIT).sum() <= 3 and np.median(sens[:-1]) < 1e-8
