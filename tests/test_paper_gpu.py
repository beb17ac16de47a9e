"""GPU parity of the paper-native record entry points (include/nasg.h: nasg_paper_*)
against the fp64 oracle (oracle/nasg_ref.c: nasg_ref_paper_*, pinned by tests/test_oracle_paper_pins.py), element by
element on the same seeded RAW values. The records are built by workloads.pack_paper_records (a re-ordering only)."""
import dataclasses

import numpy as np
import pytest
import torch

from gpu_util import BWD_TOL, FWD_TOL, p99_rel, rel_err

pytestmark = pytest.mark.gpu
GRADS = (("g_means", "means"), ("g_euler", "euler"), ("g_shp", "shp"), ("g_ampraw", "ampraw"), ("g_dc", "dc"))


@pytest.fixture(scope="module")
def B():
    assert torch.cuda.is_available(), "these tests need a CUDA device"
    from paper_2606_09794_b200 import binding
    return binding


@pytest.fixture(scope="module")
def W():
    from paper_2606_09794_b200 import workloads
    return workloads


def run_paper(B, W, inp, mode=1):
    N, K = inp["N"], inp["K"]
    params = torch.from_numpy(W.pack_paper_records(inp["means"], inp["euler"], inp["shp"], inp["ampraw"], inp["dc"])).cuda()
    campos = torch.from_numpy(inp["campos"]).cuda()
    vis = None if inp.get("vis") is None else torch.from_numpy(inp["vis"]).cuda()
    gcol = torch.from_numpy(inp["g_colors"]).cuda()
    col = B.nasg_paper_eval_fwd(params, N, K, campos, vis, mode)
    grec = B.nasg_paper_eval_bwd(params, N, K, campos, gcol, vis, mode)
    torch.cuda.synchronize()
    return col, W.unpack_paper_records(grec.cpu().numpy(), N, K), grec


def check_paper(B, W, oracle, inp, mode=1, label=""):
    col, g, _ = run_paper(B, W, inp, mode)
    rc, rg = oracle.paper_fwd(inp, mode), oracle.paper_bwd(inp, mode)
    errs = {"colors": rel_err(col, rc)}
    for gk, pk in GRADS:
        errs[gk] = rel_err(g[pk], rg[gk])
    print(label, " ".join(f"{k}={v:.2e}" for k, v in errs.items()))
    assert errs["colors"] <= FWD_TOL, (label, errs)
    for k, v in errs.items():
        if k != "colors":
            assert v <= BWD_TOL, (label, k, errs)
    return col, g


@pytest.mark.parametrize("cfg,N", [(0, None), (1, 70_001), (2, 50_003), (2, 50_016), (4, 40_007)])
@pytest.mark.parametrize("mode", [1, 0])
def test_paper_configs_small(B, W, oracle, cfg, N, mode):
    inp = W.make_paper(W.CONFIGS[cfg], N)
    check_paper(B, W, oracle, inp, mode, label=f"paper cfg{cfg} N={inp['N']} mode={mode}")


@pytest.mark.parametrize("K", [2, 4, 8])
@pytest.mark.parametrize("C", [1, 2, 3, 4])
def test_paper_all_lobe_counts_and_cameras(B, W, oracle, K, C):
    cfg = dataclasses.replace(W.CONFIGS[2], seed=400 + K * 10 + C, K=K, C=C)
    inp = W.make_paper(cfg, N=2_101 + 32 * K)
    check_paper(B, W, oracle, inp, 1, label=f"paper K={K} C={C}")


@pytest.mark.parametrize("N", [1, 31, 33, 257])
def test_paper_tiny_sizes(B, W, oracle, N):
    check_paper(B, W, oracle, W.make_paper(W.CONFIGS[2], N), 1, label=f"paper N={N}")


def test_paper_pure_nasg_mode_and_masks(B, W, oracle):
    """norm_mode 2: no carrier (k taken as 0, its gradient 0); culled pairs exactly 0, NaN g_colors there never read."""
    inp = W.make_paper(W.CONFIGS[2], 8_016)
    # k -> 0 exactly is not reachable through 20 (tanh + 1): the oracle gets raw_k = -40 (k = 2e-34 ~ 0)
    zero = dict(inp, shp=inp["shp"].copy())
    zero["shp"][..., 2] = -40.0
    rc, rg = oracle.paper_fwd(zero, 0), oracle.paper_bwd(zero, 0)
    col, g, _ = run_paper(B, W, inp, 2)
    assert rel_err(col, rc) <= FWD_TOL
    for gk, pk in (("g_means", "means"), ("g_euler", "euler"), ("g_ampraw", "ampraw"), ("g_dc", "dc")):
        assert rel_err(g[pk], rg[gk]) <= BWD_TOL, gk
    assert rel_err(g["shp"][..., :2], rg["g_shp"][..., :2]) <= BWD_TOL and (g["shp"][..., 2] == 0).all()
    gc = inp["g_colors"].copy()
    gc[inp["vis"] == 0] = np.nan
    col, g, _ = run_paper(B, W, dict(inp, g_colors=gc), 1)
    rc, rg = oracle.paper_fwd(inp, 1), oracle.paper_bwd(inp, 1)
    assert rel_err(col, rc) <= FWD_TOL and (col.cpu().numpy()[inp["vis"] == 0] == 0).all()
    for gk, pk in GRADS:
        assert rel_err(g[pk], rg[gk]) <= BWD_TOL, gk


def test_paper_extreme_raw_values_stay_finite(B, W):
    """Saturated activations (|raw| up to 30: cos = +-1 to rounding, sin = 1e-13; k = 40; w = +-1): finite colours
    and gradients (nothing divides by a sine: the 1/sin of eq.(36) cancels against tanh')."""
    inp = W.make_paper(W.CONFIGS[2], 4_096)
    r = np.random.default_rng(7)
    inp["euler"] = r.choice(np.array([-30.0, -9.0, 0.0, 9.0, 30.0], dtype=np.float32), size=inp["euler"].shape)
    inp["shp"][..., 2] = r.choice(np.array([-30.0, 0.0, 30.0], dtype=np.float32), size=inp["shp"].shape[:2])
    inp["ampraw"] = r.choice(np.array([-30.0, 0.5, 30.0], dtype=np.float32), size=inp["ampraw"].shape)
    col, g, grec = run_paper(B, W, inp, 1)
    assert torch.isfinite(col).all() and np.isfinite(grec.cpu().numpy()).all()


@pytest.mark.parametrize("cfg", [1, 2])
def test_paper_full_size_every_element(B, W, oracle, cfg):
    inp = W.make_paper(W.CONFIGS[cfg])
    col, g, _ = run_paper(B, W, inp, 1)
    rc = oracle.paper_fwd(inp, 1)
    errs, p99 = {"colors": rel_err(col, rc)}, {"colors": p99_rel(col, rc)}
    del rc, col
    rg = oracle.paper_bwd(inp, 1)
    for gk, pk in GRADS:
        errs[gk], p99[gk] = rel_err(g[pk], rg[gk]), p99_rel(g[pk], rg[gk])
    print(f"paper cfg{cfg} full N={inp['N']} all elements:", " ".join(f"{k}={errs[k]:.2e}(p99 {p99[k]:.1e})" for k in errs))
    assert errs.pop("colors") <= FWD_TOL
    for k, v in errs.items():
        assert v <= BWD_TOL, (k, v)
