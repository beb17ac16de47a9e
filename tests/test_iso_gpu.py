"""GPU parity of the isotropic Table-6 functions (include/nasg.h: nasg_iso_*) against the fp64
oracle (oracle/iso_ref.c, pinned by tests/test_oracle_iso_pins.py), element by element on the same seeded inputs."""
import dataclasses

import numpy as np
import pytest
import torch

from gpu_util import BWD_TOL, FWD_TOL, p99_rel, rel_err

pytestmark = pytest.mark.gpu
GRADS = (("g_means", "means"), ("g_axis", "axis"), ("g_shp", "shp"), ("g_amp", "amp"), ("g_dc", "dc"))
NAMES = {0: "SG", 1: "SBeta", 2: "SCauchy"}


@pytest.fixture(scope="module")
def B():
    assert torch.cuda.is_available(), "these tests need a CUDA device"
    from paper_2606_09794_b200 import binding
    return binding


@pytest.fixture(scope="module")
def W():
    from paper_2606_09794_b200 import workloads
    return workloads


def run_iso(B, W, inp, kind):
    N, K = inp["N"], inp["K"]
    params = torch.from_numpy(W.pack_iso_records(inp["means"], inp["axis"], inp["shp"], inp["amp"], inp["dc"])).cuda()
    campos = torch.from_numpy(inp["campos"]).cuda()
    vis = None if inp.get("vis") is None else torch.from_numpy(inp["vis"]).cuda()
    gcol = torch.from_numpy(inp["g_colors"]).cuda()
    col = B.nasg_iso_eval_fwd(params, N, K, campos, kind, vis)
    grec = B.nasg_iso_eval_bwd(params, N, K, campos, gcol, kind, vis)
    torch.cuda.synchronize()
    return col, W.unpack_iso_records(grec.cpu().numpy(), N, K)


def check_iso(B, W, oracle, inp, kind, label=""):
    col, g = run_iso(B, W, inp, kind)
    rc, rg = oracle.iso_fwd(inp, kind), oracle.iso_bwd(inp, kind)
    errs, p99 = {"colors": rel_err(col, rc)}, {"colors": p99_rel(col, rc)}
    for gk, pk in GRADS:
        errs[gk], p99[gk] = rel_err(g[pk], rg[gk]), p99_rel(g[pk], rg[gk])
    print(label, NAMES[kind], " ".join(f"{k}={errs[k]:.2e}(p99 {p99[k]:.1e})" for k in errs))
    assert errs["colors"] <= FWD_TOL, (label, errs)
    for k, v in errs.items():
        if k != "colors":
            assert v <= BWD_TOL, (label, k, errs)


@pytest.mark.parametrize("kind", [0, 1, 2])
@pytest.mark.parametrize("cfg,N", [(0, None), (1, 70_001), (2, 50_016), (4, 40_007)])
def test_iso_configs_small(B, W, oracle, kind, cfg, N):
    inp = W.make_iso(W.CONFIGS[cfg], N)
    check_iso(B, W, oracle, inp, kind, label=f"iso cfg{cfg} N={inp['N']}")


@pytest.mark.parametrize("kind", [0, 1, 2])
@pytest.mark.parametrize("K,C", [(2, 1), (2, 4), (4, 3), (8, 2)])
def test_iso_lobe_counts_and_cameras(B, W, oracle, kind, K, C):
    cfg = dataclasses.replace(W.CONFIGS[2], seed=600 + K * 10 + C, K=K, C=C)
    inp = W.make_iso(cfg, N=2_101 + 32 * K)
    check_iso(B, W, oracle, inp, kind, label=f"iso K={K} C={C}")


@pytest.mark.parametrize("kind", [0, 1, 2])
def test_iso_masks_and_tiny_sizes(B, W, oracle, kind):
    for N in (1, 33, 257):
        check_iso(B, W, oracle, W.make_iso(W.CONFIGS[2], N), kind, label=f"iso N={N}")
    inp = W.make_iso(W.CONFIGS[2], 6_016)
    gc = inp["g_colors"].copy()
    gc[inp["vis"] == 0] = np.nan                         # culled g_colors are never read as values
    col, g = run_iso(B, W, dict(inp, g_colors=gc), kind)
    rc, rg = oracle.iso_fwd(inp, kind), oracle.iso_bwd(inp, kind)
    assert rel_err(col, rc) <= FWD_TOL and (col.cpu().numpy()[inp["vis"] == 0] == 0).all()
    for gk, pk in GRADS:
        assert rel_err(g[pk], rg[gk]) <= BWD_TOL, gk


@pytest.mark.parametrize("kind", [0, 1, 2])
def test_iso_full_size_every_element(B, W, oracle, kind):
    check_iso(B, W, oracle, W.make_iso(W.CONFIGS[2]), kind, label="iso cfg2 full N=3000000 all elements")
