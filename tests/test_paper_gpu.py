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


@pytest.mark.parametrize("cfg", [1, 2, 4])
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


@pytest.mark.parametrize("N", [10_007, 3 * 131072 + 4099])
def test_paper_host_entry_point(B, W, N):
    """nasg_paper_eval_fwd_bwd_host (the call bench.py --layout paper times end to end): a single chunk, and the chunked
    three-stream pipeline with a ragged last chunk, are bit-identical to the device entry points on the same paper
    records (chunks are multiples of 256 Gaussians, so every chunk runs the same kernels on the same tiles). Twice in a
    row on a side stream, as test_rec_host_entry_point."""
    inp = W.make_paper(W.CONFIGS[2], N)
    K, C = inp["K"], inp["C"]
    col, _, grec = run_paper(B, W, inp, 1)
    nf = B.nasg_paper_floats(N, K)
    host = dict(params=torch.from_numpy(W.pack_paper_records(inp["means"], inp["euler"], inp["shp"], inp["ampraw"], inp["dc"])).pin_memory(),
                campos=torch.from_numpy(inp["campos"]), vis=torch.from_numpy(inp["vis"]).pin_memory(),
                g_colors=torch.from_numpy(inp["g_colors"]).pin_memory())
    out = dict(colors=torch.empty((C, N, 3)).pin_memory(), g_params=torch.zeros(nf).pin_memory())
    scratch = torch.empty(B.nasg_paper_host_scratch_bytes(N, K, C), dtype=torch.uint8, device="cuda")
    side = torch.cuda.Stream()
    want = W.unpack_paper_records(grec.cpu().numpy(), N, K)
    for _ in range(2):
        out["colors"].fill_(7.0); out["g_params"].fill_(7.0)
        with torch.cuda.stream(side):
            B.nasg_rec_eval_fwd_bwd_host(host, out, N, K, scratch, 1, stream=side, paper=True)
        side.synchronize()
        assert np.array_equal(out["colors"].numpy(), col.cpu().numpy())
        got = W.unpack_paper_records(out["g_params"].numpy(), N, K)          # (padding lanes of the last record are not results)
        for k in ("means", "euler", "shp", "ampraw", "dc"):
            assert np.array_equal(got[k], want[k]), k


@pytest.mark.parametrize("N", [50_016, None])
def test_paper_unmirrored_cameras(B, W, oracle, N):
    """The cameras as drawn, on both sides of the y = 0 plane (W.make_paper mirrors them into y <= 0 because the
    Supplementary C frame can only point lobe axes into y >= 0; R18). Half of the view
    directions now look at lobes from behind, so evaluations next to the antipode d = -z, rare with mirrored cameras,
    are common, and eq.(9) is ill-conditioned there for broad anisotropic lobes (R11;
    tests/test_oracle_conditioning.py: one rounding of one input moves the ORACLE's gradient by up to half the tolerance).
    cfg2 recipe, small and at full N, every element: colours at 1e-5 everywhere; every gradient at 1e-4 over the Gaussians
    whose oracle gradient moves by at most 0.25 BWD_TOL under a one-ulp move of the inputs
    (gpu_util.oracle_ulp_sensitivity); the others (printed; a few per million) are held to a small multiple of their own
    oracle response."""
    from gpu_util import oracle_ulp_sensitivity, split_by_conditioning
    inp = W.make_paper(W.CONFIGS[2], N, mirror_cameras=False)
    assert (inp["campos"][:, 1] > 0).any() and (inp["campos"][:, 1] < 0).any()       # cameras on both sides
    col, g, _ = run_paper(B, W, inp, 1)
    err_colors = rel_err(col, oracle.paper_fwd(inp, 1))
    bwd = lambda x: oracle.paper_bwd(x, 1)
    rg = bwd(inp)
    sens = oracle_ulp_sensitivity(bwd, inp, ("means", "campos", "euler", "shp", "ampraw", "dc"), rg)
    errs = split_by_conditioning(g, rg, sens, GRADS)
    print(f"paper cfg2 N={inp['N']} cameras as drawn: colors={err_colors:.2e}",
          " ".join(f"{k}={v:.2e}" if isinstance(v, float) else f"{k}={v}" for k, v in errs.items()),
          "largest oracle response %.2e" % sens.max())
    assert err_colors <= FWD_TOL
    assert errs["excluded"] <= max(2, 2e-5 * inp["N"]), errs["excluded"]
    for gk, _ in GRADS:
        assert errs[gk] <= BWD_TOL, (gk, errs)
    assert errs["worst_ratio"] <= 4.0, errs
