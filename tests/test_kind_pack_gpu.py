"""nasg_kind_pack / nasg_kind_unpack / nasg_rec16_unpack (include/nasg.h): records of every kind built and decoded through
the C ABI. Checked three ways per kind: (1) against the float offsets the header comment documents, spelled out here with
explicit indices; (2) bit for bit against the numpy packers of workloads.py, which every parity test feeds to the kernels;
(3) unpack(pack(x)) == x, with a ragged last record and its padding lanes."""
import numpy as np
import pytest
import torch

pytestmark = pytest.mark.gpu
KINDS = {0: 11, 1: 9, 2: 7, 4: 9}
PAD_ONE = {0: 0, 1: None, 2: 2, 4: 0}


@pytest.fixture(scope="module")
def B():
    assert torch.cuda.is_available(), "these tests need a CUDA device"
    from paper_2606_09794_b200 import binding
    return binding


@pytest.fixture(scope="module")
def W():
    from paper_2606_09794_b200 import workloads
    return workloads


def _rows(kind, K, N, seed):
    r = np.random.default_rng(seed)
    M = KINDS[kind]
    return (r.standard_normal((N, 3)).astype(np.float32), r.standard_normal((3, N)).astype(np.float32),
            r.standard_normal((K, N, M)).astype(np.float32))


@pytest.mark.parametrize("kind", [0, 1, 2, 4])
@pytest.mark.parametrize("K,N", [(2, 1), (4, 4_099), (8, 2_048)])
def test_kind_pack_matches_the_documented_offsets_and_round_trips(B, kind, K, N):
    M = KINDS[kind]
    means, dc, comp = _rows(kind, K, N, 100 * kind + K)
    rec_t = B.nasg_kind_pack(kind, torch.from_numpy(means).cuda(), torch.from_numpy(dc).cuda(), torch.from_numpy(comp).cuda())
    T = (N + 31) // 32
    assert rec_t.numel() == B.nasg_kind_floats(kind, N, K) == T * (6 + M * K) * 32
    rec = rec_t.cpu().numpy().reshape(T, (6 + M * K) * 32)
    rs = np.random.default_rng(1)
    for _ in range(400):                                       # the header comment, index by index
        n = int(rs.integers(N)); t, lane = divmod(n, 32)
        l, c = int(rs.integers(K)), int(rs.integers(M))
        j, h = divmod(l, 2)
        assert rec[t, 192 + 64 * M * j + 64 * c + 2 * lane + h] == comp[l, n, c]
        a = int(rs.integers(3))
        assert rec[t, 32 * a + lane] == means[n, a] and rec[t, 96 + 32 * a + lane] == dc[a, n]
    if N % 32:                                                  # padding lanes: zeros, a 1 where a norm would divide
        lane = 31
        for l in range(K):
            j, h = divmod(l, 2)
            for c in range(M):
                assert rec[T - 1, 192 + 64 * M * j + 64 * c + 2 * lane + h] == (1.0 if c == PAD_ONE[kind] else 0.0)
        assert rec[T - 1, lane] == 0.0 and rec[T - 1, 96 + lane] == 0.0
    back = B.nasg_kind_unpack(kind, rec_t, N, K)
    torch.cuda.synchronize()
    assert np.array_equal(back["means"].cpu().numpy(), means) and np.array_equal(back["dc"].cpu().numpy(), dc)
    assert np.array_equal(back["comp"].cpu().numpy(), comp)


def test_kind_pack_equals_the_numpy_packers_of_every_kind(B, W):
    """The records the parity tests feed to the kernels are built by workloads.pack_*_records; a C caller builds them with
    nasg_kind_pack. Same bits, every kind, ragged N; kind 0 also equals nasg_rec_pack."""
    N = 4_099
    t = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    cat = lambda *parts: np.ascontiguousarray(np.concatenate(parts, axis=2), dtype=np.float32)
    inp = W.make(2, N)
    comp = cat(inp["quat"], inp["shape"], inp["amp"].transpose(0, 2, 1))
    got = B.nasg_kind_pack(B.KIND_QUAT, t(inp["means"]), t(inp["dc"]), t(comp))
    assert np.array_equal(got.cpu().numpy(), W.pack_records(inp["means"], inp["quat"], inp["shape"], inp["amp"], inp["dc"]))
    assert torch.equal(got, B.nasg_rec_pack(t(inp["means"]), t(inp["quat"]), t(inp["shape"]), t(inp["amp"]), t(inp["dc"])))
    inp = W.make_paper(W.CONFIGS[2], N)
    comp = cat(inp["euler"], inp["shp"], inp["ampraw"].transpose(0, 2, 1))
    got = B.nasg_kind_pack(B.KIND_PAPER, t(inp["means"]), t(inp["dc"]), t(comp))
    assert np.array_equal(got.cpu().numpy(), W.pack_paper_records(inp["means"], inp["euler"], inp["shp"], inp["ampraw"], inp["dc"]))
    inp = W.make_iso(W.CONFIGS[2], N)
    comp = cat(inp["axis"], inp["shp"][..., None], inp["amp"].transpose(0, 2, 1))
    got = B.nasg_kind_pack(B.KIND_ISO, t(inp["means"]), t(inp["dc"]), t(comp))
    assert np.array_equal(got.cpu().numpy(), W.pack_iso_records(inp["means"], inp["axis"], inp["shp"], inp["amp"], inp["dc"]))
    inp = W.make_asg(W.CONFIGS[2], N)
    comp = cat(inp["quat"], inp["shp"], inp["amp"].transpose(0, 2, 1))
    got = B.nasg_kind_pack(B.KIND_ASG, t(inp["means"]), t(inp["dc"]), t(comp))
    assert np.array_equal(got.cpu().numpy(), W.pack_asg_records(inp["means"], inp["quat"], inp["shp"], inp["amp"], inp["dc"]))


def test_kind_unpack_decodes_a_gradient_record(B, W):
    """The gradient record of the paper kind, decoded through the C ABI, equals the numpy decoder the parity tests use."""
    N = 2_101
    inp = W.make_paper(W.CONFIGS[2], N)
    K = inp["K"]
    params = torch.from_numpy(W.pack_paper_records(inp["means"], inp["euler"], inp["shp"], inp["ampraw"], inp["dc"])).cuda()
    grec = B.nasg_paper_eval_bwd(params, N, K, torch.from_numpy(inp["campos"]).cuda(), torch.from_numpy(inp["g_colors"]).cuda(),
                                 torch.from_numpy(inp["vis"]).cuda(), 1)
    got = B.nasg_kind_unpack(B.KIND_PAPER, grec, N, K)
    torch.cuda.synchronize()
    want = W.unpack_paper_records(grec.cpu().numpy(), N, K)
    comp = got["comp"].cpu().numpy()
    assert np.array_equal(got["means"].cpu().numpy(), want["means"]) and np.array_equal(got["dc"].cpu().numpy(), want["dc"])
    assert np.array_equal(comp[..., 0:3], want["euler"]) and np.array_equal(comp[..., 3:6], want["shp"])
    assert np.array_equal(comp[..., 6:9].transpose(0, 2, 1), want["ampraw"])


@pytest.mark.parametrize("K,N", [(2, 33), (4, 4_099), (8, 1_024)])
def test_rec16_unpack_returns_the_rounded_values(B, W, K, N):
    import dataclasses
    inp = W.make_nasg(dataclasses.replace(W.CONFIGS[2], seed=900 + K, K=K), N=N)
    t = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    rec16 = B.nasg_rec16_pack(t(inp["means"]), t(inp["quat"]), t(inp["shape"]), t(inp["amp"]), t(inp["dc"]))
    got = B.nasg_rec16_unpack(rec16, N, K)
    torch.cuda.synchronize()
    assert np.array_equal(got["quat"].cpu().numpy(), W.to_bf16(inp["quat"])) and np.array_equal(got["amp"].cpu().numpy(), W.to_bf16(inp["amp"]))
    for k in ("means", "shape", "dc"):
        assert np.array_equal(got[k].cpu().numpy(), inp[k]), k
