"""CPU-only checks of the C-ABI library: it loads, exports every symbol include/nasg.h declares, and
its argument validation returns the documented codes without touching a GPU (no compute calls)."""
import ctypes as C
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def B():
    from paper_2606_09794_b200 import binding
    return binding


def _declared_symbols():
    text = open(os.path.join(ROOT, "include", "nasg.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b((?:nasg|sh)_[a-z_0-9]+)\s*\(", text)))


def test_library_exports_every_declared_symbol(B):
    names = _declared_symbols()
    assert {"nasg_eval_fwd", "nasg_eval_bwd", "sh_eval_fwd", "sh_eval_bwd", "nasg_workspace_bytes",
            "nasg_strerror"} <= set(names)
    lib = C.CDLL(B.LIB_PATH)
    for name in names:
        assert hasattr(lib, name), name
    assert set(B.SYMBOLS) == set(names)
    assert "sm_100a" in B.nasg_version()


def test_library_is_sm100a_only():
    import subprocess
    from paper_2606_09794_b200 import build
    out = subprocess.run(["cuobjdump", "-lelf", build.LIB], capture_output=True, text=True).stdout
    assert "sm_100a" in out and not re.search(r"sm_(?!100a)\d+", out), out


def test_error_codes_without_gpu(B):
    lib = C.CDLL(B.LIB_PATH)
    lib.nasg_eval_fwd.restype = C.c_int
    lib.nasg_eval_bwd.restype = C.c_int
    lib.sh_eval_fwd.restype = C.c_int
    lib.sh_eval_fwd.argtypes = [C.c_int64, C.c_int32] + [C.c_void_p] * 6
    buf = (C.c_float * 64)()
    p = C.addressof(buf)

    def inputs(N=4, K=2, Cn=1, **kw):
        d = dict(means=p, quat=p, shape=p, amp=p, dc=p, campos=p, vis=None)
        d.update(kw)
        return B._Inputs(N, K, Cn, d["means"], d["quat"], d["shape"], d["amp"], d["dc"], d["campos"], d["vis"])

    fwd = lambda inp, colors=p, mode=1: lib.nasg_eval_fwd(C.byref(inp), C.c_void_p(colors), mode, None)
    assert lib.nasg_eval_fwd(None, C.c_void_p(p), 1, None) == -1                 # NASG_ERR_NULL
    assert fwd(inputs(means=None)) == -1
    assert fwd(inputs(), colors=None) == -1
    assert fwd(inputs(N=-1)) == -2 and fwd(inputs(Cn=0)) == -2 and fwd(inputs(Cn=65)) == -2   # SHAPE
    assert fwd(inputs(K=6)) == -3 and fwd(inputs(K=0)) == -3                     # UNSUPPORTED_K
    assert fwd(inputs(quat=p + 4)) == -4                                        # ALIGN
    assert fwd(inputs(), mode=3) == -7                                          # NORM_MODE (0, 1, 2 are valid)
    assert fwd(inputs(N=0, means=None)) == 0                                    # N == 0 is a no-op
    g = B._Grads(p, p, p, p, p, p, None, 0)
    assert lib.nasg_eval_bwd(C.byref(inputs()), C.c_void_p(p), C.byref(g), 1, None) == -5   # WORKSPACE
    g = B._Grads(p, p + 8, p, p, p, None, None, 0)
    assert lib.nasg_eval_bwd(C.byref(inputs()), C.c_void_p(p), C.byref(g), 1, None) == -4   # ALIGN (g_quat)
    assert lib.nasg_eval_bwd(C.byref(inputs()), None, C.byref(g), 1, None) == -1
    assert lib.sh_eval_fwd(4, 0, p, p, p, None, p, None) == -2
    assert lib.sh_eval_fwd(4, 1, None, p, p, None, p, None) == -1
    # nasg_eval_bwd_noalloc (built-in scratch): argument checks come before any CUDA call, so they run without a GPU
    noalloc = lambda inp, gr: lib.nasg_eval_bwd_noalloc(C.byref(inp), C.c_void_p(p), C.byref(gr), 1, None)
    g = B._Grads(p, p, p, p, p, None, None, 0)
    assert noalloc(inputs(), g) == -1                                           # g_campos is required
    g = B._Grads(p, p, p, p, p, p, None, 0)
    assert noalloc(inputs(K=6), g) == -3 and noalloc(inputs(Cn=65), g) == -2
    cap = B.nasg_noalloc_workspace_bytes()
    assert cap == 1 << 20 == B.nasg_workspace_bytes(256 * 21845, 4, 4) + 16     # 21,845 block rows of 4 x 3 floats fit
    assert noalloc(inputs(N=256 * 21845 + 1, K=4, Cn=4), g) == -8               # one more row does not: NOALLOC_SIZE
    assert noalloc(inputs(N=256 * 87381 + 1, K=2, Cn=1), g) == -8
    assert "nasg_eval_bwd" in B.nasg_strerror(-8)
    # nasg_kind_* (records of every kind from C): sizes and argument checks
    from paper_2606_09794_b200 import workloads as W
    assert [B.nasg_kind_components(k) for k in (0, 1, 2, 4, 3, 5, -1)] == [11, 9, 7, 9, 0, 0, 0]
    for n, k in ((1, 2), (4_099, 4), (3_000_000, 8)):
        assert B.nasg_kind_floats(0, n, k) == B.nasg_rec_floats(n, k) == W.rec_floats(n, k)
        assert B.nasg_kind_floats(1, n, k) == B.nasg_paper_floats(n, k) == W.paper_rec_floats(n, k)
        assert B.nasg_kind_floats(2, n, k) == B.nasg_iso_floats(n, k) == W.iso_rec_floats(n, k)
        assert B.nasg_kind_floats(4, n, k) == B.nasg_asg_floats(n, k) == W.asg_rec_floats(n, k)
    assert B.nasg_kind_floats(3, 100, 4) == 0 and B.nasg_kind_floats(0, 100, 3) == 0
    lib.nasg_kind_pack.argtypes = [C.c_int, C.c_int64, C.c_int32] + [C.c_void_p] * 5
    lib.nasg_kind_unpack.argtypes = [C.c_int, C.c_int64, C.c_int32] + [C.c_void_p] * 5
    lib.nasg_rec16_unpack.argtypes = [C.c_int64, C.c_int32] + [C.c_void_p] * 7
    assert lib.nasg_kind_pack(3, 4, 2, p, p, p, p, None) == -7                    # unknown kind
    assert lib.nasg_kind_pack(0, 4, 3, p, p, p, p, None) == -3 and lib.nasg_kind_pack(0, -1, 2, p, p, p, p, None) == -2
    assert lib.nasg_kind_pack(1, 4, 2, p, None, p, p, None) == -1 and lib.nasg_kind_pack(1, 4, 2, p, p, p, p + 4, None) == -4
    assert lib.nasg_kind_pack(2, 0, 2, None, None, None, None, None) == 0         # N == 0 is a no-op
    assert lib.nasg_kind_unpack(5, 4, 2, p, p, p, p, None) == -7 and lib.nasg_kind_unpack(4, 4, 2, None, p, p, p, None) == -1
    assert lib.nasg_rec16_unpack(4, 5, p, p, p, p, p, p, None) == -3 and lib.nasg_rec16_unpack(4, 2, None, p, p, p, p, p, None) == -1
    for code in (0, -1, -2, -3, -4, -5, -7, -8):
        assert B.nasg_strerror(code) and "unknown" not in B.nasg_strerror(code)
    assert "unknown" in B.nasg_strerror(-99)


def test_workspace_sizes(B):
    assert B.nasg_workspace_bytes(0, 4, 4) == 0
    assert B.nasg_workspace_bytes(3_000_000, 4, 4) == ((3_000_000 + 255) // 256) * 4 * 3 * 4
    n, k, c = 1000, 4, 4
    need = n * 12 * 2 + 2 * 2 * k * n * 16 + 2 * k * n * 12 + 2 * n * 12 + c * n + 2 * c * n * 12
    assert B.nasg_host_scratch_bytes(n, k, c) >= need
    assert B.sh_host_scratch_bytes(n, c) >= 2 * n * 12 + 2 * 48 * n * 4 + c * n + 2 * c * n * 12


def test_binding_rejects_bad_tensors(B):
    import torch
    N, K = 8, 2
    t = lambda *s: torch.zeros(*s)
    with pytest.raises(ValueError):
        B._inputs(t(N, 3), t(K, N, 4), t(K, N, 4), t(K, 3, N), t(3, N), t(1, 3), None, device_type="cuda")
    with pytest.raises(ValueError):
        B._inputs(t(N, 3), t(K, N, 4), t(K, N, 3), t(K, 3, N), t(3, N), t(1, 3), None, device_type="cpu")
    B._inputs(t(N, 3), t(K, N, 4), t(K, N, 4), t(K, 3, N), t(3, N), t(1, 3), None, device_type="cpu")


def test_product_never_imports_the_oracle():
    pkg = os.path.join(ROOT, "paper_2606_09794_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle", src, flags=re.M), f
                assert "oracle/" not in src and "nasg_ref" not in src and "sh_ref" not in src, f
    for f in ("nasg_ref.c", "sh_ref.c", "ref.py"):
        src = open(os.path.join(ROOT, "oracle", f)).read()
        assert "binding" not in src and "csrc" not in src and "nasg.h" not in src, f


def test_rec_error_codes_without_gpu(B):
    import ctypes as C
    lib = B._lib
    inp = B._RecInputs(64, 3, 1, 16, 16, None)
    assert lib.nasg_rec_eval_fwd(C.byref(inp), 16, 1, None) == -3          # K = 3
    inp = B._RecInputs(64, 4, 5, 16, 16, None)
    assert lib.nasg_rec_eval_fwd(C.byref(inp), 16, 1, None) == -2          # C = 5
    inp = B._RecInputs(64, 4, 1, None, 16, None)
    assert lib.nasg_rec_eval_fwd(C.byref(inp), 16, 1, None) == -1
    inp = B._RecInputs(64, 4, 1, 20, 16, None)
    assert lib.nasg_rec_eval_fwd(C.byref(inp), 16, 1, None) == -4          # params misaligned
    inp = B._RecInputs(64, 4, 1, 16, 16, None)
    assert lib.nasg_rec_eval_fwd(C.byref(inp), 16, 7, None) == -7
    assert lib.nasg_rec_eval_bwd(C.byref(inp), 16, None, 1, None) == -1
    inp = B._RecInputs(0, 4, 1, None, None, None)
    assert lib.nasg_rec_eval_fwd(C.byref(inp), None, 1, None) == 0         # N = 0: no-op


def test_record_layout_reordering_round_trips():
    """workloads.pack_records / unpack_records (no arithmetic: the input generator's re-ordering into the tile-record
    layout of include/nasg.h) against the documented index formula."""
    import numpy as np
    from paper_2606_09794_b200 import workloads as W
    for cfg, N in ((2, 77), (4, 32), (0, 1)):
        inp = W.make(cfg, N)
        K = inp["K"]
        rec = W.pack_records(inp["means"], inp["quat"], inp["shape"], inp["amp"], inp["dc"])
        assert rec.size == W.rec_floats(N, K)
        back = W.unpack_records(rec, N, K)
        for k in ("means", "quat", "shape", "amp", "dc"):
            assert np.array_equal(back[k], inp[k]), k
        R = (6 + 11 * K) * 32
        for n in {0, N // 2, N - 1}:
            t, lane = divmod(n, 32)
            flat = rec[t * R:(t + 1) * R]
            assert flat[lane] == inp["means"][n, 0] and flat[64 + lane] == inp["means"][n, 2]
            assert flat[96 + 32 + lane] == inp["dc"][1, n]
            for l in range(K):
                j, h = divmod(l, 2)
                for c in range(4):
                    assert flat[192 + 704 * j + 64 * c + 2 * lane + h] == inp["quat"][l, n, c]
                    assert flat[192 + 704 * j + 64 * (4 + c) + 2 * lane + h] == inp["shape"][l, n, c]
                for c in range(3):
                    assert flat[192 + 704 * j + 64 * (8 + c) + 2 * lane + h] == inp["amp"][l, c, n]
