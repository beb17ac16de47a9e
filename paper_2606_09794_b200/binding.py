"""Thin ctypes binding of ``include/nasg.h`` (argument marshalling only).

Every step of the path runs in the CUDA kernels of ``libnasg_b200.so``; PyTorch is used for device
memory and streams. There is NO CPU fallback: if the library cannot be loaded (or built) the import
fails loudly, and every entry point raises :class:`NasgError` on a non-zero return code.

Names mirror the C ABI: ``nasg_eval_fwd``, ``nasg_eval_bwd``, ``sh_eval_fwd``, ``sh_eval_bwd``,
``nasg_workspace_bytes``, ``nasg_eval_fwd_bwd_host``, ``sh_eval_fwd_bwd_host``, ``nasg_strerror``.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Optional

import torch

from . import build as _build

NORM_APPROX, NORM_EXACT, NORM_NASG = 0, 1, 2
HINT_COHERENT_VIS = 0x100       # OR into norm_mode of nasg_rec_eval_fwd / bwd (include/nasg.h)
MAX_CAMERAS = 64
SYMBOLS = ("nasg_eval_fwd", "nasg_eval_bwd", "sh_eval_fwd", "sh_eval_bwd", "nasg_workspace_bytes",
           "nasg_host_scratch_bytes", "nasg_eval_fwd_bwd_host", "sh_host_scratch_bytes",
           "sh_eval_fwd_bwd_host", "nasg_strerror", "nasg_version", "nasg_launch_count", "nasg_debug_set_path",
           "nasg_rec_floats", "nasg_rec_pack", "nasg_rec_unpack", "nasg_rec_eval_fwd", "nasg_rec_eval_bwd",
           "nasg_rec_host_scratch_bytes", "nasg_rec_eval_fwd_bwd_host", "nasg_paper_floats", "nasg_paper_eval_fwd",
           "nasg_paper_eval_bwd", "nasg_paper_host_scratch_bytes", "nasg_paper_eval_fwd_bwd_host",
           "nasg_iso_floats", "nasg_iso_eval_fwd", "nasg_iso_eval_bwd",
           "nasg_asg_floats", "nasg_asg_eval_fwd", "nasg_asg_eval_bwd",
           "nasg_rec16_floats", "nasg_rec16_pack", "nasg_rec16_eval_fwd", "nasg_rec16_eval_bwd",
           "nasg_noalloc_workspace_bytes", "nasg_eval_bwd_noalloc",
           "nasg_kind_components", "nasg_kind_floats", "nasg_kind_pack", "nasg_kind_unpack", "nasg_rec16_unpack")


class NasgError(RuntimeError):
    def __init__(self, code: int, where: str):
        self.code = code
        super().__init__(f"{where} failed with code {code}: {nasg_strerror(code)}")


class _Inputs(C.Structure):
    _fields_ = [("N", C.c_int64), ("K", C.c_int32), ("C", C.c_int32), ("means", C.c_void_p),
                ("quat", C.c_void_p), ("shape", C.c_void_p), ("amp", C.c_void_p), ("dc", C.c_void_p),
                ("campos", C.c_void_p), ("vis", C.c_void_p)]


class _RecInputs(C.Structure):
    _fields_ = [("N", C.c_int64), ("K", C.c_int32), ("C", C.c_int32), ("params", C.c_void_p),
                ("campos", C.c_void_p), ("vis", C.c_void_p)]


class _Grads(C.Structure):
    _fields_ = [("g_means", C.c_void_p), ("g_quat", C.c_void_p), ("g_shape", C.c_void_p),
                ("g_amp", C.c_void_p), ("g_dc", C.c_void_p), ("g_campos", C.c_void_p),
                ("workspace", C.c_void_p), ("workspace_bytes", C.c_size_t)]


def _load():
    path = _build.LIB
    if _build.is_stale():
        try:
            _build.build()
        except Exception as exc:  # no nvcc on this machine and no prebuilt library: fail loudly
            if not os.path.exists(path):
                raise ImportError(
                    f"libnasg_b200.so is missing and could not be built ({exc}); run "
                    f"`python -m paper_2606_09794_b200.build`. There is no CPU fallback.") from exc
            import warnings       # an older library exists: say that it does not match the sources
            warnings.warn(f"libnasg_b200.so is older than its sources and the rebuild failed ({exc}); "
                          f"loading the stale library", RuntimeWarning)
    lib = C.CDLL(path)
    vp, i64, i32, sz = C.c_void_p, C.c_int64, C.c_int32, C.c_size_t
    lib.nasg_eval_fwd.argtypes = [C.POINTER(_Inputs), vp, C.c_int, vp]
    lib.nasg_eval_bwd.argtypes = [C.POINTER(_Inputs), vp, C.POINTER(_Grads), C.c_int, vp]
    lib.sh_eval_fwd.argtypes = [i64, i32, vp, vp, vp, vp, vp, vp]
    lib.sh_eval_bwd.argtypes = [i64, i32, vp, vp, vp, vp, vp, vp, vp, vp, vp, sz, vp]
    lib.nasg_workspace_bytes.argtypes = [i64, i32, i32]
    lib.nasg_workspace_bytes.restype = sz
    lib.nasg_noalloc_workspace_bytes.argtypes = []
    lib.nasg_noalloc_workspace_bytes.restype = sz
    lib.nasg_eval_bwd_noalloc.argtypes = [C.POINTER(_Inputs), vp, C.POINTER(_Grads), C.c_int, vp]
    lib.nasg_eval_bwd_noalloc.restype = C.c_int
    lib.nasg_host_scratch_bytes.argtypes = [i64, i32, i32]
    lib.nasg_host_scratch_bytes.restype = sz
    lib.sh_host_scratch_bytes.argtypes = [i64, i32]
    lib.sh_host_scratch_bytes.restype = sz
    lib.nasg_eval_fwd_bwd_host.argtypes = [C.POINTER(_Inputs), vp, vp, C.POINTER(_Grads), C.c_int, vp, sz, vp]
    lib.sh_eval_fwd_bwd_host.argtypes = [i64, i32, vp, vp, vp, vp, vp, vp, vp, vp, vp, vp, sz, vp]
    lib.nasg_strerror.argtypes = [C.c_int]
    lib.nasg_strerror.restype = C.c_char_p
    lib.nasg_version.restype = C.c_char_p
    lib.nasg_launch_count.restype = i64
    lib.nasg_debug_set_path.argtypes = [C.c_int]
    lib.nasg_debug_set_path.restype = None
    lib.nasg_rec_floats.argtypes = [i64, i32]
    lib.nasg_rec_floats.restype = sz
    lib.nasg_rec_pack.argtypes = [C.POINTER(_Inputs), vp, vp]
    lib.nasg_rec_unpack.argtypes = [i64, i32, vp, vp, vp, vp, vp, vp, vp]
    lib.nasg_rec_eval_fwd.argtypes = [C.POINTER(_RecInputs), vp, C.c_int, vp]
    lib.nasg_rec_eval_bwd.argtypes = [C.POINTER(_RecInputs), vp, vp, C.c_int, vp]
    lib.nasg_rec16_floats.argtypes = [i64, i32]
    lib.nasg_rec16_floats.restype = sz
    lib.nasg_rec16_pack.argtypes = [C.POINTER(_Inputs), vp, vp]
    lib.nasg_rec16_eval_fwd.argtypes = [C.POINTER(_RecInputs), vp, C.c_int, vp]
    lib.nasg_rec16_eval_bwd.argtypes = [C.POINTER(_RecInputs), vp, vp, C.c_int, vp]
    lib.nasg_iso_floats.argtypes = [i64, i32]
    lib.nasg_iso_floats.restype = sz
    lib.nasg_iso_eval_fwd.argtypes = [C.POINTER(_RecInputs), vp, C.c_int, vp]
    lib.nasg_iso_eval_bwd.argtypes = [C.POINTER(_RecInputs), vp, vp, C.c_int, vp]
    lib.nasg_asg_floats.argtypes = [i64, i32]
    lib.nasg_asg_floats.restype = sz
    lib.nasg_asg_eval_fwd.argtypes = [C.POINTER(_RecInputs), vp, vp]
    lib.nasg_asg_eval_bwd.argtypes = [C.POINTER(_RecInputs), vp, vp, vp]
    lib.nasg_paper_floats.argtypes = [i64, i32]
    lib.nasg_paper_floats.restype = sz
    lib.nasg_paper_eval_fwd.argtypes = [C.POINTER(_RecInputs), vp, C.c_int, vp]
    lib.nasg_paper_eval_bwd.argtypes = [C.POINTER(_RecInputs), vp, vp, C.c_int, vp]
    lib.nasg_kind_components.argtypes = [C.c_int]
    lib.nasg_kind_components.restype = i32
    lib.nasg_kind_floats.argtypes = [C.c_int, i64, i32]
    lib.nasg_kind_floats.restype = sz
    lib.nasg_kind_pack.argtypes = [C.c_int, i64, i32, vp, vp, vp, vp, vp]
    lib.nasg_kind_unpack.argtypes = [C.c_int, i64, i32, vp, vp, vp, vp, vp]
    lib.nasg_rec16_unpack.argtypes = [i64, i32, vp, vp, vp, vp, vp, vp, vp]
    for name in ("nasg_kind_pack", "nasg_kind_unpack", "nasg_rec16_unpack"):
        getattr(lib, name).restype = C.c_int
    lib.nasg_rec_host_scratch_bytes.argtypes = [i64, i32, i32]
    lib.nasg_rec_host_scratch_bytes.restype = sz
    lib.nasg_rec_eval_fwd_bwd_host.argtypes = [C.POINTER(_RecInputs), vp, vp, vp, C.c_int, vp, sz, vp]
    lib.nasg_paper_host_scratch_bytes.argtypes = [i64, i32, i32]
    lib.nasg_paper_host_scratch_bytes.restype = sz
    lib.nasg_paper_eval_fwd_bwd_host.argtypes = [C.POINTER(_RecInputs), vp, vp, vp, C.c_int, vp, sz, vp]
    for name in ("nasg_eval_fwd", "nasg_eval_bwd", "sh_eval_fwd", "sh_eval_bwd", "nasg_eval_fwd_bwd_host",
                 "sh_eval_fwd_bwd_host", "nasg_rec_pack", "nasg_rec_unpack", "nasg_rec_eval_fwd", "nasg_rec_eval_bwd",
                 "nasg_rec_eval_fwd_bwd_host", "nasg_paper_eval_fwd", "nasg_paper_eval_bwd", "nasg_paper_eval_fwd_bwd_host",
                 "nasg_iso_eval_fwd", "nasg_iso_eval_bwd", "nasg_asg_eval_fwd", "nasg_asg_eval_bwd", "nasg_rec16_pack", "nasg_rec16_eval_fwd", "nasg_rec16_eval_bwd"):
        getattr(lib, name).restype = C.c_int
    return lib


_lib = _load()
LIB_PATH = _build.LIB


def nasg_strerror(code: int) -> str:
    return _lib.nasg_strerror(int(code)).decode()


def nasg_version() -> str:
    return _lib.nasg_version().decode()


def nasg_launch_count() -> int:
    return int(_lib.nasg_launch_count())


def nasg_debug_set_path(path: int) -> None:
    """Test hook (include/nasg.h): 0 = automatic dispatch, 1 = generic kernels only, 2 = never the tile kernels."""
    _lib.nasg_debug_set_path(int(path))


def nasg_workspace_bytes(N: int, K: int, Cn: int) -> int:
    return int(_lib.nasg_workspace_bytes(N, K, Cn))


def nasg_host_scratch_bytes(N: int, K: int, Cn: int) -> int:
    return int(_lib.nasg_host_scratch_bytes(N, K, Cn))


def sh_host_scratch_bytes(N: int, Cn: int) -> int:
    return int(_lib.sh_host_scratch_bytes(N, Cn))


def _ptr(t: Optional[torch.Tensor]):
    return None if t is None else t.data_ptr()


def _stream(stream) -> Optional[int]:
    if stream is None:
        stream = torch.cuda.current_stream()
    return stream.cuda_stream if hasattr(stream, "cuda_stream") else int(stream)


def _chk(t: Optional[torch.Tensor], name: str, shape, dtype, device_type: str):
    if t is None:
        return
    if tuple(t.shape) != tuple(shape) or t.dtype != dtype or not t.is_contiguous() or t.device.type != device_type:
        raise ValueError(f"{name}: expected contiguous {dtype} {tuple(shape)} on {device_type}, got "
                         f"{t.dtype} {tuple(t.shape)} on {t.device} contiguous={t.is_contiguous()}")


def _inputs(means, quat, shape, amp, dc, campos, vis, device_type="cuda") -> _Inputs:
    K, N = int(quat.shape[0]), int(quat.shape[1])
    Cn = int(campos.shape[0])
    f32 = torch.float32
    _chk(means, "means", (N, 3), f32, device_type); _chk(quat, "quat", (K, N, 4), f32, device_type)
    _chk(shape, "shape", (K, N, 4), f32, device_type); _chk(amp, "amp", (K, 3, N), f32, device_type)
    _chk(dc, "dc", (3, N), f32, device_type); _chk(campos, "campos", (Cn, 3), f32, device_type)
    _chk(vis, "vis", (Cn, N), torch.uint8, device_type)
    return _Inputs(N, K, Cn, _ptr(means), _ptr(quat), _ptr(shape), _ptr(amp), _ptr(dc), _ptr(campos), _ptr(vis))


def nasg_eval_fwd(means, quat, shape, amp, dc, campos, vis=None, norm_mode: int = NORM_EXACT,
                  out: Optional[torch.Tensor] = None, stream=None) -> torch.Tensor:
    """colors [C,N,3] = c0 + sum_l w_l G_l(normalize(mean - campos))  (eq.(6), eq.(9), eq.(10))."""
    inp = _inputs(means, quat, shape, amp, dc, campos, vis)
    if out is None:
        out = torch.empty((inp.C, inp.N, 3), dtype=torch.float32, device=means.device)
    _chk(out, "colors", (inp.C, inp.N, 3), torch.float32, "cuda")
    rc = _lib.nasg_eval_fwd(C.byref(inp), _ptr(out), int(norm_mode), _stream(stream))
    if rc != 0:
        raise NasgError(rc, "nasg_eval_fwd")
    return out


def nasg_alloc_grads(K: int, N: int, Cn: int, device, want_campos: bool = False) -> dict:
    f32 = torch.float32
    g = dict(g_means=torch.empty((N, 3), dtype=f32, device=device), g_quat=torch.empty((K, N, 4), dtype=f32, device=device),
             g_shape=torch.empty((K, N, 4), dtype=f32, device=device), g_amp=torch.empty((K, 3, N), dtype=f32, device=device),
             g_dc=torch.empty((3, N), dtype=f32, device=device))
    if want_campos:
        g["g_campos"] = torch.empty((Cn, 3), dtype=f32, device=device)
        g["workspace"] = torch.empty(max(1, nasg_workspace_bytes(N, K, Cn)), dtype=torch.uint8, device=device)
    return g


def _grads_struct(g: dict) -> _Grads:
    ws = g.get("workspace")
    return _Grads(_ptr(g.get("g_means")), _ptr(g.get("g_quat")), _ptr(g.get("g_shape")), _ptr(g.get("g_amp")),
                  _ptr(g.get("g_dc")), _ptr(g.get("g_campos")), _ptr(ws), 0 if ws is None else ws.numel())


def nasg_eval_bwd(means, quat, shape, amp, dc, campos, g_colors, vis=None, norm_mode: int = NORM_EXACT,
                  want_campos: bool = False, out: Optional[dict] = None, stream=None) -> dict:
    """Gradients of sum(g_colors * colors): dict g_means, g_quat, g_shape, g_amp, g_dc[, g_campos]."""
    inp = _inputs(means, quat, shape, amp, dc, campos, vis)
    _chk(g_colors, "g_colors", (inp.C, inp.N, 3), torch.float32, "cuda")
    if out is None:
        out = nasg_alloc_grads(inp.K, inp.N, inp.C, means.device, want_campos)
    elif want_campos and (out.get("g_campos") is None or out.get("workspace") is None):
        raise ValueError("want_campos=True but the supplied `out` lacks g_campos / workspace (nasg_alloc_grads(..., want_campos=True))")
    gs = _grads_struct(out)
    rc = _lib.nasg_eval_bwd(C.byref(inp), _ptr(g_colors), C.byref(gs), int(norm_mode), _stream(stream))
    if rc != 0:
        raise NasgError(rc, "nasg_eval_bwd")
    return out


def nasg_noalloc_workspace_bytes() -> int:
    """Capacity of the library's built-in scratch array (include/nasg.h: NASG_NOALLOC_WS_BYTES)."""
    return int(_lib.nasg_noalloc_workspace_bytes())


def nasg_eval_bwd_noalloc(means, quat, shape, amp, dc, campos, g_colors, out: dict, vis=None,
                          norm_mode: int = NORM_EXACT, stream=None) -> dict:
    """``nasg_eval_bwd`` with ``g_campos`` for callers that cannot allocate device memory (a plug-in inside a host
    application's memory budget, a render loop that cannot afford cudaMalloc's device-wide synchronisation, a process
    whose device memory is fully handed out): the partial sums of ``g_campos`` go to a fixed 1 MiB array inside the
    library instead of a caller-provided workspace. Accordingly this wrapper creates no tensor either: ``out`` must
    hold every gradient tensor the caller wants written, ``g_campos`` [C,3] among them (no ``workspace`` entry is
    needed or looked at). Problems with ``nasg_workspace_bytes(N, K, C) > nasg_noalloc_workspace_bytes()`` raise
    ``NasgError`` (code -8). Calls share the one array per device, so calls that may overlap on the GPU race."""
    inp = _inputs(means, quat, shape, amp, dc, campos, vis)
    _chk(g_colors, "g_colors", (inp.C, inp.N, 3), torch.float32, "cuda")
    if out.get("g_campos") is None:
        raise ValueError("nasg_eval_bwd_noalloc: out['g_campos'] [C,3] is required (without it use nasg_eval_bwd)")
    gs = _Grads(_ptr(out.get("g_means")), _ptr(out.get("g_quat")), _ptr(out.get("g_shape")), _ptr(out.get("g_amp")),
                _ptr(out.get("g_dc")), _ptr(out["g_campos"]), None, 0)
    rc = _lib.nasg_eval_bwd_noalloc(C.byref(inp), _ptr(g_colors), C.byref(gs), int(norm_mode), _stream(stream))
    if rc != 0:
        raise NasgError(rc, "nasg_eval_bwd_noalloc")
    return out


def sh_eval_fwd(means, coeffs, campos, vis=None, out: Optional[torch.Tensor] = None, stream=None) -> torch.Tensor:
    """colors [C,N,3] = sum_j coeffs[j,:,n] Y_j(d), real SH degree 3 (eq.(5))."""
    N, Cn = int(means.shape[0]), int(campos.shape[0])
    f32 = torch.float32
    _chk(means, "means", (N, 3), f32, "cuda"); _chk(coeffs, "coeffs", (16, 3, N), f32, "cuda")
    _chk(campos, "campos", (Cn, 3), f32, "cuda"); _chk(vis, "vis", (Cn, N), torch.uint8, "cuda")
    if out is None:
        out = torch.empty((Cn, N, 3), dtype=f32, device=means.device)
    rc = _lib.sh_eval_fwd(N, Cn, _ptr(means), _ptr(coeffs), _ptr(campos), _ptr(vis), _ptr(out), _stream(stream))
    if rc != 0:
        raise NasgError(rc, "sh_eval_fwd")
    return out


def sh_alloc_grads(N: int, Cn: int, device, want_campos: bool = False) -> dict:
    f32 = torch.float32
    g = dict(g_means=torch.empty((N, 3), dtype=f32, device=device), g_coeffs=torch.empty((16, 3, N), dtype=f32, device=device))
    if want_campos:
        g["g_campos"] = torch.empty((Cn, 3), dtype=f32, device=device)
        g["workspace"] = torch.empty(max(1, nasg_workspace_bytes(N, 0, Cn)), dtype=torch.uint8, device=device)
    return g


def sh_eval_bwd(means, coeffs, campos, g_colors, vis=None, want_campos: bool = False, out: Optional[dict] = None,
                stream=None) -> dict:
    N, Cn = int(means.shape[0]), int(campos.shape[0])
    f32 = torch.float32
    _chk(means, "means", (N, 3), f32, "cuda"); _chk(coeffs, "coeffs", (16, 3, N), f32, "cuda")
    _chk(campos, "campos", (Cn, 3), f32, "cuda"); _chk(vis, "vis", (Cn, N), torch.uint8, "cuda")
    _chk(g_colors, "g_colors", (Cn, N, 3), f32, "cuda")
    if out is None:
        out = sh_alloc_grads(N, Cn, means.device, want_campos)
    ws = out.get("workspace")
    rc = _lib.sh_eval_bwd(N, Cn, _ptr(means), _ptr(coeffs), _ptr(campos), _ptr(vis), _ptr(g_colors),
                          _ptr(out.get("g_means")), _ptr(out.get("g_coeffs")), _ptr(out.get("g_campos")),
                          _ptr(ws), 0 if ws is None else ws.numel(), _stream(stream))
    if rc != 0:
        raise NasgError(rc, "sh_eval_bwd")
    return out


def nasg_eval_fwd_bwd_host(host: dict, host_out: dict, dev_scratch: torch.Tensor, norm_mode: int = NORM_EXACT,
                           stream=None) -> None:
    """End-to-end call with HOST tensors (pinned recommended): H2D copies, forward, backward, D2H copies,
    all enqueued on ``stream``; returns without synchronising. ``host`` holds means, quat, shape, amp, dc,
    campos, vis (or None), g_colors; ``host_out`` holds colors and any of g_means, g_quat, g_shape, g_amp,
    g_dc, g_campos."""
    inp = _inputs(host["means"], host["quat"], host["shape"], host["amp"], host["dc"], host["campos"],
                  host.get("vis"), device_type="cpu")
    _chk(host["g_colors"], "g_colors", (inp.C, inp.N, 3), torch.float32, "cpu")
    _chk(host_out["colors"], "colors", (inp.C, inp.N, 3), torch.float32, "cpu")
    gs = _grads_struct({k: v for k, v in host_out.items() if k != "colors"})
    rc = _lib.nasg_eval_fwd_bwd_host(C.byref(inp), _ptr(host["g_colors"]), _ptr(host_out["colors"]), C.byref(gs),
                                     int(norm_mode), _ptr(dev_scratch), dev_scratch.numel() * dev_scratch.element_size(),
                                     _stream(stream))
    if rc != 0:
        raise NasgError(rc, "nasg_eval_fwd_bwd_host")


def sh_eval_fwd_bwd_host(host: dict, host_out: dict, dev_scratch: torch.Tensor, stream=None) -> None:
    N, Cn = int(host["means"].shape[0]), int(host["campos"].shape[0])
    f32 = torch.float32
    _chk(host["means"], "means", (N, 3), f32, "cpu"); _chk(host["coeffs"], "coeffs", (16, 3, N), f32, "cpu")
    _chk(host["campos"], "campos", (Cn, 3), f32, "cpu"); _chk(host.get("vis"), "vis", (Cn, N), torch.uint8, "cpu")
    _chk(host["g_colors"], "g_colors", (Cn, N, 3), f32, "cpu"); _chk(host_out["colors"], "colors", (Cn, N, 3), f32, "cpu")
    _chk(host_out.get("g_means"), "g_means", (N, 3), f32, "cpu"); _chk(host_out.get("g_coeffs"), "g_coeffs", (16, 3, N), f32, "cpu")
    _chk(host_out.get("g_campos"), "g_campos", (Cn, 3), f32, "cpu")
    rc = _lib.sh_eval_fwd_bwd_host(N, Cn, _ptr(host["means"]), _ptr(host["coeffs"]), _ptr(host["campos"]),
                                   _ptr(host.get("vis")), _ptr(host["g_colors"]), _ptr(host_out["colors"]),
                                   _ptr(host_out.get("g_means")), _ptr(host_out.get("g_coeffs")),
                                   _ptr(host_out.get("g_campos")), _ptr(dev_scratch),
                                   dev_scratch.numel() * dev_scratch.element_size(), _stream(stream))
    if rc != 0:
        raise NasgError(rc, "sh_eval_fwd_bwd_host")


# ---- tile-record layout (include/nasg.h: nasg_rec_*) ----------------------------------------------
def nasg_rec_floats(N: int, K: int) -> int:
    return int(_lib.nasg_rec_floats(N, K))


def nasg_rec_pack(means, quat, shape, amp, dc, out: Optional[torch.Tensor] = None, stream=None) -> torch.Tensor:
    """Row arrays (layout v1) -> tile records: float tensor of nasg_rec_floats(N, K) elements."""
    K, N = int(quat.shape[0]), int(quat.shape[1])
    f32 = torch.float32
    _chk(means, "means", (N, 3), f32, "cuda"); _chk(quat, "quat", (K, N, 4), f32, "cuda")
    _chk(shape, "shape", (K, N, 4), f32, "cuda"); _chk(amp, "amp", (K, 3, N), f32, "cuda"); _chk(dc, "dc", (3, N), f32, "cuda")
    inp = _Inputs(N, K, 1, _ptr(means), _ptr(quat), _ptr(shape), _ptr(amp), _ptr(dc), None, None)
    if out is None:
        out = torch.empty(nasg_rec_floats(N, K), dtype=f32, device=means.device)
    _chk(out, "params", (nasg_rec_floats(N, K),), f32, "cuda")
    rc = _lib.nasg_rec_pack(C.byref(inp), _ptr(out), _stream(stream))
    if rc != 0:
        raise NasgError(rc, "nasg_rec_pack")
    return out


def nasg_rec_unpack(rec: torch.Tensor, N: int, K: int, stream=None, out: Optional[dict] = None) -> dict:
    """Tile records (parameters or gradients) -> dict of row arrays means, quat, shape, amp, dc (written into `out` if given)."""
    f32 = torch.float32
    _chk(rec, "rec", (nasg_rec_floats(N, K),), f32, "cuda")
    dev = rec.device
    if out is None:
        out = dict(means=torch.empty((N, 3), dtype=f32, device=dev), quat=torch.empty((K, N, 4), dtype=f32, device=dev),
                   shape=torch.empty((K, N, 4), dtype=f32, device=dev), amp=torch.empty((K, 3, N), dtype=f32, device=dev),
                   dc=torch.empty((3, N), dtype=f32, device=dev))
    for name, shp in (("means", (N, 3)), ("quat", (K, N, 4)), ("shape", (K, N, 4)), ("amp", (K, 3, N)), ("dc", (3, N))):
        _chk(out[name], name, shp, f32, "cuda")
    rc = _lib.nasg_rec_unpack(N, K, _ptr(rec), _ptr(out["means"]), _ptr(out["quat"]), _ptr(out["shape"]), _ptr(out["amp"]),
                              _ptr(out["dc"]), _stream(stream))
    if rc != 0:
        raise NasgError(rc, "nasg_rec_unpack")
    return out


def _rec_inputs(params, N, K, campos, vis) -> _RecInputs:
    Cn = int(campos.shape[0])
    _chk(params, "params", (nasg_rec_floats(N, K),), torch.float32, "cuda")
    _chk(campos, "campos", (Cn, 3), torch.float32, "cuda"); _chk(vis, "vis", (Cn, N), torch.uint8, "cuda")
    return _RecInputs(N, K, Cn, _ptr(params), _ptr(campos), _ptr(vis))


def nasg_rec_eval_fwd(params, N: int, K: int, campos, vis=None, norm_mode: int = NORM_EXACT,
                      out: Optional[torch.Tensor] = None, stream=None) -> torch.Tensor:
    """colors [C,N,3] from tile-record parameters (same function as nasg_eval_fwd)."""
    inp = _rec_inputs(params, N, K, campos, vis)
    if out is None:
        out = torch.empty((inp.C, N, 3), dtype=torch.float32, device=params.device)
    _chk(out, "colors", (inp.C, N, 3), torch.float32, "cuda")
    rc = _lib.nasg_rec_eval_fwd(C.byref(inp), _ptr(out), int(norm_mode), _stream(stream))
    if rc != 0:
        raise NasgError(rc, "nasg_rec_eval_fwd")
    return out


def nasg_rec_eval_bwd(params, N: int, K: int, campos, g_colors, vis=None, norm_mode: int = NORM_EXACT,
                      out: Optional[torch.Tensor] = None, stream=None) -> torch.Tensor:
    """Gradient record array (layout of `params`) of sum(g_colors * colors)."""
    inp = _rec_inputs(params, N, K, campos, vis)
    _chk(g_colors, "g_colors", (inp.C, N, 3), torch.float32, "cuda")
    if out is None:
        out = torch.zeros(nasg_rec_floats(N, K), dtype=torch.float32, device=params.device)   # (padding lanes stay 0)
    _chk(out, "g_params", (nasg_rec_floats(N, K),), torch.float32, "cuda")
    rc = _lib.nasg_rec_eval_bwd(C.byref(inp), _ptr(g_colors), _ptr(out), int(norm_mode), _stream(stream))
    if rc != 0:
        raise NasgError(rc, "nasg_rec_eval_bwd")
    return out


def nasg_rec_host_scratch_bytes(N: int, K: int, Cn: int) -> int:
    return int(_lib.nasg_rec_host_scratch_bytes(N, K, Cn))


def nasg_paper_host_scratch_bytes(N: int, K: int, Cn: int) -> int:
    return int(_lib.nasg_paper_host_scratch_bytes(N, K, Cn))


def nasg_rec_eval_fwd_bwd_host(host: dict, host_out: dict, N: int, K: int, dev_scratch: torch.Tensor,
                               norm_mode: int = NORM_EXACT, stream=None, paper: bool = False) -> None:
    """End-to-end call with HOST tensors on the tile-record layout: ``host`` holds params (records), campos, vis (or
    None), g_colors; ``host_out`` holds colors and g_params (records). paper=True: paper-native records
    (nasg_paper_eval_fwd_bwd_host)."""
    f32 = torch.float32
    Cn = int(host["campos"].shape[0])
    nf = nasg_paper_floats(N, K) if paper else nasg_rec_floats(N, K)
    _chk(host["params"], "params", (nf,), f32, "cpu"); _chk(host["campos"], "campos", (Cn, 3), f32, "cpu")
    _chk(host.get("vis"), "vis", (Cn, N), torch.uint8, "cpu"); _chk(host["g_colors"], "g_colors", (Cn, N, 3), f32, "cpu")
    _chk(host_out["colors"], "colors", (Cn, N, 3), f32, "cpu"); _chk(host_out["g_params"], "g_params", (nf,), f32, "cpu")
    inp = _RecInputs(N, K, Cn, _ptr(host["params"]), _ptr(host["campos"]), _ptr(host.get("vis")))
    fn = _lib.nasg_paper_eval_fwd_bwd_host if paper else _lib.nasg_rec_eval_fwd_bwd_host
    rc = fn(C.byref(inp), _ptr(host["g_colors"]), _ptr(host_out["colors"]), _ptr(host_out["g_params"]), int(norm_mode), _ptr(dev_scratch),
            dev_scratch.numel() * dev_scratch.element_size(), _stream(stream))
    if rc != 0:
        raise NasgError(rc, "nasg_paper_eval_fwd_bwd_host" if paper else "nasg_rec_eval_fwd_bwd_host")


# ---- the paper's own parameter record (include/nasg.h: nasg_paper_*) ---------------------------------
def nasg_paper_floats(N: int, K: int) -> int:
    return int(_lib.nasg_paper_floats(N, K))


def nasg_paper_eval_fwd(params, N: int, K: int, campos, vis=None, norm_mode: int = NORM_EXACT,
                        out: Optional[torch.Tensor] = None, stream=None) -> torch.Tensor:
    """colors [C,N,3] from paper-native tile records (raw values; Table 8 activations applied in the kernel)."""
    Cn = int(campos.shape[0])
    _chk(params, "params", (nasg_paper_floats(N, K),), torch.float32, "cuda")
    _chk(campos, "campos", (Cn, 3), torch.float32, "cuda"); _chk(vis, "vis", (Cn, N), torch.uint8, "cuda")
    inp = _RecInputs(N, K, Cn, _ptr(params), _ptr(campos), _ptr(vis))
    if out is None:
        out = torch.empty((Cn, N, 3), dtype=torch.float32, device=params.device)
    _chk(out, "colors", (Cn, N, 3), torch.float32, "cuda")
    rc = _lib.nasg_paper_eval_fwd(C.byref(inp), _ptr(out), int(norm_mode), _stream(stream))
    if rc != 0:
        raise NasgError(rc, "nasg_paper_eval_fwd")
    return out


def nasg_paper_eval_bwd(params, N: int, K: int, campos, g_colors, vis=None, norm_mode: int = NORM_EXACT,
                        out: Optional[torch.Tensor] = None, stream=None) -> torch.Tensor:
    """Gradient record array (dL/d raw values, layout of `params`)."""
    Cn = int(campos.shape[0])
    nf = nasg_paper_floats(N, K)
    _chk(params, "params", (nf,), torch.float32, "cuda"); _chk(g_colors, "g_colors", (Cn, N, 3), torch.float32, "cuda")
    _chk(campos, "campos", (Cn, 3), torch.float32, "cuda"); _chk(vis, "vis", (Cn, N), torch.uint8, "cuda")
    inp = _RecInputs(N, K, Cn, _ptr(params), _ptr(campos), _ptr(vis))
    if out is None:
        out = torch.zeros(nf, dtype=torch.float32, device=params.device)
    _chk(out, "g_params", (nf,), torch.float32, "cuda")
    rc = _lib.nasg_paper_eval_bwd(C.byref(inp), _ptr(g_colors), _ptr(out), int(norm_mode), _stream(stream))
    if rc != 0:
        raise NasgError(rc, "nasg_paper_eval_bwd")
    return out


# ---- isotropic Table-6 functions (include/nasg.h: nasg_iso_*) ---------------------------------------
ISO_SG, ISO_BETA, ISO_CAUCHY = 0, 1, 2


def nasg_iso_floats(N: int, K: int) -> int:
    return int(_lib.nasg_iso_floats(N, K))


def nasg_iso_eval_fwd(params, N: int, K: int, campos, kind: int, vis=None, out: Optional[torch.Tensor] = None, stream=None) -> torch.Tensor:
    Cn = int(campos.shape[0])
    _chk(params, "params", (nasg_iso_floats(N, K),), torch.float32, "cuda")
    _chk(campos, "campos", (Cn, 3), torch.float32, "cuda"); _chk(vis, "vis", (Cn, N), torch.uint8, "cuda")
    inp = _RecInputs(N, K, Cn, _ptr(params), _ptr(campos), _ptr(vis))
    if out is None:
        out = torch.empty((Cn, N, 3), dtype=torch.float32, device=params.device)
    _chk(out, "colors", (Cn, N, 3), torch.float32, "cuda")
    rc = _lib.nasg_iso_eval_fwd(C.byref(inp), _ptr(out), int(kind), _stream(stream))
    if rc != 0:
        raise NasgError(rc, "nasg_iso_eval_fwd")
    return out


def nasg_iso_eval_bwd(params, N: int, K: int, campos, g_colors, kind: int, vis=None, out: Optional[torch.Tensor] = None,
                      stream=None) -> torch.Tensor:
    Cn = int(campos.shape[0])
    nf = nasg_iso_floats(N, K)
    _chk(params, "params", (nf,), torch.float32, "cuda"); _chk(g_colors, "g_colors", (Cn, N, 3), torch.float32, "cuda")
    _chk(campos, "campos", (Cn, 3), torch.float32, "cuda"); _chk(vis, "vis", (Cn, N), torch.uint8, "cuda")
    inp = _RecInputs(N, K, Cn, _ptr(params), _ptr(campos), _ptr(vis))
    if out is None:
        out = torch.zeros(nf, dtype=torch.float32, device=params.device)
    _chk(out, "g_params", (nf,), torch.float32, "cuda")
    rc = _lib.nasg_iso_eval_bwd(C.byref(inp), _ptr(g_colors), _ptr(out), int(kind), _stream(stream))
    if rc != 0:
        raise NasgError(rc, "nasg_iso_eval_bwd")
    return out


# ---- Anisotropic Spherical Gaussian of Table 6 (include/nasg.h: nasg_asg_*) -------------------------
def nasg_asg_floats(N: int, K: int) -> int:
    return int(_lib.nasg_asg_floats(N, K))


def nasg_asg_eval_fwd(params, N: int, K: int, campos, vis=None, out: Optional[torch.Tensor] = None, stream=None) -> torch.Tensor:
    Cn = int(campos.shape[0])
    _chk(params, "params", (nasg_asg_floats(N, K),), torch.float32, "cuda")
    _chk(campos, "campos", (Cn, 3), torch.float32, "cuda"); _chk(vis, "vis", (Cn, N), torch.uint8, "cuda")
    inp = _RecInputs(N, K, Cn, _ptr(params), _ptr(campos), _ptr(vis))
    if out is None:
        out = torch.empty((Cn, N, 3), dtype=torch.float32, device=params.device)
    _chk(out, "colors", (Cn, N, 3), torch.float32, "cuda")
    rc = _lib.nasg_asg_eval_fwd(C.byref(inp), _ptr(out), _stream(stream))
    if rc != 0:
        raise NasgError(rc, "nasg_asg_eval_fwd")
    return out


def nasg_asg_eval_bwd(params, N: int, K: int, campos, g_colors, vis=None, out: Optional[torch.Tensor] = None, stream=None) -> torch.Tensor:
    Cn = int(campos.shape[0])
    nf = nasg_asg_floats(N, K)
    _chk(params, "params", (nf,), torch.float32, "cuda"); _chk(g_colors, "g_colors", (Cn, N, 3), torch.float32, "cuda")
    _chk(campos, "campos", (Cn, 3), torch.float32, "cuda"); _chk(vis, "vis", (Cn, N), torch.uint8, "cuda")
    inp = _RecInputs(N, K, Cn, _ptr(params), _ptr(campos), _ptr(vis))
    if out is None:
        out = torch.zeros(nf, dtype=torch.float32, device=params.device)
    _chk(out, "g_params", (nf,), torch.float32, "cuda")
    rc = _lib.nasg_asg_eval_bwd(C.byref(inp), _ptr(g_colors), _ptr(out), _stream(stream))
    if rc != 0:
        raise NasgError(rc, "nasg_asg_eval_bwd")
    return out


# ---- bf16 parameter storage (include/nasg.h: nasg_rec16_*) ------------------------------------------
def nasg_rec16_floats(N: int, K: int) -> int:
    return int(_lib.nasg_rec16_floats(N, K))


def nasg_rec16_pack(means, quat, shape, amp, dc, out: Optional[torch.Tensor] = None, stream=None) -> torch.Tensor:
    """Row arrays -> tile records with bf16 quaternion / amplitude (round to nearest even): float32-typed word tensor."""
    K, N = int(quat.shape[0]), int(quat.shape[1])
    f32 = torch.float32
    _chk(means, "means", (N, 3), f32, "cuda"); _chk(quat, "quat", (K, N, 4), f32, "cuda")
    _chk(shape, "shape", (K, N, 4), f32, "cuda"); _chk(amp, "amp", (K, 3, N), f32, "cuda"); _chk(dc, "dc", (3, N), f32, "cuda")
    inp = _Inputs(N, K, 1, _ptr(means), _ptr(quat), _ptr(shape), _ptr(amp), _ptr(dc), None, None)
    if out is None:
        out = torch.empty(nasg_rec16_floats(N, K), dtype=f32, device=means.device)
    _chk(out, "params", (nasg_rec16_floats(N, K),), f32, "cuda")
    rc = _lib.nasg_rec16_pack(C.byref(inp), _ptr(out), _stream(stream))
    if rc != 0:
        raise NasgError(rc, "nasg_rec16_pack")
    return out


def nasg_rec16_eval_fwd(params, N: int, K: int, campos, vis=None, norm_mode: int = NORM_EXACT,
                        out: Optional[torch.Tensor] = None, stream=None) -> torch.Tensor:
    Cn = int(campos.shape[0])
    _chk(params, "params", (nasg_rec16_floats(N, K),), torch.float32, "cuda")
    _chk(campos, "campos", (Cn, 3), torch.float32, "cuda"); _chk(vis, "vis", (Cn, N), torch.uint8, "cuda")
    inp = _RecInputs(N, K, Cn, _ptr(params), _ptr(campos), _ptr(vis))
    if out is None:
        out = torch.empty((Cn, N, 3), dtype=torch.float32, device=params.device)
    _chk(out, "colors", (Cn, N, 3), torch.float32, "cuda")
    rc = _lib.nasg_rec16_eval_fwd(C.byref(inp), _ptr(out), int(norm_mode), _stream(stream))
    if rc != 0:
        raise NasgError(rc, "nasg_rec16_eval_fwd")
    return out


def nasg_rec16_eval_bwd(params, N: int, K: int, campos, g_colors, vis=None, norm_mode: int = NORM_EXACT,
                        out: Optional[torch.Tensor] = None, stream=None) -> torch.Tensor:
    """fp32 gradient record array (layout of nasg_rec_eval_bwd: nasg_rec_floats(N, K) floats)."""
    Cn = int(campos.shape[0])
    _chk(params, "params", (nasg_rec16_floats(N, K),), torch.float32, "cuda"); _chk(g_colors, "g_colors", (Cn, N, 3), torch.float32, "cuda")
    _chk(campos, "campos", (Cn, 3), torch.float32, "cuda"); _chk(vis, "vis", (Cn, N), torch.uint8, "cuda")
    inp = _RecInputs(N, K, Cn, _ptr(params), _ptr(campos), _ptr(vis))
    if out is None:
        out = torch.zeros(nasg_rec_floats(N, K), dtype=torch.float32, device=params.device)
    _chk(out, "g_params", (nasg_rec_floats(N, K),), torch.float32, "cuda")
    rc = _lib.nasg_rec16_eval_bwd(C.byref(inp), _ptr(g_colors), _ptr(out), int(norm_mode), _stream(stream))
    if rc != 0:
        raise NasgError(rc, "nasg_rec16_eval_bwd")
    return out


# ---- records of every kind from row arrays and back (include/nasg.h: nasg_kind_*) -----------------------
KIND_QUAT, KIND_PAPER, KIND_ISO, KIND_ASG = 0, 1, 2, 4


def nasg_kind_components(kind: int) -> int:
    return int(_lib.nasg_kind_components(int(kind)))


def nasg_kind_floats(kind: int, N: int, K: int) -> int:
    return int(_lib.nasg_kind_floats(int(kind), N, K))


def nasg_kind_pack(kind: int, means, dc, comp, out: Optional[torch.Tensor] = None, stream=None) -> torch.Tensor:
    """means [N,3], dc [3,N], comp [K,N,M] (the M components of every lobe in the kind's order) -> record array."""
    f32 = torch.float32
    K, N, M = (int(x) for x in comp.shape)
    _chk(means, "means", (N, 3), f32, "cuda"); _chk(dc, "dc", (3, N), f32, "cuda"); _chk(comp, "comp", (K, N, M), f32, "cuda")
    if M != nasg_kind_components(kind):
        raise ValueError(f"comp has {M} components per lobe, kind {kind} has {nasg_kind_components(kind)}")
    nf = nasg_kind_floats(kind, N, K)
    if out is None:
        out = torch.empty(nf, dtype=f32, device=means.device)
    _chk(out, "rec", (nf,), f32, "cuda")
    rc = _lib.nasg_kind_pack(int(kind), N, K, _ptr(means), _ptr(dc), _ptr(comp), _ptr(out), _stream(stream))
    if rc != 0:
        raise NasgError(rc, "nasg_kind_pack")
    return out


def nasg_kind_unpack(kind: int, rec: torch.Tensor, N: int, K: int, stream=None) -> dict:
    """Record array (parameters or gradients) of a kind -> dict means [N,3], dc [3,N], comp [K,N,M]."""
    f32 = torch.float32
    M = nasg_kind_components(kind)
    _chk(rec, "rec", (nasg_kind_floats(kind, N, K),), f32, "cuda")
    out = dict(means=torch.empty((N, 3), dtype=f32, device=rec.device), dc=torch.empty((3, N), dtype=f32, device=rec.device),
               comp=torch.empty((K, N, M), dtype=f32, device=rec.device))
    rc = _lib.nasg_kind_unpack(int(kind), N, K, _ptr(rec), _ptr(out["means"]), _ptr(out["dc"]), _ptr(out["comp"]), _stream(stream))
    if rc != 0:
        raise NasgError(rc, "nasg_kind_unpack")
    return out


def nasg_rec16_unpack(rec16: torch.Tensor, N: int, K: int, stream=None) -> dict:
    """bf16 parameter record (nasg_rec16_pack) -> fp32 row arrays means, quat, shape, amp, dc (exact)."""
    f32 = torch.float32
    _chk(rec16, "rec16", (nasg_rec16_floats(N, K),), f32, "cuda")
    dev = rec16.device
    out = dict(means=torch.empty((N, 3), dtype=f32, device=dev), quat=torch.empty((K, N, 4), dtype=f32, device=dev),
               shape=torch.empty((K, N, 4), dtype=f32, device=dev), amp=torch.empty((K, 3, N), dtype=f32, device=dev),
               dc=torch.empty((3, N), dtype=f32, device=dev))
    rc = _lib.nasg_rec16_unpack(N, K, _ptr(rec16), _ptr(out["means"]), _ptr(out["quat"]), _ptr(out["shape"]), _ptr(out["amp"]),
                                _ptr(out["dc"]), _stream(stream))
    if rc != 0:
        raise NasgError(rc, "nasg_rec16_unpack")
    return out
