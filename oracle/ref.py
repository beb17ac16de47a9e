"""ctypes loader of the fp64 CPU oracle (TEST INFRASTRUCTURE, not product code).

Builds ``oracle/liboracle_ref.so`` from ``nasg_ref.c`` + ``sh_ref.c`` with gcc (``-O2 -fopenmp``, no
``-ffast-math``) and exposes numpy wrappers. Inputs are the fp32/uint8 arrays of
``paper_2606_09794_b200.workloads`` (or fp64 arrays for finite-difference tests); they are promoted
to fp64 exactly, and every output is fp64. No arithmetic of the method happens in this file.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from typing import Optional

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = [os.path.join(_HERE, "nasg_ref.c"), os.path.join(_HERE, "sh_ref.c"), os.path.join(_HERE, "iso_ref.c"),
        os.path.join(_HERE, "asg_ref.c")]
_LIB = os.path.join(_HERE, "liboracle_ref.so")
_lib = None


def build(force: bool = False) -> str:
    """Compile the oracle with gcc if the .so is missing or older than its sources."""
    stale = force or not os.path.exists(_LIB) or any(
        os.path.getmtime(s) > os.path.getmtime(_LIB) for s in _SRC)
    if stale:
        cmd = ["gcc", "-O2", "-std=c99", "-fopenmp", "-fPIC", "-shared", "-Wall", "-Wextra",
               "-o", _LIB] + _SRC + ["-lm"]
        subprocess.run(cmd, check=True)
    return _LIB


def lib():
    global _lib
    if _lib is None:
        build()
        L = C.CDLL(_LIB)
        dp, u8p, i64, i32, dbl = C.c_void_p, C.c_void_p, C.c_int64, C.c_int, C.c_double
        L.nasg_ref_fwd.argtypes = [i64, i32, i32, dp, dp, dp, dp, dp, dp, u8p, i32, dp]
        L.nasg_ref_bwd.argtypes = [i64, i32, i32, dp, dp, dp, dp, dp, dp, u8p, dp, i32,
                                   dp, dp, dp, dp, dp, dp]
        L.sh_ref_fwd.argtypes = [i64, i32, dp, dp, dp, u8p, dp]
        L.sh_ref_bwd.argtypes = [i64, i32, dp, dp, dp, u8p, dp, dp, dp, dp]
        L.nasg_ref_integral.argtypes = [dbl, dbl, dbl, i32]
        L.nasg_ref_integral.restype = dbl
        L.nasg_ref_psi.argtypes = [dbl, dbl, dp]
        L.nasg_ref_dlnI.argtypes = [dbl, dbl, dbl, i32, dp]
        L.nasg_ref_partials.argtypes = [dbl, dbl, dbl, dbl, dbl, dbl, i32, dp]
        L.nasg_ref_frame.argtypes = [dp, dp, dp]
        L.iso_ref_lobe.argtypes = [i32, dbl, dbl, dp]
        L.iso_ref_fwd.argtypes = [i64, i32, i32, i32, dp, dp, dp, dp, dp, dp, u8p, dp]
        L.iso_ref_bwd.argtypes = [i64, i32, i32, i32, dp, dp, dp, dp, dp, dp, u8p, dp, dp, dp, dp, dp, dp]
        L.iso_ref_fwd.restype = i32
        L.iso_ref_bwd.restype = i32
        L.asg_ref_frame.argtypes = [dp, dp, dp, dp]
        L.asg_ref_lobe.argtypes = [dbl, dbl, dbl, dbl, dbl, dp]
        L.asg_ref_fwd.argtypes = [i64, i32, i32, dp, dp, dp, dp, dp, dp, u8p, dp]
        L.asg_ref_bwd.argtypes = [i64, i32, i32, dp, dp, dp, dp, dp, dp, u8p, dp, dp, dp, dp, dp, dp]
        L.nasg_ref_paper_frame.argtypes = [dp, dp, dp, dp, dp]
        L.nasg_ref_paper_fwd.argtypes = [i64, i32, i32, dp, dp, dp, dp, dp, dp, u8p, i32, dp]
        L.nasg_ref_paper_bwd.argtypes = [i64, i32, i32, dp, dp, dp, dp, dp, dp, u8p, dp, i32, dp, dp, dp, dp, dp]
        L.nasg_ref_paper_fwd.restype = i32
        L.nasg_ref_paper_bwd.restype = i32
        L.sh_ref_basis.argtypes = [dp, dp, dp]
        L.nasg_ref_num_threads.restype = i32
        L.nasg_ref_set_num_threads.argtypes = [i32]
        for f in (L.nasg_ref_fwd, L.nasg_ref_bwd, L.sh_ref_fwd, L.sh_ref_bwd):
            f.restype = i32
        _lib = L
    return _lib


def _d(a) -> np.ndarray:
    return np.ascontiguousarray(a, dtype=np.float64)


def _p(a: Optional[np.ndarray]):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def num_threads() -> int:
    return int(lib().nasg_ref_num_threads())


def set_num_threads(t: int) -> None:
    """OpenMP threads of the following calls (timing harness only)."""
    lib().nasg_ref_set_num_threads(int(t))


def nasg_fwd(inp: dict, norm_mode: int = 1) -> np.ndarray:
    """colors [C,N,3] fp64."""
    N, K, Cn = int(inp["N"]), int(inp["K"]), int(inp["C"])
    means, quat, shape, amp, dc, campos = (_d(inp[k]) for k in
                                           ("means", "quat", "shape", "amp", "dc", "campos"))
    vis = None if inp.get("vis") is None else np.ascontiguousarray(inp["vis"], dtype=np.uint8)
    colors = np.empty((Cn, N, 3), dtype=np.float64)
    rc = lib().nasg_ref_fwd(N, K, Cn, _p(means), _p(quat), _p(shape), _p(amp), _p(dc), _p(campos),
                            _p(vis), norm_mode, _p(colors))
    assert rc == 0
    return colors


def nasg_bwd(inp: dict, norm_mode: int = 1, g_colors: Optional[np.ndarray] = None) -> dict:
    """dict of fp64 gradients: g_means, g_quat, g_shape, g_amp, g_dc, g_campos."""
    N, K, Cn = int(inp["N"]), int(inp["K"]), int(inp["C"])
    means, quat, shape, amp, dc, campos = (_d(inp[k]) for k in
                                           ("means", "quat", "shape", "amp", "dc", "campos"))
    gcol = _d(inp["g_colors"] if g_colors is None else g_colors)
    vis = None if inp.get("vis") is None else np.ascontiguousarray(inp["vis"], dtype=np.uint8)
    out = dict(g_means=np.empty((N, 3)), g_quat=np.empty((K, N, 4)), g_shape=np.empty((K, N, 4)),
               g_amp=np.empty((K, 3, N)), g_dc=np.empty((3, N)), g_campos=np.empty((Cn, 3)))
    rc = lib().nasg_ref_bwd(N, K, Cn, _p(means), _p(quat), _p(shape), _p(amp), _p(dc), _p(campos),
                            _p(vis), _p(gcol), norm_mode, _p(out["g_means"]), _p(out["g_quat"]),
                            _p(out["g_shape"]), _p(out["g_amp"]), _p(out["g_dc"]), _p(out["g_campos"]))
    assert rc == 0
    return out


def sh_fwd(inp: dict) -> np.ndarray:
    N, Cn = int(inp["N"]), int(inp["C"])
    means, coeffs, campos = _d(inp["means"]), _d(inp["coeffs"]), _d(inp["campos"])
    vis = None if inp.get("vis") is None else np.ascontiguousarray(inp["vis"], dtype=np.uint8)
    colors = np.empty((Cn, N, 3), dtype=np.float64)
    rc = lib().sh_ref_fwd(N, Cn, _p(means), _p(coeffs), _p(campos), _p(vis), _p(colors))
    assert rc == 0
    return colors


def sh_bwd(inp: dict, g_colors: Optional[np.ndarray] = None) -> dict:
    N, Cn = int(inp["N"]), int(inp["C"])
    means, coeffs, campos = _d(inp["means"]), _d(inp["coeffs"]), _d(inp["campos"])
    gcol = _d(inp["g_colors"] if g_colors is None else g_colors)
    vis = None if inp.get("vis") is None else np.ascontiguousarray(inp["vis"], dtype=np.uint8)
    out = dict(g_means=np.empty((N, 3)), g_coeffs=np.empty((16, 3, N)), g_campos=np.empty((Cn, 3)))
    rc = lib().sh_ref_bwd(N, Cn, _p(means), _p(coeffs), _p(campos), _p(vis), _p(gcol),
                          _p(out["g_means"]), _p(out["g_coeffs"]), _p(out["g_campos"]))
    assert rc == 0
    return out


# ---- scalar helpers used by the pins -------------------------------------------------------
def integral(lam: float, a: float, k: float, norm_mode: int = 1) -> float:
    return float(lib().nasg_ref_integral(lam, a, k, norm_mode))


def psi(Lam: float, k: float) -> np.ndarray:
    out = np.empty(3)
    lib().nasg_ref_psi(Lam, k, _p(out))
    return out


def dlnI(lam: float, a: float, k: float, norm_mode: int = 1) -> np.ndarray:
    out = np.empty(3)
    lib().nasg_ref_dlnI(lam, a, k, norm_mode, _p(out))
    return out


def partials(u, v, lam, a, k, phi, norm_mode: int = 1) -> np.ndarray:
    """[G, G_u, G_v, G_lambda, G_a, G_k, G_phi] of one normalised lobe."""
    out = np.empty(7)
    lib().nasg_ref_partials(u, v, lam, a, k, phi, norm_mode, _p(out))
    return out


def frame(q) -> tuple:
    q = _d(q)
    X, Z = np.empty(3), np.empty(3)
    lib().nasg_ref_frame(_p(q), _p(X), _p(Z))
    return X, Z


def sh_basis(d) -> tuple:
    d = _d(d)
    Y, dY = np.empty(16), np.empty((16, 3))
    lib().sh_ref_basis(_p(d), _p(Y), _p(dY))
    return Y, dY


# ---- paper-native parameter record (Table 8 activations, Supplementary C frame) -----------------
def paper_frame(euler_raw) -> tuple:
    """X, Z and their derivatives dX[i], dZ[i] with respect to the cosines (c_theta, c_phi, c_tau), eqs.(38)-(44)."""
    e = _d(euler_raw)
    X, Z, dX, dZ = np.empty(3), np.empty(3), np.empty((3, 3)), np.empty((3, 3))
    lib().nasg_ref_paper_frame(_p(e), _p(X), _p(Z), _p(dX), _p(dZ))
    return X, Z, dX, dZ


def paper_fwd(inp: dict, norm_mode: int = 1) -> np.ndarray:
    """colors [C,N,3] fp64 from the paper-native record: inp holds means, euler [K,N,3], shp [K,N,3], ampraw [K,3,N], dc."""
    N, K, Cn = int(inp["N"]), int(inp["K"]), int(inp["C"])
    means, eu, sp, aw, dc, campos = (_d(inp[k]) for k in ("means", "euler", "shp", "ampraw", "dc", "campos"))
    vis = None if inp.get("vis") is None else np.ascontiguousarray(inp["vis"], dtype=np.uint8)
    colors = np.empty((Cn, N, 3), dtype=np.float64)
    rc = lib().nasg_ref_paper_fwd(N, K, Cn, _p(means), _p(eu), _p(sp), _p(aw), _p(dc), _p(campos), _p(vis), norm_mode, _p(colors))
    assert rc == 0
    return colors


def paper_bwd(inp: dict, norm_mode: int = 1, g_colors: Optional[np.ndarray] = None) -> dict:
    """fp64 gradients with respect to the RAW values: g_means, g_euler, g_shp, g_ampraw, g_dc."""
    N, K, Cn = int(inp["N"]), int(inp["K"]), int(inp["C"])
    means, eu, sp, aw, dc, campos = (_d(inp[k]) for k in ("means", "euler", "shp", "ampraw", "dc", "campos"))
    gcol = _d(inp["g_colors"] if g_colors is None else g_colors)
    vis = None if inp.get("vis") is None else np.ascontiguousarray(inp["vis"], dtype=np.uint8)
    out = dict(g_means=np.empty((N, 3)), g_euler=np.empty((K, N, 3)), g_shp=np.empty((K, N, 3)),
               g_ampraw=np.empty((K, 3, N)), g_dc=np.empty((3, N)))
    rc = lib().nasg_ref_paper_bwd(N, K, Cn, _p(means), _p(eu), _p(sp), _p(aw), _p(dc), _p(campos), _p(vis), _p(gcol), norm_mode,
                                  _p(out["g_means"]), _p(out["g_euler"]), _p(out["g_shp"]), _p(out["g_ampraw"]), _p(out["g_dc"]))
    assert rc == 0
    return out


# ---- isotropic Table-6 functions (oracle/iso_ref.c): kind 0 = Spherical Gaussian, 1 = Spherical Beta, 2 = Spherical Cauchy
def iso_lobe(kind: int, v: float, raw: float) -> np.ndarray:
    """[F, dF/dv, dF/draw] of one normalised lobe F = c G at v = z.d."""
    out = np.empty(3)
    lib().iso_ref_lobe(int(kind), float(v), float(raw), _p(out))
    return out


def iso_fwd(inp: dict, kind: int) -> np.ndarray:
    """colors [C,N,3] fp64; inp holds means, axis [K,N,3], shp [K,N], amp [K,3,N], dc, campos, vis."""
    N, K, Cn = int(inp["N"]), int(inp["K"]), int(inp["C"])
    means, ax, sp, am, dc, campos = (_d(inp[k]) for k in ("means", "axis", "shp", "amp", "dc", "campos"))
    vis = None if inp.get("vis") is None else np.ascontiguousarray(inp["vis"], dtype=np.uint8)
    colors = np.empty((Cn, N, 3), dtype=np.float64)
    rc = lib().iso_ref_fwd(N, K, Cn, int(kind), _p(means), _p(ax), _p(sp), _p(am), _p(dc), _p(campos), _p(vis), _p(colors))
    assert rc == 0
    return colors


def iso_bwd(inp: dict, kind: int, g_colors: Optional[np.ndarray] = None) -> dict:
    N, K, Cn = int(inp["N"]), int(inp["K"]), int(inp["C"])
    means, ax, sp, am, dc, campos = (_d(inp[k]) for k in ("means", "axis", "shp", "amp", "dc", "campos"))
    gcol = _d(inp["g_colors"] if g_colors is None else g_colors)
    vis = None if inp.get("vis") is None else np.ascontiguousarray(inp["vis"], dtype=np.uint8)
    out = dict(g_means=np.empty((N, 3)), g_axis=np.empty((K, N, 3)), g_shp=np.empty((K, N)), g_amp=np.empty((K, 3, N)), g_dc=np.empty((3, N)))
    rc = lib().iso_ref_bwd(N, K, Cn, int(kind), _p(means), _p(ax), _p(sp), _p(am), _p(dc), _p(campos), _p(vis), _p(gcol),
                           _p(out["g_means"]), _p(out["g_axis"]), _p(out["g_shp"]), _p(out["g_amp"]), _p(out["g_dc"]))
    assert rc == 0
    return out


# ---- Anisotropic Spherical Gaussian of Table 6 (oracle/asg_ref.c)
def asg_frame(q) -> tuple:
    """Columns (x, y, z) of R(q/|q|), q = (w,x,y,z)."""
    q = _d(np.asarray(q, dtype=np.float64))
    X, Y, Z = np.empty(3), np.empty(3), np.empty(3)
    lib().asg_ref_frame(_p(q), _p(X), _p(Y), _p(Z))
    return X, Y, Z


def asg_lobe(u: float, t: float, v: float, raw_mu: float, raw_lam: float) -> np.ndarray:
    """[G, G_u, G_t, G_v, G_rawmu, G_rawlambda] at (u, t, v) = (d.x, d.y, d.z)."""
    out = np.empty(6)
    lib().asg_ref_lobe(float(u), float(t), float(v), float(raw_mu), float(raw_lam), _p(out))
    return out


def asg_fwd(inp: dict) -> np.ndarray:
    """colors [C,N,3] fp64; inp holds means, quat [K,N,4], shp [K,N,2] (raw mu, raw lambda), amp [K,3,N], dc, campos, vis."""
    N, K, Cn = int(inp["N"]), int(inp["K"]), int(inp["C"])
    means, qu, sp, am, dc, campos = (_d(inp[k]) for k in ("means", "quat", "shp", "amp", "dc", "campos"))
    vis = None if inp.get("vis") is None else np.ascontiguousarray(inp["vis"], dtype=np.uint8)
    colors = np.empty((Cn, N, 3), dtype=np.float64)
    rc = lib().asg_ref_fwd(N, K, Cn, _p(means), _p(qu), _p(sp), _p(am), _p(dc), _p(campos), _p(vis), _p(colors))
    assert rc == 0
    return colors


def asg_bwd(inp: dict, g_colors: Optional[np.ndarray] = None) -> dict:
    N, K, Cn = int(inp["N"]), int(inp["K"]), int(inp["C"])
    means, qu, sp, am, dc, campos = (_d(inp[k]) for k in ("means", "quat", "shp", "amp", "dc", "campos"))
    gcol = _d(inp["g_colors"] if g_colors is None else g_colors)
    vis = None if inp.get("vis") is None else np.ascontiguousarray(inp["vis"], dtype=np.uint8)
    out = dict(g_means=np.empty((N, 3)), g_quat=np.empty((K, N, 4)), g_shp=np.empty((K, N, 2)), g_amp=np.empty((K, 3, N)), g_dc=np.empty((3, N)))
    rc = lib().asg_ref_bwd(N, K, Cn, _p(means), _p(qu), _p(sp), _p(am), _p(dc), _p(campos), _p(vis), _p(gcol),
                           _p(out["g_means"]), _p(out["g_quat"]), _p(out["g_shp"]), _p(out["g_amp"]), _p(out["g_dc"]))
    assert rc == 0
    return out
