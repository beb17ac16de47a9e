"""Seeded synthetic workloads (the five BASELINE.json configs).

This module holds NO arithmetic of the method: it only draws the random inputs that both the
CUDA path and the independent fp64 oracle consume (SURVEY.md section
8(d)). Every array is drawn from its own PCG64 sub-stream ``default_rng([seed, tag])`` and cast to
fp32 (uint8 for the mask) before either implementation sees it.

Shapes follow the boundary in ``include/nasg.h``:
  means [N,3] · quat [K,N,4] (w,x,y,z) · shape [K,N,4] = (log Lambda, log lambda, k, phi)
  amp [K,3,N] · dc [3,N] · campos [C,3] · vis [C,N] uint8 or None · g_colors [C,N,3]
  SH: coeffs [16,3,N]
"""
from __future__ import annotations

from dataclasses import dataclass
from typing import Optional

import numpy as np

# sub-stream tags (one independent stream per array)
TAG_MEANS, TAG_CAMPOS, TAG_VIS, TAG_QUAT, TAG_BW, TAG_FREQ, TAG_PHASE = 0, 1, 2, 3, 4, 5, 6
TAG_AMP, TAG_DC, TAG_GCOL, TAG_SH, TAG_EULER = 7, 8, 9, 10, 11


@dataclass(frozen=True)
class Config:
    """One BASELINE.json config. ``kind`` is "nasg" or "sh"."""
    index: int
    kind: str
    seed: int
    N: int
    K: int            # lobes (0 for SH)
    C: int            # cameras
    fixed_campos: bool
    vis_p: Optional[float]      # Bernoulli probability, None = all visible (vis pointer NULL)
    bw_range: tuple             # log-bandwidth range
    k_range: tuple              # Gabor frequency range
    name: str


CONFIGS = (
    Config(0, "nasg", 0, 10_000, 2, 1, True, None, (0.0, 5.0), (0.0, 8.0), "cfg0 N=1e4 K=2 C=1"),
    Config(1, "nasg", 1, 1_000_000, 4, 1, False, None, (0.0, 5.0), (0.0, 8.0), "cfg1 N=1e6 K=4 C=1"),
    Config(2, "nasg", 2, 3_000_000, 4, 4, False, 0.6, (0.0, 5.0), (0.0, 8.0),
           "cfg2 N=3e6 K=4 C=4 vis~Bern(0.6)"),
    Config(3, "sh", 2, 3_000_000, 0, 4, False, 0.6, (0.0, 5.0), (0.0, 8.0),
           "cfg3 SH-3 N=3e6 C=4 vis~Bern(0.6)"),
    Config(4, "nasg", 4, 6_000_000, 8, 1, False, None, (3.0, 8.0), (4.0, 16.0),
           "cfg4 N=6e6 K=8 C=1 high-frequency"),
)


def _rng(seed: int, tag: int) -> np.random.Generator:
    return np.random.Generator(np.random.PCG64([seed, tag]))


def make_geometry(cfg: Config, N: Optional[int] = None, vis_cluster: int = 1) -> dict:
    """means, campos, vis, g_colors: the arrays config 3 shares with config 2 (same seed/tags). vis_cluster > 1: the
    Bernoulli draw is per (camera, run of vis_cluster consecutive Gaussians) instead of per (camera, Gaussian): the
    spatially coherent visibility of a scene stored in spatial order, where frustum culling removes whole runs (a labelled
    variant; the BASELINE configs use vis_cluster = 1, iid, the pessimistic case)."""
    N = cfg.N if N is None else int(N)
    C = cfg.C
    means = _rng(cfg.seed, TAG_MEANS).uniform(-1.0, 1.0, size=(N, 3)).astype(np.float32)
    if cfg.fixed_campos:
        campos = np.array([[0.0, 0.0, 4.0]], dtype=np.float32)
    else:
        g = _rng(cfg.seed, TAG_CAMPOS).standard_normal(size=(C, 3))
        campos = (4.0 * g / np.linalg.norm(g, axis=1, keepdims=True)).astype(np.float32)
    if cfg.vis_p is None:
        vis = None
    else:
        if vis_cluster > 1:
            runs = (N + vis_cluster - 1) // vis_cluster
            vis = np.repeat((_rng(cfg.seed, TAG_VIS).random(size=(C, runs)) < cfg.vis_p).astype(np.uint8), vis_cluster, axis=1)[:, :N]
            vis = np.ascontiguousarray(vis)
        else:
            vis = (_rng(cfg.seed, TAG_VIS).random(size=(C, N)) < cfg.vis_p).astype(np.uint8)
    g_colors = _rng(cfg.seed, TAG_GCOL).standard_normal(size=(C, N, 3)).astype(np.float32)
    return dict(N=N, C=C, means=means, campos=campos, vis=vis, g_colors=g_colors)


def make_nasg(cfg: Config, N: Optional[int] = None, vis_cluster: int = 1) -> dict:
    """Inputs of nasg_eval_fwd/bwd for a NASGabor config."""
    assert cfg.kind == "nasg"
    out = make_geometry(cfg, N, vis_cluster)
    N, K = out["N"], cfg.K
    q = _rng(cfg.seed, TAG_QUAT).standard_normal(size=(K, N, 4))
    q /= np.linalg.norm(q, axis=2, keepdims=True)
    b = _rng(cfg.seed, TAG_BW).uniform(cfg.bw_range[0], cfg.bw_range[1], size=(K, N, 2))
    shape = np.empty((K, N, 4), dtype=np.float64)
    shape[..., 0] = b.max(axis=2)      # log Lambda: first bandwidth (>= second)
    shape[..., 1] = b.min(axis=2)      # log lambda
    shape[..., 2] = _rng(cfg.seed, TAG_FREQ).uniform(cfg.k_range[0], cfg.k_range[1], size=(K, N))
    shape[..., 3] = _rng(cfg.seed, TAG_PHASE).uniform(0.0, 2.0 * np.pi, size=(K, N))
    amp = _rng(cfg.seed, TAG_AMP).normal(0.0, 0.3, size=(K, 3, N))
    dc = _rng(cfg.seed, TAG_DC).normal(0.0, 0.3, size=(3, N))
    out.update(K=K, quat=q.astype(np.float32), shape=shape.astype(np.float32),
               amp=amp.astype(np.float32), dc=dc.astype(np.float32))
    return out


def make_paper(cfg: Config, N: Optional[int] = None, mirror_cameras: bool = True) -> dict:
    """The same config with the paper-native parameter record (include/nasg.h: nasg_paper_*; Table 8): RAW
    (pre-activation) values, drawn directly so that this module applies no activation: euler [K,N,3] ~ U[-1.8,1.8]
    (cosines tanh(raw) in +-0.947), shp [K,N,3] = (lambda_raw = the smaller of the two log-bandwidth draws, a_raw = their
    difference - 0.5, k_raw ~ U[-2.5,-0.7], i.e. k in [0.3,7.9]; the high-frequency config U[-1.1,-0.2], k in [4,16]),
    ampraw ~ N(0,0.3), dc ~ N(0,0.3); geometry, masks and g_colors as make_nasg, except that every camera is mirrored
    into the y <= 0 half-space: with sin = +sqrt(1 - cos^2) the record's lobe axes z = (c s, s s, c) all have z_y >= 0
    (SURVEY.md NEXT-2 "quirk"), so only view directions d = normalize(mean - campos) with d_y > 0 can
    meet a lobe peak; a camera on the other side would see nothing but lobe tails. mirror_cameras=False keeps the
    cameras as drawn (on both sides), the labelled variant test_paper_unmirrored_cameras runs."""
    assert cfg.kind == "nasg"
    out = make_geometry(cfg, N)
    if mirror_cameras:
        out["campos"] = out["campos"].copy()
        out["campos"][:, 1] = -np.abs(out["campos"][:, 1])
    N, K = out["N"], cfg.K
    euler = _rng(cfg.seed, TAG_EULER).uniform(-1.8, 1.8, size=(K, N, 3))
    b = _rng(cfg.seed, TAG_BW).uniform(cfg.bw_range[0], cfg.bw_range[1], size=(K, N, 2))
    kr = (-2.5, -0.7) if cfg.k_range[1] <= 8.0 else (-1.1, -0.2)
    shp = np.empty((K, N, 3), dtype=np.float64)
    shp[..., 0] = b.min(axis=2)
    shp[..., 1] = b.max(axis=2) - b.min(axis=2) - 0.5
    shp[..., 2] = _rng(cfg.seed, TAG_FREQ).uniform(kr[0], kr[1], size=(K, N))
    ampraw = _rng(cfg.seed, TAG_AMP).normal(0.0, 0.3, size=(K, 3, N))
    dc = _rng(cfg.seed, TAG_DC).normal(0.0, 0.3, size=(3, N))
    out.update(K=K, euler=euler.astype(np.float32), shp=shp.astype(np.float32), ampraw=ampraw.astype(np.float32),
               dc=dc.astype(np.float32))
    return out


def make_iso(cfg: Config, N: Optional[int] = None) -> dict:
    """The same config for the isotropic Table-6 functions (include/nasg.h: nasg_iso_*): axis [K,N,3] ~ N(0,1)^3 scaled by
    U[0.5,2] (unnormalised on purpose), shp [K,N] raw ~ U[0, 4.5] (lambda, beta = e^raw in [1, 90]; rho = sigmoid in
    [0.5, 0.989]), amp ~ N(0,0.3), dc ~ N(0,0.3); geometry, masks and g_colors as make_nasg."""
    assert cfg.kind == "nasg"
    out = make_geometry(cfg, N)
    N, K = out["N"], cfg.K
    r = _rng(cfg.seed, TAG_QUAT)
    axis = r.standard_normal(size=(K, N, 3)) * r.uniform(0.5, 2.0, size=(K, N, 1))
    shp = _rng(cfg.seed, TAG_BW).uniform(0.0, 4.5, size=(K, N))
    amp = _rng(cfg.seed, TAG_AMP).normal(0.0, 0.3, size=(K, 3, N))
    dc = _rng(cfg.seed, TAG_DC).normal(0.0, 0.3, size=(3, N))
    out.update(K=K, axis=axis.astype(np.float32), shp=shp.astype(np.float32), amp=amp.astype(np.float32), dc=dc.astype(np.float32))
    return out


def make_asg(cfg: Config, N: Optional[int] = None) -> dict:
    """The same config for the Anisotropic Spherical Gaussian of Table 6 (include/nasg.h: nasg_asg_*): quat [K,N,4] ~ N(0,1)^4
    scaled by U[0.5,2] (unnormalised on purpose), shp [K,N,2] = (raw mu, raw lambda) ~ U[-1, 4.5] (bandwidths e^raw in
    [0.37, 90]), amp ~ N(0,0.3), dc ~ N(0,0.3); geometry, masks and g_colors as make_nasg."""
    assert cfg.kind == "nasg"
    out = make_geometry(cfg, N)
    N, K = out["N"], cfg.K
    r = _rng(cfg.seed, TAG_QUAT)
    quat = r.standard_normal(size=(K, N, 4)) * r.uniform(0.5, 2.0, size=(K, N, 1))
    shp = _rng(cfg.seed, TAG_BW).uniform(-1.0, 4.5, size=(K, N, 2))
    amp = _rng(cfg.seed, TAG_AMP).normal(0.0, 0.3, size=(K, 3, N))
    dc = _rng(cfg.seed, TAG_DC).normal(0.0, 0.3, size=(3, N))
    out.update(K=K, quat=quat.astype(np.float32), shp=shp.astype(np.float32), amp=amp.astype(np.float32), dc=dc.astype(np.float32))
    return out


def make_sh(cfg: Config, N: Optional[int] = None) -> dict:
    """Inputs of sh_eval_fwd/bwd (config 3): geometry of config 2 plus degree-3 coefficients."""
    assert cfg.kind == "sh"
    out = make_geometry(cfg, N)
    N = out["N"]
    coeffs = _rng(cfg.seed, TAG_SH).normal(0.0, 0.2, size=(16, 3, N))
    coeffs[0] += 0.5                   # DC band ~ N(0.5, 0.2)
    out.update(coeffs=coeffs.astype(np.float32))
    return out


def make(cfg_index: int, N: Optional[int] = None) -> dict:
    cfg = CONFIGS[cfg_index]
    return make_nasg(cfg, N) if cfg.kind == "nasg" else make_sh(cfg, N)


def take(inp: dict, idx: np.ndarray) -> dict:
    """Gather a subset of Gaussians (per-Gaussian independent path): used to check sampled
    outputs of a full-size run against the oracle."""
    idx = np.asarray(idx, dtype=np.int64)
    out = dict(inp)
    out["N"] = int(idx.size)
    out["means"] = np.ascontiguousarray(inp["means"][idx])
    out["g_colors"] = np.ascontiguousarray(inp["g_colors"][:, idx])
    if inp.get("vis") is not None:
        out["vis"] = np.ascontiguousarray(inp["vis"][:, idx])
    for key in ("quat", "shape"):
        if key in inp:
            out[key] = np.ascontiguousarray(inp[key][:, idx])
    for key in ("amp", "coeffs"):
        if key in inp:
            out[key] = np.ascontiguousarray(inp[key][:, :, idx])
    if "dc" in inp:
        out["dc"] = np.ascontiguousarray(inp["dc"][:, idx])
    return out


# ---- tile-record layout (include/nasg.h "layout v2"): pure re-ordering, no arithmetic ----------------
REC_TILE = 32


def rec_floats(N: int, K: int) -> int:
    return ((N + REC_TILE - 1) // REC_TILE) * REC_TILE * (6 + 11 * K)


def _pack(means, dc, comp) -> np.ndarray:
    """means [N,3], dc [3,N], comp [K,N,M] (the M per-lobe components) -> float32 [T, 6 + M K, 32] flattened."""
    K, N, M = comp.shape
    assert K % 2 == 0
    T = (N + REC_TILE - 1) // REC_TILE
    Np = T * REC_TILE
    rec = np.empty((T, 6 + M * K, REC_TILE), dtype=np.float32)
    rec[:, 0:3, :] = np.pad(means, ((0, Np - N), (0, 0))).reshape(T, REC_TILE, 3).transpose(0, 2, 1)
    rec[:, 3:6, :] = np.pad(dc, ((0, 0), (0, Np - N))).reshape(3, T, REC_TILE).transpose(1, 0, 2)
    comp = np.pad(comp, ((0, 0), (0, Np - N), (0, 0)))
    # [K/2, 2, T, 32, M] -> [T, K/2, M, 32, 2]
    comp = comp.reshape(K // 2, 2, T, REC_TILE, M).transpose(2, 0, 4, 3, 1)
    rec[:, 6:, :] = comp.reshape(T, (K // 2) * M * 2, REC_TILE)
    return rec.reshape(-1)


def _unpack(rec, N: int, K: int, M: int):
    T = (N + REC_TILE - 1) // REC_TILE
    rec = np.asarray(rec).reshape(T, 6 + M * K, REC_TILE)
    means = rec[:, 0:3, :].transpose(0, 2, 1).reshape(T * REC_TILE, 3)[:N]
    dc = rec[:, 3:6, :].transpose(1, 0, 2).reshape(3, T * REC_TILE)[:, :N]
    comp = rec[:, 6:, :].reshape(T, K // 2, M, REC_TILE, 2).transpose(1, 4, 0, 3, 2).reshape(K, T * REC_TILE, M)[:, :N]
    return np.ascontiguousarray(means), np.ascontiguousarray(dc), comp


def pack_records(means, quat, shape, amp, dc) -> np.ndarray:
    """Row arrays -> float32 [T, 6 + 11 K, 32] records flattened (K even). Padding lanes: unit quaternion, zeros."""
    N = quat.shape[1]
    rec = _pack(means, dc, np.concatenate([quat, shape, amp.transpose(0, 2, 1)], axis=2))
    if N % REC_TILE:
        K = quat.shape[0]
        r = rec.reshape(-1, 6 + 11 * K, REC_TILE)
        r[-1, 6:].reshape(K // 2, 11, REC_TILE, 2)[:, 0, N % REC_TILE:, :] = 1.0       # quaternion w of the padding lanes
    return rec


def unpack_records(rec: np.ndarray, N: int, K: int) -> dict:
    """Inverse of pack_records (also for gradient records): dict means, quat, shape, amp, dc."""
    means, dc, comp = _unpack(rec, N, K, 11)
    return dict(means=means, dc=dc, quat=np.ascontiguousarray(comp[..., 0:4]), shape=np.ascontiguousarray(comp[..., 4:8]),
                amp=np.ascontiguousarray(comp[..., 8:11].transpose(0, 2, 1)))


def paper_rec_floats(N: int, K: int) -> int:
    return ((N + REC_TILE - 1) // REC_TILE) * REC_TILE * (6 + 9 * K)


def pack_paper_records(means, euler, shp, ampraw, dc) -> np.ndarray:
    """Paper-native record (3 + 9 K appearance floats per Gaussian) as tile records
    float32 [T, 6 + 9 K, 32]: per lobe the components (theta, phi, tau, lambda, a, k, w_r, w_g, w_b), all RAW."""
    return _pack(means, dc, np.concatenate([euler, shp, ampraw.transpose(0, 2, 1)], axis=2))


def unpack_paper_records(rec: np.ndarray, N: int, K: int) -> dict:
    means, dc, comp = _unpack(rec, N, K, 9)
    return dict(means=means, dc=dc, euler=np.ascontiguousarray(comp[..., 0:3]), shp=np.ascontiguousarray(comp[..., 3:6]),
                ampraw=np.ascontiguousarray(comp[..., 6:9].transpose(0, 2, 1)))


def iso_rec_floats(N: int, K: int) -> int:
    return ((N + REC_TILE - 1) // REC_TILE) * REC_TILE * (6 + 7 * K)


def pack_iso_records(means, axis, shp, amp, dc) -> np.ndarray:
    """Isotropic Table-6 lobes as tile records float32 [T, 6 + 7 K, 32]: per lobe (axis x, y, z, shape raw, w_r, w_g, w_b).
    Padding lanes get the axis (0, 0, 1) so that nothing divides by zero in lanes that are never stored."""
    N = axis.shape[1]
    rec = _pack(means, dc, np.concatenate([axis, shp[..., None], amp.transpose(0, 2, 1)], axis=2))
    if N % REC_TILE:
        K = axis.shape[0]
        r = rec.reshape(-1, 6 + 7 * K, REC_TILE)
        r[-1, 6:].reshape(K // 2, 7, REC_TILE, 2)[:, 2, N % REC_TILE:, :] = 1.0
    return rec


def unpack_iso_records(rec: np.ndarray, N: int, K: int) -> dict:
    means, dc, comp = _unpack(rec, N, K, 7)
    return dict(means=means, dc=dc, axis=np.ascontiguousarray(comp[..., 0:3]), shp=np.ascontiguousarray(comp[..., 3]),
                amp=np.ascontiguousarray(comp[..., 4:7].transpose(0, 2, 1)))


def asg_rec_floats(N: int, K: int) -> int:
    return ((N + REC_TILE - 1) // REC_TILE) * REC_TILE * (6 + 9 * K)


def pack_asg_records(means, quat, shp, amp, dc) -> np.ndarray:
    """Anisotropic Spherical Gaussian lobes as tile records float32 [T, 6 + 9 K, 32]: per lobe (q_w, q_x, q_y, q_z, raw mu,
    raw lambda, w_r, w_g, w_b). Padding lanes get the unit quaternion."""
    N = quat.shape[1]
    rec = _pack(means, dc, np.concatenate([quat, shp, amp.transpose(0, 2, 1)], axis=2))
    if N % REC_TILE:
        K = quat.shape[0]
        r = rec.reshape(-1, 6 + 9 * K, REC_TILE)
        r[-1, 6:].reshape(K // 2, 9, REC_TILE, 2)[:, 0, N % REC_TILE:, :] = 1.0
    return rec


def unpack_asg_records(rec: np.ndarray, N: int, K: int) -> dict:
    means, dc, comp = _unpack(rec, N, K, 9)
    return dict(means=means, dc=dc, quat=np.ascontiguousarray(comp[..., 0:4]), shp=np.ascontiguousarray(comp[..., 4:6]),
                amp=np.ascontiguousarray(comp[..., 6:9].transpose(0, 2, 1)))


# ---- bf16 parameter storage (include/nasg.h: nasg_rec16_*): quaternion and amplitude as bfloat16, the rest fp32 -------
def to_bf16(a: np.ndarray) -> np.ndarray:
    """Round an fp32 array to bfloat16 (round to nearest even) and return it as fp32: the values a bf16 record holds.
    A NaN stays a NaN (sign and upper payload kept, quiet bit set): the rounding increment must not carry a NaN whose low
    mantissa bits are set out of the exponent field into +-0. Infinities stay infinities; a finite value beyond the largest
    bf16 rounds to infinity. The pack kernel (nasg_rec16_pack) does the same, bit for bit."""
    u = np.ascontiguousarray(a, dtype=np.float32).view(np.uint32).astype(np.uint64)
    nan = (u & 0x7FFFFFFF) > 0x7F800000
    r = (u + 0x7FFF + ((u >> 16) & 1)) & 0xFFFF0000
    r = np.where(nan, (u & 0xFFFF0000) | 0x00400000, r)
    return r.astype(np.uint32).view(np.float32).reshape(np.shape(a))


def rec16_words(N: int, K: int) -> int:
    """32-bit words of a bf16 record array: header 192 words, 480 words per lobe pair (4 x 32 quat pairs, 4 x 64 shape, 3 x 32 amp pairs)."""
    return ((N + REC_TILE - 1) // REC_TILE) * (192 + 480 * (K // 2))


def pack_records16(means, quat, shape, amp, dc) -> np.ndarray:
    """Tile records with bf16 quaternion / amplitude: uint32 words [T, 192 + 480 K/2]. Per pair: quat component c at words
    [32 c + lane] = (bf16 of lobe 2j) | (bf16 of lobe 2j+1) << 16; shape component c at [128 + 64 c + 2 lane + h] (fp32);
    amplitude c at [384 + 32 c + lane] (bf16 pair). quat and amp must already be bf16-representable (to_bf16)."""
    K, N = quat.shape[0], quat.shape[1]
    T = (N + REC_TILE - 1) // REC_TILE
    Np = T * REC_TILE
    full = pack_records(means, quat, shape, amp, dc).view(np.uint32).reshape(T, 6 + 11 * K, REC_TILE)   # fp32 records (padding: unit q)
    out = np.empty((T, 192 + 480 * (K // 2)), dtype=np.uint32)
    out[:, :192] = full[:, :6].reshape(T, 192)
    pairs = full[:, 6:].reshape(T, K // 2, 11, REC_TILE, 2)
    for j in range(K // 2):
        base = 192 + 480 * j
        for c in range(4):
            w = pairs[:, j, c]
            out[:, base + 32 * c: base + 32 * c + 32] = (w[..., 0] >> 16) | (w[..., 1] & 0xFFFF0000)
        out[:, base + 128: base + 384] = pairs[:, j, 4:8].reshape(T, 256)
        for c in range(3):
            w = pairs[:, j, 8 + c]
            out[:, base + 384 + 32 * c: base + 384 + 32 * c + 32] = (w[..., 0] >> 16) | (w[..., 1] & 0xFFFF0000)
    return out.reshape(-1)
