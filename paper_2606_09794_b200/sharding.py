"""Multi-GPU plumbing of the path.

The path shards naturally: Gaussians are independent, so every rank owns a contiguous N-range and
runs the same two kernels on it with no data-path collective. `campos` is replicated. The only
quantity that crosses shards is the optional per-camera gradient `g_campos[C,3]`, a sum over all
Gaussians: one all-reduce of 3*C floats. This module holds that host logic and nothing of the
method's arithmetic; it works with any torch.distributed backend (NCCL on the GPUs, gloo in the CPU
tests).
"""
from __future__ import annotations

import dataclasses
from typing import Tuple

import torch
import torch.distributed as dist


def shard_range(n_total: int, rank: int, world: int) -> Tuple[int, int]:
    """Contiguous [begin, end) range of rank `rank`: sizes differ by at most one, begin of every
    shard except possibly the last few is a multiple of 4 when n_total // world is (so the packed
    kernels keep their 4-byte aligned visibility rows)."""
    if not (0 <= rank < world):
        raise ValueError("rank out of range")
    base, rem = divmod(int(n_total), int(world))
    begin = rank * base + min(rank, rem)
    return begin, begin + base + (1 if rank < rem else 0)


def shard_inputs(inp: dict, rank: int, world: int) -> dict:
    """Slice a workload dict (numpy arrays, layouts of include/nasg.h) to this rank's N-range."""
    b, e = shard_range(inp["N"], rank, world)
    out = dict(inp)
    out["N"] = e - b
    out["means"] = inp["means"][b:e]
    out["g_colors"] = inp["g_colors"][:, b:e]
    if inp.get("vis") is not None:
        out["vis"] = inp["vis"][:, b:e]
    for key in ("quat", "shape"):
        if key in inp:
            out[key] = inp[key][:, b:e]
    for key in ("amp", "coeffs"):
        if key in inp:
            out[key] = inp[key][:, :, b:e]
    if "dc" in inp:
        out["dc"] = inp["dc"][:, b:e]
    return out


def weak_scaling_config(cfg, rank: int):
    """bench.py's weak-scaling recipe: every rank draws its own shard of the config's size from
    seed + 1000 * rank (rank 0 is the single-GPU workload itself)."""
    return dataclasses.replace(cfg, seed=cfg.seed + 1000 * rank)


def world_size() -> int:
    return dist.get_world_size() if dist.is_available() and dist.is_initialized() else 1


def allreduce_g_campos(g_campos: torch.Tensor) -> torch.Tensor:
    """Sum the per-shard `g_campos[C,3]` over all ranks, in place (no-op for one process)."""
    if world_size() > 1:
        dist.all_reduce(g_campos, op=dist.ReduceOp.SUM)
    return g_campos


def max_over_ranks(value: float, device="cpu") -> float:
    """Max of a per-rank scalar (the device-timed milliseconds of bench.py)."""
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    if world_size() > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())
