"""Multi-process CPU tests (gloo, world_size 2) of the N > 1 path's host logic
(`paper_2606_09794_b200/sharding.py`): contiguous N-shards with no data-path collective, one
all-reduce for `g_campos`, max-over-ranks timing. The per-shard arithmetic is done by the fp64
oracle here (tests may call it); on the GPU box the same logic runs with the CUDA kernels and NCCL."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2606_09794_b200 import sharding as S
from paper_2606_09794_b200 import workloads as W


def test_shard_ranges_partition_exactly():
    for n_total in (0, 1, 7, 10_000, 3_000_000, 3_000_001):
        for world in (1, 2, 3, 4, 8):
            ranges = [S.shard_range(n_total, r, world) for r in range(world)]
            assert ranges[0][0] == 0 and ranges[-1][1] == n_total
            assert all(ranges[i][1] == ranges[i + 1][0] for i in range(world - 1))
            sizes = [e - b for b, e in ranges]
            assert max(sizes) - min(sizes) <= 1
    with pytest.raises(ValueError):
        S.shard_range(10, 2, 2)


def test_weak_scaling_configs_are_distinct_and_rank0_is_the_workload():
    cfg = W.CONFIGS[2]
    assert S.weak_scaling_config(cfg, 0) == cfg
    a = W.make_nasg(S.weak_scaling_config(cfg, 0), 64)
    b = W.make_nasg(S.weak_scaling_config(cfg, 1), 64)
    assert not np.array_equal(a["means"], b["means"])


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank: int, world: int, port: int, out_dir: str):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        from oracle import ref
        inp = W.make(2, 2001)                                    # cfg2 recipe: K=4, C=4, Bernoulli mask
        mine = S.shard_inputs(inp, rank, world)
        col = ref.nasg_fwd(mine, 1)
        g = ref.nasg_bwd(mine, 1)
        gcam = torch.from_numpy(g["g_campos"].copy())
        S.allreduce_g_campos(gcam)                               # the path's only collective
        t = S.max_over_ranks(10.0 + rank)
        b, e = S.shard_range(inp["N"], rank, world)
        np.savez(os.path.join(out_dir, f"rank{rank}.npz"), colors=col, g_means=g["g_means"], g_quat=g["g_quat"],
                 g_campos=gcam.numpy(), t=t, b=b, e=e)
    finally:
        dist.destroy_process_group()


def test_two_rank_shards_reproduce_the_single_process_result(tmp_path):
    world, port = 2, _free_port()
    mp.spawn(_worker, args=(world, port, str(tmp_path)), nprocs=world, join=True)
    from oracle import ref
    inp = W.make(2, 2001)
    col, g = ref.nasg_fwd(inp, 1), ref.nasg_bwd(inp, 1)
    parts = [np.load(tmp_path / f"rank{r}.npz") for r in range(world)]
    assert [int(p["b"]) for p in parts] == [0, 1001] and int(parts[1]["e"]) == 2001
    np.testing.assert_array_equal(np.concatenate([p["colors"] for p in parts], axis=1), col)      # no exchange needed
    np.testing.assert_array_equal(np.concatenate([p["g_means"] for p in parts], axis=0), g["g_means"])
    np.testing.assert_array_equal(np.concatenate([p["g_quat"] for p in parts], axis=1), g["g_quat"])
    for p in parts:                                               # every rank holds the full sum after the all-reduce
        np.testing.assert_allclose(p["g_campos"], g["g_campos"], rtol=1e-12, atol=1e-14)
        assert float(p["t"]) == 11.0                              # max over ranks
