"""Multi-GPU plumbing for the sample-sharded likelihood.

The path shards over SAMPLES with no data-path collective: data, PSD and the detector
description are replicated, every rank evaluates its own batch of B samples (weak scaling:
one sampler population per GPU), and the only communication is control-plane -- a barrier
around the timed region, MAX over ranks of the device time and SUM of the units processed.
Works with the `nccl` backend on GPUs and with `gloo` on CPU (tests/test_dist_gloo.py).
"""
from __future__ import annotations

import os
from typing import Tuple

import numpy as np


def env_world() -> Tuple[int, int, int]:
    """(rank, local_rank, world_size) from the torchrun environment; (0, 0, 1) when absent."""
    return (int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0")),
            int(os.environ.get("WORLD_SIZE", "1")))


def init(backend: str):
    """Initialise torch.distributed from MASTER_ADDR/MASTER_PORT when WORLD_SIZE > 1."""
    import torch.distributed as dist
    rank, local_rank, world = env_world()
    if world > 1 and not dist.is_initialized():
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        os.environ.setdefault("MASTER_PORT", "29500")
        dist.init_process_group(backend=backend, rank=rank, world_size=world)
    return rank, local_rank, world


def rank_seed(seed: int, rank: int) -> int:
    """Seed of the parameter batch a rank draws: rank 0 keeps the config's seed."""
    return int(seed) + 1000003 * int(rank)


def shard_bounds(B: int, rank: int, world: int) -> Tuple[int, int]:
    """[lo, hi) of a contiguous, balanced split of B samples (strong-scaling helper)."""
    base, rem = divmod(int(B), int(world))
    lo = rank * base + min(rank, rem)
    return lo, lo + base + (1 if rank < rem else 0)


def barrier(device=None) -> None:
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized():
        if device is not None and device.type == "cuda":
            dist.barrier(device_ids=[device.index])
        else:
            dist.barrier()


def aggregate(elapsed_ms: float, units: float, device=None) -> Tuple[float, float]:
    """(MAX over ranks of elapsed_ms, SUM over ranks of units)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()):
        return float(elapsed_ms), float(units)
    dev = device if device is not None else torch.device("cpu")
    t = torch.tensor([float(elapsed_ms)], dtype=torch.float64, device=dev)
    u = torch.tensor([float(units)], dtype=torch.float64, device=dev)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(u, op=dist.ReduceOp.SUM)
    return float(t.item()), float(u.item())


def gather_lnL(local: "np.ndarray", device=None) -> "np.ndarray":
    """All-gather of the per-rank lnL vectors (B/G doubles each; latency-bound)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()):
        return np.asarray(local)
    dev = device if device is not None else torch.device("cpu")
    x = torch.as_tensor(np.asarray(local), dtype=torch.float64, device=dev)
    out = [torch.empty_like(x) for _ in range(dist.get_world_size())]
    dist.all_gather(out, x)
    return torch.cat(out).cpu().numpy()


class ShardedLikelihood:
    """Strong scaling over samples: every rank holds the same data set and the same batch of theta,
    evaluates the samples [lo, hi) of `shard_bounds` with `local_eval` (e.g. a `binding.Likelihood`: tensor of
    theta [b][11] -> tensor of lnL [b]) and one all-gather of ceil(B / G) doubles per rank restores the full lnL
    vector on every rank, in sample order.  No other collective touches the data path; the result of each sample is
    bit-identical to the single-GPU one (the reduction of a sample never crosses ranks)."""

    def __init__(self, local_eval):
        self.local_eval = local_eval

    def __call__(self, params: "torch.Tensor") -> "torch.Tensor":
        import torch
        import torch.distributed as dist
        B = params.shape[0]
        if not (dist.is_available() and dist.is_initialized()):
            return self.local_eval(params)          # (a one-rank group still takes the all-gather path below)
        rank, world = dist.get_rank(), dist.get_world_size()
        lo, hi = shard_bounds(B, rank, world)
        per = -(-B // world)
        mine = torch.full((per,), float("nan"), dtype=torch.float64, device=params.device)
        if hi > lo:
            mine[:hi - lo] = self.local_eval(params[lo:hi].contiguous())
        parts = [torch.empty_like(mine) for _ in range(world)]
        dist.all_gather(parts, mine)
        out = torch.empty(B, dtype=torch.float64, device=params.device)
        for r, part in enumerate(parts):
            rlo, rhi = shard_bounds(B, r, world)
            out[rlo:rhi] = part[:rhi - rlo]
        return out
