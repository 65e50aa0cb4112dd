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


def replicate(*tensors, src: int = 0):
    """Replication of the data set, the PSD (and, for strong scaling, the theta batch) from rank `src` to every rank
    ("data, weights and per-bin tables are replicated once (ncclBroadcast)"): one broadcast per
    tensor, in place; every rank passes tensors of the same shape and dtype.  Returns the tensors.  Done once per
    data set -- the hot loop has no collective besides the all-gather of ShardedCall."""
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized():
        import torch
        for t in tensors:
            dist.broadcast(torch.view_as_real(t) if t.is_complex() else t, src=src)     # (re, im) pairs: same memory
    return tensors if len(tensors) != 1 else tensors[0]


class ShardedCall:
    """Strong scaling over samples for ANY per-sample call of the library: every rank holds the same
    data set and the same batch of theta, evaluates the samples [lo, hi) of `shard_bounds` with `local_eval` (theta
    [b][11] -> a tensor [b][...] or a tuple of such tensors, `None` entries allowed: e.g. a `binding.Likelihood`
    (lnL), a `binding.LikelihoodGrad` (lnL, gradient) or a `binding.Fisher` (F, gradient)), and one all-gather of
    ceil(B / G) rows per output restores the full arrays on every rank, in sample order.  No other collective touches
    the data path; the result of each sample is bit-identical to the single-GPU one (the reduction of a sample never
    crosses ranks)."""

    def __init__(self, local_eval):
        self.local_eval = local_eval

    def __call__(self, params: "torch.Tensor"):
        import torch
        import torch.distributed as dist
        B = params.shape[0]
        if not (dist.is_available() and dist.is_initialized()):
            return self.local_eval(params)          # (a one-rank group still takes the all-gather path below)
        rank, world = dist.get_rank(), dist.get_world_size()
        lo, hi = shard_bounds(B, rank, world)
        per = -(-B // world)
        # every rank evaluates at least one sample so that the shapes of the outputs are known everywhere (a rank
        # whose slice is empty -- more ranks than samples -- evaluates sample 0 and discards it)
        local = self.local_eval(params[lo:hi].contiguous() if hi > lo else params[:1].contiguous())
        single = not isinstance(local, (tuple, list))
        outs = []
        for res in ((local,) if single else local):
            if res is None:
                outs.append(None)
                continue
            mine = torch.full((per,) + tuple(res.shape[1:]), float("nan"), dtype=res.dtype, device=res.device)
            if hi > lo:
                mine[:hi - lo] = res
            parts = [torch.empty_like(mine) for _ in range(world)]
            dist.all_gather(parts, mine)
            out = torch.empty((B,) + tuple(res.shape[1:]), dtype=res.dtype, device=res.device)
            for r, part in enumerate(parts):
                rlo, rhi = shard_bounds(B, r, world)
                out[rlo:rhi] = part[:rhi - rlo]
            outs.append(out)
        return outs[0] if single else tuple(outs)


class ShardedLikelihood(ShardedCall):
    """`ShardedCall` for a call that returns lnL [b] (kept under its round-1 name)."""
