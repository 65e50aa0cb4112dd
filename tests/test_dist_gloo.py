"""World-size-2 CPU (gloo) tests of the multi-GPU plumbing in paper_2602_12011_b200/dist.py:
sample sharding with no data-path collective, MAX/SUM aggregation of the timing,
the all-gather of per-rank lnL vectors, and per-rank parameter seeds.  The per-rank "likelihood"
here is a stand-in pure function of the parameters (no oracle, no CUDA): what is under test is
the host-side sharding and communication logic."""
import os
import socket

import numpy as np
import torch.multiprocessing as mp

from paper_2602_12011_b200 import dist as pdist
from paper_2602_12011_b200 import workloads as W


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _stand_in_lnL(params: np.ndarray) -> np.ndarray:
    return -0.5 * np.sum(params * params, axis=1)


def _worker(rank: int, world: int, port: int, B: int, out_dir: str) -> None:
    os.environ.update({"RANK": str(rank), "LOCAL_RANK": str(rank), "WORLD_SIZE": str(world),
                       "MASTER_ADDR": "127.0.0.1", "MASTER_PORT": str(port)})
    r, lr, w = pdist.init("gloo")
    assert (r, lr, w) == (rank, rank, world)
    wl = W.config(2, B=B, N=8)
    lo, hi = pdist.shard_bounds(B, rank, world)
    local = _stand_in_lnL(wl.params[lo:hi])
    pdist.barrier()
    full = pdist.gather_lnL(np.pad(local, (0, (-(-B // world)) - local.size), constant_values=np.nan))
    t_max, units = pdist.aggregate(10.0 + rank, hi - lo)
    # weak scaling: every rank draws its own batch
    mine = W.config(2, B=4, N=8, param_seed=pdist.rank_seed(1000, rank)).params
    import torch
    sharded = pdist.ShardedLikelihood(lambda p: torch.from_numpy(_stand_in_lnL(p.numpy())))
    strong = sharded(torch.from_numpy(wl.params)).numpy()          # same batch on every rank, split and gathered
    tiny = sharded(torch.from_numpy(wl.params[:1])).numpy()        # fewer samples than ranks: one rank idles
    # replication of the data set from rank 0: rank 1 starts with zeros
    d_ = torch.arange(24.0).reshape(2, 3, 4) if rank == 0 else torch.zeros(2, 3, 4)
    p_ = torch.full((5,), 7.0) if rank == 0 else torch.zeros(5)
    d_, p_ = pdist.replicate(d_, p_)
    assert torch.equal(d_, torch.arange(24.0).reshape(2, 3, 4)) and torch.equal(p_, torch.full((5,), 7.0))
    # a call with several outputs (lnL, gradient-like [b][11], nothing, Fisher-like [b][11][11])
    multi = pdist.ShardedCall(lambda p: (torch.from_numpy(_stand_in_lnL(p.numpy())), -p, None,
                                         p[:, :, None] * p[:, None, :]))
    m_lnL, m_grad, m_none, m_F = multi(torch.from_numpy(wl.params))
    assert m_none is None
    t_lnL, t_grad, _, t_F = multi(torch.from_numpy(wl.params[:1]))
    np.savez(os.path.join(out_dir, f"r{rank}.npz"), full=full, t_max=t_max, units=units, mine=mine, lo=lo, hi=hi,
             strong=strong, tiny=tiny, m_lnL=m_lnL.numpy(), m_grad=m_grad.numpy(), m_F=m_F.numpy(),
             t_grad=t_grad.numpy(), t_F=t_F.numpy())
    import torch.distributed as dist
    dist.destroy_process_group()


def test_sample_sharding_world_size_2(tmp_path):
    B, world = 37, 2
    port = _free_port()
    mp.spawn(_worker, args=(world, port, B, str(tmp_path)), nprocs=world, join=True)
    res = [np.load(tmp_path / f"r{r}.npz") for r in range(world)]
    want = _stand_in_lnL(W.config(2, B=B, N=8).params)
    per = -(-B // world)
    for r in res:
        full = r["full"]
        got = np.concatenate([full[i * per:i * per + (res[i]["hi"] - res[i]["lo"])] for i in range(world)])
        assert np.array_equal(got, want)                        # gather restores sample order, bit for bit
        assert float(r["t_max"]) == 11.0 and float(r["units"]) == B      # MAX of times, SUM of units
        assert np.array_equal(r["strong"], want) and np.array_equal(r["tiny"], want[:1])   # ShardedLikelihood
        p = W.config(2, B=B, N=8).params
        assert np.array_equal(r["m_lnL"], want) and np.array_equal(r["m_grad"], -p)            # ShardedCall, tuples
        assert np.array_equal(r["m_F"], p[:, :, None] * p[:, None, :])
        assert np.array_equal(r["t_grad"], -p[:1]) and r["t_F"].shape == (1, 11, 11)
    assert int(res[0]["lo"]) == 0 and int(res[0]["hi"]) == int(res[1]["lo"]) and int(res[1]["hi"]) == B
    assert not np.array_equal(res[0]["mine"], res[1]["mine"])    # different batches per rank
    assert np.array_equal(res[0]["mine"], W.config(2, B=4, N=8, param_seed=1000).params)   # rank 0 keeps the seed


def test_shard_bounds_cover_and_balance():
    for B in (1, 7, 64, 4096, 8191):
        for world in (1, 2, 3, 8):
            b = [pdist.shard_bounds(B, r, world) for r in range(world)]
            assert b[0][0] == 0 and b[-1][1] == B
            assert all(b[i][1] == b[i + 1][0] for i in range(world - 1))
            sizes = [hi - lo for lo, hi in b]
            assert max(sizes) - min(sizes) <= 1


def test_single_process_fallbacks():
    assert pdist.env_world()[2] >= 1
    t, u = pdist.aggregate(3.5, 12)
    assert (t, u) == (3.5, 12.0)
    x = np.arange(5.0)
    assert np.array_equal(pdist.gather_lnL(x), x)
    import torch
    y = torch.ones(3)
    assert pdist.replicate(y) is y                              # no process group: nothing to do
