"""Maximum batch sizes (include/pespace.h: the sample tiles of a call fill gridDim.y = 65535): the largest accepted batch
is evaluated correctly -- first, last and interior samples against the oracle, every result finite -- and one sample
more is refused with PESPACE_EINVAL before anything is launched.  Likelihood: 65535 x 64 samples; reverse-mode
gradient of a multi-class model: 65535 x 16; Fisher matrix: 65535 x 4."""
import numpy as np
import pytest

import oracle
from paper_2602_12011_b200 import workloads as W

pytestmark = pytest.mark.gpu

TOL = 1e-9


def dev(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def big_batch(B, grid, rng):
    base = W.draw_prior(4096, 1.0 / grid.df, rng)
    th = np.tile(base, (B // 4096 + 1, 1))[:B].copy()
    th[:, 10] += rng.uniform(0.0, 10.0, B)                    # every sample its own t_c
    return th


def test_largest_likelihood_batch_and_one_more():
    import torch
    from paper_2602_12011_b200 import binding as P
    grid = W.Grid(1e-4, 1.5e-5, 64)
    model = W.Model(W.MODES_HM, (W.lisa_like(),))
    rng = np.random.default_rng(4)
    b_max = 65535 * 64
    th = big_batch(b_max + 1, grid, rng)
    wl = W.Workload("limits", grid, model, th[:8], th[0].copy(), 5)
    psd, data = wl.psd(), wl.data(lambda p, f, m: oracle.response(p, f, m))
    d_th = dev(th)
    lik = P.Likelihood(dev(data), dev(psd), grid, model, b_max + 1)
    got = lik(d_th[:b_max])
    assert bool(torch.isfinite(got).all())
    got = got.cpu().numpy()
    idx = np.array([0, 1, 63, 64, 4095, 4096, 1000003, b_max - 65, b_max - 1])
    want = oracle.loglike(th[idx], data, psd, grid, model)
    hh = -2.0 * oracle.loglike(th[idx], np.zeros_like(data), psd, grid, model)
    assert (np.abs(got[idx] - want) / np.maximum(np.abs(want), 0.5 * hh)).max() <= TOL
    out = torch.full((b_max + 1,), 7.0, dtype=torch.float64, device="cuda")
    with pytest.raises(P.PespaceError, match="invalid argument"):
        lik(d_th, out)
    torch.cuda.synchronize()
    assert bool((out == 7.0).all())                            # refused before anything was launched


def test_largest_gradient_batch_and_one_more():
    import torch
    from paper_2602_12011_b200 import binding as P
    grid = W.Grid(1e-4, 1.5e-5, 64)
    model = W.Model(W.MODE_22 | W.MODE_33, (W.tianqin_like(),))
    rng = np.random.default_rng(6)
    b_max = 65535 * 16
    th = big_batch(b_max + 1, grid, rng)
    wl = W.Workload("limits", grid, model, th[:8], th[0].copy(), 5)
    psd, data = wl.psd(), wl.data(lambda p, f, m: oracle.response(p, f, m))
    d_th = dev(th)
    lg = P.LikelihoodGrad(dev(data), dev(psd), grid, model, b_max + 1)
    lnL, grad = lg(d_th[:b_max])
    assert bool(torch.isfinite(lnL).all()) and bool(torch.isfinite(grad).all())
    idx = np.array([0, 15, 16, 4097, 500001, b_max - 17, b_max - 1])
    Fo, go = oracle.fisher(th[idx], data, psd, grid, model)
    want = oracle.loglike(th[idx], data, psd, grid, model)
    hh = -2.0 * oracle.loglike(th[idx], np.zeros_like(data), psd, grid, model)
    assert (np.abs(lnL.cpu().numpy()[idx] - want) / np.maximum(np.abs(want), 0.5 * hh)).max() <= TOL
    d = np.sqrt(np.einsum("bii->bi", Fo))
    scale = d * np.sqrt(np.maximum(-2.0 * want, hh))[:, None]
    assert (np.abs(grad.cpu().numpy()[idx] - go) / scale).max() <= TOL
    with pytest.raises(P.PespaceError, match="invalid argument"):
        lg(d_th)


def test_largest_fisher_batch_and_one_more():
    import torch
    from paper_2602_12011_b200 import binding as P
    grid = W.Grid(1.3e-4, 1.1e-5, 96)
    model = W.Model(W.MODE_22 | W.MODE_21 | W.MODE_44, (W.lisa_like(15),))
    rng = np.random.default_rng(8)
    b_max = 65535 * 4
    th = big_batch(b_max + 1, grid, rng)
    wl = W.Workload("limits", grid, model, th[:8], th[0].copy(), 5)
    psd, data = wl.psd(), wl.data(lambda p, f, m: oracle.response(p, f, m))
    d_th = dev(th)
    fi = P.Fisher(dev(data), dev(psd), grid, model, b_max + 1)
    F, g = fi(d_th[:b_max])
    assert bool(torch.isfinite(F).all()) and bool(torch.isfinite(g).all())
    idx = np.array([0, 3, 4, 4099, 100001, b_max - 5, b_max - 1])
    Fo, go = oracle.fisher(th[idx], data, psd, grid, model)
    d = np.sqrt(np.einsum("bii->bi", Fo))
    assert (np.abs(F.cpu().numpy()[idx] - Fo) / (d[:, :, None] * d[:, None, :])).max() <= TOL
    want = oracle.loglike(th[idx], data, psd, grid, model)
    hh = -2.0 * oracle.loglike(th[idx], np.zeros_like(data), psd, grid, model)
    scale = d * np.sqrt(np.maximum(-2.0 * want, hh))[:, None]
    assert (np.abs(g.cpu().numpy()[idx] - go) / scale).max() <= TOL
    with pytest.raises(P.PespaceError, match="invalid argument"):
        fi(d_th)
