"""GPU-vs-oracle parity of pespace_loglike_grad (reverse-mode gradient).

Checker: oracle.fisher's gradient (11-tangent dual number, pinned by P12 / P13) and oracle.loglike.  Tolerances of
test_gpu_parity.py: lnL 1e-9 relative; grad_i on the Cauchy-Schwarz scale sqrt(F_ii <d-h|d-h>) at 1e-9.
"""
import dataclasses

import numpy as np
import pytest

import oracle
from paper_2602_12011_b200 import workloads as W

pytestmark = pytest.mark.gpu

TOL = 1e-9


@pytest.fixture(scope="module")
def P():
    import torch
    from paper_2602_12011_b200 import binding
    assert torch.cuda.is_available()
    return binding


def dev(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def oracle_response_fn(params, freqs, model):
    return oracle.response(params, freqs, model)


def check_grad(P, wl, data, psd, subset=None):
    idx = np.arange(wl.B) if subset is None else np.asarray(subset)
    lnL, g = P.loglike_grad(dev(wl.params), dev(data), dev(psd), wl.grid, wl.model)
    lnL, g = lnL.cpu().numpy()[idx], g.cpu().numpy()[idx]
    Fo, go = oracle.fisher(wl.params[idx], data, psd, wl.grid, wl.model)
    want = oracle.loglike(wl.params[idx], data, psd, wl.grid, wl.model)
    hh = -2.0 * oracle.loglike(wl.params[idx], np.zeros_like(data), psd, wl.grid, wl.model)
    assert (np.abs(lnL - want) / np.maximum(np.abs(want), 0.5 * hh)).max() <= TOL
    d = np.sqrt(np.einsum("bii->bi", Fo))
    d = np.where(d > 0, d, 1.0)
    rr = np.maximum(-2.0 * want, hh)
    err = np.abs(g - go) / (d * np.sqrt(rr)[:, None])
    assert err.max() <= TOL, (err.max(), np.unravel_index(np.argmax(err), err.shape), err.max(axis=0))
    return lnL, g


def test_grad_config1_full(P):
    wl = W.config(1)
    check_grad(P, wl, wl.data(oracle_response_fn), wl.psd())


@pytest.mark.parametrize("idx,B,N", [(2, 70, 3000), (3, 37, 1500), (4, 67, 1100), (5, 9, 2300)])
def test_grad_reduced_configs(P, idx, B, N):
    """several tiles (32 samples), several blocks (1024 bins), ragged tails"""
    wl = W.config(idx, B=B, N=N)
    check_grad(P, wl, wl.data(oracle_response_fn), wl.psd())


@pytest.mark.parametrize("gen", [15, 20])
def test_grad_random_sky_spinning_all_detectors(P, gen):
    rng = np.random.default_rng(5)
    th = W.draw_prior(9, 4e5, rng)
    th[:, 2] = rng.uniform(-0.8, 0.8, 9); th[:, 3] = rng.uniform(-0.8, 0.8, 9)
    dets = (dataclasses.replace(W.lisa_like(gen), lambda0=0.7), W.taiji_like(gen),
            dataclasses.replace(W.tianqin_like(gen), lambda0=1.1))
    wl = W.Workload("random", W.Grid(1e-4, 3.1e-5, 700), W.Model(W.MODES_HM, dets), th, th[3].copy(), 77)
    check_grad(P, wl, wl.data(oracle_response_fn), wl.psd())


@pytest.mark.parametrize("mask", [1, 2, 4, 8, 16, 9, 22])
def test_grad_individual_modes(P, mask):
    wl = W.config(4, B=5, N=400)
    wl = W.Workload("modes", wl.grid, W.Model(mask, wl.model.detectors), wl.params, wl.theta_inj, 5)
    check_grad(P, wl, wl.data(oracle_response_fn), wl.psd())


def test_grad_matches_forward_mode_and_is_deterministic(P):
    wl = W.config(5, B=13, N=2500)
    data, psd = wl.data(oracle_response_fn), wl.psd()
    lik = P.LikelihoodGrad(dev(data), dev(psd), wl.grid, wl.model, wl.B)
    l1, g1 = lik(dev(wl.params))
    l2, g2 = lik(dev(wl.params))
    assert np.array_equal(l1.cpu().numpy(), l2.cpu().numpy()) and np.array_equal(g1.cpu().numpy(), g2.cpu().numpy())
    F, gf = P.fisher(dev(wl.params), dev(data), dev(psd), wl.grid, wl.model)
    d = np.sqrt(np.einsum("bii->bi", F.cpu().numpy()))
    rr = -2.0 * l1.cpu().numpy()
    assert (np.abs(g1.cpu().numpy() - gf.cpu().numpy()) / (d * np.sqrt(rr)[:, None])).max() <= TOL
    plain = P.loglike(dev(wl.params), dev(data), dev(psd), wl.grid, wl.model).cpu().numpy()
    assert np.allclose(l1.cpu().numpy(), plain, rtol=1e-12, atol=0)
    # host-buffer session: same kernels, bit-identical
    ses = P.Session(wl.grid, wl.model, wl.B)
    ses.set_data(data, psd)
    ls, gs = ses.loglike_grad(wl.params)
    assert np.array_equal(ls, l1.cpu().numpy()) and np.array_equal(gs, g1.cpu().numpy())
    ses.close()


def test_grad_edge_cases(P):
    wl = W.config(5, B=6, N=300)
    data, psd = wl.data(oracle_response_fn), wl.psd()
    psd2 = psd.copy(); psd2[0, 0, 3] = 0.0; psd2[1, 1, 100] = np.inf; psd2[2, 2, 299] = np.nan
    data2 = data.copy(); data2[0, 0, 3] = np.nan
    th = wl.params.copy(); th[1, 0] = -5.0; th[4, 4] = np.nan
    lnL, g = P.loglike_grad(dev(th), dev(data2), dev(psd2), wl.grid, wl.model)
    lnL, g = lnL.cpu().numpy(), g.cpu().numpy()
    assert np.all(np.isneginf(lnL[[1, 4]])) and np.all(np.isnan(g[[1, 4]]))
    ok = [0, 2, 3, 5]
    Fo, go = oracle.fisher(th[ok], data2, psd2, wl.grid, wl.model)
    d = np.sqrt(np.einsum("bii->bi", Fo))
    rr = -2.0 * oracle.loglike(th[ok], data2, psd2, wl.grid, wl.model)
    assert (np.abs(g[ok] - go) / (d * np.sqrt(rr)[:, None])).max() <= TOL
    # B = 1, N = 1
    one = W.Workload("one", W.Grid(3e-3, 1e-5, 1), W.config(2).model, wl.params[:1], wl.theta_inj, None)
    check_grad(P, one, np.full((1, 3, 1), 1e-20 + 2e-20j), one.psd())


def test_grad_full_size_sampled(P):
    """config 5's workload at full size (B = 256, N = 262144, three detectors, five modes), 8 samples vs the oracle"""
    wl = W.config(5)
    check_grad(P, wl, wl.data(oracle_response_fn), wl.psd(), subset=[0, 37, 73, 110, 146, 183, 219, 255])
