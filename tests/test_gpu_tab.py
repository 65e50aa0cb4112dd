"""GPU-vs-oracle parity of the tabulated-waveform entry points (reading T1):
pespace_response_tab / pespace_loglike_tab against oracle.response_tab / oracle.loglike_tab on the same tables.
Tolerances as in test_gpu_parity.py: 1e-9 on lnL (relative to max(|lnL|, <h|h>/2)), 1e-8 max-abs on the response
with the 1e-12 cancellation floor of the T channel."""
import numpy as np
import pytest

import oracle
from paper_2602_12011_b200 import workloads as W

pytestmark = pytest.mark.gpu

TOL_LNL = 1e-9
TOL_RESP = 1e-8
CANCEL_FLOOR = 1e-12


@pytest.fixture(scope="module")
def P():
    import torch
    from paper_2602_12011_b200 import binding
    assert torch.cuda.is_available()
    return binding


def dev(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def dev_table(P, table):
    return P.WaveTable(*(dev(x) for x in table))


def check_response_tab(P, params, table, freqs, model):
    got = P.response_tab(dev(params), dev_table(P, table), dev(freqs), model).cpu().numpy()
    want = oracle.response_tab(params, table, freqs, model)
    assert got.shape == want.shape
    for b in range(want.shape[0]):
        for d in range(want.shape[1]):
            det_scale = np.abs(want[b, d]).max()
            assert np.abs(got[b, d] - want[b, d]).max() <= TOL_RESP * det_scale, (b, d)
            for c in range(3):
                scale = np.abs(want[b, d, c]).max()
                err = np.abs(got[b, d, c] - want[b, d, c]).max()
                assert err <= TOL_RESP * scale + CANCEL_FLOOR * det_scale, (b, d, c, err / scale, err / det_scale)
    return got, want


def check_loglike_tab(P, params, table, data, psd, grid, model):
    lik = P.LikelihoodTab(dev(data), dev(psd), grid, model, params.shape[0])
    got = lik(dev(params), dev_table(P, table)).cpu().numpy()
    want = oracle.loglike_tab(params, table, data, psd, grid, model)
    hh = -2.0 * oracle.loglike_tab(params, table, np.zeros_like(data), psd, grid, model)
    scale = np.maximum(np.abs(want), 0.5 * hh)
    rel = np.abs(got - want) / scale
    assert np.all(rel <= TOL_LNL), (rel.max(), int(np.argmax(rel)))
    return got


def noisy_data(wl, table):
    rng = np.random.default_rng(wl.noise_seed or 7)
    psd = wl.psd()
    inj = wl.theta_inj[None]
    inj_table = tuple(x if x.ndim == 1 else x[:1] for x in table)
    h = oracle.response_tab(inj, inj_table, wl.grid.freqs(), wl.model)[0]
    return h + W.coloured_noise(psd, wl.grid.df, rng), psd


@pytest.mark.parametrize("idx,B,N,K", [(2, 45, 3000, 700), (3, 21, 1500, 500), (4, 70, 1100, 900)])
def test_tab_reduced_configs_oracle_tables(P, idx, B, N, K):
    """Tables of the oracle's analytic modes (the physically shaped input), several tiles and a ragged tail."""
    wl = W.config(idx, B=B, N=N)
    f = wl.grid.freqs()
    wl.params[0] = wl.theta_inj                                           # sample 0 = the injection
    table = W.table_from_waveform_fn(wl.params, wl.model.mode_mask, W.log_nodes(f[0], f[-1], K), oracle.waveform)
    data, psd = noisy_data(wl, table)
    check_loglike_tab(P, wl.params, table, data, psd, wl.grid, wl.model)
    check_response_tab(P, wl.params[:4], tuple(x if x.ndim == 1 else x[:4] for x in table), f[::3], wl.model)


@pytest.mark.parametrize("mask", [W.MODE_22 | W.MODE_33, W.MODE_21 | W.MODE_33 | W.MODE_32,
                                  W.MODE_22 | W.MODE_21 | W.MODE_32 | W.MODE_44])
def test_tab_two_to_four_modes(P, mask):
    """mode counts other than 1 and 5: the kernel variant with the run-time mode loop (the compile-time variants
    cover the mode counts of configs 2-4 only)"""
    base = W.config(4, B=37, N=1100)
    wl = W.Workload("mask%d" % mask, base.grid, W.Model(mask, base.model.detectors), base.params, base.theta_inj,
                    base.noise_seed)
    f = wl.grid.freqs()
    wl.params[0] = wl.theta_inj
    table = W.table_from_waveform_fn(wl.params, mask, W.log_nodes(f[0], f[-1], 600), oracle.waveform)
    data, psd = noisy_data(wl, table)
    check_loglike_tab(P, wl.params, table, data, psd, wl.grid, wl.model)
    check_response_tab(P, wl.params[:4], tuple(x if x.ndim == 1 else x[:4] for x in table), f[::3], wl.model)


@pytest.mark.parametrize("gen", [15, 20])
def test_tab_random_sky_band_limited_table(P, gen):
    """Prior draws through all three detector kinds; synthetic chirp tables that end inside the grid (modes vanish
    above the last node and below the first), frequencies exactly on nodes, f <= 0 in the response call."""
    rng = np.random.default_rng(31)
    grid = W.Grid(1e-4, 3.1e-5, 700)
    th = W.draw_prior(37, 4e5, rng)
    model = W.Model(W.MODES_HM, (W.lisa_like(gen), W.taiji_like(gen), W.tianqin_like(gen)))
    fn = W.log_nodes(3e-4, 1.5e-2, 333)
    table = W.chirp_table(th, model.mode_mask, fn)
    wl = W.Workload("tab-random", grid, model, th, th[3].copy(), 79)
    psd = wl.psd()
    h = oracle.response_tab(th[3:4], tuple(x if x.ndim == 1 else x[3:4] for x in table), grid.freqs(), model)[0]
    data = h + W.coloured_noise(psd, grid.df, np.random.default_rng(79))
    check_loglike_tab(P, th, table, data, psd, grid, model)
    f = np.concatenate([[0.0, -1.0], fn[[0, 5, 100, -1]], grid.freqs()[::9]])
    got, want = check_response_tab(P, th[:5], tuple(x if x.ndim == 1 else x[:5] for x in table), f, model)
    assert np.all(got[:, :, :, :2] == 0.0)
    outside = (f < fn[0]) | (f > fn[-1])
    assert np.all(got[..., outside] == 0.0) and np.all(want[..., outside] == 0.0)


def test_tab_single_modes_edge_cases_and_determinism(P):
    grid = W.Grid(1e-4, 2e-6, 300)                                        # one ragged bin block
    th = np.tile(W.THETA_INJ, (5, 1))
    th[1, 4] = -1.0                                                       # out of domain: D_L <= 0
    th[2, 9] = np.nan                                                     # non-finite psi
    th[3, 0] = np.nan                                                     # M is NOT used by the tabulated path
    fn = W.log_nodes(1e-4, 1e-3, 64)
    for mask in (1, 2, 4, 8, 16):
        model = W.Model(mask, (W.lisa_like(), W.tianqin_like()))
        good = np.where(np.isfinite(th[:, 0]), th[:, 0], 2e6)
        tab_params = th.copy(); tab_params[:, 0] = good
        table = W.chirp_table(np.where(np.isfinite(tab_params), tab_params, 1.0), mask, fn)
        wl = W.Workload("tab-edge", grid, model, th, th[0].copy(), None)
        psd = wl.psd()
        psd[0, 1, 10:20] = 0.0                                            # weight-0 bins
        data = oracle.response_tab(th[:1], tuple(x if x.ndim == 1 else x[:1] for x in table), grid.freqs(), model)[0]
        lik = P.LikelihoodTab(dev(data), dev(psd), grid, model, 5)
        a = lik(dev(th), dev_table(P, table)).cpu().numpy()
        b = lik(dev(th), dev_table(P, table)).cpu().numpy()
        assert np.array_equal(a, b)
        want = oracle.loglike_tab(th, table, data, psd, grid, model)
        assert a[1] == -np.inf and a[2] == -np.inf and want[1] == -np.inf and want[2] == -np.inf
        hh = -2.0 * oracle.loglike_tab(th[[0, 3, 4]], tuple(x if x.ndim == 1 else x[[0, 3, 4]] for x in table),
                                       np.zeros_like(data), psd, grid, model)
        assert np.all(np.abs(a[[0, 3, 4]] - want[[0, 3, 4]]) <= TOL_LNL * np.maximum(np.abs(want[[0, 3, 4]]), 0.5 * hh))
        r = P.response_tab(dev(th), dev_table(P, table), dev(grid.freqs()), model).cpu().numpy()
        assert np.all(np.isnan(r[1])) and np.all(np.isnan(r[2])) and np.all(np.isfinite(r[[0, 3, 4]]))


def test_tab_argument_errors(P):
    import torch
    grid = W.Grid(1e-4, 2e-6, 64)
    model = W.Model(1, (W.lisa_like(),))
    th = np.tile(W.THETA_INJ, (3, 1))
    table = W.chirp_table(th, 1, W.log_nodes(1e-4, 1e-3, 16))
    with pytest.raises(P.PespaceError):                                   # table for another batch size
        P.response_tab(dev(th[:2]), dev_table(P, table), dev(grid.freqs()), model)
    with pytest.raises(P.PespaceError):                                   # K < 4
        P.response_tab(dev(th), dev_table(P, tuple(x[..., :3] for x in table)), dev(grid.freqs()), model)
    with pytest.raises(P.PespaceError):                                   # two modes in the mask, one in the table
        P.response_tab(dev(th), dev_table(P, table), dev(grid.freqs()), W.Model(3, model.detectors))


def test_tab_full_size_sampled_parity(P):
    """BASELINE config 2 size (B = 4096 x N = 262144) in the launch configuration bench.py --waveform tab times:
    synthetic chirp tables on 4096 nodes; the oracle is evaluated on sampled samples."""
    wl = W.config(2)
    f = wl.grid.freqs()
    fn = W.log_nodes(f[0], f[-1], 4096)
    table = W.chirp_table(wl.params, wl.model.mode_mask, fn)
    inj = W.chirp_table(wl.theta_inj[None], wl.model.mode_mask, fn)
    psd = wl.psd()
    data = oracle.response_tab(wl.theta_inj[None], inj, f, wl.model)[0] + \
        W.coloured_noise(psd, wl.grid.df, np.random.default_rng(101))
    lik = P.LikelihoodTab(dev(data), dev(psd), wl.grid, wl.model, wl.B)
    got = lik(dev(wl.params), dev_table(P, table)).cpu().numpy()
    idx = np.array([0, 1023, 2500, 4095])
    sub = tuple(x if x.ndim == 1 else x[idx] for x in table)
    want = oracle.loglike_tab(wl.params[idx], sub, data, psd, wl.grid, wl.model)
    assert np.all(np.isfinite(got))
    assert np.all(np.abs(got[idx] - want) <= TOL_LNL * np.abs(want)), np.abs(got[idx] - want) / np.abs(want)


def test_tab_session_matches_device_call(P):
    """pespace_session_loglike_tab (host tables) is bit-identical to pespace_loglike_tab; unordered nodes rejected."""
    wl = W.config(3, B=9, N=900)
    f = wl.grid.freqs()
    table = W.chirp_table(wl.params, wl.model.mode_mask, W.log_nodes(f[0], f[-1], 200))
    data, psd = noisy_data(wl, table)
    want = P.LikelihoodTab(dev(data), dev(psd), wl.grid, wl.model, wl.B)(dev(wl.params), dev_table(P, table)).cpu().numpy()
    ses = P.Session(wl.grid, wl.model, 16)
    ses.set_data(data, psd)
    assert np.array_equal(ses.loglike_tab(wl.params, table), want)
    assert np.array_equal(ses.loglike_tab(wl.params[:5], tuple(x if x.ndim == 1 else x[:5] for x in table)), want[:5])
    bad = (table[0][::-1].copy(),) + table[1:]
    with pytest.raises(P.PespaceError):
        ses.loglike_tab(wl.params, bad)
    ses.close()


# ------------------------------------------------------------------ T1 x S10: Fisher matrix / gradient on tables
TOL_F = 1e-9
USED = [4, 5, 6, 7, 8, 9, 10]            # D_L, iota, phi_c, lambda, beta, psi, t_c


def check_fisher_tab(P, params, table, data, psd, grid, model, with_grad=True):
    F, g = P.fisher_tab(dev(params), dev_table(P, table), dev(data) if with_grad else None, dev(psd), grid, model)
    F = F.cpu().numpy()
    Fo, go = oracle.fisher_tab(params, table, data if with_grad else None, psd, grid, model)
    assert np.all(F[:, :4, :] == 0) and np.all(F[:, :, :4] == 0)          # M, q, chi1, chi2: not parameters of this path
    ix = np.ix_(range(params.shape[0]), USED, USED)
    d = np.sqrt(np.einsum("bii->bi", Fo[ix]))
    assert np.all(d > 0)
    errF = np.abs(F[ix] - Fo[ix]) / (d[:, :, None] * d[:, None, :])
    assert errF.max() <= TOL_F, errF.max()
    assert np.array_equal(F, F.transpose(0, 2, 1))
    if with_grad:
        g = g.cpu().numpy()
        assert np.all(g[:, :4] == 0)
        rr = -2.0 * oracle.loglike_tab(params, table, data, psd, grid, model)
        errg = np.abs(g[:, USED] - go[:, USED]) / (d * np.sqrt(rr)[:, None])
        assert errg.max() <= TOL_F, errg.max()
    else:
        assert g is None
    return F


@pytest.mark.parametrize("idx,B,N,K", [(2, 11, 5000, 700), (3, 6, 2100, 500), (4, 9, 1100, 900)])
def test_fisher_tab_reduced_configs(P, idx, B, N, K):
    """several chunks and blocks, ragged tails; tables of the oracle's analytic modes; with and without data"""
    wl = W.config(idx, B=B, N=N)
    f = wl.grid.freqs()
    wl.params[0] = wl.theta_inj
    table = W.table_from_waveform_fn(wl.params, wl.model.mode_mask, W.log_nodes(f[0], f[-1], K), oracle.waveform)
    data, psd = noisy_data(wl, table)
    check_fisher_tab(P, wl.params, table, data, psd, wl.grid, wl.model)
    check_fisher_tab(P, wl.params, table, data, psd, wl.grid, wl.model, with_grad=False)


@pytest.mark.parametrize("gen", [15, 20])
def test_fisher_tab_random_sky_synthetic_tables(P, gen):
    rng = np.random.default_rng(6)
    th = W.draw_prior(7, 4e5, rng)
    dets = (W.lisa_like(gen), W.taiji_like(gen), W.tianqin_like(gen))
    model = W.Model(W.MODES_HM, dets)
    grid = W.Grid(2e-4, 3.1e-5, 600)
    f = grid.freqs()
    table = W.chirp_table(th, model.mode_mask, W.log_nodes(1.5 * f[0], 0.8 * f[-1], 200))     # band-limited tables
    wl = W.Workload("random", grid, model, th, th[2].copy(), 31)
    data, psd = noisy_data(wl, table)
    check_fisher_tab(P, th, table, data, psd, grid, model)


def test_fisher_tab_gradient_only_edge_cases_and_determinism(P):
    wl = W.config(4, B=6, N=700)
    f = wl.grid.freqs()
    table = W.table_from_waveform_fn(wl.params, wl.model.mode_mask, W.log_nodes(f[0], f[-1], 300), oracle.waveform)
    data, psd = noisy_data(wl, table)
    fis = P.FisherTab(dev(data), dev(psd), wl.grid, wl.model, wl.B)
    F, g = fis(dev(wl.params), dev_table(P, table))
    none, g1 = fis(dev(wl.params), dev_table(P, table), grad_only=True)
    assert none is None
    Fo, go = oracle.fisher_tab(wl.params, table, data, psd, wl.grid, wl.model)
    d = np.sqrt(np.einsum("bii->bi", Fo[:, 4:, 4:]))
    rr = -2.0 * oracle.loglike_tab(wl.params, table, data, psd, wl.grid, wl.model)
    assert (np.abs(g1.cpu().numpy()[:, 4:] - go[:, 4:]) / (d * np.sqrt(rr)[:, None])).max() <= TOL_F
    F2, g2 = fis(dev(wl.params), dev_table(P, table))
    assert np.array_equal(F.cpu().numpy(), F2.cpu().numpy()) and np.array_equal(g.cpu().numpy(), g2.cpu().numpy())
    th = wl.params.copy(); th[1, 4] = -1.0; th[3, 9] = np.nan; th[4, 0] = np.nan      # M is ignored: sample 4 stays valid
    Fb, gb = fis(dev(th), dev_table(P, table))
    Fb, gb = Fb.cpu().numpy(), gb.cpu().numpy()
    assert np.all(np.isnan(Fb[[1, 3]])) and np.all(np.isnan(gb[[1, 3]])) and np.all(np.isfinite(Fb[[0, 2, 4, 5]]))
    with pytest.raises(P.PespaceError):
        P.FisherTab(None, dev(psd), wl.grid, wl.model, wl.B)(dev(wl.params), dev_table(P, table), grad_only=True)


def test_fisher_tab_full_size_sampled(P):
    """config 5's workload (three detectors, five modes, N = 262144) at B = 64 on tables; oracle on 3 samples"""
    wl = W.config(5, B=64)
    f = wl.grid.freqs()
    table = W.chirp_table(wl.params, wl.model.mode_mask, W.log_nodes(f[0], f[-1], 2048))
    data, psd = noisy_data(wl, table)
    F, g = P.fisher_tab(dev(wl.params), dev_table(P, table), dev(data), dev(psd), wl.grid, wl.model)
    sub = [0, 31, 63]
    tsub = tuple(x if x.ndim == 1 else x[sub] for x in table)
    Fo, go = oracle.fisher_tab(wl.params[sub], tsub, data, psd, wl.grid, wl.model)
    ix = np.ix_(range(3), USED, USED)
    d = np.sqrt(np.einsum("bii->bi", Fo[ix]))
    assert (np.abs(F.cpu().numpy()[sub][ix] - Fo[ix]) / (d[:, :, None] * d[:, None, :])).max() <= TOL_F
    rr = -2.0 * oracle.loglike_tab(wl.params[sub], tsub, data, psd, wl.grid, wl.model)
    assert (np.abs(g.cpu().numpy()[sub][:, USED] - go[:, USED]) / (d * np.sqrt(rr)[:, None])).max() <= TOL_F
