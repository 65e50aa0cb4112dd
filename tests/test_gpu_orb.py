"""GPU-vs-oracle parity of the tabulated-orbit entry points (reading T2):
pespace_response_orb / pespace_loglike_orb against oracle.response_orb / oracle.loglike_orb on the same tables.
Tolerances of test_gpu_parity.py: 1e-9 on lnL (relative to max(|lnL|, <h|h>/2)), 1e-8 max-abs on the response with
the 1e-12 cancellation floor of the T channel."""
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


def dev_orbit(P, tab):
    return P.OrbitTable(tab[0], tab[1], dev(tab[2]), dev(tab[3]))


def time_span(params, mask, f):
    """[t_lo, t_hi] covering every t_lm(f) of the batch (the oracle's time-frequency map; test side only)"""
    tl = np.array([oracle.waveform(th, l, m, f)[2] for th in params for (l, m) in W.mask_modes(mask)])
    return tl.min() - 50.0, tl.max() + 50.0


def check_response_orb(P, params, tab, freqs, model):
    got = P.response_orb(dev(params), dev_orbit(P, tab), dev(freqs), model).cpu().numpy()
    want = oracle.response_orb(params, tab, freqs, model)
    for b in range(want.shape[0]):
        for d in range(want.shape[1]):
            det_scale = np.abs(want[b, d]).max()
            assert np.abs(got[b, d] - want[b, d]).max() <= TOL_RESP * det_scale, (b, d)
            for c in range(3):
                scale = np.abs(want[b, d, c]).max()
                err = np.abs(got[b, d, c] - want[b, d, c]).max()
                assert err <= TOL_RESP * scale + CANCEL_FLOOR * det_scale, (b, d, c, err / scale, err / det_scale)
    return got, want


def check_loglike_orb(P, wl, tab, data, psd):
    lik = P.LikelihoodOrb(dev(data), dev(psd), wl.grid, wl.model, wl.B)
    got = lik(dev(wl.params), dev_orbit(P, tab)).cpu().numpy()
    want = oracle.loglike_orb(wl.params, tab, data, psd, wl.grid, wl.model)
    hh = -2.0 * oracle.loglike_orb(wl.params, tab, np.zeros_like(data), psd, wl.grid, wl.model)
    rel = np.abs(got - want) / np.maximum(np.abs(want), 0.5 * hh)
    assert rel.max() <= TOL_LNL, (rel.max(), int(np.argmax(rel)))
    return got


@pytest.mark.parametrize("idx,B,N", [(2, 70, 3000), (3, 37, 1500), (4, 67, 1100)])
def test_orb_reduced_configs_synthetic_ephemeris(P, idx, B, N):
    """seeded toy ephemeris with breathing arms (workloads.synthetic_orbit_table), several tiles and a ragged tail"""
    wl = W.config(idx, B=B, N=N)
    f = wl.grid.freqs()
    t_lo, t_hi = time_span(wl.params, wl.model.mode_mask, f[[0, -1]])
    dt = 1800.0
    tab = W.synthetic_orbit_table(wl.model.detectors, t_lo, dt, int((t_hi - t_lo) / dt) + 2, seed=idx)
    rng = np.random.default_rng(wl.noise_seed)
    psd = wl.psd()
    data = oracle.response_orb(wl.theta_inj[None], tab, f, wl.model)[0] + W.coloured_noise(psd, wl.grid.df, rng)
    check_loglike_orb(P, wl, tab, data, psd)
    check_response_orb(P, wl.params[:4], tab, f[::5], wl.model)


@pytest.mark.parametrize("mask", [W.MODE_33, W.MODE_21 | W.MODE_33 | W.MODE_44, W.MODE_22 | W.MODE_32 | W.MODE_44])
def test_orb_other_mode_masks(P, mask):
    """class masks other than configs 2-4's: the kernel variant with the run-time class loop"""
    base = W.config(4, B=37, N=1100)
    wl = W.Workload("mask%d" % mask, base.grid, W.Model(mask, base.model.detectors), base.params, base.theta_inj,
                    base.noise_seed)
    f = wl.grid.freqs()
    t_lo, t_hi = time_span(wl.params, W.MODES_HM, f[[0, -1]])
    dt = 1800.0
    tab = W.synthetic_orbit_table(wl.model.detectors, t_lo, dt, int((t_hi - t_lo) / dt) + 2, seed=mask)
    rng = np.random.default_rng(wl.noise_seed)
    psd = wl.psd()
    data = oracle.response_orb(wl.theta_inj[None], tab, f, wl.model)[0] + W.coloured_noise(psd, wl.grid.df, rng)
    check_loglike_orb(P, wl, tab, data, psd)
    check_response_orb(P, wl.params[:4], tab, f[::5], wl.model)


@pytest.mark.parametrize("gen", [15, 20])
def test_orb_dense_analytic_tables_reproduce_the_analytic_kernels(P, gen):
    """tables sampled from the oracle's analytic orbits: the tabulated-orbit kernels must agree with the oracle on those
    tables AND (to the interpolation error, 1e-9) with the analytic-orbit kernels of pespace_response"""
    rng = np.random.default_rng(11)
    th = W.draw_prior(6, 4e5, rng)
    th[:, 0] = 10.0 ** rng.uniform(5.8, 6.6, 6)
    th[:, 2] = rng.uniform(-0.5, 0.5, 6)
    dets = (W.lisa_like(gen), W.taiji_like(gen), W.tianqin_like(gen))
    model = W.Model(W.MODES_HM, dets)
    f = np.geomspace(3e-4, 8e-2, 150)
    t_lo, t_hi = time_span(th, model.mode_mask, f)
    dt = 300.0
    tab = W.orbit_table_from_fn(dets, t_lo, dt, int((t_hi - t_lo) / dt) + 2, oracle.orbit)
    got, want = check_response_orb(P, th, tab, f, model)
    ana = P.response(dev(th), dev(f), model).cpu().numpy()
    for d in range(3):
        assert np.abs(got[:, d] - ana[:, d]).max() <= 1e-8 * np.abs(ana[:, d]).max()


def test_orb_band_limits_edge_cases_and_determinism(P):
    wl = W.config(3, B=9, N=900)
    f = wl.grid.freqs()
    _, _, t22 = oracle.waveform(wl.theta_inj, 2, 2, f)
    t_lo, t_hi = time_span(wl.params, wl.model.mode_mask, f[[0, -1]])
    dt = 3600.0
    # a table that starts in the middle of the band's time span: early t_lm (low f) fall outside
    t_start = 0.5 * (t22[300] + t22[301])
    tab = W.synthetic_orbit_table(wl.model.detectors, t_start, dt, int((t_hi - t_start) / dt) + 2, seed=5)
    m22 = W.Model(W.MODES_22_ONLY, wl.model.detectors)
    inj = wl.theta_inj[None]
    r = P.response_orb(dev(inj), dev_orbit(P, tab), dev(f), m22).cpu().numpy()[0, 0]
    ro = oracle.response_orb(inj, tab, f, m22)[0, 0]
    assert np.all(r[:, :300] == 0) and np.all(ro[:, :300] == 0) and np.all(np.abs(r[0, 302:]) > 0)
    check_response_orb(P, wl.params, tab, f[::3], wl.model)
    psd = wl.psd()
    data = oracle.response_orb(inj, tab, f, wl.model)[0]
    lnL = check_loglike_orb(P, wl, tab, data, psd)
    lik = P.LikelihoodOrb(dev(data), dev(psd), wl.grid, wl.model, wl.B)
    assert np.array_equal(lik(dev(wl.params), dev_orbit(P, tab)).cpu().numpy(), lnL)
    # out-of-domain samples; K = 2 table; bad arguments
    th = wl.params.copy(); th[1, 0] = -5.0; th[3, 4] = np.nan
    got = lik(dev(th), dev_orbit(P, tab)).cpu().numpy()
    assert np.isneginf(got[1]) and np.isneginf(got[3]) and np.isfinite(got[0])
    two = (tab[0], (tab[2].shape[1] - 1) * tab[1], tab[2][:, [0, -1]], tab[3][:, [0, -1]])
    check_response_orb(P, wl.params[:2], two, f[400::50], wl.model)
    with pytest.raises(P.PespaceError):
        P.response_orb(dev(th), P.OrbitTable(0.0, -1.0, dev(tab[2]), dev(tab[3])), dev(f), wl.model)
    with pytest.raises(P.PespaceError):
        P.response_orb(dev(th), dev_orbit(P, tab), dev(f), W.config(4, B=2, N=10).model)     # 1 table, 3 detectors


def test_orb_full_size_sampled(P):
    """config 4's workload at B = 512 x N = 262144 with a synthetic ephemeris; oracle on 6 samples"""
    wl = W.config(4, B=512)
    f = wl.grid.freqs()
    t_lo, t_hi = time_span(wl.params[::37], wl.model.mode_mask, f[[0, -1]])
    dt = 900.0
    tab = W.synthetic_orbit_table(wl.model.detectors, t_lo - 3e5, dt, int((t_hi - t_lo + 6e5) / dt) + 2, seed=9)
    rng = np.random.default_rng(3)
    psd = wl.psd()
    data = P.response_orb(dev(wl.theta_inj[None]), dev_orbit(P, tab), dev(f), wl.model).cpu().numpy()[0]
    data = data + W.coloured_noise(psd, wl.grid.df, rng)
    got = P.LikelihoodOrb(dev(data), dev(psd), wl.grid, wl.model, wl.B)(dev(wl.params), dev_orbit(P, tab)).cpu().numpy()
    sub = np.array([0, 101, 202, 303, 404, 511])
    want = oracle.loglike_orb(wl.params[sub], tab, data, psd, wl.grid, wl.model)
    assert (np.abs(got[sub] - want) / np.abs(want)).max() <= TOL_LNL
