"""GPU-vs-oracle parity (run on the B200 box: pytest -m gpu).  Every call goes through the
C ABI of libpespace.so via the ctypes binding; expected values come from oracle/ only.

Tolerances (BASELINE.json north_star): lnL and <h|h> 1e-9 relative -- relative to
max(|lnL|, 1/2 <h|h>) (reading G14: lnL ~ 0 for a noiseless injection) -- and 1e-8
relative max-abs on the response arrays.  The response array of one (sample, detector) is
[3][N]; its error is measured against its max |.| (1e-8), and ALSO per channel against that
channel's own max |.| (1e-8) plus a cancellation floor of 1e-12 of the detector's max |.|:
T = (X+Y+Z)/sqrt3 cancels to ~(2 pi f L)^3 of A at low f (pin P8), so for the short-arm
TianQin-like detector below 1 mHz T is 1e-12 of A and is rounding noise in ANY double
evaluation, the oracle's included ("Tolerances").
"""
import math

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


def oracle_response_fn(params, freqs, model):
    return oracle.response(params, freqs, model)


def check_response(P, params, freqs, model):
    got = P.response(dev(params), dev(freqs), model).cpu().numpy()
    want = oracle.response(params, freqs, model)
    assert got.shape == want.shape
    for b in range(want.shape[0]):
        for d in range(want.shape[1]):
            det_scale = np.abs(want[b, d]).max()
            assert np.abs(got[b, d] - want[b, d]).max() <= TOL_RESP * det_scale
            for c in range(3):
                scale = np.abs(want[b, d, c]).max()
                err = np.abs(got[b, d, c] - want[b, d, c]).max()
                assert err <= TOL_RESP * scale + CANCEL_FLOOR * det_scale, (b, d, c, err / scale, err / det_scale)
    return got, want


def check_loglike(P, wl, data, psd, subset=None):
    import torch
    lik = P.Likelihood(dev(data), dev(psd), wl.grid, wl.model, wl.B)
    got = lik(dev(wl.params)).cpu().numpy()
    idx = np.arange(wl.B) if subset is None else np.asarray(subset)
    want = oracle.loglike(wl.params[idx], data, psd, wl.grid, wl.model)
    hh = -2.0 * oracle.loglike(wl.params[idx], np.zeros_like(data), psd, wl.grid, wl.model)
    scale = np.maximum(np.abs(want), 0.5 * hh)
    rel = np.abs(got[idx] - want) / scale
    assert np.all(rel <= TOL_LNL), (rel.max(), idx[np.argmax(rel)])
    # <h|h> itself (data = 0)
    lik0 = P.Likelihood(dev(np.zeros_like(data)), dev(psd), wl.grid, wl.model, wl.B)
    hh_gpu = -2.0 * lik0(dev(wl.params)).cpu().numpy()[idx]
    assert np.all(np.abs(hh_gpu - hh) <= TOL_LNL * hh)
    return got


# ------------------------------------------------------------------ config 1, in full
def test_config1_response_and_loglike_full(P):
    wl = W.config(1)
    f = wl.grid.freqs()
    check_response(P, wl.params, f, wl.model)
    data, psd = wl.data(oracle_response_fn), wl.psd()
    lnL = check_loglike(P, wl, data, psd)
    # noiseless injection = sample 0: lnL ~ 0 on the scale of <h|h>, and the maximum of the batch
    assert np.argmax(lnL) == 0


# ------------------------------------------------------------------ reduced configs 2-4: several tiles + ragged tails
@pytest.mark.parametrize("idx,B,N", [(2, 70, 3000), (3, 37, 1500), (4, 67, 1100)])
def test_reduced_configs_loglike_and_response(P, idx, B, N):
    wl = W.config(idx, B=B, N=N)
    data, psd = wl.data(oracle_response_fn), wl.psd()
    check_loglike(P, wl, data, psd)
    check_response(P, wl.params[:5], wl.grid.freqs()[::7], wl.model)


@pytest.mark.parametrize("gen", [15, 20])
def test_random_sky_all_detectors_both_generations(P, gen):
    """Prior draws (random sky, inclination, masses) through all three detector kinds."""
    rng = np.random.default_rng(11)
    grid = W.Grid(1e-4, 3.1e-5, 700)
    th = W.draw_prior(19, 4e5, rng)
    th[:, 2] = rng.uniform(-0.8, 0.8, 19); th[:, 3] = rng.uniform(-0.8, 0.8, 19)
    model = W.Model(W.MODES_HM, (W.lisa_like(gen), W.taiji_like(gen), W.tianqin_like(gen)))
    wl = W.Workload("random", grid, model, th, th[3].copy(), 77)
    data, psd = wl.data(oracle_response_fn), wl.psd()
    check_loglike(P, wl, data, psd)
    check_response(P, th, grid.freqs()[::5], model)


def test_nonzero_constellation_phases(P):
    """lambda0 != 0 (kind 0: constellation rotation phase, absorbed into the per-sample constants by a frame
    rotation; kind 1: orbital phase phi0), two kind-0 detectors with DIFFERENT lambda0 in one model."""
    import dataclasses
    rng = np.random.default_rng(23)
    th = W.draw_prior(7, 4e5, rng)
    dets = (dataclasses.replace(W.lisa_like(), lambda0=0.7), dataclasses.replace(W.taiji_like(15), lambda0=-2.1),
            dataclasses.replace(W.tianqin_like(), lambda0=1.1))
    model = W.Model(W.MODES_HM, dets)
    wl = W.Workload("phases", W.Grid(1e-4, 2.9e-5, 600), model, th, th[2].copy(), 78)
    data, psd = wl.data(oracle_response_fn), wl.psd()
    check_response(P, th, wl.grid.freqs()[::3], model)
    check_loglike(P, wl, data, psd)
    check_fisher(P, wl, data, psd)


@pytest.mark.parametrize("mask", [1, 2, 4, 8, 16, 9, 22])
def test_individual_modes(P, mask):
    wl = W.config(3, B=9, N=600)
    model = W.Model(mask, wl.model.detectors)
    check_response(P, wl.params, wl.grid.freqs(), model)


# ------------------------------------------------------------------ edge cases
def test_edge_cases(P):
    import torch
    wl = W.config(2, B=5, N=300)
    f = wl.grid.freqs()
    psd = wl.psd()
    data = wl.data(oracle_response_fn)
    # B = 1, N = 1
    one = W.Workload("one", W.Grid(3e-3, 1e-5, 1), wl.model, wl.params[:1], wl.theta_inj, None)
    check_loglike(P, one, np.full((1, 3, 1), 1e-20 + 2e-20j), one.psd())
    # zero / inf / nan PSD bins carry no weight; out-of-domain samples give -inf / NaN rows
    psd2 = psd.copy(); psd2[0, 0, 3] = 0.0; psd2[0, 1, 100] = np.inf; psd2[0, 2, 299] = np.nan; psd2[0, 0, 17] = -1.0
    th = wl.params.copy(); th[1, 0] = -5.0; th[3, 4] = np.nan
    got = P.loglike(dev(th), dev(data), dev(psd2), wl.grid, wl.model).cpu().numpy()
    want = oracle.loglike(th, data, psd2, wl.grid, wl.model)
    assert np.isneginf(got[1]) and np.isneginf(got[3]) and np.isneginf(want[1])
    ok = [0, 2, 4]
    assert np.all(np.abs(got[ok] - want[ok]) <= TOL_LNL * np.abs(want[ok]))
    r = P.response(dev(th), dev(f), wl.model).cpu().numpy()
    assert np.all(np.isnan(r[1].view(np.float64))) and np.all(np.isfinite(r[0].view(np.float64)))
    # f <= 0 bins produce zeros
    f2 = f.copy(); f2[0] = 0.0; f2[5] = -1e-3
    r2 = P.response(dev(wl.params), dev(f2), wl.model).cpu().numpy()
    assert np.all(r2[:, :, :, [0, 5]] == 0) and np.all(r2[:, :, :, 1] != 0)


def test_source_along_an_arm_is_regular(P):
    """k parallel to an arm at t_f(f): 1 - (k.n)^2 -> 0 (Eq. 5's sinc argument -> 0)."""
    th = W.THETA_INJ.copy(); th[10] = 2.0e6
    det = W.lisa_like()
    f0 = 1e-3
    _, _, t = oracle.waveform(th, 2, 2, np.array([f0]))
    x = oracle.orbit(det, t[0])
    n12 = (x[0] - x[1]) / det.L_m
    th[8] = -math.asin(n12[2]); th[7] = math.atan2(-n12[1], -n12[0])
    _, _, t2 = oracle.waveform(th, 2, 2, np.array([f0]))
    assert t2[0] == t[0]
    f = np.array([f0 * (1 - 1e-9), f0, f0 * (1 + 1e-9), 2e-3, 5e-3])
    check_response(P, th[None, :], f, W.Model(1, (det,)))


def test_special_angles_and_equal_masses(P):
    """Face-on / face-off (iota = 0, pi), ecliptic poles (beta = +-pi/2), equal masses (q = 1: the odd-m amplitudes
    vanish), psi = 0, phi_c = 0, t_c at the edges of the data."""
    wl = W.config(4, B=8, N=900)
    th = np.tile(wl.theta_inj, (8, 1))
    th[0, 5] = 0.0
    th[1, 5] = np.pi
    th[2, 8] = 0.5 * np.pi
    th[3, 8] = -0.5 * np.pi
    th[4, 1] = 1.0
    th[5, 9] = 0.0; th[5, 6] = 0.0
    th[6, 10] = 0.0
    th[7, 10] = 1.0 / wl.grid.df
    wl.params = th
    data, psd = wl.data(oracle_response_fn), wl.psd()
    check_loglike(P, wl, data, psd)
    check_response(P, th, wl.grid.freqs()[::4], wl.model)
    F, g = P.fisher(dev(th), dev(data), dev(psd), wl.grid, wl.model)
    Fo, go = oracle.fisher(th, data, psd, wl.grid, wl.model)
    d = np.sqrt(np.einsum("bii->bi", Fo))
    d = np.where(d > 0, d, 1.0)                       # q = 1: d/dq of the odd-m modes is the only content of that row
    assert (np.abs(F.cpu().numpy() - Fo) / (d[:, :, None] * d[:, None, :])).max() <= TOL_F


def test_bitwise_determinism(P):
    wl = W.config(3, B=130, N=2000)
    data, psd = wl.data(oracle_response_fn), wl.psd()
    lik = P.Likelihood(dev(data), dev(psd), wl.grid, wl.model, wl.B)
    p = dev(wl.params)
    a = lik(p).cpu().numpy()
    b = lik(p).cpu().numpy()
    assert np.array_equal(a, b)
    r1 = P.response(p, dev(wl.grid.freqs()), wl.model).cpu().numpy()
    r2 = P.response(p, dev(wl.grid.freqs()), wl.model).cpu().numpy()
    assert np.array_equal(r1.view(np.float64), r2.view(np.float64))


def test_response_against_the_binary128_oracle(P):
    """The CUDA path against the oracle evaluated in IEEE binary128 (pin P14's reference): the split phase reduction
    (f t_c and the PN phase reduced modulo one turn before they are added) keeps the FP64 kernel as close to the exact
    definition as the plain double oracle is."""
    wl = W.config(1)
    f = wl.grid.freqs()[::64]
    rq = oracle.response(wl.params, f, wl.model, quad=True)
    ro = oracle.response(wl.params, f, wl.model)
    rg = P.response(dev(wl.params), dev(f), wl.model).cpu().numpy()
    scale = np.abs(rq).max(axis=(2, 3), keepdims=True)
    err_gpu, err_cpu = (np.abs(rg - rq) / scale).max(), (np.abs(ro - rq) / scale).max()
    assert err_gpu <= 1e-11, err_gpu                 # measured 2.1e-13 (double oracle: 3.8e-12)
    assert err_gpu <= 2.0 * err_cpu + 1e-13, (err_gpu, err_cpu)
    print(f"max error vs binary128: CUDA {err_gpu:.2e}, double oracle {err_cpu:.2e}")


def test_host_buffer_call_matches_device_call(P):
    wl = W.config(4, B=33, N=900)
    data, psd = wl.data(oracle_response_fn), wl.psd()
    a = P.loglike_host(wl.params, data, psd, wl.grid, wl.model)
    b = P.loglike(dev(wl.params), dev(data), dev(psd), wl.grid, wl.model).cpu().numpy()
    assert np.array_equal(a, b)


def test_session_matches_device_calls_and_oracle(P):
    """pespace_session_*: host buffers in, host buffers out; same kernels, so bit-identical to the device-pointer
    calls, and within tolerance of the oracle.  Pinned torch tensors and numpy arrays are both accepted."""
    import torch
    wl = W.config(4, B=37, N=1100)
    data, psd = wl.data(oracle_response_fn), wl.psd()
    ses = P.Session(wl.grid, wl.model, 64, want_fisher=True)
    with pytest.raises(P.PespaceError):
        ses.loglike(wl.params)                                   # no data yet
    ses.set_data(None, psd)
    F0, none = ses.fisher(wl.params, with_grad=False)             # the Fisher matrix needs only the PSD
    assert none is None
    with pytest.raises(P.PespaceError):
        ses.fisher(wl.params, with_grad=True)                    # the gradient needs the data
    ses.set_data(torch.from_numpy(data).pin_memory(), None)
    a = ses.loglike(wl.params)
    b = P.loglike(dev(wl.params), dev(data), dev(psd), wl.grid, wl.model).cpu().numpy()
    assert np.array_equal(a, b)
    want = oracle.loglike(wl.params, data, psd, wl.grid, wl.model)
    assert np.all(np.abs(a - want) <= TOL_LNL * np.abs(want))
    out = torch.empty(20, dtype=torch.float64).pin_memory()
    ses.loglike(torch.from_numpy(wl.params[:20]).pin_memory(), out)   # smaller batch, pinned buffers
    assert np.array_equal(out.numpy(), a[:20])
    F, g = ses.fisher(wl.params)
    Fd, gd = P.fisher(dev(wl.params), dev(data), dev(psd), wl.grid, wl.model)
    assert np.array_equal(F, Fd.cpu().numpy()) and np.array_equal(g, gd.cpu().numpy())
    assert np.array_equal(F0, F)
    # the per-bin table is cached per data set: a new data set must invalidate it
    ses.set_data(np.zeros_like(data), None)
    z = ses.loglike(wl.params)
    assert np.array_equal(z, P.loglike(dev(wl.params), dev(np.zeros_like(data)), dev(psd), wl.grid, wl.model).cpu().numpy())
    ses.set_data(data, None)
    assert np.array_equal(ses.loglike(wl.params), a)
    with pytest.raises(P.PespaceError):
        ses.loglike(np.tile(wl.params, (2, 1)))                  # batch larger than max_B
    ses.close()
    ses.close()                                                  # idempotent


def test_error_codes_on_device(P):
    wl = W.config(2, B=4, N=64)
    data, psd = dev(wl.data(oracle_response_fn)), dev(wl.psd())
    with pytest.raises(P.PespaceError):
        P.loglike(dev(wl.params), data, psd, W.Grid(1e-4, 0.0, 64), wl.model)
    with pytest.raises(P.PespaceError):
        P.loglike(dev(wl.params), data, psd, wl.grid, W.Model(64, wl.model.detectors))
    lik = P.Likelihood(data, psd, wl.grid, wl.model, 2)
    with pytest.raises(P.PespaceError):
        lik(dev(wl.params))                     # batch larger than the workspace


# ------------------------------------------------------------------ full size, sampled (bench.py's launch configuration)
@pytest.mark.parametrize("idx,stride_div", [(2, 32), (3, 16)])
def test_full_size_sampled_parity(P, idx, stride_div):
    wl = W.config(idx)
    data, psd = wl.data(oracle_response_fn), wl.psd()
    step = -(-wl.B // stride_div)
    subset = sorted(set([0] + list(range(0, wl.B, step))))
    check_loglike(P, wl, data, psd, subset=subset)


def test_full_size_network_sampled_parity(P):
    wl = W.config(4)
    data, psd = wl.data(oracle_response_fn), wl.psd()
    subset = [0, 1023, 4097, 8191]
    check_loglike(P, wl, data, psd, subset=subset)


# ------------------------------------------------------------------ S10: forward-mode derivatives (Eq. 13, 14)
# Tolerance: the Fisher matrix is a Gram matrix of the tangents d_i h, so an entry is
# compared on the Cauchy-Schwarz scale of its row and column, |dF_ij| <= 1e-9 sqrt(F_ii F_jj); the gradient
# <d - h | d_i h> on the scale sqrt(F_ii <d-h|d-h>).  1e-9 is the north-star tolerance of <h|h>.
TOL_F = 1e-9


def check_fisher(P, wl, data, psd, subset=None, with_grad=True):
    idx = np.arange(wl.B) if subset is None else np.asarray(subset)
    F, g = P.fisher(dev(wl.params), dev(data) if with_grad else None, dev(psd), wl.grid, wl.model)
    F = F.cpu().numpy()
    Fo, go = oracle.fisher(wl.params[idx], data if with_grad else None, psd, wl.grid, wl.model)
    d = np.sqrt(np.einsum("bii->bi", Fo))
    assert np.all(d > 0)
    errF = np.abs(F[idx] - Fo) / (d[:, :, None] * d[:, None, :])
    assert errF.max() <= TOL_F, errF.max()
    assert np.array_equal(F, F.transpose(0, 2, 1))
    if with_grad:
        rr = -2.0 * oracle.loglike(wl.params[idx], data, psd, wl.grid, wl.model)
        errg = np.abs(g.cpu().numpy()[idx] - go) / (d * np.sqrt(rr)[:, None])
        assert errg.max() <= TOL_F, errg.max()
    else:
        assert g is None
    return F


def test_fisher_config1_full(P):
    wl = W.config(1)
    data, psd = wl.data(oracle_response_fn), wl.psd()
    # noiseless data = h(sample 0): every other sample has a non-zero residual; sample 0 has d - h = 0 and
    # its gradient is compared on the scale of the batch
    F, g = P.fisher(dev(wl.params), dev(data), dev(psd), wl.grid, wl.model)
    Fo, go = oracle.fisher(wl.params, data, psd, wl.grid, wl.model)
    d = np.sqrt(np.einsum("bii->bi", Fo))
    assert (np.abs(F.cpu().numpy() - Fo) / (d[:, :, None] * d[:, None, :])).max() <= TOL_F
    rr = -2.0 * oracle.loglike(wl.params, data, psd, wl.grid, wl.model)
    hh = -2.0 * oracle.loglike(wl.params, np.zeros_like(data), psd, wl.grid, wl.model)
    scale = d * np.sqrt(np.maximum(rr, hh))[:, None]
    assert (np.abs(g.cpu().numpy() - go) / scale).max() <= TOL_F


@pytest.mark.parametrize("idx,B,N", [(2, 11, 5000), (3, 6, 2100), (5, 9, 2300)])
def test_fisher_reduced_configs(P, idx, B, N):
    """several chunks (128 bins), several blocks (2048 bins), ragged tails in bins and samples"""
    wl = W.config(idx, B=B, N=N)
    data, psd = wl.data(oracle_response_fn), wl.psd()
    check_fisher(P, wl, data, psd)
    check_fisher(P, wl, data, psd, with_grad=False)


@pytest.mark.parametrize("gen", [15, 20])
def test_fisher_random_sky_spinning(P, gen):
    rng = np.random.default_rng(5)
    th = W.draw_prior(9, 4e5, rng)
    th[:, 2] = rng.uniform(-0.8, 0.8, 9); th[:, 3] = rng.uniform(-0.8, 0.8, 9)
    model = W.Model(W.MODES_HM, (W.lisa_like(gen), W.taiji_like(gen), W.tianqin_like(gen)))
    wl = W.Workload("random", W.Grid(1e-4, 3.1e-5, 700), model, th, th[3].copy(), 77)
    check_fisher(P, wl, wl.data(oracle_response_fn), wl.psd())


@pytest.mark.parametrize("mask", [2, 4, 8, 16, 9, 22])
def test_fisher_individual_modes(P, mask):
    wl = W.config(3, B=5, N=400)
    wl = W.Workload("modes", wl.grid, W.Model(mask, wl.model.detectors), wl.params, wl.theta_inj, 5)
    check_fisher(P, wl, wl.data(oracle_response_fn), wl.psd())


def test_fisher_edge_cases_and_determinism(P):
    wl = W.config(5, B=6, N=300)
    data, psd = wl.data(oracle_response_fn), wl.psd()
    psd2 = psd.copy(); psd2[0, 0, 3] = 0.0; psd2[1, 1, 100] = np.inf; psd2[2, 2, 299] = np.nan
    th = wl.params.copy(); th[1, 0] = -5.0; th[4, 4] = np.nan
    F, g = P.fisher(dev(th), dev(data), dev(psd2), wl.grid, wl.model)
    F2, g2 = P.fisher(dev(th), dev(data), dev(psd2), wl.grid, wl.model)
    F, g = F.cpu().numpy(), g.cpu().numpy()
    assert np.array_equal(F, F2.cpu().numpy(), equal_nan=True) and np.array_equal(g, g2.cpu().numpy(), equal_nan=True)
    assert np.all(np.isnan(F[[1, 4]])) and np.all(np.isnan(g[[1, 4]]))
    ok = [0, 2, 3, 5]
    Fo, go = oracle.fisher(th[ok], data, psd2, wl.grid, wl.model)
    d = np.sqrt(np.einsum("bii->bi", Fo))
    assert (np.abs(F[ok] - Fo) / (d[:, :, None] * d[:, None, :])).max() <= TOL_F


def test_fisher_gradient_only_mode(P):
    """pespace_fisher with d_out_F = NULL returns d lnL / d theta alone: within tolerance of the oracle and of the
    full call (the reduction tree differs, so not bit-identical), deterministic, also through a session."""
    wl = W.config(5, B=13, N=2500)
    data, psd = wl.data(oracle_response_fn), wl.psd()
    fis = P.Fisher(dev(data), dev(psd), wl.grid, wl.model, wl.B)
    none, g = fis(dev(wl.params), grad_only=True)
    assert none is None
    g = g.cpu().numpy()
    Fo, go = oracle.fisher(wl.params, data, psd, wl.grid, wl.model)
    d = np.sqrt(np.einsum("bii->bi", Fo))
    rr = -2.0 * oracle.loglike(wl.params, data, psd, wl.grid, wl.model)
    assert (np.abs(g - go) / (d * np.sqrt(rr)[:, None])).max() <= TOL_F
    assert np.array_equal(g, fis(dev(wl.params), grad_only=True)[1].cpu().numpy())
    ses = P.Session(wl.grid, wl.model, wl.B, want_fisher=True)
    ses.set_data(data, psd)
    assert np.array_equal(ses.fisher(wl.params, grad_only=True)[1], g)
    ses.close()
    with pytest.raises(P.PespaceError):
        P.Fisher(None, dev(psd), wl.grid, wl.model, wl.B)(dev(wl.params), grad_only=True)


def test_fisher_gradient_is_the_derivative_of_loglike(P):
    """d lnL / d theta_i from pespace_fisher against a central difference of pespace_loglike (GPU only):
    ties the two entry points together at a size where the oracle would take minutes."""
    wl = W.config(3, B=4, N=20000)
    data, psd = wl.data(oracle_response_fn), wl.psd()
    _, g = P.fisher(dev(wl.params), dev(data), dev(psd), wl.grid, wl.model)
    g = g.cpu().numpy()
    lik = P.Likelihood(dev(data), dev(psd), wl.grid, wl.model, wl.B)
    for i, h in [(4, 1e-6), (5, 1e-7), (6, 1e-7), (9, 1e-7)]:      # D_L, iota, phi_c, psi
        tp, tm = wl.params.copy(), wl.params.copy()
        tp[:, i] += h; tm[:, i] -= h
        fd = (lik(dev(tp)).cpu().numpy() - lik(dev(tm)).cpu().numpy()) / (2 * h)
        assert np.allclose(fd, g[:, i], rtol=2e-5, atol=1e-3 * np.abs(g[:, i]).max()), (i, fd, g[:, i])


def test_fisher_full_size_sampled_parity(P):
    """config 5 at full size (B = 256 x N = 262144, three detectors, five modes), oracle on 4 samples"""
    wl = W.config(5)
    data, psd = wl.data(oracle_response_fn), wl.psd()
    check_fisher(P, wl, data, psd, subset=[0, 85, 170, 255])


# ------------------------------------------------------------------ multi-GPU plumbing on one GPU
def test_sharded_likelihood_with_the_real_binding_under_nccl(P):
    """dist.ShardedLikelihood driving binding.Likelihood inside a one-rank NCCL group (the all-gather path is taken
    even at world size 1): bit-identical to the plain call.  This is as far as one GPU goes; the world-size-2 host
    logic is covered on gloo (tests/test_dist_gloo.py)."""
    import socket
    import torch
    import torch.distributed as dist
    from paper_2602_12011_b200 import dist as pdist
    wl = W.config(3, B=70, N=3000)
    data, psd = wl.data(oracle_response_fn), wl.psd()
    lik = P.Likelihood(dev(data), dev(psd), wl.grid, wl.model, wl.B)
    plain = lik(dev(wl.params)).cpu().numpy()
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    assert not dist.is_initialized()
    dist.init_process_group("nccl", init_method=f"tcp://127.0.0.1:{port}", rank=0, world_size=1)
    try:
        rep_d, rep_p = pdist.replicate(dev(data), dev(psd))                     # NCCL broadcast (one rank: identity)
        assert torch.equal(torch.view_as_real(rep_d), torch.view_as_real(dev(data))) and torch.equal(rep_p, dev(psd))
        sharded = pdist.ShardedLikelihood(lambda p: lik(p))
        got = sharded(dev(wl.params)).cpu().numpy()
        assert np.array_equal(got, plain)
        t_max, units = pdist.aggregate(12.5, wl.B, torch.device("cuda", torch.cuda.current_device()))
        assert t_max == 12.5 and units == wl.B
        assert np.array_equal(pdist.gather_lnL(plain, torch.device("cuda", torch.cuda.current_device())), plain)
        # the calls with several outputs: adjoint gradient (lnL, grad) and Fisher matrix (F, grad)
        th = dev(wl.params[:9])
        lg = P.LikelihoodGrad(dev(data), dev(psd), wl.grid, wl.model, 9)
        want_l, want_g = (x.clone() for x in lg(th))
        got_l, got_g = pdist.ShardedCall(lambda p: lg(p))(th)
        assert torch.equal(got_l, want_l) and torch.equal(got_g, want_g)
        fi = P.Fisher(dev(data), dev(psd), wl.grid, wl.model, 9)
        want_F, want_fg = (x.clone() for x in fi(th))
        got_F, got_fg = pdist.ShardedCall(lambda p: fi(p))(th)
        assert torch.equal(got_F, want_F) and torch.equal(got_fg, want_fg)
        none_F, only_g = pdist.ShardedCall(lambda p: fi(p, grad_only=True))(th)
        assert none_F is None and only_g.shape == (9, 11)
    finally:
        dist.destroy_process_group()


# ------------------------------------------------------------------ fused multi-detector kernel: model shapes
@pytest.mark.parametrize("mask,n_det", [(1, 2), (W.MODES_HM, 8), (20, 5), (2, 3)])
def test_fused_kernel_detector_counts_and_masks(P, mask, n_det):
    """models with 2 ... PESPACE_MAX_DET detectors of mixed kinds (one launch, waveform part shared): lnL against the
    oracle, and against the sum of the one-detector calls (each detector alone goes through loglike_kernel)"""
    import dataclasses
    protos = [W.lisa_like(), W.tianqin_like(), W.taiji_like(15), dataclasses.replace(W.lisa_like(15), lambda0=0.9),
              dataclasses.replace(W.tianqin_like(15), lambda0=-0.4), W.taiji_like(),
              dataclasses.replace(W.lisa_like(), kappa=0.3, L_m=2.0e9), dataclasses.replace(W.tianqin_like(), lon=0.3, lat=0.5)]
    dets = tuple(protos[:n_det])
    rng = np.random.default_rng(40 + n_det)
    th = W.draw_prior(67, 4e5, rng)
    wl = W.Workload("fused", W.Grid(1.2e-4, 2.7e-5, 700), W.Model(mask, dets), th, th[1].copy(), 50 + n_det)
    data, psd = wl.data(oracle_response_fn), wl.psd()
    got = check_loglike(P, wl, data, psd)
    one_by_one = np.zeros(wl.B)
    for d, det in enumerate(dets):
        one_by_one += P.loglike(dev(th), dev(data[d:d + 1]), dev(psd[d:d + 1]), wl.grid, W.Model(mask, (det,))).cpu().numpy()
    assert np.allclose(got, one_by_one, rtol=1e-12, atol=0)
    # pespace_response of the same model (response_fused_kernel) against the oracle and the one-detector calls
    # (response_kernel); non-positive and repeated frequencies, out-of-domain sample, ragged bin block
    f = wl.grid.freqs()[::3].copy()
    thr = th[:9].copy()
    resp, _ = check_response(P, thr, f, wl.model)
    f[5] = 0.0; f[6] = -1e-3; f[7] = f[8]
    thr[4, 4] = -1.0
    resp = P.response(dev(thr), dev(f), wl.model).cpu().numpy()
    assert np.all(np.delete(resp, 4, axis=0)[..., 5:7] == 0.0)          # f <= 0: zeros
    assert np.all(np.isnan(resp[4])) and np.all(np.isfinite(np.delete(resp, 4, axis=0)))
    assert np.array_equal(np.delete(resp, 4, axis=0)[..., 7], np.delete(resp, 4, axis=0)[..., 8])
    for d, det in enumerate(dets):
        one = P.response(dev(thr), dev(f), W.Model(mask, (det,))).cpu().numpy()[:, 0]
        ok = np.delete(np.arange(9), 4)
        scale = np.abs(one[ok]).max(axis=(1, 2), keepdims=True)
        assert np.all(np.abs(resp[ok, d] - one[ok]) <= 1e-11 * scale)
    assert np.array_equal(resp[np.isfinite(resp)], P.response(dev(thr), dev(f), wl.model).cpu().numpy()[np.isfinite(resp)])


# ------------------------------------------------------------------ prepared data
@pytest.mark.parametrize("idx,B,N", [(2, 70, 3000), (4, 67, 1100)])
def test_prepared_calls_are_bit_identical_to_the_plain_ones(P, idx, B, N):
    """pespace_prepare once, then pespace_loglike_prepared / pespace_loglike_grad_prepared for several batches
    (full, smaller, one sample) against the same workspace: bit-identical to pespace_loglike / pespace_loglike_grad,
    which rebuild the per-bin table on every call; the table survives the calls, a mixed-precision call in between
    invalidates it and the binding falls back to the plain call."""
    import torch
    wl = W.config(idx, B=B, N=N)
    data, psd = wl.data(oracle_response_fn), wl.psd()
    th = dev(wl.params)
    plain = P.Likelihood(dev(data), dev(psd), wl.grid, wl.model, B)
    want = plain(th).clone()
    prep = P.Likelihood(dev(data), dev(psd), wl.grid, wl.model, B).prepare()
    n0 = P.launch_count()
    got = prep(th).clone()
    assert P.launch_count() - n0 == 3                                     # prep_samples, main kernel, combine
    assert prep.prepared and torch.equal(got, want)
    for b in (B - 7, 1):
        assert torch.equal(prep(th[:b].contiguous()), want[:b])
    check_loglike(P, wl, data, psd)                                       # and the oracle agrees (plain path)
    mixed = prep(th, mixed=True)
    assert not prep.prepared and torch.isfinite(mixed).all()
    assert torch.equal(prep(th), want)                                    # plain call again (rebuilds the table)
    # gradient twin: one pespace_prepare on the larger workspace serves it
    pg = P.LikelihoodGrad(dev(data), dev(psd), wl.grid, wl.model, B)
    want_l, want_g = (x.clone() for x in pg(th))
    pg.prepare()
    got_l, got_g = pg(th)
    assert torch.equal(got_l, want_l) and torch.equal(got_g, want_g)
    got_l, got_g = pg(th[:5].contiguous())
    assert torch.equal(got_l, want_l[:5]) and torch.equal(got_g, want_g[:5])
    with pytest.raises(P.PespaceError):
        P.LikelihoodOrb(dev(data), dev(psd), wl.grid, wl.model, B).prepare()
