"""Seeded random sweep of the analytic path against the oracle: shapes, grids, mode sets, detector sets and parameters
that no hand-written case has -- batch sizes around the tile sizes (31 ... 129), bin counts around the block sizes
(31 ... 2049), bands anywhere in 0.1-120 mHz, any of the 31 mode masks, one to four detectors of either kind and TDI
generation with perturbed arm lengths and orbital phases, spins, negative t_c.  Every case goes through the checkers
of the parity tests with their tolerances (1e-9 on lnL, <h|h>, gradient and Fisher entries, 1e-8 on response arrays);
every second case also runs the mixed-precision likelihood against its stated error bound.

Sums over at least 31 bins only: a one- or two-bin "likelihood" is the single-bin regime of DESIGN.md section 10, where
the floors of the per-bin tolerances apply instead of the flat 1e-9 (tests/test_gpu_fullband.py covers that regime).
t_c is drawn inside the observation span 1/df of the case's own grid, as in every config of BASELINE.json."""
import dataclasses

import numpy as np
import pytest

from paper_2602_12011_b200 import workloads as W
from test_gpu_grad import check_grad
from test_gpu_parity import check_fisher, check_loglike, check_response, dev, oracle_response_fn

pytestmark = pytest.mark.gpu

N_CASES = 160


@pytest.fixture(scope="module")
def P():
    import torch
    from paper_2602_12011_b200 import binding
    assert torch.cuda.is_available()
    return binding


def random_case(case: int):
    rng = np.random.default_rng(770000 + case)
    B = int(rng.choice([1, 2, 3, 5, 31, 33, 63, 65, 100, 129]))
    N = int(rng.choice([31, 255, 257, 511, 1025, 1500, 2049]))
    f0 = 10.0 ** rng.uniform(-4.0, -2.0)
    fmax = min(0.12, f0 * 10.0 ** rng.uniform(0.3, 2.5))
    df = (fmax - f0) / N
    grid = W.Grid(f0, df, N)
    mask = int(rng.integers(1, 32))
    dets = []
    for _ in range(int(rng.choice([1, 1, 2, 3, 4]))):
        proto = [W.lisa_like, W.taiji_like, W.tianqin_like][int(rng.integers(0, 3))](int(rng.choice([15, 20])))
        change = {"lambda0": float(rng.uniform(-3.0, 3.0))}
        if rng.random() < 0.5:
            change["L_m"] = proto.L_m * float(rng.uniform(0.5, 1.5))
        if proto.kind == 0 and rng.random() < 0.5:
            change["kappa"] = float(rng.uniform(-1.0, 1.0))
        if proto.kind == 1 and rng.random() < 0.5:
            change["lon"], change["lat"] = float(rng.uniform(0.0, 6.28)), float(rng.uniform(-1.5, 1.5))
        dets.append(dataclasses.replace(proto, **change))
    th = W.draw_prior(B, 1.0 / df, rng)
    th[:, 2], th[:, 3] = rng.uniform(-0.9, 0.9, B), rng.uniform(-0.9, 0.9, B)
    if rng.random() < 0.3:
        th[:, 10] -= rng.uniform(0.0, 0.3 / df)                       # coalescence before the start of the data
    return W.Workload("sweep%d" % case, grid, W.Model(mask, tuple(dets)), th, th[0].copy(), int(rng.integers(1, 1000)))


def check_mixed(P, wl, data, psd):
    """pespace_loglike_mixed is an approximation by design: 5e-6 of max(|lnL|, <h|h>/2) on the BASELINE configs
    (tests/test_gpu_mixed.py), plus 5e-7 / x_min with x_min = 2 pi f0 L / c of the shortest arm: FP32 brackets are
    O(x) quantities known to 6e-8 (include/pespace.h)"""
    import oracle
    x_min = min(2.0 * np.pi * wl.grid.f0 * d.L_m / W.C_SI for d in wl.model.detectors)
    tol = 5e-6 + 5e-7 / x_min
    lik = P.Likelihood(dev(data), dev(psd), wl.grid, wl.model, wl.B)
    got = lik(dev(wl.params), mixed=True).cpu().numpy()
    want = oracle.loglike(wl.params, data, psd, wl.grid, wl.model)
    hh = -2.0 * oracle.loglike(wl.params, np.zeros_like(data), psd, wl.grid, wl.model)
    assert np.all(np.isfinite(got))
    rel = np.abs(got - want) / np.maximum(np.abs(want), 0.5 * hh)
    assert rel.max() <= tol, ("mixed", rel.max(), tol)


@pytest.mark.parametrize("chunk", range(8))
def test_random_models_shapes_and_parameters(P, chunk):
    per = N_CASES // 8
    for case in range(chunk * per, (chunk + 1) * per):
        wl = random_case(case)
        psd = wl.psd()
        data = wl.data(oracle_response_fn)
        try:
            check_loglike(P, wl, data, psd)
            check_response(P, wl.params[:4], wl.grid.freqs()[::max(1, wl.grid.N // 300)], wl.model)
            if case % 2 == 0:
                check_mixed(P, wl, data, psd)
            if case % 3 == 0:
                sub = list(range(min(wl.B, 3)))
                check_grad(P, wl, data, psd, subset=sub)
                check_fisher(P, wl, data, psd, subset=sub)
        except AssertionError as exc:
            raise AssertionError(f"case {case}: B={wl.B} N={wl.grid.N} f0={wl.grid.f0:.4e} df={wl.grid.df:.4e} "
                                 f"mask={wl.model.mode_mask} detectors="
                                 f"{[(d.kind, d.tdi_gen, d.L_m) for d in wl.model.detectors]}: {exc}") from exc


@pytest.mark.parametrize("chunk", range(4))
def test_random_tables_waveforms_and_orbits(P, chunk):
    """the tabulated paths on the same random models: waveform tables of 4 ... 300 nodes that may start late or end
    early inside the band (pespace_loglike_tab, pespace_response_tab, the Fisher matrix of pespace_fisher_tab), and
    seeded toy ephemerides of 50 ... 3000 nodes that may start after the earliest t_lm (pespace_loglike_orb,
    pespace_response_orb).  The gradient of pespace_fisher_tab is left to tests/test_gpu_tab.py: its checker scales
    the error by the residual alone, which is meaningless at the SNRs of 1e6 and more that random amplitudes give."""
    import oracle
    import test_gpu_orb as TO
    import test_gpu_tab as TT
    per = 12
    for case in range(1000 + chunk * per, 1000 + (chunk + 1) * per):
        wl = random_case(case)
        rng = np.random.default_rng(case)
        wl = W.Workload(wl.name, wl.grid, wl.model, wl.params[:min(wl.B, 40)], wl.theta_inj, wl.noise_seed)
        f = wl.grid.freqs()
        psd = wl.psd()
        sub = max(1, wl.grid.N // 200)
        try:
            K = int(rng.choice([4, 5, 17, 64, 300]))
            lo = f[0] * (1.0 if rng.random() < 0.6 else rng.uniform(1.0, 1.5))
            hi = f[-1] * (1.0 if rng.random() < 0.6 else rng.uniform(0.6, 1.0))
            if hi <= lo * 1.01:
                hi = lo * 1.5
            table = W.chirp_table(wl.params, wl.model.mode_mask, W.log_nodes(lo, hi, K))
            head = tuple(x if x.ndim == 1 else x[:3] for x in table)
            data, _ = TT.noisy_data(wl, table)
            TT.check_loglike_tab(P, wl.params, table, data, psd, wl.grid, wl.model)
            TT.check_response_tab(P, wl.params[:3], head, f[::sub], wl.model)
            TT.check_fisher_tab(P, wl.params[:3], head, None, psd, wl.grid, wl.model, with_grad=False)
            if case % 2 == 0:
                t_lo, t_hi = TO.time_span(wl.params, wl.model.mode_mask, f[[0, -1]])
                if rng.random() < 0.3:
                    t_lo = t_lo + 0.3 * (t_hi - t_lo)                       # a table that starts late
                Kt = int(rng.choice([50, 400, 3000]))
                dt = max(t_hi - t_lo, 1000.0) / (Kt - 3)
                tab = W.synthetic_orbit_table(wl.model.detectors, t_lo - dt, dt, Kt, seed=case)
                d3 = oracle.response_orb(wl.theta_inj[None], tab, f, wl.model)[0] + W.coloured_noise(psd, wl.grid.df, rng)
                TO.check_loglike_orb(P, wl, tab, d3, psd)
                TO.check_response_orb(P, wl.params[:3], tab, f[::sub], wl.model)
        except AssertionError as exc:
            raise AssertionError(f"case {case}: B={wl.B} N={wl.grid.N} f0={wl.grid.f0:.4e} df={wl.grid.df:.4e} "
                                 f"mask={wl.model.mode_mask} detectors="
                                 f"{[(d.kind, d.tdi_gen, d.L_m) for d in wl.model.detectors]}: {exc}") from exc
