"""Seeded random sweep of the analytic path against the oracle: shapes, grids, mode sets, detector sets and parameters
that no hand-written case has -- batch sizes around the tile sizes (31 ... 129), bin counts around the block sizes
(31 ... 2049), bands anywhere in 0.1-120 mHz, any of the 31 mode masks, one to four detectors of either kind and TDI
generation with perturbed arm lengths and orbital phases, spins, negative t_c.  Every case goes through the checkers
of the parity tests with their tolerances (1e-9 on lnL, <h|h>, gradient and Fisher entries, 1e-8 on response arrays).

Sums over at least 31 bins only: a one- or two-bin "likelihood" is the single-bin regime of DESIGN.md section 10, where
the floors of the per-bin tolerances apply instead of the flat 1e-9 (tests/test_gpu_fullband.py covers that regime).
t_c is drawn inside the observation span 1/df of the case's own grid, as in every config of BASELINE.json."""
import dataclasses

import numpy as np
import pytest

from paper_2602_12011_b200 import workloads as W
from test_gpu_grad import check_grad
from test_gpu_parity import check_fisher, check_loglike, check_response, oracle_response_fn

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
            if case % 3 == 0:
                sub = list(range(min(wl.B, 3)))
                check_grad(P, wl, data, psd, subset=sub)
                check_fisher(P, wl, data, psd, subset=sub)
        except AssertionError as exc:
            raise AssertionError(f"case {case}: B={wl.B} N={wl.grid.N} f0={wl.grid.f0:.4e} df={wl.grid.df:.4e} "
                                 f"mask={wl.model.mode_mask} detectors="
                                 f"{[(d.kind, d.tdi_gen, d.L_m) for d in wl.model.detectors]}: {exc}") from exc
