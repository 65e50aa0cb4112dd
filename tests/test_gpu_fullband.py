"""GPU-vs-oracle parity over the WHOLE band of configs 2-5 (0.1 ... 101.2 mHz), bin by bin.

The reduced configs of test_gpu_parity.py keep df = 1/(30 d) and the first N bins, so they stop at about 1.3 mHz.
Here the response is compared element-wise on a strided sample of the full 262144-bin grid plus +-3 bins around every
in-band null of the TDI prefactor g(z) of Eq. 6 (n c/4L for generation 2.0, n c/2L for
1.5), which also covers the region v > 1 where t_22 - t_c turns positive (G2) and arm phases 2 pi f L of several
turns.  Tolerance PER BIN (not per array, so that a frequency-local error cannot hide behind the large low-frequency
amplitudes): with s_k = max_c |h_c(f_k)| of the oracle,

    |got_c(f_k) - want_c(f_k)| <= 1e-8 |want_c(f_k)| + FLOOR(f_k) s_k,
    FLOOR(f) = 16 eps (1 + 1/x) + 4 eps 2 pi f / df,     x = 2 pi f L / c,  eps = 2^-52

(`bin_floor`).  First term: both sides form X, Y, Z from six single links of relative rounding error eps whose sum
cancels to O(x) of a link (the long-wavelength limit, pin P7) and, for T = (X+Y+Z)/sqrt3, to O(x^3) (pin P8): the
absolute rounding noise of ANY double evaluation is ~ eps |y| ~ (eps / x) s_k per bin, the oracle's included.
Second term: the oracle adds 2 pi f t_c (up to 2 pi f / df = 1.6e6 rad at the top of the band) to the PN phase in
double, i.e. it carries an absolute phase error of a few eps |phase| (pin P14 over the band: the double oracle is
6e-10 from its own binary128 evaluation at 0.1 Hz; the CUDA path, which reduces the two phases separately, 5e-13).
A channel therefore agrees to 1e-8 of ITSELF or, where it is small against its neighbours (T at low f, a channel
passing through zero), to better than 1e-9 of the bin's largest channel.

The per-bin analogue for the derivatives (S10) runs pespace_fisher on ONE-bin grids: F_ij is then
4 df sum_c Re[conj(d_i h_c) d_j h_c] / S_c of that bin alone, compared entry by entry on the Cauchy-Schwarz scale.
"""
import dataclasses

import numpy as np
import pytest

import oracle
from paper_2602_12011_b200 import workloads as W

pytestmark = pytest.mark.gpu

TOL_RESP = 1e-8
TOL_LNL = 1e-9
TOL_F = 1e-9
EPS = 2.220446049250313e-16
C_SI = 299792458.0


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


def null_frequencies(det, f_lo, f_hi):
    """zeros of g(z) of Eq. 6 inside (f_lo, f_hi): z^2 = 1 at n c/2L; generation 2.0 adds z^4 = 1 at n c/4L"""
    step = C_SI / ((4.0 if det.tdi_gen == 20 else 2.0) * det.L_m)
    n = np.arange(1, int(f_hi / step) + 1)
    f = n * step
    return f[(f > f_lo) & (f < f_hi)]


def band_indices(grid, dets, stride=257, around=3):
    """strided sample of the grid + the bins within `around` of every in-band null of every detector"""
    f = grid.freqs()
    idx = set(range(0, grid.N, stride)) | {grid.N - 1}
    n_null = 0
    for det in dets:
        for fn in null_frequencies(det, f[0], f[-1]):
            k0 = int(round((fn - grid.f0) / grid.df))
            idx |= {k for k in range(k0 - around, k0 + around + 1) if 0 <= k < grid.N}
            n_null += 1
    return np.array(sorted(idx)), n_null


def cancel_floor(det, f):
    """rounding noise of the link sums relative to the bin's largest channel: 16 eps (1 + 1/x) (module docstring)"""
    x = 2.0 * np.pi * f * det.L_m / C_SI
    return 16.0 * EPS * (1.0 + 1.0 / x)


def bin_floor(det, f, df):
    """cancellation noise + the oracle's phase rounding, 4 eps 2 pi f / df (t_c <= T = 1/df)"""
    return cancel_floor(det, f) + 4.0 * EPS * 2.0 * np.pi * f / df


def check_response_per_bin(got, want, f, dets, what="", df=W.MONTH_DF):
    worst = 0.0
    for b in range(want.shape[0]):
        for d, det in enumerate(dets):
            s = np.abs(want[b, d]).max(axis=0)                     # [N]: largest channel of the bin
            assert np.all(s > 0.0)
            floor = bin_floor(det, f, df) * s
            for c in range(3):
                err = np.abs(got[b, d, c] - want[b, d, c])
                tol = TOL_RESP * np.abs(want[b, d, c]) + floor
                bad = np.nonzero(err > tol)[0]
                assert bad.size == 0, (what, b, d, c, f[bad[:5]], (err[bad[:5]] / s[bad[:5]]))
                worst = max(worst, float((err / tol).max()))
    return worst


# ---------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("gen", [20, 15])
@pytest.mark.parametrize("mask", [W.MODES_22_ONLY, W.MODES_HM])
def test_response_full_band_per_bin(P, gen, mask):
    """configs 2-4: the full 262144-bin grid sampled every 257th bin + the neighbourhood of every in-band null, all
    three detectors, per-bin tolerance.  The injection, jittered samples and one random-sky spinning sample."""
    grid = W.config(2).grid
    dets = (W.lisa_like(gen), W.taiji_like(gen), W.tianqin_like(gen))
    model = W.Model(mask, dets)
    idx, n_null = band_indices(grid, dets)
    assert n_null >= (7 if gen == 20 else 3)          # LISA-like 30/60/90 mHz, Taiji-like 25/50/75/100 mHz (2.0)
    f = grid.freqs()[idx]
    th = W.config(4, B=6).params
    th[0] = W.config(4).theta_inj
    rng = np.random.default_rng(31)
    th[5] = W.draw_prior(1, 1.0 / grid.df, rng)[0]
    th[5, 0] = 3.1e6; th[5, 2] = 0.6; th[5, 3] = -0.4
    assert (np.pi * th[0, 0] * 4.925490947641267e-6 * f[-1]) ** (1.0 / 3.0) > 1.4       # v > 1 bins are in the sample
    got = P.response(dev(th), dev(f), model).cpu().numpy()
    want = oracle.response(th, f, model)
    worst = check_response_per_bin(got, want, f, dets, f"gen {gen} mask {mask}")
    print(f"full band, gen {gen}, mask {mask}: {f.size} bins, {n_null} nulls, worst per-bin error / tolerance {worst:.3f}")


def test_response_near_nulls_dense(P):
    """every bin of a 129-bin window centred on each LISA-like / Taiji-like null (generation 2.0), five modes"""
    grid = W.config(2).grid
    fgrid = grid.freqs()
    for det in (W.lisa_like(), W.taiji_like()):
        model = W.Model(W.MODES_HM, (det,))
        th = W.config(3, B=3).params
        for fn in null_frequencies(det, fgrid[0], fgrid[-1]):
            k0 = int(round((fn - grid.f0) / grid.df))
            f = fgrid[max(0, k0 - 64):min(grid.N, k0 + 65)]
            got = P.response(dev(th), dev(f), model).cpu().numpy()
            want = oracle.response(th, f, model)
            check_response_per_bin(got, want, f, (det,), f"{det.name} null {fn:.6f}")
            # the response really dips there: |g| at the centre is tiny against the window edge
            assert np.abs(want[0, 0, 0]).min() < 0.05 * np.abs(want[0, 0, 0]).max()


@pytest.mark.parametrize("gen", [20, 15])
def test_response_tab_full_band_per_bin(P, gen):
    """pespace_response_tab (tabulated mode waveforms, reading T1) over the full band, same sample of bins and the same
    per-bin tolerance: tables of the oracle's analytic modes on 2000 log-spaced nodes, five modes, three detectors"""
    grid = W.config(2).grid
    dets = (W.lisa_like(gen), W.taiji_like(gen), W.tianqin_like(gen))
    model = W.Model(W.MODES_HM, dets)
    idx, _ = band_indices(grid, dets)
    fgrid = grid.freqs()
    f = fgrid[idx]
    th = W.config(4, B=4).params
    table = W.table_from_waveform_fn(th, model.mode_mask, W.log_nodes(fgrid[0], fgrid[-1], 2000), oracle.waveform)
    got = P.response_tab(dev(th), P.WaveTable(*(dev(x) for x in table)), dev(f), model).cpu().numpy()
    want = oracle.response_tab(th, table, f, model)
    check_response_per_bin(got, want, f, dets, f"tab gen {gen}")


def test_response_orb_full_band_per_bin(P):
    """pespace_response_orb (tabulated orbits, reading T2) over the full band with the same per-bin tolerance: seeded
    toy ephemeris with breathing arms, five modes, three detectors, the nulls of the NOMINAL arm lengths included"""
    grid = W.config(2).grid
    dets = (W.lisa_like(), W.taiji_like(), W.tianqin_like())
    model = W.Model(W.MODES_HM, dets)
    idx, _ = band_indices(grid, dets)
    f = grid.freqs()[idx]
    th = W.config(4, B=4).params
    T = 1.0 / grid.df
    tab = W.synthetic_orbit_table(dets, -16.0 * T, 1800.0, int(18.5 * T / 1800.0) + 2, seed=21)
    got = P.response_orb(dev(th), P.OrbitTable(tab[0], tab[1], dev(tab[2]), dev(tab[3])), dev(f), model).cpu().numpy()
    want = oracle.response_orb(th, tab, f, model)
    assert np.all(np.abs(want[:, :, 0]).max(axis=-1) > 0)
    worst = check_response_per_bin(got, want, f, dets, "orb")
    print(f"tabulated orbits, full band: {f.size} bins, worst per-bin error / tolerance {worst:.3f}")


def _window_workload(det_list, k0, n, B, mask, seed):
    """an n-bin stretch of the config-2 lattice starting at bin k0: same df, f0 moved"""
    base = W.config(2).grid
    f0 = base.freqs()[k0]
    wl = W.config(4, B=B, N=n)
    grid = W.Grid(float(f0), base.df, n)
    return W.Workload("window", grid, W.Model(mask, tuple(det_list)), wl.params, wl.theta_inj, seed)


@pytest.mark.parametrize("gen", [20, 15])
def test_loglike_noisy_window_straddling_a_null(P, gen):
    """lnL on short grids with NOISY data centred on in-band nulls: prep_bins_kernel divides the data by g(z) where
    |g|^2 is many orders below its median; the weighted residual must stay regular (G9)."""
    base = W.config(2).grid
    for det in (W.lisa_like(gen), W.taiji_like(gen)):
        for fn in null_frequencies(det, base.f0, base.freqs()[-1])[:3]:
            k0 = int(round((fn - base.f0) / base.df)) - 200
            wl = _window_workload([det], k0, 401, 9, W.MODES_HM, 7)
            data, psd = wl.data(oracle_response_fn), wl.psd()
            assert psd[0, 0].min() < 1e-3 * np.median(psd[0, 0])
            got = P.loglike(dev(wl.params), dev(data), dev(psd), wl.grid, wl.model).cpu().numpy()
            want = oracle.loglike(wl.params, data, psd, wl.grid, wl.model)
            hh = -2.0 * oracle.loglike(wl.params, np.zeros_like(data), psd, wl.grid, wl.model)
            rel = np.abs(got - want) / np.maximum(np.abs(want), 0.5 * hh)
            assert rel.max() <= TOL_LNL, (det.name, fn, rel.max())


def test_loglike_high_band_windows_three_detectors(P):
    """lnL and <h|h> restricted to windows high in the band (where the full-size sums carry no weight)"""
    for k0 in (60000, 130000, 200000, 261000):
        wl = _window_workload([W.lisa_like(), W.taiji_like(), W.tianqin_like()], k0, 1000, 11, W.MODES_HM, 9)
        data, psd = wl.data(oracle_response_fn), wl.psd()
        for dat in (data, np.zeros_like(data)):
            got = P.loglike(dev(wl.params), dev(dat), dev(psd), wl.grid, wl.model).cpu().numpy()
            want = oracle.loglike(wl.params, dat, psd, wl.grid, wl.model)
            hh = -2.0 * oracle.loglike(wl.params, np.zeros_like(data), psd, wl.grid, wl.model)
            rel = np.abs(got - want) / np.maximum(np.abs(want), 0.5 * hh)
            assert rel.max() <= TOL_LNL, (k0, rel.max())


# --------------------------------------------------------------------------------------------------------------- S10
def phase_floor(f, df):
    """the double oracle's phase rounding, 4 eps 2 pi f / df (module docstring; pin P14 over the band)"""
    return 4.0 * EPS * 2.0 * np.pi * f / df


def test_fisher_single_bin_grids_over_the_band(P):
    """per-bin derivative parity: pespace_fisher on ONE-bin grids placed over the band (incl. +-2 bins of the nulls and
    v > 1): every F_ij of the bin against the oracle's 11-tangent dual number on the Cauchy-Schwarz scale, and the
    gradient with noisy data.  Tolerance of a single bin: 1e-9 + 8 x the double oracle's phase rounding (the modes
    carry independent roundings of phases up to 1.6e6 rad, which moves their interference terms; measured against
    binary128 finite differences in the next test: oracle 2.2e-9 at 63 mHz, CUDA path 4e-11)."""
    base = W.config(2).grid
    fgrid = base.freqs()
    dets = (W.lisa_like(), W.taiji_like(), W.tianqin_like())
    ks = set(range(0, base.N, 262144 // 24)) | {base.N - 1}
    for det in dets[:2]:
        for fn in null_frequencies(det, fgrid[0], fgrid[-1]):
            k0 = int(round((fn - base.f0) / base.df))
            ks |= {k0 - 2, k0 + 1}
    th = W.config(5, B=3).params
    th[1, 2] = 0.5; th[1, 3] = -0.3
    worstF = worstg = 0.0
    for k in sorted(ks):
        wl = _window_workload(dets, k, 1, 3, W.MODES_HM, 13)
        wl.params = th
        data, psd = wl.data(oracle_response_fn), wl.psd()
        F, g = P.fisher(dev(th), dev(data), dev(psd), wl.grid, wl.model)
        Fo, go = oracle.fisher(th, data, psd, wl.grid, wl.model)
        d = np.sqrt(np.einsum("bii->bi", Fo))
        assert np.all(d > 0)
        eF = (np.abs(F.cpu().numpy() - Fo) / (d[:, :, None] * d[:, None, :])).max()
        rr = -2.0 * oracle.loglike(th, data, psd, wl.grid, wl.model)
        eg = (np.abs(g.cpu().numpy() - go) / (d * np.sqrt(rr)[:, None])).max()
        tol_F = TOL_F + 8.0 * phase_floor(fgrid[k], base.df)
        # gradient of ONE bin: the rounding noise of d_i h_c (cancel_floor, relative to the largest channel) enters
        # <d - h | d_i h> through every channel with weight sqrt(w_c); on the scale sqrt(F_ii <r|r>) >= sqrt(w_A) ...
        # that is cancel_floor x sqrt(S_max / S_min) -- at low f the T channel of a short-arm detector is pure
        # rounding noise (pin P8) whitened by a PSD (x^2/3) S_A.  (F itself is insensitive: the noise is multiplied by
        # the small d_j h_T.)  In sums over many bins the term averages out; here it is the whole result.
        tol_g = tol_F + max(cancel_floor(det, fgrid[k]) * np.sqrt(psd[i].max() / psd[i].min()) for i, det in enumerate(dets))
        assert eF <= tol_F and eg <= tol_g, (k, fgrid[k], eF, eg, tol_F, tol_g)
        # the reverse-mode gradient (pespace_loglike_grad) of the same single bin, same tolerance; lnL at 1e-9
        la, ga = P.loglike_grad(dev(th), dev(data), dev(psd), wl.grid, wl.model)
        ea = (np.abs(ga.cpu().numpy() - go) / (d * np.sqrt(rr)[:, None])).max()
        assert ea <= tol_g, (k, fgrid[k], ea, tol_g)
        assert (np.abs(la.cpu().numpy() + 0.5 * rr) / (0.5 * rr)).max() <= TOL_LNL
        worstF, worstg = max(worstF, eF / tol_F), max(worstg, eg / tol_g, ea / tol_g)
    print(f"single-bin Fisher over the band: {len(ks)} bins, worst F / tolerance {worstF:.2f}, worst grad / tolerance {worstg:.2f}")


def test_fisher_single_bins_against_binary128_finite_differences(P):
    """the extrinsic 6 x 6 block (D_L, iota, phi_c, lambda, beta, psi) of single-bin Fisher matrices against
    Richardson-extrapolated central differences of the oracle's response evaluated in IEEE BINARY128 (steps chosen so
    that the phase moves by 2e-3 and 1e-3 rad: truncation 1e-12, resolution of the double output 1e-13): the exact
    definition to 1e-11, at 1e-9.  (The mass and spin columns would need steps too small for the double output.)"""
    base = W.config(2).grid
    fgrid = base.freqs()
    dets = (W.lisa_like(), W.taiji_like(), W.tianqin_like())
    th = W.config(5, B=2).params
    th[1, 2] = 0.5; th[1, 3] = -0.3
    sub = [4, 5, 6, 7, 8, 9]
    for k in (20000, 77448, 130000, 163830, 233200, 261000):        # 7.8 ... 100.8 mHz; 77448: LISA-like 30 mHz null + 1
        wl = _window_workload(dets, k, 1, 2, W.MODES_HM, 13)
        wl.params = th
        psd = wl.psd()
        F, _ = P.fisher(dev(th), None, dev(psd), wl.grid, wl.model)
        f = wl.grid.freqs()
        dopp = 2.0 * np.pi * f[0] * 499.005 + 2.0                     # rad of phase per rad of sky angle (AU/c) + pattern
        sens = {4: 1.0, 5: 1.0, 6: 4.0, 7: dopp, 8: dopp, 9: 4.0}
        J = np.zeros((2, 11, 3, 3), dtype=complex)
        for i in sub:
            for b in range(2):
                est = []
                for hs in (2e-3, 1e-3):
                    h = hs / sens[i] * (abs(th[b, i]) if i == 4 else 1.0)
                    tp, tm = th[b:b + 1].copy(), th[b:b + 1].copy()
                    tp[0, i] += h; tm[0, i] -= h
                    rp = oracle.response(tp, f, wl.model, quad=True)[0, :, :, 0]
                    rm = oracle.response(tm, f, wl.model, quad=True)[0, :, :, 0]
                    est.append((rp - rm) / (tp[0, i] - tm[0, i]))
                J[b, i] = (4.0 * est[1] - est[0]) / 3.0
        w = 4.0 * wl.grid.df / psd[:, :, 0]
        Fq = np.einsum("bidc,bjdc,dc->bij", np.conj(J), J, w).real
        ix = np.ix_(range(2), sub, sub)
        d = np.sqrt(np.einsum("bii->bi", Fq[ix]))
        err = (np.abs(F.cpu().numpy()[ix] - Fq[ix]) / (d[:, :, None] * d[:, None, :])).max()
        assert err <= TOL_F, (k, fgrid[k], err)


def test_fisher_windows_at_the_nulls(P):
    """Fisher matrix and gradient on 300-bin windows straddling 30, 60, 90 mHz (LISA-like) and 25 ... 100 mHz
    (Taiji-like), five modes, noisy data"""
    base = W.config(2).grid
    for det in (W.lisa_like(), W.taiji_like()):
        for fn in null_frequencies(det, base.f0, base.freqs()[-1]):
            k0 = int(round((fn - base.f0) / base.df)) - 150
            wl = _window_workload([det], min(k0, base.N - 300), 300, 4, W.MODES_HM, 17)
            data, psd = wl.data(oracle_response_fn), wl.psd()
            F, g = P.fisher(dev(wl.params), dev(data), dev(psd), wl.grid, wl.model)
            Fo, go = oracle.fisher(wl.params, data, psd, wl.grid, wl.model)
            d = np.sqrt(np.einsum("bii->bi", Fo))
            eF = (np.abs(F.cpu().numpy() - Fo) / (d[:, :, None] * d[:, None, :])).max()
            rr = -2.0 * oracle.loglike(wl.params, data, psd, wl.grid, wl.model)
            eg = (np.abs(g.cpu().numpy() - go) / (d * np.sqrt(rr)[:, None])).max()
            assert eF <= TOL_F and eg <= TOL_F, (det.name, fn, eF, eg)


# --------------------------------------------------------------------------------------------------------------- masks
def test_masked_bins_ignore_the_data_and_exact_nulls_keep_their_weight(P):
    """Reading G9, one rule on both sides: a bin's weight depends on the PSD alone.
    (1) bins whose PSD is 0 / negative / non-finite are skipped WITHOUT reading the data: NaN / Inf data there must
        not reach lnL, the gradient or F;
    (2) a bin where g(z) is exactly 0 (2 f L / c an exact integer) but the caller's PSD is positive keeps its
        theta-independent term |d|^2 4 df / S, as the definition (Eq. 10) has it."""
    det = dataclasses.replace(W.lisa_like(), L_m=8.0 * C_SI)          # L / c = 8 s exactly
    grid = W.Grid(0.0625 - 64 * 2.0 ** -20, 2.0 ** -20, 200)          # bin 64 = 0.0625 Hz exactly: 2 f L / c = 1
    f = grid.freqs()
    assert f[64] == 0.0625 and 2.0 * f[64] * (det.L_m / C_SI) == 1.0
    model = W.Model(W.MODES_HM, (det,))
    th = W.config(3, B=5).params
    rng = np.random.default_rng(3)
    psd = np.full((1, 3, grid.N), 1e-40) * rng.uniform(0.5, 2.0, (1, 3, grid.N))
    data = W.coloured_noise(psd, grid.df, rng) + oracle.response(th[:1], f, model)[0]
    r = P.response(dev(th), dev(f), model).cpu().numpy()
    assert np.all(r[:, :, :, 64] == 0)                                # the template is identically zero there
    ro = oracle.response(th, f, model)
    assert np.abs(ro[:, :, :, 64]).max() < 1e-12 * np.abs(ro).max()   # (the oracle's sin(pi) is 1.2e-16, not 0)
    want = oracle.loglike(th, data, psd, grid, model)
    got = P.loglike(dev(th), dev(data), dev(psd), grid, model).cpu().numpy()
    assert np.abs(got - want).max() <= TOL_LNL * np.abs(want).min()
    # the null bin's own term is visible at this tolerance
    term = 0.5 * 4.0 * grid.df * (np.abs(data[0, :, 64]) ** 2 / psd[0, :, 64]).sum()
    assert term > 100 * TOL_LNL * np.abs(want).max()
    # (1) masked bins with poisoned data
    psd2, data2 = psd.copy(), data.copy()
    for c, k, s, dval in [(0, 3, 0.0, np.nan), (1, 100, np.inf, np.inf), (2, 199, np.nan, np.nan + 1j * np.inf),
                          (0, 17, -1.0, -np.inf), (1, 64, 0.0, np.nan)]:
        psd2[0, c, k] = s
        data2[0, c, k] = dval
    want2 = oracle.loglike(th, data2, psd2, grid, model)
    assert np.all(np.isfinite(want2))
    got2 = P.loglike(dev(th), dev(data2), dev(psd2), grid, model).cpu().numpy()
    assert np.abs(got2 - want2).max() <= TOL_LNL * np.abs(want2).min()
    F, g = P.fisher(dev(th), dev(data2), dev(psd2), grid, model)
    Fo, go = oracle.fisher(th, data2, psd2, grid, model)
    d = np.sqrt(np.einsum("bii->bi", Fo))
    assert (np.abs(F.cpu().numpy() - Fo) / (d[:, :, None] * d[:, None, :])).max() <= TOL_F
    rr = -2.0 * want2
    assert (np.abs(g.cpu().numpy() - go) / (d * np.sqrt(rr)[:, None])).max() <= TOL_F
    lm = P.Likelihood(dev(data2), dev(psd2), grid, model, th.shape[0])(dev(th), mixed=True).cpu().numpy()
    assert np.abs(lm - want2).max() <= 5e-6 * np.abs(want2).min()


# --------------------------------------------------------------------------------------------------------------- sizes
def test_full_size_network_every_32nd_sample(P):
    """config 4 at full size (B = 8192, three detectors, five modes): SURVEY 8(d)'s subset, every ceil(B/32)-th
    sample plus sample 0 and the last one"""
    wl = W.config(4)
    data, psd = wl.data(oracle_response_fn), wl.psd()
    subset = np.array(sorted(set(range(0, wl.B, wl.B // 32)) | {wl.B - 1}))
    assert subset.size >= 33
    got = P.Likelihood(dev(data), dev(psd), wl.grid, wl.model, wl.B)(dev(wl.params)).cpu().numpy()
    want = oracle.loglike(wl.params[subset], data, psd, wl.grid, wl.model)
    assert (np.abs(got[subset] - want) / np.abs(want)).max() <= TOL_LNL


def test_full_size_fisher_eight_samples(P):
    """config 5 at full size: 8 of the 256 samples against the oracle"""
    wl = W.config(5)
    data, psd = wl.data(oracle_response_fn), wl.psd()
    subset = np.array([0, 37, 73, 110, 146, 183, 219, 255])
    F, g = P.fisher(dev(wl.params), dev(data), dev(psd), wl.grid, wl.model)
    Fo, go = oracle.fisher(wl.params[subset], data, psd, wl.grid, wl.model)
    d = np.sqrt(np.einsum("bii->bi", Fo))
    assert (np.abs(F.cpu().numpy()[subset] - Fo) / (d[:, :, None] * d[:, None, :])).max() <= TOL_F
    rr = -2.0 * oracle.loglike(wl.params[subset], data, psd, wl.grid, wl.model)
    assert (np.abs(g.cpu().numpy()[subset] - go) / (d * np.sqrt(rr)[:, None])).max() <= TOL_F
