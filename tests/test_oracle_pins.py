"""Pins P1-P16: the oracle checked against what the paper and the
mathematics fix, NOT against itself.  Every check here uses a different formula, a closed
form, an invariant, a limit or brute force from the one the oracle evaluates.

Runs without a GPU (`-m "not gpu"`).
"""
import math
import os

import numpy as np
import pytest

import oracle
from paper_2602_12011_b200 import workloads as W

C_SI = 299792458.0
AU = 149597870700.0
YR = 31558149.763545603
TSUN = 1.3271244e20 / C_SI ** 3
GPC_S = 3.0856775814913673e25 / C_SI
EULER = 0.5772156649015329

THETA = np.array([2e6, 3.0, 0.0, 0.0, 10.0, 0.4, 1.3, 1.375, -1.2108, 2.659, 2073600.0])
LISA = W.lisa_like()
LISA15 = W.lisa_like(15)
TAIJI = W.taiji_like()
TQ = W.tianqin_like()
MODES = {(2, 2): 1, (2, 1): 2, (3, 3): 4, (3, 2): 8, (4, 4): 16}


# ------------------------------------------------------------------ test-side geometry (restated, O7)
def frame(lam, bet):
    k = -np.array([math.cos(bet) * math.cos(lam), math.cos(bet) * math.sin(lam), math.sin(bet)])
    u = np.array([math.sin(lam), -math.cos(lam), 0.0])
    v = np.array([-math.sin(bet) * math.cos(lam), -math.sin(bet) * math.sin(lam), math.cos(bet)])
    return k, u, v


def mode_tensor(l, m, iota, lam, bet, psi):
    """P^{lm} = K+ P+ + Kx Px as a complex 3x3 matrix, with the harmonics from CLOSED FORMS."""
    k, u, v = frame(lam, bet)
    ep = np.outer(u, u) - np.outer(v, v)
    ec = np.outer(u, v) + np.outer(v, u)
    Pp = math.cos(2 * psi) * ep + math.sin(2 * psi) * ec
    Pc = -math.sin(2 * psi) * ep + math.cos(2 * psi) * ec
    Yp, Ym = closed_form_swsh(l, m, iota), closed_form_swsh(l, -m, iota)
    Kp = 0.5 * (Yp + (-1) ** l * Ym)
    Kc = -0.5j * (Yp - (-1) ** l * Ym)
    return Kp * Pp + Kc * Pc


def closed_form_swsh(l, m, iota):
    c, s = math.cos(iota), math.sin(iota)
    Ch, Sh = math.cos(iota / 2), math.sin(iota / 2)
    pi = math.pi
    table = {
        (2, 2): math.sqrt(5 / (64 * pi)) * (1 + c) ** 2, (2, -2): math.sqrt(5 / (64 * pi)) * (1 - c) ** 2,
        (2, 1): math.sqrt(5 / (16 * pi)) * s * (1 + c), (2, -1): math.sqrt(5 / (16 * pi)) * s * (1 - c),
        (3, 3): -math.sqrt(21 / (2 * pi)) * Ch ** 5 * Sh, (3, -3): math.sqrt(21 / (2 * pi)) * Ch * Sh ** 5,
        (3, 2): math.sqrt(7 / pi) * Ch ** 4 * (3 * c - 2) / 2, (3, -2): math.sqrt(7 / pi) * Sh ** 4 * (3 * c + 2) / 2,
        (4, 4): 3 * math.sqrt(7 / pi) * Ch ** 6 * Sh ** 2, (4, -4): 3 * math.sqrt(7 / pi) * Ch ** 2 * Sh ** 6,
    }
    return table[(l, m)]


def inner(a, b, psd, df):
    """<a|b> of Eq. 14 with T = 1/df, summed over every leading axis."""
    return 4.0 * df * np.real(np.sum(np.conj(a) * b / psd))


# ------------------------------------------------------------------ golden: SURVEY worked example
def _golden():
    path = os.path.join(os.path.dirname(__file__), "golden", "survey_worked_example.txt")
    rows = {}
    for line in open(path):
        if line.startswith("#") or not line.strip():
            continue
        key, *vals = line.split()
        rows.setdefault(key, []).append([float(x) for x in vals])
    return rows


def test_golden_worked_example():
    g = _golden()
    th = np.array(g["theta"][0])
    for f, psi, dt, amp in g["wave"]:
        a, p, t = oracle.waveform(th, 2, 2, np.array([f]))
        assert p[0] == pytest.approx(psi, rel=1e-12)
        assert t[0] - th[10] == pytest.approx(dt, rel=1e-9)
        assert a[0] == pytest.approx(amp, rel=1e-12)
    for gen, mask, f, *vals in g["resp"]:
        r = oracle.response(th, np.array([f]), W.Model(int(mask), (W.lisa_like(int(gen)),)))[0, 0, :, 0]
        got = np.array([r[0].real, r[0].imag, r[1].real, r[1].imag, r[2].real, r[2].imag])
        want = np.array(vals)
        ok = np.isfinite(want)
        scale = np.abs(r[0])
        # T is a difference of nearly equal terms at low f; compare it on the scale of T itself
        tol = np.where(np.arange(6) < 4, 2e-9 * scale, 2e-6 * np.abs(r[2]))
        assert np.all(np.abs(got - want)[ok] <= tol[ok]), (gen, mask, f, got, want)
    for f, sa, st in g["psd"]:
        S = W.psd_aet(LISA, np.array([f]))[:, 0]
        assert S[0] == pytest.approx(sa, rel=1e-9) and S[1] == S[0] and S[2] == pytest.approx(st, rel=1e-9)
    assert np.allclose(oracle.orbit(LISA, 0.0)[0], g["sc1"][0], rtol=0, atol=2e-3)


# ------------------------------------------------------------------ P1, P2: PN phase and t_f
def taylor_t2_time(f, M, q, tc):
    """Independently stated 3.5PN TaylorT2 series t(v)."""
    Ms, eta, pi = M * TSUN, q / (1 + q) ** 2, math.pi
    v = (pi * Ms * f) ** (1.0 / 3.0)
    tau = [1.0, 0.0,
           743 / 252 + 11 * eta / 3,
           -32 * pi / 5,
           3058673 / 508032 + 5429 * eta / 504 + 617 * eta ** 2 / 72,
           -(7729 / 252 - 13 * eta / 3) * pi,
           -10052469856691 / 23471078400 + 128 * pi ** 2 / 3 + 6848 * EULER / 105
           + (3147553127 / 3048192 - 451 * pi ** 2 / 12) * eta - 15211 * eta ** 2 / 1728
           + 25565 * eta ** 3 / 1296 + 6848 / 105 * math.log(4 * v),
           (-15419335 / 127008 - 75703 * eta / 756 + 14809 * eta ** 2 / 378) * pi]
    return tc - 5 * Ms / (256 * eta * v ** 8) * sum(tau[k] * v ** k for k in range(8))


@pytest.mark.parametrize("M,q", [(2e6, 3.0), (1e5, 1.0), (1e7, 8.0), (6e5, 1.7)])
def test_P1_spa_duality_with_taylor_t2(M, q):
    th = THETA.copy(); th[0], th[1] = M, q
    f = np.array([1e-4, 3e-4, 1e-3, 5e-3, 2e-2])
    _, _, t = oracle.waveform(th, 2, 2, f)
    want = np.array([taylor_t2_time(x, M, q, th[10]) for x in f])
    assert np.allclose(t - th[10], want - th[10], rtol=1e-11, atol=1e-9)


def test_P2_tf_is_phase_derivative_and_newtonian_limit():
    th = THETA.copy()
    for f0, chi1, chi2 in ((1.3e-4, 0.0, 0.0), (1e-3, 0.0, 0.0), (7e-3, 0.0, 0.0), (2e-3, 0.6, -0.3)):
        th[2], th[3] = chi1, chi2
        est = []
        for h in (2e-3 * f0, 1e-3 * f0):
            _, p, _ = oracle.waveform(th, 2, 2, np.array([f0 - h, f0 + h]))
            est.append((p[1] - p[0]) / (2 * h) / (2 * math.pi))
        richardson = (4 * est[1] - est[0]) / 3          # Eq. 4 with Phi = -Psi
        _, _, t = oracle.waveform(th, 2, 2, np.array([f0]))
        assert t[0] - th[10] == pytest.approx(richardson - th[10], rel=2e-7)
    th[2] = th[3] = 0.0
    # low-frequency limit: t_c - (5/256) Mc^{-5/3} (pi f)^{-8/3}, deviation O(v^2)
    Ms, eta = th[0] * TSUN, th[1] / (1 + th[1]) ** 2
    Mc = eta ** 0.6 * Ms
    dev = []
    for f0 in (1e-8, 1e-7):
        _, _, t = oracle.waveform(th, 2, 2, np.array([f0]))
        newt = -(5.0 / 256.0) * Mc ** (-5.0 / 3.0) * (math.pi * f0) ** (-8.0 / 3.0)
        dev.append(abs((t[0] - th[10]) / newt - 1.0))
    assert dev[0] < 3e-4 and dev[1] < 1.5e-3 and dev[0] < dev[1]
    _, _, t = oracle.waveform(th, 2, 2, np.array([1e-4]))
    assert (t[0] - th[10]) / 86400.0 == pytest.approx(-59.16, abs=0.01)      # SURVEY P2 probe value


def test_higher_mode_maps_follow_the_22_mode():
    """O5 / G5: Psi_lm(f) = (m/2) Psi_22(2f/m), t_lm(f) = t_22(2f/m), A_lm from the listed ratios."""
    th = THETA.copy()
    f = np.array([2e-4, 1e-3, 6e-3])
    eta, delta = th[1] / (1 + th[1]) ** 2, (th[1] - 1) / (th[1] + 1)
    ratios = {(2, 1): (delta / 3, 1), (3, 3): (0.75 * math.sqrt(15 / 14) * delta, 1),
              (3, 2): (math.sqrt(5 / 7) / 3 * (1 - 3 * eta), 2), (4, 4): (8 / 9 * math.sqrt(5 / 7) * (1 - 3 * eta), 2)}
    for (l, m), (c, p) in ratios.items():
        a, ps, t = oracle.waveform(th, l, m, f)
        a2, ps2, t2 = oracle.waveform(th, 2, 2, 2 * f / m)
        vm = (math.pi * th[0] * TSUN * 2 * f / m) ** (1 / 3)
        assert np.allclose(ps, m / 2 * ps2, rtol=1e-15, atol=0)
        assert np.allclose(t, t2, rtol=0, atol=0)
        assert np.allclose(a, math.sqrt(2 / m) * c * vm ** p * a2, rtol=1e-13, atol=0)


def test_spin_terms_against_the_poisson_will_forms():
    """G3 / O2: the 1.5PN spin-orbit and 2PN spin-spin terms, pinned against the forms printed by Poisson & Will,
    Phys. Rev. D 52, 848 (1995), Eqs. (1.3)-(1.5) [also Cutler & Flanagan 1994 for beta; Kidder 1995 for sigma],
    restated here from the individual masses and NOT taken from the oracle:
        beta  = (1/12) sum_i [113 (m_i/M)^2 + 75 eta] (L.chi_i),
        sigma = (eta/48) [-247 chi_1.chi_2 + 721 (L.chi_1)(L.chi_2)]      (aligned spins: both products chi_1 chi_2),
        Psi(f) = 2 pi f t_c - phi_c - pi/4 + (3/128)(pi Mc f)^{-5/3} [1 + ... - 4 (4 pi - beta) x^{3/2}
                                                                          + 10 (3058673/1016064 + ... - sigma) x^2],
        t(f)   = t_c - (5/256) Mc (pi Mc f)^{-8/3} [1 + ... - (8/5)(4 pi - beta) x^{3/2} + 2 (... - sigma) x^2],
    with x = (pi M f)^{2/3}.  Only the spin-dependent differences are compared, so the non-spinning part (pins P1, P2)
    drops out: the phase AND the time-frequency map, each against its own printed series."""
    for M, q, chi1, chi2 in ((2e6, 3.0, 0.6, -0.3), (4e5, 1.0, -0.9, 0.7), (7e6, 7.5, 0.25, 0.8), (1e6, 2.0, 0.5, 0.0)):
        th = THETA.copy(); th[0], th[1] = M, q
        m1, m2 = q / (1 + q), 1 / (1 + q)                      # m_i / M
        eta = m1 * m2
        beta = ((113 * m1 ** 2 + 75 * eta) * chi1 + (113 * m2 ** 2 + 75 * eta) * chi2) / 12
        sigma = eta / 48 * (-247 + 721) * chi1 * chi2
        Ms = M * TSUN
        Mc = eta ** 0.6 * Ms
        f = np.array([1.3e-4, 7e-4, 3e-3, 1.1e-2])
        x = (math.pi * Ms * f) ** (2.0 / 3.0)
        th0, ths = th.copy(), th.copy()
        ths[2], ths[3] = chi1, chi2
        _, p0, t0 = oracle.waveform(th0, 2, 2, f)
        _, ps, ts = oracle.waveform(ths, 2, 2, f)
        dpsi = 3 / 128 * (math.pi * Mc * f) ** (-5.0 / 3.0) * (4 * beta * x ** 1.5 - 10 * sigma * x ** 2)
        dt = -5 / 256 * Mc * (math.pi * Mc * f) ** (-8.0 / 3.0) * (8 / 5 * beta * x ** 1.5 - 2 * sigma * x ** 2)
        assert np.allclose(ps - p0, dpsi, rtol=1e-9, atol=1e-9 * np.abs(p0).max() * 1e-3)
        assert np.allclose(ts - t0, dt, rtol=1e-9, atol=1e-12 * np.abs(t0 - th[10]).max())
        assert np.abs(dpsi).min() > 1e-2                       # the spin terms are not negligible in the comparison
    # each spin separately, equal spins, and the antisymmetric combination at q = 1 (beta keeps only 75 eta terms)
    th = THETA.copy(); th[1] = 1.0; th[2], th[3] = 0.4, -0.4
    _, ps, _ = oracle.waveform(th, 2, 2, np.array([1e-3]))
    th[2] = th[3] = 0.0
    _, p0, _ = oracle.waveform(th, 2, 2, np.array([1e-3]))
    x = (math.pi * th[0] * TSUN * 1e-3) ** (2.0 / 3.0)
    want = 3 / 128 * 4 * (math.pi * th[0] * TSUN * 1e-3) ** (-5.0 / 3.0) * (-10 * (0.25 / 48 * 474 * -0.16) * x ** 2)
    assert ps[0] - p0[0] == pytest.approx(want, rel=1e-8)     # beta = 0 by symmetry, sigma < 0


def _point_mass_moment(q, l, current):
    """Newtonian radiative multipole of two point masses on a circular orbit, mass-ratio dependence only: the mass
    moment of order l is sum_A m_A r_A^l e^{-i m phi_A}, the current moment carries one more power of r_A (r x v);
    body 2 sits opposite body 1 (phi_2 = phi_1 + pi), r_1 = (m_2/M) r, r_2 = (m_1/M) r.  Returned in units of
    mu r^l (mu r^{l+1} Omega), with the sign (-1)^power for body 2."""
    m1, m2 = q / (1 + q), 1 / (1 + q)
    p = l + 1 if current else l
    return (m1 * m2 ** p + m2 * (-m1) ** p) / (m1 * m2)


def test_mode_amplitude_ratios_against_multipole_moments_and_test_mass_fluxes():
    """O5: the c_lm v^{p_lm} table, pinned WITHOUT restating it.
    (a) Mass-ratio dependence: a mode with l + m even is a mass multipole of order l, with l + m odd a current
        multipole of order l; for two point masses these are sum_A m_A (+-r_A)^l and sum_A m_A (+-r_A)^{l+1}
        (`_point_mass_moment`), so A_lm(q) / A_lm(q_ref) at equal M, f must follow them (this is where delta and
        1 - 3 eta come from; equal masses kill the odd-m modes).
    (b) Numbers and powers of v: in the test-mass limit the energy flux carried by mode (l,m) relative to (2,2)
        at the same ORBITAL frequency is, at leading order, the black-hole-perturbation result of Poisson,
        Phys. Rev. D 47, 1497 (1993), Eq. (5.12)-(5.13) [eta_21 = v^2/36, eta_33 = (1215/896) v^2, eta_32 = (5/63) v^4,
        eta_44 = (1280/567) v^4, v = (M Omega)^{1/3}].  Flux ~ (m Omega)^2 |h_lm(t)|^2 and the stationary-phase
        transform gives |h~_lm(f = m F)|^2 = |h_lm|^2 pi / (m dOmega/dt), hence
        flux_lm / flux_22 = (m^2/4) (m/2) |h~_lm(m F)|^2 / |h~_22(2 F)|^2."""
    th = THETA.copy()
    F = np.array([2e-5, 1e-4, 7e-4])                        # orbital frequencies
    # (b) test-mass limit
    th[1] = 1e7
    poisson = {(2, 1): (1 / 36, 2), (3, 3): (1215 / 896, 2), (3, 2): (5 / 63, 4), (4, 4): (1280 / 567, 4)}
    a22, _, _ = oracle.waveform(th, 2, 2, 2 * F)
    v = (2 * math.pi * th[0] * TSUN * F) ** (1.0 / 3.0)     # (M Omega)^{1/3}
    for (l, m), (coef, power) in poisson.items():
        alm, _, _ = oracle.waveform(th, l, m, m * F)
        flux_ratio = (m * m / 4) * (m / 2) * (alm / a22) ** 2
        assert np.allclose(flux_ratio, coef * v ** power, rtol=3e-6, atol=0), (l, m)   # q = 1e7: delta, 1 - 3 eta to 1e-6
    # (a) mass-ratio dependence against the point-mass moments, normalised to the (2,2) mode (mu r^2: moment 1)
    qref = 5.0
    for q in (1.0, 1.3, 3.0, 8.0):
        for (l, m) in ((2, 1), (3, 3), (3, 2), (4, 4)):
            ratio = []
            for qq in (q, qref):
                th[1] = qq
                alm, _, _ = oracle.waveform(th, l, m, m * F)
                a22, _, _ = oracle.waveform(th, 2, 2, 2 * F)
                ratio.append(alm / a22)
            want = abs(_point_mass_moment(q, l, (l + m) % 2 == 1)) / abs(_point_mass_moment(qref, l, (l + m) % 2 == 1))
            assert np.allclose(ratio[0] / ratio[1], want, rtol=1e-12, atol=1e-15), (q, l, m)
    assert _point_mass_moment(1.0, 3, False) == 0.0 and _point_mass_moment(1.0, 2, True) == 0.0


def test_mode_constant_phase_reading_G5():
    """G5 is a READING, not a pin: BASELINE.json writes Psi_lm = (m/2) Psi_22 without argument; applied to the whole
    of Psi_22(2f/m) this gives the constant -(m/2)(pi/4) = -m pi/8 per mode (a stricter stationary-phase treatment
    would give -pi/4 for every m).  The paper fixes neither; DESIGN.md lists it as "reading, unpinned".  This test
    only makes the reading explicit: with t_c = phi_c = 0, Psi_lm(f) + m pi/8 is (m/2) x the PN part of Psi_22(2f/m),
    the PN part being pinned by P1/P2 through t_22."""
    th = THETA.copy(); th[6] = 0.0; th[10] = 0.0
    f = np.array([3e-4, 2e-3])
    for (l, m) in ((2, 1), (3, 3), (3, 2), (4, 4)):
        _, plm, _ = oracle.waveform(th, l, m, f)
        _, p22, _ = oracle.waveform(th, 2, 2, 2 * f / m)
        pn22 = p22 + math.pi / 4
        assert np.allclose(plm + m * math.pi / 8, m / 2 * pn22, rtol=1e-14, atol=0)


def test_amplitude_is_textbook_restricted_pn():
    """O4: A_22 * (Y_22 + Y_2-2)/2 equals (1+cos^2 i)/2 sqrt(5/24) pi^{-2/3} Mc^{5/6} f^{-7/6} / D."""
    th = THETA.copy()
    f = np.array([1e-4, 1e-3, 1e-2])
    a, _, _ = oracle.waveform(th, 2, 2, f)
    eta = th[1] / (1 + th[1]) ** 2
    Mc = eta ** 0.6 * th[0] * TSUN
    iota = th[5]
    hp = (1 + math.cos(iota) ** 2) / 2 * math.sqrt(5 / 24) * math.pi ** (-2 / 3) * Mc ** (5 / 6) * f ** (-7 / 6) / (th[4] * GPC_S)
    kp = 0.5 * (closed_form_swsh(2, 2, iota) + closed_form_swsh(2, -2, iota))
    assert np.allclose(a * kp, hp, rtol=1e-13, atol=0)


# ------------------------------------------------------------------ P3: orbits
@pytest.mark.parametrize("det", [LISA, TAIJI, TQ])
def test_P3_rigid_equilateral_constellation(det):
    for t in np.linspace(-3e7, 6e7, 41):
        x = oracle.orbit(det, t)
        for r, s in ((0, 1), (0, 2), (1, 2)):
            assert np.linalg.norm(x[r] - x[s]) / det.L_m == pytest.approx(1.0, abs=1e-12)
        cen = x.mean(axis=0)
        normal = np.cross(x[1] - x[0], x[2] - x[0])
        normal /= np.linalg.norm(normal)
        aE = 2 * math.pi * t / YR
        if det.kind == 0:
            a = aE + det.kappa
            assert np.allclose(cen, AU * np.array([math.cos(a), math.sin(a), 0.0]), rtol=0, atol=1e-3)
            assert abs(normal[2]) == pytest.approx(0.5, abs=1e-12)       # plane 60 deg from the ecliptic
        else:
            assert np.allclose(cen, AU * np.array([math.cos(aE), math.sin(aE), 0.0]), rtol=0, atol=1e-3)
            nh = np.array([math.cos(det.lat) * math.cos(det.lon), math.cos(det.lat) * math.sin(det.lon), math.sin(det.lat)])
            assert abs(abs(normal @ nh) - 1.0) < 1e-7                      # fixed pointing (G8)
    # orbital periods
    x0, x1 = oracle.orbit(det, 1234.5), oracle.orbit(det, 1234.5 + YR)
    if det.kind == 0:
        assert np.allclose(x0, x1, rtol=0, atol=5e-3)
    else:
        d0 = oracle.orbit(det, 100.0) - oracle.orbit(det, 100.0).mean(axis=0)
        d1 = oracle.orbit(det, 100.0 + det.period_s) - oracle.orbit(det, 100.0 + det.period_s).mean(axis=0)
        assert np.allclose(d0, d1, rtol=0, atol=1e-2)


# ------------------------------------------------------------------ P4: harmonics
def test_P4_goldberg_sum_vs_closed_forms_and_norm():
    for (l, m) in MODES:
        for mm in (m, -m):
            for iota in (0.0, 0.3, 1.1, math.pi / 2, 2.5, math.pi):
                assert oracle.swsh(l, mm, iota) == pytest.approx(closed_form_swsh(l, mm, iota), abs=3e-15)
            # int |Y|^2 dOmega = 1 (Gauss-Legendre in cos(iota))
            xg, wg = np.polynomial.legendre.leggauss(24)
            vals = np.array([oracle.swsh(l, mm, math.acos(x)) for x in xg])
            assert 2 * math.pi * np.sum(wg * vals ** 2) == pytest.approx(1.0, abs=1e-13)
    # (2,2): h_x = -i (2c/(1+c^2)) h_+  <=>  Kx/K+ = -2ic/(1+c^2)
    for iota in (0.2, 1.0, 2.8):
        Yp, Ym = oracle.swsh(2, 2, iota), oracle.swsh(2, -2, iota)
        c = math.cos(iota)
        assert (Yp - Ym) / (Yp + Ym) == pytest.approx(2 * c / (1 + c * c), rel=1e-13)


# ------------------------------------------------------------------ P5: Eq. 5 is the transform of Eq. 1
@pytest.mark.parametrize("det", [LISA, TAIJI, TQ])
@pytest.mark.parametrize("lm", list(MODES))
def test_P5_single_link_is_fourier_transform_of_eq1(det, lm):
    l, m = lm
    th = THETA.copy(); th[1] = 2.2; th[5] = 1.1
    k, u, v = frame(th[7], th[8])
    P = mode_tensor(l, m, th[5], th[7], th[8], th[9])
    Lbar = det.L_m / C_SI
    for f in (2e-4, 3e-3, 4e-2):
        a, psi, t = oracle.waveform(th, l, m, np.array([f]))
        h = a[0] * np.exp(-1j * psi[0])
        x = oracle.orbit(det, t[0]) / C_SI                      # seconds, at t_lm(f)
        y = oracle.links(th, l, m, f, det)
        for i, (r, s) in enumerate(oracle.LINK_ORDER):
            n = (x[r - 1] - x[s - 1]) / Lbar
            want = ((np.exp(-2j * math.pi * f * (Lbar + k @ x[s - 1])) - np.exp(-2j * math.pi * f * (k @ x[r - 1])))
                    / (2 * (1 - k @ n)) * (n @ P @ n) * h)
            # kind 1 forms n from positions ~1 AU apart from the origin: 3 digits lost in the TEST's n
            tol = 1e-9 if det.kind == 0 else 3e-8
            assert abs(y[i] - want) <= tol * abs(want), (det.name, lm, f, r, s)


def test_P5b_sinc_is_sin_x_over_x_and_regular_at_zero():
    """Source exactly along an arm: 1 - k.n -> 0, Eq. 5's sinc -> 1 (not numpy's sin(pi x)/(pi x))."""
    th = THETA.copy()
    x = oracle.orbit(LISA, 0.0)
    n12 = (x[0] - x[1]) / LISA.L_m
    # k = n12 requires source direction -n12; choose t_f(f) = 0 by construction: use t_c so that t_22(f)=0
    f = 1e-3
    _, _, t = oracle.waveform(th, 2, 2, np.array([f]))
    th[10] -= t[0]                                            # now t_22(f) = 0
    th[8] = math.asin(-n12[2] * -1.0) * -1.0                  # beta with -k = source dir = -n12 ... k = n12
    th[7] = math.atan2(-n12[1], -n12[0])
    k, _, _ = frame(th[7], th[8])
    assert np.allclose(k, n12, atol=1e-12)
    y = oracle.links(th, 2, 2, f, LISA)
    assert np.all(np.isfinite(y.view(np.float64)))
    # for the aligned link n.P.n = 0 (transverse wave), so y12 vanishes to rounding; y21 (k.n = -1) too
    scale = np.abs(y).max()
    assert abs(y[0]) < 1e-12 * scale and abs(y[1]) < 1e-12 * scale


# ------------------------------------------------------------------ P6: Eq. 6 is Eq. 2 with D -> z
def literal_eq2(y, z, gen):
    """Eq. 2 written out term by term (G1: 8th positive term of X_2.0 ends ... D21 D13 y31)."""
    def X(y13, y31, y12, y21):
        if gen == 15:
            return (y13 + z * y31 + z ** 2 * y12 + z ** 3 * y21
                    - y12 - z * y21 - z ** 2 * y13 - z ** 3 * y31)
        return (y13 + z * y31 + z ** 2 * y12 + z ** 3 * y21
                + z ** 4 * y12 + z ** 5 * y21 + z ** 6 * y13 + z ** 7 * y31
                - y12 - z * y21 - z ** 2 * y13 - z ** 3 * y31
                - z ** 4 * y13 - z ** 5 * y31 - z ** 6 * y12 - z ** 7 * y21)
    g = {(1, 2): y[0], (2, 1): y[1], (1, 3): y[2], (3, 1): y[3], (2, 3): y[4], (3, 2): y[5]}
    cyc = lambda i: i % 3 + 1
    out = []
    a, b, c = 1, 2, 3
    for _ in range(3):
        out.append(X(g[(a, c)], g[(c, a)], g[(a, b)], g[(b, a)]))
        a, b, c = cyc(a), cyc(b), cyc(c)
    return np.array(out)


@pytest.mark.parametrize("gen", [15, 20])
def test_P6_tdi_closed_form_equals_delay_operator_sum(gen):
    rng = np.random.default_rng(7)
    for f in (1e-4, 2.3e-3, 4.1e-2):
        y = rng.standard_normal(6) + 1j * rng.standard_normal(6)
        z = np.exp(-2j * math.pi * f * 2.5e9 / C_SI)
        got = oracle.tdi(y, f, 2.5e9, gen)
        want = literal_eq2(y, z, gen)
        assert np.allclose(got, want, rtol=1e-12, atol=1e-14)


# ------------------------------------------------------------------ P7, P8: long-wavelength limit
def long_wavelength_AE(th, det, f, l=2, m=2):
    a_, psi, t = oracle.waveform(th, l, m, np.array([f]))
    h = a_[0] * np.exp(-1j * psi[0])
    x = oracle.orbit(det, t[0]) / C_SI
    k, _, _ = frame(th[7], th[8])
    P = mode_tensor(l, m, th[5], th[7], th[8], th[9])
    Lbar = det.L_m / C_SI
    arm = lambda r, s: ((x[r] - x[s]) / Lbar) @ P @ ((x[r] - x[s]) / Lbar) * h
    a, b, c = arm(1, 2), arm(2, 0), arm(0, 1)          # arms opposite spacecraft 1, 2, 3
    p0 = x.mean(axis=0)
    Kf = 8 * math.pi ** 2 * f ** 2 * Lbar ** 2 * np.exp(-2j * math.pi * f * (k @ p0))
    if det.tdi_gen == 20:
        Kf = Kf * 8j * math.pi * f * Lbar
    return Kf * (a - 2 * b + c) / math.sqrt(2), Kf * math.sqrt(1.5) * (a - c)


@pytest.mark.parametrize("det", [LISA15, LISA, TAIJI])
def test_P7_low_frequency_response_matches_pattern_functions(det):
    th = THETA.copy()
    devs = []
    for f in (1e-6, 1e-5):
        r = oracle.response(th, np.array([f]), W.Model(1, (det,)))[0, 0, :, 0]
        A, E = long_wavelength_AE(th, det, f)
        devs.append(max(abs(r[0] - A) / abs(A), abs(r[1] - E) / abs(E)))
    assert devs[0] < 4e-4 and devs[1] < 4e-3           # SURVEY probe: 1.0e-4, 1.0e-3 for LISA-like 1.5
    assert 5.0 < devs[1] / devs[0] < 20.0              # -> 0 linearly in f


@pytest.mark.parametrize("det", [LISA15, LISA, TQ])
def test_P8_T_channel_is_suppressed_at_low_frequency(det):
    th = THETA.copy()
    f = np.array([1e-5, 1e-4, 1e-3]) if det.kind == 0 else np.array([1e-4, 1e-3, 1e-2])
    r = oracle.response(th, f, W.Model(1, (det,)))[0, 0]
    ratio = np.abs(r[2]) / np.abs(r[0])
    assert ratio[1] < 1e-7
    for i in (0, 1):
        assert 2.5 < math.log10(ratio[i + 1] / ratio[i]) < 3.5      # |T|/|A| ~ f^3


# ------------------------------------------------------------------ P9, P10: likelihood invariants
def small_workload(mask=1, dets=(LISA,), N=512):
    grid = W.Grid(1e-4, (1e-2 - 1e-4) / (N - 1), N)
    return grid, W.Model(mask, tuple(dets))


def test_P9_noiseless_lnL_zero_at_injection_and_maximal_there():
    grid, model = small_workload(mask=31)
    th0 = THETA.copy(); th0[10] = 2.0e5; th0[2] = 0.1; th0[3] = -0.2
    f = grid.freqs()
    d = oracle.response(th0, f, model)[0]
    psd = np.stack([W.psd_aet(x, f) for x in model.detectors])
    assert oracle.loglike(th0, d, psd, grid, model)[0] == 0.0
    scales = np.array([2e6, 3.0, 1.0, 1.0, 10.0, 1.0, 1.0, 1.0, 1.0, 1.0, 1.0])
    for j in range(11):
        prev = 0.0
        for eps in (1e-7, 1e-6, 1e-5, 1e-4):
            vals = []
            for sgn in (+1, -1):
                th = th0.copy(); th[j] += sgn * eps * scales[j]
                vals.append(oracle.loglike(th, d, psd, grid, model)[0])
            assert max(vals) < 0.0, (j, eps, vals)
            assert min(vals) < prev                       # falls away from the maximum
            prev = max(vals)


def test_P10_distance_scaling_and_polarisation_period():
    grid, model = small_workload(mask=31, dets=(LISA, TQ))
    f = grid.freqs()
    psd = np.stack([W.psd_aet(x, f) for x in model.detectors])
    zero = np.zeros((2, 3, grid.N), dtype=np.complex128)
    th = THETA.copy()
    hh = -2.0 * oracle.loglike(th, zero, psd, grid, model)[0]
    th2 = th.copy(); th2[4] *= 2.0
    hh2 = -2.0 * oracle.loglike(th2, zero, psd, grid, model)[0]
    assert hh2 == pytest.approx(hh / 4.0, rel=1e-15)
    thp = th.copy(); thp[9] += math.pi
    r0, r1 = oracle.response(th, f, model), oracle.response(thp, f, model)
    assert np.abs(r1 - r0).max() <= 1e-14 * np.abs(r0).max()


def test_O11_whittle_sum_brute_force():
    """lnL = -2 df sum |d-h|^2 / S (Eq. 10 with T = 1/df), brute force in numpy on a tiny case;
    bins with S = 0 or non-finite are skipped (G9)."""
    grid, model = small_workload(mask=31, dets=(LISA, TAIJI), N=97)
    f = grid.freqs()
    rng = np.random.default_rng(5)
    psd = np.stack([W.psd_aet(x, f) for x in model.detectors])
    th = np.stack([THETA, THETA * (1 + 1e-3)])
    h = oracle.response(th, f, model)
    d = h[0] + W.coloured_noise(psd, grid.df, rng)
    psd[0, 1, 5] = 0.0; psd[1, 2, 9] = np.inf; psd[1, 0, 11] = np.nan
    ok = np.isfinite(psd) & (psd > 0)
    want = [-2.0 * grid.df * np.sum((np.abs(d - h[b]) ** 2)[ok] / psd[ok]) for b in range(2)]
    got = oracle.loglike(th, d, psd, grid, model)
    assert np.allclose(got, want, rtol=1e-13, atol=0)


def test_P15_noise_expectation_fixes_the_normalisation():
    """G12 + Eq. 9/10: with d = h(theta0) + n, lnL(theta0) ~ -3 N n_det +- sqrt(3 N n_det)."""
    N = 8192
    grid = W.Grid(1e-4, W.MONTH_DF, N)
    model = W.Model(1, (LISA, TAIJI))
    f = grid.freqs()
    psd = np.stack([W.psd_aet(x, f) for x in model.detectors])
    th0 = THETA.copy()
    d = oracle.response(th0, f, model)[0] + W.coloured_noise(psd, grid.df, np.random.default_rng(101))
    lnL = oracle.loglike(th0, d, psd, grid, model)[0]
    mean, sd = -3.0 * N * 2, math.sqrt(3.0 * N * 2)
    assert abs(lnL - mean) < 4.5 * sd


# ------------------------------------------------------------------ P11: noise PSD forms (input recipe, G13)
@pytest.mark.parametrize("gen", [15, 20])
def test_P11_psd_from_link_noise_propagation(gen):
    det = W.lisa_like(gen)
    Lm = det.L_m
    for f in (1.7e-4, 2e-3, 1.3e-2, 4.7e-2):
        x = 2 * math.pi * f * Lm / C_SI
        z = np.exp(-1j * x)
        S_oms = (det.A_oms * 2 * math.pi * f / C_SI) ** 2 * (1 + (2e-3 / f) ** 4)
        S_acc = (det.A_acc / (2 * math.pi * f * C_SI)) ** 2 * (1 + (0.4e-3 / f) ** 2) * (1 + (f / 8e-3) ** 4)
        S = np.zeros(3)
        for i, (r, s) in enumerate(oracle.LINK_ORDER):
            # OMS noise of link rs: y_rs += n
            y = np.zeros(6, dtype=complex); y[i] = 1.0
            S += np.abs(aet_of(oracle.tdi(y, f, Lm, gen))) ** 2 * S_oms
            # test-mass noise on spacecraft r facing s: y_rs += a, y_sr += z a
            y = np.zeros(6, dtype=complex); y[i] = 1.0
            y[oracle.LINK_ORDER.index((s, r))] = z
            S += np.abs(aet_of(oracle.tdi(y, f, Lm, gen))) ** 2 * S_acc
        want = W.psd_aet(det, np.array([f]))[:, 0]
        assert np.allclose(S, want, rtol=1e-11, atol=0)


def aet_of(XYZ):
    X, Y, Z = XYZ
    return np.array([(Z - X) / math.sqrt(2), (X - 2 * Y + Z) / math.sqrt(6), (X + Y + Z) / math.sqrt(3)])


def test_eq3_channel_combination():
    """A, E, T of the oracle are Eq. 3 applied to the oracle's own X, Y, Z (links -> tdi)."""
    th = THETA.copy()
    for det in (LISA, LISA15, TQ):
        for f in (3e-4, 8e-3):
            tot = np.zeros(3, dtype=complex)
            for (l, m) in MODES:
                tot += aet_of(oracle.tdi(oracle.links(th, l, m, f, det), f, det.L_m, det.tdi_gen))
            r = oracle.response(th, np.array([f]), W.Model(31, (det,)))[0, 0, :, 0]
            assert np.allclose(r, tot, rtol=1e-13, atol=1e-16 * np.abs(tot).max())


# ------------------------------------------------------------------ P12, P13: forward-mode derivatives
def test_P12_snr_derivative_wrt_inclination_closed_form():
    """(2,2) only: rho^2(iota) = a g+^2 + b gx^2 + 2 c g+ gx (Fig. 3 design)."""
    grid, model = small_workload(mask=1)
    f = grid.freqs()
    psd = np.stack([W.psd_aet(x, f) for x in model.detectors])
    zero = np.zeros((1, 3, grid.N), dtype=np.complex128)
    gp = lambda i: (1 + math.cos(i) ** 2) / 2
    gx = lambda i: math.cos(i)
    th = THETA.copy()

    def rho2(iota):
        t = th.copy(); t[5] = iota
        return -2.0 * oracle.loglike(t, zero, psd, grid, model)[0]
    nodes = (0.3, 1.2, 2.4)
    Amat = np.array([[gp(i) ** 2, gx(i) ** 2, 2 * gp(i) * gx(i)] for i in nodes])
    a, b, c = np.linalg.solve(Amat, np.array([rho2(i) for i in nodes]))
    for iota in (0.4, 0.9, 1.9, 2.9):
        assert rho2(iota) == pytest.approx(a * gp(iota) ** 2 + b * gx(iota) ** 2 + 2 * c * gp(iota) * gx(iota), rel=1e-12)
        dgp, dgx = -math.cos(iota) * math.sin(iota), -math.sin(iota)
        d_rho2 = 2 * a * gp(iota) * dgp + 2 * b * gx(iota) * dgx + 2 * c * (dgp * gx(iota) + gp(iota) * dgx)
        t = th.copy(); t[5] = iota
        _, grad = oracle.fisher(t, zero, psd, grid, model)     # d = 0: grad_i = -<h|d_i h> = -1/2 d_i rho^2
        assert -2.0 * grad[0, 5] == pytest.approx(d_rho2, rel=1e-10)
        # the quantity of Fig. 3: d rho / d iota
        assert -grad[0, 5] / math.sqrt(rho2(iota)) == pytest.approx(d_rho2 / (2 * math.sqrt(rho2(iota))), rel=1e-10)


FD_STEPS = np.array([2.0, 3e-5, 1e-4, 1e-4, 1e-3, 1e-4, 1e-4, 1e-5, 1e-5, 1e-4, 1e-2])


def richardson_dh(th, j, f, model):
    """d h / d theta_j by central differences with steps h, h/2, h/4 and two Richardson levels."""
    est = []
    for div in (1.0, 2.0, 4.0):
        h = FD_STEPS[j] / div
        tp, tm = th.copy(), th.copy()
        tp[j] += h; tm[j] -= h
        est.append((oracle.response(tp, f, model)[0] - oracle.response(tm, f, model)[0]) / (2 * h))
    r1 = [(4 * est[1] - est[0]) / 3, (4 * est[2] - est[1]) / 3]
    return (16 * r1[1] - r1[0]) / 15


@pytest.mark.parametrize("mask,dets", [(1, (LISA,)), (31, (LISA, TQ))])
def test_P13_fisher_and_gradient_vs_richardson_finite_differences(mask, dets):
    grid, model = small_workload(mask=mask, dets=dets, N=384)
    f = grid.freqs()
    psd = np.stack([W.psd_aet(x, f) for x in model.detectors])
    th = THETA.copy(); th[10] = 3.0e5; th[2] = 0.3; th[3] = -0.1; th[1] = 2.5
    h = oracle.response(th, f, model)[0]
    d = h + W.coloured_noise(psd, grid.df, np.random.default_rng(3))
    F, grad = oracle.fisher(th, d, psd, grid, model)
    F, grad = F[0], grad[0]
    dh = [richardson_dh(th, j, f, model) for j in range(11)]
    hh = inner(h, h, psd, grid.df)
    for i in range(11):
        assert grad[i] == pytest.approx(inner(d - h, dh[i], psd, grid.df), rel=1e-6, abs=1e-6 * math.sqrt(F[i, i]) * math.sqrt(hh))
        for j in range(11):
            assert F[i, j] == F[j, i]
            assert abs(F[i, j] - inner(dh[i], dh[j], psd, grid.df)) <= 1e-6 * math.sqrt(F[i, i] * F[j, j])
    # closed forms: d h / d D_L = -h / D_L
    assert F[4, 4] == pytest.approx(hh / th[4] ** 2, rel=1e-12)
    assert grad[4] == pytest.approx(-inner(d - h, h, psd, grid.df) / th[4], rel=1e-9)
    if mask == 1:                                   # (2,2) only: d h / d phi_c = 2 i h
        assert F[6, 6] == pytest.approx(4 * hh, rel=1e-12)
        assert abs(F[6, 4]) <= 1e-12 * math.sqrt(F[6, 6] * F[4, 4])
    # the Fisher matrix without data equals the one with data
    F2, g2 = oracle.fisher(th, None, psd, grid, model)
    assert g2 is None and np.array_equal(F2[0], F)


# ------------------------------------------------------------------ P14: is double enough?
def test_P14_double_vs_binary128_on_config1_bins():
    wl = W.config(1)
    f = wl.grid.freqs()[::64]                        # 64 bins across the band
    r = oracle.response(wl.params, f, wl.model)
    rq = oracle.response(wl.params, f, wl.model, quad=True)
    for b in range(wl.B):
        for c in range(3):
            # tolerance: |Psi| * 2^-53 with |Psi| up to ~3e5 rad for the lightest systems -> 3e-11;
            # measured worst case is ~1e-11 (SURVEY's 1e-12 holds for M >= 1e6 only)
            assert np.abs(r[b, 0, c] - rq[b, 0, c]).max() <= 1e-10 * np.abs(rq[b, 0, c]).max()


def test_P14_double_vs_binary128_over_the_full_band_and_at_the_nulls():
    """P14 over the band of configs 2-5 (0.1 ... 101 mHz) and in the neighbourhood of every in-band zero of g(z)
    (Eq. 6; G9): bin by bin, the double oracle must agree with its own binary128 evaluation to 2e-9 of the bin's
    largest channel (2 pi f t_c reaches 1.3e6 rad: one ulp of that phase is 2.3e-10 rad; measured 6e-10), and
    also within +-3 bins of the zeros, where the expanded form 1 - z^2 - z^4 + z^6 lost up to 3e-7 (the oracle
    evaluates the product (1 - z^2)(1 - z^4) of SURVEY O10 for that reason)."""
    grid = W.config(2).grid
    fgrid = grid.freqs()
    th = W.config(4, B=2).params
    for gen in (20, 15):
        for det in (W.lisa_like(gen), W.taiji_like(gen), W.tianqin_like(gen)):
            idx = set(range(0, grid.N, 4099))
            step = C_SI / ((4.0 if gen == 20 else 2.0) * det.L_m)
            nulls = [n * step for n in range(1, int(fgrid[-1] / step) + 1)]
            for fn in nulls:
                k0 = int(round((fn - grid.f0) / grid.df))
                idx |= {k for k in range(k0 - 3, k0 + 4) if 0 <= k < grid.N}
            f = fgrid[np.array(sorted(idx))]
            model = W.Model(W.MODES_HM, (det,))
            r = oracle.response(th, f, model)[:, 0]
            rq = oracle.response(th, f, model, quad=True)[:, 0]
            s = np.abs(rq).max(axis=1, keepdims=True)
            err = (np.abs(r - rq) / s).max(axis=(0, 1))
            # the bin NEAREST a zero may sit arbitrarily close to it (LISA-like 29.979 mHz: 0.005 bin, |g| 5e-7 of
            # its typical size): there the double rounding of the argument 2 pi f L shows as 3e-9; tolerance 1e-8
            nearest = np.zeros(f.size, dtype=bool)
            for fn in nulls:
                nearest[np.argmin(np.abs(f - fn))] = True
            assert err[~nearest].max() <= 2e-9 and err.max() <= 1e-8, (gen, det.name, err.max())
            if det.kind == 0:
                assert len(nulls) >= (3 if gen == 20 else 1)


# ------------------------------------------------------------------ P16: SNR sanity on the full config-2 grid
def test_P16_snr_of_config2_injection():
    g = _golden()
    wl = W.config(2, B=1)
    f = wl.grid.freqs()
    psd = wl.psd()
    h22 = oracle.response(wl.theta_inj, f, wl.model)[0]
    assert inner(h22, h22, psd, wl.grid.df) == pytest.approx(g["snr2_22"][0][0], rel=2e-3)
    hm = oracle.response(wl.theta_inj, f, W.Model(W.MODES_HM, wl.model.detectors))[0]
    tot, sa, se, st = g["snr2_hm"][0]
    assert inner(hm, hm, psd, wl.grid.df) == pytest.approx(tot, rel=2e-3)
    for c, want in enumerate((sa, se, st)):
        assert inner(hm[0, c], hm[0, c], psd[0, c], wl.grid.df) == pytest.approx(want, rel=5e-3)


# ------------------------------------------------------------------ domain errors and argument checks
def test_out_of_domain_samples_and_bad_arguments():
    grid, model = small_workload(N=16)
    f = grid.freqs()
    psd = np.stack([W.psd_aet(x, f) for x in model.detectors])
    d = np.zeros((1, 3, 16), dtype=np.complex128)
    bad = np.stack([THETA, THETA, THETA, THETA, THETA])
    bad[1, 0] = -1.0; bad[2, 1] = 0.5; bad[3, 4] = 0.0; bad[4, 6] = np.nan
    lnL = oracle.loglike(bad, d, psd, grid, model)
    assert np.isfinite(lnL[0]) and np.all(np.isneginf(lnL[1:]))
    r = oracle.response(bad, f, model)
    assert np.all(np.isfinite(r[0].view(np.float64))) and np.all(np.isnan(r[1:].view(np.float64)))
    with pytest.raises(ValueError):
        oracle.loglike(THETA, d, psd, W.Grid(1e-4, -1.0, 16), model)
    with pytest.raises(ValueError):
        oracle.response(THETA, f, W.Model(0, (LISA,)))
    with pytest.raises(ValueError):
        oracle.response(THETA, f, W.Model(1, (W.Detector("x", 2, 20, 1e9),)))


# ------------------------------------------------------------------ T1: tabulated mode waveforms
def test_T1_interpolants_are_exact_for_cubics_and_zero_outside():
    """Cubic Hermite (phase, slopes 2 pi t_j), its derivative (t_f) and 4-node Lagrange (amplitude) reproduce
    cubic polynomials exactly on non-uniform nodes; outside the table the interpolants are undefined (mode = 0)."""
    rng = np.random.default_rng(5)
    fn = np.sort(rng.uniform(1e-3, 2e-3, 40))
    x = (fn - 1.5e-3) / 1e-3
    cp, ca = rng.normal(size=4) * [50.0, 400.0, 30.0, 20.0], rng.normal(size=4)
    P = lambda y: cp[0] + cp[1] * y + cp[2] * y ** 2 + cp[3] * y ** 3
    dP = lambda y: (cp[1] + 2 * cp[2] * y + 3 * cp[3] * y ** 2) / 1e-3
    A = lambda y: ca[0] + ca[1] * y + ca[2] * y ** 2 + ca[3] * y ** 3
    f = np.concatenate([rng.uniform(fn[0], fn[-1], 500), fn[[0, 7, -1]]])
    y = (f - 1.5e-3) / 1e-3
    a, p, t = oracle.tab_waveform(fn, A(x), P(x), dP(x) / (2 * np.pi), f)
    assert np.abs(p - P(y)).max() <= 1e-11 * np.abs(P(y)).max()
    assert np.abs(t - dP(y) / (2 * np.pi)).max() <= 1e-10 * np.abs(dP(y)).max()
    assert np.abs(a - A(y)).max() <= 1e-12 * np.abs(A(y)).max()
    a, p, t = oracle.tab_waveform(fn, A(x), P(x), dP(x) / (2 * np.pi), np.array([fn[0] * 0.999, fn[-1] * 1.001]))
    assert np.all(np.isnan(a)) and np.all(np.isnan(p)) and np.all(np.isnan(t))


@pytest.mark.parametrize("mask,dets", [(1, (LISA,)), (31, (LISA, TQ))])
def test_T1_tabulated_path_reproduces_the_analytic_path(mask, dets):
    """Tables of the oracle's own analytic modes at t_c = 0, phi_c = 0, D_L = 1 Gpc, pushed through the tabulated
    path with theta's t_c, phi_c, D_L, give the analytic response up to the interpolation error, which falls as
    K^-4 (pins mode order, the signs of the t_c and phi_c terms, the 1/D_L scaling and the stencils)."""
    model = W.Model(mask, dets)
    f = np.geomspace(1.2e-4, 0.09, 400)
    th = THETA.copy()
    th[2], th[3] = 0.3, -0.2
    want = oracle.response(th, f, model)[0]
    errs = []
    for K in (200, 400, 3000):
        table = W.table_from_waveform_fn(th, mask, W.log_nodes(1e-4, 0.1, K), oracle.waveform)
        got = oracle.response_tab(th, table, f, model)[0]
        errs.append(max(np.abs(got[d] - want[d]).max() / np.abs(want[d]).max() for d in range(len(dets))))
    assert errs[2] <= 2e-10, errs                    # floor: rounding of the 1e6 rad phase (1e-16 relative)
    assert errs[0] / errs[1] > 10.0, errs            # fourth order: 16 per halving of the node spacing


def test_T1_extrinsic_parameters_band_limits_and_likelihood():
    model = W.Model(3, (LISA,))                                  # (2,2) and (2,1)
    grid = W.Grid(1e-4, 2.5e-6, 600)
    f = grid.freqs()
    th = np.tile(THETA, (3, 1))
    th[1, 4] *= 2.0                                              # D_L doubled
    th[2, 6] += np.pi                                            # phi_c + pi: m = 2 unchanged, m = 1 flips sign
    fn = W.log_nodes(1e-4, 1.2e-3, 900)                          # the table ends inside the grid
    table = W.chirp_table(th, 3, fn)
    r = oracle.response_tab(th, table, f, model)
    inside = f <= fn[-1]
    assert np.all(r[:, :, :, ~inside] == 0.0) and np.abs(r[0, 0, 0, inside]).min() > 0.0
    assert np.allclose(r[1], 0.5 * r[0], rtol=1e-13, atol=0.0)
    only22 = oracle.response_tab(th, tuple(x if x.ndim == 1 else x[:, :1] for x in table), f, W.Model(1, (LISA,)))
    only21 = oracle.response_tab(th, tuple(x if x.ndim == 1 else x[:, 1:] for x in table), f, W.Model(2, (LISA,)))
    scale = np.abs(r[0]).max()
    assert np.abs(only22[0] + only21[0] - r[0]).max() <= 1e-13 * scale           # modes add, in bit order
    assert np.abs(only22[2] - only22[0]).max() <= 1e-9 * scale
    assert np.abs(only21[2] + only21[0]).max() <= 1e-9 * np.abs(only21[0]).max()
    # noiseless data from sample 0: lnL = 0 there, negative elsewhere, and equal to the Whittle sum written out
    psd = W.psd_aet(LISA, f)[None]
    lnL = oracle.loglike_tab(th, table, r[0], psd, grid, model)
    assert lnL[0] == 0.0 and lnL[1] < 0.0 and lnL[2] < 0.0
    brute = -0.5 * 4.0 * grid.df * np.sum(np.abs(r[0] - r[1]) ** 2 / psd)
    assert abs(lnL[1] - brute) <= 1e-12 * abs(brute)


# ------------------------------------------------------------------ T2: tabulated numerical orbits
def test_T2_hermite_is_exact_on_cubic_trajectories_and_empty_outside():
    rng = np.random.default_rng(8)
    t0, dt, K = -1000.0, 3600.0, 9
    t = t0 + dt * np.arange(K)
    co = rng.normal(size=(4, 3, 3)) * np.array([1e11, 1e4, 1e-3, 1e-10])[:, None, None]     # x = a + b t + c t^2 + d t^3
    pos = sum(co[i] * t[:, None, None] ** i for i in range(4))
    vel = sum(i * co[i] * t[:, None, None] ** (i - 1) for i in range(1, 4))
    for tt in (t0, t0 + 0.37 * dt, t0 + 4.5 * dt, t0 + 7.999 * dt, t[-1]):
        want = sum(co[i] * tt ** i for i in range(4))
        got = oracle.orbit_tab(t0, dt, pos, vel, tt)
        assert np.allclose(got, want, rtol=1e-13, atol=1e-3)
    assert oracle.orbit_tab(t0, dt, pos, vel, t0 - 1.0) is None and oracle.orbit_tab(t0, dt, pos, vel, t[-1] + 1.0) is None
    # the nodes themselves are reproduced exactly
    assert np.array_equal(oracle.orbit_tab(t0, dt, pos, vel, t[3]), pos[3])


@pytest.mark.parametrize("det,dt", [(LISA, 3600.0), (TAIJI, 3600.0), (TQ, 300.0)])
def test_T2_dense_table_reproduces_the_analytic_orbit_and_rigid_arms(det, dt):
    t0, K = 1.0e6, 200
    tab = W.orbit_table_from_fn([det], t0, dt, K, oracle.orbit)
    rng = np.random.default_rng(2)
    for tt in t0 + dt * (K - 1) * rng.uniform(0.0, 1.0, 25):
        x = oracle.orbit_tab(tab[0], tab[1], tab[2][0], tab[3][0], tt)
        assert np.allclose(x, oracle.orbit(det, tt), rtol=0, atol=2e-3)                   # metres, at 1.5e11 m
        for r, s_ in ((0, 1), (0, 2), (1, 2)):
            assert np.linalg.norm(x[r] - x[s_]) / det.L_m == pytest.approx(1.0, abs=1e-9)   # P3 on the interpolant


def test_T2_response_and_likelihood_with_dense_tables_match_the_analytic_path():
    """fed dense samples of the analytic orbits, the tabulated-orbit path reproduces O8-O11; a table that starts late
    leaves the low frequencies (early t_lm) empty; the Whittle sum is the brute-force one"""
    th = np.array([THETA, THETA * (1 + 0.01 * np.array([1, -1, 0, 0, 2, 1, -1, 1, 1, -1, 0.5]))])
    dets = (LISA, TAIJI, TQ)
    model = W.Model(W.MODES_HM, dets)
    f = np.geomspace(2e-4, 9e-2, 60)
    tl = np.array([oracle.waveform(t_, l, m, f)[2] for t_ in th for (l, m) in MODES])     # every t_lm(f) of the test
    t_lo, t_hi = tl.min() - 10.0, tl.max() + 10.0           # (t_lm is not monotonic beyond v ~ 1, G2)
    dt = 300.0
    K = int((t_hi - t_lo) / dt) + 2
    # one table per detector on the same grid; the short-period detector sets dt
    tab = W.orbit_table_from_fn(dets, t_lo, dt, K, oracle.orbit)
    got = oracle.response_orb(th, tab, f, model)
    want = oracle.response(th, f, model)
    for d in range(3):
        assert np.abs(got[:, d] - want[:, d]).max() <= 1e-9 * np.abs(want[:, d]).max()
    # late table: modes whose t_lm(f) precedes the first node vanish
    _, _, t22 = oracle.waveform(th[0], 2, 2, f)
    cut = 12                                     # still on the monotonic branch of t_22(f)
    t_start = 0.5 * (t22[cut - 1] + t22[cut])
    K2 = int((t_hi - t_start) / dt) + 2
    late = W.orbit_table_from_fn(dets[:1], t_start, dt, K2, oracle.orbit)
    m22 = W.Model(W.MODES_22_ONLY, dets[:1])
    r = oracle.response_orb(th[:1], late, f, m22)[0, 0]
    assert np.all(np.diff(t22[:cut + 8]) > 0)
    assert np.all(r[:, :cut] == 0) and np.all(np.abs(r[0, cut:cut + 8]) > 0)
    # Whittle sum by brute force
    grid = W.Grid(1e-3, 2e-5, 50)
    fg = grid.freqs()
    rng = np.random.default_rng(4)
    psd = np.stack([W.psd_aet(dd, fg) for dd in dets])
    data = W.coloured_noise(psd, grid.df, rng) + oracle.response_orb(th[:1], tab, fg, model)[0]
    h = oracle.response_orb(th, tab, fg, model)
    brute = -0.5 * 4.0 * grid.df * (np.abs(data[None] - h) ** 2 / psd[None]).sum(axis=(1, 2, 3))
    assert np.allclose(oracle.loglike_orb(th, tab, data, psd, grid, model), brute, rtol=1e-12, atol=0)


# ------------------------------------------------------------------ T1 x O12: Fisher matrix on tabulated waveforms
@pytest.mark.parametrize("mask,dets", [(1, (LISA,)), (31, (LISA, TQ))])
def test_T1_fisher_tab_vs_richardson_finite_differences_and_closed_forms(mask, dets):
    """oracle.fisher_tab (dual numbers through the tabulated path) against Richardson-extrapolated central differences
    of oracle.response_tab, the D_L / phi_c closed forms, and exact zeros for the parameters the path ignores"""
    grid, model = small_workload(mask=mask, dets=dets, N=384)
    f = grid.freqs()
    psd = np.stack([W.psd_aet(x, f) for x in model.detectors])
    th = THETA.copy(); th[10] = 3.0e5; th[1] = 2.5
    table = W.table_from_waveform_fn(th[None], mask, W.log_nodes(f[0], f[-1], 300), oracle.waveform)
    h = oracle.response_tab(th, table, f, model)[0]
    d = h + W.coloured_noise(psd, grid.df, np.random.default_rng(3))
    F, grad = oracle.fisher_tab(th, table, d, psd, grid, model)
    F, grad = F[0], grad[0]
    used = [4, 5, 6, 7, 8, 9, 10]

    def dh_tab(j):
        est = []
        for div in (1.0, 2.0, 4.0):
            st = FD_STEPS[j] / div
            tp, tm = th.copy(), th.copy()
            tp[j] += st; tm[j] -= st
            est.append((oracle.response_tab(tp, table, f, model)[0] - oracle.response_tab(tm, table, f, model)[0]) / (2 * st))
        r1 = [(4 * est[1] - est[0]) / 3, (4 * est[2] - est[1]) / 3]
        return (16 * r1[1] - r1[0]) / 15

    dh = {j: dh_tab(j) for j in used}
    hh = inner(h, h, psd, grid.df)
    for i in used:
        assert grad[i] == pytest.approx(inner(d - h, dh[i], psd, grid.df), rel=1e-6, abs=1e-6 * math.sqrt(F[i, i]) * math.sqrt(hh))
        for j in used:
            assert F[i, j] == F[j, i]
            assert abs(F[i, j] - inner(dh[i], dh[j], psd, grid.df)) <= 1e-6 * math.sqrt(F[i, i] * F[j, j])
    assert np.all(F[:4, :] == 0) and np.all(F[:, :4] == 0) and np.all(grad[:4] == 0)       # M, q, chi1, chi2: ignored
    assert F[4, 4] == pytest.approx(hh / th[4] ** 2, rel=1e-12)
    assert grad[4] == pytest.approx(-inner(d - h, h, psd, grid.df) / th[4], rel=1e-9)
    if mask == 1:                                   # (2,2) only: d h / d phi_c = 2 i h
        assert F[6, 6] == pytest.approx(4 * hh, rel=1e-12)
        assert abs(F[6, 4]) <= 1e-12 * math.sqrt(F[6, 6] * F[4, 4])
    F2, g2 = oracle.fisher_tab(th, table, None, psd, grid, model)
    assert g2 is None and np.array_equal(F2[0], F)
    # on tables of the analytic modes the extrinsic block approaches the analytic path's (fourth order in the spacing)
    Fa, _ = oracle.fisher(th, d, psd, grid, model)
    ix = np.ix_(used, used)
    dd = np.sqrt(np.diag(Fa[0]))[used]
    assert (np.abs(F[ix] - Fa[0][ix]) / np.outer(dd, dd)).max() <= 1e-5
