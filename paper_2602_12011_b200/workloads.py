"""Seeded synthetic workloads shaped like the paper's MBHB analyses.

This module is the ONE thing the CUDA path's callers (tests, bench.py, smoke) and the
oracle's callers share.  It holds input recipes only -- parameter draws, frequency
grids, detector descriptions, analytic noise PSDs (G13) and coloured Gaussian noise
(G12) -- and none of the method's arithmetic: it never evaluates a waveform, an orbit
or a response.  The injected signal is obtained from a `response_fn` the caller passes
in (the oracle in tests, the CUDA library in bench.py), so no input ever flows from
one implementation to the other's expected values.

The paper measures on simulated data, not on a public data set;
these inputs take the shapes of its analyses (1 or 3 detectors, A/E/T, 1 or 5 modes,
uniform rfft-like grid from 1e-4 Hz, Gaussian noise coloured by the analytic PSD,
injection + prior draws) and stand in for them.

RNG: numpy.random.default_rng(seed); draw order: parameter columns in theta order,
then (noise seed) per detector, per channel A, E, T: Re then Im.
"""
from __future__ import annotations

import ctypes
import ctypes.util
import dataclasses
import functools
import math
from typing import Callable, List, Optional, Sequence

import numpy as np

C_SI = 299792458.0
NPAR = 11
# theta order: M[Msun] q chi1 chi2 D_L[Gpc] iota phi_c lambda beta psi t_c[s]
PARAM_NAMES = ("M", "q", "chi1", "chi2", "D_L", "iota", "phi_c", "lambda", "beta", "psi", "t_c")

MODE_22, MODE_21, MODE_33, MODE_32, MODE_44 = 1, 2, 4, 8, 16
MODES_22_ONLY = MODE_22
MODES_HM = MODE_22 | MODE_21 | MODE_33 | MODE_32 | MODE_44


@functools.lru_cache(maxsize=16)
def _fma_grid_cached(f0: float, df: float, N: int) -> np.ndarray:
    if hasattr(math, "fma"):
        fma = math.fma
    else:
        libm = ctypes.CDLL(ctypes.util.find_library("m") or "libm.so.6")
        libm.fma.restype = ctypes.c_double
        libm.fma.argtypes = [ctypes.c_double] * 3
        fma = libm.fma
    out = np.fromiter((fma(float(k), df, f0) for k in range(N)), dtype=np.float64, count=N)
    out.setflags(write=False)
    return out


def _fma_grid(f0: float, df: float, N: int) -> np.ndarray:
    return _fma_grid_cached(float(f0), float(df), int(N)).copy()


@dataclasses.dataclass(frozen=True)
class Detector:
    """Plain description of one detector (mirrors the C struct field by field)."""
    name: str
    kind: int            # 0 heliocentric, 1 geocentric
    tdi_gen: int         # 15 or 20
    L_m: float
    kappa: float = 0.0
    lambda0: float = 0.0
    period_s: float = 0.0
    lon: float = 0.0
    lat: float = 0.0
    A_acc: float = 3e-15   # m/s^2/sqrt(Hz), noise recipe only (G13)
    A_oms: float = 15e-12  # m/sqrt(Hz)


@dataclasses.dataclass(frozen=True)
class Grid:
    f0: float
    df: float
    N: int

    def freqs(self) -> np.ndarray:
        # G11: f_k = fma(k, df, f0), one rounding (libm's fma; math.fma from Python 3.13 on).
        return _fma_grid(self.f0, self.df, self.N)


@dataclasses.dataclass(frozen=True)
class Model:
    mode_mask: int
    detectors: Sequence[Detector]


def lisa_like(tdi_gen: int = 20) -> Detector:
    return Detector("LISA-like", 0, tdi_gen, 2.5e9, kappa=math.radians(-20.0), A_acc=3e-15, A_oms=15e-12)


def taiji_like(tdi_gen: int = 20) -> Detector:
    return Detector("Taiji-like", 0, tdi_gen, 3.0e9, kappa=math.radians(+20.0), A_acc=3e-15, A_oms=8e-12)


def tianqin_like(tdi_gen: int = 20) -> Detector:
    return Detector("TianQin-like", 1, tdi_gen, math.sqrt(3.0) * 1e8, period_s=3.65 * 86400.0,
                    lon=math.radians(120.5), lat=math.radians(-4.7), A_acc=1e-15, A_oms=1e-12)


# ----------------------------------------------------------------------------- noise recipe (G13)
def psd_aet(det: Detector, f: np.ndarray) -> np.ndarray:
    """One-sided analytic S_A, S_E, S_T [3][N] in 1/Hz for the detector's TDI generation.

    Acceleration + OMS noise only.  Shape functions of SURVEY.md G13;
    pinned by P11 (propagation of six uncorrelated link noises through Eq. 6 / Eq. 3).
    """
    f = np.asarray(f, dtype=np.float64)
    x = 2.0 * np.pi * f * det.L_m / C_SI
    S_oms = (det.A_oms * 2.0 * np.pi * f / C_SI) ** 2 * (1.0 + (2e-3 / f) ** 4)
    S_acc = (det.A_acc / (2.0 * np.pi * f * C_SI)) ** 2 * (1.0 + (0.4e-3 / f) ** 2) * (1.0 + (f / 8e-3) ** 4)
    sx, cx = np.sin(x), np.cos(x)
    s_half2 = np.sin(0.5 * x) ** 2
    S_A = 8.0 * sx * sx * (2.0 * (3.0 + 2.0 * cx + np.cos(2.0 * x)) * S_acc + (2.0 + cx) * S_oms)
    S_T = 32.0 * sx * sx * s_half2 * (4.0 * s_half2 * S_acc + S_oms)
    out = np.stack([S_A, S_A.copy(), S_T])
    if det.tdi_gen == 20:
        out = out * (4.0 * np.sin(2.0 * x) ** 2)
    elif det.tdi_gen != 15:
        raise ValueError("tdi_gen must be 15 or 20")
    return out


def coloured_noise(psd: np.ndarray, df: float, rng: np.random.Generator) -> np.ndarray:
    """G12: Re and Im of n_c(f_k) iid N(0, S_c(f_k) T / 4), T = 1/df.  psd [...][N] -> complex [...][N]."""
    sigma = np.sqrt(psd / (4.0 * df))
    flat = sigma.reshape(-1, sigma.shape[-1])
    out = np.empty(flat.shape, dtype=np.complex128)
    for i in range(flat.shape[0]):          # per detector, per channel: Re then Im
        re = rng.standard_normal(flat.shape[1])
        im = rng.standard_normal(flat.shape[1])
        out[i] = (re + 1j * im) * flat[i]
    return out.reshape(sigma.shape)


# ----------------------------------------------------------------------------- parameter draws
THETA_INJ = np.array([2e6, 3.0, 0.0, 0.0, 10.0, 0.4, 1.3, 1.375, -1.2108, 2.659, 0.0])  # t_c set per grid


def draw_prior(B: int, T_obs: float, rng: np.random.Generator) -> np.ndarray:
    """Config 1 prior draws, columns in theta order."""
    th = np.zeros((B, NPAR))
    th[:, 0] = 10.0 ** rng.uniform(5.0, 7.0, B)
    th[:, 1] = rng.uniform(1.0, 8.0, B)
    th[:, 4] = rng.uniform(1.0, 20.0, B)
    th[:, 5] = np.arccos(rng.uniform(-1.0, 1.0, B))
    th[:, 6] = rng.uniform(0.0, 2.0 * np.pi, B)
    th[:, 7] = rng.uniform(0.0, 2.0 * np.pi, B)
    th[:, 8] = np.arcsin(rng.uniform(-1.0, 1.0, B))
    th[:, 9] = rng.uniform(0.0, np.pi, B)
    th[:, 10] = rng.uniform(0.0, T_obs, B)
    return th


def draw_jitter(B: int, theta_inj: np.ndarray, rng: np.random.Generator, rel: float = 0.01) -> np.ndarray:
    """Configs 2-5: theta_b = theta_inj * (1 + rel * g), g ~ N(0,1) iid (column by column); q clipped to >= 1."""
    th = np.empty((B, NPAR))
    for j in range(NPAR):
        th[:, j] = theta_inj[j] * (1.0 + rel * rng.standard_normal(B))
    th[:, 1] = np.maximum(th[:, 1], 1.0)
    return th


# ----------------------------------------------------------------------------- configs
@dataclasses.dataclass
class Workload:
    name: str
    grid: Grid
    model: Model
    params: np.ndarray              # [B][11]
    theta_inj: np.ndarray           # [11]
    noise_seed: Optional[int]       # None = noiseless
    want_fisher: bool = False

    @property
    def B(self) -> int:
        return self.params.shape[0]

    def psd(self) -> np.ndarray:
        """[n_det][3][N]"""
        f = self.grid.freqs()
        return np.stack([psd_aet(d, f) for d in self.model.detectors])

    def data(self, response_fn: Callable[[np.ndarray, np.ndarray, Model], np.ndarray]) -> np.ndarray:
        """Injection (+ noise) [n_det][3][N] complex128.

        response_fn(params[1][11], freqs[N], model) -> complex [1][n_det][3][N] is supplied
        by the caller: the oracle in tests, the CUDA library in bench.py.
        """
        f = self.grid.freqs()
        h = np.asarray(response_fn(self.theta_inj[None, :].copy(), f, self.model))[0]
        if self.noise_seed is None:
            return h.astype(np.complex128)
        rng = np.random.default_rng(self.noise_seed)
        return h + coloured_noise(self.psd(), self.grid.df, rng)


MONTH_DF = 1.0 / 2592000.0   # 1/(30 days)


def _jitter_workload(name, seed, noise_seed, B, N, mode_mask, dets, want_fisher=False) -> Workload:
    grid = Grid(1e-4, MONTH_DF, N)
    inj = THETA_INJ.copy()
    inj[10] = 2073600.0                # t_c = 0.8 T, T = 30 days
    rng = np.random.default_rng(seed)
    return Workload(name, grid, Model(mode_mask, tuple(dets)), draw_jitter(B, inj, rng), inj, noise_seed,
                    want_fisher)


CONFIG_SEEDS = {1: (0, None), 2: (1, 101), 3: (1, 101), 4: (3, 103), 5: (4, 104)}   # (params, noise)


def config(idx: int, B: Optional[int] = None, N: Optional[int] = None,
           param_seed: Optional[int] = None) -> Workload:
    """BASELINE.json configs 1-5.  B / N override the size (reduced parity cases keep f0, df
    and the draw recipe with B draws / the first N bins); param_seed overrides the seed of
    the parameter draws only (one batch per rank or per step in bench.py)."""
    if param_seed is not None and idx != 1:
        base = config(idx, B, N)
        rng = np.random.default_rng(param_seed)
        base.params = draw_jitter(base.B, base.theta_inj, rng)
        return base
    if idx == 1:
        n = 4096 if N is None else N
        grid_full_df = (1e-2 - 1e-4) / 4095
        grid = Grid(1e-4, grid_full_df, n)
        rng = np.random.default_rng(0)
        b = 16 if B is None else B
        th = draw_prior(b, 1.0 / grid_full_df, rng)
        return Workload("config1", grid, Model(MODES_22_ONLY, (lisa_like(),)), th, th[0].copy(), None)   # G15
    if idx == 2:
        return _jitter_workload("config2", 1, 101, B or 4096, N or 262144, MODES_22_ONLY, [lisa_like()])
    if idx == 3:
        return _jitter_workload("config3", 1, 101, B or 4096, N or 262144, MODES_HM, [lisa_like()])
    if idx == 4:
        return _jitter_workload("config4", 3, 103, B or 8192, N or 262144, MODES_HM,
                                [lisa_like(), taiji_like(), tianqin_like()])
    if idx == 5:
        return _jitter_workload("config5", 4, 104, B or 256, N or 262144, MODES_HM,
                                [lisa_like(), taiji_like(), tianqin_like()], want_fisher=True)
    raise ValueError("config index must be 1..5")


# ---------------------------------------------------------------- tabulated mode waveforms
# Input recipes for the *_tab entry points: tables (fnodes [K], amp, phase, tf [B][n_modes][K]) for the reference
# extrinsic values t_c = 0, phi_c = 0, D_L = 1 Gpc, modes in bit order of the mask.  Like the rest of this module
# they hold none of the method's arithmetic: `table_from_waveform_fn` tabulates whatever per-mode waveform function
# the caller passes in (the oracle's in the tests), `chirp_table` is a seeded-parameter synthetic input shaped like
# an inspiral (power laws in f), used where no waveform generator may be called (bench.py).
MODE_LM = ((2, 2), (2, 1), (3, 3), (3, 2), (4, 4))


def log_nodes(f_lo: float, f_hi: float, K: int) -> np.ndarray:
    """K log-spaced nodes covering [f_lo, f_hi] (end points widened by one part in 1e12)."""
    return np.geomspace(f_lo * (1.0 - 1e-12), f_hi * (1.0 + 1e-12), K)


def mask_modes(mode_mask: int):
    return [lm for i, lm in enumerate(MODE_LM) if mode_mask & (1 << i)]


def table_from_waveform_fn(params: np.ndarray, mode_mask: int, fnodes: np.ndarray,
                           waveform_fn: Callable[[np.ndarray, int, int, np.ndarray], tuple]):
    """waveform_fn(theta, l, m, freqs) -> (A, Psi, t_f); called with t_c = 0, phi_c = 0, D_L = 1 Gpc."""
    params = np.atleast_2d(params)
    modes = mask_modes(mode_mask)
    B, K = params.shape[0], fnodes.shape[0]
    amp, phase, tf = (np.empty((B, len(modes), K)) for _ in range(3))
    for b in range(B):
        th = params[b].copy()
        th[4], th[6], th[10] = 1.0, 0.0, 0.0
        for i, (l, m) in enumerate(modes):
            amp[b, i], phase[b, i], tf[b, i] = waveform_fn(th, l, m, fnodes)
    return fnodes, amp, phase, tf


def chirp_table(params: np.ndarray, mode_mask: int, fnodes: np.ndarray):
    """Synthetic smooth tables shaped like an inspiral: Psi = c0 (f')^(-5/3) (1 + c1 (f')^(2/3)) with f' = 2f/m,
    t_f = (1/2pi) dPsi/df exactly, A = a0 (f')^(-7/6) / m, the scales set by theta's M and q."""
    params = np.atleast_2d(params)
    modes = mask_modes(mode_mask)
    B, K = params.shape[0], fnodes.shape[0]
    amp, phase, tf = (np.empty((B, len(modes), K)) for _ in range(3))
    for b in range(B):
        Ms = params[b, 0] * 4.925490947641267e-6
        eta = params[b, 1] / (1.0 + params[b, 1]) ** 2
        c0 = 3.0 / (128.0 * eta) * (np.pi * Ms) ** (-5.0 / 3.0)
        c1 = (3715.0 / 756.0 + 55.0 * eta / 9.0) * (np.pi * Ms) ** (2.0 / 3.0)
        a0 = np.sqrt(2.0 * eta / 3.0) * np.pi ** (-1.0 / 6.0) * Ms ** (5.0 / 6.0) * Ms / 1.0292712505433901e17
        for i, (l, m) in enumerate(modes):
            fp = 2.0 * fnodes / m
            phase[b, i] = 0.5 * m * c0 * (fp ** (-5.0 / 3.0) + c1 / fp)
            dpsi_dfp = c0 * (-5.0 / 3.0 * fp ** (-8.0 / 3.0) - c1 / fp ** 2)      # d/df' of the (2,2)-like phase
            tf[b, i] = dpsi_dfp / (2.0 * np.pi)                                 # (m/2) (2/m) d/df' = d/df
            amp[b, i] = a0 * fp ** (-7.0 / 6.0) / m
    return fnodes, amp, phase, tf


# ---------------------------------------------------------------- tabulated numerical orbits
# Input recipes for the *_orb entry points: (t0, dt, pos [n_det][K][3][3] m, vel [n_det][K][3][3] m/s) on a uniform
# time grid.  `orbit_table_from_fn` samples whatever position function the caller passes in (the oracle's analytic
# orbit in the tests) and differentiates it numerically; `synthetic_orbit_table` is a seeded toy ephemeris shaped like
# a numerical orbit product (a cartwheeling triangle on a one-year circle plus small smooth perturbations), used where
# no orbit code may be called (bench.py).  Neither evaluates anything the method computes.
def orbit_table_from_fn(dets, t0: float, dt: float, K: int, orbit_fn: Callable[[Detector, float], np.ndarray],
                        h: float = 64.0):
    """orbit_fn(det, t) -> positions [3][3] in metres.  Velocities: five-point central differences with step h."""
    t = t0 + dt * np.arange(K)
    pos = np.empty((len(dets), K, 3, 3))
    vel = np.empty_like(pos)
    for d, det in enumerate(dets):
        for j, tj in enumerate(t):
            pos[d, j] = orbit_fn(det, tj)
            vel[d, j] = (-orbit_fn(det, tj + 2 * h) + 8.0 * orbit_fn(det, tj + h) - 8.0 * orbit_fn(det, tj - h)
                         + orbit_fn(det, tj - 2 * h)) / (12.0 * h)
    return float(t0), float(dt), pos, vel


def synthetic_orbit_table(dets, t0: float, dt: float, K: int, seed: int = 0, rel_pert: float = 2e-3):
    """Seeded toy ephemeris: per detector an equilateral triangle of side L_m whose centre moves on a circle of 1 au
    (one turn per 31558150 s, phase kappa; kind 1: on Earth's circle) and which turns in its own plane (heliocentric:
    once per orbit in a plane tilted by 60 degrees; geocentric: once per period_s in the plane normal to (lon, lat)),
    plus smooth perturbations of relative size rel_pert of the arm length (three harmonics per coordinate, seeded)
    standing in for the arm breathing of real numerical orbits.  Velocities are the exact time derivatives."""
    AU, YR = 149597870700.0, 31558149.763545603
    rng = np.random.default_rng(seed)
    t = t0 + dt * np.arange(K)
    pos = np.empty((len(dets), K, 3, 3))
    vel = np.empty_like(pos)
    for d, det in enumerate(dets):
        w0 = 2.0 * np.pi / YR
        a = w0 * t + (det.kappa if det.kind == 0 else 0.0)
        cen = AU * np.stack([np.cos(a), np.sin(a), np.zeros_like(a)], axis=-1)
        dcen = AU * w0 * np.stack([-np.sin(a), np.cos(a), np.zeros_like(a)], axis=-1)
        r = det.L_m / np.sqrt(3.0)
        if det.kind == 0:
            wr = w0
            e1 = np.stack([np.cos(a) * 0.5, np.sin(a) * 0.5, -np.sqrt(0.75) * np.ones_like(a)], axis=-1)   # tilted radial
            e2 = np.stack([-np.sin(a), np.cos(a), np.zeros_like(a)], axis=-1)
            de1 = w0 * np.stack([-np.sin(a) * 0.5, np.cos(a) * 0.5, np.zeros_like(a)], axis=-1)
            de2 = w0 * np.stack([-np.cos(a), -np.sin(a), np.zeros_like(a)], axis=-1)
        else:
            wr = 2.0 * np.pi / det.period_s
            n = np.array([np.cos(det.lat) * np.cos(det.lon), np.cos(det.lat) * np.sin(det.lon), np.sin(det.lat)])
            b1 = np.array([-np.sin(det.lon), np.cos(det.lon), 0.0])
            b2 = np.cross(n, b1)
            e1, e2 = np.tile(b1, (K, 1)), np.tile(b2, (K, 1))
            de1 = de2 = np.zeros((K, 3))
        for sc in range(3):
            ph = -wr * t + 2.0 * np.pi * sc / 3.0 + det.lambda0 if det.kind == 0 else wr * t + 2.0 * np.pi * sc / 3.0 + det.lambda0
            dph = -wr if det.kind == 0 else wr
            c, s_ = np.cos(ph)[:, None], np.sin(ph)[:, None]
            x = cen + r * (c * e1 + s_ * e2)
            v = dcen + r * (c * de1 + s_ * de2) + r * dph * (-s_ * e1 + c * e2)
            for ax in range(3):
                for _ in range(3):
                    amp = rel_pert * det.L_m * rng.uniform(-1.0, 1.0)
                    om = 2.0 * np.pi / (YR / rng.integers(1, 6))
                    p0 = rng.uniform(0.0, 2.0 * np.pi)
                    x[:, ax] += amp * np.sin(om * t + p0)
                    v[:, ax] += amp * om * np.cos(om * t + p0)
            pos[d, :, sc], vel[d, :, sc] = x, v
    return float(t0), float(dt), pos, vel
