"""ctypes front-end of the CPU oracle (oracle/pespace_oracle.cpp).

TEST INFRASTRUCTURE, NOT PRODUCT CODE.  Only tests/, __graft_entry__.smoke() and
bench.py's cpu_baseline / --impl reference legs may import this package.  It does not
import the CUDA package's binding or kernels; the only thing it accepts from
`paper_2602_12011_b200` is the plain Detector/Model/Grid description objects of the
workload module (duck-typed: any object with the same attribute names works).
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

from . import build as _build

NPAR = 11


class _Det(C.Structure):
    _fields_ = [("kind", C.c_int32), ("tdi_gen", C.c_int32), ("L_m", C.c_double), ("kappa", C.c_double),
                ("lambda0", C.c_double), ("period_s", C.c_double), ("lon", C.c_double), ("lat", C.c_double)]


class _Grid(C.Structure):
    _fields_ = [("f0", C.c_double), ("df", C.c_double), ("N", C.c_int64)]


class _Model(C.Structure):
    _fields_ = [("mode_mask", C.c_uint32), ("n_det", C.c_int32), ("det", C.POINTER(_Det))]


_lib = None


def lib():
    global _lib
    if _lib is None:
        path = _build.build()
        L = C.CDLL(path)
        dp = C.POINTER(C.c_double)
        L.pespace_oracle_response.argtypes = [dp, C.c_int64, dp, C.c_int64, C.POINTER(_Model), dp]
        L.pespace_oracle_response_quad.argtypes = L.pespace_oracle_response.argtypes
        L.pespace_oracle_loglike.argtypes = [dp, C.c_int64, dp, dp, C.POINTER(_Grid), C.POINTER(_Model), dp]
        L.pespace_oracle_fisher.argtypes = [dp, C.c_int64, dp, dp, C.POINTER(_Grid), C.POINTER(_Model), dp, dp]
        L.pespace_oracle_waveform.argtypes = [dp, C.c_int, C.c_int, dp, C.c_int64, dp, dp, dp]
        L.pespace_oracle_swsh.argtypes = [C.c_int, C.c_int, C.c_double, dp]
        L.pespace_oracle_orbit.argtypes = [C.POINTER(_Det), C.c_double, dp]
        L.pespace_oracle_links.argtypes = [dp, C.c_int, C.c_int, C.c_double, C.POINTER(_Det), dp]
        L.pespace_oracle_tdi.argtypes = [dp, C.c_double, C.c_double, C.c_int, dp]
        i64 = C.c_int64
        L.pespace_oracle_response_tab.argtypes = [dp, i64, i64, dp, dp, dp, dp, dp, i64, C.POINTER(_Model), dp]
        L.pespace_oracle_loglike_tab.argtypes = [dp, i64, i64, dp, dp, dp, dp, dp, dp, C.POINTER(_Grid),
                                                 C.POINTER(_Model), dp]
        L.pespace_oracle_fisher_tab.argtypes = [dp, i64, i64, dp, dp, dp, dp, dp, dp, C.POINTER(_Grid),
                                                C.POINTER(_Model), dp, dp]
        L.pespace_oracle_tab_waveform.argtypes = [i64, dp, dp, dp, dp, dp, i64, dp, dp, dp]
        dbl = C.c_double
        L.pespace_oracle_response_orb.argtypes = [dp, i64, i64, dbl, dbl, dp, dp, dp, i64, C.POINTER(_Model), dp]
        L.pespace_oracle_loglike_orb.argtypes = [dp, i64, i64, dbl, dbl, dp, dp, dp, dp, C.POINTER(_Grid),
                                                 C.POINTER(_Model), dp]
        L.pespace_oracle_orbit_tab.argtypes = [i64, dbl, dbl, dp, dp, dbl, dp]
        L.pespace_oracle_set_threads.argtypes = [C.c_int]
        L.pespace_oracle_set_threads.restype = None
        _lib = L
    return _lib


def _dp(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def _det(d) -> _Det:
    return _Det(int(d.kind), int(d.tdi_gen), float(d.L_m), float(d.kappa), float(d.lambda0),
                float(d.period_s), float(d.lon), float(d.lat))


def _model(model):
    dets = (_Det * len(model.detectors))(*[_det(d) for d in model.detectors])
    return _Model(int(model.mode_mask), len(model.detectors), dets), dets  # keep `dets` alive


def _check(rc, what):
    if rc != 0:
        raise ValueError(f"{what}: oracle rejected the arguments (rc={rc})")


def set_threads(n: int) -> None:
    lib().pespace_oracle_set_threads(int(n))


def get_threads() -> int:
    return int(lib().pespace_oracle_get_threads())


def response(params, freqs, model, quad: bool = False) -> np.ndarray:
    """complex128 [B][n_det][3][N]"""
    p, f = _f64(np.atleast_2d(params)), _f64(freqs)
    m, keep = _model(model)
    B, N, nd = p.shape[0], f.shape[0], len(model.detectors)
    out = np.empty((B, nd, 3, N, 2), dtype=np.float64)
    fn = lib().pespace_oracle_response_quad if quad else lib().pespace_oracle_response
    _check(fn(_dp(p), B, _dp(f), N, C.byref(m), _dp(out)), "response")
    return out.view(np.complex128)[..., 0]


def loglike(params, data, psd, grid, model) -> np.ndarray:
    """data complex [n_det][3][N], psd [n_det][3][N] -> lnL [B]"""
    p = _f64(np.atleast_2d(params))
    d = np.ascontiguousarray(data, dtype=np.complex128).view(np.float64)
    s = _f64(psd)
    m, keep = _model(model)
    g = _Grid(float(grid.f0), float(grid.df), int(grid.N))
    out = np.empty(p.shape[0], dtype=np.float64)
    _check(lib().pespace_oracle_loglike(_dp(p), p.shape[0], _dp(d), _dp(s), C.byref(g), C.byref(m), _dp(out)),
           "loglike")
    return out


def fisher(params, data, psd, grid, model):
    """-> (F [B][11][11], grad [B][11] or None when data is None)"""
    p = _f64(np.atleast_2d(params))
    s = _f64(psd)
    m, keep = _model(model)
    g = _Grid(float(grid.f0), float(grid.df), int(grid.N))
    B = p.shape[0]
    F = np.empty((B, NPAR, NPAR), dtype=np.float64)
    if data is None:
        _check(lib().pespace_oracle_fisher(_dp(p), B, None, _dp(s), C.byref(g), C.byref(m), _dp(F), None), "fisher")
        return F, None
    d = np.ascontiguousarray(data, dtype=np.complex128).view(np.float64)
    grad = np.empty((B, NPAR), dtype=np.float64)
    _check(lib().pespace_oracle_fisher(_dp(p), B, _dp(d), _dp(s), C.byref(g), C.byref(m), _dp(F), _dp(grad)),
           "fisher")
    return F, grad


def _table(table, B, model):
    """table = (fnodes [K], amp, phase, tf each [B][n_modes][K]) -> contiguous float64 arrays, K"""
    fn, a, ph, tf = (_f64(x) for x in table)
    nm = bin(int(model.mode_mask)).count("1")
    K = fn.shape[0]
    for x in (a, ph, tf):
        if x.shape != (B, nm, K):
            raise ValueError(f"table arrays must be [B={B}][n_modes={nm}][K={K}], got {x.shape}")
    return fn, a, ph, tf, K


def response_tab(params, table, freqs, model) -> np.ndarray:
    """T1: response from tabulated mode waveforms; complex128 [B][n_det][3][N]"""
    p, f = _f64(np.atleast_2d(params)), _f64(freqs)
    m, keep = _model(model)
    B, N, nd = p.shape[0], f.shape[0], len(model.detectors)
    fn, a, ph, tf, K = _table(table, B, model)
    out = np.empty((B, nd, 3, N, 2), dtype=np.float64)
    _check(lib().pespace_oracle_response_tab(_dp(p), B, K, _dp(fn), _dp(a), _dp(ph), _dp(tf), _dp(f), N, C.byref(m),
                                             _dp(out)), "response_tab")
    return out.view(np.complex128)[..., 0]


def loglike_tab(params, table, data, psd, grid, model) -> np.ndarray:
    """T1: lnL [B] from tabulated mode waveforms"""
    p = _f64(np.atleast_2d(params))
    d = np.ascontiguousarray(data, dtype=np.complex128).view(np.float64)
    s = _f64(psd)
    m, keep = _model(model)
    g = _Grid(float(grid.f0), float(grid.df), int(grid.N))
    B = p.shape[0]
    fn, a, ph, tf, K = _table(table, B, model)
    out = np.empty(B, dtype=np.float64)
    _check(lib().pespace_oracle_loglike_tab(_dp(p), B, K, _dp(fn), _dp(a), _dp(ph), _dp(tf), _dp(d), _dp(s), C.byref(g),
                                            C.byref(m), _dp(out)), "loglike_tab")
    return out


def fisher_tab(params, table, data, psd, grid, model):
    """T1 x O12: -> (F [B][11][11], grad [B][11] or None when data is None); rows / columns 0-3 are 0"""
    p = _f64(np.atleast_2d(params))
    s = _f64(psd)
    m, keep = _model(model)
    g = _Grid(float(grid.f0), float(grid.df), int(grid.N))
    B = p.shape[0]
    fn, a, ph, tf, K = _table(table, B, model)
    F = np.empty((B, NPAR, NPAR), dtype=np.float64)
    d = None if data is None else np.ascontiguousarray(data, dtype=np.complex128).view(np.float64)
    grad = None if data is None else np.empty((B, NPAR), dtype=np.float64)
    _check(lib().pespace_oracle_fisher_tab(_dp(p), B, K, _dp(fn), _dp(a), _dp(ph), _dp(tf), None if d is None else _dp(d),
                                           _dp(s), C.byref(g), C.byref(m), _dp(F), None if grad is None else _dp(grad)),
           "fisher_tab")
    return F, grad


def tab_waveform(fnodes, amp, phase, tf, freqs):
    """T1: the interpolants of one (sample, mode) table at freqs -> (A, Psi, t_f); NaN outside the table"""
    fn, a, ph, t, f = (_f64(x) for x in (fnodes, amp, phase, tf, freqs))
    oa, op, ot = (np.empty_like(f) for _ in range(3))
    _check(lib().pespace_oracle_tab_waveform(fn.shape[0], _dp(fn), _dp(a), _dp(ph), _dp(t), _dp(f), f.shape[0], _dp(oa),
                                             _dp(op), _dp(ot)), "tab_waveform")
    return oa, op, ot


def _orbit(orbit, nd):
    """orbit = (t0, dt, pos [n_det][K][3][3], vel [n_det][K][3][3]) -> (t0, dt, pos, vel, K)"""
    t0, dt, pos, vel = orbit
    pos, vel = _f64(pos), _f64(vel)
    if pos.ndim != 4 or pos.shape[0] != nd or pos.shape[2:] != (3, 3) or vel.shape != pos.shape:
        raise ValueError(f"orbit tables must be [n_det={nd}][K][3][3], got {pos.shape} and {vel.shape}")
    return float(t0), float(dt), pos, vel, pos.shape[1]


def response_orb(params, orbit, freqs, model) -> np.ndarray:
    """T2: response with tabulated orbits; complex128 [B][n_det][3][N]"""
    p, f = _f64(np.atleast_2d(params)), _f64(freqs)
    m, keep = _model(model)
    B, N, nd = p.shape[0], f.shape[0], len(model.detectors)
    t0, dt, pos, vel, K = _orbit(orbit, nd)
    out = np.empty((B, nd, 3, N, 2), dtype=np.float64)
    _check(lib().pespace_oracle_response_orb(_dp(p), B, K, t0, dt, _dp(pos), _dp(vel), _dp(f), N, C.byref(m), _dp(out)),
           "response_orb")
    return out.view(np.complex128)[..., 0]


def loglike_orb(params, orbit, data, psd, grid, model) -> np.ndarray:
    """T2: lnL [B] with tabulated orbits"""
    p = _f64(np.atleast_2d(params))
    d = np.ascontiguousarray(data, dtype=np.complex128).view(np.float64)
    s = _f64(psd)
    m, keep = _model(model)
    g = _Grid(float(grid.f0), float(grid.df), int(grid.N))
    t0, dt, pos, vel, K = _orbit(orbit, len(model.detectors))
    out = np.empty(p.shape[0], dtype=np.float64)
    _check(lib().pespace_oracle_loglike_orb(_dp(p), p.shape[0], K, t0, dt, _dp(pos), _dp(vel), _dp(d), _dp(s),
                                            C.byref(g), C.byref(m), _dp(out)), "loglike_orb")
    return out


def orbit_tab(t0, dt, pos, vel, t):
    """T2: interpolated positions [3][3] of one detector's table (pos, vel [K][3][3]) at t; None outside the table"""
    pos, vel = _f64(pos), _f64(vel)
    out = np.empty((3, 3), dtype=np.float64)
    rc = lib().pespace_oracle_orbit_tab(pos.shape[0], float(t0), float(dt), _dp(pos), _dp(vel), float(t), _dp(out))
    if rc == 1:
        return None
    _check(rc, "orbit_tab")
    return out


def waveform(theta, l, m, freqs):
    """-> (A_lm [s], Psi_lm [rad], t_lm [s]) on freqs"""
    th, f = _f64(theta), _f64(freqs)
    a, p, t = (np.empty_like(f) for _ in range(3))
    _check(lib().pespace_oracle_waveform(_dp(th), l, m, _dp(f), f.shape[0], _dp(a), _dp(p), _dp(t)), "waveform")
    return a, p, t


def swsh(l, m, iota) -> float:
    out = C.c_double()
    _check(lib().pespace_oracle_swsh(l, m, float(iota), C.byref(out)), "swsh")
    return out.value


def orbit(det, t) -> np.ndarray:
    """spacecraft positions [3][3] in metres"""
    out = np.empty((3, 3), dtype=np.float64)
    d = _det(det)
    _check(lib().pespace_oracle_orbit(C.byref(d), float(t), _dp(out)), "orbit")
    return out


LINK_ORDER = ((1, 2), (2, 1), (1, 3), (3, 1), (2, 3), (3, 2))   # (receiver, sender)


def links(theta, l, m, f, det) -> np.ndarray:
    """six single-link responses of one mode, complex [6] in LINK_ORDER"""
    th = _f64(theta)
    out = np.empty((6, 2), dtype=np.float64)
    d = _det(det)
    _check(lib().pespace_oracle_links(_dp(th), l, m, float(f), C.byref(d), _dp(out)), "links")
    return out.view(np.complex128)[:, 0]


def tdi(y, f, L_m, tdi_gen) -> np.ndarray:
    """X, Y, Z complex [3] from six links in LINK_ORDER"""
    yy = np.ascontiguousarray(y, dtype=np.complex128).view(np.float64)
    out = np.empty((3, 2), dtype=np.float64)
    _check(lib().pespace_oracle_tdi(_dp(yy), float(f), float(L_m), int(tdi_gen), _dp(out)), "tdi")
    return out.view(np.complex128)[:, 0]
