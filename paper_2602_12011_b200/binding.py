"""Thin ctypes binding over libpespace.so (include/pespace.h).  Argument marshalling only:
every step of the hot path runs in the CUDA kernels.  There is NO CPU fallback -- if the
shared library is missing this module raises at import, and every compute call needs a
CUDA device.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Optional

import numpy as np
import torch

NPAR = 11
_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libpespace.so")

EXPORTS = ("pespace_response", "pespace_workspace_bytes", "pespace_loglike", "pespace_fisher",
           "pespace_loglike_mixed", "pespace_workspace_bytes_grad", "pespace_loglike_grad",
           "pespace_prepare", "pespace_loglike_prepared", "pespace_loglike_grad_prepared",
           "pespace_response_noalloc", "pespace_noalloc_scratch_needed",
           "pespace_session_loglike_grad", "pespace_response_orb", "pespace_loglike_orb",
           "pespace_workspace_bytes_fisher_tab", "pespace_fisher_tab", "pespace_response_tab", "pespace_workspace_bytes_tab", "pespace_loglike_tab",
           "pespace_session_create", "pespace_session_set_data", "pespace_session_loglike", "pespace_session_loglike_mixed",
           "pespace_session_fisher", "pespace_session_loglike_tab", "pespace_session_destroy",
           "pespace_loglike_host", "pespace_fp64_peak", "pespace_profile_enable", "pespace_profile_read",
           "pespace_launch_count", "pespace_strerror",
           "pespace_version")


class PespaceError(RuntimeError):
    pass


class _Det(C.Structure):
    _fields_ = [("kind", C.c_int32), ("tdi_gen", C.c_int32), ("L_m", C.c_double), ("kappa", C.c_double),
                ("lambda0", C.c_double), ("period_s", C.c_double), ("lon", C.c_double), ("lat", C.c_double)]


class _Grid(C.Structure):
    _fields_ = [("f0", C.c_double), ("df", C.c_double), ("N", C.c_int64)]


class _Model(C.Structure):
    _fields_ = [("mode_mask", C.c_uint32), ("n_det", C.c_int32), ("det", C.POINTER(_Det))]


class _OrbitTable(C.Structure):
    _fields_ = [("K", C.c_int64), ("t0", C.c_double), ("dt", C.c_double), ("d_pos", C.c_void_p), ("d_vel", C.c_void_p)]


class _WaveTable(C.Structure):
    _fields_ = [("K", C.c_int64), ("d_fnodes", C.c_void_p), ("d_amp", C.c_void_p), ("d_phase", C.c_void_p),
                ("d_tf", C.c_void_p)]


def _load():
    if not os.path.exists(LIB_PATH):
        # not built yet (a fresh checkout: the library is not under version control): compile it in-tree with nvcc.
        # There is no CPU fallback: if the build fails, importing this module fails.
        try:
            from . import build as _build
            _build.build()
        except Exception as exc:
            raise ImportError(f"{LIB_PATH} is missing and could not be built ({exc}); run "
                              "`python -m paper_2602_12011_b200.build` (there is no CPU fallback)") from exc
    L = C.CDLL(LIB_PATH)
    vp, i64, sz = C.c_void_p, C.c_int64, C.c_size_t
    L.pespace_response.argtypes = [vp, i64, vp, i64, C.POINTER(_Model), vp, vp]
    L.pespace_response_noalloc.argtypes = [vp, i64, vp, i64, C.POINTER(_Model), vp, vp]
    L.pespace_noalloc_scratch_needed.argtypes = [i64, C.POINTER(_Model)]
    L.pespace_noalloc_scratch_needed.restype = sz
    L.pespace_workspace_bytes.argtypes = [i64, C.POINTER(_Grid), C.POINTER(_Model), C.c_int]
    L.pespace_workspace_bytes.restype = sz
    L.pespace_loglike.argtypes = [vp, i64, vp, vp, C.POINTER(_Grid), C.POINTER(_Model), vp, vp, sz, vp]
    L.pespace_loglike_mixed.argtypes = [vp, i64, vp, vp, C.POINTER(_Grid), C.POINTER(_Model), vp, vp, sz, vp]
    L.pespace_fisher.argtypes = [vp, i64, vp, vp, C.POINTER(_Grid), C.POINTER(_Model), vp, vp, vp, sz, vp]
    L.pespace_workspace_bytes_grad.argtypes = [i64, C.POINTER(_Grid), C.POINTER(_Model)]
    L.pespace_workspace_bytes_grad.restype = sz
    L.pespace_loglike_grad.argtypes = [vp, i64, vp, vp, C.POINTER(_Grid), C.POINTER(_Model), vp, vp, vp, sz, vp]
    L.pespace_prepare.argtypes = [vp, vp, C.POINTER(_Grid), C.POINTER(_Model), vp, sz, vp]
    L.pespace_loglike_prepared.argtypes = [vp, i64, C.POINTER(_Grid), C.POINTER(_Model), vp, vp, sz, vp]
    L.pespace_loglike_grad_prepared.argtypes = [vp, i64, C.POINTER(_Grid), C.POINTER(_Model), vp, vp, vp, sz, vp]
    L.pespace_workspace_bytes_fisher_tab.argtypes = [i64, C.POINTER(_Grid), C.POINTER(_Model)]
    L.pespace_workspace_bytes_fisher_tab.restype = sz
    L.pespace_fisher_tab.argtypes = [vp, i64, C.POINTER(_WaveTable), vp, vp, C.POINTER(_Grid), C.POINTER(_Model), vp, vp,
                                     vp, sz, vp]
    L.pespace_response_orb.argtypes = [vp, i64, C.POINTER(_OrbitTable), vp, i64, C.POINTER(_Model), vp, vp]
    L.pespace_loglike_orb.argtypes = [vp, i64, C.POINTER(_OrbitTable), vp, vp, C.POINTER(_Grid), C.POINTER(_Model), vp,
                                      vp, sz, vp]
    L.pespace_loglike_host.argtypes = [vp, i64, vp, vp, C.POINTER(_Grid), C.POINTER(_Model), vp]
    L.pespace_response_tab.argtypes = [vp, i64, C.POINTER(_WaveTable), vp, i64, C.POINTER(_Model), vp, vp]
    L.pespace_workspace_bytes_tab.argtypes = [i64, C.POINTER(_Grid), C.POINTER(_Model)]
    L.pespace_workspace_bytes_tab.restype = sz
    L.pespace_loglike_tab.argtypes = [vp, i64, C.POINTER(_WaveTable), vp, vp, C.POINTER(_Grid), C.POINTER(_Model), vp,
                                      vp, sz, vp]
    L.pespace_session_create.argtypes = [C.POINTER(_Grid), C.POINTER(_Model), i64, C.c_int, C.POINTER(vp)]
    L.pespace_session_set_data.argtypes = [vp, vp, vp]
    L.pespace_session_loglike.argtypes = [vp, vp, i64, vp]
    L.pespace_session_loglike_mixed.argtypes = [vp, vp, i64, vp]
    L.pespace_session_fisher.argtypes = [vp, vp, i64, vp, vp]
    L.pespace_session_loglike_grad.argtypes = [vp, vp, i64, vp, vp]
    L.pespace_session_loglike_tab.argtypes = [vp, vp, i64, i64, vp, vp, vp, vp, vp]
    L.pespace_session_destroy.argtypes = [vp]
    L.pespace_fp64_peak.argtypes = [C.c_int, C.c_int, C.POINTER(C.c_double), C.POINTER(C.c_double)]
    L.pespace_profile_enable.argtypes = [C.c_int]
    L.pespace_profile_read.argtypes = [C.POINTER(C.c_double), C.POINTER(i64)]
    L.pespace_launch_count.restype = i64
    L.pespace_strerror.argtypes = [C.c_int]
    L.pespace_strerror.restype = C.c_char_p
    L.pespace_version.restype = C.c_char_p
    return L


_lib = _load()


def lib():
    return _lib


def _check(rc: int, what: str) -> None:
    if rc != 0:
        raise PespaceError(f"{what} failed: {_lib.pespace_strerror(rc).decode()} (code {rc})")


def _model(model):
    dets = (_Det * len(model.detectors))(*[
        _Det(int(d.kind), int(d.tdi_gen), float(d.L_m), float(d.kappa), float(d.lambda0),
             float(d.period_s), float(d.lon), float(d.lat)) for d in model.detectors])
    return _Model(int(model.mode_mask), len(model.detectors), dets), dets


def _grid(grid):
    return _Grid(float(grid.f0), float(grid.df), int(grid.N))


def _dev(t: torch.Tensor, name: str) -> torch.Tensor:
    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == torch.float64 and t.is_contiguous()):
        raise PespaceError(f"{name}: expected a contiguous float64 CUDA tensor")
    return t


def _stream_ptr() -> int:
    return torch.cuda.current_stream().cuda_stream


def version() -> str:
    return _lib.pespace_version().decode()


def launch_count() -> int:
    return int(_lib.pespace_launch_count())


def workspace_bytes(B: int, grid, model, want_fisher: bool = False) -> int:
    m, keep = _model(model)
    g = _grid(grid)
    return int(_lib.pespace_workspace_bytes(int(B), C.byref(g), C.byref(m), int(want_fisher)))


def response(params: torch.Tensor, freqs: torch.Tensor, model, out: Optional[torch.Tensor] = None) -> torch.Tensor:
    """params [B][11], freqs [N] (device, f64) -> complex128 [B][n_det][3][N] (device)."""
    p, f = _dev(params, "params"), _dev(freqs, "freqs")
    B, N, nd = p.shape[0], f.shape[0], len(model.detectors)
    if out is None:
        out = torch.empty((B, nd, 3, N, 2), dtype=torch.float64, device=p.device)
    m, keep = _model(model)
    _check(_lib.pespace_response(p.data_ptr(), B, f.data_ptr(), N, C.byref(m), _dev(out, "out").data_ptr(),
                                 _stream_ptr()), "pespace_response")
    return torch.view_as_complex(out)


NOALLOC_SCRATCH_BYTES = 1 << 20      # PESPACE_NOALLOC_SCRATCH_BYTES of include/pespace.h


def noalloc_scratch_needed(B: int, model) -> int:
    m, keep = _model(model)
    return int(_lib.pespace_noalloc_scratch_needed(int(B), C.byref(m)))


def response_noalloc(params: torch.Tensor, freqs: torch.Tensor, model, out: torch.Tensor) -> torch.Tensor:
    """pespace_response_noalloc: as `response`, scratch in the library's static device array (no allocation inside
    the call, so `out` [B][n_det][3][N][2] f64 is the caller's; batches beyond the array raise PespaceError)."""
    p, f = _dev(params, "params"), _dev(freqs, "freqs")
    B, N, nd = p.shape[0], f.shape[0], len(model.detectors)
    o = _dev(out, "out")
    if tuple(o.shape) != (B, nd, 3, N, 2):
        raise PespaceError("out must be [B][n_det][3][N][2]")
    m, keep = _model(model)
    _check(_lib.pespace_response_noalloc(p.data_ptr(), B, f.data_ptr(), N, C.byref(m), o.data_ptr(), _stream_ptr()),
           "pespace_response_noalloc")
    return torch.view_as_complex(o)


class Likelihood:
    """Data, PSD and workspace resident on the device; one call per batch of samples."""

    def __init__(self, data: torch.Tensor, psd: torch.Tensor, grid, model, max_batch: int):
        nd = len(model.detectors)
        d = torch.view_as_real(data) if data.is_complex() else data
        self.data = _dev(d.contiguous(), "data")
        self.psd = _dev(psd.contiguous(), "psd")
        if tuple(self.data.shape) != (nd, 3, grid.N, 2) or tuple(self.psd.shape) != (nd, 3, grid.N):
            raise PespaceError("data must be [n_det][3][N] complex and psd [n_det][3][N]")
        self.grid, self.model, self.max_batch = grid, model, int(max_batch)
        self._m, self._keep = _model(model)
        self._g = _grid(grid)
        self.ws_bytes = workspace_bytes(max_batch, grid, model)
        self.ws = torch.empty(self.ws_bytes, dtype=torch.uint8, device=self.data.device)
        self.prepared = False

    _has_prepared = True                     # pespace_loglike and pespace_loglike_grad have a *_prepared twin

    def prepare(self) -> "Likelihood":
        """pespace_prepare: fold data and PSD into the per-bin table of the workspace once; later calls skip step S0
        (pespace_loglike_prepared / pespace_loglike_grad_prepared) until a call of another kind rewrites the table."""
        if not self._has_prepared:
            raise PespaceError("this call has no prepared variant")
        _check(_lib.pespace_prepare(self.data.data_ptr(), self.psd.data_ptr(), C.byref(self._g), C.byref(self._m),
                                    self.ws.data_ptr(), self.ws_bytes, _stream_ptr()), "pespace_prepare")
        self.prepared = True
        return self

    def __call__(self, params: torch.Tensor, out: Optional[torch.Tensor] = None, mixed: bool = False) -> torch.Tensor:
        """mixed=True: pespace_loglike_mixed (FP64 phases, FP32 geometry; ~1e-6 relative accuracy)."""
        p = _dev(params, "params")
        B = p.shape[0]
        if B > self.max_batch:
            raise PespaceError("batch larger than the workspace was sized for")
        if out is None:
            out = torch.empty(B, dtype=torch.float64, device=p.device)
        if self.prepared and not mixed and type(self) is Likelihood:
            _check(_lib.pespace_loglike_prepared(p.data_ptr(), B, C.byref(self._g), C.byref(self._m),
                                                 _dev(out, "out").data_ptr(), self.ws.data_ptr(), self.ws_bytes,
                                                 _stream_ptr()), "pespace_loglike_prepared")
            return out
        self.prepared = False                # the mixed kernel keeps its own (whitened) table in the same place
        fn, name = (_lib.pespace_loglike_mixed, "pespace_loglike_mixed") if mixed else \
            (_lib.pespace_loglike, "pespace_loglike")
        _check(fn(p.data_ptr(), B, self.data.data_ptr(), self.psd.data_ptr(), C.byref(self._g), C.byref(self._m),
                  _dev(out, "out").data_ptr(), self.ws.data_ptr(), self.ws_bytes, _stream_ptr()), name)
        return out


def loglike(params: torch.Tensor, data: torch.Tensor, psd: torch.Tensor, grid, model) -> torch.Tensor:
    return Likelihood(data, psd, grid, model, params.shape[0])(params)


class WaveTable:
    """Tabulated mode waveforms on the device (pespace_wavetable): fnodes [K], amp / phase / tf [B][n_modes][K]
    for t_c = 0, phi_c = 0, D_L = 1 Gpc, modes in bit order of the model's mode_mask."""

    def __init__(self, fnodes: torch.Tensor, amp: torch.Tensor, phase: torch.Tensor, tf: torch.Tensor):
        self.fnodes, self.amp, self.phase, self.tf = (_dev(x, n) for x, n in
                                                      ((fnodes, "fnodes"), (amp, "amp"), (phase, "phase"), (tf, "tf")))
        K = self.fnodes.shape[0]
        if self.amp.dim() != 3 or self.amp.shape[2] != K or self.phase.shape != self.amp.shape or \
                self.tf.shape != self.amp.shape:
            raise PespaceError("amp, phase and tf must be [B][n_modes][K] with K = len(fnodes)")
        self.B, self.n_modes, self.K = int(self.amp.shape[0]), int(self.amp.shape[1]), int(K)
        self.c = _WaveTable(self.K, self.fnodes.data_ptr(), self.amp.data_ptr(), self.phase.data_ptr(),
                            self.tf.data_ptr())

    def check(self, B: int, model) -> None:
        if self.B != B or self.n_modes != bin(int(model.mode_mask)).count("1"):
            raise PespaceError("table shape does not match the batch size / the number of modes of the mask")


def response_tab(params: torch.Tensor, table: WaveTable, freqs: torch.Tensor, model,
                 out: Optional[torch.Tensor] = None) -> torch.Tensor:
    """Response from tabulated mode waveforms -> complex128 [B][n_det][3][N] (device)."""
    p, f = _dev(params, "params"), _dev(freqs, "freqs")
    B, N, nd = p.shape[0], f.shape[0], len(model.detectors)
    table.check(B, model)
    if out is None:
        out = torch.empty((B, nd, 3, N, 2), dtype=torch.float64, device=p.device)
    m, keep = _model(model)
    _check(_lib.pespace_response_tab(p.data_ptr(), B, C.byref(table.c), f.data_ptr(), N, C.byref(m),
                                     _dev(out, "out").data_ptr(), _stream_ptr()), "pespace_response_tab")
    return torch.view_as_complex(out)


class LikelihoodTab(Likelihood):
    """pespace_loglike_tab with data, PSD and workspace resident on the device."""
    _has_prepared = False

    def __init__(self, data: torch.Tensor, psd: torch.Tensor, grid, model, max_batch: int):
        super().__init__(data, psd, grid, model, max_batch)
        self.ws_bytes = int(_lib.pespace_workspace_bytes_tab(int(max_batch), C.byref(self._g), C.byref(self._m)))
        self.ws = torch.empty(self.ws_bytes, dtype=torch.uint8, device=self.data.device)

    def __call__(self, params: torch.Tensor, table: WaveTable, out: Optional[torch.Tensor] = None) -> torch.Tensor:
        p = _dev(params, "params")
        B = p.shape[0]
        if B > self.max_batch:
            raise PespaceError("batch larger than the workspace was sized for")
        table.check(B, self.model)
        if out is None:
            out = torch.empty(B, dtype=torch.float64, device=p.device)
        _check(_lib.pespace_loglike_tab(p.data_ptr(), B, C.byref(table.c), self.data.data_ptr(), self.psd.data_ptr(),
                                        C.byref(self._g), C.byref(self._m), _dev(out, "out").data_ptr(),
                                        self.ws.data_ptr(), self.ws_bytes, _stream_ptr()), "pespace_loglike_tab")
        return out


class Fisher:
    """Data (optional), PSD, workspace and outputs resident on the device; one pespace_fisher call per batch."""

    def __init__(self, data: Optional[torch.Tensor], psd: torch.Tensor, grid, model, max_batch: int):
        self.psd = _dev(psd.contiguous(), "psd")
        self.data = None
        if data is not None:
            d = torch.view_as_real(data) if data.is_complex() else data
            self.data = _dev(d.contiguous(), "data")
        self.grid, self.model, self.max_batch = grid, model, int(max_batch)
        self._m, self._keep = _model(model)
        self._g = _grid(grid)
        self.ws_bytes = workspace_bytes(max_batch, grid, model, True)
        self.ws = torch.empty(max(self.ws_bytes, 16), dtype=torch.uint8, device=self.psd.device)

    def __call__(self, params: torch.Tensor, out_F: Optional[torch.Tensor] = None,
                 out_grad: Optional[torch.Tensor] = None, grad_only: bool = False):
        """-> (F, grad); grad_only=True skips the Fisher matrix (returns (None, grad): d lnL / d theta alone)."""
        p = _dev(params, "params")
        B = p.shape[0]
        if B > self.max_batch:
            raise PespaceError("batch larger than the workspace was sized for")
        if grad_only:
            if self.data is None:
                raise PespaceError("the gradient needs the data set")
            if out_grad is None:
                out_grad = torch.empty((B, NPAR), dtype=torch.float64, device=p.device)
            _check(_lib.pespace_fisher(p.data_ptr(), B, self.data.data_ptr(), self.psd.data_ptr(), C.byref(self._g),
                                       C.byref(self._m), None, _dev(out_grad, "out_grad").data_ptr(),
                                       self.ws.data_ptr(), self.ws_bytes, _stream_ptr()), "pespace_fisher")
            return None, out_grad
        if out_F is None:
            out_F = torch.empty((B, NPAR, NPAR), dtype=torch.float64, device=p.device)
        if self.data is not None and out_grad is None:
            out_grad = torch.empty((B, NPAR), dtype=torch.float64, device=p.device)
        _check(_lib.pespace_fisher(p.data_ptr(), B, None if self.data is None else self.data.data_ptr(),
                                   self.psd.data_ptr(), C.byref(self._g), C.byref(self._m),
                                   _dev(out_F, "out_F").data_ptr(),
                                   None if self.data is None else _dev(out_grad, "out_grad").data_ptr(),
                                   self.ws.data_ptr(), self.ws_bytes, _stream_ptr()), "pespace_fisher")
        return out_F, (out_grad if self.data is not None else None)


class FisherTab(Fisher):
    """pespace_fisher_tab: Fisher matrix / gradient on tabulated mode waveforms (extrinsic parameters)."""

    def __init__(self, data: Optional[torch.Tensor], psd: torch.Tensor, grid, model, max_batch: int):
        super().__init__(data, psd, grid, model, max_batch)
        self.ws_bytes = int(_lib.pespace_workspace_bytes_fisher_tab(max_batch, C.byref(self._g), C.byref(self._m)))
        self.ws = torch.empty(max(self.ws_bytes, 16), dtype=torch.uint8, device=self.psd.device)

    def __call__(self, params: torch.Tensor, table: WaveTable, grad_only: bool = False):
        """-> (F or None, grad or None)"""
        p = _dev(params, "params")
        B = p.shape[0]
        if B > self.max_batch:
            raise PespaceError("batch larger than the workspace was sized for")
        table.check(B, self.model)
        if grad_only and self.data is None:
            raise PespaceError("the gradient needs the data set")
        F = None if grad_only else torch.empty((B, NPAR, NPAR), dtype=torch.float64, device=p.device)
        g = None if self.data is None else torch.empty((B, NPAR), dtype=torch.float64, device=p.device)
        _check(_lib.pespace_fisher_tab(p.data_ptr(), B, C.byref(table.c), None if self.data is None else self.data.data_ptr(),
                                       self.psd.data_ptr(), C.byref(self._g), C.byref(self._m),
                                       None if F is None else F.data_ptr(), None if g is None else g.data_ptr(),
                                       self.ws.data_ptr(), self.ws_bytes, _stream_ptr()), "pespace_fisher_tab")
        return F, g


def fisher_tab(params: torch.Tensor, table: WaveTable, data: Optional[torch.Tensor], psd: torch.Tensor, grid, model):
    """-> (F [B][11][11], grad [B][11] or None) on tabulated mode waveforms"""
    return FisherTab(data, psd, grid, model, params.shape[0])(params, table)


def fisher(params: torch.Tensor, data: Optional[torch.Tensor], psd: torch.Tensor, grid, model):
    """-> (F [B][11][11], grad [B][11] or None)."""
    return Fisher(data, psd, grid, model, params.shape[0])(params)


class OrbitTable:
    """Device-resident orbit tables: pos, vel [n_det][K][3][3] on the time grid t0 + j dt."""

    def __init__(self, t0: float, dt: float, pos: torch.Tensor, vel: torch.Tensor):
        self.t0, self.dt = float(t0), float(dt)
        self.pos, self.vel = _dev(pos.contiguous(), "pos"), _dev(vel.contiguous(), "vel")
        if self.pos.dim() != 4 or tuple(self.pos.shape[2:]) != (3, 3) or self.vel.shape != self.pos.shape:
            raise PespaceError("orbit tables must be [n_det][K][3][3]")
        self.K = int(self.pos.shape[1])
        self.c = _OrbitTable(self.K, self.t0, self.dt, self.pos.data_ptr(), self.vel.data_ptr())

    def check(self, model) -> None:
        if self.pos.shape[0] != len(model.detectors):
            raise PespaceError(f"orbit tables hold {self.pos.shape[0]} detector(s), the model {len(model.detectors)}")


def response_orb(params: torch.Tensor, orbit: OrbitTable, freqs: torch.Tensor, model,
                 out: Optional[torch.Tensor] = None) -> torch.Tensor:
    """complex128 [B][n_det][3][N] with the spacecraft positions from `orbit`"""
    p, f = _dev(params, "params"), _dev(freqs, "freqs")
    orbit.check(model)
    B, N, nd = p.shape[0], f.shape[0], len(model.detectors)
    if out is None:
        out = torch.empty((B, nd, 3, N, 2), dtype=torch.float64, device=p.device)
    m, keep = _model(model)
    _check(_lib.pespace_response_orb(p.data_ptr(), B, C.byref(orbit.c), f.data_ptr(), N, C.byref(m),
                                     _dev(out, "out").data_ptr(), _stream_ptr()), "pespace_response_orb")
    return torch.view_as_complex(out)


class LikelihoodOrb(Likelihood):
    """pespace_loglike_orb: likelihood with tabulated orbits; data, PSD and workspace resident."""
    _has_prepared = False

    def __call__(self, params: torch.Tensor, orbit: OrbitTable, out: Optional[torch.Tensor] = None) -> torch.Tensor:
        p = _dev(params, "params")
        orbit.check(self.model)
        B = p.shape[0]
        if B > self.max_batch:
            raise PespaceError("batch larger than the workspace was sized for")
        if out is None:
            out = torch.empty(B, dtype=torch.float64, device=p.device)
        _check(_lib.pespace_loglike_orb(p.data_ptr(), B, C.byref(orbit.c), self.data.data_ptr(), self.psd.data_ptr(),
                                        C.byref(self._g), C.byref(self._m), _dev(out, "out").data_ptr(),
                                        self.ws.data_ptr(), self.ws_bytes, _stream_ptr()), "pespace_loglike_orb")
        return out


class LikelihoodGrad(Likelihood):
    """pespace_loglike_grad: lnL and d lnL / d theta in one reverse-mode pass (data, PSD, workspace resident)."""

    def __init__(self, data: torch.Tensor, psd: torch.Tensor, grid, model, max_batch: int):
        super().__init__(data, psd, grid, model, max_batch)
        self.ws_bytes = int(_lib.pespace_workspace_bytes_grad(max_batch, C.byref(self._g), C.byref(self._m)))
        if self.ws_bytes == 0:
            raise PespaceError("pespace_workspace_bytes_grad rejected the arguments")
        self.ws = torch.empty(self.ws_bytes, dtype=torch.uint8, device=self.data.device)

    def __call__(self, params: torch.Tensor, out_lnL: Optional[torch.Tensor] = None,
                 out_grad: Optional[torch.Tensor] = None):
        """-> (lnL [B], grad [B][11])"""
        p = _dev(params, "params")
        B = p.shape[0]
        if B > self.max_batch:
            raise PespaceError("batch larger than the workspace was sized for")
        if out_lnL is None:
            out_lnL = torch.empty(B, dtype=torch.float64, device=p.device)
        if out_grad is None:
            out_grad = torch.empty((B, NPAR), dtype=torch.float64, device=p.device)
        if self.prepared:
            _check(_lib.pespace_loglike_grad_prepared(p.data_ptr(), B, C.byref(self._g), C.byref(self._m),
                                                      _dev(out_lnL, "out_lnL").data_ptr(),
                                                      _dev(out_grad, "out_grad").data_ptr(), self.ws.data_ptr(),
                                                      self.ws_bytes, _stream_ptr()), "pespace_loglike_grad_prepared")
            return out_lnL, out_grad
        _check(_lib.pespace_loglike_grad(p.data_ptr(), B, self.data.data_ptr(), self.psd.data_ptr(), C.byref(self._g),
                                         C.byref(self._m), _dev(out_lnL, "out_lnL").data_ptr(),
                                         _dev(out_grad, "out_grad").data_ptr(), self.ws.data_ptr(), self.ws_bytes,
                                         _stream_ptr()), "pespace_loglike_grad")
        return out_lnL, out_grad


def loglike_grad(params: torch.Tensor, data: torch.Tensor, psd: torch.Tensor, grid, model):
    """-> (lnL [B], d lnL / d theta [B][11]) by reverse mode"""
    return LikelihoodGrad(data, psd, grid, model, params.shape[0])(params)


def loglike_host(params: np.ndarray, data: np.ndarray, psd: np.ndarray, grid, model) -> np.ndarray:
    """End-to-end call on HOST numpy buffers: H2D copies, kernels and the D2H copy of lnL all
    happen inside the C call (pespace_loglike_host)."""
    p = np.ascontiguousarray(params, dtype=np.float64)
    d = np.ascontiguousarray(data, dtype=np.complex128)
    s = np.ascontiguousarray(psd, dtype=np.float64)
    out = np.empty(p.shape[0], dtype=np.float64)
    m, keep = _model(model)
    g = _grid(grid)
    _check(_lib.pespace_loglike_host(p.ctypes.data, p.shape[0], d.ctypes.data, s.ctypes.data, C.byref(g),
                                     C.byref(m), out.ctypes.data), "pespace_loglike_host")
    return out


def _host_ptr(a, dtype, name: str):
    """Address of a contiguous host buffer: numpy array or CPU torch tensor (pinned or pageable)."""
    if isinstance(a, torch.Tensor):
        want = torch.complex128 if dtype == np.complex128 else torch.float64
        if a.is_cuda or a.dtype != want or not a.is_contiguous():
            raise PespaceError(f"{name}: expected a contiguous host tensor of {want}")
        return a.data_ptr(), a
    b = np.ascontiguousarray(a, dtype=dtype)
    return b.ctypes.data, b


class Session:
    """Host-buffer API (pespace_session_*): data set, PSD and scratch stay on the device; a call copies
    theta in and lnL (or F, grad) out.  Inputs and outputs are numpy arrays or CPU torch tensors."""

    def __init__(self, grid, model, max_batch: int, want_fisher: bool = False):
        m, self._keep = _model(model)
        g = _grid(grid)
        h = C.c_void_p()
        _check(_lib.pespace_session_create(C.byref(g), C.byref(m), int(max_batch), int(want_fisher), C.byref(h)),
               "pespace_session_create")
        self._h, self.grid, self.model, self.max_batch = h, grid, model, int(max_batch)

    def set_data(self, data=None, psd=None) -> None:
        dp = sp = None
        if data is not None:
            dp, keep_d = _host_ptr(data, np.complex128, "data")
        if psd is not None:
            sp, keep_s = _host_ptr(psd, np.float64, "psd")
        _check(_lib.pespace_session_set_data(self._h, dp, sp), "pespace_session_set_data")

    def loglike(self, params, out=None, mixed: bool = False):
        pp, p = _host_ptr(params, np.float64, "params")
        if out is None:
            out = np.empty(p.shape[0], dtype=np.float64)
        op, o = _host_ptr(out, np.float64, "out")
        if mixed:
            _check(_lib.pespace_session_loglike_mixed(self._h, pp, int(p.shape[0]), op), "pespace_session_loglike_mixed")
        else:
            _check(_lib.pespace_session_loglike(self._h, pp, int(p.shape[0]), op), "pespace_session_loglike")
        return out

    def loglike_grad(self, params, out_lnL=None, out_grad=None):
        """-> (lnL [B], d lnL / d theta [B][11]) through pespace_loglike_grad (reverse mode)"""
        pp, p = _host_ptr(params, np.float64, "params")
        B = int(p.shape[0])
        if out_lnL is None:
            out_lnL = np.empty(B, dtype=np.float64)
        if out_grad is None:
            out_grad = np.empty((B, NPAR), dtype=np.float64)
        lp, keep_l = _host_ptr(out_lnL, np.float64, "out_lnL")
        gp, keep_g = _host_ptr(out_grad, np.float64, "out_grad")
        _check(_lib.pespace_session_loglike_grad(self._h, pp, B, lp, gp), "pespace_session_loglike_grad")
        return out_lnL, out_grad

    def loglike_tab(self, params, table, out=None):
        """table = (fnodes [K], amp, phase, tf [B][n_modes][K]) as host arrays / CPU tensors"""
        pp, p = _host_ptr(params, np.float64, "params")
        B = int(p.shape[0])
        (fp, fn), (ap, a), (hp, ph), (tp, tf) = (_host_ptr(x, np.float64, n) for x, n in
                                                 zip(table, ("fnodes", "amp", "phase", "tf")))
        K = int(fn.shape[0])
        nm = bin(int(self.model.mode_mask)).count("1")
        for x in (a, ph, tf):
            if tuple(x.shape) != (B, nm, K):
                raise PespaceError(f"table arrays must be [B={B}][n_modes={nm}][K={K}]")
        if out is None:
            out = np.empty(B, dtype=np.float64)
        op, o = _host_ptr(out, np.float64, "out")
        _check(_lib.pespace_session_loglike_tab(self._h, pp, B, K, fp, ap, hp, tp, op), "pespace_session_loglike_tab")
        return out

    def fisher(self, params, with_grad: bool = True, out_F=None, out_grad=None, grad_only: bool = False):
        pp, p = _host_ptr(params, np.float64, "params")
        B = int(p.shape[0])
        if with_grad and out_grad is None:
            out_grad = np.empty((B, NPAR), dtype=np.float64)
        if grad_only:
            gp, keep_g = _host_ptr(out_grad, np.float64, "out_grad")
            _check(_lib.pespace_session_fisher(self._h, pp, B, None, gp), "pespace_session_fisher")
            return None, out_grad
        if out_F is None:
            out_F = np.empty((B, NPAR, NPAR), dtype=np.float64)
        Fp, keep_F = _host_ptr(out_F, np.float64, "out_F")
        gp = None
        if with_grad:
            gp, keep_g = _host_ptr(out_grad, np.float64, "out_grad")
        _check(_lib.pespace_session_fisher(self._h, pp, B, Fp, gp), "pespace_session_fisher")
        return out_F, (out_grad if with_grad else None)

    def close(self) -> None:
        if self._h is not None and self._h.value:
            h, self._h = self._h, None
            _check(_lib.pespace_session_destroy(h), "pespace_session_destroy")

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def fp64_peak(iters: int = 4096, mode: int = 0):
    """-> (TFLOP/s, ms) of the DFMA micro-benchmark (mode 0: two register operands, the pipe peak;
    mode 1: three distinct register operands)."""
    t, ms = C.c_double(), C.c_double()
    _check(_lib.pespace_fp64_peak(int(mode), int(iters), C.byref(t), C.byref(ms)), "pespace_fp64_peak")
    return t.value, ms.value


def profile_enable(on: bool) -> None:
    _check(_lib.pespace_profile_enable(int(bool(on))), "pespace_profile_enable")


def profile_read():
    """-> (summed ms of the dominant kernel, number of its launches) since the last read."""
    ms, n = C.c_double(), C.c_int64()
    _check(_lib.pespace_profile_read(C.byref(ms), C.byref(n)), "pespace_profile_read")
    return ms.value, int(n.value)
