"""Host-side checks that need no GPU: the C-ABI library builds, loads and exports every symbol
include/pespace.h declares; argument validation returns the documented codes before any CUDA
call; the workload recipes are reproducible."""
import ctypes as C
import glob
import os
import re

import numpy as np
import pytest

from paper_2602_12011_b200 import build as pbuild
from paper_2602_12011_b200 import workloads as W

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    return C.CDLL(pbuild.build())


def declared_symbols():
    names = set()
    for hdr in sorted(glob.glob(os.path.join(ROOT, "include", "*.h"))):
        text = re.sub(r"/\*.*?\*/", "", open(hdr).read(), flags=re.S)
        names |= set(re.findall(r"\b(pespace_[a-z0-9_]+)\s*\(", text))
    return sorted(names)


def test_library_exports_every_declared_symbol(lib):
    names = declared_symbols()
    assert {"pespace_response", "pespace_loglike", "pespace_fisher", "pespace_workspace_bytes",
            "pespace_strerror"} <= set(names)
    for n in names:
        assert hasattr(lib, n), n


def test_binding_mirrors_the_header():
    from paper_2602_12011_b200 import binding
    assert sorted(binding.EXPORTS) == declared_symbols()
    assert "sm_100a" in binding.version()


def test_argument_validation_without_a_device():
    from paper_2602_12011_b200 import binding as P
    L = P.lib()
    wl = W.config(2, B=4, N=64)
    m, keep = P._model(wl.model)
    g = P._grid(wl.grid)
    EINVAL = -1
    fake = 0x1000  # never dereferenced: validation fails first
    assert L.pespace_loglike(None, 4, fake, fake, C.byref(g), C.byref(m), fake, fake, 1 << 30, None) == EINVAL
    assert L.pespace_loglike(fake, 0, fake, fake, C.byref(g), C.byref(m), fake, fake, 1 << 30, None) == EINVAL
    assert L.pespace_loglike(fake, 4, fake, fake, C.byref(g), C.byref(m), fake, fake, 8, None) == EINVAL  # ws too small
    bad_g = P._Grid(1e-4, -1.0, 64)
    assert L.pespace_loglike(fake, 4, fake, fake, C.byref(bad_g), C.byref(m), fake, fake, 1 << 30, None) == EINVAL
    bad_m, keep2 = P._model(W.Model(0, wl.model.detectors))
    assert L.pespace_response(fake, 4, fake, 64, C.byref(bad_m), fake, None) == EINVAL
    bad_m2, keep3 = P._model(W.Model(1, (W.Detector("x", 7, 20, 1e9),)))
    assert L.pespace_response(fake, 4, fake, 64, C.byref(bad_m2), fake, None) == EINVAL
    bad_m3, keep4 = P._model(W.Model(1, (W.Detector("x", 0, 17, 1e9),)))
    assert L.pespace_fisher(fake, 4, None, fake, C.byref(g), C.byref(bad_m3), fake, None, fake, 1 << 30, None) == EINVAL
    assert L.pespace_loglike_host(None, 4, fake, fake, C.byref(g), C.byref(m), fake) == EINVAL
    # prepared-data entry points: the same checks, before any CUDA call
    assert L.pespace_prepare(None, fake, C.byref(g), C.byref(m), fake, 1 << 30, None) == EINVAL
    assert L.pespace_prepare(fake, fake, C.byref(g), C.byref(m), fake, 8, None) == EINVAL                 # ws too small
    assert L.pespace_prepare(fake, fake, C.byref(g), C.byref(m), 0x1008, 1 << 30, None) == EINVAL          # alignment
    assert L.pespace_prepare(fake, fake, C.byref(bad_g), C.byref(m), fake, 1 << 30, None) == EINVAL
    assert L.pespace_loglike_prepared(None, 4, C.byref(g), C.byref(m), fake, fake, 1 << 30, None) == EINVAL
    assert L.pespace_loglike_prepared(fake, 0, C.byref(g), C.byref(m), fake, fake, 1 << 30, None) == EINVAL
    assert L.pespace_loglike_prepared(fake, 4, C.byref(g), C.byref(m), fake, fake, 8, None) == EINVAL
    assert L.pespace_loglike_grad_prepared(fake, 4, C.byref(g), C.byref(m), None, None, fake, 1 << 30, None) == EINVAL
    assert L.pespace_loglike_grad_prepared(fake, 4, C.byref(g), C.byref(m), fake, fake, fake, 8, None) == EINVAL
    assert L.pespace_fp64_peak(0, 0, None, None) == EINVAL
    assert L.pespace_workspace_bytes(0, C.byref(g), C.byref(m), 0) == 0
    assert L.pespace_workspace_bytes(4096, C.byref(g), C.byref(m), 0) > 4096 * 8
    assert L.pespace_strerror(EINVAL) == b"invalid argument"
    assert L.pespace_strerror(0) == b"ok"


def test_workloads_are_seeded_and_shaped_like_the_configs():
    a, b = W.config(2, B=64, N=128), W.config(2, B=64, N=128)
    assert np.array_equal(a.params, b.params)
    assert a.params[:, 1].min() >= 1.0 and np.all(a.params[:, 2:4] == 0.0)
    assert np.allclose(a.params.mean(axis=0)[[0, 4]], [2e6, 10.0], rtol=0.01)
    full = W.config(2)
    assert (full.B, full.grid.N, full.grid.f0) == (4096, 262144, 1e-4)
    assert full.grid.df == 1.0 / (30 * 86400) and full.theta_inj[10] == 2073600.0
    c4 = W.config(4)
    assert c4.B == 8192 and [d.kind for d in c4.model.detectors] == [0, 0, 1] and c4.model.mode_mask == 31
    c1 = W.config(1)
    assert c1.B == 16 and c1.grid.N == 4096 and c1.noise_seed is None
    f = c1.grid.freqs()
    assert f[0] == 1e-4 and abs(f[-1] - 1e-2) < 1e-15
    # G12: noise variance
    psd = np.full((1, 3, 20000), 2.5e-40)
    n = W.coloured_noise(psd, 1e-6, np.random.default_rng(0))
    assert np.var(n.real) == pytest.approx(2.5e-40 / 4e-6, rel=0.03)
    # psd nulls of TDI 2.0 sit where sin(2x) = 0
    det = W.lisa_like()
    fn = 299792458.0 / (4 * det.L_m)
    assert W.psd_aet(det, np.array([fn]))[0, 0] < 1e-25 * W.psd_aet(det, np.array([fn * 0.9]))[0, 0]


def test_session_argument_validation_without_a_device():
    """pespace_session_* reject bad arguments before any CUDA call (include/pespace.h, host-buffer entry points)."""
    from paper_2602_12011_b200 import binding as P
    L = P.lib()
    wl = W.config(2, B=4, N=64)
    m, keep = P._model(wl.model)
    g = P._grid(wl.grid)
    EINVAL = -1
    h = C.c_void_p(0x1234)
    assert L.pespace_session_create(C.byref(g), C.byref(m), 0, 0, C.byref(h)) == EINVAL
    assert not h.value                                            # *out is NULL on failure
    bad_g = P._Grid(1e-4, 0.0, 64)
    assert L.pespace_session_create(C.byref(bad_g), C.byref(m), 4, 0, C.byref(h)) == EINVAL
    bad_m, keep2 = P._model(W.Model(64, wl.model.detectors))
    assert L.pespace_session_create(C.byref(g), C.byref(bad_m), 4, 1, C.byref(h)) == EINVAL
    assert L.pespace_session_create(C.byref(g), C.byref(m), 4, 0, None) == EINVAL
    assert L.pespace_session_set_data(None, None, None) == EINVAL
    assert L.pespace_session_loglike(None, None, 4, None) == EINVAL
    assert L.pespace_session_loglike_mixed(None, None, 4, None) == EINVAL
    assert L.pespace_session_fisher(None, None, 4, None, None) == EINVAL
    assert L.pespace_session_loglike_tab(None, None, 4, 8, None, None, None, None, None) == EINVAL
    assert L.pespace_session_destroy(None) == EINVAL
    assert L.pespace_loglike_host(None, 4, None, None, C.byref(g), C.byref(m), None) == EINVAL


def test_tab_argument_validation_without_a_device():
    """pespace_*_tab reject bad arguments before any CUDA call (include/pespace.h, tabulated mode waveforms)."""
    from paper_2602_12011_b200 import binding as P
    L = P.lib()
    wl = W.config(2, B=4, N=64)
    m, keep = P._model(wl.model)
    g = P._grid(wl.grid)
    EINVAL = -1
    fake = 0x1000
    good = P._WaveTable(16, fake, fake, fake, fake)
    assert L.pespace_response_tab(fake, 4, None, fake, 64, C.byref(m), fake, None) == EINVAL
    assert L.pespace_response_tab(fake, 4, C.byref(P._WaveTable(3, fake, fake, fake, fake)), fake, 64, C.byref(m), fake,
                                  None) == EINVAL                               # K < 4
    assert L.pespace_response_tab(fake, 4, C.byref(P._WaveTable(16, fake, None, fake, fake)), fake, 64, C.byref(m), fake,
                                  None) == EINVAL                               # missing table array
    assert L.pespace_response_tab(None, 4, C.byref(good), fake, 64, C.byref(m), fake, None) == EINVAL
    assert L.pespace_loglike_tab(fake, 4, C.byref(good), fake, fake, C.byref(g), C.byref(m), fake, fake, 8, None) == EINVAL
    assert L.pespace_loglike_tab(fake, 0, C.byref(good), fake, fake, C.byref(g), C.byref(m), fake, fake, 1 << 30,
                                 None) == EINVAL
    assert L.pespace_workspace_bytes_tab(0, C.byref(g), C.byref(m)) == 0
    ws_tab, ws = L.pespace_workspace_bytes_tab(4, C.byref(g), C.byref(m)), L.pespace_workspace_bytes(4, C.byref(g), C.byref(m), 0)
    assert ws_tab > ws > 0


def test_header_is_plain_c():
    """include/pespace.h is a C ABI: it must compile as C99 and as C++ with no other header of this repository."""
    import subprocess
    for hdr in sorted(glob.glob(os.path.join(ROOT, "include", "*.h"))):
        for cmd in (["gcc", "-x", "c", "-std=c99", "-Wall", "-Werror", "-fsyntax-only", hdr],
                    ["g++", "-x", "c++", "-Wall", "-Werror", "-fsyntax-only", hdr]):
            res = subprocess.run(cmd, capture_output=True, text=True)
            assert res.returncode == 0, res.stderr


def test_product_header_holds_no_bench_scaffolding():
    """pespace.h is the boundary; the micro-benchmark, the kernel timer and the launch counter live in
    pespace_bench.h."""
    text = open(os.path.join(ROOT, "include", "pespace.h")).read()
    for name in ("pespace_fp64_peak", "pespace_profile_enable", "pespace_profile_read", "pespace_launch_count"):
        assert name not in text


def test_grad_argument_validation_without_a_device():
    from paper_2602_12011_b200 import binding as P
    L = P.lib()
    wl = W.config(3, B=4, N=64)
    m, keep = P._model(wl.model)
    g = P._grid(wl.grid)
    fake = 0x1000
    assert L.pespace_workspace_bytes_grad(0, C.byref(g), C.byref(m)) == 0
    need = L.pespace_workspace_bytes_grad(4, C.byref(g), C.byref(m))
    assert need > L.pespace_workspace_bytes(4, C.byref(g), C.byref(m), 0)
    assert L.pespace_loglike_grad(fake, 4, fake, fake, C.byref(g), C.byref(m), None, None, fake, need, None) == -1
    assert L.pespace_loglike_grad(fake, 4, fake, fake, C.byref(g), C.byref(m), fake, fake, fake, need - 1, None) == -1
    assert L.pespace_loglike_grad(fake, 4, None, fake, C.byref(g), C.byref(m), fake, fake, fake, need, None) == -1
    assert L.pespace_session_loglike_grad(None, None, 4, None, None) == -1


def test_orb_argument_validation_without_a_device():
    from paper_2602_12011_b200 import binding as P
    L = P.lib()
    wl = W.config(3, B=4, N=64)
    m, keep = P._model(wl.model)
    g = P._grid(wl.grid)
    fake = 0x1000
    good = P._OrbitTable(16, 0.0, 100.0, fake, fake)
    assert L.pespace_response_orb(fake, 4, None, fake, 64, C.byref(m), fake, None) == -1
    assert L.pespace_response_orb(fake, 4, C.byref(P._OrbitTable(1, 0.0, 100.0, fake, fake)), fake, 64, C.byref(m), fake,
                                  None) == -1                                   # K < 2
    assert L.pespace_response_orb(fake, 4, C.byref(P._OrbitTable(16, 0.0, 0.0, fake, fake)), fake, 64, C.byref(m), fake,
                                  None) == -1                                   # dt <= 0
    assert L.pespace_response_orb(fake, 4, C.byref(P._OrbitTable(16, 0.0, 1.0, fake, None)), fake, 64, C.byref(m), fake,
                                  None) == -1
    assert L.pespace_loglike_orb(fake, 4, C.byref(good), fake, fake, C.byref(g), C.byref(m), fake, fake, 8, None) == -1
    assert L.pespace_loglike_orb(fake, 0, C.byref(good), fake, fake, C.byref(g), C.byref(m), fake, fake, 1 << 30,
                                 None) == -1


def test_a_c_program_links_against_the_library(tmp_path):
    """a caller written in C (not C++, no torch, no Python): includes include/pespace.h, links libpespace.so, asks for
    the workspace size of BASELINE config 2, checks the no-allocation limits and that a bad call is refused with
    PESPACE_EINVAL and a message -- everything that works without a GPU"""
    import subprocess
    from paper_2602_12011_b200 import binding as P     # builds the library if it is missing
    src = tmp_path / "caller.c"
    src.write_text(r'''
#include <stdio.h>
#include <string.h>
#include "pespace.h"
int main(void) {
  pespace_detector det = {0};
  det.kind = 0; det.tdi_gen = 20; det.L_m = 2.5e9; det.kappa = -0.349;
  pespace_model model = {PESPACE_MODE_22, 1, &det};
  pespace_grid grid = {1e-4, 1.0 / (30.0 * 86400.0), 262144};
  size_t ws = pespace_workspace_bytes(4096, &grid, &model, 0);
  size_t wg = pespace_workspace_bytes_grad(4096, &grid, &model);
  if (ws == 0 || wg <= ws) return 1;
  if (pespace_noalloc_scratch_needed(2016, &model) > PESPACE_NOALLOC_SCRATCH_BYTES) return 2;
  if (pespace_noalloc_scratch_needed(2017, &model) <= PESPACE_NOALLOC_SCRATCH_BYTES) return 3;
  if (pespace_loglike(NULL, 4096, NULL, NULL, &grid, &model, NULL, NULL, ws, NULL) != PESPACE_EINVAL) return 4;
  if (strcmp(pespace_strerror(PESPACE_EINVAL), "invalid argument") != 0) return 5;
  det.tdi_gen = 17;                                  /* unknown TDI generation */
  if (pespace_workspace_bytes(4096, &grid, &model, 0) != 0) return 6;
  printf("%s %zu %zu\n", pespace_version(), ws, wg);
  return 0;
}
''')
    exe = tmp_path / "caller"
    libdir = os.path.dirname(P.LIB_PATH)
    res = subprocess.run(["gcc", "-std=c99", "-Wall", "-Werror", "-I", os.path.join(ROOT, "include"), str(src), "-o", str(exe),
                          "-L", libdir, "-lpespace", "-Wl,-rpath," + libdir], capture_output=True, text=True)
    assert res.returncode == 0, res.stderr
    run = subprocess.run([str(exe)], capture_output=True, text=True)
    assert run.returncode == 0, (run.returncode, run.stdout, run.stderr)
    version, ws, wg = run.stdout.strip().rsplit(" ", 2)
    assert version == P.version() and int(ws) > 0 and int(wg) > int(ws)
