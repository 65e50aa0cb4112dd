"""The C ABI used from C, end to end on the GPU: a program written in C99 (gcc; no C++, no torch, no Python in the
process) reads theta, data and PSD from files, allocates device memory with the CUDA runtime API, calls
pespace_workspace_bytes, pespace_loglike, pespace_loglike_grad and pespace_response_noalloc of include/pespace.h, and
writes the results back.  They must equal, bit for bit, what the Python binding returns for the same inputs."""
import os
import subprocess

import numpy as np
import pytest

from paper_2602_12011_b200 import workloads as W

pytestmark = pytest.mark.gpu

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

C_SOURCE = r'''
#include <stdio.h>
#include <stdlib.h>
#include <cuda_runtime_api.h>
#include "pespace.h"

static double* load(const char* path, size_t n) {
  double* h = (double*)malloc(n * sizeof(double));
  FILE* f = fopen(path, "rb");
  if (!h || !f || fread(h, sizeof(double), n, f) != n) { fprintf(stderr, "cannot read %s\n", path); exit(10); }
  fclose(f);
  return h;
}
static double* to_device(const double* h, size_t n) {
  double* d = NULL;
  if (cudaMalloc((void**)&d, n * sizeof(double)) != cudaSuccess) exit(11);
  if (cudaMemcpy(d, h, n * sizeof(double), cudaMemcpyHostToDevice) != cudaSuccess) exit(12);
  return d;
}
static void save(const char* path, const double* d, size_t n) {
  double* h = (double*)malloc(n * sizeof(double));
  if (cudaMemcpy(h, d, n * sizeof(double), cudaMemcpyDeviceToHost) != cudaSuccess) exit(13);
  FILE* f = fopen(path, "wb");
  if (!f || fwrite(h, sizeof(double), n, f) != n) exit(14);
  fclose(f);
  free(h);
}
#define OK(call) do { int rc_ = (call); if (rc_ != PESPACE_OK) { \
  fprintf(stderr, "%s: %s\n", #call, pespace_strerror(rc_)); return 20; } } while (0)

int main(int argc, char** argv) {
  if (argc != 4) return 1;
  const long B = atol(argv[1]), N = atol(argv[2]);
  const char* dir = argv[3];
  char path[1024];
  pespace_detector det[2] = {{0}, {0}};
  det[0].kind = 0; det[0].tdi_gen = 20; det[0].L_m = 2.5e9; det[0].kappa = -0.3490658503988659;
  det[1].kind = 1; det[1].tdi_gen = 15; det[1].L_m = 1.7320508075688772e8; det[1].period_s = 315360.0;
  det[1].lon = 2.1031217584577884; det[1].lat = -0.08203047484373349;
  pespace_model model = {PESPACE_MODE_22 | PESPACE_MODE_33 | PESPACE_MODE_21, 2, det};
  pespace_grid grid = {1.2e-4, 2.5e-6, N};
  const size_t n_data = (size_t)2 * 3 * N * 2, n_psd = (size_t)2 * 3 * N;
  snprintf(path, sizeof path, "%s/theta.bin", dir); double* d_theta = to_device(load(path, (size_t)B * 11), (size_t)B * 11);
  snprintf(path, sizeof path, "%s/data.bin", dir);  double* d_data = to_device(load(path, n_data), n_data);
  snprintf(path, sizeof path, "%s/psd.bin", dir);   double* d_psd = to_device(load(path, n_psd), n_psd);
  snprintf(path, sizeof path, "%s/freqs.bin", dir); double* d_freqs = to_device(load(path, (size_t)N), (size_t)N);
  size_t ws = pespace_workspace_bytes(B, &grid, &model, 0), wg = pespace_workspace_bytes_grad(B, &grid, &model);
  if (!ws || !wg) return 2;
  void* d_ws = NULL; double *d_lnL, *d_gl, *d_grad, *d_resp;
  if (cudaMalloc(&d_ws, wg > ws ? wg : ws) != cudaSuccess) return 3;
  cudaMalloc((void**)&d_lnL, B * sizeof(double)); cudaMalloc((void**)&d_gl, B * sizeof(double));
  cudaMalloc((void**)&d_grad, B * 11 * sizeof(double));
  cudaMalloc((void**)&d_resp, (size_t)B * 2 * 3 * N * 2 * sizeof(double));
  cudaStream_t st;
  if (cudaStreamCreate(&st) != cudaSuccess) return 4;
  OK(pespace_loglike(d_theta, B, d_data, d_psd, &grid, &model, d_lnL, d_ws, ws, st));
  OK(pespace_loglike_grad(d_theta, B, d_data, d_psd, &grid, &model, d_gl, d_grad, d_ws, wg, st));
  OK(pespace_response_noalloc(d_theta, B, d_freqs, N, &model, d_resp, st));
  if (cudaStreamSynchronize(st) != cudaSuccess) return 5;
  snprintf(path, sizeof path, "%s/lnL.bin", dir);  save(path, d_lnL, (size_t)B);
  snprintf(path, sizeof path, "%s/gl.bin", dir);   save(path, d_gl, (size_t)B);
  snprintf(path, sizeof path, "%s/grad.bin", dir); save(path, d_grad, (size_t)B * 11);
  snprintf(path, sizeof path, "%s/resp.bin", dir); save(path, d_resp, (size_t)B * 2 * 3 * N * 2);
  printf("%s\n", pespace_version());
  return 0;
}
'''


def test_c_program_runs_the_hot_path_and_matches_the_binding(tmp_path):
    import torch
    from paper_2602_12011_b200 import binding as P
    assert torch.cuda.is_available()
    B, N = 70, 3000
    grid = W.Grid(1.2e-4, 2.5e-6, N)
    lisa, tq = W.lisa_like(20), W.tianqin_like(15)
    model = W.Model(W.MODE_22 | W.MODE_33 | W.MODE_21, (lisa, tq))
    rng = np.random.default_rng(5)
    theta = W.draw_prior(B, 1.0 / grid.df, rng)
    wl = W.Workload("c-caller", grid, model, theta, theta[0].copy(), 3)
    psd = wl.psd()
    data = W.coloured_noise(psd, grid.df, rng)
    for name, arr in (("theta", theta), ("data", np.ascontiguousarray(data).view(np.float64)), ("psd", psd),
                      ("freqs", grid.freqs())):
        np.ascontiguousarray(arr, dtype=np.float64).tofile(tmp_path / f"{name}.bin")
    src = tmp_path / "caller.c"
    src.write_text(C_SOURCE.replace("315360.0", repr(float(tq.period_s))).replace("2.1031217584577884", repr(float(tq.lon)))
                   .replace("-0.08203047484373349", repr(float(tq.lat))).replace("-0.3490658503988659", repr(float(lisa.kappa)))
                   .replace("1.7320508075688772e8", repr(float(tq.L_m))))
    cuda = os.environ.get("CUDA_HOME", "/usr/local/cuda")
    libdir = os.path.dirname(P.LIB_PATH)
    exe = tmp_path / "caller"
    res = subprocess.run(["gcc", "-std=c99", "-Wall", "-Werror", "-I", os.path.join(ROOT, "include"), "-I", os.path.join(cuda, "include"),
                          str(src), "-o", str(exe), "-L", libdir, "-lpespace", "-L", os.path.join(cuda, "lib64"), "-lcudart",
                          "-Wl,-rpath," + libdir, "-Wl,-rpath," + os.path.join(cuda, "lib64")], capture_output=True, text=True)
    assert res.returncode == 0, res.stderr
    run = subprocess.run([str(exe), str(B), str(N), str(tmp_path)], capture_output=True, text=True, timeout=300)
    assert run.returncode == 0, (run.returncode, run.stdout, run.stderr)
    assert run.stdout.strip() == P.version()

    dev = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    lnL = P.loglike(dev(theta), dev(data), dev(psd), grid, model).cpu().numpy()
    gl, grad = (x.cpu().numpy() for x in P.loglike_grad(dev(theta), dev(data), dev(psd), grid, model))
    resp = torch.view_as_real(P.response(dev(theta), dev(grid.freqs()), model)).cpu().numpy()
    assert np.array_equal(np.fromfile(tmp_path / "lnL.bin"), lnL)
    assert np.array_equal(np.fromfile(tmp_path / "gl.bin"), gl)
    assert np.array_equal(np.fromfile(tmp_path / "grad.bin").reshape(B, 11), grad)
    assert np.array_equal(np.fromfile(tmp_path / "resp.bin").reshape(resp.shape), resp)
