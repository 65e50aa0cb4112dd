// pespace_session.cu -- host-buffer entry points of include/pespace.h.  A session keeps the data set, the
// PSD, the workspace and the result buffers resident on the device between calls (the
// sampler-facing use is many batches of theta against ONE data set), so that a call moves only theta in and
// lnL (or F, grad) out.  Every step of the path still runs in the kernels behind pespace_loglike /
// pespace_fisher; this file only owns memory, a stream and the copies.
#include "pespace_host.hpp"

#include <new>
#include <vector>

using namespace pespace;
using namespace pespace::host;

struct pespace_session {
  pespace_grid grid;
  pespace_model model;
  std::vector<pespace_detector> det;
  long long max_B = 0;
  int want_fisher = 0;
  bool have_data = false, have_psd = false;
  bool bins_ready = false;          // the per-bin table in d_ws matches the current data set and PSD
  cudaStream_t st = nullptr;
  double *d_params = nullptr, *d_data = nullptr, *d_psd = nullptr, *d_lnL = nullptr, *d_F = nullptr, *d_grad = nullptr;
  void *d_ws = nullptr, *d_ws_f = nullptr, *d_ws_t = nullptr, *d_ws_g = nullptr;
  size_t ws_bytes = 0, ws_f_bytes = 0, ws_t_bytes = 0, ws_g_bytes = 0;
  double* d_grad_g = nullptr;       // [max_B][11], pespace_session_loglike_grad (allocated on first use)
  // zero-copy result path of pespace_session_loglike: combine_kernel writes lnL straight into mapped pinned host
  // memory (no device-to-host copy call; theta of small batches goes the same way in the other direction)
  double *h_lnL_pin = nullptr, *d_lnL_map = nullptr, *h_par_pin = nullptr, *d_par_map = nullptr;
  double* d_tab = nullptr;          // [fnodes K | amp | phase | tf], grown on demand (pespace_session_loglike_tab)
  size_t tab_doubles = 0;
  size_t n_series() const { return (size_t)model.n_det * 3 * (size_t)grid.N; }
};

namespace {

void release(pespace_session* s) {
  if (!s) return;
  cudaFree(s->d_params); cudaFree(s->d_data); cudaFree(s->d_psd); cudaFree(s->d_lnL); cudaFree(s->d_F);
  cudaFree(s->d_grad); cudaFree(s->d_ws); cudaFree(s->d_ws_f); cudaFree(s->d_ws_t); cudaFree(s->d_tab);
  cudaFree(s->d_ws_g); cudaFree(s->d_grad_g);
  if (s->h_lnL_pin) cudaFreeHost(s->h_lnL_pin);
  if (s->h_par_pin) cudaFreeHost(s->h_par_pin);
  if (s->st) cudaStreamDestroy(s->st);
  delete s;
}

}  // namespace

extern "C" {

int pespace_session_create(const pespace_grid* grid, const pespace_model* model, int64_t max_B, int want_fisher,
                           pespace_session** out) {
  if (!out) return PESPACE_EINVAL;
  *out = nullptr;
  if (max_B <= 0 || !grid_ok(grid) || !model_ok(model)) return PESPACE_EINVAL;
  pespace_session* s = new (std::nothrow) pespace_session();
  if (!s) return PESPACE_ENOMEM;
  s->grid = *grid;
  s->det.assign(model->det, model->det + model->n_det);
  s->model = *model;
  s->model.det = s->det.data();
  s->max_B = max_B;
  s->want_fisher = want_fisher != 0;
  s->ws_bytes = pespace_workspace_bytes(max_B, grid, &s->model, 0);
  s->ws_f_bytes = want_fisher ? pespace_workspace_bytes(max_B, grid, &s->model, 1) : 0;
  const size_t nS = s->n_series();
  bool ok = cudaStreamCreateWithFlags(&s->st, cudaStreamNonBlocking) == cudaSuccess &&
            cudaMalloc((void**)&s->d_params, (size_t)max_B * NPAR * 8) == cudaSuccess &&
            cudaMalloc((void**)&s->d_data, nS * 16) == cudaSuccess &&
            cudaMalloc((void**)&s->d_psd, nS * 8) == cudaSuccess &&
            cudaMalloc((void**)&s->d_lnL, (size_t)max_B * 8) == cudaSuccess &&
            cudaMalloc(&s->d_ws, s->ws_bytes) == cudaSuccess;
  constexpr int64_t kMappedThetaMax = 256;       // samples whose theta is read over the bus by the prep kernel
  ok = ok && cudaHostAlloc((void**)&s->h_lnL_pin, (size_t)max_B * 8, cudaHostAllocMapped) == cudaSuccess &&
       cudaHostGetDevicePointer((void**)&s->d_lnL_map, s->h_lnL_pin, 0) == cudaSuccess &&
       cudaHostAlloc((void**)&s->h_par_pin, (size_t)kMappedThetaMax * NPAR * 8, cudaHostAllocMapped) == cudaSuccess &&
       cudaHostGetDevicePointer((void**)&s->d_par_map, s->h_par_pin, 0) == cudaSuccess;
  if (ok && want_fisher)
    ok = cudaMalloc((void**)&s->d_F, (size_t)max_B * NPAR * NPAR * 8) == cudaSuccess &&
         cudaMalloc((void**)&s->d_grad, (size_t)max_B * NPAR * 8) == cudaSuccess &&
         cudaMalloc(&s->d_ws_f, s->ws_f_bytes) == cudaSuccess;
  if (!ok) {
    cudaGetLastError();
    release(s);
    return PESPACE_ENOMEM;
  }
  *out = s;
  return PESPACE_OK;
}

int pespace_session_destroy(pespace_session* s) {
  if (!s) return PESPACE_EINVAL;
  cudaError_t e = cudaStreamSynchronize(s->st);
  release(s);
  return e == cudaSuccess ? PESPACE_OK : cuda_fail(e);
}

int pespace_session_set_data(pespace_session* s, const double* h_data_AET, const double* h_psd) {
  if (!s || (!h_data_AET && !h_psd)) return PESPACE_EINVAL;
  const size_t nS = s->n_series();
  if (h_data_AET) {
    CU(cudaMemcpyAsync(s->d_data, h_data_AET, nS * 16, cudaMemcpyHostToDevice, s->st));
    s->have_data = true;
  }
  if (h_psd) {
    CU(cudaMemcpyAsync(s->d_psd, h_psd, nS * 8, cudaMemcpyHostToDevice, s->st));
    s->have_psd = true;
  }
  s->bins_ready = false;
  CU(cudaStreamSynchronize(s->st));   // the caller may reuse its buffers on return
  return PESPACE_OK;
}

int pespace_session_loglike(pespace_session* s, const double* h_params, int64_t B, double* h_out_lnL) {
  if (!s || !h_params || !h_out_lnL || B <= 0 || B > s->max_B || !s->have_data || !s->have_psd) return PESPACE_EINVAL;
  const double* d_theta = s->d_params;
  if (B <= 256) {                                       // small batch: theta through mapped pinned memory, no copy call
    std::memcpy(s->h_par_pin, h_params, (size_t)B * NPAR * 8);
    d_theta = s->d_par_map;
  } else {
    CU(cudaMemcpyAsync(s->d_params, h_params, (size_t)B * NPAR * 8, cudaMemcpyHostToDevice, s->st));
  }
  const int rc = loglike_impl(d_theta, B, s->d_data, s->d_psd, &s->grid, &s->model, s->d_lnL_map, s->d_ws, s->ws_bytes,
                              s->st, s->bins_ready);      // the S0 table is built once per data set
  if (rc != PESPACE_OK) { s->bins_ready = false; return rc; }
  s->bins_ready = true;
  CU(cudaStreamSynchronize(s->st));
  std::memcpy(h_out_lnL, s->h_lnL_pin, (size_t)B * 8);
  return PESPACE_OK;
}

int pespace_session_loglike_mixed(pespace_session* s, const double* h_params, int64_t B, double* h_out_lnL) {
  if (!s || !h_params || !h_out_lnL || B <= 0 || B > s->max_B || !s->have_data || !s->have_psd) return PESPACE_EINVAL;
  CU(cudaMemcpyAsync(s->d_params, h_params, (size_t)B * NPAR * 8, cudaMemcpyHostToDevice, s->st));
  s->bins_ready = false;            // the mixed kernel keeps its own (whitened) per-bin table in the same workspace
  const int rc = pespace_loglike_mixed(s->d_params, B, s->d_data, s->d_psd, &s->grid, &s->model, s->d_lnL_map, s->d_ws,
                                       s->ws_bytes, s->st);
  if (rc != PESPACE_OK) return rc;
  CU(cudaStreamSynchronize(s->st));
  std::memcpy(h_out_lnL, s->h_lnL_pin, (size_t)B * 8);
  return PESPACE_OK;
}

int pespace_session_fisher(pespace_session* s, const double* h_params, int64_t B, double* h_out_F,
                           double* h_out_grad) {
  if (!s || !s->want_fisher || !h_params || (!h_out_F && !h_out_grad) || B <= 0 || B > s->max_B || !s->have_psd)
    return PESPACE_EINVAL;
  if (h_out_grad && !s->have_data) return PESPACE_EINVAL;
  CU(cudaMemcpyAsync(s->d_params, h_params, (size_t)B * NPAR * 8, cudaMemcpyHostToDevice, s->st));
  const int rc = pespace_fisher(s->d_params, B, h_out_grad ? s->d_data : nullptr, s->d_psd, &s->grid, &s->model,
                                h_out_F ? s->d_F : nullptr, h_out_grad ? s->d_grad : nullptr, s->d_ws_f, s->ws_f_bytes,
                                s->st);
  if (rc != PESPACE_OK) return rc;
  if (h_out_F) CU(cudaMemcpyAsync(h_out_F, s->d_F, (size_t)B * NPAR * NPAR * 8, cudaMemcpyDeviceToHost, s->st));
  if (h_out_grad) CU(cudaMemcpyAsync(h_out_grad, s->d_grad, (size_t)B * NPAR * 8, cudaMemcpyDeviceToHost, s->st));
  CU(cudaStreamSynchronize(s->st));
  return PESPACE_OK;
}

int pespace_session_loglike_grad(pespace_session* s, const double* h_params, int64_t B, double* h_out_lnL,
                                 double* h_out_grad) {
  if (!s || !h_params || (!h_out_lnL && !h_out_grad) || B <= 0 || B > s->max_B || !s->have_data || !s->have_psd)
    return PESPACE_EINVAL;
  if (!s->d_ws_g) {
    s->ws_g_bytes = pespace_workspace_bytes_grad(s->max_B, &s->grid, &s->model);
    if (cudaMalloc(&s->d_ws_g, s->ws_g_bytes) != cudaSuccess ||
        cudaMalloc((void**)&s->d_grad_g, (size_t)s->max_B * NPAR * 8) != cudaSuccess) {
      cudaGetLastError();
      cudaFree(s->d_ws_g); s->d_ws_g = nullptr;
      return PESPACE_ENOMEM;
    }
  }
  CU(cudaMemcpyAsync(s->d_params, h_params, (size_t)B * NPAR * 8, cudaMemcpyHostToDevice, s->st));
  const int rc = pespace_loglike_grad(s->d_params, B, s->d_data, s->d_psd, &s->grid, &s->model,
                                      h_out_lnL ? s->d_lnL_map : nullptr, h_out_grad ? s->d_grad_g : nullptr, s->d_ws_g,
                                      s->ws_g_bytes, s->st);
  if (rc != PESPACE_OK) return rc;
  if (h_out_grad) CU(cudaMemcpyAsync(h_out_grad, s->d_grad_g, (size_t)B * NPAR * 8, cudaMemcpyDeviceToHost, s->st));
  CU(cudaStreamSynchronize(s->st));
  if (h_out_lnL) std::memcpy(h_out_lnL, s->h_lnL_pin, (size_t)B * 8);
  return PESPACE_OK;
}

int pespace_session_loglike_tab(pespace_session* s, const double* h_params, int64_t B, int64_t K,
                                const double* h_fnodes, const double* h_amp, const double* h_phase, const double* h_tf,
                                double* h_out_lnL) {
  if (!s || !h_params || !h_out_lnL || !h_fnodes || !h_amp || !h_phase || !h_tf || B <= 0 || B > s->max_B || K < 4 ||
      !s->have_data || !s->have_psd)
    return PESPACE_EINVAL;
  for (int64_t j = 0; j + 1 < K; ++j)
    if (!(h_fnodes[j + 1] > h_fnodes[j])) return PESPACE_EINVAL;      // host memory: the node order can be checked
  int n_modes = 0;
  for (int i = 0; i < 5; ++i) n_modes += (s->model.mode_mask >> i) & 1u;
  const size_t per = (size_t)B * n_modes * (size_t)K, need = (size_t)K + 3 * per;
  if (need > s->tab_doubles) {
    CU(cudaStreamSynchronize(s->st));
    cudaFree(s->d_tab);
    s->d_tab = nullptr; s->tab_doubles = 0;
    if (cudaMalloc((void**)&s->d_tab, need * 8) != cudaSuccess) { cudaGetLastError(); return PESPACE_ENOMEM; }
    s->tab_doubles = need;
  }
  if (!s->d_ws_t) {
    s->ws_t_bytes = pespace_workspace_bytes_tab(s->max_B, &s->grid, &s->model);
    if (cudaMalloc(&s->d_ws_t, s->ws_t_bytes) != cudaSuccess) { cudaGetLastError(); return PESPACE_ENOMEM; }
  }
  double *d_fn = s->d_tab, *d_amp = d_fn + K, *d_ph = d_amp + per, *d_tf = d_ph + per;
  CU(cudaMemcpyAsync(s->d_params, h_params, (size_t)B * NPAR * 8, cudaMemcpyHostToDevice, s->st));
  CU(cudaMemcpyAsync(d_fn, h_fnodes, (size_t)K * 8, cudaMemcpyHostToDevice, s->st));
  CU(cudaMemcpyAsync(d_amp, h_amp, per * 8, cudaMemcpyHostToDevice, s->st));
  CU(cudaMemcpyAsync(d_ph, h_phase, per * 8, cudaMemcpyHostToDevice, s->st));
  CU(cudaMemcpyAsync(d_tf, h_tf, per * 8, cudaMemcpyHostToDevice, s->st));
  const pespace_wavetable T = {K, d_fn, d_amp, d_ph, d_tf};
  const int rc = pespace_loglike_tab(s->d_params, B, &T, s->d_data, s->d_psd, &s->grid, &s->model, s->d_lnL, s->d_ws_t,
                                     s->ws_t_bytes, s->st);
  if (rc != PESPACE_OK) return rc;
  CU(cudaMemcpyAsync(h_out_lnL, s->d_lnL, (size_t)B * 8, cudaMemcpyDeviceToHost, s->st));
  CU(cudaStreamSynchronize(s->st));
  return PESPACE_OK;
}

int pespace_loglike_host(const double* h_params, int64_t B, const double* h_data_AET, const double* h_psd,
                         const pespace_grid* grid, const pespace_model* model, double* h_out_lnL) {
  if (!h_params || !h_data_AET || !h_psd || !h_out_lnL) return PESPACE_EINVAL;
  pespace_session* s = nullptr;
  int rc = pespace_session_create(grid, model, B, 0, &s);
  if (rc != PESPACE_OK) return rc;
  rc = pespace_session_set_data(s, h_data_AET, h_psd);
  if (rc == PESPACE_OK) rc = pespace_session_loglike(s, h_params, B, h_out_lnL);
  const int rc2 = pespace_session_destroy(s);
  return rc != PESPACE_OK ? rc : rc2;
}

}  // extern "C"
