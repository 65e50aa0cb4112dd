// pespace_grad.cu -- pespace_loglike_grad of include/pespace.h: lnL and d lnL / d theta by reverse mode (SURVEY.md
// 8(f) N4).
#include "pespace_launch.hpp"
#include "pespace_grad.cuh"

using namespace pespace;
using namespace pespace::host;

namespace {

struct GradPlan {
  long long nbx, ntile;
  size_t trig_bytes, bins_bytes, consts_bytes, du_bytes, partial_bytes;   // workspace, in this order
};
GradPlan make_grad_plan(long long B, long long N, int n_det, unsigned cmask) {
  GradPlan p;
  p.nbx = (N + (long long)BLOCK * GCHUNKS - 1) / ((long long)BLOCK * GCHUNKS);
  p.ntile = (B + grad_tile(cmask) - 1) / grad_tile(cmask);
  p.trig_bytes = align_up((size_t)NTAB * sizeof(double2), 256);
  p.bins_bytes = align_up((size_t)n_det * NBF * (size_t)N * sizeof(double), 256);
  p.consts_bytes = align_up((size_t)B * sample_stride(n_det) * sizeof(double), 256);
  p.du_bytes = align_up((size_t)B * fisher_const_stride(n_det) * sizeof(double), 256);
  p.partial_bytes = align_up((size_t)n_det * p.nbx * (size_t)B * NVP * sizeof(double), 256);
  return p;
}

}  // namespace

extern "C" {

size_t pespace_workspace_bytes_grad(int64_t B, const pespace_grid* grid, const pespace_model* model) {
  if (B <= 0 || !grid_ok(grid) || !model_ok(model)) return 0;
  const GradPlan p = make_grad_plan(B, grid->N, model->n_det, class_mask(model->mode_mask));
  return p.trig_bytes + p.bins_bytes + p.consts_bytes + p.du_bytes + p.partial_bytes;
}

int pespace_loglike_grad(const double* d_params, int64_t B, const double* d_data_AET, const double* d_psd,
                         const pespace_grid* grid, const pespace_model* model, double* d_out_lnL, double* d_out_grad,
                         void* d_workspace, size_t workspace_bytes, void* stream) {
  return loglike_grad_impl(d_params, B, d_data_AET, d_psd, grid, model, d_out_lnL, d_out_grad, d_workspace,
                           workspace_bytes, stream, false);
}

int pespace_loglike_grad_prepared(const double* d_params, int64_t B, const pespace_grid* grid,
                                  const pespace_model* model, double* d_out_lnL, double* d_out_grad, void* d_workspace,
                                  size_t workspace_bytes, void* stream) {
  return loglike_grad_impl(d_params, B, nullptr, nullptr, grid, model, d_out_lnL, d_out_grad, d_workspace,
                           workspace_bytes, stream, true);
}

}  // extern "C"

// bins_ready: the per-bin table at the head of the workspace was written by pespace_prepare (or an earlier call) for
// the same data set, PSD, grid and model
int pespace::host::loglike_grad_impl(const double* d_params, int64_t B, const double* d_data_AET, const double* d_psd,
                                     const pespace_grid* grid, const pespace_model* model, double* d_out_lnL,
                                     double* d_out_grad, void* d_workspace, size_t workspace_bytes, void* stream,
                                     bool bins_ready) {
  if (!d_params || (!bins_ready && (!d_data_AET || !d_psd)) || (!d_out_lnL && !d_out_grad) || !d_workspace || B <= 0 ||
      !grid_ok(grid) || !model_ok(model))
    return PESPACE_EINVAL;
  if (workspace_bytes < pespace_workspace_bytes_grad(B, grid, model) || ((uintptr_t)d_workspace & 15u))
    return PESPACE_EINVAL;
  const GradPlan p = make_grad_plan(B, grid->N, model->n_det, class_mask(model->mode_mask));
  if (p.ntile > 65535) return PESPACE_EINVAL;                 // gridDim.y
  cudaStream_t st = (cudaStream_t)stream;
  char* ws = (char*)d_workspace;
  double2* d_trig = (double2*)ws;
  double* d_bins = (double*)(ws + p.trig_bytes);
  double* d_consts = (double*)(ws + p.trig_bytes + p.bins_bytes);
  double* d_du = (double*)(ws + p.trig_bytes + p.bins_bytes + p.consts_bytes);
  double* d_partial = (double*)(ws + p.trig_bytes + p.bins_bytes + p.consts_bytes + p.du_bytes);
  const PrepArgs A = make_prep_args(model);
  // S1 twice: the plain constants the sweep reads, and their tangents for the chain rule of the second pass
  prep_samples_kernel<<<(unsigned)((prep_threads(B, model->n_det) + 127) / 128), 128, 0, st>>>(d_params, B, A, d_consts,
                                                                                             d_trig);
  LAUNCHED();
  prep_samples_du_kernel<<<(unsigned)((prep_du_threads(B, model->n_det) + 63) / 64), 64, 0, st>>>(d_params, B, A, d_du);
  LAUNCHED();
  const GridC G = {grid->f0, grid->df, (long long)grid->N};
  if (!bins_ready) {
    prep_bins_kernel<<<dim3((unsigned)((grid->N + 255) / 256), (unsigned)model->n_det), 256, 0, st>>>(
        (const double2*)d_data_AET, d_psd, G, A, 1, d_bins);
    LAUNCHED();
  }
  const unsigned cm = class_mask(model->mode_mask);
  const dim3 g((unsigned)p.nbx, (unsigned)p.ntile);
  for (int d = 0; d < model->n_det; ++d) {
    const DetC dc = make_det(model->det[d]);
    EvPair ev;
    if (int rc = prof_begin(ev, st); rc != PESPACE_OK) return rc;
    CU(grad_launcher(dc.kind, cm)(g, st, d_consts, d_trig, B, d_bins, G.N, dc, model->n_det, d, d_partial));
    LAUNCHED();
    if (int rc = prof_end(ev, st); rc != PESPACE_OK) return rc;
  }
  combine_grad_kernel<<<(unsigned)((B + 3) / 4), 128, 0, st>>>(d_partial, d_du, d_params, B, (int)(model->n_det * p.nbx),
                                                             model->n_det, d_out_lnL, d_out_grad);
  LAUNCHED();
  return PESPACE_OK;
}
