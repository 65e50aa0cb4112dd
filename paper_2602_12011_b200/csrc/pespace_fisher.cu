// pespace_fisher.cu -- pespace_fisher of include/pespace.h: forward-mode derivatives (S10).
#include "pespace_launch.hpp"
#include "pespace_fisher.cuh"

using namespace pespace;
using namespace pespace::host;

namespace {

struct FisherPlan {
  long long nbx, ntile;
  size_t consts_bytes, partial_bytes, bins_bytes;     // workspace: [sample constants | block partials | per-bin table]
};
FisherPlan make_fisher_plan(long long B, long long N, int n_det) {
  FisherPlan p;
  p.nbx = (N + (long long)FBLOCK * FCHUNKS - 1) / ((long long)FBLOCK * FCHUNKS);
  p.ntile = (B + FTILE - 1) / FTILE;
  p.consts_bytes = align_up((size_t)B * fisher_const_stride(n_det) * sizeof(double), 256);
  p.partial_bytes = align_up((size_t)n_det * p.nbx * (size_t)B * NG * sizeof(double), 256);
  p.bins_bytes = align_up((size_t)n_det * NBF * (size_t)N * sizeof(double), 256);
  return p;
}

}  // namespace

namespace pespace {
namespace host {
size_t fisher_workspace_bytes(long long B, long long N, int n_det) {
  const FisherPlan p = make_fisher_plan(B, N, n_det);
  return p.consts_bytes + p.partial_bytes + p.bins_bytes;
}
}  // namespace host
}  // namespace pespace

extern "C" int pespace_fisher(const double* d_params, int64_t B, const double* d_data_AET, const double* d_psd,
                              const pespace_grid* grid, const pespace_model* model, double* d_out_F,
                              double* d_out_grad, void* d_workspace, size_t workspace_bytes, void* stream) {
  if (!d_params || !d_psd || (!d_out_F && !d_out_grad) || !d_workspace || B <= 0 || !grid_ok(grid) || !model_ok(model))
    return PESPACE_EINVAL;
  const int grad_only = d_out_F == nullptr;                   // d lnL / d theta alone: row 0 of the Gram matrix
  if (d_out_grad && !d_data_AET) return PESPACE_EINVAL;       // the gradient needs the data
  if (workspace_bytes < fisher_workspace_bytes(B, grid->N, model->n_det) || ((uintptr_t)d_workspace & 15u))
    return PESPACE_EINVAL;
  const FisherPlan p = make_fisher_plan(B, grid->N, model->n_det);
  if (p.ntile > 65535) return PESPACE_EINVAL;                 // gridDim.y
  cudaStream_t st = (cudaStream_t)stream;
  double* d_consts = (double*)d_workspace;
  double* d_partial = (double*)((char*)d_workspace + p.consts_bytes);
  double* d_bins = (double*)((char*)d_workspace + p.consts_bytes + p.partial_bytes);
  const PrepArgs A = make_prep_args(model);
  const int th = 64;
  prep_samples_du_kernel<<<(unsigned)((prep_du_threads(B, model->n_det) + th - 1) / th), th, 0, st>>>(d_params, B, A,
                                                                                                    d_consts);
  LAUNCHED();
  const unsigned cm = class_mask(model->mode_mask);
  const GridC G = {grid->f0, grid->df, (long long)grid->N};
  {
    // S0: per-bin table of this data set (d_data_AET == NULL: zeros, Fisher matrix only)
    const dim3 gb((unsigned)((grid->N + 255) / 256), (unsigned)model->n_det);
    prep_bins_kernel<<<gb, 256, 0, st>>>((const double2*)d_data_AET, d_psd, G, A, 1, d_bins);
    LAUNCHED();
  }
  const dim3 g((unsigned)p.nbx, (unsigned)p.ntile);
  for (int d = 0; d < model->n_det; ++d) {
    const DetC dc = make_det(model->det[d]);
    EvPair ev;
    if (int rc = prof_begin(ev, st); rc != PESPACE_OK) return rc;
    CU(fisher_launcher(dc.kind, cm)(g, st, d_consts, B, d_bins, G.N, dc, model->n_det, d, grad_only, d_partial));
    LAUNCHED();
    if (int rc = prof_end(ev, st); rc != PESPACE_OK) return rc;
  }
  const long long nt = (long long)B * NG;
  combine_fisher_kernel<<<(unsigned)((nt + 31) / 32), dim3(32, CGROUPS), 0, st>>>(
      d_partial, d_consts, B, (int)(model->n_det * p.nbx), fisher_const_stride(model->n_det), d_out_F, d_out_grad);
  LAUNCHED();
  return PESPACE_OK;
}
