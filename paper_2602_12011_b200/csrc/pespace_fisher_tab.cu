// pespace_fisher_tab.cu -- pespace_fisher_tab of include/pespace.h: Fisher matrix / gradient on tabulated mode
// waveforms (T1 x S10).
#include "pespace_host.hpp"
#include "pespace_fisher_tab.cuh"

using namespace pespace;
using namespace pespace::host;

namespace {

struct FisherTabPlan {
  long long nbx, ntile;
  size_t consts_bytes, partial_bytes, bins_bytes, wt_bytes;     // workspace, in this order
};
FisherTabPlan make_plan(long long B, long long N, int n_det) {
  FisherTabPlan p;
  p.nbx = (N + (long long)FBLOCK * FCHUNKS - 1) / ((long long)FBLOCK * FCHUNKS);
  p.ntile = (B + FTILE - 1) / FTILE;
  p.consts_bytes = align_up((size_t)B * fisher_const_stride(n_det) * sizeof(double), 256);
  p.partial_bytes = align_up((size_t)n_det * p.nbx * (size_t)B * NG * sizeof(double), 256);
  p.bins_bytes = align_up((size_t)n_det * NBF * (size_t)N * sizeof(double), 256);
  p.wt_bytes = align_up((size_t)NWT * (size_t)N * sizeof(double), 256);
  return p;
}
bool table_ok(const pespace_wavetable* t) {
  return t && t->K >= 4 && t->d_fnodes && t->d_amp && t->d_phase && t->d_tf;
}
TabC make_tab(const pespace_wavetable* t, unsigned mode_mask) {
  TabC T;
  T.K = t->K; T.amp = t->d_amp; T.phase = t->d_phase; T.tf = t->d_tf;
  const int mm[5] = {2, 1, 3, 2, 4};
  T.n_modes = 0;
  for (int i = 0; i < 5; ++i) T.m[i] = 0;
  for (int i = 0; i < 5; ++i)
    if ((mode_mask >> i) & 1u) T.m[T.n_modes++] = mm[i];
  return T;
}
SmemOptIn g_cfg0, g_cfg1;

}  // namespace

extern "C" {

size_t pespace_workspace_bytes_fisher_tab(int64_t B, const pespace_grid* grid, const pespace_model* model) {
  if (B <= 0 || !grid_ok(grid) || !model_ok(model)) return 0;
  const FisherTabPlan p = make_plan(B, grid->N, model->n_det);
  return p.consts_bytes + p.partial_bytes + p.bins_bytes + p.wt_bytes;
}

int pespace_fisher_tab(const double* d_params, int64_t B, const pespace_wavetable* table, const double* d_data_AET,
                       const double* d_psd, const pespace_grid* grid, const pespace_model* model, double* d_out_F,
                       double* d_out_grad, void* d_workspace, size_t workspace_bytes, void* stream) {
  if (!d_params || !d_psd || (!d_out_F && !d_out_grad) || !d_workspace || B <= 0 || !grid_ok(grid) || !model_ok(model) ||
      !table_ok(table))
    return PESPACE_EINVAL;
  const int grad_only = d_out_F == nullptr;
  if (d_out_grad && !d_data_AET) return PESPACE_EINVAL;       // the gradient needs the data
  if (workspace_bytes < pespace_workspace_bytes_fisher_tab(B, grid, model) || ((uintptr_t)d_workspace & 15u))
    return PESPACE_EINVAL;
  const FisherTabPlan p = make_plan(B, grid->N, model->n_det);
  if (p.ntile > 65535) return PESPACE_EINVAL;
  cudaStream_t st = (cudaStream_t)stream;
  char* ws = (char*)d_workspace;
  double* d_consts = (double*)ws;
  double* d_partial = (double*)(ws + p.consts_bytes);
  double* d_bins = (double*)(ws + p.consts_bytes + p.partial_bytes);
  double* d_wt = (double*)(ws + p.consts_bytes + p.partial_bytes + p.bins_bytes);
  const PrepArgs A = make_prep_args(model);
  prep_samples_tab_du_kernel<<<(unsigned)((B + 63) / 64), 64, 0, st>>>(d_params, B, A, d_consts);
  LAUNCHED();
  const GridC G = {grid->f0, grid->df, (long long)grid->N};
  const unsigned nb256 = (unsigned)((grid->N + 255) / 256);
  prep_bins_kernel<<<dim3(nb256, (unsigned)model->n_det), 256, 0, st>>>((const double2*)d_data_AET, d_psd, G, A, 0, d_bins);
  LAUNCHED();
  prep_tab_weights_kernel<<<nb256, 256, 0, st>>>(G, table->d_fnodes, table->K, d_wt);
  LAUNCHED();
  const TabC T = make_tab(table, model->mode_mask);
  const dim3 g((unsigned)p.nbx, (unsigned)p.ntile);
  for (int d = 0; d < model->n_det; ++d) {
    const DetC dc = make_det(model->det[d]);
    EvPair ev;
    if (int rc = prof_begin(ev, st); rc != PESPACE_OK) return rc;
    if (dc.kind == 0) {
      CU(opt_in_smem(fisher_tab_kernel<0>, fisher_smem_bytes(), g_cfg0));
      fisher_tab_kernel<0><<<g, FBLOCK, fisher_smem_bytes(), st>>>(d_consts, B, T, d_bins, d_wt, G.N, dc, model->n_det, d,
                                                                   grad_only, d_partial);
    } else {
      CU(opt_in_smem(fisher_tab_kernel<1>, fisher_smem_bytes(), g_cfg1));
      fisher_tab_kernel<1><<<g, FBLOCK, fisher_smem_bytes(), st>>>(d_consts, B, T, d_bins, d_wt, G.N, dc, model->n_det, d,
                                                                   grad_only, d_partial);
    }
    LAUNCHED();
    if (int rc = prof_end(ev, st); rc != PESPACE_OK) return rc;
  }
  const long long nt = (long long)B * NG;
  combine_fisher_kernel<<<(unsigned)((nt + 31) / 32), dim3(32, CGROUPS), 0, st>>>(
      d_partial, d_consts, B, (int)(model->n_det * p.nbx), fisher_const_stride(model->n_det), d_out_F, d_out_grad);
  LAUNCHED();
  return PESPACE_OK;
}

}  // extern "C"
