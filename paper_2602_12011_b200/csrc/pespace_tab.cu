// pespace_tab.cu -- pespace_response_tab / pespace_loglike_tab of include/pespace.h: response and likelihood
// from tabulated mode waveforms.
#include "pespace_host.hpp"
#include "pespace_tab.cuh"

using namespace pespace;
using namespace pespace::host;

namespace {

struct TabPlan {
  int stride;
  long long nbb, ntile;
  size_t trig_bytes, consts_bytes, partial_bytes, bins_bytes, wt_bytes;
};
TabPlan make_tab_plan(long long B, long long N, int n_det) {
  TabPlan p;
  p.stride = sample_stride(n_det);
  p.nbb = (N + BLOCK - 1) / BLOCK;
  p.ntile = (B + TAB_TILE - 1) / TAB_TILE;
  p.trig_bytes = align_up((size_t)NTAB * sizeof(double2), 256);
  p.consts_bytes = align_up((size_t)B * p.stride * sizeof(double), 256);
  p.partial_bytes = align_up((size_t)n_det * p.nbb * (size_t)B * sizeof(double), 256);
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

template <class K>
cudaError_t opt_in(K kernel, SmemOptIn& done) { return opt_in_smem(kernel, tab_smem_bytes(), done); }

int run_prep_tab(const double* d_params, long long B, const pespace_model* model, double* d_consts, double2* d_trig,
                 cudaStream_t st) {
  const PrepArgs A = make_prep_args(model);
  const int th = 128;
  prep_samples_tab_kernel<<<(unsigned)((prep_threads(B) + th - 1) / th), th, 0, st>>>(d_params, B, A, d_consts, d_trig);
  LAUNCHED();
  return PESPACE_OK;
}

}  // namespace

extern "C" {

size_t pespace_workspace_bytes_tab(int64_t B, const pespace_grid* grid, const pespace_model* model) {
  if (B <= 0 || !grid_ok(grid) || !model_ok(model)) return 0;
  const TabPlan p = make_tab_plan(B, grid->N, model->n_det);
  return p.trig_bytes + p.consts_bytes + p.partial_bytes + p.bins_bytes + p.wt_bytes;
}

int pespace_response_tab(const double* d_params, int64_t B, const pespace_wavetable* table, const double* d_freqs,
                         int64_t N, const pespace_model* model, double* d_out_AET, void* stream) {
  if (!d_params || !d_freqs || !d_out_AET || B <= 0 || N <= 0 || !model_ok(model) || !table_ok(table))
    return PESPACE_EINVAL;
  cudaStream_t st = (cudaStream_t)stream;
  const TabPlan p = make_tab_plan(B, N, model->n_det);
  if (p.ntile > 65535) return PESPACE_EINVAL;
  char* d_scratch = nullptr;
  CU(cudaMallocAsync((void**)&d_scratch, p.trig_bytes + p.consts_bytes, st));
  double2* d_trig = (double2*)d_scratch;
  double* d_consts = (double*)(d_scratch + p.trig_bytes);
  int rc = run_prep_tab(d_params, B, model, d_consts, d_trig, st);
  const TabC T = make_tab(table, model->mode_mask);
  const dim3 grid((unsigned)p.nbb, (unsigned)p.ntile);
  static SmemOptIn cfg0, cfg1;
  for (int d = 0; d < model->n_det && rc == PESPACE_OK; ++d) {
    const DetC dc = make_det(model->det[d]);
    cudaError_t e;
    if (dc.kind == 0) {
      e = opt_in(response_tab_kernel<0>, cfg0);
      if (e == cudaSuccess)
        response_tab_kernel<0><<<grid, BLOCK, tab_smem_bytes(), st>>>(d_consts, d_trig, B, T, table->d_fnodes, d_freqs, N,
                                                                      dc, model->n_det, d, (double2*)d_out_AET);
    } else {
      e = opt_in(response_tab_kernel<1>, cfg1);
      if (e == cudaSuccess)
        response_tab_kernel<1><<<grid, BLOCK, tab_smem_bytes(), st>>>(d_consts, d_trig, B, T, table->d_fnodes, d_freqs, N,
                                                                      dc, model->n_det, d, (double2*)d_out_AET);
    }
    ++g_launches;
    if (e == cudaSuccess) e = cudaGetLastError();
    if (e != cudaSuccess) rc = cuda_fail(e);
  }
  cudaError_t e = cudaFreeAsync(d_scratch, st);
  if (rc == PESPACE_OK && e != cudaSuccess) rc = cuda_fail(e);
  return rc;
}

int pespace_loglike_tab(const double* d_params, int64_t B, const pespace_wavetable* table, const double* d_data_AET,
                        const double* d_psd, const pespace_grid* grid, const pespace_model* model, double* d_out_lnL,
                        void* d_workspace, size_t workspace_bytes, void* stream) {
  if (!d_params || !d_data_AET || !d_psd || !d_out_lnL || !d_workspace || B <= 0 || !grid_ok(grid) ||
      !model_ok(model) || !table_ok(table))
    return PESPACE_EINVAL;
  if (workspace_bytes < pespace_workspace_bytes_tab(B, grid, model) || ((uintptr_t)d_workspace & 15u))
    return PESPACE_EINVAL;
  cudaStream_t st = (cudaStream_t)stream;
  const TabPlan p = make_tab_plan(B, grid->N, model->n_det);
  if (p.ntile > 65535) return PESPACE_EINVAL;
  char* ws = (char*)d_workspace;
  double2* d_trig = (double2*)ws;
  double* d_consts = (double*)(ws + p.trig_bytes);
  double* d_partial = (double*)(ws + p.trig_bytes + p.consts_bytes);
  double* d_bins = (double*)(ws + p.trig_bytes + p.consts_bytes + p.partial_bytes);
  double* d_wt = (double*)(ws + p.trig_bytes + p.consts_bytes + p.partial_bytes + p.bins_bytes);
  int rc = run_prep_tab(d_params, B, model, d_consts, d_trig, st);
  if (rc != PESPACE_OK) return rc;
  const GridC G = {grid->f0, grid->df, (long long)grid->N};
  const PrepArgs A = make_prep_args(model);
  const unsigned nb256 = (unsigned)((grid->N + 255) / 256);
  prep_bins_kernel<<<dim3(nb256, (unsigned)model->n_det), 256, 0, st>>>((const double2*)d_data_AET, d_psd, G, A, 0, d_bins);
  LAUNCHED();
  prep_tab_weights_kernel<<<nb256, 256, 0, st>>>(G, table->d_fnodes, table->K, d_wt);
  LAUNCHED();
  const TabC T = make_tab(table, model->mode_mask);
  const dim3 g((unsigned)p.nbb, (unsigned)p.ntile);
  static SmemOptIn cfg[2][3];
  const int v = T.n_modes == 1 ? 1 : T.n_modes == 5 ? 2 : 0;       // kernel variant: single mode, five modes unrolled, any
  for (int d = 0; d < model->n_det; ++d) {
    const DetC dc = make_det(model->det[d]);
    EvPair ev;
    if (int rc2 = prof_begin(ev, st); rc2 != PESPACE_OK) return rc2;
#define PESPACE_TAB_LAUNCH(KIND, V, NM)                                                                              \
    if (dc.kind == KIND && v == V) {                                                                                   \
      CU(opt_in(loglike_tab_kernel<KIND, NM>, cfg[KIND][V]));                                                          \
      loglike_tab_kernel<KIND, NM><<<g, BLOCK, tab_smem_bytes(), st>>>(d_consts, d_trig, B, T, d_bins, d_wt, G.N, dc,  \
                                                                       model->n_det, d, d_partial);                   \
    }
    PESPACE_TAB_LAUNCH(0, 0, 0) PESPACE_TAB_LAUNCH(0, 1, 1) PESPACE_TAB_LAUNCH(0, 2, 5)
    PESPACE_TAB_LAUNCH(1, 0, 0) PESPACE_TAB_LAUNCH(1, 1, 1) PESPACE_TAB_LAUNCH(1, 2, 5)
#undef PESPACE_TAB_LAUNCH
    LAUNCHED();
    if (int rc2 = prof_end(ev, st); rc2 != PESPACE_OK) return rc2;
  }
  combine_kernel<<<PESPACE_COMBINE_GRID(B), 0, st>>>(d_partial, d_consts, B, (int)(model->n_det * p.nbb),
                                                                p.stride, d_out_lnL);
  LAUNCHED();
  return PESPACE_OK;
}

}  // extern "C"
