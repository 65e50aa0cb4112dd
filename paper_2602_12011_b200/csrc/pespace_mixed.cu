// pespace_mixed.cu -- pespace_loglike_mixed of include/pespace.h: the mixed-precision likelihood.
#include "pespace_host.hpp"
#include "pespace_mixed.cuh"

using namespace pespace;
using namespace pespace::host;

extern "C" int pespace_loglike_mixed(const double* d_params, int64_t B, const double* d_data_AET, const double* d_psd,
                                     const pespace_grid* grid, const pespace_model* model, double* d_out_lnL,
                                     void* d_workspace, size_t workspace_bytes, void* stream) {
  if (!d_params || !d_data_AET || !d_psd || !d_out_lnL || !d_workspace || B <= 0 || !grid_ok(grid) ||
      !model_ok(model))
    return PESPACE_EINVAL;
  if (workspace_bytes < pespace_workspace_bytes(B, grid, model, 0) || ((uintptr_t)d_workspace & 15u))
    return PESPACE_EINVAL;
  cudaStream_t st = (cudaStream_t)stream;
  // same workspace layout as pespace_loglike: [trig table | sample constants | block partials | per-bin table]
  const int n_det = model->n_det, stride = sample_stride(n_det);
  const long long N = grid->N, nbb = (N + BLOCK - 1) / BLOCK, ntile = (B + MIX_TILE - 1) / MIX_TILE;
  if (ntile > 65535) return PESPACE_EINVAL;
  const size_t trig_bytes = align_up((size_t)NTAB * sizeof(double2), 256);
  const size_t consts_bytes = align_up((size_t)B * stride * sizeof(double), 256);
  const size_t partial_bytes = align_up((size_t)n_det * nbb * (size_t)B * sizeof(double), 256);
  char* ws = (char*)d_workspace;
  double2* d_trig = (double2*)ws;
  double* d_consts = (double*)(ws + trig_bytes);
  double* d_partial = (double*)(ws + trig_bytes + consts_bytes);
  double* d_bins = (double*)(ws + trig_bytes + consts_bytes + partial_bytes);
  const PrepArgs A = make_prep_args(model);
  const int th = 128;
  prep_samples_kernel<<<(unsigned)((prep_threads(B, n_det) + th - 1) / th), th, 0, st>>>(d_params, B, A, d_consts, d_trig);
  LAUNCHED();
  const GridC G = {grid->f0, grid->df, N};
  prep_bins_kernel<<<dim3((unsigned)((N + 255) / 256), (unsigned)n_det), 256, 0, st>>>((const double2*)d_data_AET, d_psd, G,
                                                                                     A, 2, d_bins);
  LAUNCHED();
  const unsigned cm = class_mask(model->mode_mask);
  const dim3 g((unsigned)nbb, (unsigned)ntile);
  static SmemOptIn cfg[2][3];
  const int v = cm == 2u ? 1 : cm == 15u ? 2 : 0;       // kernel variant: mask 2 / mask 15 unrolled, else run-time loop
  for (int d = 0; d < n_det; ++d) {
    const DetC dc = make_det(model->det[d]);
    EvPair ev;
    if (int rc = prof_begin(ev, st); rc != PESPACE_OK) return rc;
#define PESPACE_MIX_LAUNCH(KIND, V, CM)                                                                            \
    if (dc.kind == KIND && v == V) {                                                                                 \
      CU(opt_in_smem(loglike_mixed_kernel<KIND, CM>, mixed_smem_bytes(), cfg[KIND][V]));                             \
      loglike_mixed_kernel<KIND, CM><<<g, BLOCK, mixed_smem_bytes(), st>>>(d_consts, d_trig, B, cm, d_bins, N, dc,   \
                                                                           n_det, d, d_partial);                    \
    }
    PESPACE_MIX_LAUNCH(0, 0, 0u) PESPACE_MIX_LAUNCH(0, 1, 2u) PESPACE_MIX_LAUNCH(0, 2, 15u)
    PESPACE_MIX_LAUNCH(1, 0, 0u) PESPACE_MIX_LAUNCH(1, 1, 2u) PESPACE_MIX_LAUNCH(1, 2, 15u)
#undef PESPACE_MIX_LAUNCH
    LAUNCHED();
    if (int rc = prof_end(ev, st); rc != PESPACE_OK) return rc;
  }
  combine_kernel<<<PESPACE_COMBINE_GRID(B), 0, st>>>(d_partial, d_consts, B, (int)(n_det * nbb), stride, d_out_lnL);
  LAUNCHED();
  return PESPACE_OK;
}
