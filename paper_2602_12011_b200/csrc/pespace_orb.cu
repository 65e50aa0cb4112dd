// pespace_orb.cu -- pespace_response_orb / pespace_loglike_orb of include/pespace.h: response and likelihood with
// tabulated numerical orbits.
#include "pespace_host.hpp"
#include "pespace_orb.cuh"

using namespace pespace;
using namespace pespace::host;

namespace {

struct OrbPlan {
  int stride;
  long long nbb, ntile;
  size_t trig_bytes, bins_bytes, consts_bytes, partial_bytes;   // workspace layout of pespace_loglike
};
OrbPlan make_orb_plan(long long B, long long N, int n_det) {
  OrbPlan p;
  p.stride = sample_stride(n_det);
  p.nbb = (N + BLOCK - 1) / BLOCK;
  p.ntile = (B + TAB_TILE - 1) / TAB_TILE;
  p.trig_bytes = align_up((size_t)NTAB * sizeof(double2), 256);
  p.bins_bytes = align_up((size_t)n_det * NBF * (size_t)N * sizeof(double), 256);
  p.consts_bytes = align_up((size_t)B * p.stride * sizeof(double), 256);
  p.partial_bytes = align_up((size_t)n_det * p.nbb * (size_t)B * sizeof(double), 256);
  return p;
}

bool orbit_ok(const pespace_orbittable* o) {
  return o && o->K >= 2 && o->d_pos && o->d_vel && o->dt > 0.0 && std::isfinite(o->dt) && std::isfinite(o->t0);
}
OrbC make_orb(const pespace_orbittable* o, int det) {
  OrbC O;
  O.K = o->K;
  O.dt = o->dt;
  O.ts = (kYear / kTurn) / o->dt;
  O.pos = o->d_pos + (size_t)det * (size_t)o->K * 9;
  O.vel = o->d_vel + (size_t)det * (size_t)o->K * 9;
  return O;
}
int run_prep_orb(const double* d_params, long long B, const pespace_model* model, const pespace_orbittable* o,
                 double* d_consts, double2* d_trig, cudaStream_t st) {
  const PrepArgs A = make_prep_args(model);
  const OrbPrep P = {o->t0, o->dt};
  prep_samples_orb_kernel<<<(unsigned)((prep_threads(B) + 127) / 128), 128, 0, st>>>(d_params, B, A, P, d_consts, d_trig);
  LAUNCHED();
  return PESPACE_OK;
}
SmemOptIn g_cfg_resp[3], g_cfg_like[3];
// kernel variant of a class mask: 1 -> mask 2 unrolled, 2 -> mask 15 unrolled, 0 -> run-time loop
int variant_of(unsigned cm) { return cm == 2u ? 1 : cm == 15u ? 2 : 0; }

}  // namespace

extern "C" {

int pespace_response_orb(const double* d_params, int64_t B, const pespace_orbittable* orbit, const double* d_freqs,
                         int64_t N, const pespace_model* model, double* d_out_AET, void* stream) {
  if (!d_params || !d_freqs || !d_out_AET || B <= 0 || N <= 0 || !model_ok(model) || !orbit_ok(orbit))
    return PESPACE_EINVAL;
  cudaStream_t st = (cudaStream_t)stream;
  const OrbPlan p = make_orb_plan(B, N, model->n_det);
  if (p.ntile > 65535) return PESPACE_EINVAL;
  char* d_scratch = nullptr;
  CU(cudaMallocAsync((void**)&d_scratch, p.trig_bytes + p.consts_bytes, st));
  double2* d_trig = (double2*)d_scratch;
  double* d_consts = (double*)(d_scratch + p.trig_bytes);
  int rc = run_prep_orb(d_params, B, model, orbit, d_consts, d_trig, st);
  const unsigned cm = class_mask(model->mode_mask);
  const dim3 grid((unsigned)p.nbb, (unsigned)p.ntile);
  for (int d = 0; d < model->n_det && rc == PESPACE_OK; ++d) {
    const DetC dc = make_det(model->det[d]);
    cudaError_t e = cudaSuccess;
    const OrbC O = make_orb(orbit, d);
#define PESPACE_ORB_RESP(V, CM)                                                                                       \
    if (variant_of(cm) == V) {                                                                                          \
      e = opt_in_smem(response_orb_kernel<CM>, tab_smem_bytes(), g_cfg_resp[V]);                                        \
      if (e == cudaSuccess)                                                                                             \
        response_orb_kernel<CM><<<grid, BLOCK, tab_smem_bytes(), st>>>(d_consts, d_trig, B, cm, O, d_freqs, N, dc,      \
                                                                       model->n_det, d, (double2*)d_out_AET);          \
    }
    PESPACE_ORB_RESP(0, 0u) PESPACE_ORB_RESP(1, 2u) PESPACE_ORB_RESP(2, 15u)
#undef PESPACE_ORB_RESP
    ++g_launches;
    if (e == cudaSuccess) e = cudaGetLastError();
    if (e != cudaSuccess) rc = cuda_fail(e);
  }
  cudaError_t e = cudaFreeAsync(d_scratch, st);
  if (rc == PESPACE_OK && e != cudaSuccess) rc = cuda_fail(e);
  return rc;
}

int pespace_loglike_orb(const double* d_params, int64_t B, const pespace_orbittable* orbit, const double* d_data_AET,
                        const double* d_psd, const pespace_grid* grid, const pespace_model* model, double* d_out_lnL,
                        void* d_workspace, size_t workspace_bytes, void* stream) {
  if (!d_params || !d_data_AET || !d_psd || !d_out_lnL || !d_workspace || B <= 0 || !grid_ok(grid) ||
      !model_ok(model) || !orbit_ok(orbit))
    return PESPACE_EINVAL;
  if (workspace_bytes < pespace_workspace_bytes(B, grid, model, 0) || ((uintptr_t)d_workspace & 15u))
    return PESPACE_EINVAL;
  cudaStream_t st = (cudaStream_t)stream;
  const OrbPlan p = make_orb_plan(B, grid->N, model->n_det);
  if (p.ntile > 65535) return PESPACE_EINVAL;
  char* ws = (char*)d_workspace;
  double2* d_trig = (double2*)ws;
  double* d_bins = (double*)(ws + p.trig_bytes);
  double* d_consts = (double*)(ws + p.trig_bytes + p.bins_bytes);
  double* d_partial = (double*)(ws + p.trig_bytes + p.bins_bytes + p.consts_bytes);
  int rc = run_prep_orb(d_params, B, model, orbit, d_consts, d_trig, st);
  if (rc != PESPACE_OK) return rc;
  const GridC G = {grid->f0, grid->df, (long long)grid->N};
  const PrepArgs A = make_prep_args(model);
  prep_bins_kernel<<<dim3((unsigned)((grid->N + 255) / 256), (unsigned)model->n_det), 256, 0, st>>>(
      (const double2*)d_data_AET, d_psd, G, A, 1, d_bins);
  LAUNCHED();
  const unsigned cm = class_mask(model->mode_mask);
  const dim3 g((unsigned)p.nbb, (unsigned)p.ntile);
  for (int d = 0; d < model->n_det; ++d) {
    const DetC dc = make_det(model->det[d]);
    EvPair ev;
    if (int rc2 = prof_begin(ev, st); rc2 != PESPACE_OK) return rc2;
    const OrbC O = make_orb(orbit, d);
#define PESPACE_ORB_LIKE(V, CM)                                                                                       \
    if (variant_of(cm) == V) {                                                                                          \
      CU(opt_in_smem(loglike_orb_kernel<CM>, tab_smem_bytes(), g_cfg_like[V]));                                         \
      loglike_orb_kernel<CM><<<g, BLOCK, tab_smem_bytes(), st>>>(d_consts, d_trig, B, cm, O, d_bins, G.N, dc,           \
                                                                 model->n_det, d, d_partial);                          \
    }
    PESPACE_ORB_LIKE(0, 0u) PESPACE_ORB_LIKE(1, 2u) PESPACE_ORB_LIKE(2, 15u)
#undef PESPACE_ORB_LIKE
    LAUNCHED();
    if (int rc2 = prof_end(ev, st); rc2 != PESPACE_OK) return rc2;
  }
  combine_kernel<<<PESPACE_COMBINE_GRID(B), 0, st>>>(d_partial, d_consts, B, (int)(model->n_det * p.nbb), p.stride,
                                                    d_out_lnL);
  LAUNCHED();
  return PESPACE_OK;
}

}  // extern "C"
