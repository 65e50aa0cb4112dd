// pespace_host.hpp -- host-side helpers shared by the translation units of libpespace.so
// (argument checks, detector constants, launch bookkeeping).  Not part of the public ABI.
#pragma once
#include "../../include/pespace.h"
#include "../../include/pespace_bench.h"
#include "pespace_device.cuh"

#include <atomic>
#include <cmath>
#include <cstdio>
#include <cstring>

namespace pespace {
namespace host {

extern std::atomic<long long> g_launches;
char* cuda_msg();   // thread-local message buffer behind pespace_strerror(PESPACE_ECUDA), 256 bytes

inline int cuda_fail(cudaError_t e) {
  snprintf(cuda_msg(), 256, "CUDA error: %s", cudaGetErrorString(e));
  return PESPACE_ECUDA;
}
#define CU(x) do { cudaError_t e_ = (x); if (e_ != cudaSuccess) return ::pespace::host::cuda_fail(e_); } while (0)
#define LAUNCHED() do { ++::pespace::host::g_launches; cudaError_t e_ = cudaGetLastError(); \
                        if (e_ != cudaSuccess) return ::pespace::host::cuda_fail(e_); } while (0)

inline bool model_ok(const pespace_model* m) {
  if (!m || !m->det || m->n_det < 1 || m->n_det > PESPACE_MAX_DET) return false;
  if ((m->mode_mask & 31u) == 0 || (m->mode_mask & ~31u) != 0) return false;
  for (int i = 0; i < m->n_det; ++i) {
    const pespace_detector& d = m->det[i];
    if (d.kind != 0 && d.kind != 1) return false;
    if (d.tdi_gen != 15 && d.tdi_gen != 20) return false;
    if (!(d.L_m > 0.0) || !std::isfinite(d.L_m)) return false;
    if (d.kind == 1 && !(d.period_s > 0.0)) return false;
  }
  return true;
}
inline bool grid_ok(const pespace_grid* g) {
  return g && g->N > 0 && g->df > 0.0 && g->f0 > 0.0 && std::isfinite(g->df) && std::isfinite(g->f0);
}

inline DetC make_det(const pespace_detector& d) {
  DetC c;
  std::memset(&c, 0, sizeof c);
  c.Lbar = d.L_m / kC;
  c.kind = d.kind; c.gen = d.tdi_gen;
  c.kappa = d.kappa; c.lambda0 = d.lambda0; c.period_s = d.period_s; c.lon = d.lon; c.lat = d.lat;
  c.yr_over_p = (d.kind == 1) ? kYear / d.period_s : 0.0;
  return c;
}

inline PrepArgs make_prep_args(const pespace_model* model) {
  PrepArgs A;
  std::memset(&A, 0, sizeof A);
  A.n_det = model->n_det;
  A.mode_mask = model->mode_mask;
  for (int i = 0; i < model->n_det; ++i) A.det[i] = make_det(model->det[i]);
  return A;
}

inline unsigned class_mask(unsigned mode_mask) {
  unsigned m = 0;
  if (mode_mask & PESPACE_MODE_21) m |= 1u;                       // m = 1
  if (mode_mask & (PESPACE_MODE_22 | PESPACE_MODE_32)) m |= 2u;   // m = 2
  if (mode_mask & PESPACE_MODE_33) m |= 4u;                       // m = 3
  if (mode_mask & PESPACE_MODE_44) m |= 8u;                       // m = 4
  return m;
}

inline size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

// Dynamic shared memory beyond 48 KB is an opt-in attribute of a kernel PER DEVICE: one flag per device ordinal
// (atomic: host threads may race to set it, setting it twice is harmless); ordinals >= 64 set it on every launch.
struct SmemOptIn { std::atomic<unsigned long long> done{0}; };
template <class K>
inline cudaError_t opt_in_smem(K kernel, size_t bytes, SmemOptIn& flag) {
  int dev = 0;
  if (cudaError_t e = cudaGetDevice(&dev); e != cudaSuccess) return e;
  const unsigned long long bit = (dev >= 0 && dev < 64) ? (1ull << dev) : 0ull;
  if (flag.done.load(std::memory_order_acquire) & bit) return cudaSuccess;
  const cudaError_t e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
  if (e == cudaSuccess) flag.done.fetch_or(bit, std::memory_order_release);
  return e;
}

// optional event timing of the dominant kernels (pespace_profile_enable / _read); defined in pespace_api.cu
struct EvPair { cudaEvent_t a = nullptr, b = nullptr; };
int prof_begin(EvPair& ev, cudaStream_t st);   // no-op unless profiling is enabled
int prof_end(EvPair& ev, cudaStream_t st);

// pespace_loglike with a switch for callers that keep the workspace between calls (pespace_session.cu): bins_ready =
// the per-bin table at the head of the workspace is still valid for this data set, PSD, grid and model
int loglike_impl(const double* d_params, int64_t B, const double* d_data_AET, const double* d_psd,
                 const pespace_grid* grid, const pespace_model* model, double* d_out_lnL, void* d_workspace,
                 size_t workspace_bytes, void* stream, bool bins_ready);

// pespace_loglike_grad with the same switch (pespace_grad.cu)
int loglike_grad_impl(const double* d_params, int64_t B, const double* d_data_AET, const double* d_psd,
                      const pespace_grid* grid, const pespace_model* model, double* d_out_lnL, double* d_out_grad,
                      void* d_workspace, size_t workspace_bytes, void* stream, bool bins_ready);

// Fisher path (pespace_fisher.cu)
size_t fisher_workspace_bytes(long long B, long long N, int n_det);

}  // namespace host
}  // namespace pespace
