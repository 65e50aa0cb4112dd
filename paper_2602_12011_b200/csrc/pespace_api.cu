// pespace_api.cu -- the C ABI of include/pespace.h: argument checks, workspace carving, launches.
#include "pespace_launch.hpp"

#include <mutex>
#include <vector>

using namespace pespace;
using namespace pespace::host;

namespace pespace {
namespace host {
std::atomic<long long> g_launches{0};
char* cuda_msg() {
  static thread_local char msg[256] = "";
  return msg;
}
}  // namespace host
}  // namespace pespace

namespace {

std::atomic<bool> g_profile{false};
constexpr size_t kMaxEvents = 65536;   // bound of the event list between two pespace_profile_read calls
std::vector<EvPair> g_events;
std::mutex g_ev_mutex;

struct Plan {
  int n_det, stride;
  long long nbb;          // bin blocks
  long long ntile;        // sample tiles
  size_t trig_bytes, consts_bytes, partial_bytes, bins_bytes;   // workspace: [trig table | per-bin table (likelihood
                                                                // only) | sample constants | block partials]
};
Plan make_plan(long long B, long long N, int n_det) {
  Plan p;
  p.n_det = n_det;
  p.stride = sample_stride(n_det);
  p.nbb = (N + BLOCK - 1) / BLOCK;
  p.ntile = (B + TILE - 1) / TILE;
  p.trig_bytes = align_up((size_t)NTAB * sizeof(double2), 256);
  p.consts_bytes = align_up((size_t)B * p.stride * sizeof(double), 256);
  p.partial_bytes = align_up((size_t)n_det * p.nbb * (size_t)B * sizeof(double), 256);
  p.bins_bytes = align_up((size_t)n_det * NBF * (size_t)N * sizeof(double), 256);
  return p;
}

int run_prep(const double* d_params, long long B, const pespace_model* model, double* d_consts, double2* d_trig,
             cudaStream_t st) {
  const PrepArgs A = make_prep_args(model);
  const int th = 128;
  prep_samples_kernel<<<(unsigned)((prep_threads(B, model->n_det) + th - 1) / th), th, 0, st>>>(d_params, B, A, d_consts,
                                                                                                d_trig);
  LAUNCHED();
  return PESPACE_OK;
}

}  // namespace

namespace pespace {
namespace host {
int prof_begin(EvPair& ev, cudaStream_t st) {
  ev = EvPair();
  if (!g_profile.load(std::memory_order_relaxed)) return PESPACE_OK;
  {
    std::lock_guard<std::mutex> lk(g_ev_mutex);
    if (g_events.size() >= kMaxEvents) return PESPACE_OK;
  }
  CU(cudaEventCreate(&ev.a));
  CU(cudaEventCreate(&ev.b));
  CU(cudaEventRecord(ev.a, st));
  return PESPACE_OK;
}
int prof_end(EvPair& ev, cudaStream_t st) {
  if (!ev.a) return PESPACE_OK;
  CU(cudaEventRecord(ev.b, st));
  std::lock_guard<std::mutex> lk(g_ev_mutex);
  g_events.push_back(ev);
  return PESPACE_OK;
}
}  // namespace host
}  // namespace pespace

extern "C" {

const char* pespace_version(void) { return "pespace-b200 0.1 (sm_100a, fp64)"; }

const char* pespace_strerror(int code) {
  switch (code) {
    case PESPACE_OK: return "ok";
    case PESPACE_EINVAL: return "invalid argument";
    case PESPACE_ECUDA: return cuda_msg()[0] ? cuda_msg() : "CUDA error";
    case PESPACE_ENOMEM: return "out of memory";
    case PESPACE_ETOOBIG: return cuda_msg()[0] ? cuda_msg() : "batch beyond the static scratch array";
    default: return "unknown error code";
  }
}

int64_t pespace_launch_count(void) { return (int64_t)g_launches.load(); }

int pespace_profile_enable(int on) {
  g_profile.store(on != 0);
  return PESPACE_OK;
}

int pespace_profile_read(double* h_main_ms, int64_t* h_launches) {
  std::lock_guard<std::mutex> lk(g_ev_mutex);
  double total = 0.0;
  int rc = PESPACE_OK;
  for (const EvPair& ev : g_events) {
    float ms = 0.f;
    cudaError_t e = cudaEventSynchronize(ev.b);
    if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, ev.a, ev.b);
    if (e != cudaSuccess) rc = cuda_fail(e);
    total += ms;
    cudaEventDestroy(ev.a);
    cudaEventDestroy(ev.b);
  }
  if (h_main_ms) *h_main_ms = total;
  if (h_launches) *h_launches = (int64_t)g_events.size();
  g_events.clear();
  return rc;
}

size_t pespace_workspace_bytes(int64_t B, const pespace_grid* grid, const pespace_model* model, int want_fisher) {
  if (B <= 0 || !grid_ok(grid) || !model_ok(model)) return 0;
  if (want_fisher) return fisher_workspace_bytes(B, grid->N, model->n_det);
  const Plan p = make_plan(B, grid->N, model->n_det);
  return p.trig_bytes + p.consts_bytes + p.partial_bytes + p.bins_bytes;
}

int pespace_response(const double* d_params, int64_t B, const double* d_freqs, int64_t N,
                     const pespace_model* model, double* d_out_AET, void* stream) {
  if (!d_params || !d_freqs || !d_out_AET || B <= 0 || N <= 0 || !model_ok(model)) return PESPACE_EINVAL;
  cudaStream_t st = (cudaStream_t)stream;
  const Plan p = make_plan(B, N, model->n_det);
  if (p.ntile > 65535) return PESPACE_EINVAL;                 // gridDim.y
  char* d_scratch = nullptr;
  CU(cudaMallocAsync((void**)&d_scratch, p.trig_bytes + p.consts_bytes, st));
  double2* d_trig = (double2*)d_scratch;
  double* d_consts = (double*)(d_scratch + p.trig_bytes);
  int rc = run_prep(d_params, B, model, d_consts, d_trig, st);
  if (rc == PESPACE_OK) {
    const unsigned cm = class_mask(model->mode_mask);
    if (model->n_det > 1) {
      // several detectors: ONE launch, S2/S3 evaluated once per (sample, bin) and shared (pespace_fused.cuh)
      DetSet D;
      std::memset(&D, 0, sizeof D);
      for (int d = 0; d < model->n_det; ++d) D.det[d] = make_det(model->det[d]);
      const long long ntile = (B + TILE_L - 1) / TILE_L;
      if (ntile > 65535) rc = PESPACE_EINVAL;
      if (rc == PESPACE_OK) {
        const dim3 grid((unsigned)p.nbb, (unsigned)ntile);
        cudaError_t e = fused_response_launcher(cm)(grid, st, d_consts, d_trig, B, d_freqs, N, D, model->n_det,
                                                    (double2*)d_out_AET);
        ++g_launches;
        if (e == cudaSuccess) e = cudaGetLastError();
        if (e != cudaSuccess) rc = cuda_fail(e);
      }
    } else {
      const dim3 grid((unsigned)p.nbb, (unsigned)p.ntile);
      const DetC dc = make_det(model->det[0]);
      cudaError_t e = response_launcher(dc.kind, cm)(grid, st, d_consts, d_trig, B, d_freqs, N, dc, 1, 0,
                                                     (double2*)d_out_AET);
      ++g_launches;
      if (e == cudaSuccess) e = cudaGetLastError();
      if (e != cudaSuccess) rc = cuda_fail(e);
    }
  }
  cudaError_t e = cudaFreeAsync(d_scratch, st);
  if (rc == PESPACE_OK && e != cudaSuccess) rc = cuda_fail(e);
  return rc;
}

int pespace_loglike(const double* d_params, int64_t B, const double* d_data_AET, const double* d_psd,
                    const pespace_grid* grid, const pespace_model* model, double* d_out_lnL,
                    void* d_workspace, size_t workspace_bytes, void* stream) {
  return pespace::host::loglike_impl(d_params, B, d_data_AET, d_psd, grid, model, d_out_lnL, d_workspace, workspace_bytes,
                                     stream, false);
}

int pespace_prepare(const double* d_data_AET, const double* d_psd, const pespace_grid* grid, const pespace_model* model,
                    void* d_workspace, size_t workspace_bytes, void* stream) {
  if (!d_data_AET || !d_psd || !d_workspace || !grid_ok(grid) || !model_ok(model)) return PESPACE_EINVAL;
  if (workspace_bytes < pespace_workspace_bytes(1, grid, model, 0) || ((uintptr_t)d_workspace & 15u)) return PESPACE_EINVAL;
  cudaStream_t st = (cudaStream_t)stream;
  const Plan p = make_plan(1, grid->N, model->n_det);
  double* d_bins = (double*)((char*)d_workspace + p.trig_bytes);
  const GridC G = {grid->f0, grid->df, (long long)grid->N};
  const PrepArgs A = make_prep_args(model);
  prep_bins_kernel<<<dim3((unsigned)((grid->N + 255) / 256), (unsigned)model->n_det), 256, 0, st>>>(
      (const double2*)d_data_AET, d_psd, G, A, 1, d_bins);
  LAUNCHED();
  return PESPACE_OK;
}

int pespace_loglike_prepared(const double* d_params, int64_t B, const pespace_grid* grid, const pespace_model* model,
                             double* d_out_lnL, void* d_workspace, size_t workspace_bytes, void* stream) {
  return pespace::host::loglike_impl(d_params, B, nullptr, nullptr, grid, model, d_out_lnL, d_workspace, workspace_bytes,
                                     stream, true);
}

}  // extern "C"

// pespace_loglike with one extra switch for the session calls: bins_ready = the per-bin table (S0) at the head of the
// workspace was written by an earlier call for the same data set, PSD, grid and model and is reused
int pespace::host::loglike_impl(const double* d_params, int64_t B, const double* d_data_AET, const double* d_psd,
                                const pespace_grid* grid, const pespace_model* model, double* d_out_lnL,
                                void* d_workspace, size_t workspace_bytes, void* stream, bool bins_ready) {
  if (!d_params || (!bins_ready && (!d_data_AET || !d_psd)) || !d_out_lnL || !d_workspace || B <= 0 || !grid_ok(grid) ||
      !model_ok(model))
    return PESPACE_EINVAL;
  if (workspace_bytes < pespace_workspace_bytes(B, grid, model, 0) || ((uintptr_t)d_workspace & 15u))
    return PESPACE_EINVAL;
  cudaStream_t st = (cudaStream_t)stream;
  const Plan p = make_plan(B, grid->N, model->n_det);
  if (p.ntile > 65535) return PESPACE_EINVAL;                 // gridDim.y
  double2* d_trig = (double2*)d_workspace;
  double* d_bins = (double*)((char*)d_workspace + p.trig_bytes);           // B-independent offset: reusable across calls
  double* d_consts = (double*)((char*)d_workspace + p.trig_bytes + p.bins_bytes);
  double* d_partial = (double*)((char*)d_workspace + p.trig_bytes + p.bins_bytes + p.consts_bytes);
  int rc = run_prep(d_params, B, model, d_consts, d_trig, st);
  if (rc != PESPACE_OK) return rc;
  const unsigned cm = class_mask(model->mode_mask);
  const GridC G = {grid->f0, grid->df, (long long)grid->N};
  if (!bins_ready) {
    // S0: per-bin table of this data set, once per call (once per data set through a session)
    const PrepArgs A = make_prep_args(model);
    const dim3 gb((unsigned)((grid->N + 255) / 256), (unsigned)model->n_det);
    prep_bins_kernel<<<gb, 256, 0, st>>>((const double2*)d_data_AET, d_psd, G, A, 1, d_bins);
    LAUNCHED();
  }
  int n_slices = (int)(model->n_det * p.nbb);
  if (model->n_det > 1) {
    // several detectors: ONE launch, the waveform part (S2/S3) evaluated once per (sample, bin) and shared (pespace_fused.cuh)
    DetSet D;
    std::memset(&D, 0, sizeof D);
    for (int d = 0; d < model->n_det; ++d) D.det[d] = make_det(model->det[d]);
    const long long ntile = (B + TILE_L - 1) / TILE_L;
    if (ntile > 65535) return PESPACE_EINVAL;
    const dim3 g((unsigned)p.nbb, (unsigned)ntile);
    EvPair ev;
    if (int rc2 = prof_begin(ev, st); rc2 != PESPACE_OK) return rc2;
    CU(fused_launcher(cm)(g, st, d_consts, d_trig, B, d_bins, G.N, D, model->n_det, d_partial));
    LAUNCHED();
    if (int rc2 = prof_end(ev, st); rc2 != PESPACE_OK) return rc2;
    n_slices = (int)p.nbb;
  } else {
    const dim3 g((unsigned)p.nbb, (unsigned)p.ntile);
    const DetC dc = make_det(model->det[0]);
    EvPair ev;
    if (int rc2 = prof_begin(ev, st); rc2 != PESPACE_OK) return rc2;
    CU(loglike_launcher(dc.kind, cm)(g, st, d_consts, d_trig, B, d_bins, G.N, dc, 1, 0, d_partial));
    LAUNCHED();
    if (int rc2 = prof_end(ev, st); rc2 != PESPACE_OK) return rc2;
  }
  combine_kernel<<<PESPACE_COMBINE_GRID(B), 0, st>>>(d_partial, d_consts, B, n_slices, p.stride, d_out_lnL);
  LAUNCHED();
  return PESPACE_OK;
}

extern "C" {

int pespace_fp64_peak(int mode, int iters, double* h_out_tflops, double* h_out_ms) {
  if (iters <= 0 || !h_out_tflops || mode < 0 || mode > 10) return PESPACE_EINVAL;
  int dev = 0, sms = 0;
  CU(cudaGetDevice(&dev));
  CU(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
  double *d_in = nullptr, *d_out = nullptr;
  CU(cudaMalloc((void**)&d_in, 64 * 8));
  CU(cudaMalloc((void**)&d_out, 8));
  CU(cudaMemset(d_in, 0, 64 * 8));          // all-zero operands: no overflow, full-rate DFMA
  cudaEvent_t e0, e1;
  CU(cudaEventCreate(&e0));
  CU(cudaEventCreate(&e1));
  const int blocks = sms * 8, threads = 256;
  auto go = [&](int n) {
    if (mode == 0) dfma_peak_kernel<false><<<blocks, threads>>>(n, d_in, d_out);
    else if (mode == 1) dfma_peak_kernel<true><<<blocks, threads>>>(n, d_in, d_out);
    else if (mode == 2) dmma_peak_kernel<8, 0><<<blocks, threads>>>(n, d_in, d_out);
    else if (mode == 3) dmma_peak_kernel<2, 0><<<blocks, threads>>>(n, d_in, d_out);
    else if (mode == 4) dmma_peak_kernel<8, 1><<<blocks, threads>>>(n, d_in, d_out);
    else if (mode == 5) dmma_peak_kernel<8, 4><<<blocks, threads>>>(n, d_in, d_out);
    else if (mode == 6) operand_probe_kernel<0><<<blocks, threads>>>(n, d_in, d_out);
    else if (mode == 7) operand_probe_kernel<1><<<blocks, threads>>>(n, d_in, d_out);
    else if (mode == 8) operand_probe_kernel<2><<<blocks, threads>>>(n, d_in, d_out);
    else if (mode == 9) operand_probe_kernel<3><<<blocks, threads>>>(n, d_in, d_out);
    else operand_probe_kernel<4><<<blocks, threads>>>(n, d_in, d_out);
    ++g_launches;
  };
  go(iters / 8 + 1);   // warm-up
  CU(cudaEventRecord(e0));
  go(iters);
  CU(cudaEventRecord(e1));
  CU(cudaEventSynchronize(e1));
  float ms = 0.f;
  CU(cudaEventElapsedTime(&ms, e0, e1));
  // per thread and iteration: modes 0, 1, 6, 7: 64 DFMAs; modes 2-5: 8 x NACC DMMAs of 256 FMAs per warp (8 per
  // thread) plus DFMA_MIX DFMAs per DMMA; modes 8-10: 128 FP32 FMAs
  const double fma_per_thread_iter = mode <= 1 ? 64.0 : mode == 2 ? 8.0 * 8 * 8 : mode == 3 ? 8.0 * 2 * 8
                                     : mode == 4 ? 8.0 * 8 * (8 + 1) : mode == 5 ? 8.0 * 8 * (8 + 4)
                                     : mode <= 7 ? 64.0 : 128.0;
  const double flops = 2.0 * fma_per_thread_iter * (double)iters * (double)blocks * (double)threads;
  *h_out_tflops = flops / (ms * 1e-3) / 1e12;
  if (h_out_ms) *h_out_ms = ms;
  cudaEventDestroy(e0); cudaEventDestroy(e1); cudaFree(d_in); cudaFree(d_out);
  return PESPACE_OK;
}

}  // extern "C"
