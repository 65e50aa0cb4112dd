// pespace_noalloc.cu -- pespace_response_noalloc of include/pespace.h: the detector response for callers that cannot
// call cudaMalloc (code under CUDA graph capture, tight serving loops, harnesses that forbid allocation).
//
// pespace_response needs scratch memory for step S1 -- the per-sample constants [B][40 + 24 n_det] doubles and the
// 1024-entry sine / cosine table -- and takes it from cudaMallocAsync / cudaFreeAsync on every call.  This twin keeps
// that scratch in ONE file-scope device array of PESPACE_NOALLOC_SCRATCH_BYTES (1 MiB; every GPU that loads the library
// holds it until the process exits) and launches the SAME kernels on it: prep_samples_kernel, then response_kernel
// (one detector) or response_fused_kernel (several).  It calls no cudaMalloc, cudaFree or allocating library routine.
//
// The array's name is a host-side stand-in in host code, not a device address: the address the kernels get comes from
// cudaGetSymbolAddress, taken once per device with that device current (scratch_of below).
//
// Every call shares the array and finds the last call's contents in it.  Nothing has to start at zero: the prep
// kernel of a call writes every word the response kernels of that call read (all 40 + 24 n_det constants of every
// sample b < B, out-of-domain samples included, and the whole table) before they are launched on the same stream.
// Two calls that overlap on the GPU (different streams, or different host threads on different streams) RACE on the
// array; calls on one stream are ordered and safe.
#include "pespace_launch.hpp"

#include <mutex>

using namespace pespace;
using namespace pespace::host;

static __device__ __align__(256) unsigned char pespace_noalloc_scratch[PESPACE_NOALLOC_SCRATCH_BYTES];

namespace {

constexpr int kMaxDevices = 64;
std::mutex g_scratch_mutex;
void* g_scratch_ptr[kMaxDevices] = {nullptr};

// device address of the scratch array on the CURRENT device (looked up once per device)
int scratch_of(unsigned char** out) {
  int dev = -1;
  CU(cudaGetDevice(&dev));
  if (dev < 0 || dev >= kMaxDevices) {
    snprintf(cuda_msg(), 256, "pespace_response_noalloc: device ordinal %d beyond %d", dev, kMaxDevices - 1);
    return PESPACE_ECUDA;
  }
  std::lock_guard<std::mutex> lock(g_scratch_mutex);
  if (!g_scratch_ptr[dev]) {
    void* p = nullptr;
    CU(cudaGetSymbolAddress(&p, pespace_noalloc_scratch));
    if (!p) return PESPACE_ECUDA;
    g_scratch_ptr[dev] = p;
  }
  *out = static_cast<unsigned char*>(g_scratch_ptr[dev]);
  return PESPACE_OK;
}

size_t trig_bytes() { return align_up((size_t)NTAB * sizeof(double2), 256); }

}  // namespace

extern "C" {

size_t pespace_noalloc_scratch_needed(int64_t B, const pespace_model* model) {
  if (B <= 0 || !model_ok(model)) return 0;
  return trig_bytes() + align_up((size_t)B * (size_t)sample_stride(model->n_det) * sizeof(double), 256);
}

int pespace_response_noalloc(const double* d_params, int64_t B, const double* d_freqs, int64_t N,
                             const pespace_model* model, double* d_out_AET, void* stream) {
  if (!d_params || !d_freqs || !d_out_AET || B <= 0 || N <= 0 || !model_ok(model)) return PESPACE_EINVAL;
  const size_t need = pespace_noalloc_scratch_needed(B, model);
  if (need > (size_t)PESPACE_NOALLOC_SCRATCH_BYTES) {
    snprintf(cuda_msg(), 256,
             "pespace_response_noalloc: B = %lld samples x %d detector(s) need %zu bytes of scratch, the static array "
             "holds %zu (use pespace_response, or split the batch)",
             (long long)B, (int)model->n_det, need, (size_t)PESPACE_NOALLOC_SCRATCH_BYTES);
    return PESPACE_ETOOBIG;
  }
  const long long nbb = (N + BLOCK - 1) / BLOCK;
  unsigned char* scratch = nullptr;
  if (int rc = scratch_of(&scratch); rc != PESPACE_OK) return rc;
  cudaStream_t st = (cudaStream_t)stream;
  double2* d_trig = reinterpret_cast<double2*>(scratch);
  double* d_consts = reinterpret_cast<double*>(scratch + trig_bytes());
  const PrepArgs A = make_prep_args(model);
  prep_samples_kernel<<<(unsigned)((prep_threads(B, model->n_det) + 127) / 128), 128, 0, st>>>(d_params, B, A, d_consts,
                                                                                             d_trig);
  LAUNCHED();
  const unsigned cm = class_mask(model->mode_mask);
  if (model->n_det > 1) {
    DetSet D;
    std::memset(&D, 0, sizeof D);
    for (int d = 0; d < model->n_det; ++d) D.det[d] = make_det(model->det[d]);
    const long long ntile = (B + TILE_L - 1) / TILE_L;
    if (ntile > 65535) return PESPACE_EINVAL;                 // gridDim.y (cannot happen within the scratch limit)
    CU(fused_response_launcher(cm)(dim3((unsigned)nbb, (unsigned)ntile), st, d_consts, d_trig, B, d_freqs, N, D,
                                   model->n_det, (double2*)d_out_AET));
    LAUNCHED();
  } else {
    const long long ntile = (B + TILE - 1) / TILE;
    if (ntile > 65535) return PESPACE_EINVAL;
    const DetC dc = make_det(model->det[0]);
    CU(response_launcher(dc.kind, cm)(dim3((unsigned)nbb, (unsigned)ntile), st, d_consts, d_trig, B, d_freqs, N, dc, 1, 0,
                                      (double2*)d_out_AET));
    LAUNCHED();
  }
  return PESPACE_OK;
}

}  // extern "C"
