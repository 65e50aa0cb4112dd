// pespace_inst.cuh -- body of the pespace_inst_*.cu translation units.  The including file defines
//   PESPACE_INST_WHAT  0 likelihood, 1 response, 2 Fisher, 3 adjoint gradient, 4 fused multi-detector likelihood,
//                      5 fused multi-detector response (4, 5: kind unused)
//   PESPACE_INST_KIND  0 heliocentric, 1 geocentric
//   PESPACE_INST_HALF  0 class masks 1..7, 1 class masks 8..15
#include "pespace_launch.hpp"
#if PESPACE_INST_WHAT == 2
#include "pespace_fisher.cuh"
#endif
#if PESPACE_INST_WHAT == 3
#include "pespace_grad.cuh"
#endif
#if PESPACE_INST_WHAT == 4 || PESPACE_INST_WHAT == 5
#include "pespace_fused.cuh"
#endif

namespace pespace {
namespace host {
namespace {

// the kernels use dynamic shared memory beyond 48 KB: opt in once per instantiation and device (opt_in_smem)

#if PESPACE_INST_WHAT == 0
template <int KIND, unsigned CM>
cudaError_t launch(dim3 g, cudaStream_t st, const double* consts, const double2* trig, long long B,
                   const double* bins, long long N, const DetC& dc, int n_det, int det, double* partial) {
  static SmemOptIn configured;
  if (cudaError_t e = opt_in_smem(loglike_kernel<KIND, CM>, kernel_smem_bytes(), configured); e != cudaSuccess) return e;
  loglike_kernel<KIND, CM><<<g, BLOCK, kernel_smem_bytes(), st>>>(consts, trig, B, bins, N, dc, n_det, det, partial);
  return cudaSuccess;
}
using Fn = LoglikeFn;
#elif PESPACE_INST_WHAT == 1
template <int KIND, unsigned CM>
cudaError_t launch(dim3 g, cudaStream_t st, const double* consts, const double2* trig, long long B,
                   const double* freqs, long long N, const DetC& dc, int n_det, int det, double2* out) {
  static SmemOptIn configured;
  if (cudaError_t e = opt_in_smem(response_kernel<KIND, CM>, kernel_smem_bytes(), configured); e != cudaSuccess) return e;
  response_kernel<KIND, CM><<<g, BLOCK, kernel_smem_bytes(), st>>>(consts, trig, B, freqs, N, dc, n_det, det, out);
  return cudaSuccess;
}
using Fn = ResponseFn;
#elif PESPACE_INST_WHAT == 4
template <int KIND, unsigned CM>
cudaError_t launch(dim3 g, cudaStream_t st, const double* consts, const double2* trig, long long B,
                   const double* bins, long long N, const DetSet& D, int n_det, double* partial) {
  // the dynamic shared-memory size depends on n_det: opt in for the largest model
  static SmemOptIn configured;
  if (cudaError_t e = opt_in_smem(loglike_fused_kernel<CM>, fused_smem_bytes(PESPACE_MAX_DET), configured); e != cudaSuccess)
    return e;
  loglike_fused_kernel<CM><<<g, BLOCK, fused_smem_bytes(n_det), st>>>(consts, trig, B, bins, N, D, n_det, partial);
  return cudaSuccess;
}
using Fn = FusedFn;
#elif PESPACE_INST_WHAT == 5
template <int KIND, unsigned CM>
cudaError_t launch(dim3 g, cudaStream_t st, const double* consts, const double2* trig, long long B,
                   const double* freqs, long long N, const DetSet& D, int n_det, double2* out) {
  static SmemOptIn configured;
  if (cudaError_t e = opt_in_smem(response_fused_kernel<CM>, fused_response_smem_bytes(PESPACE_MAX_DET), configured);
      e != cudaSuccess)
    return e;
  response_fused_kernel<CM><<<g, BLOCK, fused_response_smem_bytes(n_det), st>>>(consts, trig, B, freqs, N, D, n_det, out);
  return cudaSuccess;
}
using Fn = FusedResponseFn;
#elif PESPACE_INST_WHAT == 3
template <int KIND, unsigned CM>
cudaError_t launch(dim3 g, cudaStream_t st, const double* consts, const double2* trig, long long B,
                   const double* bins, long long N, const DetC& dc, int n_det, int det, double* partial) {
  static SmemOptIn configured;
  if (cudaError_t e = opt_in_smem(loglike_grad_kernel<KIND, CM>, grad_smem_bytes(CM), configured); e != cudaSuccess) return e;
  loglike_grad_kernel<KIND, CM><<<g, BLOCK, grad_smem_bytes(CM), st>>>(consts, trig, B, bins, N, dc, n_det, det, partial);
  return cudaSuccess;
}
using Fn = GradFn;
#else
template <int KIND, unsigned CM>
cudaError_t launch(dim3 g, cudaStream_t st, const double* consts, long long B, const double* bins, long long N,
                   const DetC& dc, int n_det, int det, int grad_only, double* partial) {
  static SmemOptIn configured;
  if (cudaError_t e = opt_in_smem(fisher_kernel<KIND, CM>, fisher_smem_bytes(), configured); e != cudaSuccess) return e;
  fisher_kernel<KIND, CM><<<g, FBLOCK, fisher_smem_bytes(), st>>>(consts, B, bins, N, dc, n_det, det, grad_only, partial);
  return cudaSuccess;
}
using Fn = FisherFn;
#endif

constexpr int K = PESPACE_INST_KIND;
#if PESPACE_INST_HALF == 0
const Fn kTable[8] = {nullptr, launch<K, 1>, launch<K, 2>, launch<K, 3>, launch<K, 4>, launch<K, 5>, launch<K, 6>,
                      launch<K, 7>};
constexpr unsigned kBase = 0;
#else
const Fn kTable[8] = {launch<K, 8>, launch<K, 9>, launch<K, 10>, launch<K, 11>, launch<K, 12>, launch<K, 13>,
                      launch<K, 14>, launch<K, 15>};
constexpr unsigned kBase = 8;
#endif

}  // namespace

#define PESPACE_CAT_(a, b, c, d, e) a##b##c##d##e
#define PESPACE_CAT(a, b, c, d, e) PESPACE_CAT_(a, b, c, d, e)
#if PESPACE_INST_WHAT == 0
#define PESPACE_INST_NAME PESPACE_CAT(loglike_launcher_k, PESPACE_INST_KIND, _h, PESPACE_INST_HALF, )
#elif PESPACE_INST_WHAT == 1
#define PESPACE_INST_NAME PESPACE_CAT(response_launcher_k, PESPACE_INST_KIND, _h, PESPACE_INST_HALF, )
#elif PESPACE_INST_WHAT == 4
#define PESPACE_INST_NAME PESPACE_CAT(fused_launcher_h, PESPACE_INST_HALF, , , )
#elif PESPACE_INST_WHAT == 5
#define PESPACE_INST_NAME PESPACE_CAT(fused_response_launcher_h, PESPACE_INST_HALF, , , )
#elif PESPACE_INST_WHAT == 3
#define PESPACE_INST_NAME PESPACE_CAT(grad_launcher_k, PESPACE_INST_KIND, _h, PESPACE_INST_HALF, )
#else
#define PESPACE_INST_NAME PESPACE_CAT(fisher_launcher_k, PESPACE_INST_KIND, _h, PESPACE_INST_HALF, )
#endif

Fn PESPACE_INST_NAME(unsigned cmask) {
  return (cmask - kBase < 8u) ? kTable[cmask - kBase] : nullptr;   // unsigned wrap-around rejects cmask < kBase
}

}  // namespace host
}  // namespace pespace
