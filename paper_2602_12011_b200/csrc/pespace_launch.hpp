// pespace_launch.hpp -- kernel launchers behind the C ABI.  The kernels are specialised at compile time on
// (detector kind, mode-class mask); the 2 x 15 instantiations of each entry point are spread over several
// translation units (pespace_inst_*.cu, one per entry point x kind x half of the masks) so that they
// compile in parallel.  Not part of the public ABI.
#pragma once
#include "pespace_host.hpp"
#include "pespace_fused.cuh"

namespace pespace {
namespace host {

using LoglikeFn = cudaError_t (*)(dim3, cudaStream_t, const double*, const double2*, long long, const double*,
                                  long long, const DetC&, int, int, double*);
using ResponseFn = cudaError_t (*)(dim3, cudaStream_t, const double*, const double2*, long long, const double*,
                                   long long, const DetC&, int, int, double2*);
using GradFn = cudaError_t (*)(dim3, cudaStream_t, const double*, const double2*, long long, const double*, long long,
                               const DetC&, int, int, double*);
using FusedFn = cudaError_t (*)(dim3, cudaStream_t, const double*, const double2*, long long, const double*, long long,
                                const DetSet&, int, double*);
using FusedResponseFn = cudaError_t (*)(dim3, cudaStream_t, const double*, const double2*, long long, const double*,
                                        long long, const DetSet&, int, double2*);
using FisherFn = cudaError_t (*)(dim3, cudaStream_t, const double*, long long, const double*, long long, const DetC&,
                                 int, int, int, double*);

// half 0: class masks 1..7, half 1: masks 8..15; each returns nullptr for a mask outside its half
#define PESPACE_DECLARE_INST(FN, name) \
  FN name##_k0_h0(unsigned cmask); FN name##_k0_h1(unsigned cmask); \
  FN name##_k1_h0(unsigned cmask); FN name##_k1_h1(unsigned cmask); \
  inline FN name(int kind, unsigned cmask) { \
    if (cmask < 1u || cmask > 15u) return nullptr; \
    if (kind == 0) return cmask < 8u ? name##_k0_h0(cmask) : name##_k0_h1(cmask); \
    return cmask < 8u ? name##_k1_h0(cmask) : name##_k1_h1(cmask); \
  }
PESPACE_DECLARE_INST(LoglikeFn, loglike_launcher)
PESPACE_DECLARE_INST(ResponseFn, response_launcher)
PESPACE_DECLARE_INST(FisherFn, fisher_launcher)
PESPACE_DECLARE_INST(GradFn, grad_launcher)
#undef PESPACE_DECLARE_INST
// fused multi-detector likelihood: specialised on the class mask only
FusedFn fused_launcher_h0(unsigned cmask);
FusedFn fused_launcher_h1(unsigned cmask);
inline FusedFn fused_launcher(unsigned cmask) {
  if (cmask < 1u || cmask > 15u) return nullptr;
  return cmask < 8u ? fused_launcher_h0(cmask) : fused_launcher_h1(cmask);
}
FusedResponseFn fused_response_launcher_h0(unsigned cmask);
FusedResponseFn fused_response_launcher_h1(unsigned cmask);
inline FusedResponseFn fused_response_launcher(unsigned cmask) {
  if (cmask < 1u || cmask > 15u) return nullptr;
  return cmask < 8u ? fused_response_launcher_h0(cmask) : fused_response_launcher_h1(cmask);
}

}  // namespace host
}  // namespace pespace
