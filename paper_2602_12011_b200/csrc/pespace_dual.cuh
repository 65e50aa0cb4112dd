// pespace_dual.cuh -- small forward-mode (dual-number) scalar for the device code of the Fisher
// path (Eq. 13; "forward mode").  Du<N> carries a value and N tangents.
// Used (a) with N = 7 in the per-sample constant kernel, where every constant is differentiated
// w.r.t. (M, q, chi1, chi2, iota, lambda, beta), and (b) with N = 3 in the per-bin geometry stage of
// fisher_kernel, directions (orbit time, lambda, beta).
#pragma once
#include <cuda_runtime.h>

namespace pespace {

template <int N>
struct Du {
  double v;
  double d[N];
  __host__ __device__ __forceinline__ Du() {}
  __host__ __device__ __forceinline__ Du(double x) : v(x) {
#pragma unroll
    for (int i = 0; i < N; ++i) d[i] = 0.0;
  }
};

template <int N> __device__ __forceinline__ Du<N> operator+(const Du<N>& a, const Du<N>& b) {
  Du<N> r; r.v = a.v + b.v;
#pragma unroll
  for (int i = 0; i < N; ++i) r.d[i] = a.d[i] + b.d[i];
  return r;
}
template <int N> __device__ __forceinline__ Du<N> operator-(const Du<N>& a, const Du<N>& b) {
  Du<N> r; r.v = a.v - b.v;
#pragma unroll
  for (int i = 0; i < N; ++i) r.d[i] = a.d[i] - b.d[i];
  return r;
}
template <int N> __device__ __forceinline__ Du<N> operator-(const Du<N>& a) {
  Du<N> r; r.v = -a.v;
#pragma unroll
  for (int i = 0; i < N; ++i) r.d[i] = -a.d[i];
  return r;
}
template <int N> __device__ __forceinline__ Du<N> operator*(const Du<N>& a, const Du<N>& b) {
  Du<N> r; r.v = a.v * b.v;
#pragma unroll
  for (int i = 0; i < N; ++i) r.d[i] = fma(a.v, b.d[i], a.d[i] * b.v);
  return r;
}
template <int N> __device__ __forceinline__ Du<N> operator+(const Du<N>& a, double s) { Du<N> r = a; r.v += s; return r; }
template <int N> __device__ __forceinline__ Du<N> operator+(double s, const Du<N>& a) { return a + s; }
template <int N> __device__ __forceinline__ Du<N> operator-(const Du<N>& a, double s) { Du<N> r = a; r.v -= s; return r; }
template <int N> __device__ __forceinline__ Du<N> operator-(double s, const Du<N>& a) { return (-a) + s; }
template <int N> __device__ __forceinline__ Du<N> operator*(const Du<N>& a, double s) {
  Du<N> r; r.v = a.v * s;
#pragma unroll
  for (int i = 0; i < N; ++i) r.d[i] = a.d[i] * s;
  return r;
}
template <int N> __device__ __forceinline__ Du<N> operator*(double s, const Du<N>& a) { return a * s; }
// chain rule: f(a) with f'(a) = df
template <int N> __device__ __forceinline__ Du<N> chain(const Du<N>& a, double fv, double df) {
  Du<N> r; r.v = fv;
#pragma unroll
  for (int i = 0; i < N; ++i) r.d[i] = df * a.d[i];
  return r;
}
template <int N> __device__ __forceinline__ Du<N> operator/(const Du<N>& a, const Du<N>& b) {
  const double ib = 1.0 / b.v;
  Du<N> r; r.v = a.v * ib;
#pragma unroll
  for (int i = 0; i < N; ++i) r.d[i] = (a.d[i] - r.v * b.d[i]) * ib;
  return r;
}
template <int N> __device__ __forceinline__ Du<N> operator/(const Du<N>& a, double s) { return a * (1.0 / s); }
template <int N> __device__ __forceinline__ Du<N> operator/(double s, const Du<N>& b) { return Du<N>(s) / b; }
// a*b + c
template <int N> __device__ __forceinline__ Du<N> dfma(const Du<N>& a, const Du<N>& b, const Du<N>& c) {
  Du<N> r; r.v = fma(a.v, b.v, c.v);
#pragma unroll
  for (int i = 0; i < N; ++i) r.d[i] = fma(a.v, b.d[i], fma(a.d[i], b.v, c.d[i]));
  return r;
}
// s*b + c with a plain-double multiplier
template <int N> __device__ __forceinline__ Du<N> dfma(double s, const Du<N>& b, const Du<N>& c) {
  Du<N> r; r.v = fma(s, b.v, c.v);
#pragma unroll
  for (int i = 0; i < N; ++i) r.d[i] = fma(s, b.d[i], c.d[i]);
  return r;
}

// elementary functions, double and Du overloads under one name
__device__ __forceinline__ double p_sqrt(double x) { return sqrt(x); }
__device__ __forceinline__ double p_cbrt(double x) { return cbrt(x); }
__device__ __forceinline__ double p_log(double x) { return log(x); }
__device__ __forceinline__ double p_sin(double x) { return sin(x); }
__device__ __forceinline__ double p_cos(double x) { return cos(x); }
__device__ __forceinline__ double p_val(double x) { return x; }
template <int N> __device__ __forceinline__ Du<N> p_sqrt(const Du<N>& a) {
  const double s = sqrt(a.v);
  return chain(a, s, 0.5 / s);
}
template <int N> __device__ __forceinline__ Du<N> p_cbrt(const Du<N>& a) {
  const double c = cbrt(a.v);
  return chain(a, c, c / (3.0 * a.v));
}
template <int N> __device__ __forceinline__ Du<N> p_log(const Du<N>& a) { return chain(a, log(a.v), 1.0 / a.v); }
template <int N> __device__ __forceinline__ Du<N> p_sin(const Du<N>& a) { return chain(a, sin(a.v), cos(a.v)); }
template <int N> __device__ __forceinline__ Du<N> p_cos(const Du<N>& a) { return chain(a, cos(a.v), -sin(a.v)); }
template <int N> __device__ __forceinline__ double p_val(const Du<N>& a) { return a.v; }

}  // namespace pespace
