// pespace_fused.cuh -- the likelihood kernel for models with several detectors: ONE launch, the waveform part shared.
//
// SURVEY.md 8(a) marks S2 (mode amplitude and phase) and S3 (t_lm) "shared by detectors": they depend on the sample,
// the bin and the mode class only.  loglike_kernel (pespace_device.cuh) is launched once per detector and re-evaluates
// them every time.  Here a thread evaluates, per (sample, bin), S2/S3 of every class of the mask ONCE into registers
// (psi, tau, CKp, CKc: 4 doubles per class), then walks the detectors: per detector it loads the 11 per-bin numbers of
// that detector (sin / cos 2 pi f L, folded data, weights; L1 hits after the first sample of the tile), runs S4-S7 of
// every class on the cached waveform scalars (eval_geom, the code of the per-detector kernel), forms the residual and
// adds the weighted square to ONE accumulator.  One warp reduction and one partial per (sample, block) instead of
// n_det; a three-detector single-theta call is one launch instead of three.
//
// The detector kind is a run-time property here (both eval_geom<0> and eval_geom<1> bodies are in the kernel, selected
// by a block-uniform branch), the class mask stays a compile-time parameter.  Sum order: classes inside a detector,
// detectors in model order, then the fixed warp / block / combine tree: deterministic, but not the order of the
// per-detector kernels (results differ from them in the last bits).
#pragma once
#include "pespace_device.cuh"

namespace pespace {

struct DetSet { DetC det[8]; };

#ifndef PESPACE_FTILE_L
#define PESPACE_FTILE_L 64
#endif
constexpr int TILE_L = PESPACE_FTILE_L;        // samples per block (the staged constants hold every detector's block);
                                               // config 4: 332.2 ms per step with 64, 334.1 with 32

__host__ __device__ constexpr size_t fused_smem_bytes(int n_det) {
  return sizeof(double) * ((size_t)2 * NTAB + (size_t)TILE_L * sample_stride(n_det) + (size_t)(BLOCK / 32) * TILE_L);
}
__host__ __device__ constexpr size_t fused_response_smem_bytes(int n_det) {
  return sizeof(double) * ((size_t)2 * NTAB + (size_t)TILE_L * sample_stride(n_det));
}

// S2/S3 of class m = MC + 1 (the first half of eval_class): phase psi (pu, reduced), tau = kTurn (t_lm - t_c) / yr and
// the amplitudes of the two polarisation contents
template <int MC>
__device__ __forceinline__ void eval_wave(const BinC& bc, const double* __restrict__ sc, double va, double La, double ftc,
                                          double& psi, double& tau, double& CKp, double& CKc) {
  constexpr double CB[4] = {1.2599210498948731648, 1.0, 0.87358046473629886905, 0.79370052598409973738};
  constexpr double LN3[4] = {0.23104906018664843647, 0.0, -0.13515503603605479399, -0.23104906018664843647};
  constexpr double S83[4] = {0.1574901312368591456, 1.0, 2.948334068485008683, 6.349604207872797899};
  constexpr double MH[4] = {0.5, 1.0, 1.5, 2.0};
  const double v = (MC == 1) ? va : va * CB[MC];
  const double L = (MC == 1) ? La : La + LN3[MC];
  const double v2 = v * v;
  double P = fma(sc[W_P7], v, fma(sc[W_P6L], L, sc[W_P6]));
  P = fma(P, v, fma(sc[W_P5L], L, sc[W_P5]));
  P = fma(P, v, sc[W_P4]);
  P = fma(P, v, sc[W_P3]);
  P = fma(P, v, sc[W_P2]);
  P = fma(P, v2, sc[W_P0]);
  double Q = fma(sc[W_Q7], v, fma(sc[W_Q6L], L, sc[W_Q6]));
  Q = fma(Q, v, sc[W_Q5]);
  Q = fma(Q, v, sc[W_Q4]);
  Q = fma(Q, v, sc[W_Q3]);
  Q = fma(Q, v, sc[W_Q2]);
  Q = fma(Q, v2, sc[W_Q0]);
  psi = ((MC == 1) ? bc.fm53 : S83[MC] * bc.fm53) * P;
  psi -= whole_turns(psi);
  psi += fma(MH[MC], sc[W_PH0], ftc);
  tau = ((MC == 1) ? bc.fm83 : S83[MC] * bc.fm83) * Q;
  const double* ka = sc + W_KA + 4 * MC;
  if (MC == 1) { CKp = fma(ka[1], v2, ka[0]); CKc = fma(ka[3], v2, ka[2]); }
  else if (MC == 3) { CKp = v2 * ka[0]; CKc = v2 * ka[2]; }
  else { CKp = v * ka[0]; CKc = v * ka[2]; }
}

// S4-S7 of every class of CMASK for one detector from the cached waveform scalars; scd = the sample's constants shifted
// so that this detector's block sits where eval_geom expects it (eval_geom reads detector-block offsets only)
template <int KIND, unsigned CMASK>
__device__ __forceinline__ void geom_classes(const BinC& bc, const double* __restrict__ scd, const DetC& dc,
                                             const double2* __restrict__ tab, const double (&psi)[4],
                                             const double (&tau)[4], const double (&CKp)[4], const double (&CKc)[4],
                                             double (&S)[6]) {
  constexpr bool c0 = CMASK & 1u, c1 = CMASK & 2u, c2 = CMASK & 4u, c3 = CMASK & 8u;
  if (c0) eval_geom<KIND, true, true>(bc, scd, dc, tab, psi[0], tau[0], CKp[0], CKc[0], S);
  if (c1) eval_geom<KIND, !c0, true>(bc, scd, dc, tab, psi[1], tau[1], CKp[1], CKc[1], S);
  if (c2) eval_geom<KIND, !(c0 || c1), true>(bc, scd, dc, tab, psi[2], tau[2], CKp[2], CKc[2], S);
  if (c3) eval_geom<KIND, !(c0 || c1 || c2), true>(bc, scd, dc, tab, psi[3], tau[3], CKp[3], CKc[3], S);
}

template <unsigned CMASK>
__global__ void __launch_bounds__(BLOCK, 1)
loglike_fused_kernel(const double* __restrict__ consts, const double2* __restrict__ trig, long long B,
                     const double* __restrict__ bins /* [n_det][NBF][N] */, long long N, DetSet D, int n_det,
                     double* __restrict__ partial /* [gridDim.x][B] */) {
  double2* tab = reinterpret_cast<double2*>(pespace_dyn_smem);
  double* smem = reinterpret_cast<double*>(tab + NTAB);
  const int stride = sample_stride(n_det);
  double (*red)[TILE_L] = reinterpret_cast<double (*)[TILE_L]>(smem + TILE_L * stride);
  const long long b0 = (long long)blockIdx.y * TILE_L;
  const int ns = (int)min((long long)TILE_L, B - b0);
  stage_trig(tab, trig);
  for (int i = threadIdx.x; i < ns * stride; i += BLOCK) smem[i] = consts[b0 * stride + i];   // contiguous samples
  const long long k = (long long)blockIdx.x * BLOCK + threadIdx.x;
  const bool live = k < N;
  const size_t kk = (size_t)(live ? k : N - 1);
  BinC bc;                                   // the detector-independent part of the per-bin record (from detector 0's)
  bc.fT = bins[BF_FT * N + kk]; bc.cf = bins[BF_CF * N + kk]; bc.lnf3 = bins[BF_LNF3 * N + kk];
  bc.fm53 = bins[BF_FM53 * N + kk]; bc.fm83 = bins[BF_FM83 * N + kk]; bc.fm76 = 0.0; bc.sth = 0.0; bc.cth = 1.0;
  __syncthreads();
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  for (int s = 0; s < ns; ++s) {
    const double* sc = smem + s * stride;
    const double ftc = mul_mod_turn(bc.fT, sc[W_TC]);
    const double va = sc[W_A] * bc.cf, La = bc.lnf3;
    double psi[4], tau[4], CKp[4], CKc[4];
    if (CMASK & 1u) eval_wave<0>(bc, sc, va, La, ftc, psi[0], tau[0], CKp[0], CKc[0]);
    if (CMASK & 2u) eval_wave<1>(bc, sc, va, La, ftc, psi[1], tau[1], CKp[1], CKc[1]);
    if (CMASK & 4u) eval_wave<2>(bc, sc, va, La, ftc, psi[2], tau[2], CKp[2], CKc[2]);
    if (CMASK & 8u) eval_wave<3>(bc, sc, va, La, ftc, psi[3], tau[3], CKp[3], CKc[3]);
    double acc = 0.0;
#pragma unroll 1
    for (int d = 0; d < n_det; ++d) {
      const double* bp = bins + (size_t)d * NBF * (size_t)N + kk;
      BinC bd = bc;
      bd.sth = bp[BF_STH * N]; bd.cth = bp[BF_CTH * N];
      const DetC& dc = D.det[d];
      const double* scd = sc + D_STRIDE * d;
      double S[6];
      if (dc.kind == 0) geom_classes<0, CMASK>(bd, scd, dc, tab, psi, tau, CKp, CKc, S);
      else geom_classes<1, CMASK>(bd, scd, dc, tab, psi, tau, CKp, CKc, S);
      const double Ar = S[4] - S[0], Ai = S[5] - S[1];
      const double Er_ = S[0] - 2.0 * S[2] + S[4], Ei_ = S[1] - 2.0 * S[3] + S[5];
      const double Tr = S[0] + S[2] + S[4], Ti = S[1] + S[3] + S[5];
      double r0 = bp[(BF_DR + 0) * N] - Ar, r1 = bp[(BF_DI + 0) * N] - Ai;
      acc = fma(live ? bp[(BF_W + 0) * N] : 0.0, fma(r0, r0, r1 * r1), acc);
      r0 = bp[(BF_DR + 1) * N] - Er_; r1 = bp[(BF_DI + 1) * N] - Ei_;
      acc = fma(live ? bp[(BF_W + 1) * N] : 0.0, fma(r0, r0, r1 * r1), acc);
      r0 = bp[(BF_DR + 2) * N] - Tr; r1 = bp[(BF_DI + 2) * N] - Ti;
      acc = fma(live ? bp[(BF_W + 2) * N] : 0.0, fma(r0, r0, r1 * r1), acc);
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
    if (lane == 0) red[warp][s] = acc;
  }
  __syncthreads();
  if (threadIdx.x < ns) {
    double t = 0.0;
#pragma unroll
    for (int wv = 0; wv < BLOCK / 32; ++wv) t += red[wv][threadIdx.x];
    partial[(size_t)blockIdx.x * (size_t)B + (size_t)(b0 + threadIdx.x)] = t;
  }
}

// pespace_response for models with several detectors: the same sharing for the response arrays.  The frequency array is
// arbitrary here, so the per-bin record is computed in the prologue (make_bin); its detector-dependent part (sin / cos
// 2 pi f L and the TDI prefactor g z f^{-7/6}, four doubles per detector) is kept per thread in local memory (L1) and
// read back once per (sample, detector).
template <unsigned CMASK>
__global__ void __launch_bounds__(BLOCK, 1)
response_fused_kernel(const double* __restrict__ consts, const double2* __restrict__ trig, long long B,
                      const double* __restrict__ freqs, long long N, DetSet D, int n_det,
                      double2* __restrict__ out /* [B][n_det][3][N] */) {
  double2* tab = reinterpret_cast<double2*>(pespace_dyn_smem);
  double* smem = reinterpret_cast<double*>(tab + NTAB);
  const int stride = sample_stride(n_det);
  const long long b0 = (long long)blockIdx.y * TILE_L;
  const int ns = (int)min((long long)TILE_L, B - b0);
  stage_trig(tab, trig);
  for (int i = threadIdx.x; i < ns * stride; i += BLOCK) smem[i] = consts[b0 * stride + i];
  const long long k = (long long)blockIdx.x * BLOCK + threadIdx.x;
  const bool live = k < N;
  const double fraw = freqs[live ? k : N - 1];
  const bool pos = fraw > 0.0;
  const BinC bc = make_bin(pos ? fraw : 1.0, D.det[0].Lbar);
  double pb[PESPACE_MAX_DET][4];                       // sin, cos 2 pi f L_d; prefactor (re, im)
  for (int d = 0; d < n_det; ++d) {
    BinC bd = bc;
    sincospi(2.0 * (pos ? fraw : 1.0) * D.det[d].Lbar, &bd.sth, &bd.cth);
    pb[d][0] = bd.sth; pb[d][1] = bd.cth;
    tdi_prefactor(bd, D.det[d].gen, pb[d][2], pb[d][3]);
    if (!pos) { pb[d][2] = 0.0; pb[d][3] = 0.0; }     // f <= 0: zeros (the body runs on f = 1 and is finite)
  }
  __syncthreads();
  const double i2 = 0.70710678118654752440, i6 = 0.40824829046386301637, i3 = 0.57735026918962576451;
  for (int s = 0; s < ns; ++s) {
    const double* sc = smem + s * stride;
    const double ftc = mul_mod_turn(bc.fT, sc[W_TC]);
    const double va = sc[W_A] * bc.cf, La = bc.lnf3;
    double psi[4], tau[4], CKp[4], CKc[4];
    if (CMASK & 1u) eval_wave<0>(bc, sc, va, La, ftc, psi[0], tau[0], CKp[0], CKc[0]);
    if (CMASK & 2u) eval_wave<1>(bc, sc, va, La, ftc, psi[1], tau[1], CKp[1], CKc[1]);
    if (CMASK & 4u) eval_wave<2>(bc, sc, va, La, ftc, psi[2], tau[2], CKp[2], CKc[2]);
    if (CMASK & 8u) eval_wave<3>(bc, sc, va, La, ftc, psi[3], tau[3], CKp[3], CKc[3]);
    const bool valid = sc[W_VALID] != 0.0;
#pragma unroll 1
    for (int d = 0; d < n_det; ++d) {
      BinC bd = bc;
      bd.sth = pb[d][0]; bd.cth = pb[d][1];
      const double gr = pb[d][2], gi = pb[d][3];
      const DetC& dc = D.det[d];
      const double* scd = sc + D_STRIDE * d;
      double S[6];
      if (dc.kind == 0) geom_classes<0, CMASK>(bd, scd, dc, tab, psi, tau, CKp, CKc, S);
      else geom_classes<1, CMASK>(bd, scd, dc, tab, psi, tau, CKp, CKc, S);
      double ch[6];                                    // S holds (Re, -Im)
      ch[0] = (S[4] - S[0]) * i2; ch[1] = (S[1] - S[5]) * i2;
      ch[2] = (S[0] - 2.0 * S[2] + S[4]) * i6; ch[3] = -(S[1] - 2.0 * S[3] + S[5]) * i6;
      ch[4] = (S[0] + S[2] + S[4]) * i3; ch[5] = -(S[1] + S[3] + S[5]) * i3;
      if (!live) continue;
      double2* o = out + ((size_t)(b0 + s) * n_det + d) * 3 * (size_t)N + (size_t)k;
      if (valid) {                                     // block-uniform
#pragma unroll
        for (int c = 0; c < 3; ++c)
          o[c * N] = make_double2(fma(ch[2 * c], gr, -ch[2 * c + 1] * gi), fma(ch[2 * c], gi, ch[2 * c + 1] * gr));
      } else {
        o[0] = o[N] = o[2 * N] = make_double2(CUDART_NAN, CUDART_NAN);
      }
    }
  }
}

}  // namespace pespace
