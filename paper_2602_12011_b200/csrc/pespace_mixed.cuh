// pespace_mixed.cuh -- mixed-precision likelihood (the paper's float32 mode for searches and
// coarse maximisation).  What stays FP64: every phase that enters an exponential -- the PN phase
// polynomial, 2 pi f t_c, the Doppler phase of the guiding centre, the sum psi + 2 pi f k.x_n and its reduction
// modulo one turn (phases reach 1e6..1e8 rad; FP32 has 7 digits).  What runs in FP32: the t_lm polynomial, the
// orbit angle, the projections and arm weights, the sine/cosine of the REDUCED phases, the brackets, TDI sums,
// A/E/T and the residual.  Data and template are whitened per bin and channel (r_c = sqrt(w_c) (d_c - h_c)) and the
// amplitudes carry a fixed scale 2^64, so that every FP32 quantity is of order 1e-3..1e3 for detector-like inputs
// (|sqrt(4 df / S_n) h| between ~1e-19 x 2^64 and 1e19 x 2^64 overflow / underflow is NOT detected).
// Accuracy: ~1e-6 relative on h (measured against the oracle in tests/test_gpu_mixed.py), i.e. NOT a substitute for
// pespace_loglike in parameter estimation of SNR ~ 1e3 signals; throughput: DESIGN.md 8c.
#pragma once
#include "pespace_device.cuh"

namespace pespace {

constexpr float kAmpScale = 18446744073709551616.0f;    // 2^64: amplitudes x this, sqrt(w) / this
constexpr float kMagicF = 12582912.0f;                  // 1.5 * 2^23: rounds |x| < 2^22 to an integer

__constant__ double kMixCB[4] = {1.2599210498948731648, 1.0, 0.87358046473629886905, 0.79370052598409973738};
__constant__ double kMixLN3[4] = {0.23104906018664843647, 0.0, -0.13515503603605479399, -0.23104906018664843647};
__constant__ double kMixS83[4] = {0.1574901312368591456, 1.0, 2.948334068485008683, 6.349604207872797899};

// sin, cos of a phase a (pu, |a| < 2^22) in FP32 from the float table: first-order sine and second-order cosine
// correction of the remainder |y| <= 1/2 pu (theta <= 3.1e-3: the dropped terms are < 5e-9)
__device__ __forceinline__ void sincos_f(float y, int j, const float2* __restrict__ tabf, float& s, float& c) {
  const float2 T = tabf[j & (NTAB - 1)];
  const float sl = y * (float)kRadPerPu;
  const float cl = -0.5f * sl * sl;
  s = fmaf(T.y, sl, fmaf(T.x, cl, T.x));
  c = fmaf(-T.x, sl, fmaf(T.y, cl, T.y));
}
__device__ __forceinline__ void sincos_pu_f(float a, const float2* __restrict__ tabf, float& s, float& c) {
  const float t = a + kMagicF;
  sincos_f(a - (t - kMagicF), __float_as_int(t), tabf, s, c);
}

// One mode class of one (sample, bin, detector): adds X, Y, Z (whitening and per-bin factor excluded) to S (FP32).
//   sc: FP64 constants (phase polynomial), sf: FP32 copy of the same block with the amplitudes scaled by 2^64
template <int KIND>
__device__ __forceinline__ void eval_class_mixed(int MC, bool first, double fT, double cf, double lnf3, double fm53,
                                                 float fm83f, float sthf, float cthf, float omcf, float fTLf,
                                                 const double* __restrict__ sc, const float* __restrict__ sf,
                                                 const DetC& dc, const float2* __restrict__ tabf,
                                                 const float2* __restrict__ tabm1, double va, double ftc,
                                                 float (&S)[6]) {
  // ---- S2: phase, FP64
  const double v = va * kMixCB[MC];
  const double L = lnf3 + kMixLN3[MC];
  const double v2 = v * v;
  double P = fma(sc[W_P7], v, fma(sc[W_P6L], L, sc[W_P6]));
  P = fma(P, v, fma(sc[W_P5L], L, sc[W_P5]));
  P = fma(P, v, sc[W_P4]);
  P = fma(P, v, sc[W_P3]);
  P = fma(P, v, sc[W_P2]);
  P = fma(P, v2, sc[W_P0]);
  double psi = (kMixS83[MC] * fm53) * P;
  psi -= whole_turns(psi);
  psi += fma(0.5 * (double)(MC + 1), sc[W_PH0], ftc);
  // ---- S3: t_lm, FP32
  const float vf = (float)v, Lf = (float)L, v2f = vf * vf;
  float Q = fmaf(sf[W_Q7], vf, fmaf(sf[W_Q6L], Lf, sf[W_Q6]));
  Q = fmaf(Q, vf, sf[W_Q5]);
  Q = fmaf(Q, vf, sf[W_Q4]);
  Q = fmaf(Q, vf, sf[W_Q3]);
  Q = fmaf(Q, vf, sf[W_Q2]);
  Q = fmaf(Q, v2f, sf[W_Q0]);
  const float tau = ((float)kMixS83[MC] * fm83f) * Q;
  const float* ka = sf + W_KA + 4 * MC;
  float CKp, CKc;
  if (MC == 1) { CKp = fmaf(ka[1], v2f, ka[0]); CKc = fmaf(ka[3], v2f, ka[2]); }
  else if (MC == 3) { CKp = v2f * ka[0]; CKc = v2f * ka[2]; }
  else { CKp = vf * ka[0]; CKc = vf * ka[2]; }
  // ---- S4: orbit, FP32
  float G1k, G2k, G1u, G2u, G1v, G2v, cD, sD;      // cD, sD: cos, sin of the guiding-centre (Earth) angle
  if (KIND == 0) {
    float sa, ca;
    sincos_pu_f(sf[D_BASE] + tau, tabf, sa, ca);
    const float c2 = fmaf(2.0f * ca, ca, -1.0f), s2 = 2.0f * sa * ca;
    const float* w = sf + S_K;
    G1k = fmaf(w[0], c2, fmaf(w[1], s2, fmaf(w[2], ca, w[3])));
    G2k = fmaf(w[0], s2, fmaf(-w[1], c2, fmaf(w[2], sa, w[4])));
    w = sf + S_U;
    G1u = fmaf(w[0], c2, fmaf(w[1], s2, fmaf(w[2], ca, w[3])));
    G2u = fmaf(w[0], s2, fmaf(-w[1], c2, fmaf(w[2], sa, w[4])));
    w = sf + S_V;
    G1v = fmaf(w[0], c2, fmaf(w[1], s2, fmaf(w[2], ca, w[3])));
    G2v = fmaf(w[0], s2, fmaf(-w[1], c2, fmaf(w[2], sa, w[4])));
    cD = ca; sD = sa;
  } else {
    float sp, cp;
    sincos_pu_f(sf[D_BASE] + tau, tabf, sD, cD);
    sincos_pu_f(fmaf(tau, (float)dc.yr_over_p, sf[D_BASE + 1]), tabf, sp, cp);
    const float* w = sf + D_BASE + 2;
    G1k = fmaf(w[0], cp, w[1] * sp); G2k = fmaf(w[1], cp, -w[0] * sp);
    G1u = fmaf(w[2], cp, w[3] * sp); G2u = fmaf(w[3], cp, -w[2] * sp);
    G1v = fmaf(w[4], cp, w[5] * sp); G2v = fmaf(w[5], cp, -w[4] * sp);
  }
  constexpr float R3H = 0.86602540378443864676f;
  const float tk = R3H * G2k;
  const float nun[3] = {G1k, fmaf(-0.5f, G1k, tk), fmaf(-0.5f, G1k, -tk)};
  const float ka_ = tk + tk, kb_ = fmaf(-1.5f, G1k, -tk), kc_ = fmaf(1.5f, G1k, -tk);
  const float tu = R3H * G2u, tv = R3H * G2v;
  const float ul[3] = {tu + tu, fmaf(-1.5f, G1u, -tu), fmaf(1.5f, G1u, -tu)};
  const float vl[3] = {tv + tv, fmaf(-1.5f, G1v, -tv), fmaf(1.5f, G1v, -tv)};
  // ---- S5: arm weights, FP32
  float Wr[3], Wi[3];
#pragma unroll
  for (int l = 0; l < 3; ++l) {
    const float uu = ul[l], vv = vl[l];
    const float v2_ = vv * vv;
    const float D = fmaf(uu, uu, v2_);
    float rD;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(rD) : "f"(D));        // MUFU.RCP, ~1 ulp
    rD = (D > 0.0f) ? rD : 0.0f;
    Wr[l] = (CKp * rD) * fmaf(uu, uu, -v2_);
    Wi[l] = (CKc * rD) * (uu * vv);
  }
  // ---- S6: exponentials relative to the guiding centre.  E_n = E_c (1 + delta_n), E_c = exp(-i base) with the
  // large phase base = psi + kTurn f k.x_centre reduced in FP64 (Doppler phase of the centre from the FP64 constants),
  // delta_n = exp(-i a_n) - 1 with the arm-scale phase a_n = kTurn f L k.(x_n - x_centre)/L, |a_n| < 1 turn, in FP32
  // from the (sin, cos - 1) table: at low frequency a_n -> 0 and the brackets below are differences of O(2 pi f L)
  // quantities, which this form evaluates without cancelling against 1 (FP32 would lose 1 / (2 pi f L) digits).
  const double kR = fma(sc[S_DX], (double)cD, sc[S_DY] * (double)sD);
  const double ub = fma(fT, kR, psi);
  const double tb = ub + kMagic;
  float sb, cb;
  sincos_f((float)(ub - (tb - kMagic)), __double2loint(tb), tabf, sb, cb);
  float dC[3], dS[3];                 // cos a_n - 1, sin a_n
#pragma unroll
  for (int n = 0; n < 3; ++n) {
    const float a = fTLf * nun[n];
    const float t = a + kMagicF;
    const float y = a - (t - kMagicF);
    const float2 T = tabm1[__float_as_int(t) & (NTAB - 1)];        // (sin, cos - 1) of the node
    const float sl = y * (float)kRadPerPu, cl = -0.5f * sl * sl, Ty = 1.0f + T.y;
    dS[n] = fmaf(Ty, sl, fmaf(T.x, cl, T.x));
    dC[n] = fmaf(-T.x, sl, fmaf(Ty, cl, T.y));
  }
  // ---- S7: brackets in the centre frame, B'(r,s,kap) = kap (delta_s - cos(th) delta_r + (1 - cos th)) - i sin(th) (1 + delta_r)
  float Sc[6];
  auto add = [&](float& Sr, float& Si, int r, int s_, float kap, float wr, float wi, bool init) {
    const float br = fmaf(kap, fmaf(-cthf, dC[r], dC[s_]) + omcf, -sthf * dS[r]);
    const float bi = fmaf(kap, fmaf(-cthf, dS[r], dS[s_]), fmaf(sthf, dC[r], sthf));
    if (init) {
      Sr = fmaf(wr, br, -wi * bi);
      Si = fmaf(wr, bi, wi * br);
    } else {
      Sr = fmaf(wr, br, fmaf(-wi, bi, Sr));
      Si = fmaf(wr, bi, fmaf(wi, br, Si));
    }
  };
  add(Sc[0], Sc[1], 0, 2, -kb_, Wr[1], Wi[1], true);
  add(Sc[0], Sc[1], 0, 1, kc_, -Wr[2], -Wi[2], false);
  add(Sc[2], Sc[3], 1, 0, -kc_, Wr[2], Wi[2], true);
  add(Sc[2], Sc[3], 1, 2, ka_, -Wr[0], -Wi[0], false);
  add(Sc[4], Sc[5], 2, 1, -ka_, Wr[0], Wi[0], true);
  add(Sc[4], Sc[5], 2, 0, kb_, -Wr[1], -Wi[1], false);
  // back to the SSB frame: (Sr - i Si) (cb - i sb)
#pragma unroll
  for (int c = 0; c < 3; ++c) {
    const float xr = fmaf(Sc[2 * c], cb, -Sc[2 * c + 1] * sb), xi = fmaf(Sc[2 * c], sb, Sc[2 * c + 1] * cb);
    if (first) { S[2 * c] = xr; S[2 * c + 1] = xi; }
    else { S[2 * c] += xr; S[2 * c + 1] += xi; }
  }
}

// dynamic shared memory: [float2 (sin, cos) table | float2 (sin, cos - 1) table | FP64 sample constants | FP32 copy |
// warp partials]
constexpr int MIX_TILE = 64;
constexpr size_t mixed_smem_used() {
  return 2 * sizeof(float2) * NTAB + sizeof(double) * (size_t)MIX_TILE * SMEM_STRIDE +
         sizeof(float) * (size_t)MIX_TILE * SMEM_STRIDE + sizeof(double) * (size_t)(BLOCK / 32) * MIX_TILE;
}
constexpr size_t mixed_smem_bytes() { return mixed_smem_used(); }

#ifndef PESPACE_MINBX
#define PESPACE_MINBX 2
#endif
// CMASK != 0: the classes of that mask unrolled at compile time (the masks of configs 2-4); 0: any mask, run-time loop
template <int KIND, unsigned CMASK>
__global__ void __launch_bounds__(BLOCK, PESPACE_MINBX)
loglike_mixed_kernel(const double* __restrict__ consts, const double2* __restrict__ trig, long long B, unsigned cmask,
                     const double* __restrict__ bins /* [n_det][NBF][N], built with fold mode 2 */, long long N, DetC dc,
                     int n_det, int det, double* __restrict__ partial /* [n_det][gridDim.x][B] */) {
  float2* tabf = reinterpret_cast<float2*>(pespace_dyn_smem);
  float2* tabm1 = tabf + NTAB;
  double* smem = reinterpret_cast<double*>(tabm1 + NTAB);
  float* smf = reinterpret_cast<float*>(smem + MIX_TILE * SMEM_STRIDE);
  double (*red)[MIX_TILE] = reinterpret_cast<double (*)[MIX_TILE]>(smf + MIX_TILE * SMEM_STRIDE);
  const long long b0 = (long long)blockIdx.y * MIX_TILE;
  for (int i = threadIdx.x; i < NTAB; i += blockDim.x) {
    const double2 T = trig[i];
    tabf[i] = make_float2((float)T.x, (float)T.y);
    // cos - 1 = -sin^2 / (1 + cos) where cos > 0, formed in FP64 so that the float keeps full relative accuracy
    tabm1[i] = make_float2((float)T.x, (float)(T.y > 0.0 ? -T.x * T.x / (1.0 + T.y) : T.y - 1.0));
  }
  stage_tile(smem, consts, b0, B, n_det, det);
  __syncthreads();
  for (int i = threadIdx.x; i < MIX_TILE * SMEM_STRIDE; i += blockDim.x) {
    const int j = i % SMEM_STRIDE;
    double x = smem[i];
    if (j >= W_KA && j < W_KA + 16) x *= (double)kAmpScale;       // amplitudes carry the 2^64 scale
    smf[i] = (float)x;
  }
  const long long k = (long long)blockIdx.x * BLOCK + threadIdx.x;
  const bool live = k < N;
  const double* bp = bins + (size_t)det * NBF * (size_t)N + (size_t)(live ? k : N - 1);
  const double fT = bp[BF_FT * N], cf = bp[BF_CF * N], lnf3 = bp[BF_LNF3 * N], fm53 = bp[BF_FM53 * N];
  const float fm83f = (float)bp[BF_FM83 * N], sthf = (float)bp[BF_STH * N], cthf = (float)bp[BF_CTH * N];
  const float fTLf = (float)(fT * dc.Lbar);
  const double sth = bp[BF_STH * N], cth = bp[BF_CTH * N];
  const float omcf = (float)(cth > 0.0 ? sth * sth / (1.0 + cth) : 1.0 - cth);     // 1 - cos(2 pi f L), no cancellation
  float dr[3], di[3], sw[3];
#pragma unroll
  for (int c = 0; c < 3; ++c) {
    dr[c] = (float)bp[(BF_DR + c) * N]; di[c] = (float)bp[(BF_DI + c) * N];
    sw[c] = live ? (float)bp[(BF_W + c) * N] : 0.0f;
    if (!live) { dr[c] = 0.0f; di[c] = 0.0f; }
  }
  __syncthreads();
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int ns = (int)min((long long)MIX_TILE, B - b0);
  for (int s = 0; s < ns; ++s) {
    const double* sc = smem + s * SMEM_STRIDE;
    const float* sf = smf + s * SMEM_STRIDE;
    const double ftc = mul_mod_turn(fT, sc[W_TC]);
    const double va = sc[W_A] * cf;
    float S[6];
    if constexpr (CMASK != 0u) {
#define PESPACE_MIX_CLASS(MC)                                                                                    \
      if constexpr ((CMASK >> MC) & 1u)                                                                            \
        eval_class_mixed<KIND>(MC, !(CMASK & ((1u << MC) - 1u)), fT, cf, lnf3, fm53, fm83f, sthf, cthf, omcf, fTLf, sc, sf, \
                               dc, tabf, tabm1, va, ftc, S);
      PESPACE_MIX_CLASS(0) PESPACE_MIX_CLASS(1) PESPACE_MIX_CLASS(2) PESPACE_MIX_CLASS(3)
#undef PESPACE_MIX_CLASS
    } else {
      bool first = true;
#pragma unroll 1
      for (int mc = 0; mc < 4; ++mc) {
        if (!((cmask >> mc) & 1u)) continue;
        eval_class_mixed<KIND>(mc, first, fT, cf, lnf3, fm53, fm83f, sthf, cthf, omcf, fTLf, sc, sf, dc, tabf, tabm1, va,
                               ftc, S);
        first = false;
      }
    }
    const float Ar = S[4] - S[0], Ai = S[5] - S[1];
    const float Er_ = S[0] - 2.0f * S[2] + S[4], Ei_ = S[1] - 2.0f * S[3] + S[5];
    const float Tr = S[0] + S[2] + S[4], Ti = S[1] + S[3] + S[5];
    float r0 = fmaf(-sw[0], Ar, dr[0]), r1 = fmaf(-sw[0], Ai, di[0]);
    float acc = fmaf(r0, r0, r1 * r1);
    r0 = fmaf(-sw[1], Er_, dr[1]); r1 = fmaf(-sw[1], Ei_, di[1]);
    acc += fmaf(r0, r0, r1 * r1);
    r0 = fmaf(-sw[2], Tr, dr[2]); r1 = fmaf(-sw[2], Ti, di[2]);
    acc += fmaf(r0, r0, r1 * r1);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
    if (lane == 0) red[warp][s] = (double)acc;
  }
  __syncthreads();
  if (threadIdx.x < ns) {
    double t = 0.0;
#pragma unroll
    for (int wv = 0; wv < BLOCK / 32; ++wv) t += red[wv][threadIdx.x];
    partial[((size_t)det * gridDim.x + blockIdx.x) * (size_t)B + (size_t)(b0 + threadIdx.x)] = t;
  }
}

}  // namespace pespace
