// pespace_mixed.cuh -- mixed-precision likelihood (the paper's float32 mode for searches and
// coarse maximisation).  What stays FP64: every phase that enters an exponential -- the PN phase
// polynomial, 2 pi f t_c, the Doppler phase of the guiding centre, the sum psi + 2 pi f k.x_n and its reduction
// modulo one turn (phases reach 1e6..1e8 rad; FP32 has 7 digits).  What runs in FP32: the t_lm polynomial, the
// orbit angle, the projections and arm weights, the sine/cosine of the REDUCED phases, the brackets, TDI sums,
// A/E/T and the residual.  Data and template are whitened per bin and channel (r_c = sqrt(w_c) (d_c - h_c)) and the
// amplitudes carry a fixed scale 2^64, so that every FP32 quantity is of order 1e-3..1e3 for detector-like inputs
// (|sqrt(4 df / S_n) h| between ~1e-19 x 2^64 and 1e19 x 2^64 overflow / underflow is NOT detected).
// Accuracy: ~1e-6 relative on h for the BASELINE configs (tests/test_gpu_mixed.py), growing like 5e-7 / (2 pi f L / c)
// for arms that are short against the wavelength (tests/test_gpu_random_sweep.py), i.e. NOT a substitute for
// pespace_loglike in parameter estimation of SNR ~ 1e3 signals; throughput: DESIGN.md 8c.
#pragma once
#include "pespace_device.cuh"

namespace pespace {

constexpr float kAmpScale = 18446744073709551616.0f;    // 2^64: amplitudes x this, sqrt(w) / this
constexpr float kMagicF = 12582912.0f;                  // 1.5 * 2^23: rounds |x| < 2^22 to an integer

__constant__ double kMixCB[4] = {1.2599210498948731648, 1.0, 0.87358046473629886905, 0.79370052598409973738};
__constant__ double kMixLN3[4] = {0.23104906018664843647, 0.0, -0.13515503603605479399, -0.23104906018664843647};
__constant__ double kMixS83[4] = {0.1574901312368591456, 1.0, 2.948334068485008683, 6.349604207872797899};

// ---- packed FP32 arithmetic (Blackwell FFMA2 / FMUL2 / FADD2: one instruction, two lanes).  A thread evaluates TWO
// samples of its bin at once, lane x = sample s, lane y = sample s + 1: the FP32 part is bound by the issue port, and a
// packed instruction does the work of two for one issue slot (the FP32 pipe is then busy two cycles, during which the
// FP64 phase arithmetic, the table loads and the integer work issue for free).
typedef float2 F2;
__device__ __forceinline__ F2 bc2(float a) { return make_float2(a, a); }
__device__ __forceinline__ F2 fma2(F2 a, F2 b, F2 c) { return __ffma2_rn(a, b, c); }
__device__ __forceinline__ F2 mul2(F2 a, F2 b) { return __fmul2_rn(a, b); }
__device__ __forceinline__ F2 add2(F2 a, F2 b) { return __fadd2_rn(a, b); }
__device__ __forceinline__ F2 sub2(F2 a, F2 b) { return __ffma2_rn(b, make_float2(-1.0f, -1.0f), a); }   // a - b

// the three float tables (sin, cos, cos - 1) are separate arrays so that the two lanes' entries load straight into
// the halves of a register pair
struct TabF { const float* sn; const float* cs; const float* cm1; };

// sin, cos of the node j plus the remainder y (pu, |y| <= 1/2): first-order sine and second-order cosine correction
// (theta <= 3.1e-3: the dropped terms are < 5e-9), both lanes
__device__ __forceinline__ void sincos_f2(F2 y, int j0, int j1, const TabF& T, F2& s, F2& c) {
  const F2 Tx = make_float2(T.sn[j0 & (NTAB - 1)], T.sn[j1 & (NTAB - 1)]);
  const F2 Ty = make_float2(T.cs[j0 & (NTAB - 1)], T.cs[j1 & (NTAB - 1)]);
  const F2 sl = mul2(y, bc2((float)kRadPerPu)), nsl = mul2(y, bc2(-(float)kRadPerPu));
  const F2 cl = mul2(mul2(sl, sl), bc2(-0.5f));
  s = fma2(Ty, sl, fma2(Tx, cl, Tx));
  c = fma2(Tx, nsl, fma2(Ty, cl, Ty));
}
// phase a in pu, |a| < 2^22
__device__ __forceinline__ void sincos_pu_f2(F2 a, const TabF& T, F2& s, F2& c) {
  const F2 t = add2(a, bc2(kMagicF));
  const F2 y = sub2(a, add2(t, bc2(-kMagicF)));
  sincos_f2(y, __float_as_int(t.x), __float_as_int(t.y), T, s, c);
}

// per-bin numbers of the FP32 part, broadcast to both lanes
struct BinF2 { F2 fm83, sth, nsth, ncth, omc, fTL; };

// One mode class of one (bin, detector) for the sample pair (s, s + 1): adds X, Y, Z (whitening and per-bin factor
// excluded) to S (FP32 pairs).
//   sc0, sc1: FP64 constants of the two samples (phase polynomial, Doppler phase of the centre)
//   sf: FP32 copy of the pair's blocks, constant j of both samples in one float2; amplitudes scaled by 2^64
template <int KIND>
__device__ __forceinline__ void eval_class_mixed(int MC, bool first, double fT, double lnf3, double fm53,
                                                 const BinF2& bf, const double* __restrict__ sc0,
                                                 const double* __restrict__ sc1, const F2* __restrict__ sf,
                                                 const DetC& dc, const TabF& T, double va0, double va1, double ftc0,
                                                 double ftc1, F2 (&S)[6]) {
  // ---- S2: phase, FP64, per sample
  const double L = lnf3 + kMixLN3[MC];
  const double s53 = kMixS83[MC] * fm53, mh = 0.5 * (double)(MC + 1);
  double v[2], psi[2];
#pragma unroll
  for (int h = 0; h < 2; ++h) {
    const double* sc = h ? sc1 : sc0;
    v[h] = (h ? va1 : va0) * kMixCB[MC];
    const double v2 = v[h] * v[h];
    double P = fma(sc[W_P7], v[h], fma(sc[W_P6L], L, sc[W_P6]));
    P = fma(P, v[h], fma(sc[W_P5L], L, sc[W_P5]));
    P = fma(P, v[h], sc[W_P4]);
    P = fma(P, v[h], sc[W_P3]);
    P = fma(P, v[h], sc[W_P2]);
    P = fma(P, v2, sc[W_P0]);
    double x = s53 * P;
    x -= whole_turns(x);
    psi[h] = x + fma(mh, sc[W_PH0], h ? ftc1 : ftc0);
  }
  // ---- S3: t_lm, FP32 pairs
  const F2 vf = make_float2((float)v[0], (float)v[1]), Lf = bc2((float)L), v2f = mul2(vf, vf);
  F2 Q = fma2(sf[W_Q7], vf, fma2(sf[W_Q6L], Lf, sf[W_Q6]));
  Q = fma2(Q, vf, sf[W_Q5]);
  Q = fma2(Q, vf, sf[W_Q4]);
  Q = fma2(Q, vf, sf[W_Q3]);
  Q = fma2(Q, vf, sf[W_Q2]);
  Q = fma2(Q, v2f, sf[W_Q0]);
  const F2 tau = mul2(mul2(bc2((float)kMixS83[MC]), bf.fm83), Q);
  const F2* ka = sf + W_KA + 4 * MC;
  F2 CKp, CKc;
  if (MC == 1) { CKp = fma2(ka[1], v2f, ka[0]); CKc = fma2(ka[3], v2f, ka[2]); }
  else if (MC == 3) { CKp = mul2(v2f, ka[0]); CKc = mul2(v2f, ka[2]); }
  else { CKp = mul2(vf, ka[0]); CKc = mul2(vf, ka[2]); }
  // ---- S4: orbit, FP32 pairs
  F2 G1k, G2k, G1u, G2u, G1v, G2v, cD, sD;         // cD, sD: cos, sin of the guiding-centre (Earth) angle
  if (KIND == 0) {
    F2 sa, ca;
    sincos_pu_f2(add2(sf[D_BASE], tau), T, sa, ca);
    const F2 ca2 = add2(ca, ca);
    const F2 c2 = fma2(ca2, ca, bc2(-1.0f)), nc2 = fma2(mul2(ca, bc2(-2.0f)), ca, bc2(1.0f)), s2 = mul2(add2(sa, sa), ca);
    const F2* w = sf + S_K;
    G1k = fma2(w[0], c2, fma2(w[1], s2, fma2(w[2], ca, w[3])));
    G2k = fma2(w[0], s2, fma2(w[1], nc2, fma2(w[2], sa, w[4])));
    w = sf + S_U;
    G1u = fma2(w[0], c2, fma2(w[1], s2, fma2(w[2], ca, w[3])));
    G2u = fma2(w[0], s2, fma2(w[1], nc2, fma2(w[2], sa, w[4])));
    w = sf + S_V;
    G1v = fma2(w[0], c2, fma2(w[1], s2, fma2(w[2], ca, w[3])));
    G2v = fma2(w[0], s2, fma2(w[1], nc2, fma2(w[2], sa, w[4])));
    cD = ca; sD = sa;
  } else {
    F2 sp, cp;
    sincos_pu_f2(add2(sf[D_BASE], tau), T, sD, cD);
    sincos_pu_f2(fma2(tau, bc2((float)dc.yr_over_p), sf[D_BASE + 1]), T, sp, cp);
    const F2 nsp = mul2(sp, bc2(-1.0f));
    const F2* w = sf + D_BASE + 2;
    G1k = fma2(w[0], cp, mul2(w[1], sp)); G2k = fma2(w[1], cp, mul2(w[0], nsp));
    G1u = fma2(w[2], cp, mul2(w[3], sp)); G2u = fma2(w[3], cp, mul2(w[2], nsp));
    G1v = fma2(w[4], cp, mul2(w[5], sp)); G2v = fma2(w[5], cp, mul2(w[4], nsp));
  }
  constexpr float R3H = 0.86602540378443864676f;
  const F2 tk = mul2(bc2(R3H), G2k), ntk = mul2(bc2(-R3H), G2k);
  const F2 nun[3] = {G1k, fma2(bc2(-0.5f), G1k, tk), fma2(bc2(-0.5f), G1k, ntk)};
  // -k.n_l for the arms a, b, c
  const F2 nkap[3] = {add2(ntk, ntk), fma2(bc2(1.5f), G1k, tk), fma2(bc2(-1.5f), G1k, tk)};
  const F2 tu = mul2(bc2(R3H), G2u), ntu = mul2(bc2(-R3H), G2u), tv = mul2(bc2(R3H), G2v), ntv = mul2(bc2(-R3H), G2v);
  const F2 ul[3] = {add2(tu, tu), fma2(bc2(-1.5f), G1u, ntu), fma2(bc2(1.5f), G1u, ntu)};
  const F2 vl[3] = {add2(tv, tv), fma2(bc2(-1.5f), G1v, ntv), fma2(bc2(1.5f), G1v, ntv)};
  // ---- S5: arm weights, FP32 pairs (the reciprocal is MUFU.RCP per lane, ~1 ulp)
  F2 Wr[3], Wi[3], nWi[3];
#pragma unroll
  for (int l = 0; l < 3; ++l) {
    const F2 uu = ul[l], vv = vl[l];
    const F2 v2_ = mul2(vv, vv);
    const F2 D = fma2(uu, uu, v2_);
    F2 rD;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(rD.x) : "f"(D.x));
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(rD.y) : "f"(D.y));
    rD.x = (D.x > 0.0f) ? rD.x : 0.0f;
    rD.y = (D.y > 0.0f) ? rD.y : 0.0f;
    Wr[l] = mul2(mul2(CKp, rD), fma2(bc2(-2.0f), v2_, D));        // u^2 - v^2 = (u^2 + v^2) - 2 v^2
    Wi[l] = mul2(mul2(CKc, rD), mul2(uu, vv));
    nWi[l] = mul2(Wi[l], bc2(-1.0f));
  }
  // ---- S6: exponentials relative to the guiding centre.  E_n = E_c (1 + delta_n), E_c = exp(-i base) with the
  // large phase base = psi + kTurn f k.x_centre reduced in FP64 (Doppler phase of the centre from the FP64 constants),
  // delta_n = exp(-i a_n) - 1 with the arm-scale phase a_n = kTurn f L k.(x_n - x_centre)/L, |a_n| < 1 turn, in FP32
  // from the (sin, cos - 1) table: at low frequency a_n -> 0 and the brackets below are differences of O(2 pi f L)
  // quantities, which this form evaluates without cancelling against 1 (FP32 would lose 1 / (2 pi f L) digits).
  F2 yb;
  int jb[2];
#pragma unroll
  for (int h = 0; h < 2; ++h) {
    const double* sc = h ? sc1 : sc0;
    const double kR = fma(sc[S_DX], (double)(h ? cD.y : cD.x), sc[S_DY] * (double)(h ? sD.y : sD.x));
    const double ub = fma(fT, kR, psi[h]);
    const double tb = ub + kMagic;
    (h ? yb.y : yb.x) = (float)(ub - (tb - kMagic));
    jb[h] = __double2loint(tb);
  }
  F2 sb, cb;
  sincos_f2(yb, jb[0], jb[1], T, sb, cb);
  const F2 nsb = mul2(sb, bc2(-1.0f));
  F2 dC[3], dS[3];                    // cos a_n - 1, sin a_n
#pragma unroll
  for (int n = 0; n < 3; ++n) {
    const F2 a = mul2(bf.fTL, nun[n]);
    const F2 t = add2(a, bc2(kMagicF));
    const F2 y = sub2(a, add2(t, bc2(-kMagicF)));
    const int j0 = __float_as_int(t.x) & (NTAB - 1), j1 = __float_as_int(t.y) & (NTAB - 1);
    const F2 Tx = make_float2(T.sn[j0], T.sn[j1]), Ty = make_float2(T.cs[j0], T.cs[j1]);
    const F2 Tm = make_float2(T.cm1[j0], T.cm1[j1]);               // cos - 1 of the node, full relative accuracy
    const F2 sl = mul2(y, bc2((float)kRadPerPu)), nsl = mul2(y, bc2(-(float)kRadPerPu));
    const F2 cl = mul2(mul2(sl, sl), bc2(-0.5f));
    dS[n] = fma2(Ty, sl, fma2(Tx, cl, Tx));
    dC[n] = fma2(Tx, nsl, fma2(Ty, cl, Tm));
  }
  // ---- S7: brackets in the centre frame, B'(r,s,kap) = kap (delta_s - cos(th) delta_r + (1 - cos th)) - i sin(th) (1 + delta_r).
  // The three "minus W" terms of the TDI sums are taken as W times MINUS the bracket, so that only -k.n_l is needed.
  F2 Ps[3], nPs[3], Qs[3], nQs[3];
#pragma unroll
  for (int r = 0; r < 3; ++r) {
    Ps[r] = mul2(bf.sth, dS[r]); nPs[r] = mul2(bf.nsth, dS[r]);
    Qs[r] = fma2(bf.sth, dC[r], bf.sth); nQs[r] = fma2(bf.nsth, dC[r], bf.nsth);
  }
  F2 Sc[6];
  // plus = true: + W B(r, s, kap = km);  plus = false: - W B(r, s, kap = -km)
  auto add = [&](F2& Sr, F2& Si, int r, int s_, F2 km, int l, bool plus, bool init) {
    const F2 in_r = add2(fma2(bf.ncth, dC[r], dC[s_]), bf.omc), in_i = fma2(bf.ncth, dS[r], dS[s_]);
    const F2 br = fma2(km, in_r, plus ? nPs[r] : Ps[r]);
    const F2 bi = fma2(km, in_i, plus ? Qs[r] : nQs[r]);
    if (init) {
      Sr = fma2(Wr[l], br, mul2(nWi[l], bi));
      Si = fma2(Wr[l], bi, mul2(Wi[l], br));
    } else {
      Sr = fma2(Wr[l], br, fma2(nWi[l], bi, Sr));
      Si = fma2(Wr[l], bi, fma2(Wi[l], br, Si));
    }
  };
  // arms: index 0 = a (2-3), 1 = b (3-1), 2 = c (1-2)
  add(Sc[0], Sc[1], 0, 2, nkap[1], 1, true, true);      // X: + W_b B(1,3,-k.n_b)
  add(Sc[0], Sc[1], 0, 1, nkap[2], 2, false, false);    //    - W_c B(1,2,+k.n_c)
  add(Sc[2], Sc[3], 1, 0, nkap[2], 2, true, true);      // Y: + W_c B(2,1,-k.n_c)
  add(Sc[2], Sc[3], 1, 2, nkap[0], 0, false, false);    //    - W_a B(2,3,+k.n_a)
  add(Sc[4], Sc[5], 2, 1, nkap[0], 0, true, true);      // Z: + W_a B(3,2,-k.n_a)
  add(Sc[4], Sc[5], 2, 0, nkap[1], 1, false, false);    //    - W_b B(3,1,+k.n_b)
  // back to the SSB frame: (Sr - i Si) (cb - i sb)
#pragma unroll
  for (int c = 0; c < 3; ++c) {
    if (first) {
      S[2 * c] = fma2(Sc[2 * c], cb, mul2(Sc[2 * c + 1], nsb));
      S[2 * c + 1] = fma2(Sc[2 * c], sb, mul2(Sc[2 * c + 1], cb));
    } else {
      S[2 * c] = fma2(Sc[2 * c], cb, fma2(Sc[2 * c + 1], nsb, S[2 * c]));
      S[2 * c + 1] = fma2(Sc[2 * c], sb, fma2(Sc[2 * c + 1], cb, S[2 * c + 1]));
    }
  }
}

// dynamic shared memory: [float sin | cos | cos - 1 tables | FP64 sample constants | FP32 copy, the two samples of a
// pair interleaved | warp partials]
constexpr int MIX_TILE = 64;
static_assert(MIX_TILE % 4 == 0, "sample pairs; stage_tile pads the tile to a multiple of four samples");
constexpr size_t mixed_smem_used() {
  return 3 * sizeof(float) * NTAB + sizeof(double) * (size_t)MIX_TILE * SMEM_STRIDE +
         sizeof(float) * (size_t)MIX_TILE * SMEM_STRIDE + sizeof(double) * (size_t)(BLOCK / 32) * MIX_TILE;
}
constexpr size_t mixed_smem_bytes() { return (mixed_smem_used() + 15) / 16 * 16; }

#ifndef PESPACE_MINBX
#define PESPACE_MINBX 2
#endif
// CMASK != 0: the classes of that mask unrolled at compile time (the masks of configs 2-4); 0: any mask, run-time loop
template <int KIND, unsigned CMASK>
__global__ void __launch_bounds__(BLOCK, popc4(CMASK) > 1 ? 1 : PESPACE_MINBX)      // four classes unrolled: 128 registers spill
loglike_mixed_kernel(const double* __restrict__ consts, const double2* __restrict__ trig, long long B, unsigned cmask,
                     const double* __restrict__ bins /* [n_det][NBF][N], built with fold mode 2 */, long long N, DetC dc,
                     int n_det, int det, double* __restrict__ partial /* [n_det][gridDim.x][B] */) {
  double* smem = reinterpret_cast<double*>(pespace_dyn_smem);                  // FP64 constants first: 16-byte aligned
  F2* smf = reinterpret_cast<F2*>(smem + MIX_TILE * SMEM_STRIDE);              // [MIX_TILE / 2][SMEM_STRIDE] pairs
  double (*red)[MIX_TILE] = reinterpret_cast<double (*)[MIX_TILE]>(smf + (MIX_TILE / 2) * SMEM_STRIDE);
  float* tsn = reinterpret_cast<float*>(&red[BLOCK / 32][0]);
  float* tcs = tsn + NTAB;
  float* tm1 = tcs + NTAB;
  const TabF T{tsn, tcs, tm1};
  const long long b0 = (long long)blockIdx.y * MIX_TILE;
  for (int i = threadIdx.x; i < NTAB; i += blockDim.x) {
    const double2 t = trig[i];
    tsn[i] = (float)t.x;
    tcs[i] = (float)t.y;
    // cos - 1 = -sin^2 / (1 + cos) where cos > 0, formed in FP64 so that the float keeps full relative accuracy
    tm1[i] = (float)(t.y > 0.0 ? -t.x * t.x / (1.0 + t.y) : t.y - 1.0);
  }
  stage_tile(smem, consts, b0, B, n_det, det);
  __syncthreads();
  for (int i = threadIdx.x; i < MIX_TILE * SMEM_STRIDE; i += blockDim.x) {
    const int sidx = i / SMEM_STRIDE, j = i % SMEM_STRIDE;
    double x = smem[i];
    if (j >= W_KA && j < W_KA + 16) x *= (double)kAmpScale;       // amplitudes carry the 2^64 scale
    float* dst = reinterpret_cast<float*>(smf + (sidx >> 1) * SMEM_STRIDE + j);
    dst[sidx & 1] = (float)x;
  }
  const long long k = (long long)blockIdx.x * BLOCK + threadIdx.x;
  const bool live = k < N;
  const double* bp = bins + (size_t)det * NBF * (size_t)N + (size_t)(live ? k : N - 1);
  const double fT = bp[BF_FT * N], cf = bp[BF_CF * N], lnf3 = bp[BF_LNF3 * N], fm53 = bp[BF_FM53 * N];
  const double sth = bp[BF_STH * N], cth = bp[BF_CTH * N];
  BinF2 bf;
  bf.fm83 = bc2((float)bp[BF_FM83 * N]);
  bf.sth = bc2((float)sth); bf.nsth = bc2(-(float)sth); bf.ncth = bc2(-(float)cth);
  bf.omc = bc2((float)(cth > 0.0 ? sth * sth / (1.0 + cth) : 1.0 - cth));       // 1 - cos(2 pi f L), no cancellation
  bf.fTL = bc2((float)(fT * dc.Lbar));
  F2 dr[3], di[3], nsw[3];
#pragma unroll
  for (int c = 0; c < 3; ++c) {
    dr[c] = bc2(live ? (float)bp[(BF_DR + c) * N] : 0.0f);
    di[c] = bc2(live ? (float)bp[(BF_DI + c) * N] : 0.0f);
    nsw[c] = bc2(live ? -(float)bp[(BF_W + c) * N] : 0.0f);
  }
  __syncthreads();
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int ns = (int)min((long long)MIX_TILE, B - b0);
  for (int s = 0; s < ns; s += 2) {          // the pair (s, s + 1); stage_tile pads an odd tail with a copy
    const double* sc0 = smem + s * SMEM_STRIDE;
    const double* sc1 = sc0 + SMEM_STRIDE;
    const F2* sf = smf + (s >> 1) * SMEM_STRIDE;
    const double ftc0 = mul_mod_turn(fT, sc0[W_TC]), ftc1 = mul_mod_turn(fT, sc1[W_TC]);
    const double va0 = sc0[W_A] * cf, va1 = sc1[W_A] * cf;
    F2 S[6];
    if constexpr (CMASK != 0u) {
#define PESPACE_MIX_CLASS(MC)                                                                                       \
      if constexpr ((CMASK >> MC) & 1u)                                                                               \
        eval_class_mixed<KIND>(MC, !(CMASK & ((1u << MC) - 1u)), fT, lnf3, fm53, bf, sc0, sc1, sf, dc, T, va0, va1, ftc0, \
                               ftc1, S);
      PESPACE_MIX_CLASS(0) PESPACE_MIX_CLASS(1) PESPACE_MIX_CLASS(2) PESPACE_MIX_CLASS(3)
#undef PESPACE_MIX_CLASS
    } else {
      bool first = true;
#pragma unroll 1
      for (int mc = 0; mc < 4; ++mc) {
        if (!((cmask >> mc) & 1u)) continue;
        eval_class_mixed<KIND>(mc, first, fT, lnf3, fm53, bf, sc0, sc1, sf, dc, T, va0, va1, ftc0, ftc1, S);
        first = false;
      }
    }
    const F2 Ar = sub2(S[4], S[0]), Ai = sub2(S[5], S[1]);
    const F2 Er_ = fma2(bc2(-2.0f), S[2], add2(S[0], S[4])), Ei_ = fma2(bc2(-2.0f), S[3], add2(S[1], S[5]));
    const F2 Tr = add2(add2(S[0], S[2]), S[4]), Ti = add2(add2(S[1], S[3]), S[5]);
    F2 r0 = fma2(nsw[0], Ar, dr[0]), r1 = fma2(nsw[0], Ai, di[0]);
    F2 acc2 = fma2(r0, r0, mul2(r1, r1));
    r0 = fma2(nsw[1], Er_, dr[1]); r1 = fma2(nsw[1], Ei_, di[1]);
    acc2 = fma2(r0, r0, fma2(r1, r1, acc2));
    r0 = fma2(nsw[2], Tr, dr[2]); r1 = fma2(nsw[2], Ti, di[2]);
    acc2 = fma2(r0, r0, fma2(r1, r1, acc2));
    // S9: halving butterfly: after the first level the lanes 0-15 hold sample s, the lanes 16-31 sample s + 1
    const bool up = lane & 16;
    float acc = (up ? acc2.y : acc2.x) + __shfl_xor_sync(0xffffffffu, up ? acc2.x : acc2.y, 16);
#pragma unroll
    for (int o = 8; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
    if ((lane & 15) == 0) red[warp][s + (lane >> 4)] = (double)acc;     // s + 1 <= MIX_TILE - 1 (s even)
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
