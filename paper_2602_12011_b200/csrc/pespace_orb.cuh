// pespace_orb.cuh -- tabulated numerical orbits ("Support for high-precision
// numerical orbits will be extended in future work").  Reading T2 of DESIGN.md: spacecraft positions and velocities of
// every detector on a uniform time grid t_j = t0 + j dt (SSB seconds, origin of t_c), pos / vel [n_det][K][3][3];
// between nodes every coordinate is the cubic Hermite interpolant with the node velocities as slopes; Eq. 5 / Eq. 6
// keep the nominal constant arm length L of the detector description in the delays (the paper's rigid equal-arm
// formalism), the link directions are the unit vectors (x_r - x_s) / |x_r - x_s|; a mode whose
// t_lm(f) lies outside the table contributes 0.
//
// S2/S3 (analytic TaylorF2 modes) and S5-S9 are those of the likelihood path; S4 is replaced: instead of the linear
// combinations G1, G2 of a few sines and cosines, a (sample, bin, class) gathers two nodes of the table (36 doubles;
// t_lm(f) is smooth in f, so neighbouring bins read the same nodes), interpolates the nine coordinates and projects
// them on the per-sample vectors k/c, k/L, u'/L, v'/L.  One kernel for both detector kinds (the kind, kappa, lambda0,
// period and pointing of the description are not used); the class loop is unrolled at compile time for the masks of
// configs 2-4 ((2,2) only; all five modes) and a run-time loop for the rest.
#pragma once
#include "pespace_device.cuh"
#include "pespace_fisher.cuh"   // kClassCB, kClassLN3, kClassS83
#include "pespace_tab.cuh"      // stage_tile_n

namespace pespace {

struct OrbC {            // kernel parameter: one detector's table
  long long K;
  double ts;             // node spacings per pu of tau: (yr / kTurn) / dt
  const double* pos;     // [K][3][3] metres
  const double* vel;     // [K][3][3] m/s
  double dt;
};

// detector block of the per-sample constants on this path (offsets from D_BASE + D_STRIDE det)
enum : int { OB_S0 = 0,        // (t_c - t0) / dt: node coordinate of t_c
             OB_KC = 2,        // k / c          [s/m]  x 3
             OB_KL = 5,        // k / L, u' / L, v' / L  [1/m]  x 3 each
             OB_UL = 8, OB_VL = 11 };

struct OrbPrep { double t0, dt; };

static __global__ void prep_samples_orb_kernel(const double* __restrict__ params, long long B, PrepArgs A, OrbPrep O,
                                               double* __restrict__ consts, double2* __restrict__ trig) {
  const long long b = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  fill_trig_entry(trig, b);
  if (b >= B) return;
  const double* thp = params + b * NPAR;
  const int stride = sample_stride(A.n_det);
  double* o = consts + b * stride;
  if (!sample_in_domain(thp)) {
    for (int i = 0; i < stride; ++i) o[i] = 0.0;
    o[W_A] = 1.0; o[W_VALID] = 0.0;
    return;
  }
  double th[NPAR];
  for (int i = 0; i < NPAR; ++i) th[i] = thp[i];
  prep_sample<double>(th, A, [o](int idx, double val) { o[idx] = val; });     // waveform constants (S1)
  // frame (O7) with the polarisation angle absorbed: the detector blocks are rewritten for this path
  double sl, cl, sb, cb, sp, cp;
  sincos(th[7], &sl, &cl); sincos(th[8], &sb, &cb); sincos(th[9], &sp, &cp);
  const double k[3] = {-(cb * cl), -(cb * sl), -sb};
  const double u[3] = {sl, -cl, 0.0};
  const double v[3] = {-(sb * cl), -(sb * sl), cb};
  for (int d = 0; d < A.n_det; ++d) {
    double* q = o + D_BASE + D_STRIDE * d;
    for (int i = 0; i < D_STRIDE; ++i) q[i] = 0.0;
    const double L = A.det[d].Lbar * kC;
    q[OB_S0] = (th[10] - O.t0) / O.dt;
    for (int i = 0; i < 3; ++i) {
      q[OB_KC + i] = k[i] / kC;
      q[OB_KL + i] = k[i] / L;
      q[OB_UL + i] = (cp * u[i] + sp * v[i]) / L;
      q[OB_VL + i] = (cp * v[i] - sp * u[i]) / L;
    }
  }
}

// One mode class of one (sample, bin, detector) with the orbit from the table: adds X, Y, Z (Re, -Im; without the
// common factor g z f^{-7/6}) to S.  The waveform part is eval_class's, the tail (S5-S7) eval_geom's.
__device__ __forceinline__ void orb_class(int mc, bool first, const BinC& bc, const double* __restrict__ sc,
                                          const DetC& dc, const double2* __restrict__ tab, const OrbC& O, double va,
                                          double La, double ftc, double (&S)[6]) {
  const double MH = 0.5 * (double)(mc + 1);
  const double v = va * kClassCB[mc];
  const double L = La + kClassLN3[mc];
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
  double psi = (kClassS83[mc] * bc.fm53) * P;
  psi -= whole_turns(psi);
  psi += fma(MH, sc[W_PH0], ftc);
  const double tau = (kClassS83[mc] * bc.fm83) * Q;                 // kTurn (t_lm - t_c) / yr
  const double* ka = sc + W_KA + 4 * mc;
  double CKp, CKc;
  if (mc == 1) { CKp = fma(ka[1], v2, ka[0]); CKc = fma(ka[3], v2, ka[2]); }
  else { const double vp = (mc == 3) ? v2 : v; CKp = vp * ka[0]; CKc = vp * ka[2]; }

  // ---- S4 from the table: node coordinate s = (t_lm - t0) / dt, interval j, u = s - j
  const double s = fma(tau, O.ts, sc[D_BASE + OB_S0]);
  const bool inside = (s >= 0.0) && (s <= (double)(O.K - 1));
  long long j = (long long)floor(s);
  j = j < 0 ? 0 : (j > O.K - 2 ? O.K - 2 : j);
  const double u = inside ? s - (double)j : 0.0;
  if (!inside) { CKp = 0.0; CKc = 0.0; }                             // outside the table the mode contributes 0
  const double u2 = u * u, u3 = u2 * u;
  const double h00 = fma(2.0, u3, fma(-3.0, u2, 1.0)), h01 = fma(-2.0, u3, 3.0 * u2);
  const double h10 = O.dt * (u3 - 2.0 * u2 + u), h11 = O.dt * (u3 - u2);
  const double* p0 = O.pos + j * 9;
  const double* v0 = O.vel + j * 9;
  double kx[3], kd[3], ud[3], vd[3];            // k.x_n / c and the projections of x_n on k / L, u' / L, v' / L
  const double* wkc = sc + D_BASE + OB_KC; const double* wkl = sc + D_BASE + OB_KL;
  const double* wul = sc + D_BASE + OB_UL; const double* wvl = sc + D_BASE + OB_VL;
#pragma unroll
  for (int n = 0; n < 3; ++n) {
    double x[3];
#pragma unroll
    for (int a = 0; a < 3; ++a)
      x[a] = fma(h00, p0[3 * n + a], fma(h01, p0[9 + 3 * n + a], fma(h10, v0[3 * n + a], h11 * v0[9 + 3 * n + a])));
    kx[n] = fma(wkc[0], x[0], fma(wkc[1], x[1], wkc[2] * x[2]));
    kd[n] = fma(wkl[0], x[0], fma(wkl[1], x[1], wkl[2] * x[2]));
    ud[n] = fma(wul[0], x[0], fma(wul[1], x[1], wul[2] * x[2]));
    vd[n] = fma(wvl[0], x[0], fma(wvl[1], x[1], wvl[2] * x[2]));
  }
  // arms a: 2-3, b: 3-1, c: 1-2 (spacecraft 1, 2, 3 = index 0, 1, 2): projections of (x_r - x_s) / L on the orthonormal
  // triad, then normalised to the unit link vector: |x_r - x_s|^2 / L^2 = (k.a)^2 + (u'.a)^2 + (v'.a)^2
  double kl[3] = {kd[1] - kd[2], kd[2] - kd[0], kd[0] - kd[1]};
  double ul[3] = {ud[1] - ud[2], ud[2] - ud[0], ud[0] - ud[1]};
  double vl[3] = {vd[1] - vd[2], vd[2] - vd[0], vd[0] - vd[1]};
#pragma unroll
  for (int l = 0; l < 3; ++l) {
    const double n2 = fma(kl[l], kl[l], fma(ul[l], ul[l], vl[l] * vl[l]));      // close to 1
    double y;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(n2));
    const double hn = 0.5 * n2;
    y = y * fma(-hn * y, y, 1.5);                                               // two Newton steps: 2^-20 -> 2^-80
    y = y * fma(-hn * y, y, 1.5);
    kl[l] *= y; ul[l] *= y; vl[l] *= y;
  }
  const double ka_ = kl[0], kb_ = kl[1], kc_ = kl[2];

  // ---- S5: W_l = amplitude (n_l.P.n_l) / (1 - (k.n_l)^2)
  double Wr[3], Wi[3];
#pragma unroll
  for (int l = 0; l < 3; ++l) {
    const double uu = ul[l], vv = vl[l];
    const double v2_ = vv * vv;
    const double D = fma(uu, uu, v2_);
    const double rD = (__double2hiint(D) > 0) ? rcp_pos(D) : 0.0;
    Wr[l] = (CKp * rD) * fma(uu, uu, -v2_);
    Wi[l] = (CKc * rD) * (uu * vv);
  }
  // ---- S6: h_lm E_n = exp(-i (2 pi / kTurn) (psi + kTurn f k.x_n / c))
  double Er[3], Ei[3];
#pragma unroll
  for (int n = 0; n < 3; ++n) sincos_tab(fma(bc.fT, kx[n], psi), tab, Ei[n], Er[n]);
  // ---- S7: brackets and TDI sums (see eval_geom)
  auto add = [&](double& Sr, double& Si, int r, int s_, double kap, double wr, double wi, bool init) {
    const double br = fma(kap, fma(-bc.cth, Er[r], Er[s_]), -bc.sth * Ei[r]);
    const double bi = fma(kap, fma(-bc.cth, Ei[r], Ei[s_]), bc.sth * Er[r]);
    if (init) { Sr = fma(wr, br, -wi * bi); Si = fma(wr, bi, wi * br); }
    else { Sr = fma(wr, br, fma(-wi, bi, Sr)); Si = fma(wr, bi, fma(wi, br, Si)); }
  };
  add(S[0], S[1], 0, 2, -kb_, Wr[1], Wi[1], first);
  add(S[0], S[1], 0, 1, kc_, -Wr[2], -Wi[2], false);
  add(S[2], S[3], 1, 0, -kc_, Wr[2], Wi[2], first);
  add(S[2], S[3], 1, 2, ka_, -Wr[0], -Wi[0], false);
  add(S[4], S[5], 2, 1, -ka_, Wr[0], Wi[0], first);
  add(S[4], S[5], 2, 0, kb_, -Wr[1], -Wi[1], false);
}

// CMASK != 0: the classes of that mask unrolled at compile time (instantiated for the common masks); CMASK == 0: any
// mask, run-time loop
template <unsigned CMASK>
__device__ __forceinline__ void eval_xyz_orb(unsigned cmask, const BinC& bc, const double* __restrict__ sc,
                                             const DetC& dc, const double2* __restrict__ tab, const OrbC& O,
                                             double (&S)[6]) {
  const double ftc = mul_mod_turn(bc.fT, sc[W_TC]);
  const double va = sc[W_A] * bc.cf, La = bc.lnf3;
  if constexpr (CMASK != 0u) {
#define PESPACE_ORB_CLASS(MC) \
    if constexpr ((CMASK >> MC) & 1u) orb_class(MC, !(CMASK & ((1u << MC) - 1u)), bc, sc, dc, tab, O, va, La, ftc, S);
    PESPACE_ORB_CLASS(0) PESPACE_ORB_CLASS(1) PESPACE_ORB_CLASS(2) PESPACE_ORB_CLASS(3)
#undef PESPACE_ORB_CLASS
  } else {
    bool first = true;
#pragma unroll 1
    for (int mc = 0; mc < 4; ++mc) {
      if (!((cmask >> mc) & 1u)) continue;
      orb_class(mc, first, bc, sc, dc, tab, O, va, La, ftc, S);
      first = false;
    }
  }
}

// likelihood with tabulated orbits: grid (bin blocks, sample tiles of TAB_TILE); one launch per detector
template <unsigned CMASK>
__global__ void __launch_bounds__(BLOCK, 1)
loglike_orb_kernel(const double* __restrict__ consts, const double2* __restrict__ trig, long long B, unsigned cmask,
                   OrbC O, const double* __restrict__ bins /* [n_det][NBF][N] */, long long N, DetC dc, int n_det,
                   int det, double* __restrict__ partial /* [n_det][gridDim.x][B] */) {
  double2* tab = reinterpret_cast<double2*>(pespace_dyn_smem);
  double* smem = reinterpret_cast<double*>(tab + NTAB);
  double (*red)[TAB_TILE] = reinterpret_cast<double (*)[TAB_TILE]>(smem + TAB_TILE * SMEM_STRIDE);
  const long long b0 = (long long)blockIdx.y * TAB_TILE;
  stage_trig(tab, trig);
  stage_tile_n(smem, consts, b0, B, n_det, det, TAB_TILE);
  const long long k = (long long)blockIdx.x * BLOCK + threadIdx.x;
  const bool live = k < N;
  const double* bp = bins + (size_t)det * NBF * (size_t)N + (size_t)(live ? k : N - 1);
  BinC bc;
  bc.fT = bp[BF_FT * N]; bc.cf = bp[BF_CF * N]; bc.lnf3 = bp[BF_LNF3 * N]; bc.fm53 = bp[BF_FM53 * N];
  bc.fm83 = bp[BF_FM83 * N]; bc.sth = bp[BF_STH * N]; bc.cth = bp[BF_CTH * N]; bc.fm76 = 0.0;
  double dr[3], di[3], w[3];
#pragma unroll
  for (int c = 0; c < 3; ++c) {
    dr[c] = bp[(BF_DR + c) * N]; di[c] = bp[(BF_DI + c) * N];
    w[c] = live ? bp[(BF_W + c) * N] : 0.0;
  }
  __syncthreads();
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int ns = (int)min((long long)TAB_TILE, B - b0);
  for (int s = 0; s < ns; ++s) {
    double S[6];
    eval_xyz_orb<CMASK>(cmask, bc, smem + s * SMEM_STRIDE, dc, tab, O, S);
    const double Ar = S[4] - S[0], Ai = S[5] - S[1];
    const double Er_ = S[0] - 2.0 * S[2] + S[4], Ei_ = S[1] - 2.0 * S[3] + S[5];
    const double Tr = S[0] + S[2] + S[4], Ti = S[1] + S[3] + S[5];
    double r0 = dr[0] - Ar, r1 = di[0] - Ai;
    double acc = w[0] * fma(r0, r0, r1 * r1);
    r0 = dr[1] - Er_; r1 = di[1] - Ei_;
    acc = fma(w[1], fma(r0, r0, r1 * r1), acc);
    r0 = dr[2] - Tr; r1 = di[2] - Ti;
    acc = fma(w[2], fma(r0, r0, r1 * r1), acc);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
    if (lane == 0) red[warp][s] = acc;
  }
  __syncthreads();
  if (threadIdx.x < ns) {
    double t = 0.0;
#pragma unroll
    for (int wv = 0; wv < BLOCK / 32; ++wv) t += red[wv][threadIdx.x];
    partial[((size_t)det * gridDim.x + blockIdx.x) * (size_t)B + (size_t)(b0 + threadIdx.x)] = t;
  }
}

// response with tabulated orbits on an arbitrary frequency array
template <unsigned CMASK>
__global__ void __launch_bounds__(BLOCK, 1)
response_orb_kernel(const double* __restrict__ consts, const double2* __restrict__ trig, long long B, unsigned cmask,
                    OrbC O, const double* __restrict__ freqs, long long N, DetC dc, int n_det, int det,
                    double2* __restrict__ out /* [B][n_det][3][N] */) {
  double2* tab = reinterpret_cast<double2*>(pespace_dyn_smem);
  double* smem = reinterpret_cast<double*>(tab + NTAB);
  const long long b0 = (long long)blockIdx.y * TAB_TILE;
  stage_trig(tab, trig);
  stage_tile_n(smem, consts, b0, B, n_det, det, TAB_TILE);
  const long long k = (long long)blockIdx.x * BLOCK + threadIdx.x;
  const bool live = k < N;
  const double fraw = freqs[live ? k : N - 1];
  const bool pos = fraw > 0.0;
  const BinC bc = make_bin(pos ? fraw : 1.0, dc.Lbar);
  double gr, gi;
  tdi_prefactor(bc, dc.gen, gr, gi);
  __syncthreads();
  const int ns = (int)min((long long)TAB_TILE, B - b0);
  const double i2 = 0.70710678118654752440, i6 = 0.40824829046386301637, i3 = 0.57735026918962576451;
  for (int s = 0; s < ns; ++s) {
    const double* sc = smem + s * SMEM_STRIDE;
    double S[6];
    eval_xyz_orb<CMASK>(cmask, bc, sc, dc, tab, O, S);
    double ch[6];                                      // S holds (Re, -Im)
    ch[0] = (S[4] - S[0]) * i2; ch[1] = (S[1] - S[5]) * i2;
    ch[2] = (S[0] - 2.0 * S[2] + S[4]) * i6; ch[3] = -(S[1] - 2.0 * S[3] + S[5]) * i6;
    ch[4] = (S[0] + S[2] + S[4]) * i3; ch[5] = -(S[1] + S[3] + S[5]) * i3;
    if (!live) continue;
    const bool valid = sc[W_VALID] != 0.0;
#pragma unroll
    for (int c = 0; c < 3; ++c) {
      double2 o;
      o.x = ch[2 * c] * gr - ch[2 * c + 1] * gi;
      o.y = ch[2 * c] * gi + ch[2 * c + 1] * gr;
      if (!pos) { o.x = 0.0; o.y = 0.0; }
      if (!valid) { o.x = CUDART_NAN; o.y = CUDART_NAN; }
      out[(((size_t)(b0 + s) * n_det + det) * 3 + c) * (size_t)N + (size_t)k] = o;
    }
  }
}

}  // namespace pespace
