// pespace_fisher.cuh -- forward-mode derivative kernel (S10): F_ij = <d_i h | d_j h> and
// grad_i = <d - h | d_i h> (Eq. 13, 14; "forward mode").
//
// The 11 tangents of h are NOT propagated as an 11-wide dual number.  Per mode class the response is
//     h_class = CKp Hp + i CKc Hc            (conjugate representation, as in pespace_device.cuh)
// with real amplitudes CKp, CKc (functions of M, q, D_L, iota and of v) and two complex TDI sums Hp, Hc
// built with the real arm weights xi_+/D and (n.u')(n.v')/D.  The parameters enter through
//   * the amplitudes                       (M, q, iota, D_L)          -> linear in Hp, Hc
//   * the phase psi of the class           (M, q, chi1, chi2, phi_c, t_c) -> i (pi/2) dpsi * h_class
//   * the time t_lm at which the orbit is evaluated (M, q, chi1, chi2, t_c) -> ONE geometric tangent
//   * the sky position                     (lambda, beta)             -> two geometric tangents
//   * the polarisation angle               d Hp = 4 Hc, d Hc = -Hp    -> linear in Hp, Hc
// so the per-bin geometry runs on a 3-tangent dual number (orbit angle, lambda, beta), the phase and
// time polynomials on a 4-tangent one (M, q, chi1, chi2), and everything else is closed form.
//
// Launch geometry: block = 128 threads = 128 consecutive bins ("chunk"); a block walks FCHUNKS (4) chunks and a
// tile of FTILE samples.  The 12 x 3 complex numbers (value + 11 tangents of X, Y, Z) of one (sample, bin)
// are accumulated over the mode classes in shared memory (thread-private columns), then the upper triangle
// of the 12 x 12 Gram matrix of (residual, d_1 h, ..., d_11 h) -- 78 numbers -- is formed per thread and
// reduced over the warp by a halving butterfly (96 shuffles instead of 78 x 5), fixed order throughout.
#pragma once
#include "pespace_device.cuh"

namespace pespace {

#ifndef PESPACE_FBLOCK
#define PESPACE_FBLOCK 128
#endif
#ifndef PESPACE_FMINB
#define PESPACE_FMINB 2
#endif
constexpr int FBLOCK = PESPACE_FBLOCK;   // threads = bins per chunk
#ifndef PESPACE_FTILE
#define PESPACE_FTILE 4
#endif
#ifndef PESPACE_FCHUNKS
#define PESPACE_FCHUNKS 4
#endif
constexpr int FTILE = PESPACE_FTILE;      // samples per block
constexpr int FCHUNKS = PESPACE_FCHUNKS;  // chunks per block
constexpr int NT = 12;        // value + 11 tangents
constexpr int NJ = NT * 6;    // x (X, Y, Z) x (re, im)
constexpr int NG = 78;        // upper triangle of the 12 x 12 Gram matrix
constexpr int NGP = 96;       // padded: two passes of 48 accumulators
constexpr int DUW = 8;        // doubles per constant: value + tangents (M, q, chi1, chi2, iota, lambda, beta)
constexpr int FS_STRIDE = SMEM_STRIDE * DUW;   // one sample, one detector, in shared memory

__host__ __device__ constexpr int fisher_const_stride(int n_det) { return sample_stride(n_det) * DUW; }
constexpr size_t fisher_smem_bytes() {
  return sizeof(double) * ((size_t)NJ * FBLOCK + (size_t)FTILE * FS_STRIDE + (size_t)(FBLOCK / 32) * FTILE * NGP);
}

// ---- constant accessors: sc points at one sample block [SMEM_STRIDE][DUW]
__device__ __forceinline__ double cv(const double* sc, int idx) { return sc[idx * DUW]; }
__device__ __forceinline__ double ct(const double* sc, int idx, int t) { return sc[idx * DUW + 1 + t]; }
// tangents (M, q, chi1, chi2).  A constant record is 8 doubles = 64 bytes, 64-byte aligned in shared memory: the
// tangents are fetched with 128-bit (broadcast) loads
__device__ __forceinline__ Du<4> c4(const double* sc, int idx) {
  Du<4> r;
  const double2* p = reinterpret_cast<const double2*>(sc + idx * DUW);
  const double2 a = p[0], b = p[1];
  r.v = a.x; r.d[0] = a.y; r.d[1] = b.x; r.d[2] = b.y; r.d[3] = sc[idx * DUW + 4];
  return r;
}
// geometry directions (orbit angle, lambda, beta): constants carry lambda, beta only
__device__ __forceinline__ Du<3> cg(const double* sc, int idx) {
  Du<3> r;
  const double2 t = reinterpret_cast<const double2*>(sc + idx * DUW)[3];
  r.v = sc[idx * DUW]; r.d[0] = 0.0; r.d[1] = t.x; r.d[2] = t.y;
  return r;
}
// amplitude directions (M, q, iota)
__device__ __forceinline__ Du<3> ca3(const double* sc, int idx) {
  Du<3> r;
  const double* p = sc + idx * DUW;
  const double2 a = reinterpret_cast<const double2*>(p)[0];
  r.v = a.x; r.d[0] = a.y; r.d[1] = p[2]; r.d[2] = p[5];
  return r;
}
// a Du<3> with only the orbit-angle tangent
__device__ __forceinline__ Du<3> ang(double v, double d0) {
  Du<3> r;
  r.v = v; r.d[0] = d0; r.d[1] = 0.0; r.d[2] = 0.0;
  return r;
}

// a b - c d on 3-tangent duals with the subtraction fused into the products (14 instead of 18 instructions)
__device__ __forceinline__ Du<3> prod_diff(const Du<3>& a, const Du<3>& b, const Du<3>& c, const Du<3>& d) {
  Du<3> r;
  r.v = fma(a.v, b.v, -(c.v * d.v));
#pragma unroll
  for (int i = 0; i < 3; ++i) r.d[i] = fma(a.v, b.d[i], fma(a.d[i], b.v, -fma(c.v, d.d[i], c.d[i] * d.v)));
  return r;
}

// phase-like scalars of one class handed from stage A to stage C
struct ClassScal {
  double psi;        // phase, pu (reduced)
  double tau;        // kTurn (t_lm - t_c) / yr
  double dpsi[4];    // (2 pi/kTurn) d psi / d (M, q, chi1, chi2): radians per unit parameter
  double dtau[4];    // (2 pi/kTurn) d tau / d (M, q, chi1, chi2): radians of orbit angle per unit parameter
  Du<3> CKp, CKc;    // amplitudes, tangents (M, q, iota)
};

// class constants, indexed by m - 1 at run time (the class loop of the Fisher kernel is NOT unrolled: the unrolled
// body was 154 KB of code per kernel and stalled on instruction fetch, profiles/r01_kernels_ncu.md)
__constant__ double kClassCB[4] = {1.2599210498948731648, 1.0, 0.87358046473629886905, 0.79370052598409973738};
__constant__ double kClassLN3[4] = {0.23104906018664843647, 0.0, -0.13515503603605479399, -0.23104906018664843647};
__constant__ double kClassS83[4] = {0.1574901312368591456, 1.0, 2.948334068485008683, 6.349604207872797899};

// Horner step a * x + c on (value; M, q, chi1, chi2) where x depends on M only (x = (xv; xd, 0, 0, 0)): the products
// with the structural zeros of x are not formed (6 instead of 9 instructions)
__device__ __forceinline__ Du<4> horner_m(const Du<4>& a, double xv, double xd, const Du<4>& c) {
  Du<4> r;
  r.v = fma(a.v, xv, c.v);
  r.d[0] = fma(a.v, xd, fma(a.d[0], xv, c.d[0]));
#pragma unroll
  for (int i = 1; i < 4; ++i) r.d[i] = fma(a.d[i], xv, c.d[i]);
  return r;
}

__device__ __forceinline__ void fisher_stage_a(int MC, const BinC& bc, const double* __restrict__ sc, double ftc4,
                                               ClassScal& o) {
  const double* CB = kClassCB;
  const double* LN3 = kClassLN3;
  const double* S83 = kClassS83;
  const double MHmc = 0.5 * (double)(MC + 1);
  const double sv = bc.cf * CB[MC];
  Du<4> v(0.0);
  v.v = cv(sc, W_A) * sv; v.d[0] = ct(sc, W_A, 0) * sv;
  const double L = bc.lnf3 + LN3[MC];       // ln (pi Ms)^{1/3} and its tangent are folded into W_P5, W_P6, W_Q6
  const double vv = v.v, vd = v.d[0], v2v = vv * vv, v2d = 2.0 * vv * vd;      // v^2 and its M tangent
  Du<4> P = horner_m(c4(sc, W_P7), vv, vd, dfma(L, c4(sc, W_P6L), c4(sc, W_P6)));
  P = horner_m(P, vv, vd, dfma(L, c4(sc, W_P5L), c4(sc, W_P5)));
  P = horner_m(P, vv, vd, c4(sc, W_P4));
  P = horner_m(P, vv, vd, c4(sc, W_P3));
  P = horner_m(P, vv, vd, c4(sc, W_P2));
  P = horner_m(P, v2v, v2d, c4(sc, W_P0));
  Du<4> Q = horner_m(c4(sc, W_Q7), vv, vd, dfma(L, c4(sc, W_Q6L), c4(sc, W_Q6)));
  Q = horner_m(Q, vv, vd, c4(sc, W_Q5));
  Q = horner_m(Q, vv, vd, c4(sc, W_Q4));
  Q = horner_m(Q, vv, vd, c4(sc, W_Q3));
  Q = horner_m(Q, vv, vd, c4(sc, W_Q2));
  Q = horner_m(Q, v2v, v2d, c4(sc, W_Q0));
  const double sp = S83[MC] * bc.fm53, sq = S83[MC] * bc.fm83;
  double psi = sp * P.v;
  psi -= whole_turns(psi);
  o.psi = psi + fma(MHmc, cv(sc, W_PH0), ftc4);
  o.tau = sq * Q.v;
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    o.dpsi[i] = (kRadPerPu * sp) * P.d[i];
    o.dtau[i] = (kRadPerPu * sq) * Q.d[i];
  }
  // amplitude x polarisation content, tangents (M, q, iota); v carries M only
  Du<3> va(0.0);
  va.v = v.v; va.d[0] = v.d[0];
  const int ka = W_KA + 4 * MC;
  if (MC == 1) {
    const Du<3> va2 = va * va;
    o.CKp = dfma(ca3(sc, ka + 1), va2, ca3(sc, ka));
    o.CKc = dfma(ca3(sc, ka + 3), va2, ca3(sc, ka + 2));
  } else if (MC == 3) {
    const Du<3> va2 = va * va;
    o.CKp = va2 * ca3(sc, ka);
    o.CKc = va2 * ca3(sc, ka + 2);
  } else {
    o.CKp = va * ca3(sc, ka);
    o.CKc = va * ca3(sc, ka + 2);
  }
}

// J accumulation: column of this thread in shared memory, (re, im) of entry (p, comp) at J[(p * 6 + comp * 2) * FBLOCK]
__device__ __forceinline__ void jadd(bool first, double* J, int p, int comp, double re, double im) {
  // (re, im) pairs are adjacent: one 128-bit shared-memory access per entry instead of two 64-bit ones
  double2* a = reinterpret_cast<double2*>(J + ((p * 6 + comp * 2) * FBLOCK));
  if (first) { *a = make_double2(re, im); }
  else { double2 t = *a; t.x += re; t.y += im; *a = t; }
}

// One mode class of one (sample, bin, detector): adds value and tangents of (X, Y, Z) to J.
// Tangent order p = 1..11 follows theta: M, q, chi1, chi2, D_L, iota, phi_c, lambda, beta, psi, t_c
// (D_L is filled in after the class loop: d h / d D_L = -h / D_L).
template <int KIND>
__device__ __forceinline__ void fisher_class_cs(double MMmc, bool FIRST, const ClassScal& cs, const BinC& bc,
                                                const double* __restrict__ sc, const DetC& dc, double* __restrict__ J);

template <int KIND>
__device__ __forceinline__ void fisher_class(int MC, bool FIRST, const BinC& bc, const double* __restrict__ sc,
                                          const DetC& dc, double ftc4, double* __restrict__ J) {
  ClassScal cs;
  fisher_stage_a(MC, bc, sc, ftc4, cs);
  fisher_class_cs<KIND>((double)(MC + 1), FIRST, cs, bc, sc, dc, J);
}

// S4-S7 and the tangent assembly of one class (or one tabulated mode) from its phase-like scalars cs; MMmc = m
template <int KIND>
__device__ __forceinline__ void fisher_class_cs(double MMmc, bool FIRST, const ClassScal& cs, const BinC& bc,
                                                const double* __restrict__ sc, const DetC& dc, double* __restrict__ J) {
  using G = Du<3>;

  // ---- S4 on (value, d/d alpha [rad], d/d lambda, d/d beta)
  G G1k, G2k, G1u, G2u, G1v, G2v, kR;
  // The sample constants w carry tangents in (lambda, beta) only and the trigonometric basis b in the orbit angle
  // only, so sum_i w_i b_i is written out: value sum w.v b.v, d/d alpha sum w.v b', d/d lambda sum w.dl b.v,
  // d/d beta sum w.db b.v (12 instead of 21 instructions per three-term sum; a generic dual product would multiply
  // the structural zeros).
  if (KIND == 0) {
    double sa, ca;
    sincos_pu<false>(cv(sc, D_BASE) + cs.tau, nullptr, sa, ca);
    const double c2v = fma(2.0 * ca, ca, -1.0), s2v = 2.0 * sa * ca;
    const double dc2 = -2.0 * s2v, ds2 = 2.0 * c2v;             // d/d alpha of cos 2a, sin 2a
    auto rot = [&](int off, G& g1, G& g2) {
      const double* w0 = sc + off * DUW;                        // constants off..off+4, DUW doubles each
      const double* w1 = w0 + DUW; const double* w2 = w1 + DUW; const double* w3 = w2 + DUW; const double* w4 = w3 + DUW;
      g1.v = fma(w0[0], c2v, fma(w1[0], s2v, fma(w2[0], ca, w3[0])));
      g2.v = fma(w0[0], s2v, fma(-w1[0], c2v, fma(w2[0], sa, w4[0])));
      g1.d[0] = fma(w0[0], dc2, fma(w1[0], ds2, -w2[0] * sa));
      g2.d[0] = fma(w0[0], ds2, fma(-w1[0], dc2, w2[0] * ca));
      // lambda, beta: slots 6, 7 of the constant record, one 128-bit load per constant
      const double2 t0 = reinterpret_cast<const double2*>(w0)[3], t1 = reinterpret_cast<const double2*>(w1)[3],
                    t2 = reinterpret_cast<const double2*>(w2)[3], t3 = reinterpret_cast<const double2*>(w3)[3],
                    t4 = reinterpret_cast<const double2*>(w4)[3];
      g1.d[1] = fma(t0.x, c2v, fma(t1.x, s2v, fma(t2.x, ca, t3.x)));
      g2.d[1] = fma(t0.x, s2v, fma(-t1.x, c2v, fma(t2.x, sa, t4.x)));
      g1.d[2] = fma(t0.y, c2v, fma(t1.y, s2v, fma(t2.y, ca, t3.y)));
      g2.d[2] = fma(t0.y, s2v, fma(-t1.y, c2v, fma(t2.y, sa, t4.y)));
    };
    rot(S_K, G1k, G2k);
    rot(S_U, G1u, G2u);
    rot(S_V, G1v, G2v);
    const double* dx = sc + S_DX * DUW; const double* dy = sc + S_DY * DUW;
    kR.v = fma(dx[0], ca, dy[0] * sa);
    kR.d[0] = fma(dy[0], ca, -dx[0] * sa);
    const double2 dxt = reinterpret_cast<const double2*>(dx)[3], dyt = reinterpret_cast<const double2*>(dy)[3];
    kR.d[1] = fma(dxt.x, ca, dyt.x * sa);
    kR.d[2] = fma(dxt.y, ca, dyt.y * sa);
  } else {
    double sE, cE, sp, cp;
    sincos_pu<false>(cv(sc, D_BASE) + cs.tau, nullptr, sE, cE);
    sincos_pu<false>(fma(cs.tau, dc.yr_over_p, cv(sc, D_BASE + 1)), nullptr, sp, cp);
    const double dsp = dc.yr_over_p * cp, dcp = -dc.yr_over_p * sp;     // d/d alpha of sin, cos of the spacecraft phase
    auto rot = [&](int off, G& g1, G& g2) {
      const double* w0 = sc + off * DUW; const double* w1 = w0 + DUW;
      g1.v = fma(w0[0], cp, w1[0] * sp);
      g2.v = fma(w1[0], cp, -w0[0] * sp);
      g1.d[0] = fma(w0[0], dcp, w1[0] * dsp);
      g2.d[0] = fma(w1[0], dcp, -w0[0] * dsp);
      const double2 t0 = reinterpret_cast<const double2*>(w0)[3], t1 = reinterpret_cast<const double2*>(w1)[3];
      g1.d[1] = fma(t0.x, cp, t1.x * sp); g2.d[1] = fma(t1.x, cp, -t0.x * sp);
      g1.d[2] = fma(t0.y, cp, t1.y * sp); g2.d[2] = fma(t1.y, cp, -t0.y * sp);
    };
    rot(D_BASE + 2, G1k, G2k);
    rot(D_BASE + 4, G1u, G2u);
    rot(D_BASE + 6, G1v, G2v);
    const double* dx = sc + S_DX * DUW; const double* dy = sc + S_DY * DUW;
    kR.v = fma(dx[0], cE, dy[0] * sE);
    kR.d[0] = fma(dy[0], cE, -dx[0] * sE);
    const double2 dxt = reinterpret_cast<const double2*>(dx)[3], dyt = reinterpret_cast<const double2*>(dy)[3];
    kR.d[1] = fma(dxt.x, cE, dyt.x * sE);
    kR.d[2] = fma(dxt.y, cE, dyt.y * sE);
  }
  // spacecraft at 0, 120, 240 degrees (lambda0 is absorbed by the per-sample constants): same literal
  // coefficients as eval_class
  constexpr double R3H = 0.86602540378443864676;
  const G tk = R3H * G2k, tu = R3H * G2u, tv = R3H * G2v;
  G nu[3];
  nu[0] = G1k; nu[1] = dfma(-0.5, G1k, tk); nu[2] = dfma(-0.5, G1k, -tk);
  G kap[3];                                   // k.n_23, k.n_31, k.n_12
  kap[0] = tk + tk; kap[1] = dfma(-1.5, G1k, -tk); kap[2] = dfma(1.5, G1k, -tk);
  const G ul[3] = {tu + tu, dfma(-1.5, G1u, -tu), dfma(1.5, G1u, -tu)};
  const G vl[3] = {tv + tv, dfma(-1.5, G1v, -tv), dfma(1.5, G1v, -tv)};

  // ---- S5: real arm weights xi_+/D and (n.u')(n.v')/D
  G Wp[3], Wc[3];
#pragma unroll
  for (int l = 0; l < 3; ++l) {
    const G uu = ul[l], vv = vl[l];
    G u2_, v2_, D, xi;                        // squares written out: (x^2)' = (2 x) x'
    {
      const double tu2 = uu.v + uu.v, tv2 = vv.v + vv.v;
      u2_.v = uu.v * uu.v; v2_.v = vv.v * vv.v;
#pragma unroll
      for (int i = 0; i < 3; ++i) { u2_.d[i] = tu2 * uu.d[i]; v2_.d[i] = tv2 * vv.d[i]; }
      D = u2_ + v2_;
      xi = u2_ - v2_;
    }
    G rD;
    rD.v = (__double2hiint(D.v) > 0) ? rcp_pos(D.v) : 0.0;
    const double m2 = -rD.v * rD.v;
#pragma unroll
    for (int i = 0; i < 3; ++i) rD.d[i] = m2 * D.d[i];
    Wp[l] = rD * xi;
    Wc[l] = rD * (uu * vv);
  }

  // ---- S6: E_n = exp(+i (2 pi/kTurn) (psi + kTurn f k.x_n)) (conjugate representation)
  G Er[3], Ei[3];
#pragma unroll
  for (int n = 0; n < 3; ++n) {
    const G ph = dfma(dc.Lbar, nu[n], kR);
    double s, c;
    sincos_pu<false>(fma(bc.fT, ph.v, cs.psi), nullptr, s, c);
    Er[n].v = c; Ei[n].v = s;
    const double sc4 = kRadPerPu * bc.fT;
#pragma unroll
    for (int i = 0; i < 3; ++i) {
      const double t = sc4 * ph.d[i];
      Er[n].d[i] = -s * t;
      Ei[n].d[i] = c * t;
    }
  }

  // ---- S7 + tangent assembly, one of X, Y, Z at a time
  auto bracket = [&](int r, int s_, const G& kp, G& br, G& bi) {
    br = dfma(kp, dfma(-bc.cth, Er[r], Er[s_]), (-bc.sth) * Ei[r]);
    bi = dfma(kp, dfma(-bc.cth, Ei[r], Ei[s_]), bc.sth * Er[r]);
  };
  auto component = [&](int comp, int r, int s1, const G& k1, int l1, int s2, const G& k2, int l2) {
    // H = W[l1] B(r, s1, k1) - W[l2] B(r, s2, k2)
    G b1r, b1i, b2r, b2i;
    bracket(r, s1, k1, b1r, b1i);
    bracket(r, s2, k2, b2r, b2i);
    const G Hpr = prod_diff(Wp[l1], b1r, Wp[l2], b2r), Hpi = prod_diff(Wp[l1], b1i, Wp[l2], b2i);
    const G Hcr = prod_diff(Wc[l1], b1r, Wc[l2], b2r), Hci = prod_diff(Wc[l1], b1i, Wc[l2], b2i);
    const double kp = cs.CKp.v, kc = cs.CKc.v;
    const double hr = fma(kp, Hpr.v, -kc * Hci.v), hi = fma(kp, Hpi.v, kc * Hcr.v);      // CKp Hp + i CKc Hc
    double Tr[3], Ti[3];
#pragma unroll
    for (int g = 0; g < 3; ++g) {
      Tr[g] = fma(kp, Hpr.d[g], -kc * Hci.d[g]);
      Ti[g] = fma(kp, Hpi.d[g], kc * Hcr.d[g]);
    }
    jadd(FIRST, J, 0, comp, hr, hi);
    // M, q: amplitude + phase + orbit time;  chi1, chi2: phase + orbit time
#pragma unroll
    for (int i = 0; i < 2; ++i) {
      const double ap = cs.CKp.d[i], ac = cs.CKc.d[i];
      const double re = fma(ap, Hpr.v, fma(-ac, Hci.v, fma(-cs.dpsi[i], hi, cs.dtau[i] * Tr[0])));
      const double im = fma(ap, Hpi.v, fma(ac, Hcr.v, fma(cs.dpsi[i], hr, cs.dtau[i] * Ti[0])));
      jadd(FIRST, J, 1 + i, comp, re, im);
    }
#pragma unroll
    for (int i = 2; i < 4; ++i)
      jadd(FIRST, J, 1 + i, comp, fma(-cs.dpsi[i], hi, cs.dtau[i] * Tr[0]), fma(cs.dpsi[i], hr, cs.dtau[i] * Ti[0]));
    // iota: amplitudes only
    jadd(FIRST, J, 6, comp, fma(cs.CKp.d[2], Hpr.v, -cs.CKc.d[2] * Hci.v), fma(cs.CKp.d[2], Hpi.v, cs.CKc.d[2] * Hcr.v));
    // phi_c: d psi = -m d phi_c (radians) -> -m i h
    jadd(FIRST, J, 7, comp, MMmc * hi, -MMmc * hr);
    // lambda, beta
    jadd(FIRST, J, 8, comp, Tr[1], Ti[1]);
    jadd(FIRST, J, 9, comp, Tr[2], Ti[2]);
    // polarisation angle: d Hp = 4 Hc, d Hc = -Hp
    jadd(FIRST, J, 10, comp, fma(4.0 * kp, Hcr.v, kc * Hpi.v), fma(4.0 * kp, Hci.v, -kc * Hpr.v));
    // t_c: phase 2 pi f, orbit angle 2 pi / yr
    const double wp = kRadPerPu * bc.fT, wt = kRadPerPu * kTurn / kYear;
    jadd(FIRST, J, 11, comp, fma(-wp, hi, wt * Tr[0]), fma(wp, hr, wt * Ti[0]));
  };
  // arms: index 0 = a (2-3), 1 = b (3-1), 2 = c (1-2); same terms as eval_class
  component(0, 0, 2, -kap[1], 1, 1, kap[2], 2);    // X = W_b B(1,3,k13) - W_c B(1,2,k12)
  component(1, 1, 0, -kap[2], 2, 2, kap[0], 0);    // Y = W_c B(2,1,k21) - W_a B(2,3,k23)
  component(2, 2, 1, -kap[0], 0, 0, kap[1], 1);    // Z = W_a B(3,2,k32) - W_b B(3,1,k31)
}

// ---- per-sample constants with tangents: consts_du [B][sample_stride(n_det)][DUW].  Like prep_samples_kernel the
// grid covers prep_du_threads(B, n_det) threads: warp w works on section w % (2 + n_det) (prep_sample) of the samples
// 32 (w / (2 + n_det)) + lane
__host__ __device__ constexpr long long prep_du_threads(long long B, int n_det) {
  return ((B + 31) / 32) * 32 * (2 + n_det);
}
static __global__ void prep_samples_du_kernel(const double* __restrict__ params, long long B, PrepArgs A,
                                       double* __restrict__ consts) {
  const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  const int nsec = 2 + A.n_det;
  const long long w = t >> 5;
  const int sec = (int)(w % nsec);
  const long long b = (w / nsec) * 32 + (t & 31);
  if (b >= B) return;
  const double* thp = params + b * NPAR;
  const int stride = sample_stride(A.n_det);
  double* o = consts + b * (long long)stride * DUW;
  if (!sample_in_domain(thp)) {
    if (sec == 0) {
      for (int i = 0; i < stride * DUW; ++i) o[i] = 0.0;
      o[W_A * DUW] = 1.0;
    }
    return;
  }
  // tangent slots: M, q, chi1, chi2, iota, lambda, beta.  D_L, phi_c, psi and t_c are closed form.
  const int slot[NPAR] = {0, 1, 2, 3, -1, 4, -1, 5, 6, -1, -1};
  Du<7> th[NPAR];
  for (int i = 0; i < NPAR; ++i) {
    th[i] = Du<7>(thp[i]);
    if (slot[i] >= 0) th[i].d[slot[i]] = 1.0;
  }
  prep_sample<Du<7>>(th, A, [o](int idx, const Du<7>& val) {
    double* p = o + idx * DUW;
    p[0] = val.v;
    for (int t = 0; t < 7; ++t) p[1 + t] = val.d[t];
  }, sec);
}

__device__ __forceinline__ void stage_tile_du(double* smem, const double* __restrict__ consts, long long b0,
                                              long long B, int n_det, int det) {
  const int stride = sample_stride(n_det);
  for (int i = threadIdx.x; i < FTILE * FS_STRIDE; i += blockDim.x) {
    const int s = i / FS_STRIDE, r = i % FS_STRIDE, j = r / DUW, t = r % DUW;
    long long b = b0 + s;
    if (b >= B) b = B - 1;
    const int src = (j < D_BASE) ? j : (D_BASE + D_STRIDE * det + (j - D_BASE));
    smem[i] = consts[(b * stride + src) * DUW + t];
  }
}

// index of (p, q), p <= q, in the packed upper triangle of the 12 x 12 Gram matrix
__host__ __device__ constexpr int gram_index(int p, int q) { return p * NT - p * (p - 1) / 2 + (q - p); }

// The 78 Gram entries are formed in two passes over J (rows 0..3: 42 entries, rows 4..11: 36 entries) so that at
// most NGH = 48 accumulators are live at a time (one pass over all 78 needed 255 registers and spilled).
constexpr int NGH = 48;                 // accumulators per pass (42 and 36 used)
constexpr int GRAM_SPLIT = 4;           // first row of the second pass
static_assert(NGP == 2 * NGH, "two passes");

// Halving butterfly over NGH values per lane: after the four halving levels lane l holds, in a[0..2], partial sums
// of the entries  j + 24 b4 + 12 b3 + 6 b2 + 3 b1  (b_i = bit i of l), j = 0..2; the last level adds lanes l, l ^ 1.
template <int HALF, int OFF>
__device__ __forceinline__ void butterfly_level(double (&a)[NGH], int lane) {
  const bool up = lane & OFF;
#pragma unroll
  for (int i = 0; i < HALF; ++i) {
    const double keep = up ? a[i + HALF] : a[i];
    const double send = up ? a[i] : a[i + HALF];
    a[i] = keep + __shfl_xor_sync(0xffffffffu, send, OFF);
  }
}
// slot (pass, l16 = lane >> 1, j) of the per-warp partials -> packed Gram index, or -1 for padding
__host__ __device__ inline int butterfly_slot_index(int slot) {
  const int pass = slot / NGH, r = slot % NGH, l16 = r / 3, j = r % 3;
  const int li = j + 24 * ((l16 >> 3) & 1) + 12 * ((l16 >> 2) & 1) + 6 * ((l16 >> 1) & 1) + 3 * (l16 & 1);
  const int base = pass == 0 ? 0 : gram_index(GRAM_SPLIT, GRAM_SPLIT);
  const int count = pass == 0 ? gram_index(GRAM_SPLIT, GRAM_SPLIT) : NG - gram_index(GRAM_SPLIT, GRAM_SPLIT);
  return li < count ? base + li : -1;
}

// Rows P0..P1-1 of the Gram matrix of a_0 = d - h, a_p = d_p h (p = 1..11) over the channels A, E, T for this
// thread's bin, reduced over the warp and added to the warp's partials r[NGH] (slot order of butterfly_slot_index).
template <int P0, int P1>
__device__ __forceinline__ void gram_rows(const double* __restrict__ J, const double (&dr)[3], const double (&di)[3],
                                          const double (&w)[3], double mDL, int lane, double* __restrict__ r) {
  double a[NGH];
#pragma unroll
  for (int i = 0; i < NGH; ++i) a[i] = 0.0;
#pragma unroll
  for (int c = 0; c < 3; ++c) {
    double ar[NT], ai[NT];
#pragma unroll
    for (int pp = 0; pp < NT; ++pp) {
      if (pp == 5) continue;                                  // D_L: from the value, below
      if (pp < P0 && !(pp == 0 && P0 <= 5)) continue;         // not needed by this pass
      const double* jp = J + pp * 6 * FBLOCK;
      const double2 X2 = *reinterpret_cast<const double2*>(jp), Y2 = *reinterpret_cast<const double2*>(jp + 2 * FBLOCK),
                    Z2 = *reinterpret_cast<const double2*>(jp + 4 * FBLOCK);
      const double xr = X2.x, xi = X2.y, yr = Y2.x, yi = Y2.y, zr = Z2.x, zi = Z2.y;
      if (c == 0) { ar[pp] = zr - xr; ai[pp] = zi - xi; }
      else if (c == 1) { ar[pp] = xr - 2.0 * yr + zr; ai[pp] = xi - 2.0 * yi + zi; }
      else { ar[pp] = xr + yr + zr; ai[pp] = xi + yi + zi; }
    }
    if (P0 <= 5) { ar[5] = mDL * ar[0]; ai[5] = mDL * ai[0]; }   // d h / d D_L = -h / D_L
    if (P0 == 0) { ar[0] = dr[c] - ar[0]; ai[0] = di[c] - ai[0]; }
#pragma unroll
    for (int pp = P0; pp < P1; ++pp) {
      const double wr = w[c] * ar[pp], wi = w[c] * ai[pp];
#pragma unroll
      for (int q = pp; q < NT; ++q) {
        const int li = gram_index(pp, q) - gram_index(P0, P0);
        a[li] = fma(wr, ar[q], fma(wi, ai[q], a[li]));
      }
    }
  }
  butterfly_level<24, 16>(a, lane);
  butterfly_level<12, 8>(a, lane);
  butterfly_level<6, 4>(a, lane);
  butterfly_level<3, 2>(a, lane);
#pragma unroll
  for (int j = 0; j < 3; ++j) a[j] += __shfl_xor_sync(0xffffffffu, a[j], 1);
  if (!(lane & 1)) {
    double* rr = r + (lane >> 1) * 3;
    rr[0] += a[0]; rr[1] += a[1]; rr[2] += a[2];
  }
}

// Gradient only (pespace_fisher with d_out_F = NULL): row 0 of the Gram matrix, <d - h | d_p h> for p = 0..11, reduced
// over the warp with two halving levels (12 -> 6 -> 3 values) and three plain ones; lanes 0, 8, 16, 24 add their
// three sums to slots (lane >> 3) * 3 + j of r, i.e. Gram entries j + 6 b4 + 3 b3.
__device__ __forceinline__ void gram_row0(const double* __restrict__ J, const double (&dr)[3], const double (&di)[3],
                                          const double (&w)[3], double mDL, int lane, double* __restrict__ r) {
  double a[NT];
#pragma unroll
  for (int i = 0; i < NT; ++i) a[i] = 0.0;
#pragma unroll
  for (int c = 0; c < 3; ++c) {
    double ar[NT], ai[NT];
#pragma unroll
    for (int pp = 0; pp < NT; ++pp) {
      if (pp == 5) continue;
      const double* jp = J + pp * 6 * FBLOCK;
      const double2 X2 = *reinterpret_cast<const double2*>(jp), Y2 = *reinterpret_cast<const double2*>(jp + 2 * FBLOCK),
                    Z2 = *reinterpret_cast<const double2*>(jp + 4 * FBLOCK);
      const double xr = X2.x, xi = X2.y, yr = Y2.x, yi = Y2.y, zr = Z2.x, zi = Z2.y;
      if (c == 0) { ar[pp] = zr - xr; ai[pp] = zi - xi; }
      else if (c == 1) { ar[pp] = xr - 2.0 * yr + zr; ai[pp] = xi - 2.0 * yi + zi; }
      else { ar[pp] = xr + yr + zr; ai[pp] = xi + yi + zi; }
    }
    ar[5] = mDL * ar[0]; ai[5] = mDL * ai[0];
    ar[0] = dr[c] - ar[0]; ai[0] = di[c] - ai[0];
    const double wr = w[c] * ar[0], wi = w[c] * ai[0];
#pragma unroll
    for (int q = 0; q < NT; ++q) a[q] = fma(wr, ar[q], fma(wi, ai[q], a[q]));
  }
  {
    const bool up = lane & 16;
#pragma unroll
    for (int i = 0; i < 6; ++i) {
      const double keep = up ? a[i + 6] : a[i], send = up ? a[i] : a[i + 6];
      a[i] = keep + __shfl_xor_sync(0xffffffffu, send, 16);
    }
  }
  {
    const bool up = lane & 8;
#pragma unroll
    for (int i = 0; i < 3; ++i) {
      const double keep = up ? a[i + 3] : a[i], send = up ? a[i] : a[i + 3];
      a[i] = keep + __shfl_xor_sync(0xffffffffu, send, 8);
    }
  }
#pragma unroll
  for (int o = 4; o > 0; o >>= 1)
#pragma unroll
    for (int j = 0; j < 3; ++j) a[j] += __shfl_xor_sync(0xffffffffu, a[j], o);
  if (!(lane & 7)) {
    double* rr = r + (lane >> 3) * 3;
    rr[0] += a[0]; rr[1] += a[1]; rr[2] += a[2];
  }
}

template <int KIND, unsigned CMASK>
__global__ void __launch_bounds__(FBLOCK, PESPACE_FMINB)
fisher_kernel(const double* __restrict__ consts, long long B, const double* __restrict__ bins /* [n_det][NBF][N] */,
              long long N, DetC dc, int n_det, int det, int grad_only,
              double* __restrict__ partial /* [n_det][gridDim.x][B][NG] */) {
  extern __shared__ __align__(16) double fsm[];
  double* Jsm = fsm;                                   // [NT x 3][FBLOCK] (re, im) pairs
  double* csm = Jsm + NJ * FBLOCK;                     // [FTILE][SMEM_STRIDE][DUW]
  double* red = csm + FTILE * FS_STRIDE;               // [warps][FTILE][NGP]
  const long long b0 = (long long)blockIdx.y * FTILE;
  stage_tile_du(csm, consts, b0, B, n_det, det);
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  for (int i = threadIdx.x; i < (FBLOCK / 32) * FTILE * NGP; i += FBLOCK) red[i] = 0.0;
  __syncthreads();
  double* J = Jsm + 2 * threadIdx.x;
  const int ns = (int)min((long long)FTILE, B - b0);
  for (int ch = 0; ch < FCHUNKS; ++ch) {
    const long long kbase = ((long long)blockIdx.x * FCHUNKS + ch) * FBLOCK;
    if (kbase >= N) break;
    const long long k = kbase + threadIdx.x;
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
    for (int s = 0; s < ns; ++s) {
      const double* sc = csm + s * FS_STRIDE;
      const double tc = cv(sc, W_TC);
      const double ftc4 = mul_mod_turn(bc.fT, tc);
      {
        bool first = true;
#pragma unroll 1
        for (int mc = 0; mc < 4; ++mc) {
          if (!((CMASK >> mc) & 1u)) continue;
          fisher_class<KIND>(mc, first, bc, sc, dc, ftc4, J);
          first = false;
        }
      }
      const double mDL = cv(sc, W_MDL);
      double* r = red + (warp * FTILE + s) * NGP;
      if (grad_only) {
        gram_row0(J, dr, di, w, mDL, lane, r);
      } else {
        gram_rows<0, GRAM_SPLIT>(J, dr, di, w, mDL, lane, r);
        gram_rows<GRAM_SPLIT, NT>(J, dr, di, w, mDL, lane, r + NGH);
      }
    }
  }
  __syncthreads();
  // cross-warp sum in fixed order; thread t < 96 owns slot t of the per-warp partials
  if (threadIdx.x < NGP) {
    // gradient only: slot t < 12 holds Gram entry (0, t) = packed index t
    const int gidx = grad_only ? (threadIdx.x < NT ? (int)threadIdx.x : -1) : butterfly_slot_index(threadIdx.x);
    if (gidx >= 0) {
      for (int s = 0; s < ns; ++s) {
        double t = 0.0;
#pragma unroll
        for (int wv = 0; wv < FBLOCK / 32; ++wv) t += red[(wv * FTILE + s) * NGP + threadIdx.x];
        partial[(((size_t)det * gridDim.x + blockIdx.x) * (size_t)B + (size_t)(b0 + s)) * NG + gidx] = t;
      }
    }
  }
}

// second pass: fixed-order sum over (detector, bin block); scatter to F (symmetric, full) and grad.
static __global__ void combine_fisher_kernel(const double* __restrict__ partial, const double* __restrict__ consts,
                                      long long B, int n_slices, int const_stride, double* __restrict__ outF,
                                      double* __restrict__ out_grad) {
  // block = 32 consecutive (sample, Gram entry) pairs x CGROUPS slice groups, added in the order of the groups
  __shared__ double part[CGROUPS][33];
  const int x = threadIdx.x, g = threadIdx.y;
  const long long t = (long long)blockIdx.x * 32 + x;
  const bool live = t < B * NG;
  const long long b = live ? t / NG : 0;
  const int idx = live ? (int)(t % NG) : 0;
  const bool wanted = live && (outF || idx < NT);          // gradient only: the kernel wrote row 0 of the Gram matrix only
  double acc = 0.0;
  if (wanted)
    for (int i = g; i < n_slices; i += CGROUPS) acc += partial[((size_t)i * (size_t)B + (size_t)b) * NG + idx];
  part[g][x] = acc;
  __syncthreads();
  if (g != 0 || !wanted) return;
  double sum = 0.0;
#pragma unroll
  for (int k = 0; k < CGROUPS; ++k) sum += part[k][x];
  // W_A is 1 with all tangents 0 only for out-of-domain samples (prep_samples_du_kernel)
  const bool valid = consts[(size_t)b * const_stride + W_A * DUW + 1] != 0.0;
  if (!valid) sum = CUDART_NAN;
  int p = 0, rem = idx;
  while (rem >= NT - p) { rem -= NT - p; ++p; }
  const int q = p + rem;
  if (p == 0) {
    if (q > 0 && out_grad) out_grad[b * NPAR + (q - 1)] = sum;
  } else {
    outF[(b * NPAR + (p - 1)) * NPAR + (q - 1)] = sum;
    outF[(b * NPAR + (q - 1)) * NPAR + (p - 1)] = sum;
  }
}

}  // namespace pespace
