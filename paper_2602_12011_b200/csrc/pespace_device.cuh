// pespace_device.cuh -- device code of libpespace.so (sm_100a, FP64).
//
// One thread owns one frequency bin and walks over a tile of samples whose
// per-sample constants sit in shared memory (broadcast reads).  For every
// (sample, bin, detector) it evaluates, per mode class m (modes sharing m share
// phase, t_lm and orbit):
//   S2/S3  TaylorF2 phase (in turns) and t_lm(f) from two Horner polynomials in
//          v = (pi Ms 2f/m)^{1/3}                                [Eq. 4, PAPER.md:92]
//   S4     orbit phase at t_lm -> the projections k.x_n, k.n_l, u'.n_l, v'.n_l
//          (all linear in a few sines/cosines, SURVEY.md O8 note)
//   S5-S7  single links + TDI in the algebraically reduced form
//            X = g z h { W_b [k13 (E_3 - cos(th) E_1) - i sin(th) E_1]
//                      - W_c [k12 (E_2 - cos(th) E_1) - i sin(th) E_1] },  th = 2 pi f L,
//          E_n = exp(-2 pi i f k.x_n), W_l = (n_l.P.n_l)/(1-(k.n_l)^2), which is Eq. 5
//           inserted into Eq. 6 -- derivation in DESIGN.md
//   S8     residual against data, weighted by 1/S_n         [Eq. 10, PAPER.md:124]
// The per-bin factors (f^{1/3}, ln f, f^{-5/3}, f^{-8/3}, sin/cos 2 pi f L) and the data and
// weights with g z f^{-7/6} folded in are written once per call by prep_bins_kernel (S0), so the
// inner loop never touches a transcendental or a division of the library.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>
#include <math_constants.h>

#include "pespace_dual.cuh"

namespace pespace {

constexpr int NPAR = 11;

// ---- physical constants (restated, not shared with the oracle)
constexpr double kC = 299792458.0;
constexpr double kGMsun = 1.3271244e20;
constexpr double kGpc = 3.0856775814913673e25;
constexpr double kAU = 149597870700.0;
constexpr double kYear = 31558149.763545603;
constexpr double kEuler = 0.5772156649015329;
constexpr double kPi = 3.14159265358979323846;

// ---- phase units.  Every phase of the inner loop is carried in units of 1/1024 turn ("pu"): range
// reduction is then a subtraction of a multiple of 1024, the integer part of a phase indexes a
// 1024-entry sine/cosine table directly, and no multiplication by 2 pi ever happens per bin.
constexpr double kTurn = 1024.0;                 // pu per turn
constexpr double kRadPerPu = 2.0 * kPi / kTurn;  // radians per pu
constexpr int NTAB = 1024;                       // table entries per turn (one per pu)
constexpr double kMagic = 6755399441055744.0;    // 1.5 * 2^52: x + kMagic rounds x to an integer (|x| < 2^51)

// ---- per-sample constant block (doubles)
enum : int {
  W_A = 0,      // (pi Ms)^{1/3}
  W_LNA,        // ln of it (kept for reference: the kernels use the folded W_P5, W_P6, W_Q6 below)
  W_TC,         // t_c
  W_PH0,        // -(phi_c/pi + 1/8): constant phase of the (2,2) mode in turns
  W_P0, W_P2, W_P3, W_P4, W_P5, W_P5L, W_P6, W_P6L, W_P7,   // phase polynomial (turns * f'^{5/3})
  W_Q0, W_Q2, W_Q3, W_Q4, W_Q5, W_Q6, W_Q6L, W_Q7,          // (t_lm - t_c)/yr polynomial
  W_VALID,      // 1.0 valid, 0.0 out of domain
  W_KA,         // [4 mode classes][a+, b+, ax, bx]
  W_MDL = W_KA + 16,   // -1 / D_L (Fisher path)
  W_PAD,
  D_BASE,           // per detector, D_STRIDE doubles
  // offsets of the staged (one detector) view; the block of detector d starts at D_BASE + d D_STRIDE
  S_K = D_BASE + 2,    // kind 0: k/(4 sqrt3): x, y, -z/2*..., -3x, -3y  (5 each), in the frame rotated by lambda0
  S_U = S_K + 5,
  S_V = S_U + 5,
  S_DX = S_V + 5,      // (AU/c) k_x, (AU/c) k_y: Doppler phase of the guiding centre (kind 0: rotated frame)
  S_DY,
};
constexpr int D_STRIDE = 24;
// [19..22] (both kinds): (AU/c) u'_x, u'_y, v'_x, v'_y in the frame of S_DX, S_DY -- the Doppler part of the sky
// "torques" of the adjoint gradient (pespace_grad.cuh); unused by the other kernels
enum : int { S_UX = D_BASE + 19, S_UY, S_VX, S_VY };
// kind 0: [0] alpha0 - lambda0 (pu), [2..16] S_K, S_U, S_V, [17..18] S_DX, S_DY.  The constellation with rotation
//         phase lambda0 is the lambda0 = 0 constellation at orbital phase alpha - lambda0, rotated about z by lambda0:
//         the rotation is applied to k, u', v' here, so the kernels only ever see spacecraft at 0, 120, 240 degrees.
// kind 1: [0] alphaE0, [1] phi0 (pu), [2..7] (w.e1, w.e2)/sqrt3 for w = k, u', v', [17..18] S_DX, S_DY
constexpr int SMEM_STRIDE = D_BASE + D_STRIDE;   // one sample, one detector
static_assert(SMEM_STRIDE == 64, "sample block is 64 doubles");
__host__ __device__ constexpr int sample_stride(int n_det) { return D_BASE + D_STRIDE * n_det; }

// (m/2)^{7/6} for the amplitude (host/prep side)
__device__ constexpr double kM76[4] = {0.44544935907016965237, 1.0, 1.6048697909004944263, 2.2449240966187459629};

// ---- per-detector constants (kernel parameter)
struct DetC {
  double Lbar;        // L / c  (s)
  double yr_over_p;   // kind 1
  double kappa, lambda0, period_s, lon, lat;   // raw, for the prep kernel
  int kind, gen;
};

struct GridC { double f0, df; long long N; };

// ---- per-bin constants (registers)
struct BinC { double fT, cf, lnf3, fm53, fm83, fm76, sth, cth; };   // fT = kTurn f

// ---- FP64 helpers written for this kernel (the library sincospi/division carry quadrant,
// special-value and slow-path logic that the FP64-bound inner loop cannot afford)

// round to nearest integer without FRND/F2I (quarter-rate conversion unit): two full-rate DADDs
__device__ __forceinline__ double rint_magic(double x) { return (x + kMagic) - kMagic; }
// nearest multiple of one turn (kTurn = 2^10 pu) the same way: 1.5 * 2^62 has ulp 2^10 (|x| < 2^61)
constexpr double kMagicTurn = 6917529027641081856.0;
static_assert(kTurn == 1024.0, "kMagicTurn rounds to multiples of 2^10");
__device__ __forceinline__ double whole_turns(double x) { return (x + kMagicTurn) - kMagicTurn; }
// x * y modulo one turn with a single rounding: the multiple of kTurn nearest to the rounded product is removed
// inside an fma (the exact product minus that multiple is at most ~kTurn/2 in magnitude)
__device__ __forceinline__ double mul_mod_turn(double x, double y) { return fma(x, y, -whole_turns(x * y)); }

// sin and cos of (pi/2) x, x in QUARTER TURNS, |x| < 2^30.  Octant reduction y = x - rint(x),
// then near-minimax polynomials in y^2 on |y| <= 1/2 (max abs error 1.2e-16 / 1.8e-16,
// coefficients from a Chebyshev-node fit in 60-digit arithmetic).
__device__ __forceinline__ void sincos_qt(double x, double& s_out, double& c_out) {
  const double qf = rint(x);
  const double y = x - qf;
  const int q = __double2int_rn(qf);
  const double z = y * y;
  double ps = fma(5.633933781537854e-08, z, -3.59864335298231e-06);
  ps = fma(ps, z, 0.0001604411507421909);
  ps = fma(ps, z, -0.004681754132340976);
  ps = fma(ps, z, 0.07969262624604301);
  ps = fma(ps, z, -0.6459640975062443);
  ps = fma(ps, z, 1.5707963267948966);
  ps *= y;
  double pc = fma(4.6552961874867623e-07, z, -2.520013526428479e-05);
  pc = fma(pc, z, 0.000919259950041661);
  pc = fma(pc, z, -0.02086348073494657);
  pc = fma(pc, z, 0.25366950789986475);
  pc = fma(pc, z, -1.2337005501361513);
  pc = fma(pc, z, 1.0);
  // quadrant: q odd swaps, sign of sin = bit1(q), sign of cos = bit1(q+1); applied on the high words
  const bool odd = q & 1;
  int sh = __double2hiint(odd ? pc : ps), sl = __double2loint(odd ? pc : ps);
  int ch = __double2hiint(odd ? ps : pc), cl = __double2loint(odd ? ps : pc);
  sh ^= (q & 2) << 30;
  ch ^= ((q + 1) & 2) << 30;
  s_out = __hiloint2double(sh, sl);
  c_out = __hiloint2double(ch, cl);
}

// 1/x for x > 0: hardware seed (rcp.approx.ftz.f64, ~2^-20) + one cubic Newton step (3 DFMA)
__device__ __forceinline__ double rcp_pos(double x) {
  double r;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(x));
  const double e = fma(-x, r, 1.0);
  const double t = fma(e, e, e);
  return fma(r, t, r);
}

// sin and cos of a phase u in pu (|u| < 2^31) from the 1024-entry table T[j] = (sin, cos)(2 pi j / 1024)
// in shared memory: j = rint(u) mod 1024 (low word of u + kMagic), y = u - rint(u) in [-1/2, 1/2] pu,
// i.e. |theta| <= pi/1024, where sin(theta) = y (A1 + A3 y^2) and cos(theta) - 1 = y^2 (B2 + B4 y^2)
// (Taylor with the theta^5 term economised onto the lower ones: max error 1.4e-16 / 1.2e-18), then
// the angle-addition formulas.  12 FP64 instructions, no quadrant logic, no conversion instructions.
// (Evaluating the two small terms in FP32 was tried and dropped: every non-FP64 instruction costs an issue
// cycle that the FP64 pipe cannot use, and the 1e-12 error shows in the cancelling T channel.)
constexpr double kHh = 0.5 * kRadPerPu;   // half-width of the reduced interval, radians
constexpr double kA1 = kRadPerPu * (1.0 - (5.0 / 16.0) * (kHh * kHh * kHh * kHh) / 120.0);
constexpr double kA3 = kRadPerPu * kRadPerPu * kRadPerPu * (-1.0 / 6.0 + (5.0 / 4.0) * (kHh * kHh) / 120.0);
constexpr double kB2 = -0.5 * kRadPerPu * kRadPerPu;
constexpr double kB4 = kRadPerPu * kRadPerPu * kRadPerPu * kRadPerPu / 24.0;

__device__ __forceinline__ void sincos_tab(double u, const double2* __restrict__ tab, double& s_out, double& c_out) {
  const double t = u + kMagic;
  const double y = u - (t - kMagic);
  const double2 T = tab[__double2loint(t) & (NTAB - 1)];
  const double z = y * y;
  const double sl = y * fma(kA3, z, kA1);
  const double cl = z * fma(kB4, z, kB2);
  s_out = fma(T.y, sl, fma(T.x, cl, T.x));
  c_out = fma(-T.x, sl, fma(T.y, cl, T.y));
}

// phase in pu -> sin, cos; TAB selects the table (likelihood / response kernels) or the polynomial
// (kernels whose shared memory is spoken for)
template <bool TAB>
__device__ __forceinline__ void sincos_pu(double u, const double2* __restrict__ tab, double& s_out, double& c_out) {
  if constexpr (TAB) sincos_tab(u, tab, s_out, c_out);
  else sincos_qt(u * (4.0 / kTurn), s_out, c_out);
}

__device__ __forceinline__ BinC make_bin(double f, double Lbar) {
  BinC b;
  b.fT = kTurn * f;
  b.cf = cbrt(f);
  b.lnf3 = log(f) * (1.0 / 3.0);
  const double cf2 = b.cf * b.cf;
  b.fm53 = 1.0 / (f * cf2);
  b.fm83 = b.fm53 / f;
  b.fm76 = sqrt(b.fm53 / cf2);
  sincospi(2.0 * f * Lbar, &b.sth, &b.cth);   // theta = 2 pi f L
  return b;
}

// g(z) z f^{-7/6} of Eq. 6 (z = e^{-i theta})
__device__ __forceinline__ void tdi_prefactor(const BinC& b, int gen, double& gr, double& gi) {
  const double zr = b.cth, zi = -b.sth;
  const double z2r = zr * zr - zi * zi, z2i = 2.0 * zr * zi;
  double ar = 1.0 - z2r, ai = -z2i;                        // 1 - z^2
  if (gen == 20) {
    const double z4r = z2r * z2r - z2i * z2i, z4i = 2.0 * z2r * z2i;
    const double br = 1.0 - z4r, bi = -z4i;                // 1 - z^4
    const double tr = ar * br - ai * bi, ti = ar * bi + ai * br;
    ar = tr; ai = ti;
  }
  gr = (ar * zr - ai * zi) * b.fm76;
  gi = (ar * zi + ai * zr) * b.fm76;
}

template <int KIND, bool FIRST, bool TAB>
__device__ __forceinline__ void eval_geom(const BinC& bc, const double* __restrict__ sc, const DetC& dc,
                                          const double2* __restrict__ tab, double psi, double tau, double CKp,
                                          double CKc, double (&S)[6]);

// ---------------------------------------------------------------------------------------------
// One mode class (m = MC + 1) of one (sample, bin, detector): adds its X, Y, Z (without the common
// factor g z f^{-7/6}) to S.  All phases are carried in pu = 1/1024 turn (the prep kernel scales the
// polynomial coefficients by kTurn) so that the sine/cosine evaluation needs no multiply.
template <int KIND, int MC, bool FIRST, bool TAB>
__device__ __forceinline__ void eval_class(const BinC& bc, const double* __restrict__ sc, const DetC& dc,
                                           const double2* __restrict__ tab, double va, double La, double ftc,
                                           double (&S)[6]) {
  // compile-time class constants: (2/m)^{1/3}, ln(2/m)/3, (m/2)^{8/3}, m/2
  constexpr double CB[4] = {1.2599210498948731648, 1.0, 0.87358046473629886905, 0.79370052598409973738};
  constexpr double LN3[4] = {0.23104906018664843647, 0.0, -0.13515503603605479399, -0.23104906018664843647};
  constexpr double S83[4] = {0.1574901312368591456, 1.0, 2.948334068485008683, 6.349604207872797899};
  constexpr double MH[4] = {0.5, 1.0, 1.5, 2.0};
  // ---- S2/S3: v, ln v, phase and t_lm
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
  double psi = ((MC == 1) ? bc.fm53 : S83[MC] * bc.fm53) * P;     // PN phase, pu (up to ~1e8 and beyond)
  psi -= whole_turns(psi);                                         // mod one turn, exact
  psi += fma(MH[MC], sc[W_PH0], ftc);                              // + kTurn [f t_c - (m/2)(phi_c/pi + 1/8)]
  const double tau = ((MC == 1) ? bc.fm83 : S83[MC] * bc.fm83) * Q;   // kTurn (t_lm - t_c) / yr

  // ---- amplitude x polarisation content of the class: vp (a + b v^2)
  const double* ka = sc + W_KA + 4 * MC;
  double CKp, CKc;
  if (MC == 1) { CKp = fma(ka[1], v2, ka[0]); CKc = fma(ka[3], v2, ka[2]); }
  else if (MC == 3) { CKp = v2 * ka[0]; CKc = v2 * ka[2]; }
  else { CKp = v * ka[0]; CKc = v * ka[2]; }

  eval_geom<KIND, FIRST, TAB>(bc, sc, dc, tab, psi, tau, CKp, CKc, S);
}

// S4-S7 of one mode (class) of one (sample, bin, detector) from its phase psi (pu, reduced), its time tau =
// kTurn (t_lm - t_c) / yr and its amplitudes CKp, CKc (amplitude x polarisation content): adds X, Y, Z (without
// the common per-bin factor) to S.  Shared by the analytic classes (eval_class) and the tabulated modes.
template <int KIND, bool FIRST, bool TAB>
__device__ __forceinline__ void eval_geom(const BinC& bc, const double* __restrict__ sc, const DetC& dc,
                                          const double2* __restrict__ tab, double psi, double tau, double CKp,
                                          double CKc, double (&S)[6]) {
  // ---- S4: orbit phase(s) and the two rotating combinations G1, G2 of each of k, u', v'
  double G1k, G2k, G1u, G2u, G1v, G2v, kR;
  if (KIND == 0) {
    double sa, ca;
    sincos_pu<TAB>(sc[D_BASE] + tau, tab, sa, ca);
    const double c2 = fma(2.0 * ca, ca, -1.0), s2 = 2.0 * sa * ca;
    const double* w = sc + S_K;
    G1k = fma(w[0], c2, fma(w[1], s2, fma(w[2], ca, w[3])));
    G2k = fma(w[0], s2, fma(-w[1], c2, fma(w[2], sa, w[4])));
    w = sc + S_U;
    G1u = fma(w[0], c2, fma(w[1], s2, fma(w[2], ca, w[3])));
    G2u = fma(w[0], s2, fma(-w[1], c2, fma(w[2], sa, w[4])));
    w = sc + S_V;
    G1v = fma(w[0], c2, fma(w[1], s2, fma(w[2], ca, w[3])));
    G2v = fma(w[0], s2, fma(-w[1], c2, fma(w[2], sa, w[4])));
    kR = fma(sc[S_DX], ca, sc[S_DY] * sa);
  } else {
    double sE, cE, sp, cp;
    sincos_pu<TAB>(sc[D_BASE] + tau, tab, sE, cE);
    sincos_pu<TAB>(fma(tau, dc.yr_over_p, sc[D_BASE + 1]), tab, sp, cp);
    const double* w = sc + D_BASE + 2;
    G1k = fma(w[0], cp, w[1] * sp); G2k = fma(w[1], cp, -w[0] * sp);
    G1u = fma(w[2], cp, w[3] * sp); G2u = fma(w[3], cp, -w[2] * sp);
    G1v = fma(w[4], cp, w[5] * sp); G2v = fma(w[5], cp, -w[4] * sp);
    kR = fma(sc[S_DX], cE, sc[S_DY] * sE);
  }
  // Spacecraft n sits at angle 2 pi (n-1)/3 (cos = 1, -1/2, -1/2; sin = 0, r, -r with r = sqrt3/2), so
  // w.delta_n / L = (G1, -G1/2 + r G2, -G1/2 - r G2) and along the arms a: 2-3, b: 3-1, c: 1-2
  // w.n_l = (2 r G2, -3/2 G1 - r G2, 3/2 G1 - r G2): literal coefficients, no per-detector constants.
  constexpr double R3H = 0.86602540378443864676;
  const double tk = R3H * G2k;
  const double nu0 = G1k, nu1 = fma(-0.5, G1k, tk), nu2 = fma(-0.5, G1k, -tk);     // k.delta_n / L
  const double ka_ = tk + tk, kb_ = fma(-1.5, G1k, -tk), kc_ = fma(1.5, G1k, -tk);  // k.n_23, k.n_31, k.n_12
  const double tu = R3H * G2u, tv = R3H * G2v;
  const double ul[3] = {tu + tu, fma(-1.5, G1u, -tu), fma(1.5, G1u, -tu)};
  const double vl[3] = {tv + tv, fma(-1.5, G1v, -tv), fma(1.5, G1v, -tv)};

  // ---- S5: W_l = amplitude * (n_l.P.n_l) / (1 - (k.n_l)^2), with 1-(k.n)^2 = (u'.n)^2 + (v'.n)^2
  double Wr[3], Wi[3];
#pragma unroll
  for (int l = 0; l < 3; ++l) {
    const double uu = ul[l], vv = vl[l];
    const double v2_ = vv * vv;
    const double D = fma(uu, uu, v2_);
    const double rD = (__double2hiint(D) > 0) ? rcp_pos(D) : 0.0;   // D >= 0: sign/exponent test on the ALU pipe
    Wr[l] = (CKp * rD) * fma(uu, uu, -v2_);
    Wi[l] = (CKc * rD) * (uu * vv);
  }

  // ---- S6: h_lm E_n = exp(-i (2 pi / kTurn) (psi + kTurn f k.x_n)) for the three spacecraft
  double Er[3], Ei[3];
  {
    const double nun[3] = {nu0, nu1, nu2};
    const double fTL = bc.fT * dc.Lbar;              // per bin: hoisted out of the sample loop
    const double base = fma(bc.fT, kR, psi);         // phase at the guiding centre
#pragma unroll
    for (int n = 0; n < 3; ++n) {
      double s, c;
      sincos_pu<TAB>(fma(fTL, nun[n], base), tab, s, c);
      Er[n] = c; Ei[n] = s;          // note: Ei holds +sin; the minus sign is carried below
    }
  }
  // ---- S7: brackets  B(r,s,kap) = kap (E_s - cos(th) E_r) - i sin(th) E_r  and the TDI sums, with
  // E = Er - i Ei and W = Wr - i Wi:   Re(W B) = Wr Br - Wi Bi',  -Im(W B) = Wr Bi' + Wi Br
  // (Bi' = -Im B).  S accumulates (Re, -Im); the sign is restored when the residual is formed.
  auto add = [&](double& Sr, double& Si, int r, int s_, double kap, double wr, double wi, bool init) {
    const double br = fma(kap, fma(-bc.cth, Er[r], Er[s_]), -bc.sth * Ei[r]);
    const double bi = fma(kap, fma(-bc.cth, Ei[r], Ei[s_]), bc.sth * Er[r]);
    if (init) {
      Sr = fma(wr, br, -wi * bi);
      Si = fma(wr, bi, wi * br);
    } else {
      Sr = fma(wr, br, fma(-wi, bi, Sr));
      Si = fma(wr, bi, fma(wi, br, Si));
    }
  };
  // arms: index 0 = a (2-3), 1 = b (3-1), 2 = c (1-2)
  add(S[0], S[1], 0, 2, -kb_, Wr[1], Wi[1], FIRST);   // X: + W_b B(1,3,k13)
  add(S[0], S[1], 0, 1, kc_, -Wr[2], -Wi[2], false);  //    - W_c B(1,2,k12)
  add(S[2], S[3], 1, 0, -kc_, Wr[2], Wi[2], FIRST);   // Y: + W_c B(2,1,k21)
  add(S[2], S[3], 1, 2, ka_, -Wr[0], -Wi[0], false);  //    - W_a B(2,3,k23)
  add(S[4], S[5], 2, 1, -ka_, Wr[0], Wi[0], FIRST);   // Z: + W_a B(3,2,k32)
  add(S[4], S[5], 2, 0, kb_, -Wr[1], -Wi[1], false);  //    - W_b B(3,1,k31)
}

// X, Y, Z of one (sample, bin, detector) summed over the mode classes of CMASK (compile time;
// bit m-1 set = class m present).  Returns (Re, -Im) pairs in S.
template <int KIND, unsigned CMASK, bool TAB>
__device__ __forceinline__ void eval_xyz(const BinC& bc, const double* __restrict__ sc, const DetC& dc,
                                         const double2* __restrict__ tab, double (&S)[6]) {
  const double tc = sc[W_TC];
  // kTurn f t_c in pu mod one turn, with the rounding error of the product recovered by fma
  const double ftc = mul_mod_turn(bc.fT, tc);
  const double va = sc[W_A] * bc.cf, La = bc.lnf3;     // ln (pi Ms)^{1/3} is folded into W_P5, W_P6, W_Q6
  constexpr bool c0 = CMASK & 1u, c1 = CMASK & 2u, c2 = CMASK & 4u, c3 = CMASK & 8u;
  if (c0) eval_class<KIND, 0, true, TAB>(bc, sc, dc, tab, va, La, ftc, S);
  if (c1) eval_class<KIND, 1, !c0, TAB>(bc, sc, dc, tab, va, La, ftc, S);
  if (c2) eval_class<KIND, 2, !(c0 || c1), TAB>(bc, sc, dc, tab, va, La, ftc, S);
  if (c3) eval_class<KIND, 3, !(c0 || c1 || c2), TAB>(bc, sc, dc, tab, va, La, ftc, S);
}

// ---------------------------------------------------------------------------------------------
// S1: per-sample constants.  One thread per sample; plain double-precision library math.  The body
// is written once on a scalar type T: double for the likelihood / response path, Du<7> (tangents
// w.r.t. M, q, chi1, chi2, iota, lambda, beta) for the Fisher path.  `put(idx, value)` stores one
// constant of the sample block.
struct PrepArgs { DetC det[8]; int n_det; unsigned mode_mask; };

template <class T>
__device__ __forceinline__ void swsh_pairs(const T& iota, T Yp[5], T Ym[5]) {
  // -2Y_lm(iota, 0) closed forms for (2,2),(2,1),(3,3),(3,2),(4,4) and their -m partners
  const T c = p_cos(iota), s = p_sin(iota), C = p_cos(iota * 0.5), Sh = p_sin(iota * 0.5);
  const double n22 = 0.15769578262626000302, n21 = 0.31539156525252000603;
  const double n33 = 1.8281831978578629446, n3 = 1.4927053303604615657;
  const T C2 = C * C, S2 = Sh * Sh;
  Yp[0] = n22 * ((1.0 + c) * (1.0 + c));        Ym[0] = n22 * ((1.0 - c) * (1.0 - c));
  Yp[1] = n21 * (s * (1.0 + c));                Ym[1] = n21 * (s * (1.0 - c));
  Yp[2] = -n33 * (C2 * C2 * C * Sh);            Ym[2] = n33 * (C * S2 * S2 * Sh);
  Yp[3] = (n3 * 0.5) * (C2 * C2 * (3.0 * c - 2.0));  Ym[3] = (n3 * 0.5) * (S2 * S2 * (3.0 * c + 2.0));
  Yp[4] = (3.0 * n3) * (C2 * C2 * C2 * S2);     Ym[4] = (3.0 * n3) * (C2 * S2 * S2 * S2);
}

__device__ __forceinline__ bool sample_in_domain(const double* th) {
  bool ok = true;
  for (int i = 0; i < NPAR; ++i) ok = ok && isfinite(th[i]);
  return ok && th[0] > 0.0 && th[1] >= 1.0 && th[4] > 0.0;
}

// Frame and detector blocks of the per-sample constants (O7, O8): the sky basis with the polarisation angle
// absorbed, projected on the orbit basis of every detector, and the orbital phases at t_c.
template <class T, class Put>
__device__ void prep_frame(const T& lam, const T& bet, const T& pol, const T& tc, const PrepArgs& A, Put put,
                           int det_lo = 0, int det_hi = PESPACE_MAX_DET) {
  // detectors det_lo <= d < min(det_hi, n_det): all of them by default; one per thread in prep_samples_kernel
  // frame (O7) with the polarisation angle absorbed into the basis: u' = cos(psi) u + sin(psi) v, ...
  const T cl = p_cos(lam), sl = p_sin(lam), cb = p_cos(bet), sb = p_sin(bet), cp = p_cos(pol), sp = p_sin(pol);
  const T k[3] = {-(cb * cl), -(cb * sl), -sb};
  const T u[3] = {sl, -cl, T(0.0)};
  const T v[3] = {-(sb * cl), -(sb * sl), cb};
  T up[3], vp[3];
  for (int i = 0; i < 3; ++i) { up[i] = cp * u[i] + sp * v[i]; vp[i] = cp * v[i] - sp * u[i]; }
  const double r43 = 1.0 / (4.0 * sqrt(3.0));
  const T* W3[3] = {k, up, vp};
  const int off[3] = {S_K - D_BASE, S_U - D_BASE, S_V - D_BASE};
  const double tcv = p_val(tc);
  for (int dI = det_lo; dI < A.n_det && dI < det_hi; ++dI) {
    const DetC& D = A.det[dI];
    const int base = D_BASE + D_STRIDE * dI;
    for (int i = 0; i < D_STRIDE; ++i) put(base + i, T(0.0));
    double a0 = tcv / kYear;
    a0 -= rint(a0);
    if (D.kind == 0) {
      // orbital phase and sky basis in the frame rotated about z by lambda0 (see the layout note above)
      put(base, T(kTurn * (a0 + (D.kappa - D.lambda0) / (2.0 * kPi))));
      const double cL0 = cos(D.lambda0), sL0 = sin(D.lambda0);
      for (int j = 0; j < 3; ++j) {
        const T* w = W3[j];
        const T wx = cL0 * w[0] + sL0 * w[1], wy = cL0 * w[1] - sL0 * w[0];
        put(base + off[j] + 0, wx * r43); put(base + off[j] + 1, wy * r43); put(base + off[j] + 2, -0.5 * w[2]);
        put(base + off[j] + 3, -3.0 * r43 * wx); put(base + off[j] + 4, -3.0 * r43 * wy);
        if (j == 0) { put(base + (S_DX - D_BASE), (kAU / kC) * wx); put(base + (S_DY - D_BASE), (kAU / kC) * wy); }
        if (j == 1) { put(base + (S_UX - D_BASE), (kAU / kC) * wx); put(base + (S_UY - D_BASE), (kAU / kC) * wy); }
        if (j == 2) { put(base + (S_VX - D_BASE), (kAU / kC) * wx); put(base + (S_VY - D_BASE), (kAU / kC) * wy); }
      }
    } else {
      put(base + (S_DX - D_BASE), (kAU / kC) * k[0]); put(base + (S_DY - D_BASE), (kAU / kC) * k[1]);
      put(base + (S_UX - D_BASE), (kAU / kC) * up[0]); put(base + (S_UY - D_BASE), (kAU / kC) * up[1]);
      put(base + (S_VX - D_BASE), (kAU / kC) * vp[0]); put(base + (S_VY - D_BASE), (kAU / kC) * vp[1]);
      put(base, T(kTurn * a0));
      double p0 = tcv / D.period_s;
      p0 -= rint(p0);
      put(base + 1, T(kTurn * (p0 + D.lambda0 / (2.0 * kPi))));
      const double cL = cos(D.lon), sL = sin(D.lon), cB = cos(D.lat), sB = sin(D.lat);
      const double nh[3] = {cB * cL, cB * sL, sB};
      const double e1[3] = {-sL, cL, 0.0};
      const double e2[3] = {nh[1] * e1[2] - nh[2] * e1[1], nh[2] * e1[0] - nh[0] * e1[2], nh[0] * e1[1] - nh[1] * e1[0]};
      const double r3 = 1.0 / sqrt(3.0);
      for (int j = 0; j < 3; ++j) {
        const T* w = W3[j];
        put(base + 2 + 2 * j, r3 * (w[0] * e1[0] + w[1] * e1[1] + w[2] * e1[2]));
        put(base + 3 + 2 * j, r3 * (w[0] * e2[0] + w[1] * e2[1] + w[2] * e2[2]));
      }
    }
  }
}

// sec < 0: the whole block of constants (one thread per sample: the Fisher / gradient tangents, the orbit-table path).
// sec >= 0: one of its 2 + n_det independent SECTIONS -- 0: phase and time polynomials, 1: mode amplitudes and
// polarisation content, 2 + d: sky basis on the orbit basis of detector d -- so that prep_samples_kernel can give a
// sample to 2 + n_det threads: the one-thread version is a chain of ~20 dependent library calls (cbrt, log, ten
// divisions, eight sine / cosine pairs), 9.6 us for a single sample, which is the floor of the single-theta regime
// (DESIGN.md 5.5).  Every constant is computed by the same expression in either mode.
template <class T, class Put>
__device__ void prep_sample(const T (&th)[NPAR], const PrepArgs& A, Put put, int sec = -1) {
  const T M = th[0], q = th[1], chi1 = th[2], chi2 = th[3], DL = th[4], iota = th[5], phic = th[6],
          lam = th[7], bet = th[8], pol = th[9], tc = th[10];
  if (sec >= 2) {
    prep_frame(lam, bet, pol, tc, A, put, sec - 2, sec - 1);
    return;
  }
  const T Ms = M * (kGMsun / (kC * kC * kC));
  const T eta = q / ((1.0 + q) * (1.0 + q)), delta = (q - 1.0) / (q + 1.0);
  const T mu1 = q / (1.0 + q), mu2 = 1.0 / (1.0 + q);
  const T Ds = DL * (kGpc / kC);
  if (sec <= 0) {                                        // ---- section 0: phase and time polynomials
    const T a = p_cbrt(kPi * Ms);
    const T lna = p_log(a);
    put(W_A, a); put(W_LNA, lna); put(W_TC, tc);
    put(W_PH0, -kTurn * (phic / kPi + 0.125));            // pu, for m/2 = 1
    put(W_VALID, T(1.0));
    // TaylorF2 3.5PN coefficients, spin terms per G3
    const double pi2 = kPi * kPi;
    const T bso = (113.0 / 12.0 * (mu1 * mu1) + 6.25 * eta) * chi1 + (113.0 / 12.0 * (mu2 * mu2) + 6.25 * eta) * chi2;
    const T sss = 79.0 / 8.0 * (eta * chi1 * chi2);
    const T ph2 = 3715.0 / 756.0 + 55.0 / 9.0 * eta;
    const T ph3 = -16.0 * kPi + 4.0 * bso;
    const T ph4 = 15293365.0 / 508032.0 + 27145.0 / 504.0 * eta + 3085.0 / 72.0 * (eta * eta) - 10.0 * sss;
    const T ph5a = kPi * (38645.0 / 756.0 - 65.0 / 9.0 * eta);          // phi5 = ph5a (1 + 3 ln v)
    const T ph6a = 11583231236531.0 / 4694215680.0 - 640.0 / 3.0 * pi2 - 6848.0 / 21.0 * kEuler +
                   eta * (-15737765635.0 / 3048192.0 + 2255.0 / 12.0 * pi2) + 76055.0 / 1728.0 * (eta * eta) -
                   127825.0 / 1296.0 * (eta * eta * eta) - 6848.0 / 21.0 * log(4.0);   // phi6 = ph6a - 6848/21 ln v
    const double ph6l = -6848.0 / 21.0;
    const T ph7 = kPi * (77096675.0 / 254016.0 + 378515.0 / 1512.0 * eta - 74045.0 / 756.0 * (eta * eta));
    const T a5 = 1.0 / (a * a * a * a * a);
    const T cP = kTurn * 3.0 / (256.0 * kPi * eta) * a5;  // kTurn Psi/(2 pi) = f'^{-5/3} * sum (cP phi_k) v^k
    put(W_P0, cP); put(W_P2, cP * ph2); put(W_P3, cP * ph3); put(W_P4, cP * ph4);
    // ln v = ln (pi Ms)^{1/3} + ln f'^{1/3}: the sample part of the logarithm is folded into the constant terms, so
    // the kernels multiply the *L coefficients by ln f'^{1/3} only (one add less per bin, no tangent on L)
    put(W_P5, cP * ph5a + cP * 3.0 * ph5a * lna); put(W_P5L, cP * 3.0 * ph5a);
    put(W_P6, cP * ph6a + cP * ph6l * lna); put(W_P6L, cP * ph6l); put(W_P7, cP * ph7);
    const T cQ = cP / (3.0 * kYear);                       // kTurn (t - t_c)/yr = f'^{-8/3} * sum (cQ q_k) v^k
    put(W_Q0, -5.0 * cQ); put(W_Q2, -3.0 * cQ * ph2); put(W_Q3, -2.0 * cQ * ph3); put(W_Q4, -(cQ * ph4));
    put(W_Q5, 3.0 * cQ * ph5a); put(W_Q6, cQ * (ph6a + ph6l) + cQ * ph6l * lna); put(W_Q6L, cQ * ph6l);
    put(W_Q7, 2.0 * cQ * ph7);
    put(W_MDL, -1.0 / DL); put(W_PAD, T(0.0));
  }
  if (sec == 0) return;
  // ---- section 1: amplitudes (O4, O5) and polarisation content (O6) per mode, gathered per class m
  const T amp0 = p_sqrt(2.0 * eta / 3.0) * 0.82630748711075811083 * (Ms * Ms / Ds) / (Ms * p_sqrt(p_cbrt(Ms)));
  const double s57 = sqrt(5.0 / 7.0);
  const T clm[5] = {T(1.0), delta / 3.0, 0.75 * sqrt(15.0 / 14.0) * delta, s57 / 3.0 * (1.0 - 3.0 * eta),
                    8.0 / 9.0 * s57 * (1.0 - 3.0 * eta)};
  const int mm[5] = {2, 1, 3, 2, 4}, ll[5] = {2, 2, 3, 3, 4};
  T Yp[5], Ym[5];
  swsh_pairs(iota, Yp, Ym);
  T kam[16];
  for (int i = 0; i < 16; ++i) kam[i] = T(0.0);
  for (int i = 0; i < 5; ++i) {
    if (!((A.mode_mask >> i) & 1u)) continue;
    const int m = mm[i];
    const double sg = (ll[i] & 1) ? -1.0 : 1.0;
    const T Alm = sqrt(2.0 / m) * clm[i] * amp0 * kM76[m - 1];
    const T Kp = 0.5 * (Yp[i] + sg * Ym[i]);           // K+ (real)
    const T Kc = 0.5 * (Yp[i] - sg * Ym[i]);           // Kx = -i Kc
    const int slot = (i == 3) ? 1 : 0;                 // (3,2) rides on the m=2 class with an extra v^2
    kam[4 * (m - 1) + slot] = Alm * Kp;
    kam[4 * (m - 1) + 2 + slot] = 2.0 * Alm * Kc;      // factor 2 of n.e_x.n = 2 (n.u)(n.v)
  }
  for (int i = 0; i < 16; ++i) put(W_KA + i, kam[i]);
  if (sec == 1) return;
  prep_frame(lam, bet, pol, tc, A, put);                 // ---- sections 2 + d (all of them here: sec < 0)
}

// sine/cosine table of sincos_tab: trig[j] = (sin, cos)(2 pi j / NTAB), |error| <= 1 ulp (sincospi)
__device__ __forceinline__ void fill_trig_entry(double2* __restrict__ trig, long long j) {
  if (trig && j < NTAB) {
    double s, c;
    sincospi((double)j * (2.0 / NTAB), &s, &c);
    trig[j] = make_double2(s, c);
  }
}
__host__ __device__ constexpr long long prep_threads(long long B) { return B > NTAB ? B : (long long)NTAB; }
// threads of prep_samples_kernel: 2 + n_det sections per sample (prep_sample), each section of 32 samples in a warp of
// its own (sections in one warp would run one after the other), at least NTAB threads for the table
__host__ __device__ constexpr long long prep_threads(long long B, int n_det) {
  return ((B + 31) / 32) * 32 * (2 + n_det) > NTAB ? ((B + 31) / 32) * 32 * (2 + n_det) : (long long)NTAB;
}

// grid covers prep_threads(B, n_det) threads: thread j < NTAB also writes table entry j (trig may be null); warp w
// works on section w % (2 + n_det) of the samples 32 (w / (2 + n_det)) + lane
static __global__ void prep_samples_kernel(const double* __restrict__ params, long long B, PrepArgs A,
                                    double* __restrict__ consts, double2* __restrict__ trig) {
  const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  fill_trig_entry(trig, t);
  const int nsec = 2 + A.n_det;
  const long long w = t >> 5;
  const int sec = (int)(w % nsec);
  const long long b = (w / nsec) * 32 + (t & 31);
  if (b >= B) return;
  const double* thp = params + b * NPAR;
  const int stride = sample_stride(A.n_det);
  double* o = consts + b * stride;
  if (!sample_in_domain(thp)) {
    if (sec == 0) {
      for (int i = 0; i < stride; ++i) o[i] = 0.0;
      o[W_A] = 1.0; o[W_VALID] = 0.0;
    }
    return;
  }
  double th[NPAR];
  for (int i = 0; i < NPAR; ++i) th[i] = thp[i];
  prep_sample<double>(th, A, [o](int idx, double val) { o[idx] = val; }, sec);
}

// ---------------------------------------------------------------------------------------------
#ifndef PESPACE_BLOCK
#define PESPACE_BLOCK 256
#endif
constexpr int BLOCK = PESPACE_BLOCK;      // threads = bins per block
#ifndef PESPACE_TILE
#define PESPACE_TILE 64
#endif
constexpr int TILE = PESPACE_TILE;        // samples staged in shared memory per block

// dynamic shared memory of the likelihood / response kernels: [trig table | sample constants | warp partials]
extern __shared__ __align__(16) unsigned char pespace_dyn_smem[];
constexpr size_t kernel_smem_bytes() {
  return sizeof(double) * ((size_t)2 * NTAB + (size_t)TILE * SMEM_STRIDE + (size_t)(BLOCK / 32) * TILE);
}
__device__ __forceinline__ void stage_trig(double2* tab, const double2* __restrict__ trig) {
  for (int i = threadIdx.x; i < NTAB; i += blockDim.x) tab[i] = trig[i];
}

__device__ __forceinline__ void stage_tile(double* smem, const double* __restrict__ consts, long long b0,
                                           long long B, int n_det, int det) {
  // copy [wave+sky | this detector's block] of the tile's samples into smem[.][64]: min(TILE, B - b0) of them, rounded
  // up to a multiple of four (the single-class kernels evaluate four samples per trip) with the tail clamped to B - 1
  const int stride = sample_stride(n_det);
  const int lim = (int)min((long long)TILE, ((B - b0 + 3) / 4) * 4) * SMEM_STRIDE;
  // fixed trip count with a guard inside, so that the loads of a thread are issued together
#pragma unroll
  for (int it = 0; it < TILE * SMEM_STRIDE / BLOCK; ++it) {
    const int i = it * BLOCK + (int)threadIdx.x;
    if (i < lim) {
      const int s = i / SMEM_STRIDE, j = i % SMEM_STRIDE;
      long long b = b0 + s;
      if (b >= B) b = B - 1;
      const int src = (j < D_BASE) ? j : (D_BASE + D_STRIDE * det + (j - D_BASE));
      smem[i] = consts[b * stride + src];
    }
  }
}
static_assert((TILE * SMEM_STRIDE) % BLOCK == 0, "stage_tile assumes BLOCK threads");

// S0: per-bin table of one data set, written once per pespace_loglike call and read by every
// sample tile: [n_det][NBF][N] doubles = the per-bin factors of make_bin and the data / weights with
// g z f^{-7/6} and the 1/sqrt2, 1/sqrt6, 1/sqrt3 of Eq. 3 folded in (Eq. 10: w = 4 df / S_n).
enum : int { BF_FT = 0, BF_CF, BF_LNF3, BF_FM53, BF_FM83, BF_STH, BF_CTH, BF_DR, BF_DI = BF_DR + 3, BF_W = BF_DI + 3,
             NBF = BF_W + 3 };
static_assert(NBF == 16, "bin record is 16 doubles");

static __global__ void prep_bins_kernel(const double2* __restrict__ data, const double* __restrict__ psd, GridC G,
                                        PrepArgs A, int fold_f76, double* __restrict__ bins /* [n_det][NBF][N] */) {
  const long long k = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  const int det = blockIdx.y;
  if (k >= G.N) return;
  const DetC& dc = A.det[det];
  BinC bc = make_bin(fma((double)k, G.df, G.f0), dc.Lbar);
  if (!fold_f76) bc.fm76 = 1.0;          // 0: tabulated waveforms carry their own amplitude (pespace_tab.cuh)
  double gr, gi;
  tdi_prefactor(bc, dc.gen, gr, gi);
  double g2 = gr * gr + gi * gi;
  // Reading G9: the weight of a bin depends on the PSD alone.  Where g(z) is EXACTLY 0 (2 f L / c an exact integer:
  // the template vanishes identically) the bin keeps its theta-independent term |d|^2 4 df / S of Eq. 10: a stand-in
  // prefactor of 1e-100 makes the folded data d / g huge against the (then negligible) folded template while
  // w |g|^2 |d / g|^2 = w |d|^2 stays exact; nothing over- or underflows for |d|, 1/S of detector-like magnitude.
  if (!(g2 > 0.0)) { gr = 1e-100; gi = 0.0; g2 = 1e-200; }
  double* o = bins + (size_t)det * NBF * (size_t)G.N + (size_t)k;
  const size_t N = (size_t)G.N;
  o[BF_FT * N] = bc.fT; o[BF_CF * N] = bc.cf; o[BF_LNF3 * N] = bc.lnf3; o[BF_FM53 * N] = bc.fm53;
  o[BF_FM83 * N] = bc.fm83; o[BF_STH * N] = bc.sth; o[BF_CTH * N] = bc.cth;
  const double nrm[3] = {1.4142135623730950488, 2.4494897427831780982, 1.7320508075688772935};
#pragma unroll
  for (int c = 0; c < 3; ++c) {
    const size_t idx = ((size_t)det * 3 + c) * N + (size_t)k;
    const double Sn = psd[idx];
    const bool use = isfinite(Sn) && Sn > 0.0;
    // a masked bin (PSD 0, negative or non-finite) is skipped WITHOUT looking at its data: NaN / Inf there must not
    // reach the sums (0 * NaN = NaN)
    double vr = 0.0, vi = 0.0, vw = 0.0;
    if (use) {
      const double2 d = data ? data[idx] : make_double2(0.0, 0.0);   // no data set: Fisher matrix only
      const double sc_ = nrm[c] / g2;
      vr = (d.x * gr + d.y * gi) * sc_;                    // d * conj(g) / |g|^2 * nrm
      vi = (d.x * gi - d.y * gr) * sc_;                    // MINUS the imaginary part: eval_xyz returns (Re, -Im)
      vw = (4.0 * G.df / Sn) * g2 / (nrm[c] * nrm[c]);
    }
    if (fold_f76 == 2) {           // mixed-precision kernel (pespace_mixed.cuh): whitened data, sqrt(w) / 2^64
      const double sq = sqrt(vw);
      vr *= sq; vi *= sq; vw = sq * (1.0 / 18446744073709551616.0);
    }
    o[(BF_DR + c) * N] = vr;
    o[(BF_DI + c) * N] = vi;
    o[(BF_W + c) * N] = vw;
  }
}

// K_main: grid (bin blocks, sample tiles); one launch per detector.
__host__ __device__ constexpr int popc4(unsigned m) { return (m & 1) + ((m >> 1) & 1) + ((m >> 2) & 1) + ((m >> 3) & 1); }

template <int KIND, unsigned CMASK>
// single-class kernels: two resident blocks per SM (128 registers) run 1.7 % faster than three (80 registers, with
// re-materialised constants and a spill), and 5 % faster than one
#ifndef PESPACE_MINB1
#define PESPACE_MINB1 2
#endif
// multi-class kernels: ONE resident block per SM (255 registers, no spills) beats two at 128 registers with 58
// spill instructions per unit (config 3: 59.5 vs 63.9 ms); 8 warps per SM keep the FP64 issue port busy
#ifndef PESPACE_MINBM
#define PESPACE_MINBM 1
#endif
__global__ void __launch_bounds__(BLOCK, popc4(CMASK) == 1 ? PESPACE_MINB1 : PESPACE_MINBM)
loglike_kernel(const double* __restrict__ consts, const double2* __restrict__ trig, long long B,
               const double* __restrict__ bins /* [n_det][NBF][N] */, long long N, DetC dc, int n_det, int det,
               double* __restrict__ partial /* [n_det][gridDim.x][B] */) {
  double2* tab = reinterpret_cast<double2*>(pespace_dyn_smem);
  double* smem = reinterpret_cast<double*>(tab + NTAB);
  double (*red)[TILE] = reinterpret_cast<double (*)[TILE]>(smem + TILE * SMEM_STRIDE);
  const long long b0 = (long long)blockIdx.y * TILE;
  stage_trig(tab, trig);
  stage_tile(smem, consts, b0, B, n_det, det);

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
  const int ns = (int)min((long long)TILE, B - b0);
  // weighted |d - h|^2 of this thread's bin for sample s of the tile (S8)
  auto term = [&](int s) {
    double S[6];
    eval_xyz<KIND, CMASK, true>(bc, smem + s * SMEM_STRIDE, dc, tab, S);
    const double Ar = S[4] - S[0], Ai = S[5] - S[1];                         // Z - X
    const double Er_ = S[0] - 2.0 * S[2] + S[4], Ei_ = S[1] - 2.0 * S[3] + S[5];   // X - 2Y + Z
    const double Tr = S[0] + S[2] + S[4], Ti = S[1] + S[3] + S[5];           // X + Y + Z
    double r0 = dr[0] - Ar, r1 = di[0] - Ai;
    double acc = w[0] * fma(r0, r0, r1 * r1);
    r0 = dr[1] - Er_; r1 = di[1] - Ei_;
    acc = fma(w[1], fma(r0, r0, r1 * r1), acc);
    r0 = dr[2] - Tr; r1 = di[2] - Ti;
    return fma(w[2], fma(r0, r0, r1 * r1), acc);
  };
  if constexpr (popc4(CMASK) == 1) {
    // S9, single-class kernels: four samples per trip, reduced over the warp by a halving butterfly (two halving
    // levels, then three plain ones on ONE value: 6 shuffle-adds per 4 samples instead of 20).  After the halving
    // levels the lanes with bits (4, 3) = (b4, b3) hold sample 2 b4 + b3 of the group.  The ragged tail of a tile
    // (fewer than four samples left) takes the plain five-level tree below.
    const int ns4 = ns & ~3;
    for (int s0 = 0; s0 < ns4; s0 += 4) {
      double a[4];
#pragma unroll
      for (int j = 0; j < 4; ++j) a[j] = term(s0 + j);
      const bool up4 = lane & 16, up3 = lane & 8;
      const double k0 = (up4 ? a[2] : a[0]) + __shfl_xor_sync(0xffffffffu, up4 ? a[0] : a[2], 16);
      const double k1 = (up4 ? a[3] : a[1]) + __shfl_xor_sync(0xffffffffu, up4 ? a[1] : a[3], 16);
      double acc = (up3 ? k1 : k0) + __shfl_xor_sync(0xffffffffu, up3 ? k0 : k1, 8);
#pragma unroll
      for (int o = 4; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
      if ((lane & 7) == 0) red[warp][s0 + (lane >> 3)] = acc;
    }
    for (int s = ns4; s < ns; ++s) {        // ragged tail of the tile (and batches of fewer than four samples)
      double acc = term(s);
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
      if (lane == 0) red[warp][s] = acc;
    }
  } else {
    for (int s = 0; s < ns; ++s) {
      double acc = term(s);
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
      if (lane == 0) red[warp][s] = acc;
    }
  }
  __syncthreads();
  if (threadIdx.x < ns) {
    double t = 0.0;
#pragma unroll
    for (int wv = 0; wv < BLOCK / 32; ++wv) t += red[wv][threadIdx.x];
    partial[((size_t)det * gridDim.x + blockIdx.x) * (size_t)B + (size_t)(b0 + threadIdx.x)] = t;
  }
}

// K_combine: fixed-order sum over (detector, bin block); lnL = -1/2 sum; out-of-domain -> -inf.  Block = 32 samples x
// CGROUPS slice groups: thread (x, g) sums the slices g, g + CGROUPS, ... of sample 32 blockIdx.x + x (rows of 32
// consecutive samples: coalesced), then the groups are added in the order 0, 1, ... (one thread per sample used to walk
// all slices alone: 0.11 ms per call whatever B)
constexpr int CGROUPS = 16;
static __global__ void combine_kernel(const double* __restrict__ partial, const double* __restrict__ consts, long long B,
                               int n_slices, int stride, double* __restrict__ out) {
  __shared__ double part[CGROUPS][33];
  const int x = threadIdx.x, g = threadIdx.y;
  const long long b = (long long)blockIdx.x * 32 + x;
  double t = 0.0;
  if (b < B) {
    // the loads of eight slices are issued together, the additions keep the order g, g + CGROUPS, ...
    int i = g;
    for (; i + 7 * CGROUPS < n_slices; i += 8 * CGROUPS) {
      double v[8];
#pragma unroll
      for (int u = 0; u < 8; ++u) v[u] = partial[(size_t)(i + u * CGROUPS) * (size_t)B + (size_t)b];
#pragma unroll
      for (int u = 0; u < 8; ++u) t += v[u];
    }
    for (; i < n_slices; i += CGROUPS) t += partial[(size_t)i * (size_t)B + (size_t)b];
  }
  part[g][x] = t;
  __syncthreads();
  if (g == 0 && b < B) {
    double sum = 0.0;
#pragma unroll
    for (int k = 0; k < CGROUPS; ++k) sum += part[k][x];
    out[b] = (consts[b * stride + W_VALID] != 0.0) ? -0.5 * sum : -CUDART_INF;
  }
}
// launch configuration of combine_kernel
#define PESPACE_COMBINE_GRID(B) (unsigned)(((B) + 31) / 32), dim3(32, pespace::CGROUPS)

// pespace_response: same body, writes A, E, T (with the common factor restored).  Like the likelihood kernel the
// single-class instantiations evaluate four samples per trip (independent dependency chains for the FP64 pipe) and all
// instantiations are compiled for the block count per SM that suits their register need.  Non-positive frequencies
// are handled by a zero prefactor, out-of-domain samples by a block-uniform branch: no selects in the sample loop.
template <int KIND, unsigned CMASK>
__global__ void __launch_bounds__(BLOCK, popc4(CMASK) == 1 ? PESPACE_MINB1 : PESPACE_MINBM)
response_kernel(const double* __restrict__ consts, const double2* __restrict__ trig, long long B,
                const double* __restrict__ freqs, long long N, DetC dc, int n_det, int det,
                double2* __restrict__ out /* [B][n_det][3][N] */) {
  double2* tab = reinterpret_cast<double2*>(pespace_dyn_smem);
  double* smem = reinterpret_cast<double*>(tab + NTAB);
  const long long b0 = (long long)blockIdx.y * TILE;
  stage_trig(tab, trig);
  stage_tile(smem, consts, b0, B, n_det, det);
  const long long k = (long long)blockIdx.x * BLOCK + threadIdx.x;
  const bool live = k < N;
  const double fraw = freqs[live ? k : N - 1];
  const bool pos = fraw > 0.0;
  const BinC bc = make_bin(pos ? fraw : 1.0, dc.Lbar);
  double gr, gi;
  tdi_prefactor(bc, dc.gen, gr, gi);
  const double i2 = 0.70710678118654752440, i6 = 0.40824829046386301637, i3 = 0.57735026918962576451;
  // the channel normalisations folded into the prefactor; f <= 0: zeros (the body runs on f = 1 and is finite)
  const double gA[2] = {pos ? gr * i2 : 0.0, pos ? gi * i2 : 0.0};
  const double gE[2] = {pos ? gr * i6 : 0.0, pos ? gi * i6 : 0.0};
  const double gT[2] = {pos ? gr * i3 : 0.0, pos ? gi * i3 : 0.0};
  __syncthreads();
  const int ns = (int)min((long long)TILE, B - b0);
  double2* const obase = out + ((size_t)b0 * n_det + det) * 3 * (size_t)N + (size_t)(live ? k : 0);
  const size_t sstride = (size_t)n_det * 3 * (size_t)N;
  auto eval = [&](int s, double (&ch)[6]) {
    double S[6];
    eval_xyz<KIND, CMASK, true>(bc, smem + s * SMEM_STRIDE, dc, tab, S);   // S holds (Re, -Im)
    ch[0] = S[4] - S[0]; ch[1] = S[1] - S[5];
    ch[2] = S[0] - 2.0 * S[2] + S[4]; ch[3] = -(S[1] - 2.0 * S[3] + S[5]);
    ch[4] = S[0] + S[2] + S[4]; ch[5] = -(S[1] + S[3] + S[5]);
  };
  auto store = [&](int s, const double (&ch)[6]) {
    if (!live) return;
    double2* o = obase + (size_t)s * sstride;
    if (smem[s * SMEM_STRIDE + W_VALID] != 0.0) {
      o[0] = make_double2(fma(ch[0], gA[0], -ch[1] * gA[1]), fma(ch[0], gA[1], ch[1] * gA[0]));
      o[N] = make_double2(fma(ch[2], gE[0], -ch[3] * gE[1]), fma(ch[2], gE[1], ch[3] * gE[0]));
      o[2 * N] = make_double2(fma(ch[4], gT[0], -ch[5] * gT[1]), fma(ch[4], gT[1], ch[5] * gT[0]));
    } else {
      o[0] = o[N] = o[2 * N] = make_double2(CUDART_NAN, CUDART_NAN);
    }
  };
  int s = 0;
  if constexpr (popc4(CMASK) == 1) {
    for (; s + 4 <= ns; s += 4) {
      double ch[4][6];
#pragma unroll
      for (int j = 0; j < 4; ++j) eval(s + j, ch[j]);
#pragma unroll
      for (int j = 0; j < 4; ++j) store(s + j, ch[j]);
    }
  }
  for (; s < ns; ++s) {
    double ch[6];
    eval(s, ch);
    store(s, ch);
  }
}

// FP64 FMA peak: 8 independent chains per thread.  THREE = false: the multiplier and addend are
// shared by the chains (two register operands per DFMA); THREE = true: three distinct registers.
template <bool THREE>
__global__ void __launch_bounds__(256) dfma_peak_kernel(int iters, const double* __restrict__ in,
                                                        double* __restrict__ out) {
  double a[8], b[8], c[8];
#pragma unroll
  for (int j = 0; j < 8; ++j) {
    a[j] = in[(threadIdx.x + j) & 63];
    b[j] = in[(threadIdx.x + 2 * j + 1) & 63];
    c[j] = in[(threadIdx.x + 3 * j + 2) & 63];
  }
  for (int i = 0; i < iters; ++i) {
#pragma unroll
    for (int r = 0; r < 8; ++r) {
#pragma unroll
      for (int j = 0; j < 8; ++j) a[j] = THREE ? fma(a[j], b[j], c[j]) : fma(a[j], b[0], c[0]);
    }
  }
  const double r = ((a[0] + a[1]) + (a[2] + a[3])) + ((a[4] + a[5]) + (a[6] + a[7]));
  if (r == 12345.678) out[0] = r;   // never true; keeps the chains alive
}

// Register-operand probes (profiles/r02_operand_reuse.md).  Eight rounds of 8 FP64 / 16 FP32 / 8 packed-FP32 chains:
//   MODE 0: DFMA a_j = a_j m + c_j       one operand (m) shared with the preceding instruction
//   MODE 1: DFMA a_j = a_j b_{j&1} + c_j one operand shared with the instruction before the preceding one
//   MODE 2: FFMA a_j = a_j b_j + c_j     three distinct registers
//   MODE 3: FFMA2 (two FP32 lanes per instruction) p_j = p_j q_j + r_j, three distinct register pairs
//   MODE 4: FFMA a_j = a_j m + c         multiplier and addend shared (the FP32 pipe peak)
template <int MODE>
__global__ void __launch_bounds__(256) operand_probe_kernel(int iters, const double* __restrict__ in,
                                                            double* __restrict__ out) {
  double a[8], b[8], c[8];
  float fa[16], fb[16], fc[16];
  float2 p[8], q[8], r[8];
  const double m = in[threadIdx.x & 31];
#pragma unroll
  for (int j = 0; j < 8; ++j) {
    a[j] = in[(threadIdx.x + j) & 63];
    b[j] = in[(threadIdx.x + 2 * j + 1) & 63];
    c[j] = in[(threadIdx.x + 3 * j + 2) & 63];
  }
#pragma unroll
  for (int j = 0; j < 16; ++j) {
    fa[j] = (float)in[(threadIdx.x + j) & 63];
    fb[j] = (float)in[(threadIdx.x + 2 * j + 1) & 63];
    fc[j] = (float)in[(threadIdx.x + 3 * j + 2) & 63];
  }
#pragma unroll
  for (int j = 0; j < 8; ++j) {
    p[j] = make_float2(fa[2 * j], fa[2 * j + 1]);
    q[j] = make_float2(fb[2 * j], fb[2 * j + 1]);
    r[j] = make_float2(fc[2 * j], fc[2 * j + 1]);
  }
  const float fm = (float)m, fcc = fc[0];
  for (int i = 0; i < iters; ++i) {
#pragma unroll
    for (int rr = 0; rr < 8; ++rr) {
      if (MODE == 0) {
#pragma unroll
        for (int j = 0; j < 8; ++j) a[j] = fma(a[j], m, c[j]);
      } else if (MODE == 1) {
#pragma unroll
        for (int j = 0; j < 8; ++j) a[j] = fma(a[j], b[j & 1], c[j]);
      } else if (MODE == 2) {
#pragma unroll
        for (int j = 0; j < 16; ++j) fa[j] = fmaf(fa[j], fb[j], fc[j]);
      } else if (MODE == 3) {
#pragma unroll
        for (int j = 0; j < 8; ++j) p[j] = __ffma2_rn(p[j], q[j], r[j]);
      } else {
#pragma unroll
        for (int j = 0; j < 16; ++j) fa[j] = fmaf(fa[j], fm, fcc);
      }
    }
  }
  double t = 0.0;
#pragma unroll
  for (int j = 0; j < 8; ++j) t += a[j] + (double)p[j].x + (double)p[j].y;
#pragma unroll
  for (int j = 0; j < 16; ++j) t += (double)fa[j];
  if (t == 12345.678) out[0] = t;
}


// FP64 tensor-core probe: chains of mma.sync.aligned.m8n8k4 (DMMA, 8 x 8 x 4 = 256 FMAs per warp instruction) on NACC
// independent accumulator fragments per warp; DFMA_MIX > 0 interleaves that many independent DFMAs per DMMA, to see
// whether the two share the FP64 issue port (profiles/r02_dmma.md)
template <int NACC, int DFMA_MIX>
__global__ void __launch_bounds__(256) dmma_peak_kernel(int iters, const double* __restrict__ in,
                                                        double* __restrict__ out) {
  double c0[NACC], c1[NACC], x[DFMA_MIX > 0 ? DFMA_MIX : 1];
  const double a = in[threadIdx.x & 63], b = in[(threadIdx.x + 7) & 63];
#pragma unroll
  for (int j = 0; j < NACC; ++j) { c0[j] = in[(threadIdx.x + j) & 63]; c1[j] = in[(threadIdx.x + 2 * j + 1) & 63]; }
#pragma unroll
  for (int j = 0; j < (DFMA_MIX > 0 ? DFMA_MIX : 1); ++j) x[j] = in[(threadIdx.x + 3 * j) & 63];
  for (int i = 0; i < iters; ++i) {
#pragma unroll
    for (int r = 0; r < 8; ++r) {
#pragma unroll
      for (int j = 0; j < NACC; ++j) {
        asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0, %1}, {%2}, {%3}, {%0, %1};"
                     : "+d"(c0[j]), "+d"(c1[j]) : "d"(a), "d"(b));
#pragma unroll
        for (int q = 0; q < DFMA_MIX; ++q) x[q] = fma(x[q], a, b);
      }
    }
  }
  double r = 0.0;
#pragma unroll
  for (int j = 0; j < NACC; ++j) r += c0[j] + c1[j];
#pragma unroll
  for (int j = 0; j < (DFMA_MIX > 0 ? DFMA_MIX : 1); ++j) r += x[j];
  if (r == 12345.678) out[0] = r;   // never true; keeps the chains alive
}

}  // namespace pespace
