// pespace_grad.cuh -- reverse-mode (adjoint) gradient of the likelihood: lnL and d lnL / d theta in one pass
// ("The backward mode ... is more suitable for cases of large inputs and small
// output such as computing the gradients of the likelihood function", :163, :171 gradient-based samplers).
//
// The forward code is that of loglike_kernel (pespace_device.cuh): per (sample, bin, detector) the mode classes are
// summed into X, Y, Z, the residual against the folded data is formed and weighted.  With
//     L = -1/2 sum_c w_c [ (dr_c - Re h_c)^2 + (di_c - Im' h_c)^2 ]
// the adjoint of (X, Y, Z) is seeded with w_c (d_c - h_c) (one complex number per channel, the same for every mode
// class) and pushed back through S7 -> S2 of every class by hand-written reverse-mode differentiation of that forward
// code.  The sweep stops at the PER-SAMPLE CONSTANTS: what a thread accumulates, and what is reduced over the bins,
// is the adjoint of the constants the forward pass reads (plus three "torques", below) -- NV = 34 numbers per sample
// instead of 12 tangents x 6 components per (sample, bin).  The chain rule from the constants to theta needs the
// tangents of the constants, which prep_samples_du_kernel (the Fisher path's S1 on Du<7>) provides; it is applied
// once per sample by combine_grad_kernel.
//
//   phase polynomial     psi  = sp sum_k c_k b_k(v),  b = (1, v^2, v^3, v^4, v^5, v^5 L, v^6, v^6 L, v^7)
//                        -> moments  PM_k = sum psi_bar sp b_k        (adjoint of W_P0 ... W_P7)
//   time polynomial      tau  = sq sum_k q_k b'_k(v), b' = (1, v^2, v^3, v^4, v^5, v^6, v^6 L, v^7)
//                        -> moments  QM_k = sum tau_bar sq b'_k       (adjoint of W_Q0 ... W_Q7)
//   v = a f^{1/3} (2/m)^{1/3}: d b_k / d ln a = deg_k b_k, so the adjoint of W_A follows from the same moments
//   amplitudes           CK = v^p (ka0 + ka1 v^2)  -> adjoint of W_KA[.]
//   phi_c, t_c           psi contains (m/2) PH0 + fT t_c; the orbit angle(s) contain t_c / yr
//   sky and polarisation the forward pass sees the triad (k, u', v') only through G1_w = w . g1(alpha),
//                        G2_w = w . g2(alpha) and k . R(alpha).  A change of lambda, beta or psi ROTATES the triad,
//                        dw = omega x w, and omega x k = -om_u v' + om_v u', omega x u' = om_k v' - om_v k,
//                        omega x v' = -om_k u' + om_u k, so that
//                            dL = om_k T_k + om_u T_u + om_v T_v,
//                        T_k = sum G1u_bar G1v - G1v_bar G1u + (same with G2),   (the polarisation angle: omega = k)
//                        T_u = sum -G1k_bar G1v + G1v_bar G1k + ... - kR_bar (v'.R),
//                        T_v = sum  G1k_bar G1u - G1u_bar G1k + ... + kR_bar (u'.R):
//                        three numbers per (sample, bin) whatever the detector or class; omega for lambda is z^ and
//                        for beta is u, in triad components (-sin b, sin p cos b, cos p cos b) and (0, cos p, -sin p).
//
// Cost: single-class kernels run forward once and backward once with the forward state in registers.  Multi-class
// kernels need the total response before any adjoint exists: pass 1 runs the classes forward and parks the expensive
// part of each class's state (the six G's, sin / cos of the orbit angle, three reciprocals, three exponentials: NST =
// 17 doubles) in a thread-private shared-memory column; pass 2 reloads it, re-derives the cheap rest and sweeps
// back (pass 1 unrolled over the classes, pass 2 a run-time loop).  No tangent is carried per bin.
#pragma once
#include "pespace_device.cuh"
#include "pespace_fisher.cuh"

namespace pespace {

#ifndef PESPACE_GTILE
#define PESPACE_GTILE 32
#endif
#ifndef PESPACE_GCHUNKS
#define PESPACE_GCHUNKS 4
#endif
constexpr int GTILE = PESPACE_GTILE;       // samples per block, single-class kernels
constexpr int GTILE_M = 16;                // samples per block, multi-class kernels (shared memory holds the state stash)
constexpr int GCHUNKS = PESPACE_GCHUNKS;   // chunks of BLOCK bins per block
constexpr int NST = 17;                    // stashed doubles per class (multi-class kernels)
__host__ __device__ constexpr int grad_tile(unsigned cmask) { return popc4(cmask) == 1 ? GTILE : GTILE_M; }

// reduced vector of one (sample, block)
enum : int {
  GV_LNL = 0,                 // sum w |d - h|^2
  GV_PM = 1,                  // 9 phase moments (order of W_P0, P2, P3, P4, P5, P5L, P6, P6L, P7)
  GV_QM = 10,                 // 8 time moments (order of W_Q0, Q2, Q3, Q4, Q5, Q6, Q6L, Q7)
  GV_PHIC = 18,               // sum (m/2) psi_bar            [per radian of phase]
  GV_TCP = 19,                // sum psi_bar kappa fT         (d psi / d t_c)
  GV_ALPHA = 20,              // sum alpha_bar kappa          (orbit angle(s), in pu)
  GV_TK = 21, GV_TU = 22, GV_TV = 23,
  GV_KA = 24,                 // adjoints of W_KA: class m=2 (a+, ax, b+, bx), then (a+, ax) of m = 1, 3, 4
  NV = 34,
  NVP = 36                    // padded row
};
__host__ __device__ constexpr int grad_ka_slot(int mc, int j /* 0 a+, 1 b+, 2 ax, 3 bx */) {
  return mc == 1 ? GV_KA + (j == 0 ? 0 : j == 2 ? 1 : j == 1 ? 2 : 3)
                 : GV_KA + 4 + 2 * (mc == 0 ? 0 : mc - 1) + (j == 2 ? 1 : 0);
}
// number of leading slots a kernel with class mask CMASK can touch
__host__ __device__ constexpr int grad_nv(unsigned cmask) { return (cmask & 8u) ? 34 : (cmask & 4u) ? 32 : (cmask & 1u) ? 30 : 28; }

// per-warp scratch region (doubles): the state stash of the multi-class kernels ([class][NST][32 lanes]) and the
// transpose buffer of the reduction ([32 values][33]) share it -- the stash is dead once pass 2 of a sample is done
__host__ __device__ constexpr int grad_region(unsigned cmask) {
  return (popc4(cmask) > 1 && popc4(cmask) * NST * 32 > 32 * 33) ? popc4(cmask) * NST * 32 : 32 * 33;
}
__host__ __device__ constexpr size_t grad_smem_bytes(unsigned cmask) {
  return sizeof(double) * ((size_t)2 * NTAB + (size_t)grad_tile(cmask) * SMEM_STRIDE +
                           (size_t)(BLOCK / 32) * grad_tile(cmask) * NVP + (size_t)(BLOCK / 32) * grad_region(cmask));
}
static_assert(grad_smem_bytes(15u) <= 227u * 1024u && grad_smem_bytes(2u) <= 227u * 1024u, "one block per SM");
static_assert(S_VY < D_BASE + D_STRIDE, "detector block holds the torque constants S_UX ... S_VY");

// forward state of one mode class that the backward sweep needs
template <int KIND>
struct ClassState {
  double v, v2, L, sp, sq, CKp, CKc;
  double s1, c1, s2, c2;          // kind 0: sin/cos alpha, sin/cos 2 alpha; kind 1: sin/cos alpha_E, sin/cos phi
  double G1k, G2k, G1u, G2u, G1v, G2v;
  double kb_, kc_, ka_;
  double uu[3], vv[3], rD[3], pl[3], ql[3];
  double Er[3], Ei[3];
};

// forward pass of one class: the code of eval_class / eval_geom with the class index at run time and the
// intermediates kept.  Adds X, Y, Z (Re, -Im) to S (FIRST: initialises S).
template <int KIND>
__device__ __forceinline__ void grad_fwd_class(int mc, bool first, const BinC& bc, const double* __restrict__ sc,
                                               const DetC& dc, const double2* __restrict__ tab, double va, double La,
                                               double ftc, ClassState<KIND>& st, double (&S)[6]) {
  const double MH = 0.5 * (double)(mc + 1);
  const double v = va * kClassCB[mc];
  const double L = La + kClassLN3[mc];
  const double v2 = v * v;
  st.v = v; st.v2 = v2; st.L = L;
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
  st.sp = kClassS83[mc] * bc.fm53;
  st.sq = kClassS83[mc] * bc.fm83;
  double psi = st.sp * P;
  psi -= whole_turns(psi);
  psi += fma(MH, sc[W_PH0], ftc);
  const double tau = st.sq * Q;
  const double* ka = sc + W_KA + 4 * mc;
  if (mc == 1) { st.CKp = fma(ka[1], v2, ka[0]); st.CKc = fma(ka[3], v2, ka[2]); }
  else { const double vp = (mc == 3) ? v2 : v; st.CKp = vp * ka[0]; st.CKc = vp * ka[2]; }

  double kR;
  if (KIND == 0) {
    double sa, ca;
    sincos_tab(sc[D_BASE] + tau, tab, sa, ca);
    const double c2 = fma(2.0 * ca, ca, -1.0), s2 = 2.0 * sa * ca;
    st.s1 = sa; st.c1 = ca; st.s2 = s2; st.c2 = c2;
    const double* w = sc + S_K;
    st.G1k = fma(w[0], c2, fma(w[1], s2, fma(w[2], ca, w[3])));
    st.G2k = fma(w[0], s2, fma(-w[1], c2, fma(w[2], sa, w[4])));
    w = sc + S_U;
    st.G1u = fma(w[0], c2, fma(w[1], s2, fma(w[2], ca, w[3])));
    st.G2u = fma(w[0], s2, fma(-w[1], c2, fma(w[2], sa, w[4])));
    w = sc + S_V;
    st.G1v = fma(w[0], c2, fma(w[1], s2, fma(w[2], ca, w[3])));
    st.G2v = fma(w[0], s2, fma(-w[1], c2, fma(w[2], sa, w[4])));
    kR = fma(sc[S_DX], ca, sc[S_DY] * sa);
  } else {
    double sE, cE, sp, cp;
    sincos_tab(sc[D_BASE] + tau, tab, sE, cE);
    sincos_tab(fma(tau, dc.yr_over_p, sc[D_BASE + 1]), tab, sp, cp);
    st.s1 = sE; st.c1 = cE; st.s2 = sp; st.c2 = cp;
    const double* w = sc + D_BASE + 2;
    st.G1k = fma(w[0], cp, w[1] * sp); st.G2k = fma(w[1], cp, -w[0] * sp);
    st.G1u = fma(w[2], cp, w[3] * sp); st.G2u = fma(w[3], cp, -w[2] * sp);
    st.G1v = fma(w[4], cp, w[5] * sp); st.G2v = fma(w[5], cp, -w[4] * sp);
    kR = fma(sc[S_DX], cE, sc[S_DY] * sE);
  }
  constexpr double R3H = 0.86602540378443864676;
  const double tk = R3H * st.G2k;
  const double nun[3] = {st.G1k, fma(-0.5, st.G1k, tk), fma(-0.5, st.G1k, -tk)};
  st.ka_ = tk + tk; st.kb_ = fma(-1.5, st.G1k, -tk); st.kc_ = fma(1.5, st.G1k, -tk);
  const double tu = R3H * st.G2u, tv = R3H * st.G2v;
  st.uu[0] = tu + tu; st.uu[1] = fma(-1.5, st.G1u, -tu); st.uu[2] = fma(1.5, st.G1u, -tu);
  st.vv[0] = tv + tv; st.vv[1] = fma(-1.5, st.G1v, -tv); st.vv[2] = fma(1.5, st.G1v, -tv);
  double Wr[3], Wi[3];
#pragma unroll
  for (int l = 0; l < 3; ++l) {
    const double uu = st.uu[l], vv = st.vv[l];
    const double v2_ = vv * vv;
    const double D = fma(uu, uu, v2_);
    const double rD = (__double2hiint(D) > 0) ? rcp_pos(D) : 0.0;
    st.rD[l] = rD;
    st.pl[l] = rD * fma(uu, uu, -v2_);
    st.ql[l] = rD * (uu * vv);
    Wr[l] = st.CKp * st.pl[l];
    Wi[l] = st.CKc * st.ql[l];
  }
  {
    const double fTL = bc.fT * dc.Lbar;
    const double base = fma(bc.fT, kR, psi);
#pragma unroll
    for (int n = 0; n < 3; ++n) sincos_tab(fma(fTL, nun[n], base), tab, st.Ei[n], st.Er[n]);
  }
  auto add = [&](double& Sr, double& Si, int r, int s_, double kap, double wr, double wi, bool init) {
    const double br = fma(kap, fma(-bc.cth, st.Er[r], st.Er[s_]), -bc.sth * st.Ei[r]);
    const double bi = fma(kap, fma(-bc.cth, st.Ei[r], st.Ei[s_]), bc.sth * st.Er[r]);
    if (init) { Sr = fma(wr, br, -wi * bi); Si = fma(wr, bi, wi * br); }
    else { Sr = fma(wr, br, fma(-wi, bi, Sr)); Si = fma(wr, bi, fma(wi, br, Si)); }
  };
  add(S[0], S[1], 0, 2, -st.kb_, Wr[1], Wi[1], first);
  add(S[0], S[1], 0, 1, st.kc_, -Wr[2], -Wi[2], false);
  add(S[2], S[3], 1, 0, -st.kc_, Wr[2], Wi[2], first);
  add(S[2], S[3], 1, 2, st.ka_, -Wr[0], -Wi[0], false);
  add(S[4], S[5], 2, 1, -st.ka_, Wr[0], Wi[0], first);
  add(S[4], S[5], 2, 0, st.kb_, -Wr[1], -Wi[1], false);
}

// multi-class kernels: park / reload the expensive part of a class's forward state (col = this lane's column in the
// warp's region, stride 32)
template <int KIND>
__device__ __forceinline__ void grad_store_state(const ClassState<KIND>& st, double* __restrict__ col) {
  col[0 * 32] = st.G1k; col[1 * 32] = st.G2k; col[2 * 32] = st.G1u; col[3 * 32] = st.G2u;
  col[4 * 32] = st.G1v; col[5 * 32] = st.G2v; col[6 * 32] = st.s1; col[7 * 32] = st.c1;
#pragma unroll
  for (int i = 0; i < 3; ++i) {
    col[(8 + i) * 32] = st.rD[i]; col[(11 + i) * 32] = st.Er[i]; col[(14 + i) * 32] = st.Ei[i];
  }
}
template <int KIND>
__device__ __forceinline__ void grad_restore_state(int mc, const BinC& bc, const double* __restrict__ sc, double va,
                                                   double La, const double* __restrict__ col, ClassState<KIND>& st) {
  const double v = va * kClassCB[mc], v2 = v * v;
  st.v = v; st.v2 = v2; st.L = La + kClassLN3[mc];
  st.sp = kClassS83[mc] * bc.fm53;
  st.sq = kClassS83[mc] * bc.fm83;
  const double* ka = sc + W_KA + 4 * mc;
  if (mc == 1) { st.CKp = fma(ka[1], v2, ka[0]); st.CKc = fma(ka[3], v2, ka[2]); }
  else { const double vp = (mc == 3) ? v2 : v; st.CKp = vp * ka[0]; st.CKc = vp * ka[2]; }
  st.G1k = col[0 * 32]; st.G2k = col[1 * 32]; st.G1u = col[2 * 32]; st.G2u = col[3 * 32];
  st.G1v = col[4 * 32]; st.G2v = col[5 * 32]; st.s1 = col[6 * 32]; st.c1 = col[7 * 32];
  if (KIND == 0) { st.c2 = fma(2.0 * st.c1, st.c1, -1.0); st.s2 = 2.0 * st.s1 * st.c1; }
  else { st.c2 = 0.0; st.s2 = 0.0; }                       // kind 1: the backward sweep does not use them
  constexpr double R3H = 0.86602540378443864676;
  const double tk = R3H * st.G2k, tu = R3H * st.G2u, tv = R3H * st.G2v;
  st.ka_ = tk + tk; st.kb_ = fma(-1.5, st.G1k, -tk); st.kc_ = fma(1.5, st.G1k, -tk);
  st.uu[0] = tu + tu; st.uu[1] = fma(-1.5, st.G1u, -tu); st.uu[2] = fma(1.5, st.G1u, -tu);
  st.vv[0] = tv + tv; st.vv[1] = fma(-1.5, st.G1v, -tv); st.vv[2] = fma(1.5, st.G1v, -tv);
#pragma unroll
  for (int i = 0; i < 3; ++i) {
    st.rD[i] = col[(8 + i) * 32]; st.Er[i] = col[(11 + i) * 32]; st.Ei[i] = col[(14 + i) * 32];
    st.pl[i] = st.rD[i] * fma(st.uu[i], st.uu[i], -st.vv[i] * st.vv[i]);
    st.ql[i] = st.rD[i] * (st.uu[i] * st.vv[i]);
  }
}

// backward sweep of one class: Sb = adjoint of S (Re, -Im parts of X, Y, Z); adds to acc.  Written as FMA chains
// (accumulators as addends, signs on the small factors): every DADD / DMUL saved is two issue cycles of the FP64 pipe.
template <int KIND>
__device__ __forceinline__ void grad_bwd_class(int mc, const BinC& bc, const double* __restrict__ sc, const DetC& dc,
                                               const ClassState<KIND>& st, const double (&Sb)[6], double (&acc)[NV]) {
  const double MH = 0.5 * (double)(mc + 1);
  double Wrb[3] = {0.0, 0.0, 0.0}, Wib[3] = {0.0, 0.0, 0.0}, Erb[3] = {0.0, 0.0, 0.0}, Eib[3] = {0.0, 0.0, 0.0};
  double kab = 0.0, kbb = 0.0, kcb = 0.0;
  const double Wr[3] = {st.CKp * st.pl[0], st.CKp * st.pl[1], st.CKp * st.pl[2]};
  const double Wi[3] = {st.CKc * st.ql[0], st.CKc * st.ql[1], st.CKc * st.ql[2]};
  const double sEr[3] = {bc.sth * st.Er[0], bc.sth * st.Er[1], bc.sth * st.Er[2]};
  const double sEi[3] = {bc.sth * st.Ei[0], bc.sth * st.Ei[1], bc.sth * st.Ei[2]};
  const double kac = st.ka_ * bc.cth, kbc = st.kb_ * bc.cth, kcc = st.kc_ * bc.cth;
  // adjoint of  S += sg W_l B(r, s, kap),  B = kap (E_s - cth E_r) -/+ i sth E_r,  kap = ks k  (see `add` of the
  // forward pass).  (tr, ti) = sg (Sbr, Sbi); k = |kap| factor with sign ks; kc = k cth
  auto back = [&](double tr, double ti, int r, int s_, double k, double kc, double ks, double& kb_adj, int l) {
    const double er = fma(-bc.cth, st.Er[r], st.Er[s_]), ei = fma(-bc.cth, st.Ei[r], st.Ei[s_]);
    const double br = fma(ks * k, er, -sEi[r]);
    const double bi = fma(ks * k, ei, sEr[r]);
    Wrb[l] = fma(tr, br, fma(ti, bi, Wrb[l]));
    Wib[l] = fma(ti, br, fma(-tr, bi, Wib[l]));
    const double brb = fma(tr, Wr[l], ti * Wi[l]), bib = fma(ti, Wr[l], -tr * Wi[l]);
    kb_adj = fma(ks * brb, er, fma(ks * bib, ei, kb_adj));
    Erb[s_] = fma(ks * k, brb, Erb[s_]);
    Eib[s_] = fma(ks * k, bib, Eib[s_]);
    Erb[r] = fma(-ks * kc, brb, fma(bc.sth, bib, Erb[r]));
    Eib[r] = fma(-ks * kc, bib, fma(-bc.sth, brb, Eib[r]));
  };
  back(Sb[0], Sb[1], 0, 2, st.kb_, kbc, -1.0, kbb, 1);        // X: + W_b B(1,3,-kb)
  back(-Sb[0], -Sb[1], 0, 1, st.kc_, kcc, 1.0, kcb, 2);       //    - W_c B(1,2, kc)
  back(Sb[2], Sb[3], 1, 0, st.kc_, kcc, -1.0, kcb, 2);        // Y: + W_c B(2,1,-kc)
  back(-Sb[2], -Sb[3], 1, 2, st.ka_, kac, 1.0, kab, 0);       //    - W_a B(2,3, ka)
  back(Sb[4], Sb[5], 2, 1, st.ka_, kac, -1.0, kab, 0);        // Z: + W_a B(3,2,-ka)
  back(-Sb[4], -Sb[5], 2, 0, st.kb_, kbc, 1.0, kbb, 1);       //    - W_b B(3,1, kb)

  // ---- exponentials: phase_n [rad] = kappa (fTL nu_n + fT kR + psi),  E_n = (cos, sin)
  const double pb0 = fma(st.Er[0], Eib[0], -st.Ei[0] * Erb[0]);
  const double pb1 = fma(st.Er[1], Eib[1], -st.Ei[1] * Erb[1]);
  const double pb2 = fma(st.Er[2], Eib[2], -st.Ei[2] * Erb[2]);
  const double psib = (pb0 + pb1) + pb2;                    // per radian of the class phase
  const double kfT = kRadPerPu * bc.fT;
  const double kfTL = kfT * dc.Lbar;
  const double kRb = kfT * psib;

  // ---- arm weights: Wr = CKp pl, Wi = CKc ql, pl = rD (uu^2 - vv^2), ql = rD uu vv, rD = 1 / (uu^2 + vv^2)
  double CKpb = 0.0, CKcb = 0.0, uub[3], vvb[3];
#pragma unroll
  for (int l = 0; l < 3; ++l) {
    CKpb = fma(Wrb[l], st.pl[l], CKpb);
    CKcb = fma(Wib[l], st.ql[l], CKcb);
    const double plb = Wrb[l] * st.CKp, qlb = Wib[l] * st.CKc;
    const double rD2 = st.rD[l] + st.rD[l];
    const double xib2 = plb * rD2, chb = qlb * st.rD[l];                   // 2 xi_bar, chi_bar
    const double Db2 = -rD2 * fma(plb, st.pl[l], qlb * st.ql[l]);           // 2 D_bar
    uub[l] = fma(st.vv[l], chb, st.uu[l] * (Db2 + xib2));
    vvb[l] = fma(st.uu[l], chb, st.vv[l] * (Db2 - xib2));
  }
  // ---- projections on the arms and the spacecraft (nu_n_bar = kfTL pb_n folded in)
  constexpr double R3H = 0.86602540378443864676;
  const double G1ub = 1.5 * (uub[2] - uub[1]), G2ub = R3H * (fma(2.0, uub[0], -uub[1]) - uub[2]);
  const double G1vb = 1.5 * (vvb[2] - vvb[1]), G2vb = R3H * (fma(2.0, vvb[0], -vvb[1]) - vvb[2]);
  const double G1kb = fma(1.5, kcb - kbb, kfTL * fma(-0.5, pb1 + pb2, pb0));
  const double G2kb = R3H * fma(kfTL, pb1 - pb2, fma(2.0, kab, -kbb) - kcb);

  // ---- torques and orbit angle(s)
  double alphab;                     // per radian of the orbit angle (kind 1: alpha_E + (yr / P) phi)
  const double uR = fma(sc[S_UX], st.c1, sc[S_UY] * st.s1);
  const double vR = fma(sc[S_VX], st.c1, sc[S_VY] * st.s1);
  if (KIND == 0) {
    const double* wk = sc + S_K; const double* wu = sc + S_U; const double* wv = sc + S_V;
    const double c2b = fma(G1kb, wk[0], fma(-G2kb, wk[1], fma(G1ub, wu[0], fma(-G2ub, wu[1], fma(G1vb, wv[0], -G2vb * wv[1])))));
    const double s2b = fma(G1kb, wk[1], fma(G2kb, wk[0], fma(G1ub, wu[1], fma(G2ub, wu[0], fma(G1vb, wv[1], G2vb * wv[0])))));
    const double cab = fma(G1kb, wk[2], fma(G1ub, wu[2], fma(G1vb, wv[2], kRb * sc[S_DX])));
    const double sab = fma(G2kb, wk[2], fma(G2ub, wu[2], fma(G2vb, wv[2], kRb * sc[S_DY])));
    alphab = fma(-2.0 * st.s2, c2b, fma(2.0 * st.c2, s2b, fma(-st.s1, cab, st.c1 * sab)));
  } else {
    const double phib = fma(G1kb, st.G2k, fma(-G2kb, st.G1k, fma(G1ub, st.G2u, fma(-G2ub, st.G1u, fma(G1vb, st.G2v, -G2vb * st.G1v)))));
    const double aEb = kRb * fma(sc[S_DY], st.c1, -sc[S_DX] * st.s1);
    alphab = fma(dc.yr_over_p, phib, aEb);
  }
  acc[GV_TK] = fma(G1ub, st.G1v, fma(-G1vb, st.G1u, fma(G2ub, st.G2v, fma(-G2vb, st.G2u, acc[GV_TK]))));
  acc[GV_TU] = fma(-G1kb, st.G1v, fma(G1vb, st.G1k, fma(-G2kb, st.G2v, fma(G2vb, st.G2k, fma(-kRb, vR, acc[GV_TU])))));
  acc[GV_TV] = fma(G1kb, st.G1u, fma(-G1ub, st.G1k, fma(G2kb, st.G2u, fma(-G2ub, st.G2k, fma(kRb, uR, acc[GV_TV])))));

  // ---- phase and time polynomials: moments of the basis
  const double pm = (kRadPerPu * st.sp) * psib, qm = (kRadPerPu * st.sq) * alphab;
  const double v = st.v, v2 = st.v2, v3 = v2 * v, v4 = v2 * v2, v5 = v4 * v, v6 = v5 * v, v7 = v6 * v;
  const double v5L = v5 * st.L, v6L = v6 * st.L;
  acc[GV_PM + 0] += pm;
  acc[GV_PM + 1] = fma(pm, v2, acc[GV_PM + 1]);
  acc[GV_PM + 2] = fma(pm, v3, acc[GV_PM + 2]);
  acc[GV_PM + 3] = fma(pm, v4, acc[GV_PM + 3]);
  acc[GV_PM + 4] = fma(pm, v5, acc[GV_PM + 4]);
  acc[GV_PM + 5] = fma(pm, v5L, acc[GV_PM + 5]);
  acc[GV_PM + 6] = fma(pm, v6, acc[GV_PM + 6]);
  acc[GV_PM + 7] = fma(pm, v6L, acc[GV_PM + 7]);
  acc[GV_PM + 8] = fma(pm, v7, acc[GV_PM + 8]);
  acc[GV_QM + 0] += qm;
  acc[GV_QM + 1] = fma(qm, v2, acc[GV_QM + 1]);
  acc[GV_QM + 2] = fma(qm, v3, acc[GV_QM + 2]);
  acc[GV_QM + 3] = fma(qm, v4, acc[GV_QM + 3]);
  acc[GV_QM + 4] = fma(qm, v5, acc[GV_QM + 4]);
  acc[GV_QM + 5] = fma(qm, v6, acc[GV_QM + 5]);
  acc[GV_QM + 6] = fma(qm, v6L, acc[GV_QM + 6]);
  acc[GV_QM + 7] = fma(qm, v7, acc[GV_QM + 7]);
  acc[GV_PHIC] = fma(MH, psib, acc[GV_PHIC]);
  acc[GV_TCP] = fma(kfT, psib, acc[GV_TCP]);
  acc[GV_ALPHA] = fma(kRadPerPu, alphab, acc[GV_ALPHA]);
  // ---- amplitudes
  if (mc == 1) {
    acc[grad_ka_slot(1, 0)] += CKpb;
    acc[grad_ka_slot(1, 2)] += CKcb;
    acc[grad_ka_slot(1, 1)] = fma(CKpb, v2, acc[grad_ka_slot(1, 1)]);
    acc[grad_ka_slot(1, 3)] = fma(CKcb, v2, acc[grad_ka_slot(1, 3)]);
  } else if (mc == 0) {
    acc[grad_ka_slot(0, 0)] = fma(CKpb, v, acc[grad_ka_slot(0, 0)]);
    acc[grad_ka_slot(0, 2)] = fma(CKcb, v, acc[grad_ka_slot(0, 2)]);
  } else if (mc == 2) {
    acc[grad_ka_slot(2, 0)] = fma(CKpb, v, acc[grad_ka_slot(2, 0)]);
    acc[grad_ka_slot(2, 2)] = fma(CKcb, v, acc[grad_ka_slot(2, 2)]);
  } else {
    acc[grad_ka_slot(3, 0)] = fma(CKpb, v2, acc[grad_ka_slot(3, 0)]);
    acc[grad_ka_slot(3, 2)] = fma(CKcb, v2, acc[grad_ka_slot(3, 2)]);
  }
}

// Sum over the warp of NVL <= NV values per lane, added into the warp's row r[NVP]; fixed order.  Values 0..31 go
// through a shared-memory transpose (scr: [32][33] doubles, conflict-free both ways): every lane stores its values,
// lane j then adds up row j -- 32 STS + 32 LDS + 31 DADD per thread instead of the 31 shuffle-adds and 124 selects of a
// halving butterfly on 64-bit values.  Values 32, 33 (kernels with the m = 4 class) take a plain shuffle tree.
template <int NVL>
__device__ __forceinline__ void grad_warp_reduce(double (&a)[NV], int lane, double* __restrict__ scr,
                                                 double* __restrict__ r) {
#pragma unroll
  for (int j = 32; j < NVL; ++j) {
    double x = a[j];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) x += __shfl_xor_sync(0xffffffffu, x, o);
    if (lane == j - 32) r[j] += x;
  }
  constexpr int NR = NVL < 32 ? NVL : 32;
  __syncwarp();                                   // every lane is done with the stash that shares this region
#pragma unroll
  for (int j = 0; j < NR; ++j) scr[j * 33 + lane] = a[j];
  __syncwarp();
  if (lane < NR) {
    const double* row = scr + lane * 33;
    double t0 = row[0], t1 = row[1], t2 = row[2], t3 = row[3];
#pragma unroll
    for (int i = 4; i < 32; i += 4) { t0 += row[i]; t1 += row[i + 1]; t2 += row[i + 2]; t3 += row[i + 3]; }
    r[lane] += (t0 + t1) + (t2 + t3);
  }
  __syncwarp();                                   // before the next sample's stash / transpose overwrites the region
}

template <int KIND, unsigned CMASK>
__global__ void __launch_bounds__(BLOCK, 1)
loglike_grad_kernel(const double* __restrict__ consts, const double2* __restrict__ trig, long long B,
                    const double* __restrict__ bins /* [n_det][NBF][N] */, long long N, DetC dc, int n_det, int det,
                    double* __restrict__ partial /* [n_det][gridDim.x][B][NVP] */) {
  constexpr int NCLS = popc4(CMASK);
  constexpr int NVL = grad_nv(CMASK);
  constexpr int TILE_G = grad_tile(CMASK);
  constexpr int MCL = (CMASK & 8u) ? 3 : (CMASK & 4u) ? 2 : (CMASK & 2u) ? 1 : 0;   // the last class of the mask
  double2* tab = reinterpret_cast<double2*>(pespace_dyn_smem);
  double* smem = reinterpret_cast<double*>(tab + NTAB);
  double* red = smem + TILE_G * SMEM_STRIDE;                     // [warps][TILE_G][NVP]
  double* region = red + (BLOCK / 32) * TILE_G * NVP + (threadIdx.x >> 5) * grad_region(CMASK);   // this warp's scratch
  double* stash = region + (threadIdx.x & 31);                   // [class][NST][32]: this lane's column
  const long long b0 = (long long)blockIdx.y * TILE_G;
  stage_trig(tab, trig);
  {
    const int stride = sample_stride(n_det);
    for (int i = threadIdx.x; i < TILE_G * SMEM_STRIDE; i += BLOCK) {
      const int s = i / SMEM_STRIDE, j = i % SMEM_STRIDE;
      long long b = b0 + s;
      if (b >= B) b = B - 1;
      const int src = (j < D_BASE) ? j : (D_BASE + D_STRIDE * det + (j - D_BASE));
      smem[i] = consts[b * stride + src];
    }
  }
  for (int i = threadIdx.x; i < (BLOCK / 32) * TILE_G * NVP; i += BLOCK) red[i] = 0.0;
  __syncthreads();
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int ns = (int)min((long long)TILE_G, B - b0);
  for (int ch = 0; ch < GCHUNKS; ++ch) {
    const long long kbase = ((long long)blockIdx.x * GCHUNKS + ch) * BLOCK;
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
      const double* sc = smem + s * SMEM_STRIDE;
      const double ftc = mul_mod_turn(bc.fT, sc[W_TC]);
      const double va = sc[W_A] * bc.cf, La = bc.lnf3;
      double S[6];
      ClassState<KIND> st;
      if constexpr (NCLS == 1) {
        constexpr int MC0 = (CMASK & 1u) ? 0 : (CMASK & 2u) ? 1 : (CMASK & 4u) ? 2 : 3;
        grad_fwd_class<KIND>(MC0, true, bc, sc, dc, tab, va, La, ftc, st, S);
      } else {
        // pass 1: every class forward, the expensive part of its state parked in shared memory (the last class of the
        // mask stays in registers).  Pass 2 below is a RUN-TIME loop: with its bodies unrolled as well the kernel
        // carried 0.9-1.6 KB of spills per thread and ran 1.3-1.7x slower
        // pass 1, unrolled over the classes at compile time (forward bodies only: 30.7 instead of 34.0 ms per step on
        // config 5's workload); the slot of class MC in the stash = number of classes below it
#define PESPACE_G1(MC)                                                                                         \
        if constexpr ((CMASK >> MC) & 1u) {                                                                      \
          grad_fwd_class<KIND>(MC, !(CMASK & ((1u << MC) - 1u)), bc, sc, dc, tab, va, La, ftc, st, S);           \
          if (MC != MCL) grad_store_state<KIND>(st, stash + popc4(CMASK & ((1u << MC) - 1u)) * (NST * 32));      \
        }
        PESPACE_G1(0) PESPACE_G1(1) PESPACE_G1(2) PESPACE_G1(3)
#undef PESPACE_G1
      }
      double acc[NV];
#pragma unroll
      for (int i = 0; i < NV; ++i) acc[i] = 0.0;
      double Sb[6];
      {
        // residual and its weight: adjoint seeds of A = Z - X, E = X - 2Y + Z, T = X + Y + Z (unnormalised, as folded)
        const double ra0 = dr[0] - (S[4] - S[0]), ra1 = di[0] - (S[5] - S[1]);
        const double re0 = dr[1] - (S[0] - 2.0 * S[2] + S[4]), re1 = di[1] - (S[1] - 2.0 * S[3] + S[5]);
        const double rt0 = dr[2] - (S[0] + S[2] + S[4]), rt1 = di[2] - (S[1] + S[3] + S[5]);
        const double a0 = w[0] * ra0, a1 = w[0] * ra1, e0 = w[1] * re0, e1 = w[1] * re1, t0 = w[2] * rt0, t1 = w[2] * rt1;
        acc[GV_LNL] = fma(t1, rt1, fma(t0, rt0, fma(e1, re1, fma(e0, re0, fma(a1, ra1, a0 * ra0)))));
        Sb[0] = (e0 + t0) - a0; Sb[1] = (e1 + t1) - a1;
        Sb[2] = fma(-2.0, e0, t0); Sb[3] = fma(-2.0, e1, t1);
        Sb[4] = (e0 + t0) + a0; Sb[5] = (e1 + t1) + a1;
      }
      if constexpr (NCLS == 1) {
        constexpr int MC0 = (CMASK & 1u) ? 0 : (CMASK & 2u) ? 1 : (CMASK & 4u) ? 2 : 3;
        grad_bwd_class<KIND>(MC0, bc, sc, dc, st, Sb, acc);
      } else {
        grad_bwd_class<KIND>(MCL, bc, sc, dc, st, Sb, acc);       // pass 2: the last class first, its state is still live
        int slot = 0;
#pragma unroll 1
        for (int mc = 0; mc < MCL; ++mc) {
          if (!((CMASK >> mc) & 1u)) continue;
          grad_restore_state<KIND>(mc, bc, sc, va, La, stash + slot * (NST * 32), st);
          grad_bwd_class<KIND>(mc, bc, sc, dc, st, Sb, acc);
          ++slot;
        }
      }
      grad_warp_reduce<NVL>(acc, lane, region, red + (warp * TILE_G + s) * NVP);
    }
  }
  __syncthreads();
  // cross-warp sum in fixed order
  for (int i = threadIdx.x; i < ns * NVP; i += BLOCK) {
    const int s = i / NVP, j = i % NVP;
    double t = 0.0;
#pragma unroll
    for (int wv = 0; wv < BLOCK / 32; ++wv) t += red[(wv * TILE_G + s) * NVP + j];
    partial[(((size_t)det * gridDim.x + blockIdx.x) * (size_t)B + (size_t)(b0 + s)) * NVP + j] = t;
  }
}

// Second pass: fixed-order sum over (detector, bin block) of the NV adjoints of one sample, then the chain rule from
// the per-sample constants to theta with the tangents of consts_du (prep_samples_du_kernel: value + d/d(M, q, chi1,
// chi2, iota, lambda, beta) per constant).  One warp per sample: lane j < NV sums value j, lane 0 contracts.
static __global__ void combine_grad_kernel(const double* __restrict__ partial, const double* __restrict__ consts_du,
                                           const double* __restrict__ params, long long B, int n_slices, int n_det,
                                           double* __restrict__ out_lnL, double* __restrict__ out_grad) {
  __shared__ double vals[4][NVP];
  const int wv = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const long long b = (long long)blockIdx.x * 4 + wv;
  if (b < B) {
    for (int j = lane; j < NV; j += 32) {
      double t = 0.0;
      for (int i = 0; i < n_slices; ++i) t += partial[((size_t)i * (size_t)B + (size_t)b) * NVP + j];
      vals[wv][j] = t;
    }
  }
  __syncwarp();
  if (b >= B || lane != 0) return;
  const double* V = vals[wv];
  const double* cd = consts_du + (size_t)b * fisher_const_stride(n_det);
  const double* th = params + b * NPAR;
  const bool valid = cd[W_A * DUW + 1] != 0.0;            // W_A has a non-zero M tangent for every in-domain sample
  if (out_lnL) out_lnL[b] = valid ? -0.5 * V[GV_LNL] : -CUDART_INF;
  if (!out_grad) return;
  double g[NPAR];
  if (!valid) {
    for (int i = 0; i < NPAR; ++i) out_grad[b * NPAR + i] = CUDART_NAN;
    return;
  }
  const int pidx[9] = {W_P0, W_P2, W_P3, W_P4, W_P5, W_P5L, W_P6, W_P6L, W_P7};
  const double pdeg[9] = {0.0, 2.0, 3.0, 4.0, 5.0, 5.0, 6.0, 6.0, 7.0};
  const int qidx[8] = {W_Q0, W_Q2, W_Q3, W_Q4, W_Q5, W_Q6, W_Q6L, W_Q7};
  const double qdeg[8] = {0.0, 2.0, 3.0, 4.0, 5.0, 6.0, 6.0, 7.0};
  // adjoint of ln a (v = a f^{1/3} (2/m)^{1/3}) and the D_L sum from the values of the constants
  double lnab = 0.0, kasum = 0.0;
  for (int k = 0; k < 9; ++k) lnab = fma(pdeg[k] * cd[pidx[k] * DUW], V[GV_PM + k], lnab);
  for (int k = 0; k < 8; ++k) lnab = fma(qdeg[k] * cd[qidx[k] * DUW], V[GV_QM + k], lnab);
  for (int mc = 0; mc < 4; ++mc)
    for (int j = 0; j < 4; ++j) {
      if (mc != 1 && (j & 1)) continue;
      const double kav = cd[(W_KA + 4 * mc + j) * DUW], kab = V[grad_ka_slot(mc, j)];
      const double deg = (mc == 1) ? ((j & 1) ? 2.0 : 0.0) : (mc == 3 ? 2.0 : 1.0);
      lnab = fma(deg * kav, kab, lnab);
      kasum = fma(kav, kab, kasum);
    }
  // tangent slots of consts_du: 1 + (M, q, chi1, chi2, iota, lambda, beta)
  const int slot_of[5] = {0, 1, 2, 3, 4};
  const int par_of[5] = {0, 1, 2, 3, 5};
  for (int t = 0; t < 5; ++t) {
    const int sl = 1 + slot_of[t];
    double acc = lnab * cd[W_LNA * DUW + sl];
    for (int k = 0; k < 9; ++k) acc = fma(cd[pidx[k] * DUW + sl], V[GV_PM + k], acc);
    for (int k = 0; k < 8; ++k) acc = fma(cd[qidx[k] * DUW + sl], V[GV_QM + k], acc);
    for (int mc = 0; mc < 4; ++mc)
      for (int j = 0; j < 4; ++j) {
        if (mc != 1 && (j & 1)) continue;
        acc = fma(cd[(W_KA + 4 * mc + j) * DUW + sl], V[grad_ka_slot(mc, j)], acc);
      }
    g[par_of[t]] = acc;
  }
  g[4] = -kasum / th[4];                                             // D_L: every amplitude is ~ 1 / D_L
  g[6] = -2.0 * V[GV_PHIC];                                          // phi_c: psi[rad] contains -(m/2) 2 phi_c
  g[10] = fma(kTurn / kYear, V[GV_ALPHA], V[GV_TCP]);                // t_c: phase and orbit angle(s)
  double sb, cb, sp, cp;
  sincos(th[8], &sb, &cb);
  sincos(th[9], &sp, &cp);
  g[7] = fma(-sb, V[GV_TK], cb * fma(sp, V[GV_TU], cp * V[GV_TV]));   // lambda: omega = z^
  g[8] = fma(cp, V[GV_TU], -sp * V[GV_TV]);                           // beta:   omega = u
  g[9] = V[GV_TK];                                                    // psi:    omega = k
  for (int i = 0; i < NPAR; ++i) out_grad[b * NPAR + i] = g[i];
}

}  // namespace pespace
