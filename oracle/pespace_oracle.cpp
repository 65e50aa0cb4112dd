// pespace_oracle.cpp -- plain, slow, double-precision CPU oracle.
//
// TEST INFRASTRUCTURE, NOT PRODUCT CODE (see pespace_oracle.h).  It is the
// definition written out: PAPER.md Eq. 3 (A,E,T), Eq. 4 (t_f), Eq. 5 (single
// link), Eq. 6 (TDI), Eq. 10/11 (Whittle likelihood), Eq. 13/14 (Fisher, inner
// product), with the readings O0-O12 / G1-G16 of SURVEY.md 8(c) for everything
// the paper only cites (TaylorF2 waveform from BASELINE.json, analytic orbits,
// frame conventions).  No blocking, fusion, tables or algebraic shortcuts: one
// (sample, bin, detector, mode) at a time, in the paper's order.
//
// One source, three scalar types: double (the oracle), Dual<11> (forward-mode
// derivatives, O12) and __float128 (pin P14: is double enough?).
//
// Tabulated mode waveforms (T1 block below, reading T1 of DESIGN.md): the interpolation is an
// approximation of the caller's waveform, so it follows its definition step by step (binary search, cubic Hermite
// with slopes 2 pi t_j, its derivative, 4-node Lagrange); pinned by the T1 tests (exactness on cubics, reproduction
// of the analytic path at fourth order, extrinsic scalings, band limits, brute-force Whittle sum).
//
// Tabulated orbits (T2 block, reading T2 of DESIGN.md): cubic Hermite in time on the caller's
// position / velocity tables; pinned by the T2 tests (exact on cubic trajectories, reproduces the analytic orbit and
// its response when fed dense samples of it, rigid arms between nodes, zero outside the table).
//
// Pins (tests/test_oracle_pins.py): P1-P16 of SURVEY.md 8(c), the spin terms of G3 against the Poisson-Will forms
// of beta and sigma (phase and time series), the c_lm v^p table of O5 against point-mass multipole moments and the
// test-mass mode fluxes.  "Parity unpinned": the absolute values of the Taiji-/TianQin-like results (G8, G13 are
// proposals, not in the paper) and the constant per-mode phase -m pi/8 of reading G5.
//
// Build: g++ -O2 -std=gnu++17 -ffp-contract=off -fopenmp -shared -fPIC (oracle/build.py)

#include "pespace_oracle.h"

#include <cmath>
#include <cstdint>
#include <cstring>
#include <limits>
#include <vector>
#include <quadmath.h>
#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

// ---------------------------------------------------------------- O0 constants
constexpr double C_SI = 299792458.0;               // m/s
constexpr double GMSUN = 1.3271244e20;             // m^3/s^2
constexpr double GPC_M = 3.0856775814913673e25;    // m
constexpr double AU_M = 149597870700.0;            // m
constexpr double YR_S = 31558149.763545603;        // sidereal year, s
constexpr int NPAR = 11;

typedef __float128 quad;

// ---------------------------------------------------------------- dual numbers (O12)
template <int NT>
struct Dual {
  double v;
  double d[NT];
  Dual() : v(0.0) { for (int i = 0; i < NT; ++i) d[i] = 0.0; }
  Dual(double x) : v(x) { for (int i = 0; i < NT; ++i) d[i] = 0.0; }
};
template <int NT> Dual<NT> operator+(const Dual<NT>& a, const Dual<NT>& b) {
  Dual<NT> r; r.v = a.v + b.v; for (int i = 0; i < NT; ++i) r.d[i] = a.d[i] + b.d[i]; return r; }
template <int NT> Dual<NT> operator-(const Dual<NT>& a, const Dual<NT>& b) {
  Dual<NT> r; r.v = a.v - b.v; for (int i = 0; i < NT; ++i) r.d[i] = a.d[i] - b.d[i]; return r; }
template <int NT> Dual<NT> operator-(const Dual<NT>& a) {
  Dual<NT> r; r.v = -a.v; for (int i = 0; i < NT; ++i) r.d[i] = -a.d[i]; return r; }
template <int NT> Dual<NT> operator*(const Dual<NT>& a, const Dual<NT>& b) {
  Dual<NT> r; r.v = a.v * b.v; for (int i = 0; i < NT; ++i) r.d[i] = a.d[i] * b.v + a.v * b.d[i]; return r; }
template <int NT> Dual<NT> operator/(const Dual<NT>& a, const Dual<NT>& b) {
  Dual<NT> r; r.v = a.v / b.v;
  for (int i = 0; i < NT; ++i) r.d[i] = (a.d[i] - r.v * b.d[i]) / b.v;
  return r; }
template <int NT> Dual<NT> chain(const Dual<NT>& a, double fv, double dfv) {  // f(a), f'(a)
  Dual<NT> r; r.v = fv; for (int i = 0; i < NT; ++i) r.d[i] = dfv * a.d[i]; return r; }

// elementary functions, one overload set per scalar type
inline double o_sqrt(double x) { return std::sqrt(x); }
inline double o_cbrt(double x) { return std::cbrt(x); }
inline double o_log(double x) { return std::log(x); }
inline double o_sin(double x) { return std::sin(x); }
inline double o_cos(double x) { return std::cos(x); }
inline double o_val(double x) { return x; }
inline quad o_sqrt(quad x) { return sqrtq(x); }
inline quad o_cbrt(quad x) { return cbrtq(x); }
inline quad o_log(quad x) { return logq(x); }
inline quad o_sin(quad x) { return sinq(x); }
inline quad o_cos(quad x) { return cosq(x); }
inline double o_val(quad x) { return (double)x; }
template <int NT> Dual<NT> o_sqrt(const Dual<NT>& a) { double s = std::sqrt(a.v); return chain(a, s, 0.5 / s); }
template <int NT> Dual<NT> o_cbrt(const Dual<NT>& a) { double c = std::cbrt(a.v); return chain(a, c, c / (3.0 * a.v)); }
template <int NT> Dual<NT> o_log(const Dual<NT>& a) { return chain(a, std::log(a.v), 1.0 / a.v); }
template <int NT> Dual<NT> o_sin(const Dual<NT>& a) { return chain(a, std::sin(a.v), std::cos(a.v)); }
template <int NT> Dual<NT> o_cos(const Dual<NT>& a) { return chain(a, std::cos(a.v), -std::sin(a.v)); }
template <int NT> double o_val(const Dual<NT>& a) { return a.v; }

// pi and Euler's constant in the working precision
template <class T> struct K {
  static T pi() { return T(3.14159265358979323846264338327950288); }
  static T euler() { return T(0.5772156649015329); }  // O0
};
template <> struct K<quad> {
  static quad pi() { return M_PIq; }
  static quad euler() { return 0.57721566490153286060651209008240243Q; }
};

// ---------------------------------------------------------------- complex pairs
template <class T> struct Cx { T re, im; };
template <class T> Cx<T> cx(const T& re, const T& im) { Cx<T> r; r.re = re; r.im = im; return r; }
template <class T> Cx<T> operator+(const Cx<T>& a, const Cx<T>& b) { return cx<T>(a.re + b.re, a.im + b.im); }
template <class T> Cx<T> operator-(const Cx<T>& a, const Cx<T>& b) { return cx<T>(a.re - b.re, a.im - b.im); }
template <class T> Cx<T> operator*(const Cx<T>& a, const Cx<T>& b) {
  return cx<T>(a.re * b.re - a.im * b.im, a.re * b.im + a.im * b.re); }
template <class T> Cx<T> scale(const Cx<T>& a, const T& s) { return cx<T>(a.re * s, a.im * s); }
template <class T> Cx<T> expi(const T& phase) { return cx<T>(o_cos(phase), o_sin(phase)); }  // e^{i phase}

template <class T> struct V3 { T x, y, z; };
template <class T> T dot(const V3<T>& a, const V3<T>& b) { return a.x * b.x + a.y * b.y + a.z * b.z; }
template <class T> V3<T> operator+(const V3<T>& a, const V3<T>& b) { V3<T> r = {a.x + b.x, a.y + b.y, a.z + b.z}; return r; }
template <class T> V3<T> operator-(const V3<T>& a, const V3<T>& b) { V3<T> r = {a.x - b.x, a.y - b.y, a.z - b.z}; return r; }
template <class T> V3<T> smul(const V3<T>& a, const T& s) { V3<T> r = {a.x * s, a.y * s, a.z * s}; return r; }

// ---------------------------------------------------------------- O1 source scalars
template <class T> struct Source {
  T Ms, eta, delta, mu1, mu2, Ds;                 // O1
  T chi1, chi2, iota, phic, lam, bet, psi, tc;    // theta entries, raw
};
template <class T> Source<T> make_source(const T th[NPAR]) {
  Source<T> s;
  const T M = th[0], q = th[1];
  const T Tsun = T(GMSUN) / (T(C_SI) * T(C_SI) * T(C_SI));  // = 4.925490947641267e-6 s
  s.Ms = M * Tsun;
  s.eta = q / ((T(1.0) + q) * (T(1.0) + q));
  s.delta = (q - T(1.0)) / (q + T(1.0));
  s.mu1 = q / (T(1.0) + q);
  s.mu2 = T(1.0) / (T(1.0) + q);
  s.chi1 = th[2]; s.chi2 = th[3];
  s.Ds = th[4] * T(GPC_M) / T(C_SI);
  s.iota = th[5]; s.phic = th[6]; s.lam = th[7]; s.bet = th[8]; s.psi = th[9]; s.tc = th[10];
  return s;
}

// ---------------------------------------------------------------- O2 / O3: TaylorF2 3.5PN
// phi_k(v) of O2 and their d/dln v parts phi_k^{ln} of O3.
template <class T> void pn_coefficients(const Source<T>& s, const T& v, T phi[8], T philn[8]) {
  const T pi = K<T>::pi(), eta = s.eta, lnv = o_log(v);
  const T beta_so = (T(113.0) * s.mu1 * s.mu1 / T(12.0) + T(25.0) * eta / T(4.0)) * s.chi1 +
                    (T(113.0) * s.mu2 * s.mu2 / T(12.0) + T(25.0) * eta / T(4.0)) * s.chi2;   // G3
  const T sigma_ss = T(79.0) / T(8.0) * eta * s.chi1 * s.chi2;                                 // G3
  phi[0] = T(1.0);
  phi[1] = T(0.0);
  phi[2] = T(3715.0) / T(756.0) + T(55.0) * eta / T(9.0);
  phi[3] = T(-16.0) * pi + T(4.0) * beta_so;
  phi[4] = T(15293365.0) / T(508032.0) + T(27145.0) * eta / T(504.0) + T(3085.0) * eta * eta / T(72.0) -
           T(10.0) * sigma_ss;
  phi[5] = pi * (T(38645.0) / T(756.0) - T(65.0) * eta / T(9.0)) * (T(1.0) + T(3.0) * lnv);
  phi[6] = T(11583231236531.0) / T(4694215680.0) - T(640.0) * pi * pi / T(3.0) -
           T(6848.0) * K<T>::euler() / T(21.0) +
           eta * (T(-15737765635.0) / T(3048192.0) + T(2255.0) * pi * pi / T(12.0)) +
           T(76055.0) * eta * eta / T(1728.0) - T(127825.0) * eta * eta * eta / T(1296.0) -
           T(6848.0) / T(21.0) * o_log(T(4.0) * v);
  phi[7] = pi * (T(77096675.0) / T(254016.0) + T(378515.0) * eta / T(1512.0) -
                 T(74045.0) * eta * eta / T(756.0));
  for (int k = 0; k < 8; ++k) philn[k] = T(0.0);
  philn[5] = T(3.0) * pi * (T(38645.0) / T(756.0) - T(65.0) * eta / T(9.0));
  philn[6] = T(-6848.0) / T(21.0);
}

// v^{k-5}, k = 0..7
template <class T> void v_powers(const T& v, T vp[8]) {
  vp[5] = T(1.0);
  for (int k = 4; k >= 0; --k) vp[k] = vp[k + 1] / v;
  for (int k = 6; k < 8; ++k) vp[k] = vp[k - 1] * v;
}

// O2: Psi_22(f) = 2 pi f t_c - 2 phi_c - pi/4 + 3/(128 eta) sum_k phi_k v^{k-5}
template <class T> T psi22(const Source<T>& s, const T& f) {
  const T pi = K<T>::pi();
  const T v = o_cbrt(pi * s.Ms * f);
  T phi[8], philn[8], vp[8];
  pn_coefficients(s, v, phi, philn);
  v_powers(v, vp);
  T sum = T(0.0);
  for (int k = 0; k < 8; ++k) sum = sum + phi[k] * vp[k];
  return T(2.0) * pi * f * s.tc - T(2.0) * s.phic - pi / T(4.0) + T(3.0) / (T(128.0) * s.eta) * sum;
}

// O3 (Eq. 4 with Phi = -Psi): t_22(f) = t_c + 1/(2 pi) 1/(128 eta f) sum_k [(k-5) phi_k + phi_k^{ln}] v^{k-5}
template <class T> T t22(const Source<T>& s, const T& f) {
  const T pi = K<T>::pi();
  const T v = o_cbrt(pi * s.Ms * f);
  T phi[8], philn[8], vp[8];
  pn_coefficients(s, v, phi, philn);
  v_powers(v, vp);
  T sum = T(0.0);
  for (int k = 0; k < 8; ++k) sum = sum + (T((double)(k - 5)) * phi[k] + philn[k]) * vp[k];
  return s.tc + sum / (T(2.0) * pi * T(128.0) * s.eta * f);
}

// O4: A_22(f) = sqrt(2 eta / 3) pi^{-1/6} (Ms^2 / Ds) (Ms f)^{-7/6}
template <class T> T amp22(const Source<T>& s, const T& f) {
  const T pi = K<T>::pi();
  const T x = s.Ms * f;
  const T x16 = o_sqrt(o_cbrt(x));            // x^{1/6}
  const T pi16 = o_sqrt(o_cbrt(pi));          // pi^{1/6}
  return o_sqrt(T(2.0) * s.eta / T(3.0)) / pi16 * (s.Ms * s.Ms / s.Ds) / (x * x16);
}

// O5: per-mode amplitude, phase and time-frequency map.  f' = 2 f / m.
struct ModeId { int l, m; };
const ModeId MODE_TABLE[5] = {{2, 2}, {2, 1}, {3, 3}, {3, 2}, {4, 4}};

template <class T> bool mode_constants(const Source<T>& s, int l, int m, T* c_lm, int* p_lm) {
  if (l == 2 && m == 2) { *c_lm = T(1.0); *p_lm = 0; return true; }
  if (l == 2 && m == 1) { *c_lm = s.delta / T(3.0); *p_lm = 1; return true; }
  if (l == 3 && m == 3) { *c_lm = T(3.0) / T(4.0) * o_sqrt(T(15.0) / T(14.0)) * s.delta; *p_lm = 1; return true; }
  if (l == 3 && m == 2) { *c_lm = T(1.0) / T(3.0) * o_sqrt(T(5.0) / T(7.0)) * (T(1.0) - T(3.0) * s.eta); *p_lm = 2; return true; }
  if (l == 4 && m == 4) { *c_lm = T(8.0) / T(9.0) * o_sqrt(T(5.0) / T(7.0)) * (T(1.0) - T(3.0) * s.eta); *p_lm = 2; return true; }
  return false;
}

template <class T> bool mode_waveform(const Source<T>& s, int l, int m, double f, T* amp, T* psi, T* tf) {
  T c_lm; int p_lm;
  if (!mode_constants(s, l, m, &c_lm, &p_lm)) return false;
  const T fp = T(2.0) * T(f) / T((double)m);                    // f' = 2f/m
  const T vm = o_cbrt(K<T>::pi() * s.Ms * fp);
  T vpow = T(1.0);
  for (int i = 0; i < p_lm; ++i) vpow = vpow * vm;
  *amp = o_sqrt(T(2.0) / T((double)m)) * c_lm * vpow * amp22(s, fp);   // A_lm
  *psi = T((double)m) / T(2.0) * psi22(s, fp);                          // Psi_lm (G5)
  *tf = t22(s, fp);                                                     // t_lm
  return true;
}

// ---------------------------------------------------------------- O6: spin-weight -2 harmonics
double factorial(int n) { double r = 1.0; for (int i = 2; i <= n; ++i) r *= i; return r; }
double binomial(int n, int k) { if (k < 0 || k > n) return 0.0; return factorial(n) / (factorial(k) * factorial(n - k)); }

// Goldberg et al. finite sum, spin weight s = -2, phi = 0:
//  sYlm = (-1)^{l+m-s} sqrt[(l+m)!(l-m)!(2l+1) / (4 pi (l+s)!(l-s)!)]
//         sum_r (-1)^r C(l-s, r) C(l+s, r+s-m) cos^{2r+s-m}(iota/2) sin^{2l-2r-s+m}(iota/2)
template <class T> T swsh_m2(int l, int m, const T& iota) {
  const int s = -2;
  const T ch = o_cos(iota / T(2.0)), sh = o_sin(iota / T(2.0));
  const double norm2 = factorial(l + m) * factorial(l - m) * (2 * l + 1) / (factorial(l + s) * factorial(l - s));
  T sum = T(0.0);
  for (int r = 0; r <= l - s; ++r) {
    const double cc = binomial(l - s, r) * binomial(l + s, r + s - m);
    if (cc == 0.0) continue;
    const int pc = 2 * r + s - m, ps = 2 * l - 2 * r - s + m;
    T term = T(cc);
    for (int i = 0; i < pc; ++i) term = term * ch;
    for (int i = 0; i < ps; ++i) term = term * sh;
    sum = (r % 2 == 0) ? sum + term : sum - term;
  }
  const T pref = o_sqrt(T(norm2) / (T(4.0) * K<T>::pi()));
  return (((l + m - s) % 2 + 2) % 2 == 0) ? pref * sum : -(pref * sum);
}

// K_+^{lm}, K_x^{lm} of O6 (complex)
template <class T> void mode_polarisation(int l, int m, const T& iota, Cx<T>* Kp, Cx<T>* Kc) {
  const T Yp = swsh_m2(l, m, iota), Ym = swsh_m2(l, -m, iota);
  const T sgn = (l % 2 == 0) ? T(1.0) : T(-1.0);
  *Kp = cx<T>(T(0.5) * (Yp + sgn * Ym), T(0.0));
  *Kc = cx<T>(T(0.0), T(-0.5) * (Yp - sgn * Ym));
}

// ---------------------------------------------------------------- O7: frames
template <class T> struct Frame { V3<T> k, u, v; T c2psi, s2psi; };
template <class T> Frame<T> make_frame(const Source<T>& s) {
  Frame<T> F;
  const T cl = o_cos(s.lam), sl = o_sin(s.lam), cb = o_cos(s.bet), sb = o_sin(s.bet);
  F.k.x = -(cb * cl); F.k.y = -(cb * sl); F.k.z = -sb;
  F.u.x = sl; F.u.y = -cl; F.u.z = T(0.0);
  F.v.x = -(sb * cl); F.v.y = -(sb * sl); F.v.z = cb;
  F.c2psi = o_cos(T(2.0) * s.psi); F.s2psi = o_sin(T(2.0) * s.psi);
  return F;
}
// n . P^{lm} . n = K_+ (n.P_+.n) + K_x (n.P_x.n),  P_+ = cos2psi e_+ + sin2psi e_x,  P_x = -sin2psi e_+ + cos2psi e_x
template <class T> Cx<T> arm_projection(const Frame<T>& F, const V3<T>& n, const Cx<T>& Kp, const Cx<T>& Kc) {
  const T nu = dot(n, F.u), nv = dot(n, F.v);
  const T ep = nu * nu - nv * nv, ec = T(2.0) * nu * nv;       // n.e_+.n, n.e_x.n
  const T pp = F.c2psi * ep + F.s2psi * ec;
  const T pc = -(F.s2psi * ep) + F.c2psi * ec;
  return scale(Kp, pp) + scale(Kc, pc);
}

// ---------------------------------------------------------------- O8: orbits
// Positions are returned as centre + offset_n (metres) so that arm vectors can be
// formed from the offsets alone; x_n = centre + offset_n is the definition.
template <class T> void orbit(const pespace_oracle_detector& D, const T& t, V3<T>* centre, V3<T> off[3]) {
  const T pi = K<T>::pi();
  const T alphaE = T(2.0) * pi * t / T(YR_S);
  if (D.kind == 0) {
    const T alpha = alphaE + T(D.kappa);
    const T e = T(D.L_m) / (T(2.0) * o_sqrt(T(3.0)) * T(AU_M));
    centre->x = T(AU_M) * o_cos(alpha); centre->y = T(AU_M) * o_sin(alpha); centre->z = T(0.0);
    for (int n = 0; n < 3; ++n) {
      const T bn = T(2.0) * pi * T((double)n) / T(3.0) + T(D.lambda0);
      off[n].x = T(0.5) * e * T(AU_M) * (o_cos(T(2.0) * alpha - bn) - T(3.0) * o_cos(bn));
      off[n].y = T(0.5) * e * T(AU_M) * (o_sin(T(2.0) * alpha - bn) - T(3.0) * o_sin(bn));
      off[n].z = -(o_sqrt(T(3.0)) * e * T(AU_M) * o_cos(alpha - bn));
    }
  } else {
    const T r = T(D.L_m) / o_sqrt(T(3.0));
    const T cl = o_cos(T(D.lon)), sl = o_sin(T(D.lon)), cb = o_cos(T(D.lat)), sb = o_sin(T(D.lat));
    const V3<T> nh = {cb * cl, cb * sl, sb};
    const V3<T> e1 = {-sl, cl, T(0.0)};
    const V3<T> e2 = {nh.y * e1.z - nh.z * e1.y, nh.z * e1.x - nh.x * e1.z, nh.x * e1.y - nh.y * e1.x};
    centre->x = T(AU_M) * o_cos(alphaE); centre->y = T(AU_M) * o_sin(alphaE); centre->z = T(0.0);
    for (int n = 0; n < 3; ++n) {
      const T ph = T(2.0) * pi * t / T(D.period_s) + T(2.0) * pi * T((double)n) / T(3.0) + T(D.lambda0);
      off[n] = smul(e1, r * o_cos(ph)) + smul(e2, r * o_sin(ph));
    }
  }
}

// ---------------------------------------------------------------- T2: tabulated numerical orbits
// "Support for high-precision numerical orbits will be extended in future work".  Reading T2 of
// the spacecraft positions arrive as tables on a uniform time grid t_j = t0 + j dt, j = 0..K-1 (SSB time,
// same origin as t_c): pos [K][3 spacecraft][3] in metres and vel [K][3][3] in m/s.  Between nodes every coordinate
// is the cubic Hermite interpolant with the node velocities as slopes,
//   x(t) = h00(u) x_j + h10(u) dt v_j + h01(u) x_{j+1} + h11(u) dt v_{j+1},  u = (t - t_j) / dt,
//   h00 = 2u^3 - 3u^2 + 1, h10 = u^3 - 2u^2 + u, h01 = -2u^3 + 3u^2, h11 = u^3 - u^2.
// The delays keep the constant nominal arm length L of the detector description (the paper's formalism is the rigid
// equal-arm one); the single link is the transform of Eq. 1 with the positions and the unit link
// vectors n_rs = (x_r - x_s) / |x_r - x_s| from the table (see single_link), Eq. 6 is unchanged.  A mode whose
// t_lm(f) falls outside [t0, t0 + (K-1) dt] contributes 0 at that frequency.
struct OrbitTab { int64_t K; double t0, dt; const double *pos, *vel; };

template <class T> bool orbit_tab(const OrbitTab& O, const T& t, V3<T>* centre, V3<T> off[3]) {
  const double tv = o_val(t);
  const double t_end = O.t0 + (double)(O.K - 1) * O.dt;
  if (!(tv >= O.t0) || !(tv <= t_end)) return false;
  int64_t j = (int64_t)std::floor((tv - O.t0) / O.dt);
  if (j < 0) j = 0;
  if (j > O.K - 2) j = O.K - 2;
  const T u = (t - T(O.t0 + (double)j * O.dt)) / T(O.dt);
  const T u2 = u * u, u3 = u2 * u;
  const T h00 = T(2.0) * u3 - T(3.0) * u2 + T(1.0), h10 = u3 - T(2.0) * u2 + u;
  const T h01 = T(3.0) * u2 - T(2.0) * u3, h11 = u3 - u2;
  const double *p0 = O.pos + (size_t)j * 9, *p1 = p0 + 9, *v0 = O.vel + (size_t)j * 9, *v1 = v0 + 9;
  centre->x = T(0.0); centre->y = T(0.0); centre->z = T(0.0);
  for (int n = 0; n < 3; ++n) {
    T c[3];
    for (int a = 0; a < 3; ++a)
      c[a] = h00 * T(p0[3 * n + a]) + h10 * T(O.dt * v0[3 * n + a]) + h01 * T(p1[3 * n + a]) + h11 * T(O.dt * v1[3 * n + a]);
    off[n].x = c[0]; off[n].y = c[1]; off[n].z = c[2];
  }
  return true;
}
bool orbit_tab_ok(const OrbitTab& O) {
  return O.K >= 2 && O.pos && O.vel && O.dt > 0.0 && std::isfinite(O.dt) && std::isfinite(O.t0);
}

// ---------------------------------------------------------------- O9: single link, Eq. 5
template <class T> T sinc(const T& x) {
  const double ax = std::fabs(o_val(x));
  if (ax < 1e-4) return T(1.0) - x * x / T(6.0);
  return o_sin(x) / x;
}
// y_rs for receiver r, sender s (0-based), one mode.  Times in seconds.
template <class T> Cx<T> single_link(const T& f, double L_m, const Frame<T>& F, const V3<T>& centre,
                                     const V3<T> off[3], int r, int s, const Cx<T>& Kp, const Cx<T>& Kc,
                                     const Cx<T>& hlm, bool unit_arms = false) {
  const T pi = K<T>::pi();
  const T Lbar = T(L_m) / T(C_SI);
  const V3<T> dx = off[r] - off[s];
  const V3<T> xr = centre + off[r], xs = centre + off[s];
  const Cx<T> minus_i = cx<T>(T(0.0), T(-1.0));
  if (unit_arms) {
    // T2, tabulated orbits: the arms breathe, so k.(x_r - x_s) = L k.n_rs no longer holds and Eq. 5 is not the
    // transform of Eq. 1 any more.  Eq. 1 is the definition; its transform at frozen geometry is
    //   y_rs = [ e^{-2 pi i f (L + k.x_s)} - e^{-2 pi i f k.x_r} ] / (2 (1 - k.n_rs)) n_rs.h.n_rs
    // with the UNIT link vector n_rs = (x_r - x_s) / |x_r - x_s| and the nominal L (pin P5: equal to Eq. 5 for
    // rigid arms).  The pole at k.n_rs = 1 is cancelled by n.P.n = O(1 - (k.n)^2); no special case is made for it.
    const V3<T> n = smul(dx, T(1.0) / o_sqrt(dot(dx, dx)));
    const T kn = dot(F.k, n);
    // the difference of the two exponentials is written as -2 i sin(a) e^{-i pi f [L + k.(x_r + x_s)]} with
    // a = pi f [L - k.(x_r - x_s)] (= the sinc argument of Eq. 5 when the arms are rigid): same number, no cancellation
    const T a = pi * f * (Lbar - dot(F.k, dx) / T(C_SI));
    const T kxx = dot(F.k, xr + xs) / T(C_SI);
    const Cx<T> pref = scale(minus_i, o_sin(a) / (T(1.0) - kn));
    const Cx<T> ph = expi(-(pi * f * (Lbar + kxx)));
    const Cx<T> nPn = arm_projection(F, n, Kp, Kc);
    return pref * ph * nPn * hlm;
  }
  const V3<T> n = smul(dx, T(1.0) / T(L_m));                               // n_rs = (x_r - x_s)/L
  const T kn = dot(F.k, n);
  const T kxx = dot(F.k, xr + xs) / T(C_SI);                               // k.(x_r + x_s)/c
  const T x = pi * f * Lbar * (T(1.0) - kn);
  const Cx<T> pref = scale(minus_i, pi * f * Lbar * sinc(x));              // -i pi f L sinc[...]
  const Cx<T> ph = expi(-(pi * f * (Lbar + kxx)));                         // exp{-i pi f [L + k.(x_r+x_s)]}
  const Cx<T> nPn = arm_projection(F, n, Kp, Kc);                          // n.P^{lm}.n
  return pref * ph * nPn * hlm;
}

// ---------------------------------------------------------------- O10: TDI (Eq. 6) and A,E,T (Eq. 3)
// y[0..5] = y12 y21 y13 y31 y23 y32
template <class T> void tdi_xyz(const Cx<T> y[6], const T& f, double L_m, int gen, Cx<T> XYZ[3]) {
  const T Lbar = T(L_m) / T(C_SI);
  const Cx<T> z = expi(-(T(2.0) * K<T>::pi() * f * Lbar));
  const Cx<T> one = cx<T>(T(1.0), T(0.0));
  const Cx<T> z2 = z * z;
  // g(z) = 1 - z^2 (generation 1.5) or (1 - z^2)(1 - z^4) = 1 - z^2 - z^4 + z^6 (2.0): Eq. 6 as SURVEY O10 states it.
  // The PRODUCT form is evaluated: where z^2 = 1 (f = n c / 2L, inside the band of configs 2-5, G9) both factors
  // vanish and the expanded sum of four O(1) terms keeps only ~1e-16 / |g| relative digits -- 3e-7 one bin from
  // the null against this definition's own binary128 evaluation (pin P14 extended to the nulls), the product 1e-11.
  Cx<T> g = one - z2;
  if (gen == 20) g = g * (one - z2 * z2);
  const Cx<T>&y12 = y[0], &y21 = y[1], &y13 = y[2], &y31 = y[3], &y23 = y[4], &y32 = y[5];
  XYZ[0] = g * (y13 - y12 + z * (y31 - y21));
  XYZ[1] = g * (y21 - y23 + z * (y12 - y32));
  XYZ[2] = g * (y32 - y31 + z * (y23 - y13));
}
template <class T> void aet(const Cx<T> XYZ[3], Cx<T> AET[3]) {
  const Cx<T>&X = XYZ[0], &Y = XYZ[1], &Z = XYZ[2];
  AET[0] = scale(Z - X, T(1.0) / o_sqrt(T(2.0)));
  AET[1] = scale(X - scale(Y, T(2.0)) + Z, T(1.0) / o_sqrt(T(6.0)));
  AET[2] = scale(X + Y + Z, T(1.0) / o_sqrt(T(3.0)));
}

// six links of one mode at one frequency for one detector
// six links of one mode from its amplitude, phase and time-frequency map at f
template <class T> void links_from_waveform(const T& iota, const Frame<T>& F, int l, int m, double f, const T& amp,
                                            const T& psi, const T& tf, const pespace_oracle_detector& D, Cx<T> y[6],
                                            const OrbitTab* ot = nullptr) {
  const Cx<T> hlm = scale(expi(-psi), amp);                                // h_lm = A e^{-i Psi}
  Cx<T> Kp, Kc;
  mode_polarisation(l, m, iota, &Kp, &Kc);
  V3<T> centre, off[3];
  if (ot) {                                                                // T2: positions from the orbit table
    if (!orbit_tab(*ot, tf, &centre, off)) {
      for (int i = 0; i < 6; ++i) y[i] = cx<T>(T(0.0), T(0.0));
      return;
    }
  } else {
    orbit(D, tf, &centre, off);                                            // geometry at t = t_lm(f)
  }
  const int R[6] = {0, 1, 0, 2, 1, 2}, S[6] = {1, 0, 2, 0, 2, 1};
  for (int i = 0; i < 6; ++i) y[i] = single_link(T(f), D.L_m, F, centre, off, R[i], S[i], Kp, Kc, hlm, ot != nullptr);
}

template <class T> bool mode_links(const Source<T>& s, const Frame<T>& F, int l, int m, double f,
                                   const pespace_oracle_detector& D, Cx<T> y[6], const OrbitTab* ot = nullptr) {
  T amp, psi, tf;
  if (!mode_waveform(s, l, m, f, &amp, &psi, &tf)) return false;
  links_from_waveform(s.iota, F, l, m, f, amp, psi, tf, D, y, ot);
  return true;
}

// A,E,T of one detector at one frequency, summed over the modes of the mask
template <class T> void response_bin(const Source<T>& s, const Frame<T>& F, double f, uint32_t mode_mask,
                                     const pespace_oracle_detector& D, Cx<T> AET[3], const OrbitTab* ot = nullptr) {
  Cx<T> sum[3];
  for (int c = 0; c < 3; ++c) sum[c] = cx<T>(T(0.0), T(0.0));
  for (int im = 0; im < 5; ++im) {
    if (!(mode_mask & (1u << im))) continue;
    Cx<T> y[6], XYZ[3], ch[3];
    mode_links(s, F, MODE_TABLE[im].l, MODE_TABLE[im].m, f, D, y, ot);
    tdi_xyz(y, T(f), D.L_m, D.tdi_gen, XYZ);
    aet(XYZ, ch);
    for (int c = 0; c < 3; ++c) sum[c] = sum[c] + ch[c];
  }
  for (int c = 0; c < 3; ++c) AET[c] = sum[c];
}

// ---------------------------------------------------------------- argument checks
bool model_ok(const pespace_oracle_model* m) {
  if (!m || !m->det || m->n_det <= 0) return false;
  if ((m->mode_mask & 31u) == 0 || (m->mode_mask & ~31u) != 0) return false;
  for (int i = 0; i < m->n_det; ++i) {
    const pespace_oracle_detector& D = m->det[i];
    if (D.kind != 0 && D.kind != 1) return false;
    if (D.tdi_gen != 15 && D.tdi_gen != 20) return false;
    if (!(D.L_m > 0.0)) return false;
    if (D.kind == 1 && !(D.period_s > 0.0)) return false;
  }
  return true;
}
bool grid_ok(const pespace_oracle_grid* g) { return g && g->N > 0 && g->df > 0.0 && g->f0 > 0.0; }
bool sample_ok(const double* th) {
  for (int i = 0; i < NPAR; ++i) if (!std::isfinite(th[i])) return false;
  return th[0] > 0.0 && th[1] >= 1.0 && th[4] > 0.0;
}
bool weight_ok(double S) { return std::isfinite(S) && S > 0.0; }

int g_threads = 0;

template <class T>
int response_impl(const double* params, int64_t B, const double* freqs, int64_t N,
                  const pespace_oracle_model* model, double* out, const OrbitTab* tabs = nullptr) {
  if (!params || !freqs || !out || B <= 0 || N <= 0 || !model_ok(model)) return -1;
  const int nd = model->n_det;
  const double nan = std::numeric_limits<double>::quiet_NaN();
#pragma omp parallel for schedule(dynamic, 1) num_threads(g_threads > 0 ? g_threads : omp_get_max_threads())
  for (int64_t b = 0; b < B; ++b) {
    double* ob = out + (size_t)b * nd * 3 * N * 2;
    if (!sample_ok(params + b * NPAR)) {
      for (int64_t i = 0; i < (int64_t)nd * 3 * N * 2; ++i) ob[i] = nan;
      continue;
    }
    T th[NPAR];
    for (int i = 0; i < NPAR; ++i) th[i] = T(params[b * NPAR + i]);
    const Source<T> s = make_source(th);
    const Frame<T> F = make_frame(s);
    for (int d = 0; d < nd; ++d)
      for (int64_t k = 0; k < N; ++k) {
        Cx<T> ch[3];
        if (freqs[k] > 0.0) response_bin(s, F, freqs[k], model->mode_mask, model->det[d], ch, tabs ? tabs + d : nullptr);
        else for (int c = 0; c < 3; ++c) ch[c] = cx<T>(T(0.0), T(0.0));
        for (int c = 0; c < 3; ++c) {
          ob[(((size_t)d * 3 + c) * N + k) * 2 + 0] = o_val(ch[c].re);
          ob[(((size_t)d * 3 + c) * N + k) * 2 + 1] = o_val(ch[c].im);
        }
      }
  }
  return 0;
}

// ---------------------------------------------------------------- T1: tabulated waveforms
// The paper's pipeline hands per-mode amplitude, phase and t_f from the waveform generator to the response
// (PAPER.md:151-157).  Here they arrive as tables on K shared nodes f_0 < ... < f_{K-1}, per sample and per mode of
// the mask (bit order), for the reference extrinsic values t_c = 0, phi_c = 0, D_L = 1 Gpc (reading T1):
//   Psi_lm(f) = Psi_tab(f) + 2 pi f t_c - m phi_c,   t_lm(f) = t_tab(f) + t_c,   A_lm(f) = A_tab(f) / D_L[Gpc].
// Between nodes: Psi_tab is the cubic Hermite interpolant of the node values with node slopes 2 pi t_j (Eq. 4),
// t_tab is (1/2pi) times the derivative of that interpolant, A_tab the cubic Lagrange polynomial through the four
// nodes j-1..j+2 around the interval (stencil shifted to stay inside the table).  Outside [f_0, f_{K-1}] the mode is 0.
struct WaveTable { int64_t K; const double *fn, *amp, *psi, *tf; int n_modes; };

// interval index j with fn[j] <= f <= fn[j+1] (largest such j, at most K-2); -1 outside the table
int64_t tab_interval(const WaveTable& W, double f) {
  if (!(f >= W.fn[0]) || !(f <= W.fn[W.K - 1])) return -1;
  int64_t lo = 0, hi = W.K - 1;                       // invariant: fn[lo] <= f, f <= fn[hi]
  while (hi - lo > 1) {
    const int64_t mid = (lo + hi) / 2;
    if (W.fn[mid] <= f) lo = mid; else hi = mid;
  }
  return lo;
}

bool tab_waveform(const WaveTable& W, int64_t b, int imode, double f, double* amp, double* psi, double* tf) {
  const int64_t j = tab_interval(W, f);
  if (j < 0) return false;
  const size_t base = ((size_t)b * W.n_modes + imode) * (size_t)W.K;
  const double *P = W.psi + base, *Tt = W.tf + base, *A = W.amp + base;
  const double h = W.fn[j + 1] - W.fn[j], s = (f - W.fn[j]) / h;
  const double twopi = 2.0 * K<double>::pi();
  // cubic Hermite basis and its derivative in s
  const double h00 = (1.0 + 2.0 * s) * (1.0 - s) * (1.0 - s), h10 = s * (1.0 - s) * (1.0 - s);
  const double h01 = s * s * (3.0 - 2.0 * s), h11 = s * s * (s - 1.0);
  const double d00 = 6.0 * s * (s - 1.0), d10 = (1.0 - s) * (1.0 - 3.0 * s), d01 = -d00, d11 = s * (3.0 * s - 2.0);
  *psi = h00 * P[j] + h01 * P[j + 1] + h * twopi * (h10 * Tt[j] + h11 * Tt[j + 1]);
  *tf = (d00 * P[j] + d01 * P[j + 1]) / (h * twopi) + d10 * Tt[j] + d11 * Tt[j + 1];
  int64_t j0 = j - 1;
  if (j0 < 0) j0 = 0;
  if (j0 > W.K - 4) j0 = W.K - 4;
  double a = 0.0;
  for (int i = 0; i < 4; ++i) {                       // Lagrange form
    double w = 1.0;
    for (int q = 0; q < 4; ++q)
      if (q != i) w *= (f - W.fn[j0 + q]) / (W.fn[j0 + i] - W.fn[j0 + q]);
    a += w * A[j0 + i];
  }
  *amp = a;
  return true;
}

bool tab_sample_ok(const double* th) {                // M, q, chi1, chi2 are not used by the tabulated path
  for (int i = 4; i < NPAR; ++i) if (!std::isfinite(th[i])) return false;
  return th[4] > 0.0;
}
bool table_ok(const WaveTable& W) {
  if (W.K < 4 || !W.fn || !W.amp || !W.psi || !W.tf) return false;
  for (int64_t j = 0; j + 1 < W.K; ++j) if (!(W.fn[j + 1] > W.fn[j])) return false;
  return W.fn[0] > 0.0;
}

// A, E, T of one detector at one frequency from the tables, summed over the modes of the mask.  T = double, or
// Dual<11> for the derivatives w.r.t. the parameters this path uses (D_L, iota, phi_c, lambda, beta, psi, t_c): the
// table values are plain numbers, theta and the frame carry the tangents.
template <class T>
void response_bin_tab(const WaveTable& W, int64_t b, const T* th, const Frame<T>& F, double f,
                      uint32_t mode_mask, const pespace_oracle_detector& D, Cx<T> AET[3]) {
  for (int c = 0; c < 3; ++c) AET[c] = cx<T>(T(0.0), T(0.0));
  const T DL = th[4], iota = th[5], phic = th[6], tc = th[10];
  int imode = 0;
  for (int im = 0; im < 5; ++im) {
    if (!(mode_mask & (1u << im))) continue;
    const int l = MODE_TABLE[im].l, m = MODE_TABLE[im].m;
    double a, p, t;
    if (tab_waveform(W, b, imode, f, &a, &p, &t)) {
      const T amp = T(a) / DL;
      const T psi = T(p) + T(2.0) * K<T>::pi() * T(f) * tc - T((double)m) * phic;
      const T tf = T(t) + tc;
      Cx<T> y[6], XYZ[3], ch[3];
      links_from_waveform(iota, F, l, m, f, amp, psi, tf, D, y);
      tdi_xyz(y, T(f), D.L_m, D.tdi_gen, XYZ);
      aet(XYZ, ch);
      for (int c = 0; c < 3; ++c) AET[c] = AET[c] + ch[c];
    }
    ++imode;
  }
}

template <class T> Frame<T> tab_frame(const T* th) {
  Source<T> s = Source<T>();
  s.lam = th[7]; s.bet = th[8]; s.psi = th[9];
  return make_frame(s);
}
int popcount5(uint32_t m) { int n = 0; for (int i = 0; i < 5; ++i) n += (m >> i) & 1u; return n; }

}  // namespace

// =================================================================== C ABI
extern "C" {

void pespace_oracle_set_threads(int n) { g_threads = n; }
int pespace_oracle_get_threads(void) {
#ifdef _OPENMP
  return g_threads > 0 ? g_threads : omp_get_max_threads();
#else
  return 1;
#endif
}

int pespace_oracle_response(const double* params, int64_t B, const double* freqs, int64_t N,
                            const pespace_oracle_model* model, double* out_AET) {
  return response_impl<double>(params, B, freqs, N, model, out_AET);
}
int pespace_oracle_response_quad(const double* params, int64_t B, const double* freqs, int64_t N,
                                 const pespace_oracle_model* model, double* out_AET) {
  return response_impl<quad>(params, B, freqs, N, model, out_AET);
}

// T1: response and likelihood from tabulated mode waveforms (see the T1 block above)
int pespace_oracle_response_tab(const double* params, int64_t B, int64_t K, const double* fnodes, const double* amp,
                                const double* phase, const double* tf, const double* freqs, int64_t N,
                                const pespace_oracle_model* model, double* out) {
  if (!params || !freqs || !out || B <= 0 || N <= 0 || !model_ok(model)) return -1;
  const WaveTable W = {K, fnodes, amp, phase, tf, popcount5(model->mode_mask)};
  if (!table_ok(W)) return -1;
  const int nd = model->n_det;
  const double nan = std::numeric_limits<double>::quiet_NaN();
#pragma omp parallel for schedule(dynamic, 1) num_threads(g_threads > 0 ? g_threads : omp_get_max_threads())
  for (int64_t b = 0; b < B; ++b) {
    double* ob = out + (size_t)b * nd * 3 * N * 2;
    const double* th = params + b * NPAR;
    if (!tab_sample_ok(th)) {
      for (int64_t i = 0; i < (int64_t)nd * 3 * N * 2; ++i) ob[i] = nan;
      continue;
    }
    const Frame<double> F = tab_frame(th);
    for (int d = 0; d < nd; ++d)
      for (int64_t k = 0; k < N; ++k) {
        Cx<double> ch[3];
        if (freqs[k] > 0.0) response_bin_tab(W, b, th, F, freqs[k], model->mode_mask, model->det[d], ch);
        else for (int c = 0; c < 3; ++c) ch[c] = cx<double>(0.0, 0.0);
        for (int c = 0; c < 3; ++c) {
          ob[(((size_t)d * 3 + c) * N + k) * 2 + 0] = ch[c].re;
          ob[(((size_t)d * 3 + c) * N + k) * 2 + 1] = ch[c].im;
        }
      }
  }
  return 0;
}

int pespace_oracle_loglike_tab(const double* params, int64_t B, int64_t K, const double* fnodes, const double* amp,
                               const double* phase, const double* tf, const double* data, const double* psd,
                               const pespace_oracle_grid* grid, const pespace_oracle_model* model, double* out_lnL) {
  if (!params || !data || !psd || !out_lnL || B <= 0 || !grid_ok(grid) || !model_ok(model)) return -1;
  const WaveTable W = {K, fnodes, amp, phase, tf, popcount5(model->mode_mask)};
  if (!table_ok(W)) return -1;
  const int nd = model->n_det;
  const int64_t N = grid->N;
#pragma omp parallel for schedule(dynamic, 1) num_threads(g_threads > 0 ? g_threads : omp_get_max_threads())
  for (int64_t b = 0; b < B; ++b) {
    const double* th = params + b * NPAR;
    if (!tab_sample_ok(th)) { out_lnL[b] = -std::numeric_limits<double>::infinity(); continue; }
    const Frame<double> F = tab_frame(th);
    long double sum = 0.0L;
    for (int d = 0; d < nd; ++d)
      for (int64_t k = 0; k < N; ++k) {
        const double f = std::fma((double)k, grid->df, grid->f0);          // G11
        Cx<double> h[3];
        response_bin_tab(W, b, th, F, f, model->mode_mask, model->det[d], h);
        for (int c = 0; c < 3; ++c) {
          const size_t idx = ((size_t)d * 3 + c) * N + k;
          const double S = psd[idx];
          if (!weight_ok(S)) continue;                                      // G9
          const double rr = data[2 * idx] - h[c].re, ri = data[2 * idx + 1] - h[c].im;
          sum += (long double)(rr * rr + ri * ri) / (long double)S;
        }
      }
    out_lnL[b] = (double)(-0.5L * 4.0L * (long double)grid->df * sum);
  }
  return 0;
}

// T1 x O12: F_ij and grad_i with tabulated mode waveforms (the paper's own Fisher use: the waveform is
// fixed and the derivatives are taken w.r.t. extrinsic parameters).  Derivatives w.r.t. the raw theta entries the
// tabulated path uses (D_L, iota, phi_c, lambda, beta, psi, t_c); rows and columns of M, q, chi1, chi2 are exactly 0.
int pespace_oracle_fisher_tab(const double* params, int64_t B, int64_t K, const double* fnodes, const double* amp,
                              const double* phase, const double* tf, const double* data, const double* psd,
                              const pespace_oracle_grid* grid, const pespace_oracle_model* model, double* out_F,
                              double* out_grad) {
  if (!params || !psd || !out_F || B <= 0 || !grid_ok(grid) || !model_ok(model)) return -1;
  const WaveTable W = {K, fnodes, amp, phase, tf, popcount5(model->mode_mask)};
  if (!table_ok(W)) return -1;
  typedef Dual<NPAR> D11;
  const int nd = model->n_det;
  const int64_t N = grid->N;
  const double nan = std::numeric_limits<double>::quiet_NaN();
#pragma omp parallel for schedule(dynamic, 1) num_threads(g_threads > 0 ? g_threads : omp_get_max_threads())
  for (int64_t b = 0; b < B; ++b) {
    const double* th0 = params + b * NPAR;
    double* Fb = out_F + b * NPAR * NPAR;
    double* gb = (out_grad && data) ? out_grad + b * NPAR : nullptr;
    if (!tab_sample_ok(th0)) {
      for (int i = 0; i < NPAR * NPAR; ++i) Fb[i] = nan;
      if (gb) for (int i = 0; i < NPAR; ++i) gb[i] = nan;
      continue;
    }
    D11 th[NPAR];
    for (int i = 0; i < NPAR; ++i) { th[i] = D11(th0[i]); th[i].d[i] = 1.0; }  // identity seed (M, q, chi: unused)
    const Frame<D11> F = tab_frame(th);
    long double accF[NPAR][NPAR] = {}, accg[NPAR] = {};
    for (int d = 0; d < nd; ++d)
      for (int64_t k = 0; k < N; ++k) {
        const double f = std::fma((double)k, grid->df, grid->f0);
        Cx<D11> h[3];
        response_bin_tab(W, b, th, F, f, model->mode_mask, model->det[d], h);
        for (int c = 0; c < 3; ++c) {
          const size_t idx = ((size_t)d * 3 + c) * N + k;
          const double S = psd[idx];
          if (!weight_ok(S)) continue;
          const long double w = 1.0L / (long double)S;
          for (int i = 0; i < NPAR; ++i)
            for (int j = i; j < NPAR; ++j)
              accF[i][j] += w * (long double)(h[c].re.d[i] * h[c].re.d[j] + h[c].im.d[i] * h[c].im.d[j]);
          if (gb) {
            const double rr = data[2 * idx] - h[c].re.v, ri = data[2 * idx + 1] - h[c].im.v;
            for (int i = 0; i < NPAR; ++i) accg[i] += w * (long double)(rr * h[c].re.d[i] + ri * h[c].im.d[i]);
          }
        }
      }
    const long double norm = 4.0L * (long double)grid->df;
    for (int i = 0; i < NPAR; ++i)
      for (int j = i; j < NPAR; ++j) Fb[i * NPAR + j] = Fb[j * NPAR + i] = (double)(norm * accF[i][j]);
    if (gb) for (int i = 0; i < NPAR; ++i) gb[i] = (double)(norm * accg[i]);
  }
  return 0;
}

/* one mode's interpolated table values at the frequencies freqs (reference extrinsic values); out-of-table -> NaN */
int pespace_oracle_tab_waveform(int64_t K, const double* fnodes, const double* amp, const double* phase,
                                const double* tf, const double* freqs, int64_t N, double* out_amp, double* out_psi,
                                double* out_tf) {
  const WaveTable W = {K, fnodes, amp, phase, tf, 1};
  if (!table_ok(W) || !freqs || !out_amp || !out_psi || !out_tf || N <= 0) return -1;
  const double nan = std::numeric_limits<double>::quiet_NaN();
  for (int64_t k = 0; k < N; ++k)
    if (!tab_waveform(W, 0, 0, freqs[k], &out_amp[k], &out_psi[k], &out_tf[k])) out_amp[k] = out_psi[k] = out_tf[k] = nan;
  return 0;
}

// O11: lnL = -1/2 sum_det sum_c 4 df sum_k |d - h|^2 / S   (Eq. 10, 11, 14 with T = 1/df)
static int loglike_impl(const double* params, int64_t B, const double* data, const double* psd,
                        const pespace_oracle_grid* grid, const pespace_oracle_model* model, double* out_lnL,
                        const OrbitTab* tabs) {
  if (!params || !data || !psd || !out_lnL || B <= 0 || !grid_ok(grid) || !model_ok(model)) return -1;
  const int nd = model->n_det;
  const int64_t N = grid->N;
#pragma omp parallel for schedule(dynamic, 1) num_threads(g_threads > 0 ? g_threads : omp_get_max_threads())
  for (int64_t b = 0; b < B; ++b) {
    const double* th = params + b * NPAR;
    if (!sample_ok(th)) { out_lnL[b] = -std::numeric_limits<double>::infinity(); continue; }
    const Source<double> s = make_source(th);
    const Frame<double> F = make_frame(s);
    long double sum = 0.0L;
    for (int d = 0; d < nd; ++d)
      for (int64_t k = 0; k < N; ++k) {
        const double f = std::fma((double)k, grid->df, grid->f0);          // G11
        Cx<double> h[3];
        response_bin(s, F, f, model->mode_mask, model->det[d], h, tabs ? tabs + d : nullptr);
        for (int c = 0; c < 3; ++c) {
          const size_t idx = ((size_t)d * 3 + c) * N + k;
          const double S = psd[idx];
          if (!weight_ok(S)) continue;                                      // G9
          const double rr = data[2 * idx] - h[c].re, ri = data[2 * idx + 1] - h[c].im;
          sum += (long double)(rr * rr + ri * ri) / (long double)S;
        }
      }
    out_lnL[b] = (double)(-0.5L * 4.0L * (long double)grid->df * sum);
  }
  return 0;
}
int pespace_oracle_loglike(const double* params, int64_t B, const double* data, const double* psd,
                           const pespace_oracle_grid* grid, const pespace_oracle_model* model,
                           double* out_lnL) {
  return loglike_impl(params, B, data, psd, grid, model, out_lnL, nullptr);
}

// T2: response and likelihood with tabulated orbits; pos, vel [n_det][K][3][3]
static bool make_orbit_tabs(const pespace_oracle_model* model, int64_t K, double t0, double dt, const double* pos,
                            const double* vel, std::vector<OrbitTab>* out) {
  if (!model_ok(model)) return false;
  for (int d = 0; d < model->n_det; ++d) {
    const OrbitTab O = {K, t0, dt, pos ? pos + (size_t)d * K * 9 : nullptr, vel ? vel + (size_t)d * K * 9 : nullptr};
    if (!orbit_tab_ok(O)) return false;
    out->push_back(O);
  }
  return true;
}
int pespace_oracle_response_orb(const double* params, int64_t B, int64_t K, double t0, double dt, const double* pos,
                                const double* vel, const double* freqs, int64_t N, const pespace_oracle_model* model,
                                double* out_AET) {
  std::vector<OrbitTab> tabs;
  if (!make_orbit_tabs(model, K, t0, dt, pos, vel, &tabs)) return -1;
  return response_impl<double>(params, B, freqs, N, model, out_AET, tabs.data());
}
int pespace_oracle_loglike_orb(const double* params, int64_t B, int64_t K, double t0, double dt, const double* pos,
                               const double* vel, const double* data, const double* psd,
                               const pespace_oracle_grid* grid, const pespace_oracle_model* model, double* out_lnL) {
  std::vector<OrbitTab> tabs;
  if (!make_orbit_tabs(model, K, t0, dt, pos, vel, &tabs)) return -1;
  return loglike_impl(params, B, data, psd, grid, model, out_lnL, tabs.data());
}
/* the interpolated positions [3][3] (metres) of ONE detector's table at time t; returns 1 outside the table */
int pespace_oracle_orbit_tab(int64_t K, double t0, double dt, const double* pos, const double* vel, double t,
                             double* out_xyz) {
  const OrbitTab O = {K, t0, dt, pos, vel};
  if (!orbit_tab_ok(O) || !out_xyz) return -1;
  V3<double> c, off[3];
  if (!orbit_tab<double>(O, t, &c, off)) return 1;
  for (int n = 0; n < 3; ++n) { out_xyz[3 * n] = off[n].x; out_xyz[3 * n + 1] = off[n].y; out_xyz[3 * n + 2] = off[n].z; }
  return 0;
}

// O12: F_ij = 4 df Re sum conj(d_i h) d_j h / S ;  grad_i = 4 df Re sum conj(d - h) d_i h / S
int pespace_oracle_fisher(const double* params, int64_t B, const double* data, const double* psd,
                          const pespace_oracle_grid* grid, const pespace_oracle_model* model,
                          double* out_F, double* out_grad) {
  if (!params || !psd || !out_F || B <= 0 || !grid_ok(grid) || !model_ok(model)) return -1;
  typedef Dual<NPAR> D11;
  const int nd = model->n_det;
  const int64_t N = grid->N;
  const double nan = std::numeric_limits<double>::quiet_NaN();
#pragma omp parallel for schedule(dynamic, 1) num_threads(g_threads > 0 ? g_threads : omp_get_max_threads())
  for (int64_t b = 0; b < B; ++b) {
    const double* th0 = params + b * NPAR;
    double* Fb = out_F + b * NPAR * NPAR;
    double* gb = (out_grad && data) ? out_grad + b * NPAR : nullptr;
    if (!sample_ok(th0)) {
      for (int i = 0; i < NPAR * NPAR; ++i) Fb[i] = nan;
      if (gb) for (int i = 0; i < NPAR; ++i) gb[i] = nan;
      continue;
    }
    D11 th[NPAR];
    for (int i = 0; i < NPAR; ++i) { th[i] = D11(th0[i]); th[i].d[i] = 1.0; }  // identity seed
    const Source<D11> s = make_source(th);
    const Frame<D11> F = make_frame(s);
    long double accF[NPAR][NPAR] = {}, accg[NPAR] = {};
    for (int d = 0; d < nd; ++d)
      for (int64_t k = 0; k < N; ++k) {
        const double f = std::fma((double)k, grid->df, grid->f0);
        Cx<D11> h[3];
        response_bin(s, F, f, model->mode_mask, model->det[d], h);
        for (int c = 0; c < 3; ++c) {
          const size_t idx = ((size_t)d * 3 + c) * N + k;
          const double S = psd[idx];
          if (!weight_ok(S)) continue;
          const long double w = 1.0L / (long double)S;
          for (int i = 0; i < NPAR; ++i)
            for (int j = i; j < NPAR; ++j)
              accF[i][j] += w * (long double)(h[c].re.d[i] * h[c].re.d[j] + h[c].im.d[i] * h[c].im.d[j]);
          if (gb) {
            const double rr = data[2 * idx] - h[c].re.v, ri = data[2 * idx + 1] - h[c].im.v;
            for (int i = 0; i < NPAR; ++i) accg[i] += w * (long double)(rr * h[c].re.d[i] + ri * h[c].im.d[i]);
          }
        }
      }
    const long double norm = 4.0L * (long double)grid->df;
    for (int i = 0; i < NPAR; ++i)
      for (int j = i; j < NPAR; ++j) Fb[i * NPAR + j] = Fb[j * NPAR + i] = (double)(norm * accF[i][j]);
    if (gb) for (int i = 0; i < NPAR; ++i) gb[i] = (double)(norm * accg[i]);
  }
  return 0;
}

int pespace_oracle_waveform(const double* theta, int l, int m, const double* freqs, int64_t N,
                            double* out_amp, double* out_psi, double* out_tf) {
  if (!theta || !freqs || N <= 0 || !sample_ok(theta)) return -1;
  const Source<double> s = make_source(theta);
  for (int64_t k = 0; k < N; ++k) {
    double a, p, t;
    if (!mode_waveform(s, l, m, freqs[k], &a, &p, &t)) return -1;
    if (out_amp) out_amp[k] = a;
    if (out_psi) out_psi[k] = p;
    if (out_tf) out_tf[k] = t;
  }
  return 0;
}

int pespace_oracle_swsh(int l, int m, double iota, double* out) {
  if (!out || l < 2 || std::abs(m) > l) return -1;
  *out = swsh_m2<double>(l, m, iota);
  return 0;
}

int pespace_oracle_orbit(const pespace_oracle_detector* det, double t, double* out_xyz) {
  if (!det || !out_xyz) return -1;
  V3<double> c, off[3];
  orbit<double>(*det, t, &c, off);
  for (int n = 0; n < 3; ++n) {
    const V3<double> x = c + off[n];
    out_xyz[3 * n + 0] = x.x; out_xyz[3 * n + 1] = x.y; out_xyz[3 * n + 2] = x.z;
  }
  return 0;
}

int pespace_oracle_links(const double* theta, int l, int m, double f, const pespace_oracle_detector* det,
                         double* out_y) {
  if (!theta || !det || !out_y || !sample_ok(theta) || !(f > 0.0)) return -1;
  const Source<double> s = make_source(theta);
  const Frame<double> F = make_frame(s);
  Cx<double> y[6];
  if (!mode_links(s, F, l, m, f, *det, y)) return -1;
  for (int i = 0; i < 6; ++i) { out_y[2 * i] = y[i].re; out_y[2 * i + 1] = y[i].im; }
  return 0;
}

int pespace_oracle_tdi(const double* y, double f, double L_m, int tdi_gen, double* out_XYZ) {
  if (!y || !out_XYZ || (tdi_gen != 15 && tdi_gen != 20)) return -1;
  Cx<double> yy[6], XYZ[3];
  for (int i = 0; i < 6; ++i) yy[i] = cx<double>(y[2 * i], y[2 * i + 1]);
  tdi_xyz<double>(yy, f, L_m, tdi_gen, XYZ);
  for (int i = 0; i < 3; ++i) { out_XYZ[2 * i] = XYZ[i].re; out_XYZ[2 * i + 1] = XYZ[i].im; }
  return 0;
}

}  // extern "C"
