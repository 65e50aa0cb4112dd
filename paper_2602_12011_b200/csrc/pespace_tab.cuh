// pespace_tab.cuh -- tabulated mode waveforms (amplitude, phase and t_f of
// every mode come from the waveform generator).  The tables live on K shared nodes f_0 < ... < f_{K-1}, per sample
// and per mode of the mask (bit order), for t_c = 0, phi_c = 0, D_L = 1 Gpc; theta supplies D_L, iota, phi_c,
// lambda, beta, psi, t_c (reading T1 of DESIGN.md):
//   Psi_lm(f) = Psi_tab(f) + 2 pi f t_c - m phi_c,   t_lm(f) = t_tab(f) + t_c,   A_lm(f) = A_tab(f) / D_L.
// Psi_tab: cubic Hermite interpolant of the node phases with node slopes 2 pi t_j (Eq. 4); t_tab: its
// derivative / 2 pi; A_tab: cubic Lagrange polynomial through 4 nodes; a mode is 0 outside the table.
//
// All interpolation weights depend on the bin only (the nodes are shared), so they are computed once per call into a
// per-bin table; per (sample, mode, bin) the kernel gathers 4 phase/time nodes and 4 amplitude nodes (neighbouring
// bins read the same nodes: broadcast within the warp, L1/L2 hits across warps) and hands phase, time and amplitude
// to the same geometry / TDI code as the analytic path (eval_geom).  Each mode is its own class here.
#pragma once
#include "pespace_device.cuh"

namespace pespace {

struct TabC {            // kernel parameter: the tables
  long long K;
  const double* amp;     // [B][n_modes][K]
  const double* phase;
  const double* tf;
  int n_modes;
  int m[5];              // azimuthal number of mode i
};

// per-bin interpolation record [NWT][N]
enum : int { WT_J = 0,      // interval index j (as a double)
             WT_J0,         // first node of the amplitude stencil
             WT_H01,        // Psi = Psi_j + H01 (Psi_{j+1} - Psi_j) + (C10 t_j + C11 t_{j+1}) / (kTurn / 2 pi)
             WT_C10, WT_C11,     // kTurn h h10, kTurn h h11: phase contribution of the slopes, in pu
             WT_Q01, WT_Q10, WT_Q11,   // kTurn/yr x weights of (Psi_{j+1} - Psi_j), t_j, t_{j+1} in t_tab
             WT_L0,         // four Lagrange weights (0 outside the table)
             NWT = WT_L0 + 4 };
static_assert(NWT == 12, "interpolation record is 12 doubles");

// per-sample constants of the tabulated path: W_TC, W_PH0 (= -kTurn phi_c / 2 pi, times m in the kernel), W_VALID,
// W_KA + 2 i: K+ / D_L and 2 Kc / D_L of mode i; detector blocks as in the analytic path.
static __global__ void prep_samples_tab_kernel(const double* __restrict__ params, long long B, PrepArgs A,
                                               double* __restrict__ consts, double2* __restrict__ trig) {
  const long long b = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  fill_trig_entry(trig, b);
  if (b >= B) return;
  const double* th = params + b * NPAR;
  const int stride = sample_stride(A.n_det);
  double* o = consts + b * stride;
  for (int i = 0; i < stride; ++i) o[i] = 0.0;
  bool ok = th[4] > 0.0;
  for (int i = 4; i < NPAR; ++i) ok = ok && isfinite(th[i]);      // M, q, chi1, chi2 are not used here
  o[W_A] = 1.0;
  if (!ok) return;                                                // W_VALID stays 0
  o[W_VALID] = 1.0;
  o[W_TC] = th[10];
  o[W_PH0] = -kTurn * th[6] / (2.0 * kPi);
  double Yp[5], Ym[5];
  swsh_pairs(th[5], Yp, Ym);
  const int ll[5] = {2, 2, 3, 3, 4};
  int slot = 0;
  for (int i = 0; i < 5; ++i) {
    if (!((A.mode_mask >> i) & 1u)) continue;
    const double sg = (ll[i] & 1) ? -1.0 : 1.0;
    o[W_KA + 2 * slot] = 0.5 * (Yp[i] + sg * Ym[i]) / th[4];        // K+ / D_L
    o[W_KA + 2 * slot + 1] = (Yp[i] - sg * Ym[i]) / th[4];          // 2 Kc / D_L  (n.e_x.n = 2 (n.u)(n.v))
    ++slot;
  }
  prep_frame<double>(th[7], th[8], th[9], th[10], A, [o](int idx, double val) { o[idx] = val; });
}

// interpolation record of one frequency
__device__ __forceinline__ void tab_weights(double f, const double* __restrict__ fn, long long K, double (&w)[NWT]) {
#pragma unroll
  for (int i = 0; i < NWT; ++i) w[i] = 0.0;
  if (!(f >= fn[0]) || !(f <= fn[K - 1])) return;                  // outside: amplitude weights 0, nodes 0..3
  long long lo = 0, hi = K - 1;
  while (hi - lo > 1) {
    const long long mid = (lo + hi) / 2;
    if (fn[mid] <= f) lo = mid; else hi = mid;
  }
  const double h = fn[lo + 1] - fn[lo], s = (f - fn[lo]) / h;
  const double h10 = s * (1.0 - s) * (1.0 - s), h01 = s * s * (3.0 - 2.0 * s), h11 = s * s * (s - 1.0);
  const double d01 = 6.0 * s * (1.0 - s), d10 = (1.0 - s) * (1.0 - 3.0 * s), d11 = s * (3.0 * s - 2.0);
  long long j0 = lo - 1;
  if (j0 < 0) j0 = 0;
  if (j0 > K - 4) j0 = K - 4;
  w[WT_J] = (double)lo; w[WT_J0] = (double)j0;
  w[WT_H01] = h01; w[WT_C10] = kTurn * h * h10; w[WT_C11] = kTurn * h * h11;
  const double ty = kTurn / kYear;
  w[WT_Q01] = ty * d01 / (h * 2.0 * kPi); w[WT_Q10] = ty * d10; w[WT_Q11] = ty * d11;
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    double L = 1.0;
#pragma unroll
    for (int q = 0; q < 4; ++q)
      if (q != i) L *= (f - fn[j0 + q]) / (fn[j0 + i] - fn[j0 + q]);
    w[WT_L0 + i] = L;
  }
}

static __global__ void prep_tab_weights_kernel(GridC G, const double* __restrict__ fn, long long K,
                                               double* __restrict__ wt /* [NWT][N] */) {
  const long long k = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= G.N) return;
  double w[NWT];
  tab_weights(fma((double)k, G.df, G.f0), fn, K, w);
#pragma unroll
  for (int i = 0; i < NWT; ++i) wt[(size_t)i * (size_t)G.N + (size_t)k] = w[i];
}

// phase (pu, reduced), tau = kTurn t_tab / yr and amplitude of tabulated mode i of sample b at this bin
__device__ __forceinline__ void tab_mode(int i, const double (&w)[NWT], long long j, long long j0,
                                         const double* __restrict__ sc, const TabC& T, long long b, double ftc,
                                         double& psi, double& tau, double& a) {
  const size_t base = ((size_t)b * T.n_modes + i) * (size_t)T.K;
  const double* P = T.phase + base + j;
  const double* Tt = T.tf + base + j;
  const double* A = T.amp + base + j0;
  const double P0 = P[0], dP = P[1] - P0, t0 = Tt[0], t1 = Tt[1];
  psi = fma(w[WT_H01], dP, P0) * (kTurn / (2.0 * kPi));            // node part of Psi_tab, pu (up to ~1e8)
  psi -= whole_turns(psi);                                         // mod one turn, exact
  psi += fma(w[WT_C10], t0, w[WT_C11] * t1);                       // slope part (small)
  psi += fma((double)T.m[i], sc[W_PH0], ftc);                      // + kTurn [f t_c - m phi_c / 2 pi]
  tau = fma(w[WT_Q01], dP, fma(w[WT_Q10], t0, w[WT_Q11] * t1));    // kTurn t_tab / yr
  a = fma(w[WT_L0], A[0], fma(w[WT_L0 + 1], A[1], fma(w[WT_L0 + 2], A[2], w[WT_L0 + 3] * A[3])));
}

// X, Y, Z of one (sample, bin, detector) summed over the tabulated modes.  Returns (Re, -Im) pairs in S.  NM = number of
// modes known at compile time (1: no loop; 5: unrolled) or 0: run-time loop over T.n_modes.
template <int KIND, int NM>
__device__ __forceinline__ void eval_xyz_tab(const BinC& bc, const double (&w)[NWT], const double* __restrict__ sc,
                                             const DetC& dc, const double2* __restrict__ tab, const TabC& T,
                                             long long b, double (&S)[6]) {
  const double tc = sc[W_TC];
  const double ftc = mul_mod_turn(bc.fT, tc);
  const long long j = (long long)w[WT_J], j0 = (long long)w[WT_J0];
  if constexpr (NM > 0) {
#pragma unroll
    for (int i = 0; i < NM; ++i) {
      double psi, tau, a;
      tab_mode(i, w, j, j0, sc, T, b, ftc, psi, tau, a);
      if (i == 0) eval_geom<KIND, true, true>(bc, sc, dc, tab, psi, tau, a * sc[W_KA], a * sc[W_KA + 1], S);
      else eval_geom<KIND, false, true>(bc, sc, dc, tab, psi, tau, a * sc[W_KA + 2 * i], a * sc[W_KA + 2 * i + 1], S);
    }
  } else {
#pragma unroll
    for (int i = 0; i < 6; ++i) S[i] = 0.0;
#pragma unroll 1
    for (int i = 0; i < T.n_modes; ++i) {
      double psi, tau, a;
      tab_mode(i, w, j, j0, sc, T, b, ftc, psi, tau, a);
      eval_geom<KIND, false, true>(bc, sc, dc, tab, psi, tau, a * sc[W_KA + 2 * i], a * sc[W_KA + 2 * i + 1], S);
    }
  }
}

#ifndef PESPACE_TAB_TILE
#define PESPACE_TAB_TILE 64
#endif
constexpr int TAB_TILE = PESPACE_TAB_TILE;     // samples per block
constexpr size_t tab_smem_bytes() {
  return sizeof(double) * ((size_t)2 * NTAB + (size_t)TAB_TILE * SMEM_STRIDE + (size_t)(BLOCK / 32) * TAB_TILE);
}
__device__ __forceinline__ void stage_tile_n(double* smem, const double* __restrict__ consts, long long b0,
                                             long long B, int n_det, int det, int tile) {
  const int stride = sample_stride(n_det);
  for (int i = threadIdx.x; i < tile * SMEM_STRIDE; i += blockDim.x) {
    const int s = i / SMEM_STRIDE, j = i % SMEM_STRIDE;
    long long b = b0 + s;
    if (b >= B) b = B - 1;
    const int src = (j < D_BASE) ? j : (D_BASE + D_STRIDE * det + (j - D_BASE));
    smem[i] = consts[b * stride + src];
  }
}

// likelihood from tables: grid (bin blocks, sample tiles of TAB_TILE); one launch per detector
#ifndef PESPACE_MINBT
#define PESPACE_MINBT 2
#endif
template <int KIND, int NM>
__global__ void __launch_bounds__(BLOCK, PESPACE_MINBT)
loglike_tab_kernel(const double* __restrict__ consts, const double2* __restrict__ trig, long long B, TabC T,
                   const double* __restrict__ bins /* [n_det][NBF][N] */, const double* __restrict__ wt /* [NWT][N] */,
                   long long N, DetC dc, int n_det, int det, double* __restrict__ partial /* [n_det][gridDim.x][B] */) {
  double2* tab = reinterpret_cast<double2*>(pespace_dyn_smem);
  double* smem = reinterpret_cast<double*>(tab + NTAB);
  double (*red)[TAB_TILE] = reinterpret_cast<double (*)[TAB_TILE]>(smem + TAB_TILE * SMEM_STRIDE);
  const long long b0 = (long long)blockIdx.y * TAB_TILE;
  stage_trig(tab, trig);
  stage_tile_n(smem, consts, b0, B, n_det, det, TAB_TILE);
  const long long k = (long long)blockIdx.x * BLOCK + threadIdx.x;
  const bool live = k < N;
  const size_t kk = (size_t)(live ? k : N - 1);
  const double* bp = bins + (size_t)det * NBF * (size_t)N + kk;
  BinC bc;
  bc.fT = bp[BF_FT * N]; bc.sth = bp[BF_STH * N]; bc.cth = bp[BF_CTH * N];
  bc.cf = bc.lnf3 = bc.fm53 = bc.fm83 = bc.fm76 = 0.0;
  double dr[3], di[3], w[3], iw[NWT];
#pragma unroll
  for (int c = 0; c < 3; ++c) {
    dr[c] = bp[(BF_DR + c) * N]; di[c] = bp[(BF_DI + c) * N];
    w[c] = live ? bp[(BF_W + c) * N] : 0.0;
  }
#pragma unroll
  for (int i = 0; i < NWT; ++i) iw[i] = wt[(size_t)i * (size_t)N + kk];
  __syncthreads();
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int ns = (int)min((long long)TAB_TILE, B - b0);
  for (int s = 0; s < ns; ++s) {
    double S[6];
    eval_xyz_tab<KIND, NM>(bc, iw, smem + s * SMEM_STRIDE, dc, tab, T, b0 + s, S);
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

// response from tables on an arbitrary frequency array (weights computed in the kernel, once per thread)
template <int KIND>
__global__ void __launch_bounds__(BLOCK, 2)
response_tab_kernel(const double* __restrict__ consts, const double2* __restrict__ trig, long long B, TabC T,
                    const double* __restrict__ fn, const double* __restrict__ freqs, long long N, DetC dc, int n_det,
                    int det, double2* __restrict__ out /* [B][n_det][3][N] */) {
  double2* tab = reinterpret_cast<double2*>(pespace_dyn_smem);
  double* smem = reinterpret_cast<double*>(tab + NTAB);
  const long long b0 = (long long)blockIdx.y * TAB_TILE;
  stage_trig(tab, trig);
  stage_tile_n(smem, consts, b0, B, n_det, det, TAB_TILE);
  const long long k = (long long)blockIdx.x * BLOCK + threadIdx.x;
  const bool live = k < N;
  const double fraw = freqs[live ? k : N - 1];
  const bool pos = fraw > 0.0;
  const double f = pos ? fraw : 1.0;
  BinC bc;
  bc.fT = kTurn * f;
  sincospi(2.0 * f * dc.Lbar, &bc.sth, &bc.cth);
  bc.cf = bc.lnf3 = bc.fm53 = bc.fm83 = 0.0;
  bc.fm76 = 1.0;                                         // the amplitude comes from the table
  double gr, gi, iw[NWT];
  tdi_prefactor(bc, dc.gen, gr, gi);
  tab_weights(f, fn, T.K, iw);
  __syncthreads();
  const int ns = (int)min((long long)TAB_TILE, B - b0);
  const double i2 = 0.70710678118654752440, i6 = 0.40824829046386301637, i3 = 0.57735026918962576451;
  for (int s = 0; s < ns; ++s) {
    const double* sc = smem + s * SMEM_STRIDE;
    double S[6];
    eval_xyz_tab<KIND, 0>(bc, iw, sc, dc, tab, T, b0 + s, S);
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
