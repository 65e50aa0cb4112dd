// pespace_fisher_tab.cuh -- Fisher matrix and gradient on tabulated mode waveforms (T1 x S10).  This is the paper's
// own Fisher use: the waveform is fixed (PhenomX from the generator) and F is taken over extrinsic parameters
// (Fig. 3 design :193).  With tables, theta enters through D_L, iota, phi_c, lambda, beta, psi, t_c only
// (reading T1): the 4-tangent phase / time polynomials of the analytic Fisher path drop out, the geometry keeps its
// 3-tangent dual number (orbit angle, lambda, beta), the rest is closed form.  The kernel is fisher_kernel with stage A
// replaced by the table interpolation of pespace_tab.cuh and one "class" per tabulated mode; Gram step, reduction and
// combine_fisher_kernel are shared.  Rows and columns of M, q, chi1, chi2 come out exactly 0.
#pragma once
#include "pespace_fisher.cuh"
#include "pespace_tab.cuh"

namespace pespace {

// per-sample constants with tangents for this path: [sample_stride][DUW], slots (M, q, chi1, chi2, iota, lambda, beta)
static __global__ void prep_samples_tab_du_kernel(const double* __restrict__ params, long long B, PrepArgs A,
                                                  double* __restrict__ consts) {
  const long long b = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (b >= B) return;
  const double* thp = params + b * NPAR;
  const int stride = sample_stride(A.n_det);
  double* o = consts + b * (long long)stride * DUW;
  for (int i = 0; i < stride * DUW; ++i) o[i] = 0.0;
  bool ok = thp[4] > 0.0;
  for (int i = 4; i < NPAR; ++i) ok = ok && isfinite(thp[i]);      // M, q, chi1, chi2 are not used here
  o[W_A * DUW] = 1.0;
  if (!ok) return;
  o[W_A * DUW + 1] = 1.0;                  // validity flag read by combine_fisher_kernel (a non-zero "M tangent" of W_A)
  auto put = [o](int idx, const Du<7>& val) {
    double* p = o + idx * DUW;
    p[0] = val.v;
    for (int t = 0; t < 7; ++t) p[1 + t] = val.d[t];
  };
  Du<7> iota(thp[5]), lam(thp[7]), bet(thp[8]);
  iota.d[4] = 1.0; lam.d[5] = 1.0; bet.d[6] = 1.0;
  const Du<7> pol(thp[9]), tc(thp[10]);
  put(W_TC, tc);
  put(W_PH0, Du<7>(-kTurn * thp[6] / (2.0 * kPi)));
  put(W_MDL, Du<7>(-1.0 / thp[4]));
  Du<7> Yp[5], Ym[5];
  swsh_pairs(iota, Yp, Ym);
  const int ll[5] = {2, 2, 3, 3, 4};
  int slot = 0;
  for (int i = 0; i < 5; ++i) {
    if (!((A.mode_mask >> i) & 1u)) continue;
    const double sg = (ll[i] & 1) ? -1.0 : 1.0;
    put(W_KA + 2 * slot, (0.5 / thp[4]) * (Yp[i] + sg * Ym[i]));        // K+ / D_L
    put(W_KA + 2 * slot + 1, (1.0 / thp[4]) * (Yp[i] - sg * Ym[i]));    // 2 Kc / D_L
    ++slot;
  }
  prep_frame<Du<7>>(lam, bet, pol, tc, A, put);
}

// phase-like scalars of tabulated mode i at this bin (no M, q, chi tangents; amplitude tangent: iota only)
__device__ __forceinline__ void fisher_stage_tab(int i, const double (&w)[NWT], const double* __restrict__ sc,
                                                 const TabC& T, long long b, double ftc, ClassScal& o) {
  const long long j = (long long)w[WT_J], j0 = (long long)w[WT_J0];
  const size_t base = ((size_t)b * T.n_modes + i) * (size_t)T.K;
  const double* P = T.phase + base + j;
  const double* Tt = T.tf + base + j;
  const double* A = T.amp + base + j0;
  const double P0 = P[0], dP = P[1] - P0, t0 = Tt[0], t1 = Tt[1];
  double psi = fma(w[WT_H01], dP, P0) * (kTurn / (2.0 * kPi));
  psi -= whole_turns(psi);
  psi += fma(w[WT_C10], t0, w[WT_C11] * t1);
  o.psi = psi + fma((double)T.m[i], cv(sc, W_PH0), ftc);
  o.tau = fma(w[WT_Q01], dP, fma(w[WT_Q10], t0, w[WT_Q11] * t1));
#pragma unroll
  for (int q = 0; q < 4; ++q) { o.dpsi[q] = 0.0; o.dtau[q] = 0.0; }
  const double a = fma(w[WT_L0], A[0], fma(w[WT_L0 + 1], A[1], fma(w[WT_L0 + 2], A[2], w[WT_L0 + 3] * A[3])));
  o.CKp = a * ca3(sc, W_KA + 2 * i);
  o.CKc = a * ca3(sc, W_KA + 2 * i + 1);
}

template <int KIND>
__global__ void __launch_bounds__(FBLOCK, PESPACE_FMINB)
fisher_tab_kernel(const double* __restrict__ consts, long long B, TabC T, const double* __restrict__ bins /* [n_det][NBF][N] */,
                  const double* __restrict__ wt /* [NWT][N] */, long long N, DetC dc, int n_det, int det, int grad_only,
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
    for (int s = 0; s < ns; ++s) {
      const double* sc = csm + s * FS_STRIDE;
      const double ftc = mul_mod_turn(bc.fT, cv(sc, W_TC));
#pragma unroll 1
      for (int i = 0; i < T.n_modes; ++i) {
        ClassScal cs;
        fisher_stage_tab(i, iw, sc, T, b0 + s, ftc, cs);
        fisher_class_cs<KIND>((double)T.m[i], i == 0, cs, bc, sc, dc, J);
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
  if (threadIdx.x < NGP) {
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

}  // namespace pespace
