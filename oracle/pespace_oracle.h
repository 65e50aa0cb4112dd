/* pespace_oracle.h -- C ABI of the CPU oracle (HOST pointers only).
 *
 * TEST INFRASTRUCTURE, NOT PRODUCT CODE.  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may load this library.
 * It shares no code, header, table or constant generator with the CUDA path
 * (paper_2602_12011_b200/csrc, include/pespace.h); the struct layouts below are
 * restated here on purpose.
 *
 * What it computes: the plain definition of the frequency-domain detector
 * response and Whittle likelihood of arxiv 2602.12011 ("pespace"), PAPER.md
 * Eq. 3, 4, 5, 6, 10, 11, 13, 14, with the waveform / orbit / frame readings
 * O0-O12 and G1-G16 of SURVEY.md section 8(c) (listed in DESIGN.md).
 *
 * All arithmetic IEEE double; sums over bins in extended precision, in bin
 * order.  Return value 0 = OK, -1 = invalid argument.
 */
#ifndef PESPACE_ORACLE_H
#define PESPACE_ORACLE_H
#include <stddef.h>
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

typedef struct {
  int32_t kind;     /* 0 heliocentric (LISA-/Taiji-like), 1 geocentric (TianQin-like) */
  int32_t tdi_gen;  /* 15 or 20 (Eq. 6) */
  double L_m;       /* arm length, metres */
  double kappa;     /* kind 0: guiding-centre phase relative to Earth at t=0, rad */
  double lambda0;   /* kind 0: constellation rotation phase; kind 1: phi0, rad */
  double period_s;  /* kind 1: spacecraft orbital period, s */
  double lon, lat;  /* kind 1: pointing of the orbit normal (ecliptic), rad */
} pespace_oracle_detector;

typedef struct { double f0, df; int64_t N; } pespace_oracle_grid; /* f_k = fma(k, df, f0) */

typedef struct {
  uint32_t mode_mask; /* bit0 (2,2) bit1 (2,1) bit2 (3,3) bit3 (3,2) bit4 (4,4) */
  int32_t n_det;
  const pespace_oracle_detector* det;
} pespace_oracle_model;

/* theta (11 doubles per sample): M[Msun] q chi1 chi2 D_L[Gpc] iota phi_c lambda beta psi t_c[s] */

/* out_AET [B][n_det][3][N][2] : A, E, T of Eq. 3 after Eq. 5, 6, summed over modes. */
int pespace_oracle_response(const double* params, int64_t B, const double* freqs, int64_t N,
                            const pespace_oracle_model* model, double* out_AET);
/* same, evaluated internally in IEEE binary128 (pin P14); slow. */
int pespace_oracle_response_quad(const double* params, int64_t B, const double* freqs, int64_t N,
                                 const pespace_oracle_model* model, double* out_AET);

/* data_AET [n_det][3][N][2], psd [n_det][3][N]; out_lnL [B] (Eq. 10, 11; T = 1/df). */
int pespace_oracle_loglike(const double* params, int64_t B, const double* data_AET,
                           const double* psd, const pespace_oracle_grid* grid,
                           const pespace_oracle_model* model, double* out_lnL);

/* out_F [B][11][11] (Eq. 13, 14), out_grad [B][11] = d lnL / d theta (may be NULL;
 * skipped if data_AET is NULL).  Forward-mode dual numbers, SURVEY O12. */
int pespace_oracle_fisher(const double* params, int64_t B, const double* data_AET,
                          const double* psd, const pespace_oracle_grid* grid,
                          const pespace_oracle_model* model, double* out_F, double* out_grad);

/* ---- T1: tabulated mode waveforms (amplitude, phase and t_f per mode come
 * from the waveform generator).  Tables on K >= 4 shared nodes fnodes[K] (strictly increasing, Hz): amp, phase, tf
 * [B][n_modes][K], modes in bit order of the mask, for t_c = 0, phi_c = 0, D_L = 1 Gpc.  The call applies
 * Psi += 2 pi f t_c - m phi_c, t_f += t_c, A /= D_L from theta; M, q, chi1, chi2 of theta are ignored.
 * Interpolation: Psi cubic Hermite with node slopes 2 pi tf_j, t_f its derivative / 2 pi, A cubic Lagrange on
 * 4 nodes; a mode is 0 outside [fnodes[0], fnodes[K-1]]. */
int pespace_oracle_response_tab(const double* params, int64_t B, int64_t K, const double* fnodes,
                                const double* amp, const double* phase, const double* tf,
                                const double* freqs, int64_t N, const pespace_oracle_model* model,
                                double* out_AET);
int pespace_oracle_loglike_tab(const double* params, int64_t B, int64_t K, const double* fnodes,
                               const double* amp, const double* phase, const double* tf,
                               const double* data_AET, const double* psd, const pespace_oracle_grid* grid,
                               const pespace_oracle_model* model, double* out_lnL);
/* T1 x O12: Fisher matrix and gradient with tabulated mode waveforms; derivatives w.r.t. the theta entries this path
 * uses (D_L, iota, phi_c, lambda, beta, psi, t_c), rows / columns of M, q, chi1, chi2 exactly 0.  out_grad may be
 * NULL; skipped if data_AET is NULL. */
int pespace_oracle_fisher_tab(const double* params, int64_t B, int64_t K, const double* fnodes,
                              const double* amp, const double* phase, const double* tf, const double* data_AET,
                              const double* psd, const pespace_oracle_grid* grid, const pespace_oracle_model* model,
                              double* out_F, double* out_grad);
/* the interpolants of ONE (sample, mode) table at freqs[N]; NaN outside the table */
int pespace_oracle_tab_waveform(int64_t K, const double* fnodes, const double* amp, const double* phase,
                                const double* tf, const double* freqs, int64_t N, double* out_amp,
                                double* out_psi, double* out_tf);

/* ---- T2: tabulated numerical orbits.  Positions pos [n_det][K][3 spacecraft][3]
 * (metres) and velocities vel [n_det][K][3][3] (m/s) on the uniform time grid t0 + j dt (SSB seconds, origin of t_c);
 * cubic Hermite in time; Eq. 5 / 6 keep the nominal L of the detector description, the link directions are the unit
 * vectors (x_r - x_s) / |x_r - x_s|; a mode whose t_lm(f) lies outside the table contributes 0.  The detector's kind / kappa / lambda0 / period / pointing are ignored. */
int pespace_oracle_response_orb(const double* params, int64_t B, int64_t K, double t0, double dt, const double* pos,
                                const double* vel, const double* freqs, int64_t N, const pespace_oracle_model* model,
                                double* out_AET);
int pespace_oracle_loglike_orb(const double* params, int64_t B, int64_t K, double t0, double dt, const double* pos,
                               const double* vel, const double* data_AET, const double* psd,
                               const pespace_oracle_grid* grid, const pespace_oracle_model* model, double* out_lnL);
/* interpolated positions [3][3] of ONE detector's table (pos, vel [K][3][3]) at time t; returns 1 outside the table */
int pespace_oracle_orbit_tab(int64_t K, double t0, double dt, const double* pos, const double* vel, double t,
                             double* out_xyz);

/* ---- pieces, exported so that the pins can check them one at a time ---- */

/* per-mode amplitude A_lm(f) [s], phase Psi_lm(f) [rad], t_lm(f) [s]   (O2-O5) */
int pespace_oracle_waveform(const double* theta, int l, int m, const double* freqs, int64_t N,
                            double* out_amp, double* out_psi, double* out_tf);
/* spin-weight -2 spherical harmonic (Goldberg sum), phi = 0            (O6) */
int pespace_oracle_swsh(int l, int m, double iota, double* out);
/* spacecraft positions [3][3] in metres at SSB time t                  (O8) */
int pespace_oracle_orbit(const pespace_oracle_detector* det, double t, double* out_xyz);
/* six single-link responses of ONE mode at ONE frequency               (O9, Eq. 5)
 * order: y12 y21 y13 y31 y23 y32, each (re, im)                          */
int pespace_oracle_links(const double* theta, int l, int m, double f,
                         const pespace_oracle_detector* det, double* out_y);
/* TDI X, Y, Z of Eq. 6 from six links in the order above               (O10) */
int pespace_oracle_tdi(const double* y, double f, double L_m, int tdi_gen, double* out_XYZ);

void pespace_oracle_set_threads(int n); /* OpenMP threads over samples; <=0 = all cores */
int pespace_oracle_get_threads(void);

#ifdef __cplusplus
}
#endif
#endif
