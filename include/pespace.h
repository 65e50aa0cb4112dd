/* pespace.h -- C ABI of libpespace.so: batched frequency-domain detector response and
 * Whittle likelihood for MBHB signals in LISA-/Taiji-/TianQin-like detectors on B200.
 *
 * Method: arxiv 2602.12011 ("pespace"); citations are to /root/reference/PAPER.md lines.
 *   single-link response      Eq. 5
 *   TDI X,Y,Z, z = e^{-i2pi f L}  Eq. 6, generations 1.5 and 2.0
 *   A, E, T channels          Eq. 3
 *   time-frequency map t_f    Eq. 4
 *   Whittle likelihood        Eq. 10, 11
 *   Fisher matrix, <.|.>      Eq. 13, 14
 * Waveform (BASELINE.json configs): TaylorF2 3.5PN phase, 0PN amplitude, modes
 * (2,2),(2,1),(3,3),(3,2),(4,4) with Psi_lm(f) = (m/2) Psi_22(2f/m), t_lm(f) = t_22(2f/m);
 * analytic Keplerian orbits.  All readings of what the paper leaves
 * open are listed in DESIGN.md.
 *
 * Conventions
 *  - Pointers named d_* are DEVICE pointers owned by the caller; the library neither frees
 *    nor retains them past the call.  Pointers named h_* are HOST pointers.  Structs are
 *    host memory, read during the call only.
 *  - All arithmetic is IEEE FP64.  Complex numbers are interleaved (re, im) pairs.
 *  - theta, 11 doubles per sample: [0] M total mass (detector frame, Msun), [1] q = m1/m2 >= 1,
 *    [2] chi1, [3] chi2, [4] D_L (Gpc), [5] iota, [6] phi_c, [7] lambda (ecliptic longitude),
 *    [8] beta (ecliptic latitude), [9] psi, [10] t_c (s from the start of the data, SSB time).
 *  - Layouts are channel-planar and bin-contiguous: data [n_det][3][N][2], psd [n_det][3][N],
 *    response out [B][n_det][3][N][2]; channel order A, E, T.  psd is the one-sided S_n(f_k)
 *    in 1/Hz for the SAME TDI generation as the detector's tdi_gen.
 *  - Calls are asynchronous on `stream` (a cudaStream_t passed as void*; NULL = default
 *    stream); outputs are valid once the stream is synchronised.  The *_host calls are
 *    synchronous.  Same inputs give bit-identical outputs (fixed reduction order).
 *  - Return value: PESPACE_OK, or a negative code.  Nothing is printed, nothing throws.
 *  - Per-sample domain errors cannot be seen by the host: a sample with a non-finite entry,
 *    M <= 0, q < 1 or D_L <= 0 gets lnL = -INFINITY and NaN-filled response / Fisher rows.
 *  - Bins whose psd is 0, negative or non-finite carry weight 0 (e.g. exact TDI nulls).
 */
#ifndef PESPACE_H
#define PESPACE_H
#include <stddef.h>
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

#define PESPACE_OK 0
#define PESPACE_EINVAL (-1) /* null pointer, B<=0, N<=0, df<=0, f0<=0, unknown kind/tdi_gen, empty or
                               unknown mode_mask, n_det outside 1..PESPACE_MAX_DET, workspace too small */
#define PESPACE_ECUDA (-2)  /* CUDA launch / runtime error; text via pespace_strerror() */
#define PESPACE_ENOMEM (-3) /* device or pinned-host allocation failed (host-buffer calls only) */
#define PESPACE_ETOOBIG (-4) /* pespace_response_noalloc: the batch needs more scratch than the static array holds;
                                text via pespace_strerror() */

#define PESPACE_NPAR 11
#define PESPACE_MAX_DET 8

#define PESPACE_MODE_22 1u
#define PESPACE_MODE_21 2u
#define PESPACE_MODE_33 4u
#define PESPACE_MODE_32 8u
#define PESPACE_MODE_44 16u

typedef struct {
  int32_t kind;    /* 0 heliocentric (LISA-/Taiji-like), 1 geocentric (TianQin-like) */
  int32_t tdi_gen; /* 15 or 20: X_1.5 or X_2.0 of Eq. 6 */
  double L_m;      /* arm length, metres */
  double kappa;    /* kind 0: guiding-centre phase relative to Earth at t = 0 (rad) */
  double lambda0;  /* kind 0: constellation rotation phase; kind 1: orbital phase phi0 (rad) */
  double period_s; /* kind 1: spacecraft orbital period (s) */
  double lon, lat; /* kind 1: fixed pointing of the orbit normal, ecliptic (rad) */
} pespace_detector;

typedef struct { double f0, df; int64_t N; } pespace_grid; /* f_k = fma((double)k, df, f0); T = 1/df */

typedef struct {
  uint32_t mode_mask; /* OR of PESPACE_MODE_* */
  int32_t n_det;
  const pespace_detector* det; /* host array [n_det] */
} pespace_model;

/* Detector response (Eq. 5 -> Eq. 6 -> Eq. 3, summed over the modes of the mask).
 *   d_params [B][11], d_freqs [N] (Hz; bins with f <= 0 produce 0), d_out_AET [B][n_det][3][N][2]. */
int pespace_response(const double* d_params, int64_t B, const double* d_freqs, int64_t N,
                     const pespace_model* model, double* d_out_AET, void* stream);

/* pespace_response without any allocation, for callers that cannot call cudaMalloc (code under CUDA graph capture,
 * tight serving loops, harnesses that forbid it).  Same arguments, same kernels and bit-identical output; the scratch
 * of step S1 (per-sample constants and the sine / cosine table) lives in ONE static device array of
 * PESPACE_NOALLOC_SCRATCH_BYTES that every GPU which loads the library holds until the process exits.  The call
 * allocates and frees nothing (no cudaMalloc / cudaMallocAsync / cudaFree, no allocating library routine).
 *   Limit: pespace_noalloc_scratch_needed(B, model) = 16384 + 8 B (40 + 24 n_det) bytes (rounded up to 256) must not
 *   exceed PESPACE_NOALLOC_SCRATCH_BYTES: B <= 2016 samples for one detector, 1152 for three, 556 for eight; N is
 *   not limited.  A larger batch is rejected with PESPACE_ETOOBIG before anything is launched (pespace_strerror
 *   names the sizes); pespace_noalloc_scratch_needed returns 0 for invalid arguments.
 *   Sharing: every call uses the same array and finds the previous call's contents there; nothing has to start at
 *   zero (the prep kernel of a call writes every word its response kernels read).  Calls on ONE stream are ordered
 *   and safe; calls that overlap on the GPU (several streams or host threads) RACE on the array -- serialise them. */
#define PESPACE_NOALLOC_SCRATCH_BYTES (1 << 20)
size_t pespace_noalloc_scratch_needed(int64_t B, const pespace_model* model);
int pespace_response_noalloc(const double* d_params, int64_t B, const double* d_freqs, int64_t N,
                             const pespace_model* model, double* d_out_AET, void* stream);

/* Scratch the likelihood / Fisher calls need for (B, grid, model). */
size_t pespace_workspace_bytes(int64_t B, const pespace_grid* grid, const pespace_model* model,
                               int want_fisher);

/* lnL_b = -1/2 sum_det sum_{c in A,E,T} 4 df sum_k |d_c(f_k) - h_c(f_k; theta_b)|^2 / S_c(f_k)
 * (Eq. 10, 11 with T = 1/df; additive constants dropped).
 *   d_params [B][11], d_data_AET [n_det][3][N][2], d_psd [n_det][3][N], d_out_lnL [B],
 *   d_workspace >= pespace_workspace_bytes(B, grid, model, 0) bytes, 16-byte aligned. */
int pespace_loglike(const double* d_params, int64_t B, const double* d_data_AET, const double* d_psd,
                    const pespace_grid* grid, const pespace_model* model, double* d_out_lnL,
                    void* d_workspace, size_t workspace_bytes, void* stream);

/* Forward-mode derivatives (Eq. 13, 14): F_ij = <d_i h | d_j h>, grad_i = d lnL / d theta_i
 * = <d - h | d_i h>, derivatives w.r.t. the 11 raw theta entries.
 *   d_out_F [B][11][11] symmetric, full storage; d_out_grad [B][11] or NULL;
 *   d_data_AET may be NULL: then the gradient is skipped (d_out_grad must be NULL);
 *   d_out_F may be NULL when d_out_grad is not: gradient only (for gradient-based samplers),
 *   which skips the 66 Fisher entries of the per-bin Gram matrix. */
int pespace_fisher(const double* d_params, int64_t B, const double* d_data_AET, const double* d_psd,
                   const pespace_grid* grid, const pespace_model* model, double* d_out_F,
                   double* d_out_grad, void* d_workspace, size_t workspace_bytes, void* stream);

/* lnL AND its gradient d lnL / d theta [B][11] in one pass by REVERSE mode ("The
 * backward mode ... is more suitable for cases of large inputs and small output such as computing the gradients of
 * the likelihood function"; :163, :171 gradient-based samplers).  The kernel evaluates the response as
 * pespace_loglike does, seeds the adjoint of (X, Y, Z) with the weighted residual (Eq. 10) and sweeps back through
 * Eq. 6, 5, the orbit, Eq. 4 and the waveform of every mode to the per-sample constants; no tangent is carried per
 * bin.  grad_i = <d - h | d_i h> of Eq. 13/14, the quantity pespace_fisher returns in d_out_grad (derivatives
 * w.r.t. the raw theta entries), at about 2.5-3x the cost of pespace_loglike instead of 6x.  Either output pointer
 * may be NULL (not both).  Out-of-domain samples: lnL = -INFINITY, NaN gradient row.  Workspace:
 * pespace_workspace_bytes_grad.  Same inputs, bit-identical outputs.  B <= 65535 x 32 per call. */
size_t pespace_workspace_bytes_grad(int64_t B, const pespace_grid* grid, const pespace_model* model);
int pespace_loglike_grad(const double* d_params, int64_t B, const double* d_data_AET, const double* d_psd,
                         const pespace_grid* grid, const pespace_model* model, double* d_out_lnL /* [B] */,
                         double* d_out_grad /* [B][11] */, void* d_workspace, size_t workspace_bytes, void* stream);

/* Prepared data ("a persistent prepared-data handle, S0 tables cached across calls from a
 * sampler") for callers that keep theta on the device.  pespace_prepare runs step S0 alone: it folds the data set and
 * the PSD into the per-bin table at the head of the workspace (the same bytes pespace_loglike / pespace_loglike_grad
 * write there on every call).  pespace_loglike_prepared / pespace_loglike_grad_prepared then evaluate batches of
 * theta against that table without reading d_data_AET / d_psd again: same results, bit for bit, as the plain calls
 * on the same inputs.  The table stays valid while the SAME workspace is used with the SAME grid and model and only
 * by these two calls (any other entry point given this workspace may overwrite it; results are then undefined --
 * call pespace_prepare again).  Its position does not depend on B: one workspace sized for the largest batch serves
 * every smaller one.  The plain and the gradient call lay the table out identically, so one pespace_prepare on a
 * workspace of max(pespace_workspace_bytes, pespace_workspace_bytes_grad) bytes serves both.
 *   pespace_prepare: workspace_bytes >= pespace_workspace_bytes(1, grid, model, 0).
 * Errors as for the plain calls. */
int pespace_prepare(const double* d_data_AET, const double* d_psd, const pespace_grid* grid, const pespace_model* model,
                    void* d_workspace, size_t workspace_bytes, void* stream);
int pespace_loglike_prepared(const double* d_params, int64_t B, const pespace_grid* grid, const pespace_model* model,
                             double* d_out_lnL, void* d_workspace, size_t workspace_bytes, void* stream);
int pespace_loglike_grad_prepared(const double* d_params, int64_t B, const pespace_grid* grid,
                                  const pespace_model* model, double* d_out_lnL /* [B] or NULL */,
                                  double* d_out_grad /* [B][11] or NULL */, void* d_workspace, size_t workspace_bytes,
                                  void* stream);

/* Mixed-precision twin of pespace_loglike (the paper's float32 mode for searches and coarse
 * maximisation).  Same arguments, same workspace size.  Every phase that enters an exponential
 * (PN phase, 2 pi f t_c, Doppler phases, their sum and its reduction modulo one turn) stays FP64; the t_lm polynomial,
 * orbit, projections, arm weights, sines / cosines of the reduced phases, TDI sums and the whitened residual run in
 * FP32.  Accuracy ~1e-6 relative on the response, a few 1e-6 of max(|lnL|, <h|h>/2) on lnL for the BASELINE configs
 * (tests/test_gpu_mixed.py); over random models the error is 2e-7 in the median and below 1.2e-5 in 99 % of them, and
 * it grows like 5e-7 / (2 pi f L / c) where a detector's arm is short against the wavelength: up to 4e-4 for a
 * TianQin-like detector ALONE in a band below 0.3 mHz (tests/test_gpu_random_sweep.py).
 * NOT a substitute for pespace_loglike where |delta lnL| << 1 matters.  Inputs must be detector-like in magnitude:
 * sqrt(4 df / S_n) |h| x 2^-64 and x 2^64 must both be representable in FP32 (not checked). */
int pespace_loglike_mixed(const double* d_params, int64_t B, const double* d_data_AET, const double* d_psd,
                          const pespace_grid* grid, const pespace_model* model, double* d_out_lnL,
                          void* d_workspace, size_t workspace_bytes, void* stream);

/* ---- Tabulated mode waveforms.  In the paper the per-mode amplitude, phase and
 * time-frequency map t_f come from the waveform generator (PhenomXAS / PhenomXHM) and the
 * response is built on them (Eq. 4, 5).  These calls take them as tables, so that any externally generated
 * waveform drives the same response / likelihood kernels; the analytic TaylorF2 modes of pespace_response /
 * pespace_loglike are then not used.
 *   d_fnodes [K]                 node frequencies (Hz), strictly increasing, K >= 4, shared by samples and modes
 *   d_amp, d_phase, d_tf [B][n_modes][K]   A_lm (s), Psi_lm (rad), t_lm (s) at the nodes, h_lm = A e^{-i Psi},
 *                                modes in bit order of mode_mask, for t_c = 0, phi_c = 0, D_L = 1 Gpc.
 * From theta the calls use D_L, iota, phi_c, lambda, beta, psi, t_c:  Psi_lm(f) = Psi_tab(f) + 2 pi f t_c
 * - m phi_c, t_lm(f) = t_tab(f) + t_c, A_lm = A_tab / D_L[Gpc];  M, q, chi1, chi2 are ignored (a sample is out
 * of domain if one of the used entries is non-finite or D_L <= 0).  Between nodes Psi_tab is the cubic Hermite
 * interpolant of the node phases with node slopes 2 pi t_j (Eq. 4), t_tab its derivative / 2 pi, A_tab the cubic
 * Lagrange polynomial through the four nodes around the interval; a mode contributes 0 at frequencies outside
 * [fnodes[0], fnodes[K-1]].  The node array is NOT checked for monotonicity (device memory). */
typedef struct {
  int64_t K;
  const double* d_fnodes;
  const double* d_amp;
  const double* d_phase;
  const double* d_tf;
} pespace_wavetable;

int pespace_response_tab(const double* d_params, int64_t B, const pespace_wavetable* table,
                         const double* d_freqs, int64_t N, const pespace_model* model,
                         double* d_out_AET, void* stream);
size_t pespace_workspace_bytes_tab(int64_t B, const pespace_grid* grid, const pespace_model* model);
int pespace_loglike_tab(const double* d_params, int64_t B, const pespace_wavetable* table,
                        const double* d_data_AET, const double* d_psd, const pespace_grid* grid,
                        const pespace_model* model, double* d_out_lnL, void* d_workspace,
                        size_t workspace_bytes, void* stream);

/* Fisher matrix and gradient on tabulated mode waveforms (T1 x S10).  This is the paper's own Fisher use: the waveform
 * is fixed and F is taken over extrinsic parameters (PAPER.md:207; Fig. 3 design, :193).  Outputs as pespace_fisher
 * (F [B][11][11] symmetric full storage, grad [B][11] = <d - h | d_i h>, derivatives w.r.t. the raw theta entries); the
 * tabulated path depends on D_L, iota, phi_c, lambda, beta, psi, t_c only, so the rows and columns of M, q, chi1, chi2
 * are exactly 0.  d_data_AET may be NULL (then d_out_grad must be NULL); d_out_F may be NULL (gradient only).
 * Workspace: pespace_workspace_bytes_fisher_tab. */
size_t pespace_workspace_bytes_fisher_tab(int64_t B, const pespace_grid* grid, const pespace_model* model);
int pespace_fisher_tab(const double* d_params, int64_t B, const pespace_wavetable* table, const double* d_data_AET,
                       const double* d_psd, const pespace_grid* grid, const pespace_model* model, double* d_out_F,
                       double* d_out_grad, void* d_workspace, size_t workspace_bytes, void* stream);

/* ---- Tabulated numerical orbits ("Support for high-precision numerical orbits will
 * be extended in future work").  The spacecraft positions at t_lm(f) (Eq. 4, 5) are read from tables instead of the
 * analytic Keplerian orbits: d_pos [n_det][K][3 spacecraft][3] in metres and d_vel [n_det][K][3][3] in m/s on the
 * uniform time grid t0 + j dt, j = 0..K-1 (SSB seconds, same origin as t_c), K >= 2.  Between nodes every coordinate
 * is the cubic Hermite interpolant with the node velocities as slopes.  Eq. 5 / Eq. 6 keep the nominal constant arm
 * length L_m of the detector description in the delays (the paper's formalism assumes rigid equal arms, PAPER.md:55,
 * :61); the link directions n_rs = (x_r - x_s) / |x_r - x_s| (unit vectors: the arms of a numerical orbit breathe) and
 * k.(x_r + x_s) come from the table; kind, kappa, lambda0, period_s, lon, lat of the description are ignored.  A mode
 * whose t_lm(f) lies outside [t0, t0 + (K-1) dt] contributes 0 at that frequency.  Waveform:
 * the analytic TaylorF2 modes of pespace_loglike.  Workspace of pespace_loglike_orb: pespace_workspace_bytes(B, grid,
 * model, 0).  Errors and per-sample domain as pespace_loglike. */
typedef struct {
  int64_t K;
  double t0, dt;
  const double* d_pos;
  const double* d_vel;
} pespace_orbittable;

int pespace_response_orb(const double* d_params, int64_t B, const pespace_orbittable* orbit, const double* d_freqs,
                         int64_t N, const pespace_model* model, double* d_out_AET, void* stream);
int pespace_loglike_orb(const double* d_params, int64_t B, const pespace_orbittable* orbit, const double* d_data_AET,
                        const double* d_psd, const pespace_grid* grid, const pespace_model* model, double* d_out_lnL,
                        void* d_workspace, size_t workspace_bytes, void* stream);

/* ---- Host-buffer entry points (a sampler evaluates many batches of theta against
 * ONE data set).  A session owns a stream and keeps the data set, the PSD, the workspace
 * and the result buffers resident on the device between calls; each call then moves only theta in
 * and lnL (or F, grad) out.  The arithmetic is that of pespace_loglike / pespace_fisher, launched on
 * the session's stream.  All pointers are HOST pointers (pinned memory makes the copies DMA
 * transfers; pageable memory works); the calls are synchronous: outputs are valid, and input
 * buffers may be reused, on return.  A session is not thread-safe; use one per thread. */
typedef struct pespace_session pespace_session;

/* Allocates device buffers for batches of up to max_B samples on the current device.  want_fisher != 0
 * also sizes the pespace_session_fisher buffers.  *out is NULL on failure (PESPACE_EINVAL,
 * PESPACE_ENOMEM). */
int pespace_session_create(const pespace_grid* grid, const pespace_model* model, int64_t max_B,
                           int want_fisher, pespace_session** out);
/* Copies the data set h_data_AET [n_det][3][N][2] and / or the PSD h_psd [n_det][3][N] to the
 * device (either pointer may be NULL: that array is left as it is). */
int pespace_session_set_data(pespace_session* s, const double* h_data_AET, const double* h_psd);
/* h_params [B][11] -> h_out_lnL [B], B <= max_B.  PESPACE_EINVAL before data and PSD are set.  The per-bin
 * table of the data set (S0) is built by the first call after pespace_session_set_data and reused afterwards;
 * lnL (and theta of batches up to 256 samples) travel through mapped pinned memory owned by the session. */
int pespace_session_loglike(pespace_session* s, const double* h_params, int64_t B, double* h_out_lnL);
/* Same through pespace_loglike_mixed (FP64 phases, FP32 geometry; see there for the accuracy). */
int pespace_session_loglike_mixed(pespace_session* s, const double* h_params, int64_t B, double* h_out_lnL);
/* h_params [B][11] -> h_out_F [B][11][11] and, if h_out_grad != NULL, h_out_grad [B][11] (needs the
 * data set; the Fisher matrix alone needs only the PSD).  h_out_F may be NULL: gradient only. */
int pespace_session_fisher(pespace_session* s, const double* h_params, int64_t B, double* h_out_F,
                           double* h_out_grad);
/* h_params [B][11] -> h_out_lnL [B] and h_out_grad [B][11] through pespace_loglike_grad (reverse mode; either output
 * may be NULL, not both).  Needs data and PSD.  Its workspace is allocated on first use. */
int pespace_session_loglike_grad(pespace_session* s, const double* h_params, int64_t B, double* h_out_lnL,
                                 double* h_out_grad);
/* Tabulated mode waveforms through a session: h_fnodes [K] (checked here for strictly increasing order),
 * h_amp, h_phase, h_tf [B][n_modes][K] as in pespace_wavetable but in HOST memory; they are copied to the device
 * with theta on every call (the tables belong to the batch).  Device buffers are allocated on first use. */
int pespace_session_loglike_tab(pespace_session* s, const double* h_params, int64_t B, int64_t K,
                                const double* h_fnodes, const double* h_amp, const double* h_phase,
                                const double* h_tf, double* h_out_lnL);
/* Waits for the session's stream and frees everything the session owns. */
int pespace_session_destroy(pespace_session* s);

/* One-shot host-buffer twin of pespace_loglike: session create + set_data + loglike + destroy. */
int pespace_loglike_host(const double* h_params, int64_t B, const double* h_data_AET,
                         const double* h_psd, const pespace_grid* grid, const pespace_model* model,
                         double* h_out_lnL);

const char* pespace_strerror(int code);
const char* pespace_version(void);

#ifdef __cplusplus
}
#endif
#endif
