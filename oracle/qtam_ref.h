/* qtam_ref.h -- CPU ORACLE for the QTAM forward / inverse Q-transform.
 *
 * TEST INFRASTRUCTURE, NOT PRODUCT CODE.  Only tests/, __graft_entry__.smoke() and the
 * `cpu_baseline` / `--impl reference` legs of bench.py may load this library.  It shares no code,
 * header, table or constant generator with the CUDA library (paper_2603_29785_b200/csrc); the
 * CUDA path never calls it.
 *
 * What it is: the plain definition of the transform of arxiv/paper_2603_29785, evaluated
 * slowly in fp64 (long-double accumulation in the naive DFT sums), on host pointers.  Every entry
 * point cites the passage it follows; the readings R1..R14 where the paper is silent or garbled are
 * listed in DESIGN.md section "Readings".
 *
 * Layouts (identical to the CUDA library's, include/qtam.h): x is [batch][N] real; coefficients are
 * [batch][coeffs_per_segment] complex interleaved (re,im), row k of a segment at `offset_k`, time
 * index fastest.  All floating point here is double; an fp32 configuration is checked by feeding
 * the oracle the fp32-rounded input promoted to double.
 *
 * Pins (tests/test_oracle_*.py, all `-m "not gpu"`): P1 brute-force circular convolution, P2 decimated
 * = samples of the demodulated dense tile, P3 per-row energy, P4 round trip, P5 linearity, P6 frame
 * energy identity and bounds, P7 closed form for a pure sinusoid, P8 shift covariance, P9 impulse
 * symmetry, P10 white-noise variance, P11 FFT engine vs naive DFT, P12 plan invariants, plus
 * closed-form window values (tests/golden/).  Unpinned: the paper's printed residuals and shapes
 * -- they need GWOSC data / unstated defaults ("parity unpinned" for those
 * numbers only; no oracle function depends on them).
 */
#ifndef QTAM_REF_H
#define QTAM_REF_H
#include <stddef.h>
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

typedef struct qtam_ref_plan qtam_ref_plan;

typedef struct {
  int     window;                   /* 0 bisquare (PAPER.md:67 Eq. 6, :272 A1), 1 Hann (A2 :276), 2 Kaiser
                                       (A3 :280), 3 Tukey (A4 :284), 4 Planck-taper (A5-A6 :293-299)    */
  int     clamp_mode;               /* 0 none, 1 auto (PAPER.md:307 Eq. A7), 2 manual                */
  double  clamp_overlap;            /* multiplies N_t*Delta f_max in A7; 1.0 = paper literal (R7)    */
  int64_t max_window_bins;          /* L_max when clamp_mode == 2                                    */
  double  cover_floor;              /* R9, default 1e-2                                              */
  int     rows_are_bins_per_octave; /* 0: `spacing` = rows per plane; 1: bins per octave B (:303)    */
  double  window_param;             /* Kaiser beta > 0, Tukey alpha_T in (0,1], Planck alpha_P in (0,1] */
  const double *freqs;              /* manual grid (:303): n_freqs ascending centre frequencies; when    */
  int     n_freqs;                  /* n_freqs >= 2 it replaces fmin / fmax / spacing                    */
  int64_t tile_length;              /* output length per row: 0 = nextpow2(L_k) per row (R5, default);
                                       -1 = uniform, nextpow2 of the largest window (the paper's padded
                                       layout :127-129); n > 0 = uniform user-set n, a power of two >= max L */
  double  epsilon;                  /* Eq. 12 (:143): unnormalised window value outside the support, used by
                                       the dense tiles and their single-tile inversion only; 0 = none       */
  const int *plane_window;          /* composite filter bank (:327 "scanning not only across varying Quality
                                       factors Q ... but also across diverse windowing functions and their
                                       associated shape parameters"): nQ window families, one per plane (the Q
                                       list may repeat a value); NULL = `window` for every plane           */
  const double *plane_window_param; /* nQ shape parameters (NULL = 0 for every plane)                      */
} qtam_ref_options;

typedef struct {
  int plane, row; double q, f_request, f_center;
  int64_t kc, dk, L, M, offset; double norm;
} qtam_ref_row;

typedef struct {
  int n_planes, n_rows; int64_t n, n_bins, coeffs_per_segment, sum_L;
  int64_t cover_lo, cover_hi, holes, cover_count; double frame_A, frame_B;
} qtam_ref_info;

/* engine: 0 = naive O(n^2) DFT sums with long-double accumulation (THE definition);
 *         1 = the oracle's own textbook recursive radix-2 FFT (validated against 0 by pin P11).   */

/* O-plan: grid, centre bin (:75, R2), bandwidth (R1), clamp (A7/A8 :307-311),
 * bisquare window (Eq. 6 :67), unit-energy normalisation (Eq. 5 :63 as read in R3),
 * frame operator P (C36 :536), cover set (R9). Returns 0 on success, nonzero on invalid input. */
int  qtam_ref_plan_create(qtam_ref_plan **out, double fs, int64_t N, const double *Q, int nQ,
                          double fmin, double fmax, double spacing, const qtam_ref_options *opt);
void qtam_ref_plan_destroy(qtam_ref_plan *p);
int  qtam_ref_plan_info(const qtam_ref_plan *p, qtam_ref_info *out);
int  qtam_ref_plan_rows(const qtam_ref_plan *p, qtam_ref_row *out, int capacity);
/* normalised window W_k[j], j=-dk..dk, L values */
int  qtam_ref_plan_window(const qtam_ref_plan *p, int row, double *out);
/* frame operator and cover set, plane = -1 joint, else that plane (C36, R9, R10); n_bins values */
int  qtam_ref_plan_frame(const qtam_ref_plan *p, int plane, double *P_out, uint8_t *cover_out);

/* O-forward (PAPER.md:323 A9, :583 C46, :589 C47, scale R4): coef[b][offset_k+n] */
int  qtam_ref_forward(const qtam_ref_plan *p, const double *x, int batch, double *coef, int engine);
/* O-inverse (PAPER.md:135 Eq. 11, :598 C49, :602 C50; pseudo-inverse on the cover set, R9/R10) */
int  qtam_ref_inverse(const qtam_ref_plan *p, const double *coef, int batch, int plane,
                      double *x_out, int engine);
/* O-dense (PAPER.md:377 C3): out[b][row-row_begin][tau] complex, tau = 0..N-1 */
int  qtam_ref_dense(const qtam_ref_plan *p, const double *x, int batch, int row_begin, int row_end,
                    double *out, int engine);
/* O-brute (PAPER.md:382-388 C4/C5): T_k[tau] = sum_n x[n] h_k[(tau-n) mod N], no DFT of x. One
 * segment, one row; out is N complex. */
int  qtam_ref_brute_tile(const qtam_ref_plan *p, const double *x, int row, double *out);
/* O-threshold (BASELINE.json config 5, R11): zero Y_k[n] where |Y_k[n]| < kappa*median_n|Y_k[n]|.
 * fp64 decision; the _f32 variant takes every decision in IEEE binary32 with the operation order
 * stated in DESIGN.md ("threshold arithmetic") so that a float kernel can match it bit for bit. */
int  qtam_ref_threshold_rowmedian(const qtam_ref_plan *p, double *coef, int batch, double kappa);
int  qtam_ref_threshold_rowmedian_f32(const qtam_ref_plan *p, float *coef, int batch, float kappa);

/* Single-tile inversion by spectral division (Eq. 13 :148), demodulation bypassed: tile = ONE dense tile T_k
 * of every segment ([batch][N] complex, as qtam_ref_dense writes it with epsilon > 0);
 * x = F^{-1}{ F[T_k][f] / W_k[f] }, W_k[f] = norm_k * (window on the support, epsilon elsewhere), f = 0..N/2.
 * Returns nonzero when the plan's epsilon is 0 (the division is undefined off the support). */
int  qtam_ref_dense_invert(const qtam_ref_plan *p, const double *tile, int batch, int row, double *x_out);

/* Re-modulation (Eq. 10a :113-117, :129): out[b][offset_k + n] = sqrt(M_k/N) e^{+2 pi i kc n/M_k} Y_k[n]
 * = the dense tile T_k at tau = n N/M_k (identity P2).  Same layout as the coefficients. */
int  qtam_ref_remodulate(const qtam_ref_plan *p, const double *coef, int batch, double *out);

/* Instantaneous frequency (Fig. 5): out[b][offset_k + n] =
 * (kc + (M_k/2 pi) Arg(Y_k[(n+1) mod M_k] conj Y_k[n])) / T in Hz (reading R16). out: real, coefficient layout. */
int  qtam_ref_instantaneous_frequency(const qtam_ref_plan *p, const double *coef, int batch, double *out);

/* Multi-Q scan: out_metric[batch][n_planes] = total energy (metric 0) or peak pixel
 * (metric 1) of every plane's |Y|^2, out_best[batch] = the plane with the largest value per segment
 * (lowest index on ties; may be NULL). */
int  qtam_ref_plane_metric(const qtam_ref_plan *p, const double *coef, int batch, int metric,
                           double *out_metric, int32_t *out_best);
/* Projection onto the cover set: one-sided DFT of x, zero the bins outside C, inverse (R9). */
int  qtam_ref_project_cover(const qtam_ref_plan *p, const double *x, int batch, int plane,
                            double *x_out, int engine);
/* The paper's output-length options (A22: PAPER.md:150, :158-160, :184, :343): every row resampled to the same
 * n time samples, n any integer >= the largest window.  qtam_ref_output_length: mode -1 "standard" N/2+1, mode -2
 * "minimal" = the largest 2 dk + 1.  forward_length: out [batch][rows][n] complex,
 * Y'_k[m] = (N n)^{-1/2} sum_j X[kc+j] W_k[j] e^{+2 pi i j m/n} (C46/C47 with N_out = n).  inverse_length: Eq. 11
 * from such an image (C49 with N_out = n).  resample: [rows][n_in] -> [rows][n_out] through each row's band
 * (:160, Fig. 3).  Naive long-double sums; `engine` only selects the long transform of x. */
int64_t qtam_ref_output_length(const qtam_ref_plan *p, int mode);
int  qtam_ref_forward_length(const qtam_ref_plan *p, const double *x, int batch, int64_t n, double *out, int engine);
int  qtam_ref_inverse_length(const qtam_ref_plan *p, const double *in, int batch, int64_t n, int plane, double *x_out,
                             int engine);
int  qtam_ref_resample(const qtam_ref_plan *p, const double *in, int batch, int64_t n_in, int64_t n_out, double *out);
/* Clusters of active pixels of one Q-plane's [rows][M] image (R19): connected components
 * under 4-connectivity, time axis circular; components smaller than min_area dropped.  mask: [batch][rows][M]
 * non-zero = active.  labels: [batch][rows][M], 0 or 1 + the smallest pixel index of the cluster.  count: [batch]. */
int  qtam_ref_cluster_labels(const uint8_t *mask, int batch, int rows, int64_t M, int min_area, int32_t *labels,
                             int32_t *count);
/* One-sided spectrum X[f], f=0..N/2 (PAPER.md:365 C1); out is n_bins complex per segment. */
int  qtam_ref_spectrum(const qtam_ref_plan *p, const double *x, int batch, double *X_out, int engine);

/* Raw DFT engines on n complex points (interleaved); sign = -1 forward (C1), +1 inverse kernel,
 * never scaled. qtam_ref_dft: naive sums. qtam_ref_fft: recursive radix-2 with a radix-3 step,
 * n = 2^a or 3 * 2^a.                                                                            */
int  qtam_ref_dft(const double *in, double *out, int64_t n, int sign);
int  qtam_ref_fft(const double *in, double *out, int64_t n, int sign);
/* Optimal-selection output: out[batch][max_p C_p] complex, plane best[b] of segment b at its
 * start, zero after it. */
int  qtam_ref_gather_plane(const qtam_ref_plan *p, const double *coef, int batch, const int32_t *best, double *out);

/* Number of OpenMP threads the batch loops use. */
int  qtam_ref_threads(void);
void qtam_ref_set_threads(int n);

#ifdef __cplusplus
}
#endif
#endif
