/* qtam.h -- C ABI of libqtam: QTAM forward / inverse Q-transform on NVIDIA B200 (sm_100a).
 *
 * Method: arxiv/paper_2603_29785 ("QTAM: Q-Transform Amplitude Modulation"), cited below as
 * PAPER.md:<line>.  The library implements the data-parallel hot path only:
 *   forward  x[b][N] real  ->  one long real FFT (C1 :365)
 *                          ->  per Q-plane and log-spaced frequency row: multiply the band under the
 *                              row's frequency window (A9 :323), shift it to baseband (C46 :583) and
 *                              run a short inverse FFT of the window's support scaled by
 *                              sqrt(N_out/N_in) (C47 :589)  ->  complex envelope Y_k[n]
 *   inverse  Y -> per-row FFT, amplitude correction sqrt(N_in/N_out) and shift back (C49 :598),
 *                 times the window, summed over rows, divided by the frame operator
 *                 P[f] = sum_k |W_k[f]|^2 (Eq. 11 :135, C36 :536, C50 :602), one long inverse FFT.
 * The readings taken where the paper is silent or garbled (bandwidth constant, centre-bin rounding,
 * window normalisation, clamp, cover set ...) are R1-R14 of DESIGN.md.
 *
 * Conventions
 *   - Pointers named d_* are DEVICE pointers (cudaMalloc'ed or torch CUDA tensors); every other
 *     pointer is a HOST pointer.  `stream` is a cudaStream_t passed as void* (NULL = default stream).
 *   - d_x:    [batch][N] real, contiguous, float (QTAM_F32) or double (QTAM_F64).
 *   - d_coef: [batch][coeffs_per_segment] complex interleaved (re,im) of the same width; row k of
 *             segment b starts at element b*coeffs_per_segment + offset_k and holds M_k values, time
 *             index fastest; t_n = n*T/M_k.
 *   - Ownership: the caller owns every buffer it passes and keeps it alive until the stream reaches
 *     the call.  The plan owns its device tables and a workspace sized for `max_batch` segments;
 *     qtam_plan_destroy frees them.
 *   - Calls are asynchronous on `stream`, never synchronise the host, never allocate, do not modify
 *     their inputs, and in/out buffers must not alias.  One in-flight call per plan.  A call may run
 *     independent kernels on streams the plan owns; they start after the work already on `stream` and
 *     `stream` waits for them before anything issued after the call (event fork / join: capturable in
 *     a CUDA graph).
 *   - Errors: status codes only; nothing is thrown across the ABI; outputs are untouched on failure.
 *     There is no CPU fallback: without a CUDA device every compute call returns QTAM_ERR_CUDA.
 */
#ifndef QTAM_H
#define QTAM_H
#include <stddef.h>
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

typedef struct qtam_plan qtam_plan;                      /* opaque, owned by the library */

typedef enum { QTAM_F32 = 0, QTAM_F64 = 1 } qtam_dtype;  /* real in / complex out of that width */

typedef enum {
  QTAM_OK = 0,
  QTAM_ERR_INVALID_ARG = 1,   /* NULL pointer, N neither 2^k nor 3 * 2^k (k >= 3), fmax >= fs/2, fmin <= 0,
                                 Q < sqrt(11), half-width < 1 bin, batch > max_batch, bad row range,
                                 max_batch > 65535 */
  QTAM_ERR_UNSUPPORTED = 2,   /* window family / size outside what this build implements */
  QTAM_ERR_ALLOC = 3,         /* host or device allocation failed at plan creation */
  QTAM_ERR_CUDA = 4,          /* a CUDA runtime call or launch failed (or no device) */
  QTAM_ERR_EMPTY_FRAME = 5,   /* the plan's cover set is empty */
  QTAM_ERR_TOO_LARGE = 6      /* qtam_cluster_noalloc only: the problem does not fit the library's fixed scratch */
} qtam_status;

/* All fields optional; pass NULL for the defaults. struct_size = sizeof(qtam_options) (ABI version). */
typedef struct {
  size_t  struct_size;
  int     window;                   /* PAPER.md App. A: 0 bisquare (Eq. 6 :67, A1 :272) [default], 1 Hann
                                       (A2 :276), 2 Kaiser (A3 :280), 3 Tukey (A4 :284), 4 Planck-taper
                                       (A5-A6 :293-299, R15).  The half-width is the same for
                                       every family (R1)                                               */
  int     clamp_mode;               /* 0 none, 1 auto = Eq. A7 [default], 2 manual  */
  double  clamp_overlap;            /* multiplies N_t*Delta f_max in A7; default 1.0 = paper (R7)  */
  int64_t max_window_bins;          /* L_max when clamp_mode == 2                                  */
  double  cover_floor;              /* R9: a bin is invertible iff some unnormalised window value
                                       there is >= cover_floor; default 1e-2                       */
  int     rows_are_bins_per_octave; /* 0: `spacing` = rows per plane, endpoints inclusive;
                                       1: `spacing` = bins per octave B, f = fmin*2^(r/B) (:303)   */
  int     max_batch;                /* workspace is sized for this many segments; default 1; at most
                                       65535 (the batch index is a grid dimension of several kernels) */
  double  window_param;             /* Kaiser beta > 0; Tukey alpha_T, Planck alpha_P in (0, 1]     */
  const double *freqs;              /* manual grid (:303): n_freqs ascending centre frequencies in Hz
                                       (host pointer, read during plan creation only); when           */
  int     n_freqs;                  /* n_freqs >= 2 they replace fmin / fmax / spacing              */
  int64_t tile_length;              /* output samples per row: 0 = nextpow2(L_k) per row (R5) [default];
                                       -1 = uniform, nextpow2 of the largest window: the paper's
                                       zero-padded layout (:127-129), coefficients = [rows][M] per
                                       segment; n > 0 = uniform, user-set power of two >= max L     */
  double  epsilon;                  /* Eq. 12 (R17): unnormalised window value
                                       off the support (and floor on it) for qtam_dense and
                                       qtam_dense_invert only; 0 = plain windows [default]           */
  const int *plane_window;          /* composite filter bank (:327 "scanning not only across varying Quality
                                       factors Q ... but also across diverse windowing functions and their
                                       associated shape parameters"): nQ window families, one per plane (the Q
                                       list may repeat a value; host pointer, read during plan creation only);
                                       NULL = `window` for every plane [default]                         */
  const double *plane_window_param; /* nQ shape parameters (NULL = 0 for every plane)                    */
  int64_t out_length;               /* the paper's output-resolution option (:150, :158-160, :184, :343) for
                                       qtam_forward_length / _inverse_length / _resample: 0 = not used
                                       [default]; -1 = "standard" N/2 + 1; -2 = "minimal", the largest
                                       window's 2 dk + 1 (= ceil(N_t Delta f_max) + 1, R18);
                                       n > 0 = user-set, any integer >= the largest window             */
} qtam_options;

/* Host-side row table entry; rows are ordered plane-major (Q list order), ascending frequency. */
typedef struct {
  int plane, row;
  double q, f_request, f_center;    /* f_center = kc/T, the bin the window is really centred on (R2) */
  int64_t kc, dk, L, M, offset;     /* centre bin, half-width, L = 2dk+1, M = nextpow2(L), offset_k  */
  double norm;                      /* 1/sqrt(sum_j W'[j]^2), Eq. 5 as read in R3                    */
} qtam_row;

typedef struct {
  int n_planes, n_rows;
  int64_t n, n_bins, coeffs_per_segment, sum_L;
  int64_t cover_lo, cover_hi, holes;      /* joint cover set: first/last bin, gaps in between      */
  double frame_A, frame_B;                /* min of P over the cover set, max of P (C39 :550)       */
  size_t workspace_bytes;                 /* device memory the plan holds                           */
} qtam_info;

/* Plan (host, once): frequency grid f_r = fmin*(fmax/fmin)^(r/(R-1)) or fmin*2^(r/B),
 * centre bins, bandwidths, clamp A7/A8 (:307-311), the windows (App. A) and their normalisation
 * (Eq. 5-7 :63-72), output lengths, the frame operator and cover sets, device tables + workspace.
 * Q: nQ quality factors (host pointer), one plane each.  *out is written only on QTAM_OK.
 * N = 2^k or 3 * 2^k samples (the paper's benchmark segments are 6 s at 4096 Hz = 24576 = 3 * 2^13, PAPER.md:178,
 * :339): the long transforms of the latter take one radix-3 step around power-of-two transforms. */
qtam_status qtam_plan_create(qtam_plan **out, double fs, int64_t N, const double *Q, int nQ,
                             double fmin, double fmax, double spacing, qtam_dtype dtype,
                             const qtam_options *opt);
/* Same plan, host tables only: needs no CUDA device.  info/rows/window/frame work; every compute
 * call on it returns QTAM_ERR_CUDA.  For inspecting a tiling before committing device memory. */
qtam_status qtam_plan_create_host(qtam_plan **out, double fs, int64_t N, const double *Q, int nQ,
                                  double fmin, double fmax, double spacing, qtam_dtype dtype,
                                  const qtam_options *opt);
qtam_status qtam_plan_destroy(qtam_plan *p);
qtam_status qtam_plan_info(const qtam_plan *p, qtam_info *out);
/* copies n_rows entries into `out` (host); capacity must be >= n_rows */
qtam_status qtam_plan_rows(const qtam_plan *p, qtam_row *out, int capacity);
/* normalised window W_k[j], j = -dk..dk, as the device tables hold it before rounding to the plan's
 * dtype (host doubles, L values) */
qtam_status qtam_plan_window(const qtam_plan *p, int row, double *out);
/* frame operator P[f] and cover set, f = 0..N/2; plane = -1 joint, else that plane; either output
 * may be NULL (host pointers) */
qtam_status qtam_plan_frame(const qtam_plan *p, int plane, double *P_out, uint8_t *cover_out);

/* Forward: rows a1-a3 of the hot path.
 *   Y_k[n] = (N*M_k)^(-1/2) * sum_j X[kc+j] W_k[j] e^{+2 pi i j n / M_k},  n = 0..M_k-1         */
qtam_status qtam_forward(qtam_plan *p, const void *d_x, int batch, void *d_coef, void *stream);

/* Inverse: rows a5-a8 (PAPER.md:133-138 Eq. 11, :596-603).  plane = -1 inverts the joint frame of
 * all planes, plane = p >= 0 only that plane's rows with that plane's P (R10).  Bins outside the
 * cover set are set to zero (pseudo-inverse, R9), so inverse(forward(x)) = Pi_C x.               */
qtam_status qtam_inverse(qtam_plan *p, const void *d_coef, int batch, int plane, void *d_x_out,
                         void *stream);

/* Dense (non-decimated) tiles, the check path for shift invariance (C3):
 *   T_k[tau] = (1/N) sum_j X[kc+j] W_k[j] e^{+2 pi i (kc+j) tau / N},  tau = 0..N-1
 * d_out: [batch][row_end-row_begin][N] complex.                                                   */
qtam_status qtam_dense(qtam_plan *p, const void *d_x, int batch, int row_begin, int row_end,
                       void *d_out, void *stream);

/* Single-tile inversion by spectral division (Eq. 13; demodulation bypassed): d_tile = ONE dense
 * tile T_row per segment, [batch][N] complex as qtam_dense writes it on a plan with epsilon > 0;
 * x = F^{-1}{ F[T_row][f] / W_row[f] } -> d_x_out [batch][N] real.  Conditioning: errors of the tile are
 * amplified by up to 1/epsilon.  N up to 8192 (float) / 4096 (double): a check path like qtam_dense.
 * QTAM_ERR_INVALID_ARG when the plan's epsilon is 0. */
qtam_status qtam_dense_invert(qtam_plan *p, const void *d_tile, int batch, int row, void *d_x_out, void *stream);

/* The paper's output-length options (plans created with out_length != 0).
 * Every row at the same number n = qtam_output_length(p, 0) of time samples, n any integer >= the largest window
 * (no power of two): d_img = [batch][n_rows][n] complex, row k at time t_m = m T / n,
 *   forward_length   Y'_k[m] = (N n)^(-1/2) sum_j X[kc+j] W_k[j] e^{+2 pi i j m / n}      (C46 / C47 with N_out = n)
 *   inverse_length   Eq. 11 from such an image (C49 with N_out = n); plane as in qtam_inverse
 *   resample         to_standard = 1: [n_rows][n] -> [n_rows][N/2+1]  ("up-sampling the compressed image back to
 *                    the original size", :160, Fig. 3); 0: the reverse.  Exact: every row is band limited to its window.
 * qtam_output_length: mode 0 = the plan's n, -1 = N/2 + 1, -2 = the largest window (0 when the plan has none).
 * The short transforms are direct sums over the window's support, O(n L) per row: a layout converter for images of
 * the paper's sizes, not a step of the hot path.  QTAM_ERR_INVALID_ARG on a plan created with out_length = 0. */
int64_t     qtam_output_length(const qtam_plan *p, int mode);
qtam_status qtam_forward_length(qtam_plan *p, const void *d_x, int batch, void *d_img, void *stream);
qtam_status qtam_inverse_length(qtam_plan *p, const void *d_img, int batch, int plane, void *d_x_out, void *stream);
qtam_status qtam_resample(qtam_plan *p, const void *d_in, int batch, int to_standard, void *d_out, void *stream);

/* Clusters of active pixels and their binary masks ("a clustering algorithm to identify contiguous
 * energetic regions based on a tunable normalized threshold and minimum area. For each identified cluster, we
 * generated a binary mask applied to the complex CQT, which was subsequently inverted"; R19).  For plans
 * in the uniform-tile layout (tile_length != 0), where Q-plane `plane` is an image of R rows x M samples; call
 * qtam_threshold_rowmedian (the normalized threshold) first: a pixel is ACTIVE where its coefficient is non-zero.
 * qtam_cluster: connected components of the active pixels under 4-connectivity, time axis circular, frequency
 *   axis not; components of fewer than min_area pixels are dropped.  d_labels [batch][R*M] int32 (device, caller-
 *   owned): 0 = background / dropped, else 1 + the smallest pixel index (row*M + n) of the pixel's cluster;
 *   d_count [batch] int32: clusters kept.  qtam_plane_pixels(p, plane) = R*M (0 if the plane is no image).
 * qtam_mask: d_out [batch][coeffs_per_segment] = d_coef on the plane's pixels whose label equals `label` (label > 0)
 *   or is non-zero (label = 0), zero everywhere else, the other planes included; d_out may equal d_coef.
 *   qtam_inverse(d_out, plane) then gives the cluster's time series. */
int64_t     qtam_plane_pixels(const qtam_plan *p, int plane);
qtam_status qtam_cluster(qtam_plan *p, const void *d_coef, int batch, int plane, int min_area, int32_t *d_labels,
                         int32_t *d_count, void *stream);
qtam_status qtam_mask(qtam_plan *p, const void *d_coef, int batch, int plane, const int32_t *d_labels, int label,
                      void *d_out, void *stream);

/* Cluster labelling for callers that cannot allocate device memory.
 * Every call above needs a qtam_plan, and creating one calls cudaMalloc.  That rules the library out for a stage of a
 * running low-latency pipeline (a cudaMalloc or cudaFree there synchronises the device and holds up every stream), for
 * a plug-in of an application whose own pool already owns the free device memory, and for code that is only ever
 * lent its buffers.  This one entry point serves them: it takes no plan, and it calls neither cudaMalloc nor cudaFree
 * nor anything else that allocates, on the host or on the device.  The labels, the counts and the image are the
 * caller's; the single piece of scratch the method needs (a pixel counter per component root) is a fixed array that
 * is part of the library's device image: QTAM_CLUSTER_NOALLOC_MAX_PIXELS 32-bit counters = 4 MiB on every GPU on
 * which the process uses libqtam.so, held from the moment the CUDA runtime loads the library's kernels until exit.
 *   d_img: the image of segment 0, [rows][samples] complex of `dtype`, contiguous (for a plan in the uniform-tile
 *     layout: d_coef + the offset of the plane's first row, rows = the plane's rows, samples = M); segment b starts
 *     segment_stride complex elements after segment b - 1 (coeffs_per_segment for a plan's array, rows * samples for
 *     a bare stack of images).  Not modified.  A pixel is active where its coefficient is non-zero.
 *   d_labels [batch][rows * samples] int32, d_count [batch] int32, min_area >= 1: exactly as for qtam_cluster, and
 *     with the same values as qtam_cluster gives on the same image, bit for bit.
 * Limit: batch * rows * samples <= QTAM_CLUSTER_NOALLOC_MAX_PIXELS (and batch <= 65535).  Beyond it the call
 *   returns QTAM_ERR_TOO_LARGE, checked before anything touches the GPU; split the batch, or use qtam_cluster.
 * First call: the first call on each device (that device being current, as for every call here) asks the runtime
 *   where the array lives on that device and remembers the answer.  This is a host-side query that may make the
 *   runtime load the library's device code; do it once at start-up (a call with batch = 1 on a small image will do),
 *   before any stream capture begins.  Every later call on that device only enqueues kernels on `stream`.
 * Sharing: all calls on one GPU use the same array, from any thread or stream.  A call first clears the counters it
 *   is about to use, so what an earlier call left behind does no harm; but two calls whose kernels run at the same
 *   time on one GPU overwrite each other's counters and return wrong labels.  Keep the calls of a device on one
 *   stream, or order them with events. */
#define QTAM_CLUSTER_NOALLOC_MAX_PIXELS 1048576
qtam_status qtam_cluster_noalloc(qtam_dtype dtype, const void *d_img, int64_t segment_stride, int batch, int rows,
                                 int samples, int min_area, int32_t *d_labels, int32_t *d_count, void *stream);

/* Row-median threshold in place (BASELINE.json config 5; R11): per (segment,row),
 * m = median_n |Y_k[n]| (two middle values averaged), zero every Y_k[n] with |Y_k[n]| < kappa*m.
 * The decision is taken in the plan's dtype with the operation order of DESIGN.md.               */
qtam_status qtam_threshold_rowmedian(qtam_plan *p, void *d_coef, int batch, double kappa,
                                     void *stream);

/* Re-modulation with the carrier (Eq. 10a): d_out[b][offset_k + n] =
 * sqrt(M_k/N) e^{+2 pi i kc n/M_k} Y_k[n], which is the dense tile T_k at tau = n N/M_k (P2).
 * d_coef, d_out: [batch][coeffs_per_segment], same layout; d_out may equal d_coef (in place). */
qtam_status qtam_remodulate(qtam_plan *p, const void *d_coef, int batch, void *d_out, void *stream);

/* Instantaneous frequency of the demodulated tiles (Fig. 5 "the time-derivative of the unwrapped
 * phase"; R16): d_out[b][offset_k + n] = (kc + (M_k/2 pi) Arg(Y_k[(n+1) mod M_k] conj Y_k[n])) / T in Hz.
 * d_out: [batch][coeffs_per_segment] REAL of the plan's dtype (device, caller-owned); must not alias d_coef. */
qtam_status qtam_instantaneous_frequency(qtam_plan *p, const void *d_coef, int batch, void *d_out, void *stream);

/* Multi-Q scan selection ("for each resolution plane ... a signal quality metric (e.g., total
 * energy or peak pixel intensity)"; "optimal selection mode ... independently for each signal in the batch").
 * metric 0: sum over the plane's rows k and samples n of |Y_k[n]|^2; metric 1: max of |Y_k[n]|^2.
 * d_coef: [batch][coeffs_per_segment] as written by qtam_forward (not modified).
 * d_metric: [batch][n_planes] real of the plan's dtype (device, caller-owned, overwritten).
 * d_best: [batch] int32 (device) = the plane with the largest metric, lowest index on ties; may be NULL. */
typedef enum { QTAM_METRIC_ENERGY = 0, QTAM_METRIC_PEAK = 1 } qtam_metric;
qtam_status qtam_plane_metric(qtam_plan *p, const void *d_coef, int batch, int metric, void *d_metric,
                              int32_t *d_best, void *stream);

/* qtam_forward followed by qtam_threshold_rowmedian(kappa) on its output, with the same result bit for bit
 * (BASELINE.json config 5: "forward -> zero decimated coeffs with |c| below 3x row-median").  For float plans the
 * threshold runs in the epilogue of the row kernel while a row is still in registers (rows of at most 1024
 * points), so the coefficients are written once, already thresholded, and never re-read. */
qtam_status qtam_forward_threshold(qtam_plan *p, const void *d_x, int batch, double kappa, void *d_coef,
                                   void *stream);

/* Optimal-selection output ("a composite output tensor constructed from the optimal planes"):
 * d_out[b][0 .. C_q) = the coefficients of plane q = d_best[b] of segment b (its rows in layout order), zero up
 * to qtam_max_plane_coeffs(p), the row length of d_out ([batch][max plane size] complex, device, caller-owned).
 * d_best: [batch] int32 on the device, e.g. from qtam_plane_metric; out-of-range entries are clamped. */
int64_t     qtam_max_plane_coeffs(const qtam_plan *p);
qtam_status qtam_gather_plane(qtam_plan *p, const void *d_coef, int batch, const int32_t *d_best, void *d_out,
                              void *stream);

/* Number of kernel launches the last forward / inverse / threshold / dense call on this plan issued
 * (host counter, for bench.py's gpu_launches). */
int         qtam_last_launch_count(const qtam_plan *p);
const char *qtam_status_string(qtam_status s);

/* Launch profile for bench.py's roofline line.  While enabled, every kernel launch of the compute
 * calls is bracketed by CUDA events on the launch stream, and the library issues all of its launches on the
 * caller's stream (otherwise independent row kernels of one call run concurrently on the plan's own streams,
 * forked from and joined back to the caller's stream with events, and a kernel's elapsed time would include its
 * neighbours').  The events are pre-created: up to `max_launches` launches between two reads; further ones are
 * not recorded.  qtam_profile_read waits for the recorded events,
 * sums per kernel the launches, the device time (ms), the COMPULSORY bytes of those launches (algo_bytes:
 * input samples read, coefficients written or read, output samples written -- SURVEY.md 8(d)) and the bytes
 * the launches move by design (design_bytes: compulsory + spectrum, partial sums, band workspace, scratch;
 * DESIGN.md "Kernels"), writes up to `capacity` entries to `out` (host), clears the record and returns the
 * number of entries (-1 on error). */
typedef struct { char name[48]; int launches; double ms; double algo_bytes; double design_bytes; } qtam_kernel_stat;
qtam_status qtam_profile_enable(qtam_plan *p, int on, int max_launches);
int         qtam_profile_read(qtam_plan *p, qtam_kernel_stat *out, int capacity);

#ifdef __cplusplus
}
#endif
#endif
