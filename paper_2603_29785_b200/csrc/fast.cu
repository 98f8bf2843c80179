// fast.cu -- the tuned float path of libqtam for sm_100a.
//   K1 k_r2c_fast      a1      one CTA per segment: long real FFT in shared memory (ctafft.cuh), spectrum
//                              to the plan's L2-resident spectrum buffer (N = 2^12 .. 2^15)
//   K2 k_rows_fast<.,true>  a2+a3 [+a4]  one launch, one wave of CTAs, for every row with M <= 1024: window
//                              gather + baseband shift + short inverse FFT with the warp-level engine of
//                              rowfft.cuh (G = M/32 lanes per row, 32 points per lane in registers); one
//                              transform per set of identical rows (same centre bin and half-width), stored
//                              to every member; rows shorter than 32 points ride along, one thread each
//                              (tinyrow.cuh); THRESH: the row-median threshold in the epilogue (thrselect.cuh)
//   K3 k_rows_fast<.,false> a5 per-row forward FFT, sqrt(N/M), window; band values to the band workspace
//                              (plans whose inverse does not run in inv_tiled.cu)
//   K4 k_c2c_fast        a8    one CTA per segment: the half-length complex FFT behind the long C2R for plans
//                              whose spectrum comes out of k_combine_runs (N <= 2^15)
// Rows of 2^11 .. 2^13 points run in rows_cta.cu, 2^14 .. 2^17 in rows_cluster.cu, N = 2^16 .. 2^20 in
// long_fft.cu, double precision in generic.cu.
#include <type_traits>

#include "cplx.cuh"
#include "ctafft.cuh"
#include "device_plan.hpp"
#include "rowfft.cuh"
#include "thrselect.cuh"
#include "tinyrow.cuh"

namespace qtam {

extern __shared__ __align__(16) unsigned char qtam_fast_smem[];

// --------------------------------------------------------------------------------------------------
// K1: long R2C.  z[m] = x[2m] + i x[2m+1]; Z = FFT_Nc(z);
//     X[f] = (Z[f] + conj Z[Nc-f])/2 - (i/2) e^{-2 pi i f/N} (Z[f] - conj Z[Nc-f]),  f = 0..Nc  (C1)
// --------------------------------------------------------------------------------------------------
template <int LOG2NC>
__global__ void __launch_bounds__(CtaFftPlan<LOG2NC>::NT)
k_r2c_fast(const float *__restrict__ x, float2 *__restrict__ spec, long long xstride,
           const float2 *__restrict__ tw, int log2twn, const float2 *__restrict__ ptw) {
  constexpr int NC = 1 << LOG2NC, NT = CtaFftPlan<LOG2NC>::NT;
  float2 *s = reinterpret_cast<float2 *>(qtam_fast_smem);
  const float2 *gin = reinterpret_cast<const float2 *>(x) + (size_t)blockIdx.x * NC;
  cta_fft<LOG2NC, NT, -1, true, false>(s, gin, nullptr, ptw, 1.f);
  float2 *X = spec + (size_t)blockIdx.x * xstride;
  for (int f = threadIdx.x; f <= NC / 2; f += NT) {
    const int g = NC - f;
    const float2 A = s[f];
    const float2 B = (f == 0) ? A : s[g];
    const float2 E = make_float2(0.5f * (A.x + B.x), 0.5f * (A.y - B.y));
    const float2 D = make_float2(0.5f * (A.x - B.x), 0.5f * (A.y + B.y));
    float2 w = __ldg(tw + ((size_t)f << (log2twn - LOG2NC - 1)));   // e^{+2 pi i f/N}
    w.y = -w.y;
    const float2 t = make_float2(w.x * D.x - w.y * D.y, w.x * D.y + w.y * D.x);
    X[f] = make_float2(E.x + t.y, E.y - t.x);
    if (g != f) X[g] = make_float2(E.x - t.y, -E.y - t.x);
  }
}

// --------------------------------------------------------------------------------------------------
// Rows shorter than 32 points (M = 4, 8, 16): one thread per (segment, row), the whole row in registers.
// Forward: B[j] = X[kc + jj] W[jj] at j = jj mod M (R6; the spectrum's zero pads implement R8),
// Y = (N M)^{-1/2} IFFT_M(B) (C47).  Inverse: G[jj] = sqrt(N/M) FFT_M(Y)[jj mod M] W[jj] to the band
// workspace (C49).  For tiny rows FastRow::goff holds log2 M and FastRow::wpad the band offset.
// --------------------------------------------------------------------------------------------------
template <bool FORWARD, bool THRESH = false>
__device__ __forceinline__ void tiny_dispatch(long long id, const FastRow *__restrict__ tiny, int n_tiny,
                                              const float *__restrict__ fwin, const float2 *__restrict__ spec,
                                              long long xstride, int nbins, float2 *__restrict__ coef, long long ctot,
                                              float2 *__restrict__ band, long long sumL, int plane, float n_samples,
                                              float kappa = 0.f) {
  const int seg = (int)(id / n_tiny);
  const FastRow row = tiny[id - (long long)seg * n_tiny];
  if (!FORWARD && plane >= 0 && row.plane != plane) return;
  const float2 *X = spec + (size_t)seg * xstride;
  float2 *Y = coef + (size_t)seg * ctot + row.offset;
  float2 *Gb = band + (size_t)seg * sumL + row.wpad + row.dk;
  const float Mf = (float)(1 << row.goff);
  const float scale = FORWARD ? rsqrtf(n_samples * Mf) : sqrtf(n_samples / Mf);
  switch (row.goff) {
    case 2: tiny_row<4, FORWARD, THRESH>(row, X, fwin, Y, Gb, nbins, scale, kappa); break;
    case 3: tiny_row<8, FORWARD, THRESH>(row, X, fwin, Y, Gb, nbins, scale, kappa); break;
    case 4: tiny_row<16, FORWARD, THRESH>(row, X, fwin, Y, Gb, nbins, scale, kappa); break;
    default: break;
  }
}

template <bool FORWARD>
__global__ void __launch_bounds__(128)
k_tiny_rows(const FastRow *__restrict__ tiny, int n_tiny, const float *__restrict__ fwin,
            const float2 *__restrict__ spec, long long xstride, int nbins, float2 *__restrict__ coef,
            long long ctot, float2 *__restrict__ band, long long sumL, int batch, int plane, float n_samples) {
  const long long id = (long long)blockIdx.x * 128 + threadIdx.x;
  if (id >= (long long)n_tiny * batch) return;
  tiny_dispatch<FORWARD>(id, tiny, n_tiny, fwin, spec, xstride, nbins, coef, ctot, band, sumL, plane, n_samples);
}

// --------------------------------------------------------------------------------------------------
// K2 / K3: rows.  Work items are ordered bucket-major (largest M first), then segment, then row group;
// a CTA takes NWARPS consecutive items, i.e. neighbouring rows of one segment, so that the bands its
// warps read overlap in L1.
// --------------------------------------------------------------------------------------------------
template <int LOG2G, bool THRESH = false>
__device__ __forceinline__ void fwd_group(const FastBucket &B, const FastRow *__restrict__ frows, int seg, int grp,
                                       int lane, float2 *ex, const float2 *tw1,
                                       const float2 *__restrict__ spec, long long xstride,
                                       const float *__restrict__ fwinp, float2 *__restrict__ coef,
                                       long long ctot, const int *__restrict__ fmem, float kappa = 0.f) {
  constexpr int G = 1 << LOG2G, F = 32 / G, M = 32 * G;
  const int t = lane & (G - 1), rw = lane >> LOG2G;
  const int r = grp * F + rw;
  const bool valid = r < B.nrows;
  // lanes past the end of the bucket recompute its first row and simply do not store
  const FastRow row = frows[B.row_base + (valid ? r : 0)];
  // B_k[j] = X[kc + jj(j)] * Wpad[j]: the window table is zero outside the support and the spectrum
  // buffer has zero pads, so neither the support (A9) nor the clipping at DC / Nyquist (R8) needs a test
  const float2 *X = spec + (size_t)seg * xstride + row.kc + t;
  const float *W = fwinp + row.wpad + t;
  // ... and outside the support nothing is loaded at all: one compare per element saves the two loads
  // of the 40-50 % of the M-array that the window leaves empty
  const int hi = row.dk - t, lo = -row.dk - t;
  float2 v[32];
#pragma unroll
  for (int j1 = 0; j1 < 32; ++j1) {
    const int jj = (j1 < 16) ? (G * j1) : (G * j1 - M);     // signed offset from the centre (R6), minus t
    v[j1] = make_float2(0.f, 0.f);
    if ((j1 < 16) ? (jj <= hi) : (jj >= lo)) {
      const float2 xv = X[jj];
      const float w = W[G * j1];
      v[j1] = make_float2(xv.x * w, xv.y * w);
    }
  }
  // the first member's offset is fetched before the transform, every further one an iteration ahead
  int moff = __ldg(fmem + row.pad);
  RowFFT<LOG2G, +1>::run(v, ex, tw1, lane);
  if constexpr (THRESH) {
    // a4 fused into the epilogue: the row is in the registers of its G lanes; same decisions, bit for bit,
    // as qtam_threshold_rowmedian on the stored coefficients (thrselect.cuh)
    unsigned x[32], vor = 0u, vand = ~0u;
#pragma unroll
    for (int e = 0; e < 32; ++e) {
      x[e] = Bits<float>::of(Bits<float>::add(Bits<float>::mul(v[e].x, v[e].x), Bits<float>::mul(v[e].y, v[e].y)));
      vor |= x[e]; vand &= x[e];
    }
    unsigned prefix;
    const unsigned cut = thr_select<float, 32>(x, vor, vand, G, kappa, prefix);
#pragma unroll
    for (int e = 0; e < 32; ++e) if ((x[e] ^ prefix) < cut) v[e] = make_float2(0.f, 0.f);
  }
  if (valid) {
    // every member of the leader's set (rows with this centre bin and half-width) gets the same values
#pragma unroll 1
    for (int m = 0; m < row.plane; ++m) {
      float2 *dst = coef + (size_t)seg * ctot + moff + t;
      if (m + 1 < row.plane) moff = __ldg(fmem + row.pad + m + 1);
#pragma unroll
      for (int i = 0; i < F; ++i)
#pragma unroll
        for (int n2 = 0; n2 < G; ++n2) __stcs(dst + G * i + 32 * n2, v[i * G + n2]);
    }
  }
}

template <int LOG2G>
__device__ __forceinline__ void inv_group(const FastBucket &B, const FastRow *__restrict__ frows, int seg, int grp,
                                          int lane, float2 *ex, const float2 *tw1,
                                          const float2 *__restrict__ coef, long long ctot, int nbins,
                                          const float *__restrict__ fwin, float2 *__restrict__ band,
                                          long long sumL, int plane) {
  constexpr int G = 1 << LOG2G, F = 32 / G, M = 32 * G;
  const int t = lane & (G - 1), rw = lane >> LOG2G;
  const int r = grp * F + rw;
  FastRow row;
  bool valid = r < B.nrows;
  if (valid) row = frows[B.row_base + r];
  else { row.kc = 0; row.dk = -1; row.woff = 0; row.goff = 0; row.offset = 0; row.plane = -1; }
  if (plane >= 0 && row.plane != plane) valid = false;
  // a whole warp whose rows are all skipped can leave (uniform decision)
  if (__ballot_sync(0xffffffffu, valid) == 0u) return;
  const float2 *Y = coef + (size_t)seg * ctot + row.offset + t;
  float2 v[32];
#pragma unroll
  for (int j1 = 0; j1 < 32; ++j1) v[j1] = valid ? __ldcs(Y + G * j1) : make_float2(0.f, 0.f);
  RowFFT<LOG2G, -1>::run(v, ex, tw1, lane);
  if (valid) {
    float2 *Gb = band + (size_t)seg * sumL + row.goff + row.dk;
    const float *W = fwin + row.woff + row.dk;
#pragma unroll
    for (int i = 0; i < F; ++i)
#pragma unroll
      for (int n2 = 0; n2 < G; ++n2) {
        const int j = (t + G * i) + 32 * n2;
        const int jj = (G == 1) ? (j < 16 ? j : j - M) : (n2 < G / 2 ? j : j - M);
        const int f = row.kc + jj;
        if (jj <= row.dk && jj >= -row.dk && f >= 0 && f < nbins) Gb[jj] = pscale(v[i * G + n2], W[jj]);
      }
  }
}

template <int NWARPS, bool FORWARD, bool THRESH = false>
__global__ void __launch_bounds__(NWARPS * 32, NWARPS <= 8 ? 2 : 1)
k_rows_fast(FastParams P, const FastRow *frows, const void *__restrict__ tw1g_,
            const float *__restrict__ fwin, const float *__restrict__ fwinp,
            const float2 *__restrict__ spec, long long xstride, int nbins,
            float2 *__restrict__ coef, long long ctot, float2 *__restrict__ band, long long sumL,
            int batch, int plane, const FastRow *__restrict__ tiny, int n_tiny, float n_samples,
            const int *__restrict__ fmem, float kappa) {
  typedef float2 TW;
  const TW *tw1g = static_cast<const TW *>(tw1g_);
  TW *tw1s = reinterpret_cast<TW *>(qtam_fast_smem);
  float2 *exall = reinterpret_cast<float2 *>(qtam_fast_smem + sizeof(float2) * (size_t)((P.tw_total + 1) & ~1));
  for (int i = threadIdx.x; i < P.tw_total; i += NWARPS * 32) tw1s[i] = tw1g[i];
  // the row table too, when it fits (P.rows_smem): a row's record is then one shared-memory read away
  // instead of a global load the gather addresses have to wait for
  if (P.rows_smem) {
    int4 *dst = reinterpret_cast<int4 *>(exall + NWARPS * kExPerWarp);
    const int4 *src = reinterpret_cast<const int4 *>(frows);
    for (int i = threadIdx.x; i < 2 * P.rows_smem; i += NWARPS * 32) dst[i] = src[i];
    frows = reinterpret_cast<const FastRow *>(dst);
  }
  __syncthreads();
  // rows shorter than 32 points ride along, one thread per (segment, row) (n_tiny = 0: separate launch)
  if constexpr (FORWARD) {
    for (long long id = (long long)blockIdx.x * (NWARPS * 32) + threadIdx.x; id < (long long)n_tiny * batch;
         id += (long long)gridDim.x * (NWARPS * 32))
      tiny_dispatch<true, THRESH>(id, tiny, n_tiny, fwin, spec, xstride, nbins, coef, ctot, band, sumL, -1, n_samples, kappa);
  }
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  float2 *ex = exall + warp * kExPerWarp;
  // (the host keeps groups_per_seg * batch below 2^31)
  const unsigned total = (unsigned)P.groups_per_seg * (unsigned)batch;
  for (unsigned item = blockIdx.x * NWARPS + warp; item < total; item += gridDim.x * NWARPS) {
    // decode: buckets in order, each spanning ngroups*batch items
    int q = 0;
    unsigned rem = item;
    while (q + 1 < P.nbuckets && rem >= (unsigned)P.b[q].ngroups * (unsigned)batch) {
      rem -= (unsigned)P.b[q].ngroups * (unsigned)batch;
      ++q;
    }
    const FastBucket B = P.b[q];
    const int seg = (int)(rem / (unsigned)B.ngroups);
    const int grp = (int)(rem - (unsigned)seg * (unsigned)B.ngroups);
    const TW *tw1 = tw1s + B.tw_base;
#define QTAM_ROW_CASE(L)                                                                              \
  case L:                                                                                             \
    if constexpr (FORWARD) fwd_group<L, THRESH>(B, frows, seg, grp, lane, ex, tw1, spec, xstride, fwinp, coef, ctot, fmem, kappa); \
    else inv_group<L>(B, frows, seg, grp, lane, ex, tw1, coef, ctot, nbins, fwin, band, sumL, plane);  \
    break;
    switch (B.log2G) {
      QTAM_ROW_CASE(5) QTAM_ROW_CASE(4) QTAM_ROW_CASE(3) QTAM_ROW_CASE(2) QTAM_ROW_CASE(1) QTAM_ROW_CASE(0)
      default: break;
    }
#undef QTAM_ROW_CASE
  }
}

// --------------------------------------------------------------------------------------------------
// K4: the half-length complex FFT of the long C2R (row a8) for N <= 2^15, one CTA per segment: Z (already
//     pre-processed by k_combine_runs) from the spectrum buffer straight to x_out
// --------------------------------------------------------------------------------------------------
template <int LOG2NC>
__global__ void __launch_bounds__(CtaFftPlan<LOG2NC>::NT)
k_c2c_fast(const float2 *__restrict__ spec, long long xstride, const float2 *__restrict__ ptw, float *__restrict__ x_out) {
  constexpr int NC = 1 << LOG2NC, NT = CtaFftPlan<LOG2NC>::NT;
  float2 *s = reinterpret_cast<float2 *>(qtam_fast_smem);
  cta_fft<LOG2NC, NT, +1, true, true>(s, spec + (size_t)blockIdx.x * xstride,
                                      reinterpret_cast<float2 *>(x_out) + (size_t)blockIdx.x * NC, ptw, 1.f);
}

// --------------------------------------------------------------------------------------------------
// host side
// --------------------------------------------------------------------------------------------------
static int ilog2(long long v) { int l = 0; while ((1LL << l) < v) ++l; return l; }

constexpr int kRowWarps = 8;   // warps per CTA of k_rows_fast (two CTAs per SM)

template <int LOG2NC> static qtam_status r2c_launch(qtam_plan *p, const void *d_x, int batch, cudaStream_t st) {
  const size_t smem = p->cfg_r2c.smem;
  {
    LaunchScope ls(p, st, K_R2C_FAST, (double)batch * 4.0 * (double)p->hp.N,
                   (double)batch * (4.0 * (double)p->hp.N + 8.0 * (double)p->hp.nb));
    k_r2c_fast<LOG2NC><<<batch, CtaFftPlan<LOG2NC>::NT, smem, st>>>(
        static_cast<const float *>(d_x), static_cast<float2 *>(p->d_spec), p->xstride,
        static_cast<const float2 *>(p->d_tw), ilog2(p->twn), static_cast<const float2 *>(p->d_ptw));
  }
  QTAM_LAUNCH_CHECK();
  return QTAM_OK;
}

// pass tables of the long FFT (ctafft.cuh); every kernel that runs the long transform of 2^LOG2NC points
// uses radices equal to those of CtaFftPlan<LOG2NC>::NT (static_asserts at the kernels)
qtam_status build_long_tables(qtam_plan *p) {
  std::vector<float> t;
  switch (ilog2(p->hp.N) - 1) {
    case 11: fill_cta_fft_tables<11, CtaFftPlan<11>::NT>(t); break;
    case 12: fill_cta_fft_tables<12, CtaFftPlan<12>::NT>(t); break;
    case 13: fill_cta_fft_tables<13, CtaFftPlan<13>::NT>(t); break;
    case 14: fill_cta_fft_tables<14, CtaFftPlan<14>::NT>(t); break;
    default: return QTAM_OK;
  }
  if (cudaMalloc(&p->d_ptw, t.size() * sizeof(float)) != cudaSuccess) return QTAM_ERR_ALLOC;
  p->device_bytes += t.size() * sizeof(float);
  if (cudaMemcpy(p->d_ptw, t.data(), t.size() * sizeof(float), cudaMemcpyHostToDevice) != cudaSuccess)
    return QTAM_ERR_CUDA;
  return QTAM_OK;
}

qtam_status fast_r2c(qtam_plan *p, const void *d_x, int batch, cudaStream_t st) {
  switch (ilog2(p->hp.N) - 1) {
    case 11: return r2c_launch<11>(p, d_x, batch, st);
    case 12: return r2c_launch<12>(p, d_x, batch, st);
    case 13: return r2c_launch<13>(p, d_x, batch, st);
    case 14: return r2c_launch<14>(p, d_x, batch, st);
    default: return QTAM_ERR_UNSUPPORTED;
  }
}

template <int NW, bool FORWARD, bool THRESH = false>
static qtam_status rows_launch_nw(qtam_plan *p, int batch, const void *d_coef_in, void *d_coef_out, int plane,
                                  cudaStream_t st, bool *tiny_rode, float kappa = 0.f) {
  const FastParams &P = FORWARD ? p->fast_fwd : p->fast;
  if (tiny_rode) *tiny_rode = false;
  if (P.groups_per_seg == 0) return QTAM_OK;
  const KernelCfg &cfg = FORWARD ? (THRESH ? p->cfg_rows_thr : p->cfg_rows_fwd) : p->cfg_rows_inv;
  if (!cfg.ready) return QTAM_ERR_CUDA;
  const size_t smem = cfg.smem;
  if ((long long)P.groups_per_seg * batch >= (1LL << 31)) return QTAM_ERR_UNSUPPORTED;
  auto kern = k_rows_fast<NW, FORWARD, THRESH>;
  const long long total = (long long)P.groups_per_seg * batch;
  long long want = (total + NW - 1) / NW;
  const long long resident = (long long)p->num_sms * cfg.occ;
  // one wave of resident CTAs, each looping over its items
  int grid = (int)(want < resident ? want : resident);
  if (grid < 1) grid = 1;
  // the forward launch also takes the rows shorter than 32 points, one thread per (segment, row)
  const bool ride = FORWARD && p->n_tiny > 0;    // grid-stride loop in the kernel: any count rides
  // compulsory: the coefficients written (forward) or read (inverse); by design also the spectrum / the bands
  const double bytes = (double)batch * 8.0 * (P.sum_M + (ride ? p->tiny_sumM : 0.0));
  const double design = bytes + (double)batch * 8.0 * (FORWARD ? (double)p->hp.nb : P.sum_L);
  {
    LaunchScope ls(p, st, FORWARD ? (THRESH ? K_FWD_ROWS_THR : K_FWD_ROWS_FAST) : K_INV_ROWS_FAST, bytes, design);
    kern<<<grid, NW * 32, smem, st>>>(
        P, FORWARD ? p->d_frows_fwd : p->d_frows, static_cast<const void *>(FORWARD ? p->d_ftw_fwd : p->d_ftw_inv),
        static_cast<const float *>(p->d_fwin), static_cast<const float *>(p->d_fwinp),
        static_cast<const float2 *>(p->d_spec), p->xstride,
        (int)p->hp.nb,
        FORWARD ? static_cast<float2 *>(d_coef_out) : const_cast<float2 *>(static_cast<const float2 *>(d_coef_in)),
        p->hp.ctot, static_cast<float2 *>(p->d_band), p->hp.sumL, batch, plane, p->d_tiny, ride ? p->n_tiny : 0,
        (float)p->hp.N, p->d_fmem, kappa);
  }
  QTAM_LAUNCH_CHECK();
  if (tiny_rode) *tiny_rode = ride;
  return QTAM_OK;
}

template <bool FORWARD>
static qtam_status rows_launch(qtam_plan *p, int batch, const void *d_coef_in, void *d_coef_out, int plane,
                               cudaStream_t st, bool *tiny_rode) {
  return rows_launch_nw<kRowWarps, FORWARD>(p, batch, d_coef_in, d_coef_out, plane, st, tiny_rode);
}

template <bool FORWARD>
static qtam_status tiny_launch(qtam_plan *p, int batch, const void *d_coef, int plane, cudaStream_t st) {
  if (p->n_tiny == 0) return QTAM_OK;
  const long long total = (long long)p->n_tiny * batch;
  {
    LaunchScope ls(p, st, FORWARD ? K_TINY_FWD : K_TINY_INV, (double)batch * 8.0 * p->tiny_sumM,
                   (double)batch * 8.0 * (p->tiny_sumM + p->tiny_sumL));
    k_tiny_rows<FORWARD><<<(unsigned)((total + 127) / 128), 128, 0, st>>>(
        p->d_tiny, p->n_tiny, static_cast<const float *>(p->d_fwin), static_cast<const float2 *>(p->d_spec),
        p->xstride, (int)p->hp.nb, const_cast<float2 *>(static_cast<const float2 *>(d_coef)), p->hp.ctot,
        static_cast<float2 *>(p->d_band), p->hp.sumL, batch, plane, (float)p->hp.N);
  }
  QTAM_LAUNCH_CHECK();
  return QTAM_OK;
}

qtam_status fast_forward_rows(qtam_plan *p, int batch, void *d_coef, cudaStream_t st) {
  bool rode = false;
  const qtam_status s = rows_launch<true>(p, batch, nullptr, d_coef, -1, st, &rode);
  if (s != QTAM_OK || rode) return s;
  return tiny_launch<true>(p, batch, d_coef, -1, st);
}

// a2 + a3 + a4 in one launch for every row of at most 1024 points; `*done` = false when the plan's rows
// shorter than 32 points could not ride along (the caller then runs forward and threshold separately)
qtam_status fast_forward_rows_threshold(qtam_plan *p, int batch, void *d_coef, float kappa, cudaStream_t st,
                                        bool *done) {
  *done = false;
  const FastParams &P = p->fast_fwd;
  if (P.groups_per_seg == 0) return QTAM_OK;
  bool rode = false;
  const qtam_status s = rows_launch_nw<kRowWarps, true, true>(p, batch, nullptr, d_coef, -1, st, &rode, kappa);
  if (s != QTAM_OK) return s;
  if (p->n_tiny > 0 && !rode) return QTAM_ERR_UNSUPPORTED;   // cannot happen given the test above
  *done = true;
  return QTAM_OK;
}

// rows of 32 .. 1024 points to the band workspace (plans whose rows have no tiles)
qtam_status fast_inverse_rows(qtam_plan *p, const void *d_coef, int batch, int plane, cudaStream_t st) {
  return rows_launch<false>(p, batch, d_coef, nullptr, plane, st, nullptr);
}
// rows shorter than 32 points to the band workspace
qtam_status fast_tiny_inverse(qtam_plan *p, const void *d_coef, int batch, int plane, cudaStream_t st) {
  return tiny_launch<false>(p, batch, d_coef, plane, st);
}

template <int LOG2NC>
static qtam_status c2c_launch(qtam_plan *p, int batch, void *d_x_out, cudaStream_t st) {
  {
    LaunchScope ls(p, st, K_C2C_FAST, (double)batch * 4.0 * (double)p->hp.N, (double)batch * 8.0 * (double)p->hp.N);
    k_c2c_fast<LOG2NC><<<batch, CtaFftPlan<LOG2NC>::NT, p->cfg_c2c.smem, st>>>(
        static_cast<const float2 *>(p->d_spec), p->xstride, static_cast<const float2 *>(p->d_ptw),
        static_cast<float *>(d_x_out));
  }
  QTAM_LAUNCH_CHECK();
  return QTAM_OK;
}

// launch configurations of this file's kernels, fixed at plan creation
template <int LOG2NC> static bool prepare_long(qtam_plan *p) {
  const size_t smem = sizeof(float2) * (size_t)cta_fft_smem_elems<LOG2NC>();
  return kernel_prepare(p->cfg_r2c, k_r2c_fast<LOG2NC>, CtaFftPlan<LOG2NC>::NT, smem) &&
         kernel_prepare(p->cfg_c2c, k_c2c_fast<LOG2NC>, CtaFftPlan<LOG2NC>::NT, smem);
}

qtam_status prepare_fast(qtam_plan *p) {
  if (p->fast_long) {
    bool ok = false;
    switch (ilog2(p->hp.N) - 1) {
      case 11: ok = prepare_long<11>(p); break;
      case 12: ok = prepare_long<12>(p); break;
      case 13: ok = prepare_long<13>(p); break;
      case 14: ok = prepare_long<14>(p); break;
      default: break;
    }
    if (!ok) return QTAM_ERR_CUDA;
  }
  if (p->fast_rows) {
    auto smem_of = [](const FastParams &P) {
      return sizeof(float2) * (size_t)((P.tw_total + 1) & ~1) + sizeof(float2) * (size_t)kRowWarps * kExPerWarp +
             sizeof(FastRow) * (size_t)P.rows_smem;
    };
    if (!kernel_prepare(p->cfg_rows_fwd, k_rows_fast<kRowWarps, true, false>, kRowWarps * 32, smem_of(p->fast_fwd)) ||
        !kernel_prepare(p->cfg_rows_thr, k_rows_fast<kRowWarps, true, true>, kRowWarps * 32, smem_of(p->fast_fwd)) ||
        !kernel_prepare(p->cfg_rows_inv, k_rows_fast<kRowWarps, false, false>, kRowWarps * 32, smem_of(p->fast)))
      return QTAM_ERR_CUDA;
  }
  return QTAM_OK;
}

qtam_status fast_c2c_out(qtam_plan *p, int batch, void *d_x_out, cudaStream_t st) {
  switch (ilog2(p->hp.N) - 1) {
    case 11: return c2c_launch<11>(p, batch, d_x_out, st);
    case 12: return c2c_launch<12>(p, batch, d_x_out, st);
    case 13: return c2c_launch<13>(p, batch, d_x_out, st);
    case 14: return c2c_launch<14>(p, batch, d_x_out, st);
    default: return QTAM_ERR_UNSUPPORTED;
  }
}

}  // namespace qtam
