// scan.cu -- multi-Q scan selection: per (segment, Q-plane) a quality metric of the plane's
// spectrogram |Y_k[n]|^2 (total energy or peak pixel) and, per segment, the plane that maximises it.
// The coefficients of a plane are contiguous in the ABI layout (rows are plane-major), so the metric is one
// streaming reduction per (plane, segment): one CTA each, 128-bit loads, per-thread partial results in the
// plan's dtype, then a fixed shuffle / shared-memory tree in double (same result on every run, no atomics).
#include <algorithm>

#include "cplx.cuh"
#include "device_plan.hpp"

namespace qtam {

template <typename T> struct Vec4;
template <> struct Vec4<float> { typedef float4 type; };
template <> struct Vec4<double> { typedef double4 type; };

template <typename T, int METRIC>
__global__ void __launch_bounds__(512)
k_plane_metric(const C2<T> *__restrict__ coef, long long ctot, const long long *__restrict__ plane_off, int nP,
               T *__restrict__ out) {
  typedef typename Vec4<T>::type V4;
  const int q = blockIdx.x, seg = blockIdx.y;
  const long long lo = plane_off[q], n = plane_off[q + 1] - lo;     // both multiples of 4 (every M >= 4)
  const V4 *src = reinterpret_cast<const V4 *>(coef + (size_t)seg * ctot + lo);
  T acc[4] = {0, 0, 0, 0};
  const long long n2 = n / 2;                                       // two coefficients per load
  for (long long i = threadIdx.x; i < n2; i += 4 * 512) {
#pragma unroll
    for (int u = 0; u < 4; ++u) {
      const long long k = i + (long long)u * 512;
      if (k < n2) {
        const V4 v = src[k];
        const T e0 = v.x * v.x + v.y * v.y, e1 = v.z * v.z + v.w * v.w;
        if (METRIC == 0) acc[u] += e0 + e1;
        else acc[u] = fmax(acc[u], fmax(e0, e1));
      }
    }
  }
  double r = METRIC == 0 ? ((double)acc[0] + (double)acc[1]) + ((double)acc[2] + (double)acc[3])
                         : fmax(fmax((double)acc[0], (double)acc[1]), fmax((double)acc[2], (double)acc[3]));
  for (int o = 16; o > 0; o >>= 1) {
    const double other = __shfl_xor_sync(0xffffffffu, r, o);
    r = METRIC == 0 ? r + other : fmax(r, other);
  }
  __shared__ double part[16];
  if ((threadIdx.x & 31) == 0) part[threadIdx.x >> 5] = r;
  __syncthreads();
  if (threadIdx.x < 32) {
    r = threadIdx.x < 16 ? part[threadIdx.x] : 0.0;
    for (int o = 8; o > 0; o >>= 1) {
      const double other = __shfl_xor_sync(0xffffffffu, r, o);
      r = METRIC == 0 ? r + other : fmax(r, other);
    }
    if (threadIdx.x == 0) out[(size_t)seg * nP + q] = (T)r;
  }
}

// optimal selection: the plane with the largest metric, lowest index on ties, independently per segment
template <typename T>
__global__ void k_best_plane(const T *__restrict__ metric, int nP, int batch, int32_t *__restrict__ best) {
  const int seg = blockIdx.x * blockDim.x + threadIdx.x;
  if (seg >= batch) return;
  const T *m = metric + (size_t)seg * nP;
  int b = 0;
  for (int q = 1; q < nP; ++q) if (m[q] > m[b]) b = q;
  best[seg] = b;
}

// Re-modulation (Eq. 10a :113-117): out = sqrt(M/N) e^{+2 pi i kc n/M} Y_k[n].  One CTA per (row, segment);
// the phase index kc n mod M is reduced in integers (R12) and goes through sincospi.
template <typename T>
__global__ void __launch_bounds__(128)
k_remodulate(const RowDev *__restrict__ rows, const C2<T> *__restrict__ coef, long long ctot, int n_samples,
             C2<T> *__restrict__ out) {
  const RowDev r = rows[blockIdx.x];
  const C2<T> *Y = coef + (size_t)blockIdx.y * ctot + r.offset;
  C2<T> *O = out + (size_t)blockIdx.y * ctot + r.offset;
  const T amp = sqrt((T)r.M / (T)n_samples);
  const T inv = (T)2 / (T)r.M;
  for (int n = threadIdx.x; n < r.M; n += 128) {
    const int m = (int)(((long long)r.kc * n) & (r.M - 1));
    T s, c;
    sincospi((T)m * inv, &s, &c);
    const C2<T> y = Y[n];
    O[n] = cmk<T>(amp * (y.x * c - y.y * s), amp * (y.x * s + y.y * c));
  }
}

// Instantaneous frequency (Fig. 5; R16): the circular forward difference of the
// unwrapped baseband phase, Arg(Y[n+1] conj Y[n]), scaled to Hz on the row's time grid, plus the carrier kc/T.
template <typename T>
__global__ void __launch_bounds__(128)
k_inst_freq(const RowDev *__restrict__ rows, const C2<T> *__restrict__ coef, long long ctot, T inv_duration,
            T *__restrict__ out) {
  const RowDev r = rows[blockIdx.x];
  const C2<T> *Y = coef + (size_t)blockIdx.y * ctot + r.offset;
  T *O = out + (size_t)blockIdx.y * ctot + r.offset;
  const T scale = (T)r.M * (T)0.15915494309189533577 * inv_duration;      // M / (2 pi T)
  const T carrier = (T)r.kc * inv_duration;
  for (int n = threadIdx.x; n < r.M; n += 128) {
    const C2<T> a = Y[n], c = Y[(n + 1) & (r.M - 1)];
    const T re = c.x * a.x + c.y * a.y, im = c.y * a.x - c.x * a.y;
    O[n] = carrier + scale * atan2(im, re);
  }
}

qtam_status instantaneous_frequency(qtam_plan *p, const void *d_coef, int batch, void *d_out, cudaStream_t st) {
  dim3 g((unsigned)p->hp.rows.size(), batch);
  const double inv_t = p->hp.fs / (double)p->hp.N;
  {
    LaunchScope ls(p, st, K_INST_FREQ, 3.0 * p->esz * (double)batch * (double)p->hp.ctot);
    if (p->esz == 4)
      k_inst_freq<float><<<g, 128, 0, st>>>(p->d_rows, static_cast<const float2 *>(d_coef), p->hp.ctot, (float)inv_t,
                                           static_cast<float *>(d_out));
    else
      k_inst_freq<double><<<g, 128, 0, st>>>(p->d_rows, static_cast<const double2 *>(d_coef), p->hp.ctot, inv_t,
                                            static_cast<double *>(d_out));
  }
  QTAM_LAUNCH_CHECK();
  return QTAM_OK;
}

qtam_status remodulate(qtam_plan *p, const void *d_coef, int batch, void *d_out, cudaStream_t st) {
  dim3 g((unsigned)p->hp.rows.size(), batch);
  {
    LaunchScope ls(p, st, K_REMODULATE, 4.0 * p->esz * (double)batch * (double)p->hp.ctot);
    if (p->esz == 4)
      k_remodulate<float><<<g, 128, 0, st>>>(p->d_rows, static_cast<const float2 *>(d_coef), p->hp.ctot, (int)p->hp.N,
                                            static_cast<float2 *>(d_out));
    else
      k_remodulate<double><<<g, 128, 0, st>>>(p->d_rows, static_cast<const double2 *>(d_coef), p->hp.ctot,
                                             (int)p->hp.N, static_cast<double2 *>(d_out));
  }
  QTAM_LAUNCH_CHECK();
  return QTAM_OK;
}

// the composite output of the optimal-selection mode (:329): plane best[seg] of every segment, copied to the
// start of out[seg][cmax] and zero padded (planes differ in size in the ragged layout).  16-byte copies.
template <typename T>
__global__ void __launch_bounds__(256)
k_gather_plane(const C2<T> *__restrict__ coef, long long ctot, const long long *__restrict__ plane_off, int nP,
               const int32_t *__restrict__ best, long long cmax, C2<T> *__restrict__ out) {
  typedef typename Vec4<T>::type V4;
  const int seg = blockIdx.y;
  int q = best[seg];
  q = q < 0 ? 0 : (q >= nP ? nP - 1 : q);
  const long long lo = plane_off[q], n2 = (plane_off[q + 1] - lo) / 2, c2 = cmax / 2;
  const V4 *src = reinterpret_cast<const V4 *>(coef + (size_t)seg * ctot + lo);
  V4 *dst = reinterpret_cast<V4 *>(out + (size_t)seg * cmax);
  V4 zero; zero.x = zero.y = zero.z = zero.w = 0;
  for (long long i = (long long)blockIdx.x * 256 + threadIdx.x; i < c2; i += (long long)gridDim.x * 256)
    dst[i] = i < n2 ? src[i] : zero;
}

qtam_status gather_plane(qtam_plan *p, const void *d_coef, int batch, const int32_t *d_best, void *d_out,
                         cudaStream_t st) {
  const long long cmax = p->max_plane_coeffs;
  dim3 g((unsigned)std::min<long long>((cmax / 2 + 255) / 256, 64), batch);
  {
    LaunchScope ls(p, st, K_GATHER_PLANE, 4.0 * p->esz * (double)batch * (double)cmax);
    if (p->esz == 4)
      k_gather_plane<float><<<g, 256, 0, st>>>(static_cast<const float2 *>(d_coef), p->hp.ctot, p->d_plane_off, p->hp.nP,
                                              d_best, cmax, static_cast<float2 *>(d_out));
    else
      k_gather_plane<double><<<g, 256, 0, st>>>(static_cast<const double2 *>(d_coef), p->hp.ctot, p->d_plane_off,
                                               p->hp.nP, d_best, cmax, static_cast<double2 *>(d_out));
  }
  QTAM_LAUNCH_CHECK();
  return QTAM_OK;
}

template <typename T>
static qtam_status metric_t(qtam_plan *p, const void *d_coef, int batch, int metric, void *d_metric,
                            int32_t *d_best, cudaStream_t st) {
  dim3 g(p->hp.nP, batch);
  {
    LaunchScope ls(p, st, K_PLANE_METRIC, (double)batch * (sizeof(C2<T>) * (double)p->hp.ctot));
    if (metric == 0)
      k_plane_metric<T, 0><<<g, 512, 0, st>>>(static_cast<const C2<T> *>(d_coef), p->hp.ctot, p->d_plane_off,
                                              p->hp.nP, static_cast<T *>(d_metric));
    else
      k_plane_metric<T, 1><<<g, 512, 0, st>>>(static_cast<const C2<T> *>(d_coef), p->hp.ctot, p->d_plane_off,
                                              p->hp.nP, static_cast<T *>(d_metric));
  }
  QTAM_LAUNCH_CHECK();
  if (d_best) {
    LaunchScope ls(p, st, K_BEST_PLANE, (double)batch * (sizeof(T) * (double)p->hp.nP + 4.0));
    k_best_plane<T><<<(batch + 127) / 128, 128, 0, st>>>(static_cast<const T *>(d_metric), p->hp.nP, batch, d_best);
  }
  QTAM_LAUNCH_CHECK();
  return QTAM_OK;
}

qtam_status plane_metric(qtam_plan *p, const void *d_coef, int batch, int metric, void *d_metric, int32_t *d_best,
                         cudaStream_t st) {
  return p->esz == 4 ? metric_t<float>(p, d_coef, batch, metric, d_metric, d_best, st)
                     : metric_t<double>(p, d_coef, batch, metric, d_metric, d_best, st);
}

}  // namespace qtam
