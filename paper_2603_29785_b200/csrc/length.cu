// length.cu -- the paper's output-length options (A22: PAPER.md:150, :158-160, :184, :343):
// every row of the time-frequency image at the same number n of time samples, n ANY integer >= the largest
// window -- "standard" n = N/2 + 1 (64 x 410, 62 x 12289), "minimal" n = ceil(N_t Delta f_max) + 1 = the largest
// 2 dk + 1 (64 x 33, 62 x 669), or user-set -- and the re-sampling between the plan's length and the standard one
// (:160 "up-sampling the compressed image back to the original size", Fig. 3).
//   forward   Y'_k[m] = (N n)^{-1/2} sum_j X[kc + j] W_k[j] e^{+2 pi i j m / n}        (C46 / C47 with N_out = n)
//   inverse   Bhat_k[j] = sqrt(N/n) sum_m Y'_k[m] e^{-2 pi i j m / n}, then Eq. 11     (C49 with N_out = n)
//   resample  Y''[m] = (n_in n_out)^{-1/2} sum_{|j| <= dk} (sum_l Y'[l] e^{-2 pi i j l / n_in}) e^{+2 pi i j m / n_out}
// n is no power of two in general (N/2 + 1 is often prime), so the short transforms are direct sums over the
// window's support -- O(n L) per row, exact phases from a table e^{2 pi i m / n} indexed by (j m) mod n kept in
// integers (R12), double-precision accumulation.  Outside the hot path: a layout converter, not a bench step.
#include <algorithm>
#include <cmath>
#include <vector>

#include "cplx.cuh"
#include "device_plan.hpp"

namespace qtam {

constexpr int kLenThreads = 256;

// band[j + dk] = X[kc + j] W_k[j], zero where kc + j leaves the one-sided spectrum (R8)
template <typename T>
__global__ void __launch_bounds__(kLenThreads)
k_len_band(const RowDev *__restrict__ rows, const C2<T> *__restrict__ spec, long long xstride, int nbins,
           const T *__restrict__ win, C2<T> *__restrict__ band, long long sumL) {
  const RowDev r = rows[blockIdx.x];
  const C2<T> *X = spec + (long long)blockIdx.y * xstride;
  C2<T> *B = band + (long long)blockIdx.y * sumL + r.woff;
  for (int i = threadIdx.x; i <= 2 * r.dk; i += kLenThreads) {
    const int f = r.kc + i - r.dk;
    B[i] = (f >= 0 && f < nbins) ? cscale(X[f], win[r.woff + i]) : cmk<T>(0, 0);
  }
}

// out[m] = scale * sum_{|j| <= dk} band[j + dk] e^{+2 pi i j m / n}, m = 0..n-1; tw[k] = e^{2 pi i k / n}
template <typename T>
__global__ void __launch_bounds__(kLenThreads)
k_len_synth(const RowDev *__restrict__ rows, const C2<T> *__restrict__ band, long long sumL,
            const C2<T> *__restrict__ tw, int n, T scale, C2<T> *__restrict__ out, int n_rows) {
  const RowDev r = rows[blockIdx.x];
  const C2<T> *B = band + (long long)blockIdx.y * sumL + r.woff;
  C2<T> *O = out + ((long long)blockIdx.y * n_rows + blockIdx.x) * n;
  const int L = 2 * r.dk + 1;
  const int j0 = ((-r.dk) % n + n) % n;                      // (-dk) mod n
  for (int m = blockIdx.z * kLenThreads + threadIdx.x; m < n; m += gridDim.z * kLenThreads) {
    int ph = (int)(((long long)j0 * m) % n);                 // (j m) mod n at j = -dk, then += m per step
    double ax = 0.0, ay = 0.0;
    for (int i = 0; i < L; ++i) {
      const C2<T> b = B[i], w = tw[ph];
      ax += (double)b.x * (double)w.x - (double)b.y * (double)w.y;
      ay += (double)b.x * (double)w.y + (double)b.y * (double)w.x;
      ph += m; if (ph >= n) ph -= n;
    }
    O[m] = cmk<T>((T)(ax * (double)scale), (T)(ay * (double)scale));
  }
}

// band[j + dk] = amp * w(j) * sum_m in[m] e^{-2 pi i j m / n}; w = W_k[j] (inverse) or 1 (re-sampling);
// zero where kc + j leaves the one-sided spectrum
template <typename T, bool WINDOW>
__global__ void __launch_bounds__(kLenThreads)
k_len_analysis(const RowDev *__restrict__ rows, const C2<T> *__restrict__ in, int n_rows, const C2<T> *__restrict__ tw,
               int n, T amp, const T *__restrict__ win, int nbins, int plane, C2<T> *__restrict__ band, long long sumL) {
  const RowDev r = rows[blockIdx.x];
  if (plane >= 0 && r.plane != plane) return;
  const C2<T> *Y = in + ((long long)blockIdx.y * n_rows + blockIdx.x) * n;
  C2<T> *B = band + (long long)blockIdx.y * sumL + r.woff;
  for (int i = blockIdx.z * kLenThreads + threadIdx.x; i <= 2 * r.dk; i += gridDim.z * kLenThreads) {
    const int j = i - r.dk, f = r.kc + j;
    const int step = (n - ((j % n + n) % n)) % n;            // (-j) mod n: the phase advances by it per sample
    int ph = 0;
    double ax = 0.0, ay = 0.0;
    for (int m = 0; m < n; ++m) {
      const C2<T> y = Y[m], w = tw[ph];
      ax += (double)y.x * (double)w.x - (double)y.y * (double)w.y;
      ay += (double)y.x * (double)w.y + (double)y.y * (double)w.x;
      ph += step; if (ph >= n) ph -= n;
    }
    double g = (double)amp;
    if (WINDOW) g = (f >= 0 && f < nbins) ? g * (double)win[r.woff + i] : 0.0;
    B[i] = cmk<T>((T)(ax * g), (T)(ay * g));
  }
}

static int ilog2(long long v) { int l = 0; while ((1LL << l) < v) ++l; return l; }

template <typename T> static bool upload_tw(void **dst, long long n, size_t *total) {
  std::vector<T> t((size_t)(2 * n));
  const long double tau = 6.283185307179586476925286766559005768L;
  for (long long k = 0; k < n; ++k) {
    const long double a = tau * (long double)k / (long double)n;
    t[(size_t)(2 * k)] = (T)cosl(a); t[(size_t)(2 * k + 1)] = (T)sinl(a);
  }
  if (cudaMalloc(dst, t.size() * sizeof(T)) != cudaSuccess) return false;
  *total += t.size() * sizeof(T);
  return cudaMemcpy(*dst, t.data(), t.size() * sizeof(T), cudaMemcpyHostToDevice) == cudaSuccess;
}

long long length_resolve(const HostPlan &hp, long long mode) {
  long long lmax = 0;
  for (const HostRow &h : hp.rows) lmax = std::max<long long>(lmax, h.L);
  if (mode == -1) return hp.N / 2 + 1;
  if (mode == -2) return lmax;
  return mode >= lmax ? mode : 0;      // 0: refused (a length below the largest window would alias)
}

qtam_status build_length(qtam_plan *p) {
  p->len_n = 0;
  const long long mode = p->hp.opt.out_length;
  if (mode == 0) return QTAM_OK;
  const long long n = length_resolve(p->hp, mode);
  if (n <= 0 || n >= (1LL << 30)) return QTAM_ERR_INVALID_ARG;
  p->len_n = n; p->len_std = p->hp.N / 2 + 1;
  const bool ok = p->esz == 4 ? upload_tw<float>(&p->d_len_tw[0], n, &p->device_bytes) &&
                                    upload_tw<float>(&p->d_len_tw[1], p->len_std, &p->device_bytes)
                              : upload_tw<double>(&p->d_len_tw[0], n, &p->device_bytes) &&
                                    upload_tw<double>(&p->d_len_tw[1], p->len_std, &p->device_bytes);
  return ok ? QTAM_OK : QTAM_ERR_ALLOC;
}

// z-blocks so that short batches still fill the machine
static unsigned zblocks(const qtam_plan *p, long long work_items, int batch) {
  const long long ctas = (long long)p->hp.rows.size() * batch;
  long long z = (4LL * p->num_sms + ctas - 1) / std::max<long long>(ctas, 1);
  const long long zmax = (work_items + kLenThreads - 1) / kLenThreads;
  z = std::max<long long>(1, std::min<long long>(std::min<long long>(z, zmax), 64));
  return (unsigned)z;
}

template <typename T>
static qtam_status forward_length_t(qtam_plan *p, int batch, void *d_out, cudaStream_t st) {
  const int K = (int)p->hp.rows.size();
  const int n = (int)p->len_n;
  dim3 g((unsigned)K, (unsigned)batch);
  {
    LaunchScope ls(p, st, K_LEN_BAND, 0.0, 2.0 * sizeof(C2<T>) * (double)batch * (double)p->hp.sumL);
    k_len_band<T><<<g, kLenThreads, 0, st>>>(p->d_rows, static_cast<const C2<T> *>(p->d_spec), p->xstride, (int)p->hp.nb,
                                            static_cast<const T *>(p->d_win), static_cast<C2<T> *>(p->d_band), p->hp.sumL);
  }
  QTAM_LAUNCH_CHECK();
  dim3 gs((unsigned)K, (unsigned)batch, zblocks(p, n, batch));
  {
    LaunchScope ls(p, st, K_LEN_SYNTH, sizeof(C2<T>) * (double)batch * (double)K * (double)n);
    k_len_synth<T><<<gs, kLenThreads, 0, st>>>(p->d_rows, static_cast<const C2<T> *>(p->d_band), p->hp.sumL,
                                              static_cast<const C2<T> *>(p->d_len_tw[0]), n,
                                              (T)(1.0 / std::sqrt((double)p->hp.N * (double)n)),
                                              static_cast<C2<T> *>(d_out), K);
  }
  QTAM_LAUNCH_CHECK();
  return QTAM_OK;
}

qtam_status length_forward(qtam_plan *p, int batch, void *d_out, cudaStream_t st) {
  return p->esz == 4 ? forward_length_t<float>(p, batch, d_out, st) : forward_length_t<double>(p, batch, d_out, st);
}

template <typename T>
static qtam_status analysis_t(qtam_plan *p, const void *d_in, int batch, int which, bool window, int plane, cudaStream_t st) {
  const int K = (int)p->hp.rows.size();
  const int n = (int)(which == 0 ? p->len_n : p->len_std);
  long long lmax = 0;
  for (const HostRow &h : p->hp.rows) lmax = std::max<long long>(lmax, h.L);
  dim3 g((unsigned)K, (unsigned)batch, zblocks(p, lmax, batch));
  const T amp = (T)std::sqrt((double)p->hp.N / (double)n);
  {
    LaunchScope ls(p, st, K_LEN_ANALYSIS, sizeof(C2<T>) * (double)batch * (double)K * (double)n);
    if (window)
      k_len_analysis<T, true><<<g, kLenThreads, 0, st>>>(p->d_rows, static_cast<const C2<T> *>(d_in), K,
          static_cast<const C2<T> *>(p->d_len_tw[which]), n, amp, static_cast<const T *>(p->d_win), (int)p->hp.nb, plane,
          static_cast<C2<T> *>(p->d_band), p->hp.sumL);
    else
      k_len_analysis<T, false><<<g, kLenThreads, 0, st>>>(p->d_rows, static_cast<const C2<T> *>(d_in), K,
          static_cast<const C2<T> *>(p->d_len_tw[which]), n, amp, static_cast<const T *>(p->d_win), (int)p->hp.nb, plane,
          static_cast<C2<T> *>(p->d_band), p->hp.sumL);
  }
  QTAM_LAUNCH_CHECK();
  return QTAM_OK;
}

// windowed band values of every row (of the plane) into the band workspace; the caller reduces them (Eq. 11)
qtam_status length_inverse_bands(qtam_plan *p, const void *d_in, int batch, int plane, cudaStream_t st) {
  return p->esz == 4 ? analysis_t<float>(p, d_in, batch, 0, true, plane, st)
                     : analysis_t<double>(p, d_in, batch, 0, true, plane, st);
}

template <typename T>
static qtam_status resample_t(qtam_plan *p, const void *d_in, int batch, int to_standard, void *d_out, cudaStream_t st) {
  const int K = (int)p->hp.rows.size();
  const int from = to_standard ? 0 : 1, to = 1 - from;
  qtam_status s = analysis_t<T>(p, d_in, batch, from, false, -1, st);      // band = sqrt(N/n_in) DFT of the row
  if (s != QTAM_OK) return s;
  const int n = (int)(to == 0 ? p->len_n : p->len_std);
  dim3 gs((unsigned)K, (unsigned)batch, zblocks(p, n, batch));
  {
    LaunchScope ls(p, st, K_LEN_SYNTH, sizeof(C2<T>) * (double)batch * (double)K * (double)n);
    k_len_synth<T><<<gs, kLenThreads, 0, st>>>(p->d_rows, static_cast<const C2<T> *>(p->d_band), p->hp.sumL,
                                              static_cast<const C2<T> *>(p->d_len_tw[to]), n,
                                              (T)(1.0 / std::sqrt((double)p->hp.N * (double)n)),
                                              static_cast<C2<T> *>(d_out), K);
  }
  QTAM_LAUNCH_CHECK();
  return QTAM_OK;
}

qtam_status length_resample(qtam_plan *p, const void *d_in, int batch, int to_standard, void *d_out, cudaStream_t st) {
  return p->esz == 4 ? resample_t<float>(p, d_in, batch, to_standard, d_out, st)
                     : resample_t<double>(p, d_in, batch, to_standard, d_out, st);
}

}  // namespace qtam
