// qtam_ref.cpp -- CPU ORACLE (test infrastructure, see qtam_ref.h).  Plain, slow, written from
// PAPER.md; no blocking, fusion or reordering beyond what each cited formula states.  Shares no
// code with the CUDA library.
#include "qtam_ref.h"

#include <algorithm>
#include <cmath>
#include <complex>
#include <cstring>
#include <new>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef long double ld;
typedef std::complex<double> cd;
typedef std::complex<long double> cld;

namespace {

const ld TWO_PI_L = 6.283185307179586476925286766559005768L;

// e^{2 pi i a/b}; the phase index is reduced mod b in 64-bit integers first (reading R12).
inline cld cis(int64_t a, int64_t b) {
  int64_t r = a % b;
  if (r < 0) r += b;
  // exact values on the axes so that textbook special cases (b = 1, 2, 4) are exact
  if (r == 0) return cld(1, 0);
  if (4 * r == b) return cld(0, 1);
  if (2 * r == b) return cld(-1, 0);
  if (4 * r == 3 * b) return cld(0, -1);
  ld ang = TWO_PI_L * (ld)r / (ld)b;
  return cld(cosl(ang), sinl(ang));
}

struct Row {
  int plane, row;
  double q, f_request, f_center;
  int64_t kc, dk, L, M, offset;
  double norm;                 // 1/sqrt(sum_j W'^2)
  std::vector<double> wraw;    // W'_k[j], j=-dk..dk   (Eq. 6 / A1)
  std::vector<double> w;       // W_k[j] = W'_k[j]*norm (Eq. 5 as read in R3)
};

}  // namespace

struct qtam_ref_plan {
  double epsilon = 0.0;   // Eq. 12: unnormalised stop-band value of the dense windows
  double fs;
  int64_t N, nb;   // nb = N/2+1 one-sided bins
  int nP, nR;      // planes, rows per plane
  std::vector<double> Q;
  std::vector<Row> rows;
  int64_t ctot, sumL;
  // index 0 = joint frame, 1+p = plane p
  std::vector<std::vector<double>> P;
  std::vector<std::vector<uint8_t>> cover;
};

namespace {

int64_t next_pow2(int64_t v) {
  int64_t m = 1;
  while (m < v) m <<= 1;
  return m;
}
bool is_pow2(int64_t v) { return v > 0 && (v & (v - 1)) == 0; }
bool is_fft_length(int64_t v) { return is_pow2(v) || (v % 3 == 0 && is_pow2(v / 3)); }   // 2^a or 3 * 2^a

// ---- DFT engines ------------------------------------------------------------------------------

// naive: out[k] = sum_j in[j] e^{sign 2 pi i jk/n}   (C1 / C2 kernels)
void dft_naive(const cd *in, cd *out, int64_t n, int sign) {
  std::vector<cld> tw((size_t)n);
  for (int64_t m = 0; m < n; ++m) tw[(size_t)m] = cis(sign * m, n);
  for (int64_t k = 0; k < n; ++k) {
    cld acc(0, 0);
    for (int64_t j = 0; j < n; ++j) acc += cld(in[j]) * tw[(size_t)((j * k) % n)];
    out[k] = cd((double)acc.real(), (double)acc.imag());
  }
}

// textbook recursive decimation in time, radix 2 while the length is even and radix 3 for a remaining factor 3
// (segment lengths N = 3 * 2^k: the paper's own benchmark shape is 6 s at 4096 Hz = 24576 samples, PAPER.md:178,
// :339); tw[m] = e^{sign 2 pi i m/ntop}, m = 0 .. ntop-1
void fft_rec(cd *a, cd *tmp, int64_t n, const cd *tw, int64_t tw_step, int64_t ntop) {
  if (n == 1) return;
  if (n % 2 == 0) {
    int64_t h = n / 2;
    for (int64_t i = 0; i < h; ++i) {
      tmp[i] = a[2 * i];
      tmp[h + i] = a[2 * i + 1];
    }
    std::memcpy(a, tmp, sizeof(cd) * (size_t)n);
    fft_rec(a, tmp, h, tw, tw_step * 2, ntop);
    fft_rec(a + h, tmp, h, tw, tw_step * 2, ntop);
    for (int64_t k = 0; k < h; ++k) {
      cd e = a[k], o = a[h + k] * tw[(size_t)(k * tw_step)];
      a[k] = e + o;
      a[h + k] = e - o;
    }
  } else {
    // n = 3 h: X[k + m h] = F0[k] + w_n^{k + m h} F1[k] + w_n^{2 (k + m h)} F2[k], F_r = DFT_h of a[3 i + r]
    int64_t h = n / 3;
    for (int64_t i = 0; i < h; ++i) {
      tmp[i] = a[3 * i];
      tmp[h + i] = a[3 * i + 1];
      tmp[2 * h + i] = a[3 * i + 2];
    }
    std::memcpy(a, tmp, sizeof(cd) * (size_t)n);
    for (int r = 0; r < 3; ++r) fft_rec(a + r * h, tmp, h, tw, tw_step * 3, ntop);
    for (int64_t k = 0; k < h; ++k) {
      const cd f0 = a[k], f1 = a[h + k], f2 = a[2 * h + k];
      for (int64_t m = 0; m < 3; ++m) {
        const int64_t e1 = ((k + m * h) * tw_step) % ntop, e2 = (2 * (k + m * h) * tw_step) % ntop;
        tmp[k + m * h] = f0 + f1 * tw[(size_t)e1] + f2 * tw[(size_t)e2];
      }
    }
    std::memcpy(a, tmp, sizeof(cd) * (size_t)n);
  }
}

// n = 2^a or 3 * 2^a
void fft_radix2(const cd *in, cd *out, int64_t n, int sign) {
  std::vector<cd> tw((size_t)std::max<int64_t>(n, 1)), tmp((size_t)n);
  for (int64_t m = 0; m < n; ++m) {
    cld c = cis(sign * m, n);
    tw[(size_t)m] = cd((double)c.real(), (double)c.imag());
  }
  if (out != in) std::memcpy(out, in, sizeof(cd) * (size_t)n);
  fft_rec(out, tmp.data(), n, tw.data(), 1, n);
}

// One-sided spectrum X[f] = sum_n x[n] e^{-2 pi i fn/N}, f = 0..N/2 (C1).
// `need` (may be null) marks the bins the caller uses; engine 0 skips the others (leaves 0).
void spectrum_onesided(const double *x, int64_t N, cd *X, const uint8_t *need, int engine) {
  int64_t nb = N / 2 + 1;
  if (engine == 0) {
    std::vector<cld> tw((size_t)N);
    for (int64_t m = 0; m < N; ++m) tw[(size_t)m] = cis(-m, N);
    for (int64_t f = 0; f < nb; ++f) {
      if (need && !need[f]) { X[f] = cd(0, 0); continue; }
      cld acc(0, 0);
      for (int64_t n = 0; n < N; ++n) acc += (ld)x[n] * tw[(size_t)((f * n) % N)];
      X[f] = cd((double)acc.real(), (double)acc.imag());
    }
  } else {
    std::vector<cd> a((size_t)N), b((size_t)N);
    for (int64_t n = 0; n < N; ++n) a[(size_t)n] = cd(x[n], 0.0);
    fft_radix2(a.data(), b.data(), N, -1);
    for (int64_t f = 0; f < nb; ++f) X[f] = b[(size_t)f];
  }
}

// x[n] = (1/N)[Re X[0] + (-1)^n Re X[N/2] + 2 Re sum_{f=1}^{N/2-1} X[f] e^{2 pi i fn/N}]
// (C2 restricted to a Hermitian spectrum)
void inverse_onesided(const cd *X, int64_t N, double *x, int engine) {
  int64_t h = N / 2;
  if (engine == 0) {
    std::vector<cld> tw((size_t)N);
    for (int64_t m = 0; m < N; ++m) tw[(size_t)m] = cis(m, N);
    for (int64_t n = 0; n < N; ++n) {
      ld acc = (ld)X[0].real() + ((n & 1) ? -(ld)X[h].real() : (ld)X[h].real());
      for (int64_t f = 1; f < h; ++f) {
        cld t = cld(X[f]) * tw[(size_t)((f * n) % N)];
        acc += 2 * t.real();
      }
      x[n] = (double)(acc / (ld)N);
    }
  } else {
    std::vector<cd> a((size_t)N), b((size_t)N);
    a[0] = cd(X[0].real(), 0.0);
    a[(size_t)h] = cd(X[h].real(), 0.0);
    for (int64_t f = 1; f < h; ++f) {
      a[(size_t)f] = X[f];
      a[(size_t)(N - f)] = std::conj(X[f]);
    }
    fft_radix2(a.data(), b.data(), N, +1);
    for (int64_t n = 0; n < N; ++n) x[n] = b[(size_t)n].real() / (double)N;
  }
}

// bins any row touches (so engine 0 need not evaluate the rest of the spectrum)
std::vector<uint8_t> needed_bins(const qtam_ref_plan *p, int row_begin, int row_end) {
  std::vector<uint8_t> need((size_t)p->nb, 0);
  for (int k = row_begin; k < row_end; ++k) {
    const Row &r = p->rows[(size_t)k];
    for (int64_t j = -r.dk; j <= r.dk; ++j) {
      int64_t f = r.kc + j;
      if (f >= 0 && f < p->nb) need[(size_t)f] = 1;
    }
  }
  return need;
}

}  // namespace

extern "C" {

int qtam_ref_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

// lets the caller undo a launcher's OMP_NUM_THREADS=1 default (torchrun sets it for every rank)
void qtam_ref_set_threads(int n) {
#ifdef _OPENMP
  if (n > 0) omp_set_num_threads(n);
#else
  (void)n;
#endif
}

int qtam_ref_dft(const double *in, double *out, int64_t n, int sign) {
  if (!in || !out || n < 1 || (sign != 1 && sign != -1)) return 1;
  dft_naive(reinterpret_cast<const cd *>(in), reinterpret_cast<cd *>(out), n, sign);
  return 0;
}

int qtam_ref_fft(const double *in, double *out, int64_t n, int sign) {
  if (!in || !out || !is_fft_length(n) || (sign != 1 && sign != -1)) return 1;
  fft_radix2(reinterpret_cast<const cd *>(in), reinterpret_cast<cd *>(out), n, sign);
  return 0;
}

// I_0(x), modified Bessel function of the first kind, by its power series sum_k ((x/2)^k / k!)^2
static long double bessel_i0(long double x) {
  const long double h = 0.5L * x;
  long double term = 1.0L, sum = 1.0L;
  for (int k = 1; k < 500; ++k) {
    term *= (h / (long double)k) * (h / (long double)k);
    sum += term;
    if (term < 1e-22L * sum) break;
  }
  return sum;
}

// Unnormalised window value at offset j of a row with half-width dk (u = j/dk), App. A:
//   0 bisquare (A1 :272)  (1 - u^2)^2
//   1 Hann (A2 :276)      (1 + cos(pi u))/2
//   2 Kaiser (A3 :280)    I0(beta sqrt(1 - u^2)) / I0(beta)
//   3 Tukey (A4 :284)     1 for |u| <= 1 - a;  (1 + cos(pi (|u| - (1 - a))/a))/2 up to |u| = 1
//   4 Planck-taper (A5-A6 :293-299)  1 for |u| <= 1 - a, 0 at |u| = 1, else 1/(e^Z + 1) with, d = 1 - |u|,
//       Z = a/d + a/(d - a)   (reading R15: A6 as printed has the second denominator's sign flipped, which
//       would make the window tend to 0 instead of 1 at the inner edge of the transition)
static double raw_window(int type, double par, int64_t j, int64_t dk) {
  const long double PI = 3.141592653589793238462643383279502884L;
  const long double u = (long double)j / (long double)dk, au = fabsl(u);
  switch (type) {
    case 0: { const double ud = (double)j / (double)dk; return (1.0 - ud * ud) * (1.0 - ud * ud); }   // as before the families
    case 1: return (double)(0.5L * (1.0L + cosl(PI * u)));
    case 2: return (double)(bessel_i0((long double)par * sqrtl(1.0L - u * u)) / bessel_i0((long double)par));
    case 3: {
      const long double a = par;
      if (au <= 1.0L - a) return 1.0;
      return (double)(0.5L * (1.0L + cosl(PI * (au - (1.0L - a)) / a)));
    }
    default: {
      const long double a = par, d = 1.0L - au;
      if (d >= a) return 1.0;
      if (d <= 0.0L) return 0.0;
      const long double Z = a / d + a / (d - a);
      return (double)(1.0L / (expl(Z) + 1.0L));
    }
  }
}

int qtam_ref_plan_create(qtam_ref_plan **out, double fs, int64_t N, const double *Q, int nQ,
                         double fmin, double fmax, double spacing, const qtam_ref_options *opt) {
  if (!out || !Q || nQ < 1 || !(fs > 0) || !is_fft_length(N) || N % 8 != 0 || N < 8) return 1;
  qtam_ref_options o;
  o.window = 0; o.clamp_mode = 1; o.clamp_overlap = 1.0; o.max_window_bins = 0;
  o.cover_floor = 1e-2; o.rows_are_bins_per_octave = 0; o.window_param = 0.0; o.freqs = nullptr; o.n_freqs = 0; o.tile_length = 0; o.epsilon = 0.0;
  o.plane_window = nullptr; o.plane_window_param = nullptr;
  if (opt) o = *opt;
  const bool manual = o.freqs != nullptr && o.n_freqs >= 2;
  if (manual) { fmin = o.freqs[0]; fmax = o.freqs[o.n_freqs - 1]; }
  if (!(fmin > 0) || !(fmax > fmin) || !(fmax < fs / 2)) return 1;
  if (o.window < 0 || o.window > 4) return 2;
  if (o.window == 2 && !(o.window_param > 0)) return 1;
  if (o.window >= 3 && !(o.window_param > 0 && o.window_param <= 1.0)) return 1;
  if (!(o.epsilon >= 0.0)) return 1;
  for (int pl = 0; o.plane_window && pl < nQ; ++pl) {          // a composite bank: one window family per plane (:327)
    const int wt = o.plane_window[pl];
    const double wp = o.plane_window_param ? o.plane_window_param[pl] : 0.0;
    if (wt < 0 || wt > 4) return 2;
    if (wt == 2 && !(wp > 0)) return 1;
    if (wt >= 3 && !(wp > 0 && wp <= 1.0)) return 1;
  }
  if (!(o.clamp_overlap > 0)) o.clamp_overlap = 1.0;
  if (!(o.cover_floor > 0)) o.cover_floor = 1e-2;

  const double T = (double)N / fs;            // duration, the paper's N_t
  const double SQRT11 = std::sqrt(11.0);      // R1: bisquare tile half-width f*sqrt(11)/Q

  // frequency grid (R14)
  std::vector<double> f;
  if (manual) {
    for (int r = 0; r < o.n_freqs; ++r) {
      if (r > 0 && !(o.freqs[r] > o.freqs[r - 1])) return 1;   // ascending
      f.push_back(o.freqs[r]);
    }
  } else if (o.rows_are_bins_per_octave) {
    if (!(spacing > 0)) return 1;
    for (int r = 0;; ++r) {
      double fr = fmin * std::pow(2.0, (double)r / spacing);
      if (fr > fmax) break;
      f.push_back(fr);
    }
  } else {
    int R = (int)spacing;
    if (R < 2 || (double)R != spacing) return 1;
    for (int r = 0; r < R; ++r) f.push_back(fmin * std::pow(fmax / fmin, (double)r / (double)(R - 1)));
  }
  const int R = (int)f.size();
  if (R < 2) return 1;

  // clamp (A7): largest gap between consecutive centres
  double dfmax = 0;
  for (int r = 0; r + 1 < R; ++r) dfmax = std::max(dfmax, f[(size_t)r + 1] - f[(size_t)r]);
  int64_t Lmax = 0;  // 0 = unclamped
  if (o.clamp_mode == 1) Lmax = 2 * ((int64_t)std::ceil(o.clamp_overlap * T * dfmax) / 2) + 1;
  else if (o.clamp_mode == 2) {
    if (o.max_window_bins < 3) return 1;
    Lmax = 2 * ((o.max_window_bins - 1) / 2) + 1;  // odd, <= request
  } else if (o.clamp_mode != 0) return 1;

  // uniform tile length (every row zero-padded to the largest window): the longest support
  int64_t Luni = 0;
  for (int pl = 0; pl < nQ; ++pl)
    for (int r = 0; r < R; ++r) {
      int64_t L = 2 * (int64_t)std::floor(f[(size_t)r] * T * SQRT11 / Q[pl]) + 1;
      if (Lmax > 0) L = std::min(L, Lmax);
      Luni = std::max(Luni, L);
    }
  int64_t Muni = 0;
  if (o.tile_length == -1) Muni = next_pow2(Luni);
  else if (o.tile_length > 0) {
    if (!is_pow2(o.tile_length) || o.tile_length < Luni) return 1;
    Muni = o.tile_length;
  } else if (o.tile_length != 0) return 1;

  qtam_ref_plan *p = new (std::nothrow) qtam_ref_plan;
  if (!p) return 3;
  p->fs = fs; p->N = N; p->nb = N / 2 + 1; p->nP = nQ; p->nR = R; p->epsilon = o.epsilon;
  p->Q.assign(Q, Q + nQ);
  int64_t offset = 0, sumL = 0;
  for (int pl = 0; pl < nQ; ++pl) {
    if (!(Q[pl] >= SQRT11)) { delete p; return 1; }
    for (int r = 0; r < R; ++r) {
      Row row;
      row.plane = pl; row.row = r; row.q = Q[pl]; row.f_request = f[(size_t)r];
      row.kc = (int64_t)std::floor(f[(size_t)r] * T + 0.5);                 // R2
      int64_t dk_ideal = (int64_t)std::floor(f[(size_t)r] * T * SQRT11 / Q[pl]);  // R1
      int64_t L = 2 * dk_ideal + 1;                                         // Eq. 7
      if (Lmax > 0) L = std::min(L, Lmax);                                  // A8
      row.L = L; row.dk = (L - 1) / 2;
      if (row.dk < 1) { delete p; return 1; }                               // R13
      row.M = Muni > 0 ? Muni : next_pow2(L);                               // R5 / uniform layout
      row.f_center = (double)row.kc / T;
      row.offset = offset; offset += row.M; sumL += L;
      // the plane's window (Eq. 6; App. A; a composite bank gives every plane its own family,
      // :327) and unit-energy normalisation (Eq. 5 / R3); the sum runs over the unclipped support (R8)
      const int wtype = o.plane_window ? o.plane_window[pl] : o.window;
      const double wpar = o.plane_window_param ? o.plane_window_param[pl] : o.window_param;
      row.wraw.resize((size_t)L); row.w.resize((size_t)L);
      ld e = 0;
      for (int64_t j = -row.dk; j <= row.dk; ++j) {
        double v = raw_window(wtype, wpar, j, row.dk);
        row.wraw[(size_t)(j + row.dk)] = v;
        e += (ld)v * (ld)v;
      }
      row.norm = (double)(1.0L / sqrtl(e));
      for (int64_t i = 0; i < L; ++i) row.w[(size_t)i] = row.wraw[(size_t)i] * row.norm;
      p->rows.push_back(row);
    }
  }
  p->ctot = offset; p->sumL = sumL;

  // frame operator P[f] = sum_k |W_k[f]|^2 (C36) and cover sets (R9), joint and
  // per plane (R10); terms outside 0..N/2 are dropped (R8)
  p->P.assign((size_t)nQ + 1, std::vector<double>((size_t)p->nb, 0.0));
  p->cover.assign((size_t)nQ + 1, std::vector<uint8_t>((size_t)p->nb, 0));
  {
    std::vector<std::vector<ld>> acc((size_t)nQ + 1, std::vector<ld>((size_t)p->nb, 0.0L));
    for (const Row &r : p->rows)
      for (int64_t j = -r.dk; j <= r.dk; ++j) {
        int64_t b = r.kc + j;
        if (b < 0 || b >= p->nb) continue;
        ld w = r.w[(size_t)(j + r.dk)];
        acc[0][(size_t)b] += w * w;
        acc[(size_t)r.plane + 1][(size_t)b] += w * w;
        if (r.wraw[(size_t)(j + r.dk)] >= o.cover_floor) {
          p->cover[0][(size_t)b] = 1;
          p->cover[(size_t)r.plane + 1][(size_t)b] = 1;
        }
      }
    for (size_t s = 0; s < acc.size(); ++s)
      for (int64_t b = 0; b < p->nb; ++b) p->P[s][(size_t)b] = (double)acc[s][(size_t)b];
  }
  bool any = false;
  for (int64_t b = 0; b < p->nb; ++b) any = any || p->cover[0][(size_t)b];
  if (!any) { delete p; return 5; }
  *out = p;
  return 0;
}

void qtam_ref_plan_destroy(qtam_ref_plan *p) { delete p; }

int qtam_ref_plan_info(const qtam_ref_plan *p, qtam_ref_info *o) {
  if (!p || !o) return 1;
  o->n_planes = p->nP; o->n_rows = (int)p->rows.size(); o->n = p->N; o->n_bins = p->nb;
  o->coeffs_per_segment = p->ctot; o->sum_L = p->sumL;
  int64_t lo = -1, hi = -1, cnt = 0;
  double A = 0, B = 0;
  for (int64_t b = 0; b < p->nb; ++b) {
    B = std::max(B, p->P[0][(size_t)b]);
    if (!p->cover[0][(size_t)b]) continue;
    if (lo < 0) { lo = b; A = p->P[0][(size_t)b]; }
    hi = b; ++cnt;
    A = std::min(A, p->P[0][(size_t)b]);
  }
  o->cover_lo = lo; o->cover_hi = hi; o->cover_count = cnt;
  o->holes = (hi - lo + 1) - cnt;
  o->frame_A = A; o->frame_B = B;
  return 0;
}

int qtam_ref_plan_rows(const qtam_ref_plan *p, qtam_ref_row *out, int capacity) {
  if (!p || !out || capacity < (int)p->rows.size()) return 1;
  for (size_t k = 0; k < p->rows.size(); ++k) {
    const Row &r = p->rows[k];
    qtam_ref_row &o = out[k];
    o.plane = r.plane; o.row = r.row; o.q = r.q; o.f_request = r.f_request;
    o.f_center = r.f_center; o.kc = r.kc; o.dk = r.dk; o.L = r.L; o.M = r.M;
    o.offset = r.offset; o.norm = r.norm;
  }
  return 0;
}

int qtam_ref_plan_window(const qtam_ref_plan *p, int row, double *out) {
  if (!p || !out || row < 0 || row >= (int)p->rows.size()) return 1;
  const Row &r = p->rows[(size_t)row];
  std::copy(r.w.begin(), r.w.end(), out);
  return 0;
}

int qtam_ref_plan_frame(const qtam_ref_plan *p, int plane, double *P_out, uint8_t *cover_out) {
  if (!p || plane < -1 || plane >= p->nP) return 1;
  size_t s = (size_t)(plane + 1);
  if (P_out) std::copy(p->P[s].begin(), p->P[s].end(), P_out);
  if (cover_out) std::copy(p->cover[s].begin(), p->cover[s].end(), cover_out);
  return 0;
}

int qtam_ref_spectrum(const qtam_ref_plan *p, const double *x, int batch, double *X_out, int engine) {
  if (!p || !x || !X_out || batch < 0) return 1;
#pragma omp parallel for schedule(dynamic)
  for (int b = 0; b < batch; ++b)
    spectrum_onesided(x + (size_t)b * p->N, p->N, reinterpret_cast<cd *>(X_out) + (size_t)b * p->nb,
                      nullptr, engine);
  return 0;
}

// Y_k[n] = (N M)^{-1/2} sum_{j=-dk, 0<=kc+j<=N/2}^{dk} X[kc+j] W_k[j] e^{+2 pi i jn/M}, n=0..M-1
// (A9 PAPER.md:323; shift to baseband C46 :583; short inverse DFT and scale C47 :589, R4, R6, R8)
int qtam_ref_forward(const qtam_ref_plan *p, const double *x, int batch, double *coef, int engine) {
  if (!p || !x || !coef || batch < 0) return 1;
  const int K = (int)p->rows.size();
  std::vector<uint8_t> need = needed_bins(p, 0, K);
  for (int b = 0; b < batch; ++b) {
    std::vector<cd> X((size_t)p->nb);
    spectrum_onesided(x + (size_t)b * p->N, p->N, X.data(), need.data(), engine);
    cd *Y = reinterpret_cast<cd *>(coef) + (size_t)b * p->ctot;
#pragma omp parallel for schedule(dynamic)
    for (int k = 0; k < K; ++k) {
      const Row &r = p->rows[(size_t)k];
      const ld scale = 1.0L / sqrtl((ld)p->N * (ld)r.M);
      if (engine == 0) {
        std::vector<cld> tw((size_t)r.M);
        for (int64_t m = 0; m < r.M; ++m) tw[(size_t)m] = cis(m, r.M);
        for (int64_t n = 0; n < r.M; ++n) {
          cld acc(0, 0);
          for (int64_t j = -r.dk; j <= r.dk; ++j) {
            int64_t f = r.kc + j;
            if (f < 0 || f >= p->nb) continue;
            int64_t ph = ((j % r.M + r.M) % r.M) * n % r.M;
            acc += cld(X[(size_t)f]) * (ld)r.w[(size_t)(j + r.dk)] * tw[(size_t)ph];
          }
          acc *= scale;
          Y[r.offset + n] = cd((double)acc.real(), (double)acc.imag());
        }
      } else {
        std::vector<cd> a((size_t)r.M, cd(0, 0)), o((size_t)r.M);
        for (int64_t j = -r.dk; j <= r.dk; ++j) {
          int64_t f = r.kc + j;
          if (f < 0 || f >= p->nb) continue;
          a[(size_t)((j % r.M + r.M) % r.M)] = X[(size_t)f] * r.w[(size_t)(j + r.dk)];
        }
        fft_radix2(a.data(), o.data(), r.M, +1);
        for (int64_t n = 0; n < r.M; ++n) Y[r.offset + n] = o[(size_t)n] * (double)scale;
      }
    }
  }
  return 0;
}

// Eq. 12 as read in R17: the dense window of row r at bin f is norm * max(W'[f - kc], epsilon)
// on the support and norm * epsilon off it (the floor also lifts the window's exact zeros at |j| = dk, which
// Eq. 12 as printed would leave non-invertible).  epsilon = 0: the plain window, zero off the support.
static inline double dense_window(const qtam_ref_plan *p, const Row &r, int64_t f) {
  const int64_t j = f - r.kc;
  if (j < -r.dk || j > r.dk) return p->epsilon * r.norm;
  if (p->epsilon > 0) return std::max(r.wraw[(size_t)(j + r.dk)], p->epsilon) * r.norm;
  return r.w[(size_t)(j + r.dk)];
}

// T_k[tau] = (1/N) sum_j X[kc+j] W_k[j] e^{+2 pi i (kc+j) tau/N}, tau = 0..N-1 (C3)
int qtam_ref_dense(const qtam_ref_plan *p, const double *x, int batch, int row_begin, int row_end,
                   double *out, int engine) {
  if (!p || !x || !out || batch < 0 || row_begin < 0 || row_end > (int)p->rows.size() ||
      row_begin > row_end)
    return 1;
  const int64_t N = p->N;
  const int nr = row_end - row_begin;
  std::vector<uint8_t> need = needed_bins(p, row_begin, row_end);
  if (p->epsilon > 0) std::fill(need.begin(), need.end(), (uint8_t)1);
  for (int b = 0; b < batch; ++b) {
    std::vector<cd> X((size_t)p->nb);
    spectrum_onesided(x + (size_t)b * N, N, X.data(), need.data(), engine);
#pragma omp parallel for schedule(dynamic)
    for (int k = row_begin; k < row_end; ++k) {
      const Row &r = p->rows[(size_t)k];
      cd *Tk = reinterpret_cast<cd *>(out) + ((size_t)b * nr + (size_t)(k - row_begin)) * (size_t)N;
      if (engine == 0) {
        std::vector<cld> tw((size_t)N);
        for (int64_t m = 0; m < N; ++m) tw[(size_t)m] = cis(m, N);
        for (int64_t tau = 0; tau < N; ++tau) {
          cld acc(0, 0);
          if (p->epsilon > 0) {             // Eq. 12: every one-sided bin takes part
            for (int64_t f = 0; f < p->nb; ++f)
              acc += cld(X[(size_t)f]) * (ld)dense_window(p, r, f) * tw[(size_t)((f * tau) % N)];
          } else {
            for (int64_t j = -r.dk; j <= r.dk; ++j) {
              int64_t f = r.kc + j;
              if (f < 0 || f >= p->nb) continue;
              acc += cld(X[(size_t)f]) * (ld)r.w[(size_t)(j + r.dk)] * tw[(size_t)((f * tau) % N)];
            }
          }
          acc /= (ld)N;
          Tk[tau] = cd((double)acc.real(), (double)acc.imag());
        }
      } else {
        std::vector<cd> a((size_t)N, cd(0, 0)), o((size_t)N);
        for (int64_t j = -r.dk; j <= r.dk; ++j) {
          int64_t f = r.kc + j;
          if (f < 0 || f >= p->nb) continue;
          a[(size_t)f] = X[(size_t)f] * r.w[(size_t)(j + r.dk)];
        }
        if (p->epsilon > 0)
          for (int64_t f = 0; f < p->nb; ++f) a[(size_t)f] = X[(size_t)f] * dense_window(p, r, f);
        fft_radix2(a.data(), o.data(), N, +1);
        for (int64_t tau = 0; tau < N; ++tau) Tk[tau] = o[(size_t)tau] / (double)N;
      }
    }
  }
  return 0;
}

// atom h_k[m] = (1/N) sum_j W_k[j] e^{+2 pi i (kc+j) m/N} (C4 with tau folded in);
// T_k[tau] = sum_n x[n] h_k[(tau-n) mod N]  (= <x, g_{k,tau}> of C5, with the
// conjugation convention that makes C5 equal C3).  No DFT of x is taken anywhere here.
int qtam_ref_brute_tile(const qtam_ref_plan *p, const double *x, int row, double *out) {
  if (!p || !x || !out || row < 0 || row >= (int)p->rows.size()) return 1;
  const Row &r = p->rows[(size_t)row];
  const int64_t N = p->N;
  std::vector<cld> h((size_t)N);
  for (int64_t m = 0; m < N; ++m) {
    cld acc(0, 0);
    for (int64_t j = -r.dk; j <= r.dk; ++j) {
      int64_t f = r.kc + j;
      if (f < 0 || f >= p->nb) continue;
      acc += (ld)r.w[(size_t)(j + r.dk)] * cis(f * m, N);
    }
    h[(size_t)m] = acc / (ld)N;
  }
  cd *Tk = reinterpret_cast<cd *>(out);
  for (int64_t tau = 0; tau < N; ++tau) {
    cld acc(0, 0);
    for (int64_t n = 0; n < N; ++n) acc += (ld)x[n] * h[(size_t)(((tau - n) % N + N) % N)];
    Tk[tau] = cd((double)acc.real(), (double)acc.imag());
  }
  return 0;
}

// Eq. 11 = C42/C50 (:563, :602) with the tile spectra restored by C49 (:598):
//   Bhat_k[j] = sqrt(N/M) sum_n Y_k[n] e^{-2 pi i jn/M},  |j| <= dk
//   S[f] = sum_{k,j: kc+j=f} Bhat_k[j] W_k[j];  Xhat[f] = S[f]/P[f] on the cover set, else 0 (R9)
//   x = one-sided inverse DFT of Xhat (C2).  plane = -1: joint frame; plane = p: that plane (R10).
int qtam_ref_inverse(const qtam_ref_plan *p, const double *coef, int batch, int plane, double *x_out,
                     int engine) {
  if (!p || !coef || !x_out || batch < 0 || plane < -1 || plane >= p->nP) return 1;
  const int K = (int)p->rows.size();
  const std::vector<double> &P = p->P[(size_t)(plane + 1)];
  const std::vector<uint8_t> &C = p->cover[(size_t)(plane + 1)];
#pragma omp parallel for schedule(dynamic)
  for (int b = 0; b < batch; ++b) {
    const cd *Y = reinterpret_cast<const cd *>(coef) + (size_t)b * p->ctot;
    std::vector<cld> S((size_t)p->nb, cld(0, 0));
    for (int k = 0; k < K; ++k) {
      const Row &r = p->rows[(size_t)k];
      if (plane >= 0 && r.plane != plane) continue;
      const ld amp = sqrtl((ld)p->N / (ld)r.M);
      if (engine == 0) {
        std::vector<cld> tw((size_t)r.M);
        for (int64_t m = 0; m < r.M; ++m) tw[(size_t)m] = cis(-m, r.M);
        for (int64_t j = -r.dk; j <= r.dk; ++j) {
          int64_t f = r.kc + j;
          if (f < 0 || f >= p->nb) continue;
          int64_t jm = (j % r.M + r.M) % r.M;
          cld acc(0, 0);
          for (int64_t n = 0; n < r.M; ++n) acc += cld(Y[r.offset + n]) * tw[(size_t)(jm * n % r.M)];
          S[(size_t)f] += acc * amp * (ld)r.w[(size_t)(j + r.dk)];
        }
      } else {
        std::vector<cd> o((size_t)r.M);
        fft_radix2(Y + r.offset, o.data(), r.M, -1);
        for (int64_t j = -r.dk; j <= r.dk; ++j) {
          int64_t f = r.kc + j;
          if (f < 0 || f >= p->nb) continue;
          int64_t jm = (j % r.M + r.M) % r.M;
          S[(size_t)f] += cld(o[(size_t)jm]) * amp * (ld)r.w[(size_t)(j + r.dk)];
        }
      }
    }
    std::vector<cd> Xh((size_t)p->nb, cd(0, 0));
    for (int64_t f = 0; f < p->nb; ++f)
      if (C[(size_t)f]) {
        cld v = S[(size_t)f] / (ld)P[(size_t)f];
        Xh[(size_t)f] = cd((double)v.real(), (double)v.imag());
      }
    inverse_onesided(Xh.data(), p->N, x_out + (size_t)b * p->N, engine);
  }
  return 0;
}

// ---- the paper's output-length options (A22: PAPER.md:150, :158-160, :184, :343) ---------------------------------
// Every row resampled to the same number n of time samples, n any integer >= the largest window (no power of two
// needed): "standard" n = N/2 + 1 (64 x 410, 62 x 12289), "minimal" n = ceil(N_t Delta f_max) + 1 = the largest
// window's 2 dk + 1 bins (64 x 33, 62 x 669), or user-set.  C46/C47 with N_out = n:
//   Y'_k[m] = (N n)^{-1/2} sum_j X[kc + j] W_k[j] e^{+2 pi i j m / n},  m = 0..n-1.
// Naive long-double sums (the definition); `engine` only selects how the long transform of x is evaluated.
int64_t qtam_ref_output_length(const qtam_ref_plan *p, int mode) {
  if (!p) return 0;
  if (mode == -1) return p->N / 2 + 1;
  int64_t lmax = 0;
  for (const Row &r : p->rows) lmax = std::max(lmax, 2 * r.dk + 1);
  return mode == -2 ? lmax : 0;
}

int qtam_ref_forward_length(const qtam_ref_plan *p, const double *x, int batch, int64_t n, double *out, int engine) {
  if (!p || !x || !out || batch < 0 || n < qtam_ref_output_length(p, -2)) return 1;
  const int K = (int)p->rows.size();
  std::vector<uint8_t> need = needed_bins(p, 0, K);
  std::vector<cld> tw((size_t)n);
  for (int64_t m = 0; m < n; ++m) tw[(size_t)m] = cis(m, n);
#pragma omp parallel for schedule(dynamic)
  for (int b = 0; b < batch; ++b) {
    std::vector<cd> X((size_t)p->nb);
    spectrum_onesided(x + (size_t)b * p->N, p->N, X.data(), need.data(), engine);
    cd *Y = reinterpret_cast<cd *>(out) + (size_t)b * (size_t)K * (size_t)n;
    for (int k = 0; k < K; ++k) {
      const Row &r = p->rows[(size_t)k];
      const ld scale = 1.0L / sqrtl((ld)p->N * (ld)n);
      for (int64_t m = 0; m < n; ++m) {
        cld acc(0, 0);
        for (int64_t j = -r.dk; j <= r.dk; ++j) {
          const int64_t f = r.kc + j;
          if (f < 0 || f >= p->nb) continue;
          const int64_t ph = ((j % n + n) % n) * m % n;
          acc += cld(X[(size_t)f]) * (ld)r.w[(size_t)(j + r.dk)] * tw[(size_t)ph];
        }
        acc *= scale;
        Y[(size_t)k * (size_t)n + (size_t)m] = cd((double)acc.real(), (double)acc.imag());
      }
    }
  }
  return 0;
}

// band values of one resampled row: Bhat[j] = sqrt(N/n) sum_m Y'[m] e^{-2 pi i j m / n}, |j| <= dk (C49 with N_out = n)
static void band_from_length(const qtam_ref_plan *p, const Row &r, const cd *Y, int64_t n, const std::vector<cld> &twn,
                             std::vector<cld> &B) {
  B.assign((size_t)(2 * r.dk + 1), cld(0, 0));
  const ld amp = sqrtl((ld)p->N / (ld)n);
  for (int64_t j = -r.dk; j <= r.dk; ++j) {
    const int64_t jm = (j % n + n) % n;
    cld acc(0, 0);
    for (int64_t m = 0; m < n; ++m) acc += cld(Y[m]) * std::conj(twn[(size_t)(jm * m % n)]);
    B[(size_t)(j + r.dk)] = acc * amp;
  }
}

int qtam_ref_inverse_length(const qtam_ref_plan *p, const double *in, int batch, int64_t n, int plane, double *x_out,
                            int engine) {
  if (!p || !in || !x_out || batch < 0 || plane < -1 || plane >= p->nP || n < qtam_ref_output_length(p, -2)) return 1;
  const int K = (int)p->rows.size();
  const std::vector<double> &P = p->P[(size_t)(plane + 1)];
  const std::vector<uint8_t> &C = p->cover[(size_t)(plane + 1)];
  std::vector<cld> tw((size_t)n);
  for (int64_t m = 0; m < n; ++m) tw[(size_t)m] = cis(m, n);
#pragma omp parallel for schedule(dynamic)
  for (int b = 0; b < batch; ++b) {
    const cd *Y = reinterpret_cast<const cd *>(in) + (size_t)b * (size_t)K * (size_t)n;
    std::vector<cld> S((size_t)p->nb, cld(0, 0)), B;
    for (int k = 0; k < K; ++k) {
      const Row &r = p->rows[(size_t)k];
      if (plane >= 0 && r.plane != plane) continue;
      band_from_length(p, r, Y + (size_t)k * (size_t)n, n, tw, B);
      for (int64_t j = -r.dk; j <= r.dk; ++j) {
        const int64_t f = r.kc + j;
        if (f < 0 || f >= p->nb) continue;
        S[(size_t)f] += B[(size_t)(j + r.dk)] * (ld)r.w[(size_t)(j + r.dk)];
      }
    }
    std::vector<cd> Xh((size_t)p->nb, cd(0, 0));
    for (int64_t f = 0; f < p->nb; ++f)
      if (C[(size_t)f]) {
        cld v = S[(size_t)f] / (ld)P[(size_t)f];
        Xh[(size_t)f] = cd((double)v.real(), (double)v.imag());
      }
    inverse_onesided(Xh.data(), p->N, x_out + (size_t)b * p->N, engine);
  }
  return 0;
}

// Re-sampling of a [rows][n_in] image to [rows][n_out] (:160 "up-sampling the compressed image back to the original
// size", Fig. 3): every row is band limited to its window's 2 dk + 1 bins, so its n_in samples determine the band
// exactly (n_in >= 2 dk + 1) and the band determines the n_out samples.  With the energy normalisation of C47:
//   Y''[m] = (n_in n_out)^{-1/2} sum_{|j| <= dk} ( sum_l Y'[l] e^{-2 pi i j l / n_in} ) e^{+2 pi i j m / n_out}.
int qtam_ref_resample(const qtam_ref_plan *p, const double *in, int batch, int64_t n_in, int64_t n_out, double *out) {
  const int64_t lmax = qtam_ref_output_length(p, -2);
  if (!p || !in || !out || batch < 0 || n_in < lmax || n_out < lmax) return 1;
  const int K = (int)p->rows.size();
  std::vector<cld> twi((size_t)n_in), two((size_t)n_out);
  for (int64_t m = 0; m < n_in; ++m) twi[(size_t)m] = cis(m, n_in);
  for (int64_t m = 0; m < n_out; ++m) two[(size_t)m] = cis(m, n_out);
#pragma omp parallel for schedule(dynamic) collapse(2)
  for (int b = 0; b < batch; ++b)
    for (int k = 0; k < K; ++k) {
      const Row &r = p->rows[(size_t)k];
      const cd *Y = reinterpret_cast<const cd *>(in) + ((size_t)b * (size_t)K + (size_t)k) * (size_t)n_in;
      cd *O = reinterpret_cast<cd *>(out) + ((size_t)b * (size_t)K + (size_t)k) * (size_t)n_out;
      std::vector<cld> B;
      band_from_length(p, r, Y, n_in, twi, B);            // = sqrt(N/n_in) DFT
      const ld scale = 1.0L / sqrtl((ld)p->N * (ld)n_out);
      for (int64_t m = 0; m < n_out; ++m) {
        cld acc(0, 0);
        for (int64_t j = -r.dk; j <= r.dk; ++j)
          acc += B[(size_t)(j + r.dk)] * two[(size_t)(((j % n_out + n_out) % n_out) * m % n_out)];
        acc *= scale;
        O[m] = cd((double)acc.real(), (double)acc.imag());
      }
    }
  return 0;
}

// ---- clusters of active pixels ("a clustering algorithm to identify contiguous energetic regions
// based on a tunable normalized threshold and minimum area ... a binary mask applied to the complex CQT") ----------
// The image is one Q-plane in the uniform-tile layout, rows x M pixels; a pixel is ACTIVE where `mask` is non-zero
// (the caller makes it from the row-median threshold, the "normalized threshold").  Clusters are the connected
// components of the active pixels under 4-connectivity, the time axis circular like the transform, the frequency
// axis not (R19); components with fewer than min_area pixels are dropped.  Plain flood fill.
// labels[pixel] = 0 for background / dropped, else 1 + the smallest pixel index (row * M + n) of its cluster: a
// canonical numbering, so that two implementations can be compared label by label.  count[b] = clusters kept.
int qtam_ref_cluster_labels(const uint8_t *mask, int batch, int rows, int64_t M, int min_area, int32_t *labels,
                            int32_t *count) {
  if (!mask || !labels || batch < 0 || rows < 1 || M < 1 || (int64_t)rows * M >= (int64_t(1) << 31)) return 1;
  const int64_t npx = (int64_t)rows * M;
  for (int b = 0; b < batch; ++b) {
    const uint8_t *A = mask + (size_t)b * (size_t)npx;
    int32_t *Lb = labels + (size_t)b * (size_t)npx;
    std::fill(Lb, Lb + npx, 0);
    std::vector<uint8_t> seen((size_t)npx, 0);
    std::vector<int64_t> stack, members;
    int32_t kept = 0;
    for (int64_t start = 0; start < npx; ++start) {        // ascending: `start` is the cluster's smallest index
      if (!A[start] || seen[(size_t)start]) continue;
      stack.assign(1, start); members.clear();
      seen[(size_t)start] = 1;
      while (!stack.empty()) {
        const int64_t i = stack.back(); stack.pop_back();
        members.push_back(i);
        const int64_t r = i / M, n = i % M;
        const int64_t nb[4] = {r * M + (n + 1) % M, r * M + (n + M - 1) % M, r + 1 < rows ? (r + 1) * M + n : -1,
                               r > 0 ? (r - 1) * M + n : -1};
        for (int64_t j : nb)
          if (j >= 0 && A[j] && !seen[(size_t)j]) { seen[(size_t)j] = 1; stack.push_back(j); }
      }
      if ((int64_t)members.size() >= (int64_t)min_area) {
        for (int64_t i : members) Lb[i] = (int32_t)(start + 1);
        ++kept;
      }
    }
    if (count) count[b] = kept;
  }
  return 0;
}

int qtam_ref_project_cover(const qtam_ref_plan *p, const double *x, int batch, int plane,
                           double *x_out, int engine) {
  if (!p || !x || !x_out || batch < 0 || plane < -1 || plane >= p->nP) return 1;
  const std::vector<uint8_t> &C = p->cover[(size_t)(plane + 1)];
#pragma omp parallel for schedule(dynamic)
  for (int b = 0; b < batch; ++b) {
    std::vector<cd> X((size_t)p->nb);
    spectrum_onesided(x + (size_t)b * p->N, p->N, X.data(), C.data(), engine);
    for (int64_t f = 0; f < p->nb; ++f)
      if (!C[(size_t)f]) X[(size_t)f] = cd(0, 0);
    inverse_onesided(X.data(), p->N, x_out + (size_t)b * p->N, engine);
  }
  return 0;
}

// BASELINE.json config 5 / R11: m = median_n |Y_k[n]| (two middle values averaged, M is even);
// zero every Y_k[n] with |Y_k[n]| < kappa*m (strict), per (segment, row).
int qtam_ref_threshold_rowmedian(const qtam_ref_plan *p, double *coef, int batch, double kappa) {
  if (!p || !coef || batch < 0) return 1;
  for (int b = 0; b < batch; ++b)
    for (const Row &r : p->rows) {
      cd *Y = reinterpret_cast<cd *>(coef) + (size_t)b * p->ctot + r.offset;
      std::vector<double> mag((size_t)r.M), s;
      for (int64_t n = 0; n < r.M; ++n) mag[(size_t)n] = std::sqrt(Y[n].real() * Y[n].real() + Y[n].imag() * Y[n].imag());
      s = mag;
      std::sort(s.begin(), s.end());
      double m = 0.5 * (s[(size_t)(r.M / 2 - 1)] + s[(size_t)(r.M / 2)]);
      double t = kappa * m;
      for (int64_t n = 0; n < r.M; ++n)
        if (mag[(size_t)n] < t) Y[n] = cd(0, 0);
    }
  return 0;
}

// Same rule with every operation in IEEE binary32, round-to-nearest, no fused multiply-add
// (this file is compiled with -ffp-contract=off):
//   a = fl(fl(re*re) + fl(im*im)); mag = fl(sqrt(a)); m = fl(0.5*fl(lo+hi)); t = fl(kappa*m).
int qtam_ref_threshold_rowmedian_f32(const qtam_ref_plan *p, float *coef, int batch, float kappa) {
  if (!p || !coef || batch < 0) return 1;
  for (int b = 0; b < batch; ++b)
    for (const Row &r : p->rows) {
      float *Y = coef + 2 * ((size_t)b * p->ctot + r.offset);
      std::vector<float> mag((size_t)r.M), s;
      for (int64_t n = 0; n < r.M; ++n) {
        volatile float rr = Y[2 * n] * Y[2 * n];
        volatile float ii = Y[2 * n + 1] * Y[2 * n + 1];
        volatile float a = rr + ii;
        mag[(size_t)n] = std::sqrt((float)a);
      }
      s = mag;
      std::sort(s.begin(), s.end());
      volatile float sum = s[(size_t)(r.M / 2 - 1)] + s[(size_t)(r.M / 2)];
      volatile float m = 0.5f * sum;
      volatile float t = kappa * m;
      for (int64_t n = 0; n < r.M; ++n)
        if (mag[(size_t)n] < t) { Y[2 * n] = 0.0f; Y[2 * n + 1] = 0.0f; }
    }
  return 0;
}

// Eq. 13: x = F^{-1}{ T~_k[f] / W~_k[f] } from ONE dense tile, with the window of Eq. 12
// (epsilon off the support).  T~_k[f] = sum_tau T_k[tau] e^{-2 pi i f tau/N} = X[f] W_k[f] for f = 0..N/2 (C33
// :523); the real series comes back through the one-sided inverse DFT of C2 (:371).  Naive sums throughout.
int qtam_ref_dense_invert(const qtam_ref_plan *p, const double *tile, int batch, int row, double *x_out) {
  if (!p || !tile || !x_out || batch < 0 || row < 0 || row >= (int)p->rows.size()) return 1;
  if (!(p->epsilon > 0)) return 2;
  const int64_t N = p->N;
  const Row &r = p->rows[(size_t)row];
  std::vector<cld> tw((size_t)N);
  for (int64_t m = 0; m < N; ++m) tw[(size_t)m] = cis(m, N);
  for (int b = 0; b < batch; ++b) {
    const cd *Tk = reinterpret_cast<const cd *>(tile) + (size_t)b * N;
    std::vector<cld> Xh((size_t)p->nb);
    for (int64_t f = 0; f < p->nb; ++f) {
      cld acc(0, 0);
      for (int64_t tau = 0; tau < N; ++tau) acc += cld(Tk[tau]) * std::conj(tw[(size_t)((f * tau) % N)]);
      Xh[(size_t)f] = acc / (ld)dense_window(p, r, f);
    }
    for (int64_t n = 0; n < N; ++n) {
      ld acc = Xh[0].real() + ((n & 1) ? -1.0L : 1.0L) * Xh[(size_t)(N / 2)].real();
      for (int64_t f = 1; f < N / 2; ++f) acc += 2.0L * (Xh[(size_t)f] * tw[(size_t)((f * n) % N)]).real();
      x_out[(size_t)b * N + n] = (double)(acc / (ld)N);
    }
  }
  return 0;
}

// Re-modulation with the carrier (Eq. 10a :113-117; :129 "re-modulated with the carrier to recover the
// original T_k"): the decimated envelope times e^{+2 pi i kc n / M_k}, and the amplitude of C47 undone, gives
// the dense tile on the coarse time grid t_n = n T / M_k:  T_k[n N/M_k] = sqrt(M_k/N) e^{2 pi i kc n/M_k} Y_k[n].
int qtam_ref_remodulate(const qtam_ref_plan *p, const double *coef, int batch, double *out) {
  if (!p || !coef || !out || batch < 0) return 1;
  const ld TAU = 6.283185307179586476925286766559005768L;
  for (int b = 0; b < batch; ++b)
    for (const Row &r : p->rows) {
      const cd *Y = reinterpret_cast<const cd *>(coef) + (size_t)b * p->ctot + r.offset;
      cd *O = reinterpret_cast<cd *>(out) + (size_t)b * p->ctot + r.offset;
      const ld amp = sqrtl((ld)r.M / (ld)p->N);
      for (int64_t n = 0; n < r.M; ++n) {
        const int64_t m = (int64_t)(((__int128)r.kc * n) % r.M);       // R12: index reduced in integers
        const ld a = TAU * (ld)m / (ld)r.M;
        const ld c = cosl(a), s = sinl(a);
        O[n] = cd((double)(amp * ((ld)Y[n].real() * c - (ld)Y[n].imag() * s)),
                  (double)(amp * ((ld)Y[n].real() * s + (ld)Y[n].imag() * c)));
      }
    }
  return 0;
}

// Instantaneous frequency (Fig. 5 :182: "the time-derivative of the unwrapped phase" of the
// demodulated tile).  Reading R16: the derivative is the forward difference on the row's own time grid
// t_n = n T/M_k, circular like the transform; unwrapping makes successive phase differences fall in
// (-pi, pi], so the difference of the unwrapped phase is Arg(Y[n+1] conj Y[n]).  The carrier the
// demodulation removed is added back:  f_inst[n] = (kc + (M_k / 2 pi) Arg(Y_k[(n+1) mod M_k] conj Y_k[n])) / T  [Hz].
int qtam_ref_instantaneous_frequency(const qtam_ref_plan *p, const double *coef, int batch, double *out) {
  if (!p || !coef || !out || batch < 0) return 1;
  const ld TAU = 6.283185307179586476925286766559005768L;
  const ld T = (ld)p->N / (ld)p->fs;
  for (int b = 0; b < batch; ++b)
    for (const Row &r : p->rows) {
      const cd *Y = reinterpret_cast<const cd *>(coef) + (size_t)b * p->ctot + r.offset;
      double *O = out + (size_t)b * p->ctot + r.offset;
      for (int64_t n = 0; n < r.M; ++n) {
        const cd a = Y[n], c = Y[(n + 1) % r.M];
        const ld re = (ld)c.real() * (ld)a.real() + (ld)c.imag() * (ld)a.imag();
        const ld im = (ld)c.imag() * (ld)a.real() - (ld)c.real() * (ld)a.imag();
        const ld dphi = atan2l(im, re);
        O[n] = (double)(((ld)r.kc + (ld)r.M * dphi / TAU) / T);
      }
    }
  return 0;
}

// Multi-Q scan: per (segment, Q-plane) a quality metric of the plane's spectrogram
// |Y_k[n]|^2 -- metric 0: total energy sum_{k in plane} sum_n |Y_k[n]|^2, metric 1: peak pixel
// max_{k,n} |Y_k[n]|^2 -- and "optimal selection": the plane with the largest metric, independently for
// every segment (lowest plane index on ties).
int qtam_ref_plane_metric(const qtam_ref_plan *p, const double *coef, int batch, int metric,
                          double *out_metric, int32_t *out_best) {
  if (!p || !coef || batch < 0 || !out_metric || metric < 0 || metric > 1) return 1;
  for (int b = 0; b < batch; ++b) {
    std::vector<ld> val((size_t)p->nP, 0.0L);
    for (const Row &r : p->rows) {
      const cd *Y = reinterpret_cast<const cd *>(coef) + (size_t)b * p->ctot + r.offset;
      for (int64_t n = 0; n < r.M; ++n) {
        const ld e = (ld)Y[n].real() * (ld)Y[n].real() + (ld)Y[n].imag() * (ld)Y[n].imag();
        if (metric == 0) val[(size_t)r.plane] += e;
        else if (e > val[(size_t)r.plane]) val[(size_t)r.plane] = e;
      }
    }
    int best = 0;
    for (int q = 0; q < p->nP; ++q) {
      out_metric[(size_t)b * p->nP + q] = (double)val[(size_t)q];
      if (val[(size_t)q] > val[(size_t)best]) best = q;
    }
    if (out_best) out_best[b] = best;
  }
  return 0;
}

// "Optimal selection mode": the composite output built from each segment's best plane.  Planes
// have different sizes in the ragged layout, so the output is [batch][max_p C_p], plane best[b] of segment b
// copied to its start and the rest zero.
int qtam_ref_gather_plane(const qtam_ref_plan *p, const double *coef, int batch, const int32_t *best, double *out) {
  if (!p || !coef || !best || !out || batch < 0) return 1;
  std::vector<int64_t> lo((size_t)p->nP, p->ctot), hi((size_t)p->nP, 0);
  for (const Row &r : p->rows) {
    lo[(size_t)r.plane] = std::min(lo[(size_t)r.plane], r.offset);
    hi[(size_t)r.plane] = std::max(hi[(size_t)r.plane], r.offset + r.M);
  }
  int64_t cmax = 0;
  for (int q = 0; q < p->nP; ++q) cmax = std::max(cmax, hi[(size_t)q] - lo[(size_t)q]);
  for (int b = 0; b < batch; ++b) {
    if (best[b] < 0 || best[b] >= p->nP) return 1;
    const int64_t a = lo[(size_t)best[b]], n = hi[(size_t)best[b]] - a;
    for (int64_t i = 0; i < cmax; ++i) {
      out[2 * ((size_t)b * cmax + i)] = i < n ? coef[2 * ((size_t)b * p->ctot + a + i)] : 0.0;
      out[2 * ((size_t)b * cmax + i) + 1] = i < n ? coef[2 * ((size_t)b * p->ctot + a + i) + 1] : 0.0;
    }
  }
  return 0;
}

}  // extern "C"
