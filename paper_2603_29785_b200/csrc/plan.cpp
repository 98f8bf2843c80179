// plan.cpp -- host plan of libqtam: grid, centre bins, clamp, windows, output lengths, frame
// operator, cover sets and the bin->band CSR used by the inverse's segmented reduction.
// Follows PAPER.md App. A (:303-321) and Eq. 5-7 (:63-72) with the readings R1-R14 of DESIGN.md.
#include <algorithm>
#include <cmath>

#include "qtam_internal.hpp"

namespace qtam {

static bool pow2(int64_t v) { return v > 0 && (v & (v - 1)) == 0; }

// Unnormalised window value at offset j of a row with half-width dk, u = j/dk (App. A):
// bisquare A1 :272, Hann A2 :276, Kaiser A3 :280 (I_0 from <cmath>), Tukey A4 :284, Planck-taper A5-A6
// :293-299 with Z = a/d + a/(d - a), d = 1 - |u| (R15).
static double window_value(int type, double par, int64_t j, int64_t dk) {
  const double pi = 3.14159265358979323846;
  const double u = double(j) / double(dk), au = std::fabs(u);
  switch (type) {
    case 1: return 0.5 * (1.0 + std::cos(pi * u));
    case 2: return std::cyl_bessel_i(0.0, par * std::sqrt(std::max(0.0, 1.0 - u * u))) / std::cyl_bessel_i(0.0, par);
    case 3:
      if (au <= 1.0 - par) return 1.0;
      return 0.5 * (1.0 + std::cos(pi * (au - (1.0 - par)) / par));
    case 4: {
      const double d = 1.0 - au;
      if (d >= par) return 1.0;
      if (d <= 0.0) return 0.0;
      return 1.0 / (std::exp(par / d + par / (d - par)) + 1.0);
    }
    default: return (1.0 - u * u) * (1.0 - u * u);
  }
}

qtam_status build_host_plan(HostPlan &hp, double fs, int64_t N, const double *Q, int nQ, double fmin,
                            double fmax, double spacing, qtam_dtype dtype, const qtam_options *uopt) {
  // segment lengths: 2^k, or 3 * 2^k (the paper's own benchmark shape is 6 s at 4096 Hz = 24576 samples, :178, :339)
  const bool n_ok = pow2(N) || (N % 3 == 0 && pow2(N / 3));
  if (!Q || nQ < 1 || !(fs > 0.0) || !n_ok || N < 8 || N % 8 != 0) return QTAM_ERR_INVALID_ARG;
  if (dtype != QTAM_F32 && dtype != QTAM_F64) return QTAM_ERR_INVALID_ARG;
  if (N > (int64_t(1) << 26)) return QTAM_ERR_UNSUPPORTED;

  qtam_options o{};
  o.struct_size = sizeof(qtam_options);
  o.clamp_mode = 1;
  o.clamp_overlap = 1.0;
  o.cover_floor = 1e-2;
  o.max_batch = 1;
  if (uopt) {
    if (uopt->struct_size != sizeof(qtam_options)) return QTAM_ERR_INVALID_ARG;
    o = *uopt;
    if (!(o.clamp_overlap > 0.0)) o.clamp_overlap = 1.0;
    if (!(o.cover_floor > 0.0)) o.cover_floor = 1e-2;
    if (o.max_batch < 1) o.max_batch = 1;
  }
  if (o.window < 0 || o.window > 4) return QTAM_ERR_UNSUPPORTED;
  if (o.window == 2 && !(o.window_param > 0.0)) return QTAM_ERR_INVALID_ARG;
  if (o.window >= 3 && !(o.window_param > 0.0 && o.window_param <= 1.0)) return QTAM_ERR_INVALID_ARG;
  if (!(o.epsilon >= 0.0)) return QTAM_ERR_INVALID_ARG;
  if (o.out_length < -2) return QTAM_ERR_INVALID_ARG;
  // a composite bank: one window family (and shape parameter) per plane (:327)
  std::vector<int> wtype(size_t(nQ), o.window);
  std::vector<double> wpar(size_t(nQ), o.window_param);
  std::vector<int> wident(size_t(nQ), 0);
  for (int pl = 0; o.plane_window && pl < nQ; ++pl) {
    wtype[size_t(pl)] = o.plane_window[pl];
    wpar[size_t(pl)] = o.plane_window_param ? o.plane_window_param[pl] : 0.0;
    if (wtype[size_t(pl)] < 0 || wtype[size_t(pl)] > 4) return QTAM_ERR_UNSUPPORTED;
    if (wtype[size_t(pl)] == 2 && !(wpar[size_t(pl)] > 0.0)) return QTAM_ERR_INVALID_ARG;
    if (wtype[size_t(pl)] >= 3 && !(wpar[size_t(pl)] > 0.0 && wpar[size_t(pl)] <= 1.0)) return QTAM_ERR_INVALID_ARG;
    wident[size_t(pl)] = pl;
    for (int q = 0; q < pl; ++q)
      if (wtype[size_t(q)] == wtype[size_t(pl)] && wpar[size_t(q)] == wpar[size_t(pl)]) { wident[size_t(pl)] = wident[size_t(q)]; break; }
  }
  const bool manual = o.freqs != nullptr && o.n_freqs >= 2;
  if (manual) { fmin = o.freqs[0]; fmax = o.freqs[o.n_freqs - 1]; }
  if (!(fmin > 0.0) || !(fmax > fmin) || !(fmax < 0.5 * fs)) return QTAM_ERR_INVALID_ARG;
  if (o.clamp_mode < 0 || o.clamp_mode > 2) return QTAM_ERR_INVALID_ARG;

  hp.fs = fs; hp.N = N; hp.nb = N / 2 + 1; hp.nP = nQ; hp.dtype = dtype; hp.opt = o;
  hp.opt.freqs = nullptr;                     // the caller's lists are only read here
  hp.opt.plane_window = nullptr; hp.opt.plane_window_param = nullptr;
  const double dur = double(N) / fs;          // N_t of the paper (:75)
  const double tile_c = std::sqrt(11.0);      // R1

  // centre frequencies (:303, R14)
  std::vector<double> fc;
  if (manual) {
    for (int r = 0; r < o.n_freqs; ++r) {
      if (r > 0 && !(o.freqs[r] > o.freqs[r - 1])) return QTAM_ERR_INVALID_ARG;   // ascending
      fc.push_back(o.freqs[r]);
    }
  } else if (o.rows_are_bins_per_octave) {
    if (!(spacing > 0.0)) return QTAM_ERR_INVALID_ARG;
    for (int r = 0; r < (1 << 20); ++r) {
      const double v = fmin * std::pow(2.0, double(r) / spacing);
      if (v > fmax) break;
      fc.push_back(v);
    }
  } else {
    const int R = int(spacing);
    if (R < 2 || double(R) != spacing) return QTAM_ERR_INVALID_ARG;
    fc.resize(size_t(R));
    for (int r = 0; r < R; ++r) fc[size_t(r)] = fmin * std::pow(fmax / fmin, double(r) / double(R - 1));
  }
  if (fc.size() < 2) return QTAM_ERR_INVALID_ARG;
  hp.nR = int(fc.size());

  // width cap (A7 :307 / manual); 0 means "no cap"
  int64_t cap = 0;
  if (o.clamp_mode == 1) {
    double gap = 0.0;
    for (size_t r = 1; r < fc.size(); ++r) gap = std::max(gap, fc[r] - fc[r - 1]);
    const int64_t c = int64_t(std::ceil(o.clamp_overlap * dur * gap));
    cap = 2 * (c / 2) + 1;
  } else if (o.clamp_mode == 2) {
    if (o.max_window_bins < 3) return QTAM_ERR_INVALID_ARG;
    cap = 2 * ((o.max_window_bins - 1) / 2) + 1;
  }

  // uniform tile length (:127-129, every row zero-padded to the largest window) or per-row lengths (R5)
  int64_t m_uniform = 0;
  if (o.tile_length != 0) {
    int64_t lmaxrow = 0;
    for (int pl = 0; pl < nQ; ++pl)
      for (int r = 0; r < hp.nR; ++r) {
        int64_t len = 2 * int64_t(std::floor(fc[size_t(r)] * dur * tile_c / Q[pl])) + 1;
        if (cap > 0 && len > cap) len = cap;
        lmaxrow = std::max(lmaxrow, len);
      }
    if (o.tile_length == -1) { m_uniform = 1; while (m_uniform < lmaxrow) m_uniform <<= 1; }
    else if (o.tile_length > 0 && pow2(o.tile_length) && o.tile_length >= lmaxrow) m_uniform = o.tile_length;
    else return QTAM_ERR_INVALID_ARG;
  }

  hp.rows.clear();
  hp.win.clear();
  int64_t coff = 0, woff = 0, mmax = 0;
  for (int pl = 0; pl < nQ; ++pl) {
    if (!(Q[pl] >= tile_c)) return QTAM_ERR_INVALID_ARG;
    for (int r = 0; r < hp.nR; ++r) {
      HostRow h{};
      h.plane = pl; h.row = r; h.q = Q[pl]; h.f_request = fc[size_t(r)];
      h.kc = int64_t(std::floor(fc[size_t(r)] * dur + 0.5));                      // R2
      int64_t len = 2 * int64_t(std::floor(fc[size_t(r)] * dur * tile_c / Q[pl])) + 1;  // R1, Eq. 7
      if (cap > 0 && len > cap) len = cap;                                       // A8 :311
      h.L = len; h.dk = (len - 1) / 2;
      if (h.dk < 1) return QTAM_ERR_INVALID_ARG;                                  // R13
      int64_t m = 1;
      while (m < len) m <<= 1;                                                   // R5
      if (m_uniform > 0) m = m_uniform;
      h.M = m; mmax = std::max(mmax, m);
      h.f_center = double(h.kc) / dur;
      h.offset = coff; coff += m;
      h.woff = woff; h.goff = woff; woff += len;
      h.wid = wident[size_t(pl)];
      // the window (App. A), unit l2 energy over the unclipped support (Eq. 5 :63, R3, R8)
      const size_t base = hp.win.size();
      hp.win.resize(base + size_t(len));
      long double energy = 0.0L;
      for (int64_t j = -h.dk; j <= h.dk; ++j) {
        const double raw = window_value(wtype[size_t(pl)], wpar[size_t(pl)], j, h.dk);
        hp.win[base + size_t(j + h.dk)] = raw;
        energy += (long double)raw * (long double)raw;
      }
      h.norm = double(1.0L / sqrtl(energy));
      hp.rows.push_back(h);
    }
  }
  hp.ctot = coff; hp.sumL = woff; hp.Mmax = mmax;
  if (hp.sumL >= (int64_t(1) << 31) || hp.ctot >= (int64_t(1) << 40)) return QTAM_ERR_UNSUPPORTED;

  // frame operator (C36 :536), cover sets (R9), joint and per plane (R10); out-of-range bins clipped (R8)
  const size_t nsets = size_t(nQ) + 1;
  std::vector<std::vector<long double>> acc(nsets, std::vector<long double>(size_t(hp.nb), 0.0L));
  hp.cover.assign(nsets, std::vector<uint8_t>(size_t(hp.nb), 0));
  std::vector<int32_t> count(size_t(hp.nb) * nsets + 1, 0);   // per (bin, plane) entry counts
  for (const HostRow &h : hp.rows) {
    for (int64_t j = -h.dk; j <= h.dk; ++j) {
      const int64_t f = h.kc + j;
      if (f < 0 || f >= hp.nb) continue;
      const double raw = hp.win[size_t(h.woff + j + h.dk)];
      const long double w = (long double)(raw * h.norm);
      acc[0][size_t(f)] += w * w;
      acc[size_t(h.plane) + 1][size_t(f)] += w * w;
      if (raw >= o.cover_floor) {
        hp.cover[0][size_t(f)] = 1;
        hp.cover[size_t(h.plane) + 1][size_t(f)] = 1;
      }
      count[size_t(f) * nsets + size_t(h.plane)] += 1;
    }
  }
  // normalise the stored windows now that the raw values have been used for the cover test
  for (const HostRow &h : hp.rows)
    for (int64_t i = 0; i < h.L; ++i) hp.win[size_t(h.woff + i)] *= h.norm;

  hp.P.assign(nsets, std::vector<double>(size_t(hp.nb), 0.0));
  for (size_t s = 0; s < nsets; ++s)
    for (int64_t f = 0; f < hp.nb; ++f) hp.P[s][size_t(f)] = double(acc[s][size_t(f)]);

  hp.cover_lo = hp.cover_hi = -1;
  int64_t ncov = 0;
  hp.frame_A = 0; hp.frame_B = 0;
  for (int64_t f = 0; f < hp.nb; ++f) {
    hp.frame_B = std::max(hp.frame_B, hp.P[0][size_t(f)]);
    if (!hp.cover[0][size_t(f)]) continue;
    if (hp.cover_lo < 0) { hp.cover_lo = f; hp.frame_A = hp.P[0][size_t(f)]; }
    hp.cover_hi = f; ++ncov;
    hp.frame_A = std::min(hp.frame_A, hp.P[0][size_t(f)]);
  }
  if (ncov == 0) return QTAM_ERR_EMPTY_FRAME;
  hp.holes = (hp.cover_hi - hp.cover_lo + 1) - ncov;

  // CSR: exclusive scan of the counts, then fill in row order (rows are plane-major, so the entries
  // of one (bin, plane) cell are in ascending row order: a fixed summation order)
  hp.csr_ptr.assign(size_t(hp.nb) * nsets + 1, 0);
  {
    // count[] was indexed [f*nsets + plane] with nsets = nP+1 slots per bin; slot nP is unused (0)
    int64_t run = 0;
    for (size_t i = 0; i < size_t(hp.nb) * nsets; ++i) {
      hp.csr_ptr[i] = int32_t(run);
      run += count[i];
    }
    hp.csr_ptr[size_t(hp.nb) * nsets] = int32_t(run);
    hp.csr_idx.assign(size_t(run), 0);
    std::vector<int32_t> fill(hp.csr_ptr.begin(), hp.csr_ptr.end() - 1);
    for (const HostRow &h : hp.rows)
      for (int64_t j = -h.dk; j <= h.dk; ++j) {
        const int64_t f = h.kc + j;
        if (f < 0 || f >= hp.nb) continue;
        hp.csr_idx[size_t(fill[size_t(f) * nsets + size_t(h.plane)]++)] = int32_t(h.goff + j + h.dk);
      }
  }
  return QTAM_OK;
}

}  // namespace qtam
