// api.cu -- the C ABI of libqtam (include/qtam.h): plan life cycle, argument checks, dispatch.
#include <algorithm>
#include <cmath>
#include <cstdlib>
#include <cstring>
#include <new>
#include <utility>
#include <vector>

#include "cplx.cuh"
#include "device_plan.hpp"

namespace qtam {
int generic_class_of(int log2M2);
}

using namespace qtam;

namespace {

int ilog2(long long v) { int l = 0; while ((1LL << l) < v) ++l; return l; }

template <typename T> bool upload(T **dst, const void *src, size_t count, size_t *total) {
  *dst = nullptr;
  if (count == 0) count = 1;
  if (cudaMalloc(reinterpret_cast<void **>(dst), count * sizeof(T)) != cudaSuccess) return false;
  *total += count * sizeof(T);
  if (src && cudaMemcpy(*dst, src, count * sizeof(T), cudaMemcpyHostToDevice) != cudaSuccess) return false;
  return true;
}

bool dev_alloc(void **dst, size_t bytes, size_t *total) {
  *dst = nullptr;
  if (bytes == 0) bytes = 16;
  if (cudaMalloc(dst, bytes) != cudaSuccess) return false;
  *total += bytes;
  return true;
}

void free_plan(qtam_plan *p) {
  if (!p) return;
  if (p->host_only) { delete p; return; }
  cudaFree(p->d_rows); cudaFree(p->d_win); cudaFree(p->d_invP);
  if (p->d_twN != p->d_tw) cudaFree(p->d_twN);
  cudaFree(p->d_tw); cudaFree(p->d_ws3);
  cudaFree(p->d_csr_ptr); cudaFree(p->d_csr_idx); cudaFree(p->d_plane_off);
  for (int c = 0; c < qtam_plan::kClasses; ++c) { cudaFree(p->d_items[c]); cudaFree(p->d_items_fwd[c]); }
  cudaFree(p->d_gfol_ptr); cudaFree(p->d_gfol_off); cudaFree(p->d_gfol_woff);
  cudaFree(p->d_bigrows); cudaFree(p->d_spec_alloc); cudaFree(p->d_ws); cudaFree(p->d_band);
  cudaFree(p->d_fwinp); cudaFree(p->d_red);
  cudaFree(p->d_frows); cudaFree(p->d_fwin); cudaFree(p->d_ftw_fwd); cudaFree(p->d_ftw_inv);
  cudaFree(p->d_tiny); cudaFree(p->d_ptw); cudaFree(p->d_ptw_long); cudaFree(p->d_frows_fwd); cudaFree(p->d_fmem); cudaFree(p->d_tmem);
  cudaFree(p->d_thr_tasks); cudaFree(p->d_thr_offs);
  for (int c = 0; c < kCtaClasses; ++c) { cudaFree(p->d_cta_lead[c]); cudaFree(p->d_ptw_rows[c]); cudaFree(p->d_cta_groups[c]); cudaFree(p->d_cta_mem[c]); }
  cudaFree(p->d_sp_tw2);
  for (int c = 0; c < kClClasses; ++c) { cudaFree(p->d_sp_ftw[c]); cudaFree(p->d_sp_scratch[c]); cudaFree(p->d_sp_ctl[c]); cudaFree(p->d_sp_order[c]); cudaFree(p->d_sp_wt[c]); cudaFree(p->d_sp_wtoff[c]); }
  cudaFree(p->d_sp_xt); cudaFree(p->d_ptw_mid); cudaFree(p->d_tw_2k);
  for (int c = 0; c < kClClasses; ++c) { cudaFree(p->d_cl_lead[c]); cudaFree(p->d_cl_mem[c]); cudaFree(p->d_cl_groups[c]); cudaFree(p->d_cl_ftw[c]); }
  cudaFree(p->d_cl_ptw);
  cudaFree(p->d_runs); cudaFree(p->d_run_ptr); cudaFree(p->d_run_idx);
  cudaFree(p->d_len_tw[0]); cudaFree(p->d_len_tw[1]); cudaFree(p->d_ccl_area);
  cudaFree(p->d_trows); cudaFree(p->d_titems); cudaFree(p->d_part); cudaFree(p->d_counter);
  for (ProfRec &r : p->prof_pool) { cudaEventDestroy(r.e0); cudaEventDestroy(r.e1); }
  for (int i = 0; i < p->n_side; ++i) { cudaStreamDestroy(p->side[i]); cudaEventDestroy(p->ev_join[i]); }
  if (p->ev_fork) cudaEventDestroy(p->ev_fork);
  delete p;
}

// e^{+2 pi i k/n} for k = 0..n-1, evaluated in long double from the first octant (exact symmetries)
template <typename T> void fill_twiddles(std::vector<T> &tw, int64_t n) {
  tw.resize(size_t(2 * n));
  const long double tau = 6.283185307179586476925286766559005768L;
  for (int64_t k = 0; k < n; ++k) {
    long double c, s;
    // quarter-turn reduction keeps the argument of cosl/sinl in [0, pi/2)
    const int64_t quarter = n / 4;
    const int64_t qq = k / quarter, rr = k % quarter;
    long double ang = tau * (long double)rr / (long double)n;
    long double c0 = cosl(ang), s0 = sinl(ang);
    if (rr == 0) { c0 = 1.0L; s0 = 0.0L; }
    if (2 * rr == quarter) { c0 = s0 = 0.707106781186547524400844362104849039L; }
    switch (qq & 3) {
      case 0: c = c0; s = s0; break;
      case 1: c = -s0; s = c0; break;
      case 2: c = -c0; s = -s0; break;
      default: c = s0; s = -c0; break;
    }
    tw[size_t(2 * k)] = (T)c;
    tw[size_t(2 * k + 1)] = (T)s;
  }
}

// tables of the fast float path (fast.cu)
qtam_status build_fast(qtam_plan *p) {
  const HostPlan &hp = p->hp;
  size_t *tot = &p->device_bytes;
  FastParams &F = p->fast;
  std::memset(&F, 0, sizeof(F));
  // one window per distinct half-width (the clamped rows all share one)
  std::vector<float> fwin;
  std::vector<std::pair<int64_t, int>> seen;   // (dk and window identity, offset)
  // the pair (half-width, window identity) as one key: wid is a plane index, so nP + 1 keeps any number of planes apart
  const int64_t wid_span = (int64_t)hp.nP + 1;
  auto wkey = [wid_span](const HostRow &h) -> int64_t { return h.dk * wid_span + h.wid; };
  auto window_of = [&](const HostRow &h) -> int {
    for (auto &e : seen) if (e.first == wkey(h)) return e.second;
    const int off = (int)fwin.size();
    for (int64_t i = 0; i < h.L; ++i) fwin.push_back((float)hp.win[(size_t)(h.woff + i)]);
    seen.push_back({wkey(h), off});
    return off;
  };
  // the same windows zero-padded to the M points of the row's short FFT and stored at the M-array
  // index (j mod M): the fast gather multiplies without testing the support
  std::vector<float> fwinp;
  std::vector<std::pair<int64_t, int>> seen2;
  auto wpad_of = [&](const HostRow &h) -> int {
    for (auto &e : seen2) if (e.first == wkey(h)) return e.second;
    const int off = (int)fwinp.size();
    fwinp.resize(fwinp.size() + (size_t)h.M, 0.0f);
    for (int64_t jj = -h.dk; jj <= h.dk; ++jj)
      fwinp[(size_t)(off + (jj + h.M) % h.M)] = (float)hp.win[(size_t)(h.woff + jj + h.dk)];
    seen2.push_back({wkey(h), off});
    return off;
  };
  std::vector<FastRow> frows;
  std::vector<int4> red;
  // forward table: rows of one bucket with the same centre bin and half-width (the clamped rows of
  // different Q-planes, A7/A8 :307-311: one window for all of them) have identical coefficients, so
  // the forward transforms one "leader" per such set and stores the result at every member's offset.
  // Leader records reuse FastRow: plane = number of members, pad = first entry in the member table.
  FastParams &FF = p->fast_fwd;
  std::memset(&FF, 0, sizeof(FF));
  std::vector<FastRow> frowsF;
  std::vector<int> fmem;
  std::vector<float> twf, twi;   // (wx, wy) per entry
  const long double tau = 6.283185307179586476925286766559005768L;
  for (int lg = 5; lg >= 0; --lg) {
    const int G = 1 << lg, M = 32 * G, Fr = 32 / G;
    FastBucket B{};
    B.log2G = lg; B.row_base = (int)frows.size(); B.tw_base = (int)(twf.size() / 2);
    std::vector<FastRow> leaders;
    std::vector<std::vector<int>> members;
    for (size_t k = 0; k < hp.rows.size(); ++k) {
      const HostRow &h = hp.rows[k];
      if (h.M != M) continue;
      FastRow r{};
      r.kc = (int)h.kc; r.dk = (int)h.dk; r.woff = window_of(h); r.goff = (int)h.goff;
      r.offset = (int)h.offset; r.plane = h.plane; r.wpad = wpad_of(h);
      frows.push_back(r);
      {
        size_t l = 0;
        // identical rows: same centre bin, half-width and window (the same entry of the window table)
        while (l < leaders.size() && !(leaders[l].kc == r.kc && leaders[l].dk == r.dk && leaders[l].woff == r.woff)) ++l;
        if (l == leaders.size()) { leaders.push_back(r); members.emplace_back(); }
        members[l].push_back(r.offset);
      }
      {
        const int64_t lo = h.kc - h.dk;
        const int64_t jb = lo < 0 ? -lo : 0, je = std::min<int64_t>(h.L, hp.nb - lo);
        red.push_back(make_int4((int)(lo + jb), (int)std::max<int64_t>(je - jb, 0), (int)jb, h.plane));
      }
      F.sum_M += (double)h.M; F.sum_L += (double)h.L;
    }
    B.nrows = (int)frows.size() - B.row_base;
    if (B.nrows == 0) continue;
    B.ngroups = (B.nrows + Fr - 1) / Fr;
    FastBucket BF = B;
    BF.row_base = (int)frowsF.size();
    BF.nrows = (int)leaders.size();
    BF.ngroups = (BF.nrows + Fr - 1) / Fr;
    for (size_t l = 0; l < leaders.size(); ++l) {
      leaders[l].plane = (int)members[l].size();
      leaders[l].pad = (int)fmem.size();
      fmem.insert(fmem.end(), members[l].begin(), members[l].end());
      frowsF.push_back(leaders[l]);
    }
    const double sf = 1.0 / std::sqrt((double)hp.N * (double)M), si = std::sqrt((double)hp.N / (double)M);
    for (int n1 = 0; n1 < 32; ++n1)
      for (int t = 0; t < G; ++t) {
        const int m = (n1 * t) % M;
        const long double a = tau * (long double)m / (long double)M;
        const double c = (double)cosl(a), s = (double)sinl(a);
        twf.push_back((float)(c * sf)); twf.push_back((float)(s * sf));
        twi.push_back((float)(c * si)); twi.push_back((float)(-s * si));
      }
    F.groups_per_seg += B.ngroups;
    F.b[F.nbuckets++] = B;
    FF.groups_per_seg += BF.ngroups;
    FF.b[FF.nbuckets++] = BF;
  }
  F.tw_total = (int)(twf.size() / 2);
  F.rows_smem = frows.size() <= 1024 ? (int)frows.size() : 0;
  FF.tw_total = F.tw_total; FF.sum_M = F.sum_M; FF.sum_L = F.sum_L;
  FF.rows_smem = frowsF.size() <= 1024 ? (int)frowsF.size() : 0;
  // rows shorter than 32 points
  std::vector<FastRow> tiny;
  for (size_t k = 0; k < hp.rows.size(); ++k) {
    const HostRow &h = hp.rows[k];
    if (h.M >= 32) continue;
    FastRow r{};
    r.kc = (int)h.kc; r.dk = (int)h.dk; r.woff = window_of(h); r.goff = ilog2(h.M);
    r.offset = (int)h.offset; r.plane = h.plane; r.wpad = (int)h.goff;   // wpad: band offset (tiny rows)
    p->tiny_sumM += (double)h.M; p->tiny_sumL += (double)h.L;
    tiny.push_back(r);
  }
  p->n_tiny = (int)tiny.size();
  if (!upload(&p->d_tiny, tiny.data(), tiny.size(), tot)) return QTAM_ERR_ALLOC;
  if (!upload(&p->d_frows, frows.data(), frows.size(), tot)) return QTAM_ERR_ALLOC;
  p->h_frows = frows;
  if (!upload(&p->d_frows_fwd, frowsF.data(), frowsF.size(), tot)) return QTAM_ERR_ALLOC;
  if (!upload(&p->d_fmem, fmem.data(), fmem.size(), tot)) return QTAM_ERR_ALLOC;
  float *d = nullptr;
  if (!upload(&d, fwin.data(), fwin.size(), tot)) return QTAM_ERR_ALLOC;
  p->d_fwin = d;
  if (!upload(&d, fwinp.data(), fwinp.size(), tot)) return QTAM_ERR_ALLOC;
  p->d_fwinp = d;
  if (!upload(&p->d_red, red.data(), red.size(), tot)) return QTAM_ERR_ALLOC;
  if (!upload(&d, twf.data(), twf.size(), tot)) return QTAM_ERR_ALLOC;
  p->d_ftw_fwd = d;
  if (!upload(&d, twi.data(), twi.size(), tot)) return QTAM_ERR_ALLOC;
  p->d_ftw_inv = d;
  return QTAM_OK;
}

template <typename T> qtam_status build_device(qtam_plan *p) {
  const HostPlan &hp = p->hp;
  size_t *tot = &p->device_bytes;
  // rows
  std::vector<RowDev> rd(hp.rows.size());
  for (size_t k = 0; k < hp.rows.size(); ++k) {
    const HostRow &h = hp.rows[k];
    RowDev &d = rd[k];
    d.kc = (int)h.kc; d.dk = (int)h.dk; d.M = (int)h.M; d.log2M = ilog2(h.M);
    d.plane = h.plane; d.pad0 = 0; d.offset = h.offset; d.woff = h.woff;
    d.fwd_scale = 1.0 / std::sqrt((double)hp.N * (double)h.M);
    d.inv_amp = std::sqrt((double)hp.N / (double)h.M);
  }
  if (!upload(&p->d_rows, rd.data(), rd.size(), tot)) return QTAM_ERR_ALLOC;
  // windows, rounded once to the plan's dtype
  {
    std::vector<T> w(hp.win.size());
    for (size_t i = 0; i < w.size(); ++i) w[i] = (T)hp.win[i];
    T *d = nullptr;
    if (!upload(&d, w.data(), w.size(), tot)) return QTAM_ERR_ALLOC;
    p->d_win = d;
  }
  // twiddles
  {
    std::vector<T> tw;
    fill_twiddles<T>(tw, p->twn);
    T *d = nullptr;
    if (!upload(&d, tw.data(), tw.size(), tot)) return QTAM_ERR_ALLOC;
    p->d_tw = d;
    p->d_twN = d;
    if (!p->n_pow2) {
      // e^{2 pi i k/N} for the steps whose period is the segment length (radix-3 combine, real pre / post-processing)
      fill_twiddles<T>(tw, hp.N);
      if (!upload(&d, tw.data(), tw.size(), tot)) return QTAM_ERR_ALLOC;
      p->d_twN = d;
      if (!dev_alloc(&p->d_ws3, 2 * 2 * sizeof(T) * size_t(p->max_batch) * size_t(hp.N), tot)) return QTAM_ERR_ALLOC;
    }
  }
  // 1/P on the cover set, 0 elsewhere (a7; R9)
  {
    const size_t nsets = size_t(hp.nP) + 1;
    std::vector<T> ip(nsets * size_t(hp.nb));
    for (size_t s = 0; s < nsets; ++s)
      for (int64_t f = 0; f < hp.nb; ++f)
        ip[s * size_t(hp.nb) + size_t(f)] = hp.cover[s][size_t(f)] ? (T)(1.0 / hp.P[s][size_t(f)]) : (T)0;
    T *d = nullptr;
    if (!upload(&d, ip.data(), ip.size(), tot)) return QTAM_ERR_ALLOC;
    p->d_invP = d;
  }
  {
    std::vector<long long> po(size_t(hp.nP) + 1, hp.ctot);
    for (size_t k = hp.rows.size(); k-- > 0;) po[size_t(hp.rows[k].plane)] = hp.rows[k].offset;
    if (!upload(&p->d_plane_off, po.data(), po.size(), tot)) return QTAM_ERR_ALLOC;
    for (int q = 0; q < hp.nP; ++q) p->max_plane_coeffs = std::max(p->max_plane_coeffs, po[size_t(q) + 1] - po[size_t(q)]);
  }
  if (!upload(&p->d_csr_ptr, hp.csr_ptr.data(), hp.csr_ptr.size(), tot)) return QTAM_ERR_ALLOC;
  if (!upload(&p->d_csr_idx, hp.csr_idx.data(), hp.csr_idx.size(), tot)) return QTAM_ERR_ALLOC;
  // generic-path work lists
  {
    std::vector<WorkItem> items[qtam_plan::kClasses], items_fwd[qtam_plan::kClasses];
    std::vector<int> big;
    std::vector<std::vector<long long>> followers(hp.rows.size());   // per leader row: follower offsets
    std::vector<std::vector<long long>> followers_w(hp.rows.size()); // ... and their band offsets
    std::vector<int> gen_leaders;                                    // single-transform rows seen so far
    for (size_t k = 0; k < hp.rows.size(); ++k) {
      const int lm = ilog2(hp.rows[k].M);
      if (p->fast_rows && lm <= 10) continue;   // handled by fast.cu (32..1024: warp engine; < 32: one thread per row)
      if (p->fast_rows && lm >= kCtaLog2Min && lm <= kCtaLog2Max) continue;   // rows_cta.cu, rows_cluster.cu
      if (lm <= p->cap_log2) {
        const int c = generic_class_of(lm);
        items[c].push_back(WorkItem{(int)k, 0, 1, lm});
        {
          // forward: identical rows (same centre bin and half-width) are transformed once
          int leader = -1;
          for (int l : gen_leaders)
            if (hp.rows[(size_t)l].kc == hp.rows[k].kc && hp.rows[(size_t)l].dk == hp.rows[k].dk &&
                hp.rows[(size_t)l].M == hp.rows[k].M && hp.rows[(size_t)l].wid == hp.rows[k].wid) { leader = l; break; }
          if (leader < 0) { gen_leaders.push_back((int)k); items_fwd[c].push_back(WorkItem{(int)k, 0, 1, lm}); }
          else { followers[(size_t)leader].push_back(hp.rows[k].offset); followers_w[(size_t)leader].push_back(hp.rows[k].woff); }
        }
        p->class_L[c] += (double)hp.rows[k].L; p->class_M[c] += (double)hp.rows[k].M;
      } else {
        const int R1 = 1 << (lm - p->cap_log2);
        if (R1 > 16) return QTAM_ERR_UNSUPPORTED;
        for (int j1 = 0; j1 < R1; ++j1)
          {
            items[generic_class_of(p->cap_log2)].push_back(WorkItem{(int)k, j1, R1, p->cap_log2});
            items_fwd[generic_class_of(p->cap_log2)].push_back(WorkItem{(int)k, j1, R1, p->cap_log2});
          }
        big.push_back((int)k);
        p->class_L[generic_class_of(p->cap_log2)] += (double)hp.rows[k].L;
        p->class_M[generic_class_of(p->cap_log2)] += (double)hp.rows[k].M;
        p->big_M += (double)hp.rows[k].M;
        if (R1 > p->big_R1max) p->big_R1max = R1;
      }
    }
    for (int c = 0; c < qtam_plan::kClasses; ++c) {
      // largest first: the tail of the launch is then made of the short rows
      std::stable_sort(items[c].begin(), items[c].end(),
                       [](const WorkItem &a, const WorkItem &b) { return a.log2M2 > b.log2M2; });
      p->n_items[c] = (int)items[c].size();
      if (!upload(&p->d_items[c], items[c].data(), items[c].size(), tot)) return QTAM_ERR_ALLOC;
      std::stable_sort(items_fwd[c].begin(), items_fwd[c].end(),
                       [](const WorkItem &a, const WorkItem &b) { return a.log2M2 > b.log2M2; });
      p->n_items_fwd[c] = (int)items_fwd[c].size();
      if (!upload(&p->d_items_fwd[c], items_fwd[c].data(), items_fwd[c].size(), tot)) return QTAM_ERR_ALLOC;
    }
    {
      std::vector<int> fptr(hp.rows.size() + 1, 0);
      std::vector<long long> foff, fwoff;
      for (size_t k = 0; k < hp.rows.size(); ++k) {
        fptr[k] = (int)foff.size();
        foff.insert(foff.end(), followers[k].begin(), followers[k].end());
        fwoff.insert(fwoff.end(), followers_w[k].begin(), followers_w[k].end());
      }
      fptr[hp.rows.size()] = (int)foff.size();
      if (!upload(&p->d_gfol_ptr, fptr.data(), fptr.size(), tot)) return QTAM_ERR_ALLOC;
      if (!upload(&p->d_gfol_off, foff.data(), foff.size(), tot)) return QTAM_ERR_ALLOC;
      if (!upload(&p->d_gfol_woff, fwoff.data(), fwoff.size(), tot)) return QTAM_ERR_ALLOC;
    }
    p->n_bigrows = (int)big.size();
    if (!upload(&p->d_bigrows, big.data(), big.size(), tot)) return QTAM_ERR_ALLOC;
  }
  // workspace
  const size_t csz = 2 * sizeof(T);
  {
    // every segment's spectrum has kSpecPad zero bins before and after it, so that the fast gather can
    // read a full M-point neighbourhood of any centre bin without bounds checks (R8 clipping for free)
    const size_t bytes = csz * (size_t(p->max_batch) * size_t(p->xstride) + 2 * size_t(kSpecPad));
    if (!dev_alloc(&p->d_spec_alloc, bytes, tot)) return QTAM_ERR_ALLOC;
    if (cudaMemset(p->d_spec_alloc, 0, bytes) != cudaSuccess) return QTAM_ERR_CUDA;
    p->d_spec = static_cast<char *>(p->d_spec_alloc) + csz * size_t(kSpecPad);
  }
  if (!dev_alloc(&p->d_ws, csz * size_t(p->max_batch) * size_t(hp.N), tot)) return QTAM_ERR_ALLOC;
  if (!dev_alloc(&p->d_band, csz * size_t(p->max_batch) * size_t(hp.sumL), tot)) return QTAM_ERR_ALLOC;
  return QTAM_OK;
}

bool check_call(const qtam_plan *p, const void *a, const void *b, int batch) {
  if (!(p && !p->host_only && a && b && batch >= 0 && batch <= p->max_batch)) return false;
  cudaGetLastError();   // clear a stale error of an earlier (foreign) call: the launch checks below report only ours
  return true;
}

}  // namespace

extern "C" {

qtam_status qtam_plan_create(qtam_plan **out, double fs, int64_t N, const double *Q, int nQ,
                             double fmin, double fmax, double spacing, qtam_dtype dtype,
                             const qtam_options *opt) {
  if (!out) return QTAM_ERR_INVALID_ARG;
  qtam_plan *p = new (std::nothrow) qtam_plan;
  if (!p) return QTAM_ERR_ALLOC;
  qtam_status s = build_host_plan(p->hp, fs, N, Q, nQ, fmin, fmax, spacing, dtype, opt);
  if (s != QTAM_OK) { delete p; return s; }
  // the batch index is a grid dimension (y or z) of several kernels: 65535 at most
  if (p->hp.opt.max_batch > 65535) { delete p; return QTAM_ERR_INVALID_ARG; }
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) { delete p; return QTAM_ERR_CUDA; }
  p->esz = dtype == QTAM_F32 ? 4 : 8;
  p->max_batch = p->hp.opt.max_batch;
  p->xstride = ((p->hp.nb + kSpecPad + 31) / 32) * 32;
  p->n_pow2 = (N & (N - 1)) == 0;
  // power-of-two periods come from tw (short FFTs of up to nextpow2(N/2 + 1) points, the power-of-two part of
  // the long transform); for N = 3 * 2^k that is a table of 2^(k+1) entries
  p->twn = p->n_pow2 ? N : (N / 3) * 2;
  p->sub_n = p->n_pow2 ? N / 2 : N / 6;
  p->cap_log2 = dtype == QTAM_F32 ? 13 : 12;
  {
    int dev = 0, sms = 148;
    if (cudaGetDevice(&dev) == cudaSuccess &&
        cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) == cudaSuccess && sms > 0)
      p->num_sms = sms;
    const int lnc = p->n_pow2 ? ilog2(N) - 1 : -1;     // the tuned long transforms take N = 2^k only
    // the tuned float kernels keep coefficient offsets in 32-bit integers; a plan with more coefficients per
    // segment runs every row in the generic kernels (64-bit offsets)
    p->fast_rows = dtype == QTAM_F32 && p->hp.ctot < (int64_t(1) << 31);
    p->fast_long = dtype == QTAM_F32 && lnc >= 11 && lnc <= 14;
  }
  cudaGetLastError();   // an error left behind by an earlier library call is not this plan's
  s = dtype == QTAM_F32 ? build_device<float>(p) : build_device<double>(p);
  if (s == QTAM_OK) s = prepare_generic(p);
  if (s == QTAM_OK) s = build_thr_fast(p);
  if (s == QTAM_OK && p->fast_rows) s = build_fast(p);
  if (s == QTAM_OK && p->fast_long) s = build_long_tables(p);
  if (s == QTAM_OK && p->fast_rows) s = build_long_fft(p);
  // the inverse's partial sums, in summation order: tiles, CTA groups, cluster groups (then the band slots)
  if (s == QTAM_OK && p->fast_rows) s = build_inv_tiled(p);
  if (s == QTAM_OK && p->fast_rows) s = build_rows_cta(p);
  if (s == QTAM_OK && p->fast_rows) s = build_rows_2k(p);
  if (s == QTAM_OK && p->fast_rows) s = build_rows_cluster(p);
  if (s == QTAM_OK && p->fast_rows) s = build_runs(p);
  if (s == QTAM_OK) s = prepare_fast(p);
  if (s == QTAM_OK) s = build_length(p);
  if (s == QTAM_OK) s = build_cluster(p);
  if (s == QTAM_OK && (p->cta_rows || p->cl_rows)) {
    // side streams for the concurrent row launches (plans whose rows run in several kernels)
    if (cudaEventCreateWithFlags(&p->ev_fork, cudaEventDisableTiming) != cudaSuccess) s = QTAM_ERR_CUDA;
    for (int i = 0; s == QTAM_OK && i < qtam_plan::kSide; ++i) {
      if (cudaStreamCreateWithFlags(&p->side[i], cudaStreamNonBlocking) != cudaSuccess ||
          cudaEventCreateWithFlags(&p->ev_join[i], cudaEventDisableTiming) != cudaSuccess) s = QTAM_ERR_CUDA;
      else p->n_side = i + 1;
    }
  }
  if (s != QTAM_OK) { free_plan(p); cudaGetLastError(); return s; }
  if (cudaDeviceSynchronize() != cudaSuccess) { free_plan(p); return QTAM_ERR_CUDA; }
  *out = p;
  return QTAM_OK;
}

qtam_status qtam_plan_create_host(qtam_plan **out, double fs, int64_t N, const double *Q, int nQ,
                                  double fmin, double fmax, double spacing, qtam_dtype dtype,
                                  const qtam_options *opt) {
  if (!out) return QTAM_ERR_INVALID_ARG;
  qtam_plan *p = new (std::nothrow) qtam_plan;
  if (!p) return QTAM_ERR_ALLOC;
  qtam_status s = build_host_plan(p->hp, fs, N, Q, nQ, fmin, fmax, spacing, dtype, opt);
  if (s != QTAM_OK) { delete p; return s; }
  p->esz = dtype == QTAM_F32 ? 4 : 8;
  p->max_batch = 0;            // no workspace: every compute call is refused
  p->host_only = true;
  *out = p;
  return QTAM_OK;
}

qtam_status qtam_plan_destroy(qtam_plan *p) {
  if (!p) return QTAM_ERR_INVALID_ARG;
  free_plan(p);
  return QTAM_OK;
}

qtam_status qtam_plan_info(const qtam_plan *p, qtam_info *o) {
  if (!p || !o) return QTAM_ERR_INVALID_ARG;
  const HostPlan &hp = p->hp;
  o->n_planes = hp.nP; o->n_rows = (int)hp.rows.size(); o->n = hp.N; o->n_bins = hp.nb;
  o->coeffs_per_segment = hp.ctot; o->sum_L = hp.sumL;
  o->cover_lo = hp.cover_lo; o->cover_hi = hp.cover_hi; o->holes = hp.holes;
  o->frame_A = hp.frame_A; o->frame_B = hp.frame_B;
  o->workspace_bytes = p->device_bytes;
  return QTAM_OK;
}

qtam_status qtam_plan_rows(const qtam_plan *p, qtam_row *out, int capacity) {
  if (!p || !out || capacity < (int)p->hp.rows.size()) return QTAM_ERR_INVALID_ARG;
  for (size_t k = 0; k < p->hp.rows.size(); ++k) {
    const HostRow &h = p->hp.rows[k];
    qtam_row &o = out[k];
    o.plane = h.plane; o.row = h.row; o.q = h.q; o.f_request = h.f_request; o.f_center = h.f_center;
    o.kc = h.kc; o.dk = h.dk; o.L = h.L; o.M = h.M; o.offset = h.offset; o.norm = h.norm;
  }
  return QTAM_OK;
}

qtam_status qtam_plan_window(const qtam_plan *p, int row, double *out) {
  if (!p || !out || row < 0 || row >= (int)p->hp.rows.size()) return QTAM_ERR_INVALID_ARG;
  const HostRow &h = p->hp.rows[(size_t)row];
  std::memcpy(out, p->hp.win.data() + h.woff, sizeof(double) * (size_t)h.L);
  return QTAM_OK;
}

qtam_status qtam_plan_frame(const qtam_plan *p, int plane, double *P_out, uint8_t *cover_out) {
  if (!p || plane < -1 || plane >= p->hp.nP) return QTAM_ERR_INVALID_ARG;
  const size_t s = (size_t)(plane + 1);
  if (P_out) std::memcpy(P_out, p->hp.P[s].data(), sizeof(double) * (size_t)p->hp.nb);
  if (cover_out) std::memcpy(cover_out, p->hp.cover[s].data(), (size_t)p->hp.nb);
  return QTAM_OK;
}

qtam_status qtam_forward(qtam_plan *p, const void *d_x, int batch, void *d_coef, void *stream) {
  if (p && p->host_only) return QTAM_ERR_CUDA;
  if (!check_call(p, d_x, d_coef, batch)) return QTAM_ERR_INVALID_ARG;
  p->last_launches = 0;
  if (batch == 0) return QTAM_OK;
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  qtam_status s = p->fast_long ? fast_r2c(p, d_x, batch, st) : generic_r2c(p, d_x, batch, st);
  if (s != QTAM_OK) return s;
  // the row launches are independent of each other (they read the spectrum and write disjoint coefficients):
  // the longest rows first, every launch on a stream of its own, joined before the call returns to the caller's
  Fork fk(p, st);
  if (p->cl_rows) s = cluster_forward_rows(p, batch, d_coef, fk);
  if (s == QTAM_OK && p->cta_rows) s = cta_forward_rows(p, batch, d_coef, fk);
  if (s == QTAM_OK && p->fast_rows) s = fast_forward_rows(p, batch, d_coef, st);
  if (s == QTAM_OK) s = generic_forward_rows(p, batch, d_coef, st);
  fk.join();
  return s;
}

qtam_status qtam_forward_threshold(qtam_plan *p, const void *d_x, int batch, double kappa, void *d_coef,
                                   void *stream) {
  if (p && p->host_only) return QTAM_ERR_CUDA;
  if (!check_call(p, d_x, d_coef, batch) || !(kappa >= 0.0)) return QTAM_ERR_INVALID_ARG;
  p->last_launches = 0;
  if (batch == 0) return QTAM_OK;
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  if (p->fast_rows && p->esz == 4) {
    // the threshold rides in the epilogue of the row kernel for every row of at most 1024 points
      qtam_status s = p->fast_long ? fast_r2c(p, d_x, batch, st) : generic_r2c(p, d_x, batch, st);
      if (s != QTAM_OK) return s;
    bool fused = false;
    s = fast_forward_rows_threshold(p, batch, d_coef, (float)kappa, st, &fused);
    if (s != QTAM_OK) return s;
    if (fused) {
      Fork fk(p, st);
      if (p->cl_rows) s = cluster_forward_rows(p, batch, d_coef, fk);
      if (s == QTAM_OK && p->cta_rows) s = cta_forward_rows(p, batch, d_coef, fk);
      fk.join();
      if (s != QTAM_OK) return s;
      s = generic_forward_rows(p, batch, d_coef, st);
      if (s != QTAM_OK || !p->thr_has_big) return s;
      return generic_threshold(p, d_coef, batch, kappa, kThrFastLog2Max + 1, st);   // rows longer than 1024 points
    }
    // not fusable for this plan / batch: the two steps one after the other
    s = fast_forward_rows(p, batch, d_coef, st);
    {
      Fork fk(p, st);
      if (s == QTAM_OK && p->cl_rows) s = cluster_forward_rows(p, batch, d_coef, fk);
      if (s == QTAM_OK && p->cta_rows) s = cta_forward_rows(p, batch, d_coef, fk);
      fk.join();
    }
    if (s == QTAM_OK) s = generic_forward_rows(p, batch, d_coef, st);
    if (s != QTAM_OK) return s;
    const int n1 = p->last_launches;
    s = qtam_threshold_rowmedian(p, d_coef, batch, kappa, stream);
    p->last_launches += n1;
    return s;
  }
  qtam_status s = qtam_forward(p, d_x, batch, d_coef, stream);
  if (s != QTAM_OK) return s;
  const int n1 = p->last_launches;
  s = qtam_threshold_rowmedian(p, d_coef, batch, kappa, stream);
  p->last_launches += n1;
  return s;
}

qtam_status qtam_inverse(qtam_plan *p, const void *d_coef, int batch, int plane, void *d_x_out,
                         void *stream) {
  if (p && p->host_only) return QTAM_ERR_CUDA;
  if (!check_call(p, d_coef, d_x_out, batch) || plane < -1 || plane >= p->hp.nP)
    return QTAM_ERR_INVALID_ARG;
  p->last_launches = 0;
  if (batch == 0) return QTAM_OK;
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  if (p->tiled_inv) return tiled_inverse(p, d_coef, batch, plane, d_x_out, st);
  qtam_status s = QTAM_OK;
  if (p->use_runs) {
    // float plans: every row kernel leaves its contributions as runs (tiles' and groups' partial sums, the band
    // slots of the shortest rows); one pass adds them, applies 1/P and prepares the long C2R
    // (independent launches, disjoint partial sums: forked onto the plan's side streams, the longest rows first)
    Fork fk(p, st);
    if (p->cl_rows) s = cluster_inverse_rows(p, d_coef, batch, plane, fk);
    if (s == QTAM_OK && p->cta_rows) s = cta_inverse_rows(p, d_coef, batch, plane, fk);
    if (s == QTAM_OK) s = p->tiles_ok ? tiles_only(p, d_coef, batch, plane, st) : fast_inverse_rows(p, d_coef, batch, plane, st);
    if (s == QTAM_OK) s = fast_tiny_inverse(p, d_coef, batch, plane, fk.next());
    if (s == QTAM_OK) s = generic_inverse_rows(p, d_coef, batch, plane, st);   // (no items on these plans)
    fk.join();
    if (s == QTAM_OK) s = combine_runs(p, batch, plane, st);
    if (s != QTAM_OK) return s;
    if (p->fast_long) return fast_c2c_out(p, batch, d_x_out, st);
    return generic_c2c_out(p, batch, d_x_out, st);
  }
  s = generic_inverse_rows(p, d_coef, batch, plane, st);
  if (s != QTAM_OK) return s;
  s = generic_inverse_reduce(p, batch, plane, st);
  if (s != QTAM_OK) return s;
  return generic_c2r(p, batch, d_x_out, st);
}

qtam_status qtam_dense(qtam_plan *p, const void *d_x, int batch, int row_begin, int row_end,
                       void *d_out, void *stream) {
  if (p && p->host_only) return QTAM_ERR_CUDA;
  if (!check_call(p, d_x, d_out, batch) || row_begin < 0 || row_end > (int)p->hp.rows.size() ||
      row_begin > row_end)
    return QTAM_ERR_INVALID_ARG;
  p->last_launches = 0;
  if (batch == 0 || row_begin == row_end) return QTAM_OK;
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  qtam_status s = p->fast_long ? fast_r2c(p, d_x, batch, st) : generic_r2c(p, d_x, batch, st);
  if (s != QTAM_OK) return s;
  return generic_dense(p, batch, row_begin, row_end, d_out, st);
}

qtam_status qtam_dense_invert(qtam_plan *p, const void *d_tile, int batch, int row, void *d_x_out, void *stream) {
  if (p && p->host_only) return QTAM_ERR_CUDA;
  if (!check_call(p, d_tile, d_x_out, batch) || row < 0 || row >= (int)p->hp.rows.size() ||
      !(p->hp.opt.epsilon > 0.0))
    return QTAM_ERR_INVALID_ARG;
  p->last_launches = 0;
  if (batch == 0) return QTAM_OK;
  return generic_dense_invert(p, d_tile, batch, row, d_x_out, static_cast<cudaStream_t>(stream));
}

int64_t qtam_plane_pixels(const qtam_plan *p, int plane) {
  long long off; int R, M;
  if (!p || plane < 0 || plane >= p->hp.nP || !plane_image(p, plane, &off, &R, &M)) return 0;
  return (int64_t)R * M;
}

qtam_status qtam_cluster(qtam_plan *p, const void *d_coef, int batch, int plane, int min_area, int32_t *d_labels,
                         int32_t *d_count, void *stream) {
  if (p && p->host_only) return QTAM_ERR_CUDA;
  if (!check_call(p, d_coef, d_labels, batch) || !d_count || plane < 0 || plane >= p->hp.nP || min_area < 1)
    return QTAM_ERR_INVALID_ARG;
  p->last_launches = 0;
  if (batch == 0) return QTAM_OK;
  return cluster_labels(p, d_coef, batch, plane, min_area, d_labels, d_count, static_cast<cudaStream_t>(stream));
}

qtam_status qtam_mask(qtam_plan *p, const void *d_coef, int batch, int plane, const int32_t *d_labels, int label,
                      void *d_out, void *stream) {
  if (p && p->host_only) return QTAM_ERR_CUDA;
  if (!check_call(p, d_coef, d_out, batch) || !d_labels || plane < 0 || plane >= p->hp.nP || label < 0)
    return QTAM_ERR_INVALID_ARG;
  p->last_launches = 0;
  if (batch == 0) return QTAM_OK;
  return cluster_mask(p, d_coef, batch, plane, d_labels, label, d_out, static_cast<cudaStream_t>(stream));
}

int64_t qtam_output_length(const qtam_plan *p, int mode) {
  if (!p) return 0;
  if (mode == 0) return p->host_only ? length_resolve(p->hp, p->hp.opt.out_length) : p->len_n;
  return mode == -1 || mode == -2 ? length_resolve(p->hp, mode) : 0;
}

qtam_status qtam_forward_length(qtam_plan *p, const void *d_x, int batch, void *d_img, void *stream) {
  if (p && p->host_only) return QTAM_ERR_CUDA;
  if (!check_call(p, d_x, d_img, batch) || p->len_n == 0) return QTAM_ERR_INVALID_ARG;
  p->last_launches = 0;
  if (batch == 0) return QTAM_OK;
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  const qtam_status s = p->fast_long ? fast_r2c(p, d_x, batch, st) : generic_r2c(p, d_x, batch, st);
  if (s != QTAM_OK) return s;
  return length_forward(p, batch, d_img, st);
}

qtam_status qtam_inverse_length(qtam_plan *p, const void *d_img, int batch, int plane, void *d_x_out, void *stream) {
  if (p && p->host_only) return QTAM_ERR_CUDA;
  if (!check_call(p, d_img, d_x_out, batch) || p->len_n == 0 || plane < -1 || plane >= p->hp.nP)
    return QTAM_ERR_INVALID_ARG;
  p->last_launches = 0;
  if (batch == 0) return QTAM_OK;
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  qtam_status s = length_inverse_bands(p, d_img, batch, plane, st);       // every row's windowed band (C49)
  if (s == QTAM_OK) s = generic_inverse_reduce(p, batch, plane, st);      // sum over rows, 1/P (Eq. 11)
  if (s == QTAM_OK) s = generic_c2r(p, batch, d_x_out, st);
  return s;
}

qtam_status qtam_resample(qtam_plan *p, const void *d_in, int batch, int to_standard, void *d_out, void *stream) {
  if (p && p->host_only) return QTAM_ERR_CUDA;
  if (!check_call(p, d_in, d_out, batch) || p->len_n == 0) return QTAM_ERR_INVALID_ARG;
  p->last_launches = 0;
  if (batch == 0) return QTAM_OK;
  return length_resample(p, d_in, batch, to_standard != 0, d_out, static_cast<cudaStream_t>(stream));
}

qtam_status qtam_threshold_rowmedian(qtam_plan *p, void *d_coef, int batch, double kappa, void *stream) {
  if (p && p->host_only) return QTAM_ERR_CUDA;
  if (!check_call(p, d_coef, d_coef, batch) || !(kappa >= 0.0)) return QTAM_ERR_INVALID_ARG;
  p->last_launches = 0;
  if (batch == 0) return QTAM_OK;
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  const qtam_status s = fast_threshold(p, d_coef, batch, kappa, st);
  if (s != QTAM_OK || !p->thr_has_big) return s;
  return generic_threshold(p, d_coef, batch, kappa, p->n_thr_tasks > 0 ? kThrFastLog2Max + 1 : 0, st);
}

qtam_status qtam_remodulate(qtam_plan *p, const void *d_coef, int batch, void *d_out, void *stream) {
  if (p && p->host_only) return QTAM_ERR_CUDA;
  if (!check_call(p, d_coef, d_out, batch)) return QTAM_ERR_INVALID_ARG;
  p->last_launches = 0;
  if (batch == 0) return QTAM_OK;
  return remodulate(p, d_coef, batch, d_out, static_cast<cudaStream_t>(stream));
}

qtam_status qtam_instantaneous_frequency(qtam_plan *p, const void *d_coef, int batch, void *d_out, void *stream) {
  if (p && p->host_only) return QTAM_ERR_CUDA;
  if (!check_call(p, d_coef, d_out, batch)) return QTAM_ERR_INVALID_ARG;
  p->last_launches = 0;
  if (batch == 0) return QTAM_OK;
  return instantaneous_frequency(p, d_coef, batch, d_out, static_cast<cudaStream_t>(stream));
}

qtam_status qtam_gather_plane(qtam_plan *p, const void *d_coef, int batch, const int32_t *d_best, void *d_out,
                              void *stream) {
  if (p && p->host_only) return QTAM_ERR_CUDA;
  if (!check_call(p, d_coef, d_out, batch) || !d_best) return QTAM_ERR_INVALID_ARG;
  p->last_launches = 0;
  if (batch == 0) return QTAM_OK;
  return gather_plane(p, d_coef, batch, d_best, d_out, static_cast<cudaStream_t>(stream));
}

int64_t qtam_max_plane_coeffs(const qtam_plan *p) {
  if (!p) return 0;
  std::vector<int64_t> size(size_t(p->hp.nP), 0);
  for (const HostRow &h : p->hp.rows) size[size_t(h.plane)] += h.M;
  return *std::max_element(size.begin(), size.end());
}

qtam_status qtam_plane_metric(qtam_plan *p, const void *d_coef, int batch, int metric, void *d_metric,
                              int32_t *d_best, void *stream) {
  if (p && p->host_only) return QTAM_ERR_CUDA;
  if (!check_call(p, d_coef, d_metric, batch) || metric < 0 || metric > 1) return QTAM_ERR_INVALID_ARG;
  p->last_launches = 0;
  if (batch == 0) return QTAM_OK;
  return plane_metric(p, d_coef, batch, metric, d_metric, d_best, static_cast<cudaStream_t>(stream));
}

int qtam_last_launch_count(const qtam_plan *p) { return p ? p->last_launches : 0; }

static const char *const kKernelNames[K_COUNT] = {
    "cfft_seq", "cfft_cols", "cfft_rows", "r2c_post", "c2r_pre", "fwd_rows", "fwd_combine",
    "inv_rows", "inv_reduce", "dense_place", "threshold", "r2c_fast", "fwd_rows_fast", "inv_rows_fast",
    "reduce_c2r_fast", "inv_fused", "inv_tiles", "combine_c2r", "threshold_fast", "rows_cta_fwd", "rows_cta_inv",
    "tiny_rows_fwd", "tiny_rows_inv", "long_fft_a", "long_fft_b", "plane_metric", "best_plane", "remodulate", "inst_freq", "fwd_rows_thr", "gather_plane",
    "rows_cl_fwd", "rows_cl_inv", "combine_runs", "c2c_fast", "split3", "combine3", "len_band", "len_synth", "len_analysis", "cluster", "mask", "spec_residues",
    "rows_2p14_fwd", "rows_2p15_fwd", "rows_2p16_fwd", "rows_2p17_fwd", "rows_2p14_inv", "rows_2p15_inv", "rows_2p16_inv", "rows_2p17_inv"};

qtam_status qtam_profile_enable(qtam_plan *p, int on, int max_launches) {
  if (!p || p->host_only) return QTAM_ERR_INVALID_ARG;
  if (on) {
    if (max_launches < 1) max_launches = 4096;
    while ((int)p->prof_pool.size() < max_launches) {
      ProfRec r{};
      if (cudaEventCreate(&r.e0) != cudaSuccess || cudaEventCreate(&r.e1) != cudaSuccess) return QTAM_ERR_CUDA;
      p->prof_pool.push_back(r);
    }
  }
  p->prof_on = on != 0;
  p->prof_used = 0;
  p->prof_dropped = 0;
  return QTAM_OK;
}

int qtam_profile_read(qtam_plan *p, qtam_kernel_stat *out, int capacity) {
  if (!p || !out || capacity < 1) return -1;
  qtam_kernel_stat acc[K_COUNT];
  for (int k = 0; k < K_COUNT; ++k) {
    std::memset(&acc[k], 0, sizeof(acc[k]));
    std::strncpy(acc[k].name, kKernelNames[k], sizeof(acc[k].name) - 1);
  }
  for (int i = 0; i < p->prof_used; ++i) {
    ProfRec &r = p->prof_pool[(size_t)i];
    if (cudaEventSynchronize(r.e1) != cudaSuccess) return -1;
    float ms = 0.f;
    if (cudaEventElapsedTime(&ms, r.e0, r.e1) != cudaSuccess) return -1;
    acc[r.kid].launches += 1;
    acc[r.kid].ms += (double)ms;
    acc[r.kid].algo_bytes += r.bytes;
    acc[r.kid].design_bytes += r.design;
  }
  p->prof_used = 0;
  int n = 0;
  for (int k = 0; k < K_COUNT && n < capacity; ++k)
    if (acc[k].launches > 0) out[n++] = acc[k];
  return n;
}

const char *qtam_status_string(qtam_status s) {
  switch (s) {
    case QTAM_OK: return "ok";
    case QTAM_ERR_INVALID_ARG: return "invalid argument";
    case QTAM_ERR_UNSUPPORTED: return "unsupported configuration";
    case QTAM_ERR_ALLOC: return "allocation failed";
    case QTAM_ERR_CUDA: return "CUDA error (or no CUDA device)";
    case QTAM_ERR_EMPTY_FRAME: return "empty cover set";
    case QTAM_ERR_TOO_LARGE: return "problem larger than the library's fixed scratch (QTAM_CLUSTER_NOALLOC_MAX_PIXELS)";
  }
  return "unknown status";
}

}  // extern "C"
