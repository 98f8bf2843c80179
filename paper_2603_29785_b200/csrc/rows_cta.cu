// rows_cta.cu -- rows of 2^11 .. 2^17 points (float): one CTA per (segment, row), the row's short FFT in
// shared memory with the Stockham engine of ctafft.cuh.
//
//   M <= 2^14 : the whole row in one transform.  Forward (a2 + a3): pass 1 gathers X[kc + jj] W_k[jj]
//               straight from the spectrum (only the support is read, the rest of the M-array is zero;
//               A9 :323, C46 :583), the last pass writes the scaled coefficients (C47 :589).  Inverse (a5):
//               pass 1 reads the coefficients, the result is multiplied by sqrt(N/M) W_k and written to
//               the band workspace (C49 :598).
//   M = Mb 2^14, Mb = 2, 4, 8 : decimation in time for the forward, in frequency for the inverse, so
//               that both global sides stay contiguous:
//                 forward  Z_jb[n'] = sum_j' B[jb + Mb j'] w_M2^{j' n'}   (Mb transforms, strided gather)
//                          Y[n' + M2 nb] = s sum_jb w_Mb^{jb nb} w_M^{jb n'} Z_jb[n']   (radix-Mb step)
//                 inverse  u_jb[n'] = w_M^{-jb n'} sum_nb Y[n' + M2 nb] w_Mb^{-jb nb}   (radix-Mb step)
//                          Bhat[jb + Mb j'] = sum_n' u_jb[n'] w_M2^{-j' n'}             (Mb transforms)
//               The Mb intermediate sequences live in a per-CTA scratch region in global memory that the
//               CTA rewrites for every row it takes, so it stays in L2.
// Grids are persistent (CTAs loop over work items) because the scratch is per resident CTA.
#include <algorithm>
#include <cmath>
#include <cstdint>
#include <vector>

#include "ctafft.cuh"
#include "device_plan.hpp"

namespace qtam {

extern __shared__ __align__(16) unsigned char qtam_cta_smem[];

static int ilog2(long long v) { int l = 0; while ((1LL << l) < v) ++l; return l; }

struct TwbTables { const float2 *t[3]; };   // e^{+2 pi i n'/M}, n' < 2^14, for M = 2^15, 2^16, 2^17

// w^0 .. w^(MB-1) from w (products of at most three factors)
template <int MB> __device__ __forceinline__ void powers(float2 w, float2 (&pw)[MB]) {
  pw[0] = make_float2(1.f, 0.f);
  if constexpr (MB > 1) pw[1] = w;
#pragma unroll
  for (int k = 2; k < MB; ++k) pw[k] = (k & 1) ? pcmul(pw[k - 1], w) : pcmul(pw[k / 2], pw[k / 2]);
}

// forward radix-MB step: scratch [jb][n'] -> coefficients
template <int MB, int NT, int M2>
__device__ __forceinline__ void fwd_combine(const float2 *__restrict__ z, const float2 *__restrict__ twb,
                                            float2 *__restrict__ Yseg, const long long *off, int nm, float scale) {
#pragma unroll 1
  for (int n = threadIdx.x; n < M2; n += NT) {
    float2 v[MB], pw[MB];
    powers<MB>(__ldg(twb + n), pw);
#pragma unroll
    for (int jb = 0; jb < MB; ++jb) v[jb] = __ldcg(z + jb * M2 + n);
#pragma unroll
    for (int jb = 1; jb < MB; ++jb) v[jb] = pcmul(v[jb], pw[jb]);
    RegFFT<MB, +1>::run(v);
#pragma unroll
    for (int nb = 0; nb < MB; ++nb) v[nb] = pscale(v[nb], scale);
    for (int m = 0; m < nm; ++m) {
      float2 *Y = Yseg + off[m] + n;
#pragma unroll
      for (int nb = 0; nb < MB; ++nb) __stcs(Y + nb * M2, v[nb]);
    }
  }
}

// inverse radix-MB step: coefficients -> scratch [jb][n']
template <int MB, int NT, int M2>
__device__ __forceinline__ void inv_split(const float2 *__restrict__ Yseg, const long long *off, int nm,
                                          const float2 *__restrict__ twb, float2 *__restrict__ z) {
#pragma unroll 1
  for (int n = threadIdx.x; n < M2; n += NT) {
    float2 v[MB], pw[MB];
    float2 w = __ldg(twb + n);
    w.y = -w.y;
    powers<MB>(w, pw);
#pragma unroll
    for (int nb = 0; nb < MB; ++nb) v[nb] = __ldcs(Yseg + off[0] + n + nb * M2);
    for (int m = 1; m < nm; ++m) {      // members of the leader's set: rows are added before the transform
      const float2 *Y = Yseg + off[m] + n;
#pragma unroll
      for (int nb = 0; nb < MB; ++nb) v[nb] = padd(v[nb], __ldcs(Y + nb * M2));
    }
    RegFFT<MB, -1>::run(v);
#pragma unroll
    for (int jb = 0; jb < MB; ++jb) z[jb * M2 + n] = jb ? pcmul(v[jb], pw[jb]) : v[0];
  }
}

struct GatherIn {      // B[j] = X[kc + jj] W_k[jj] at M-array index j = jb + Mb a (R6), zero off the support (R8)
  const float2 *__restrict__ X; const float *__restrict__ W;
  int kc, dk, nbins, M, lb, jb;
  __device__ __forceinline__ float2 operator()(int a) const {
    const int j = jb + (a << lb);
    const int jj = j < (M >> 1) ? j : j - M;
    const int f = kc + jj;
    float2 v = make_float2(0.f, 0.f);
    if (jj >= -dk && jj <= dk && (unsigned)f < (unsigned)nbins) {
      const float2 x = __ldg(X + f);
      const float w = __ldg(W + jj);
      v = make_float2(x.x * w, x.y * w);
    }
    return v;
  }
};
struct CoefOut {      // the same coefficients go to every member of the leader's set
  float2 *__restrict__ seg; const long long *off; int nm; float scale;
  __device__ __forceinline__ void operator()(int a, float2 v) const {
    v = pscale(v, scale);
    for (int m = 0; m < nm; ++m) __stcs(seg + off[m] + a, v);
  }
};
struct CoefIn {       // sum of the members' coefficients
  const float2 *__restrict__ seg; const long long *off; int nm;
  __device__ __forceinline__ float2 operator()(int a) const {
    float2 v = __ldcs(seg + off[0] + a);
    for (int m = 1; m < nm; ++m) v = padd(v, __ldcs(seg + off[m] + a));
    return v;
  }
};
struct ScratchOut {
  float2 *__restrict__ p;
  __device__ __forceinline__ void operator()(int a, float2 v) const { p[a] = v; }
};
struct ScratchIn {
  const float2 *__restrict__ p;
  __device__ __forceinline__ float2 operator()(int a) const { return __ldcg(p + a); }
};

template <int L2, bool FORWARD>
__global__ void __launch_bounds__(CtaFftPlan<L2>::NT, (L2 == 13 || L2 == 12) ? 2 : 1)
k_rows_cta(const int *__restrict__ rowidx, const int *__restrict__ memptr, const int *__restrict__ mem, int nrows,
           const RowDev *__restrict__ rows,
           const float *__restrict__ win, const float2 *__restrict__ spec, long long xstride, int nbins,
           float2 *__restrict__ coef, long long ctot, float2 *__restrict__ band, long long sumL,
           float2 *__restrict__ scratch, long long scratch_stride, const float2 *__restrict__ ptw,
           TwbTables twb, int batch, int plane) {
  constexpr int M2 = 1 << L2, NT = CtaFftPlan<L2>::NT;
  float2 *s = reinterpret_cast<float2 *>(qtam_cta_smem);
  float2 *z = scratch + (size_t)blockIdx.x * scratch_stride;
  // rows with the same centre bin and half-width (the clamped rows of different Q-planes) have the same
  // window: `rowidx` lists one leader per such set, mem[memptr[i] .. memptr[i+1]) its members.  Forward:
  // one transform, stored at every member's offset; inverse: the members' rows are added first.
  __shared__ int s_nm;
  __shared__ long long s_off[kCtaMaxMembers];
  __shared__ long long s_slot;      // inverse: band slot that takes the sum (the first member taking part)
  const long long total = (long long)nrows * batch;
  for (long long item = blockIdx.x; item < total; item += gridDim.x) {
    const int seg = (int)(item / nrows);
    const int li = (int)(item - (long long)seg * nrows);
    const RowDev r = rows[rowidx[li]];
    __syncthreads();
    if (threadIdx.x == 0) {
      int n = 0;
      for (int m = memptr[li]; m < memptr[li + 1]; ++m) {
        const RowDev &rm = rows[mem[m]];
        if (FORWARD || plane < 0 || rm.plane == plane) {
          if (n == 0) s_slot = rm.woff;
          s_off[n++] = rm.offset;
        }
      }
      s_nm = n;
    }
    __syncthreads();
    const int nm = s_nm;
    if (nm == 0) continue;
    const int lb = r.log2M - L2, Mb = 1 << lb;
    const float *W = win + r.woff + r.dk;
    float2 *Yseg = coef + (size_t)seg * ctot;
    const float2 *tb = lb > 0 ? twb.t[lb - 1] : nullptr;
    if constexpr (FORWARD) {
      GatherIn in{spec + (size_t)seg * xstride, W, r.kc, r.dk, nbins, r.M, lb, 0};
      if (Mb == 1) {
        cta_fft_io<L2, NT, +1, true, true>(s, in, CoefOut{Yseg, s_off, nm, (float)r.fwd_scale}, ptw);
        __syncthreads();
      } else {
        for (int jb = 0; jb < Mb; ++jb) {
          in.jb = jb;
          cta_fft_io<L2, NT, +1, true, true>(s, in, ScratchOut{z + (size_t)jb * M2}, ptw);
          __syncthreads();
        }
        switch (lb) {
          case 1: fwd_combine<2, NT, M2>(z, tb, Yseg, s_off, nm, (float)r.fwd_scale); break;
          case 2: fwd_combine<4, NT, M2>(z, tb, Yseg, s_off, nm, (float)r.fwd_scale); break;
          default: fwd_combine<8, NT, M2>(z, tb, Yseg, s_off, nm, (float)r.fwd_scale); break;
        }
        __syncthreads();   // the scratch is rewritten by the next row
      }
    } else {
      if (Mb > 1) {
        switch (lb) {
          case 1: inv_split<2, NT, M2>(Yseg, s_off, nm, tb, z); break;
          case 2: inv_split<4, NT, M2>(Yseg, s_off, nm, tb, z); break;
          default: inv_split<8, NT, M2>(Yseg, s_off, nm, tb, z); break;
        }
        __syncthreads();
      }
      float2 *Gb = band + (size_t)seg * sumL + s_slot + r.dk;
      const float amp = (float)r.inv_amp;
      for (int jb = 0; jb < Mb; ++jb) {
        if (Mb == 1) cta_fft_io<L2, NT, -1, true, false>(s, CoefIn{Yseg, s_off, nm}, CtaFftNone{}, ptw);
        else cta_fft_io<L2, NT, -1, true, false>(s, ScratchIn{z + (size_t)jb * M2}, CtaFftNone{}, ptw);
        // G_k[jj] = sqrt(N/M) Bhat[jj] W_k[jj] on the support, clipped to the one-sided spectrum (R8)
        for (int jp = threadIdx.x; jp < M2; jp += NT) {
          const int j = jb + (jp << lb);
          const int jj = j < (r.M >> 1) ? j : j - r.M;
          const int f = r.kc + jj;
          if (jj >= -r.dk && jj <= r.dk && (unsigned)f < (unsigned)nbins) Gb[jj] = pscale(s[jp], amp * __ldg(W + jj));
        }
        __syncthreads();
      }
    }
  }
}

// --------------------------------------------------------------------------------------------------
// host side
// --------------------------------------------------------------------------------------------------
template <int L2> static void fill_class_table(std::vector<float> &t) { fill_cta_fft_tables<L2, CtaFftPlan<L2>::NT>(t); }
template <int L2> static bool prepare_class(qtam_plan *p, int c) {
  const size_t smem = sizeof(float2) * (size_t)cta_fft_smem_elems<L2>();
  return kernel_prepare(p->cfg_rows_cta[c][1], k_rows_cta<L2, true>, CtaFftPlan<L2>::NT, smem) &&
         kernel_prepare(p->cfg_rows_cta[c][0], k_rows_cta<L2, false>, CtaFftPlan<L2>::NT, smem);
}

qtam_status build_rows_cta(qtam_plan *p) {
  const HostPlan &hp = p->hp;
  p->cta_rows = false;
  if (!p->fast_rows) return QTAM_OK;
  auto up = [&](void **dst, const void *src, size_t bytes) -> bool {
    *dst = nullptr;
    if (cudaMalloc(dst, bytes ? bytes : 16) != cudaSuccess) return false;
    p->device_bytes += bytes;
    return bytes == 0 || cudaMemcpy(*dst, src, bytes, cudaMemcpyHostToDevice) == cudaSuccess;
  };
  bool need_twb[3] = {false, false, false};
  std::vector<int> followers;   // rows whose band slot the joint inverse leaves unwritten
  for (int c = 0; c < 4; ++c) {
    const int L2 = kCtaLog2Min + c;
    std::vector<int> idx;
    for (size_t k = 0; k < hp.rows.size(); ++k) {
      const int lm = ilog2(hp.rows[k].M);
      const bool mine = (lm == L2) || (c == 3 && lm > L2 && lm <= kCtaLog2Max);
      if (!mine) continue;
      idx.push_back((int)k);
      p->cta_sumM[c] += (double)hp.rows[k].M; p->cta_sumL[c] += (double)hp.rows[k].L;
      if (lm > L2) { need_twb[lm - L2 - 1] = true; p->cta_maxM = std::max<int64_t>(p->cta_maxM, hp.rows[k].M); }
    }
    // longest rows first within a segment
    std::stable_sort(idx.begin(), idx.end(), [&](int a, int b) { return hp.rows[(size_t)a].M > hp.rows[(size_t)b].M; });
    if (idx.empty()) { p->n_cta_rows[c] = 0; continue; }
    // one leader per set of rows with the same centre bin and half-width
    std::vector<int> lead;
    std::vector<std::vector<int>> members;
    for (int k : idx) {
      size_t l = 0;
      while (l < lead.size() && !(hp.rows[(size_t)lead[l]].kc == hp.rows[(size_t)k].kc &&
                                  hp.rows[(size_t)lead[l]].dk == hp.rows[(size_t)k].dk &&
                                  (int)members[l].size() < kCtaMaxMembers &&
                                  std::none_of(members[l].begin(), members[l].end(), [&](int m) {
                                    return hp.rows[(size_t)m].plane == hp.rows[(size_t)k].plane; }))) ++l;
      if (l == lead.size()) { lead.push_back(k); members.emplace_back(); }
      members[l].push_back(k);
    }
    std::vector<int> memptr(1, 0), mem;
    for (auto &m : members) {
      mem.insert(mem.end(), m.begin(), m.end()); memptr.push_back((int)mem.size());
      for (size_t i = 1; i < m.size(); ++i) followers.push_back(m[i]);
    }
    p->n_cta_rows[c] = (int)lead.size();
    if (!up(reinterpret_cast<void **>(&p->d_cta_rowidx[c]), lead.data(), lead.size() * sizeof(int))) return QTAM_ERR_ALLOC;
    if (!up(reinterpret_cast<void **>(&p->d_cta_memptr[c]), memptr.data(), memptr.size() * sizeof(int))) return QTAM_ERR_ALLOC;
    if (!up(reinterpret_cast<void **>(&p->d_cta_mem[c]), mem.data(), mem.size() * sizeof(int))) return QTAM_ERR_ALLOC;
    std::vector<float> t;
    bool ok = false;
    switch (L2) {
      case 11: fill_class_table<11>(t); ok = prepare_class<11>(p, c); break;
      case 12: fill_class_table<12>(t); ok = prepare_class<12>(p, c); break;
      case 13: fill_class_table<13>(t); ok = prepare_class<13>(p, c); break;
      default: fill_class_table<14>(t); ok = prepare_class<14>(p, c); break;
    }
    if (!ok) return QTAM_ERR_CUDA;
    if (!up(&p->d_ptw_rows[c], t.data(), t.size() * sizeof(float))) return QTAM_ERR_ALLOC;
    p->cta_rows = true;
  }
  if (!followers.empty()) {
    // joint CSR (one set per bin) without the followers' band slots
    std::vector<uint8_t> skip((size_t)hp.sumL, 0);
    for (int k : followers)
      for (int64_t i = 0; i < hp.rows[(size_t)k].L; ++i) skip[(size_t)(hp.rows[(size_t)k].goff + i)] = 1;
    const int nsets = hp.nP + 1;
    std::vector<int32_t> jptr((size_t)hp.nb + 1, 0), jidx;
    for (int64_t f = 0; f < hp.nb; ++f) {
      jptr[(size_t)f] = (int32_t)jidx.size();
      for (int32_t e = hp.csr_ptr[(size_t)(f * nsets)]; e < hp.csr_ptr[(size_t)(f * nsets + hp.nP)]; ++e)
        if (!skip[(size_t)hp.csr_idx[(size_t)e]]) jidx.push_back(hp.csr_idx[(size_t)e]);
    }
    jptr[(size_t)hp.nb] = (int32_t)jidx.size();
    if (!up(reinterpret_cast<void **>(&p->d_csrj_ptr), jptr.data(), jptr.size() * sizeof(int32_t))) return QTAM_ERR_ALLOC;
    if (!up(reinterpret_cast<void **>(&p->d_csrj_idx), jidx.data(), jidx.size() * sizeof(int32_t))) return QTAM_ERR_ALLOC;
  }
  const long double tau = 6.283185307179586476925286766559005768L;
  for (int b = 0; b < 3; ++b) {
    if (!need_twb[b]) continue;
    const int64_t M = int64_t(1) << (kCtaLog2Min + 3 + b + 1), M2 = int64_t(1) << (kCtaLog2Min + 3);
    std::vector<float> t((size_t)(2 * M2));
    for (int64_t n = 0; n < M2; ++n) {
      const long double a = tau * (long double)n / (long double)M;
      t[(size_t)(2 * n)] = (float)cosl(a); t[(size_t)(2 * n + 1)] = (float)sinl(a);
    }
    if (!up(&p->d_twb[b], t.data(), t.size() * sizeof(float))) return QTAM_ERR_ALLOC;
  }
  return QTAM_OK;
}

template <int L2, bool FORWARD>
static qtam_status rows_cta_launch(qtam_plan *p, int c, int batch, void *d_coef, int plane, cudaStream_t st) {
  if (p->n_cta_rows[c] == 0) return QTAM_OK;
  constexpr int NT = CtaFftPlan<L2>::NT;
  const KernelCfg &cfg = p->cfg_rows_cta[c][FORWARD ? 1 : 0];
  if (!cfg.ready) return QTAM_ERR_CUDA;
  const size_t smem = cfg.smem;
  auto kern = k_rows_cta<L2, FORWARD>;
  const long long total = (long long)p->n_cta_rows[c] * batch;
  long long grid = std::min<long long>(total, (long long)p->num_sms * cfg.occ);
  // per-CTA scratch (rows longer than one transform) comes out of the plan's [max_batch][N] workspace
  long long stride = 0;
  if (c == 3 && p->cta_maxM > 0) {
    stride = p->cta_maxM;
    grid = std::min<long long>(grid, ((long long)p->max_batch * p->hp.N) / stride);
    if (grid < 1) return QTAM_ERR_UNSUPPORTED;
  }
  TwbTables tb;
  for (int b = 0; b < 3; ++b) tb.t[b] = static_cast<const float2 *>(p->d_twb[b]);
  const double bytes = (double)batch * 8.0 * p->cta_sumM[c];     // compulsory: the coefficients
  {
    LaunchScope ls(p, st, FORWARD ? K_ROWS_CTA_FWD : K_ROWS_CTA_INV, bytes, bytes + (double)batch * 8.0 * p->cta_sumL[c]);
    kern<<<(unsigned)grid, NT, smem, st>>>(
        p->d_cta_rowidx[c], p->d_cta_memptr[c], p->d_cta_mem[c], p->n_cta_rows[c], p->d_rows, static_cast<const float *>(p->d_win),
        static_cast<const float2 *>(p->d_spec), p->xstride, (int)p->hp.nb, static_cast<float2 *>(d_coef),
        p->hp.ctot, static_cast<float2 *>(p->d_band), p->hp.sumL, static_cast<float2 *>(p->d_ws), stride,
        static_cast<const float2 *>(p->d_ptw_rows[c]), tb, batch, plane);
  }
  QTAM_LAUNCH_CHECK();
  return QTAM_OK;
}

template <bool FORWARD>
static qtam_status rows_cta_all(qtam_plan *p, int batch, void *d_coef, int plane, cudaStream_t st) {
  qtam_status s = rows_cta_launch<14, FORWARD>(p, 3, batch, d_coef, plane, st);
  if (s == QTAM_OK) s = rows_cta_launch<13, FORWARD>(p, 2, batch, d_coef, plane, st);
  if (s == QTAM_OK) s = rows_cta_launch<12, FORWARD>(p, 1, batch, d_coef, plane, st);
  if (s == QTAM_OK) s = rows_cta_launch<11, FORWARD>(p, 0, batch, d_coef, plane, st);
  return s;
}

qtam_status cta_forward_rows(qtam_plan *p, int batch, void *d_coef, cudaStream_t st) {
  return rows_cta_all<true>(p, batch, d_coef, -1, st);
}
qtam_status cta_inverse_rows(qtam_plan *p, const void *d_coef, int batch, int plane, cudaStream_t st) {
  return rows_cta_all<false>(p, batch, const_cast<void *>(d_coef), plane, st);
}

}  // namespace qtam
