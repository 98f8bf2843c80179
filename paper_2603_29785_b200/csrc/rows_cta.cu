// rows_cta.cu -- rows of 2^11 .. 2^13 points (float): one CTA per (segment, row), the row's short FFT in
// shared memory with the Stockham engine of ctafft.cuh (longer rows: rows_cluster.cu, rows_split.cu; the FORWARD of
// the 2^11-point rows: rows_2k.cu, one warp per row).
//
//   forward (a2 + a3)  pass 1 gathers X[kc + jj] W_k[jj] straight from the spectrum (only the support is read,
//                      the rest of the M-array is zero; A9 :323, C46 :583), the last pass writes the scaled
//                      coefficients (C47 :589) to every member of the leader's set (identical rows -- same centre
//                      bin and half-width, the clamped rows of different Q-planes -- are transformed once).
//   inverse (a5 + a6)  a CTA takes a GROUP of leaders consecutive in centre bin, one after the other: pass 1 adds
//                      the members' coefficient rows, the result times sqrt(N/M) W_k (C49 :598) is added into the
//                      group's partial spectrum by plain read-modify-write (one CTA owns the group, the rows come
//                      in a fixed order: a segmented reduction without atomics and without a band workspace).
//                      The groups' partial sums are added up by k_combine_runs (combine_runs.cu).
#include <algorithm>
#include <cmath>
#include <cstdint>
#include <vector>

#include "ctafft.cuh"
#include "device_plan.hpp"

namespace qtam {

extern __shared__ __align__(16) unsigned char qtam_cta_smem[];

struct GatherIn {      // B[j] = X[kc + jj] W_k[jj] at M-array index j (R6), zero off the support (R8)
  const float2 *__restrict__ X; const float *__restrict__ W;
  int kc, dk, nbins, M;
  __device__ __forceinline__ float2 operator()(int j) const {
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
  float2 *__restrict__ seg; const int *off; int nm; float scale;
  __device__ __forceinline__ void operator()(int a, float2 v) const {
    v = pscale(v, scale);
    for (int m = 0; m < nm; ++m) __stcs(seg + off[m] + a, v);
  }
};
struct CoefIn {       // sum of the members' coefficients
  const float2 *__restrict__ seg; const int *off; int nm;
  __device__ __forceinline__ float2 operator()(int a) const {
    float2 v = __ldcs(seg + off[0] + a);
    for (int m = 1; m < nm; ++m) v = padd(v, __ldcs(seg + off[m] + a));
    return v;
  }
};

template <int L2, bool FORWARD>
__global__ void __launch_bounds__(CtaFftPlan<L2>::NT, (L2 == 13 || L2 == 12) ? 2 : 1)
k_rows_cta(const ClLeader *__restrict__ lead, const int2 *__restrict__ mem, int nlead,
           const ClGroup *__restrict__ groups, int ngroups,
           const float *__restrict__ win, const float2 *__restrict__ spec, long long xstride, int nbins,
           float2 *__restrict__ coef, long long ctot, float2 *__restrict__ part, long long part_stride,
           const float2 *__restrict__ ptw, int batch, int plane) {
  constexpr int M = 1 << L2, NT = CtaFftPlan<L2>::NT;
  float2 *s = reinterpret_cast<float2 *>(qtam_cta_smem);
  __shared__ int s_nm;
  __shared__ int s_off[kCtaMaxMembers];
  if constexpr (FORWARD) {
    const long long total = (long long)nlead * batch;
    for (long long item = blockIdx.x; item < total; item += gridDim.x) {
      const int seg = (int)(item / nlead);
      const ClLeader L = lead[item - (long long)seg * nlead];
      __syncthreads();
      if (threadIdx.x < L.nmem) s_off[threadIdx.x] = mem[L.mem0 + threadIdx.x].x;
      __syncthreads();
      GatherIn in{spec + (size_t)seg * xstride, win + L.woff + L.dk, L.kc, L.dk, nbins, M};
      cta_fft_io<L2, NT, +1, true, true>(s, in, CoefOut{coef + (size_t)seg * ctot, s_off, L.nmem, L.fwd_scale}, ptw);
    }
  } else {
    const long long total = (long long)ngroups * batch;
    for (long long item = blockIdx.x; item < total; item += gridDim.x) {
      const int seg = (int)(item / ngroups);
      const ClGroup Gp = groups[item - (long long)seg * ngroups];
      float2 *pg = part + (size_t)seg * part_stride + Gp.part_off;
      {
        float4 *z = reinterpret_cast<float4 *>(pg);
        const int n4 = ((Gp.nb + 1) & ~1) / 2;
        for (int i = threadIdx.x; i < n4; i += NT) z[i] = make_float4(0.f, 0.f, 0.f, 0.f);
      }
      const float2 *Yseg = coef + (size_t)seg * ctot;
#pragma unroll 1
      for (int l = 0; l < Gp.nlead; ++l) {
        const ClLeader L = lead[Gp.lead0 + l];
        __syncthreads();      // the previous row's updates of the partial sum and its reads of s_off are done
        if (threadIdx.x < 32) {
          // members that take part (all of them, or those of the requested plane), compacted in order
          const bool ok = threadIdx.x < L.nmem && (plane < 0 || mem[L.mem0 + threadIdx.x].y == plane);
          const unsigned b = __ballot_sync(0xffffffffu, ok);
          if (ok) s_off[__popc(b & ((1u << threadIdx.x) - 1u))] = mem[L.mem0 + threadIdx.x].x;
          if (threadIdx.x == 0) s_nm = __popc(b);
        }
        __syncthreads();
        const int nm = s_nm;
        if (nm == 0) continue;
        cta_fft_io<L2, NT, -1, true, false>(s, CoefIn{Yseg, s_off, nm}, CtaFftNone{}, ptw);
        // G_k[jj] = sqrt(N/M) Bhat[jj] W_k[jj] on the support, clipped to the one-sided spectrum (R8); the loads
        // of a batch are issued before its stores (a store may not be overtaken by a later load of the same array)
        const float *W = win + L.woff + L.dk;
        float2 *pb = pg + (L.kc - Gp.lo);
        constexpr int CH = 8;
        static_assert(M % (CH * NT) == 0 || M < CH * NT, "batches must tile the row");
#pragma unroll 1
        for (int j0 = threadIdx.x; j0 < M; j0 += CH * NT) {
          float2 old[CH]; float w[CH]; int jjs[CH];
#pragma unroll
          for (int c = 0; c < CH; ++c) {
            const int j = j0 + c * NT;
            const int jj = j < (M >> 1) ? j : j - M;
            const int f = L.kc + jj;
            const bool ok = j < M && jj >= -L.dk && jj <= L.dk && (unsigned)f < (unsigned)nbins;
            jjs[c] = ok ? jj : (1 << 30);
            old[c] = make_float2(0.f, 0.f); w[c] = 0.f;
            if (ok) { old[c] = __ldcg(pb + jj); w[c] = __ldg(W + jj); }
          }
#pragma unroll
          for (int c = 0; c < CH; ++c)
            if (jjs[c] != (1 << 30)) {
              const float a = L.inv_amp * w[c];
              pb[jjs[c]] = pfma(s[j0 + c * NT], make_float2(a, a), old[c]);
            }
        }
      }
    }
  }
}

// --------------------------------------------------------------------------------------------------
// host side
// --------------------------------------------------------------------------------------------------
static int ilog2(long long v) { int l = 0; while ((1LL << l) < v) ++l; return l; }

template <int L2> static void fill_class_table(std::vector<float> &t) { fill_cta_fft_tables<L2, CtaFftPlan<L2>::NT>(t); }
template <int L2> static bool prepare_class(qtam_plan *p, int c) {
  const size_t smem = sizeof(float2) * (size_t)cta_fft_smem_elems<L2>();
  return kernel_prepare(p->cfg_rows_cta[c][1], k_rows_cta<L2, true>, CtaFftPlan<L2>::NT, smem) &&
         kernel_prepare(p->cfg_rows_cta[c][0], k_rows_cta<L2, false>, CtaFftPlan<L2>::NT, smem);
}

// Leaders (one per set of rows with the same centre bin and half-width, at most one row of a plane per set) in
// ascending centre bin, and groups of consecutive leaders for the inverse; the groups' partial sums are appended
// to the plan's per-segment partial-sum layout and registered as runs for k_combine_runs.
void build_leaders_and_groups(qtam_plan *p, const std::vector<int> &rows_in, int groups_wanted,
                              std::vector<ClLeader> &lead, std::vector<int2> &mem, std::vector<ClGroup> &groups,
                              int by_residue_max_lead, int by_residue_max_mem, bool *by_residue) {
  const HostPlan &hp = p->hp;
  std::vector<int> idx = rows_in;
  std::stable_sort(idx.begin(), idx.end(), [&](int a, int b) {
    return hp.rows[(size_t)a].kc != hp.rows[(size_t)b].kc ? hp.rows[(size_t)a].kc < hp.rows[(size_t)b].kc
                                                          : hp.rows[(size_t)a].dk < hp.rows[(size_t)b].dk; });
  // sets first (members of a set are stored contiguously), then one leader record per set
  std::vector<std::vector<int>> sets;
  for (int k : idx) {
    const HostRow &h = hp.rows[(size_t)k];
    bool joined = false;
    for (size_t l = sets.size(); l-- > 0 && !joined;) {
      const HostRow &hb = hp.rows[(size_t)sets[l][0]];
      if (hb.kc != h.kc) break;
      if (hb.dk != h.dk || hb.wid != h.wid || (int)sets[l].size() >= kCtaMaxMembers) continue;
      bool plane_free = true;
      for (int m : sets[l]) if (hp.rows[(size_t)m].plane == h.plane) plane_free = false;
      if (!plane_free) continue;
      sets[l].push_back(k); joined = true;
    }
    if (!joined) sets.push_back(std::vector<int>(1, k));
  }
  for (const auto &st : sets) {
    const HostRow &h = hp.rows[(size_t)st[0]];
    ClLeader L{};
    L.kc = (int)h.kc; L.dk = (int)h.dk; L.woff = (int)h.woff; L.mem0 = (int)mem.size(); L.nmem = (int)st.size();
    L.row = st[0];
    L.fwd_scale = (float)(1.0 / std::sqrt((double)hp.N * (double)h.M));
    L.inv_amp = (float)std::sqrt((double)hp.N / (double)h.M);
    lead.push_back(L);
    for (int k : st) mem.push_back(make_int2((int)hp.rows[(size_t)k].offset, hp.rows[(size_t)k].plane));
  }
  // partial sums sorted by residue mod 64 (rows_split.cu) when the class is small enough for that kernel
  const bool res64 = (int)lead.size() <= by_residue_max_lead && (int)mem.size() <= by_residue_max_mem;
  if (by_residue) *by_residue = res64;
  const int per = std::max<int>(1, ((int)lead.size() + groups_wanted - 1) / groups_wanted);
  for (size_t i = 0; i < lead.size(); i += (size_t)per) {
    ClGroup g{};
    g.lead0 = (int)i; g.nlead = (int)std::min(lead.size() - i, (size_t)per);
    int64_t lo = hp.nb, hi = -1;
    for (int l = 0; l < g.nlead; ++l) {
      const HostRow &h = hp.rows[(size_t)lead[i + (size_t)l].row];
      lo = std::min<int64_t>(lo, std::max<int64_t>(h.kc - h.dk, 0));
      hi = std::max<int64_t>(hi, std::min<int64_t>(h.kc + h.dk, hp.nb - 1));
    }
    if (hi < lo) { lo = 0; hi = -1; }
    g.lo = (int)lo; g.nb = (int)(hi - lo + 1);
    g.part_off = p->part_stride;
    if (res64 && g.nb > 0) {
      p->part_stride += 64 * (((lo + g.nb - 1) >> 6) - (lo >> 6) + 1);
      p->runs.push_back(HostRun{(int)lo, g.nb, g.part_off, 2, -1});
    } else {
      p->part_stride += (g.nb + 1) & ~1;
      p->runs.push_back(HostRun{(int)lo, g.nb, g.part_off, 1, -1});
    }
    groups.push_back(g);
  }
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
  for (int c = 0; c < kCtaClasses; ++c) {
    const int L2 = kCtaLog2Min + c;
    std::vector<int> idx;
    for (size_t k = 0; k < hp.rows.size(); ++k) {
      if (ilog2(hp.rows[k].M) != L2) continue;
      idx.push_back((int)k);
      p->cta_sumM[c] += (double)hp.rows[k].M; p->cta_sumL[c] += (double)hp.rows[k].L;
    }
    p->n_cta_rows[c] = 0; p->n_cta_groups[c] = 0;
    if (idx.empty()) continue;
    std::vector<ClLeader> lead;
    std::vector<int2> mem;
    std::vector<ClGroup> groups;
    build_leaders_and_groups(p, idx, 12, lead, mem, groups, 0, 0, nullptr);
    p->n_cta_rows[c] = (int)lead.size(); p->n_cta_groups[c] = (int)groups.size();
    if (!up(reinterpret_cast<void **>(&p->d_cta_lead[c]), lead.data(), lead.size() * sizeof(ClLeader))) return QTAM_ERR_ALLOC;
    if (!up(reinterpret_cast<void **>(&p->d_cta_mem[c]), mem.data(), mem.size() * sizeof(int2))) return QTAM_ERR_ALLOC;
    if (!up(reinterpret_cast<void **>(&p->d_cta_groups[c]), groups.data(), groups.size() * sizeof(ClGroup))) return QTAM_ERR_ALLOC;
    std::vector<float> t;
    bool ok = false;
    switch (L2) {
      case 11: fill_class_table<11>(t); ok = prepare_class<11>(p, c); break;
      case 12: fill_class_table<12>(t); ok = prepare_class<12>(p, c); break;
      default: fill_class_table<13>(t); ok = prepare_class<13>(p, c); break;
    }
    if (!ok) return QTAM_ERR_CUDA;
    if (!up(&p->d_ptw_rows[c], t.data(), t.size() * sizeof(float))) return QTAM_ERR_ALLOC;
    p->cta_rows = true;
  }
  return QTAM_OK;
}

template <int L2, bool FORWARD>
static qtam_status rows_cta_launch(qtam_plan *p, int c, int batch, void *d_coef, int plane, cudaStream_t st) {
  if (p->n_cta_rows[c] == 0) return QTAM_OK;
  constexpr int NT = CtaFftPlan<L2>::NT;
  const KernelCfg &cfg = p->cfg_rows_cta[c][FORWARD ? 1 : 0];
  if (!cfg.ready) return QTAM_ERR_CUDA;
  const long long total = (long long)(FORWARD ? p->n_cta_rows[c] : p->n_cta_groups[c]) * batch;
  const long long grid = std::min<long long>(total, (long long)p->num_sms * cfg.occ);
  const double bytes = (double)batch * 8.0 * p->cta_sumM[c];     // compulsory: the coefficients
  {
    LaunchScope ls(p, st, FORWARD ? K_ROWS_CTA_FWD : K_ROWS_CTA_INV, bytes, bytes + (double)batch * 8.0 * p->cta_sumL[c]);
    k_rows_cta<L2, FORWARD><<<(unsigned)grid, NT, cfg.smem, st>>>(
        p->d_cta_lead[c], p->d_cta_mem[c], p->n_cta_rows[c], p->d_cta_groups[c], p->n_cta_groups[c],
        static_cast<const float *>(p->d_win), static_cast<const float2 *>(p->d_spec), p->xstride, (int)p->hp.nb,
        static_cast<float2 *>(d_coef), p->hp.ctot, static_cast<float2 *>(p->d_part), p->part_stride,
        static_cast<const float2 *>(p->d_ptw_rows[c]), batch, plane);
  }
  QTAM_LAUNCH_CHECK();
  return QTAM_OK;
}

// every class on a stream of its own (the classes write disjoint coefficients / partial sums)
template <bool FORWARD>
static qtam_status rows_cta_all(qtam_plan *p, int batch, void *d_coef, int plane, Fork &fk) {
  qtam_status s = QTAM_OK;
  if (p->n_cta_rows[2]) s = rows_cta_launch<13, FORWARD>(p, 2, batch, d_coef, plane, fk.next());
  if (s == QTAM_OK && p->n_cta_rows[1]) s = rows_cta_launch<12, FORWARD>(p, 1, batch, d_coef, plane, fk.next());
  if (s == QTAM_OK && p->n_cta_rows[0])
    s = FORWARD && p->rows2k_ok ? rows_2k_forward(p, batch, d_coef, fk.next())
                                : rows_cta_launch<11, FORWARD>(p, 0, batch, d_coef, plane, fk.next());
  return s;
}

qtam_status cta_forward_rows(qtam_plan *p, int batch, void *d_coef, Fork &fk) {
  return rows_cta_all<true>(p, batch, d_coef, -1, fk);
}
qtam_status cta_inverse_rows(qtam_plan *p, const void *d_coef, int batch, int plane, Fork &fk) {
  return rows_cta_all<false>(p, batch, const_cast<void *>(d_coef), plane, fk);
}

}  // namespace qtam
