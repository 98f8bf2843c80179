// rows_cluster.cu -- rows of 2^14 .. 2^17 points (float): one thread-block CLUSTER per (segment, row), the row's
// short FFT split over the cluster's CTAs with the engine of clfft.cuh.  (The classes of 2^15 and 2^16 points run
// as the dataflow of rows_split.cu -- 502 -> 372 us forward, 577 -> 420 us inverse at config 4 -- whenever their
// tables fit its shared memory; this kernel then serves 2^14 points, one CTA per row, and 2^17.)  Nothing but the compulsory bytes leaves
// the chip: the intermediate of the split transform crosses between the CTAs through distributed shared memory.
//
//   forward (a2 + a3)  every CTA gathers its residues of the band, X[kc + jj] W_k[jj] (N M)^{-1/2} (A9 :323,
//                      C46 :583, C47 :589), four consecutive bins every F bins, runs its four P-point
//                      sub-transforms in shared memory, and after one cluster barrier takes the radix-F stage for
//                      its P/CL values of nc: F inputs from the F/4 CTAs, F outputs Y[nc + P m] stored to every
//                      member of the leader's set (identical rows are transformed once).
//   inverse (a5 + a6)  the mirror image: the members' coefficient rows are added while they are loaded (Eq. 11's
//                      sum over k by linearity), radix-F stage, scattered to the CTAs, P-point sub-transforms,
//                      times sqrt(N/M) W_k (C49 :598), and ADDED into the partial spectrum of the leader's group:
//                      a group is a run of leaders consecutive in centre bin that one cluster takes one after the
//                      other, so every bin of the group's partial sum is updated in a fixed order by plain
//                      read-modify-write from one cluster (cluster barriers order the updates): a segmented
//                      reduction without atomics and without a band workspace.  The groups' partial sums are
//                      added up, in a fixed order, by k_combine_runs (combine_runs.cu).
// Classes: M = 4 P CL with P = 4096 (512 threads, one CTA per SM) and CL = 1, 2, 4, 8 CTAs per cluster for
// M = 2^14 .. 2^17 (CL = 1: no exchange at all).  Measured on cfg4 against P = 2048 with twice the CTAs per
// cluster and two CTAs per SM: the smaller cluster wins (less data through distributed shared memory, which
// moves about 20 B/cycle/SM, and fewer CTAs to wait for at the cluster barrier).
#include <cooperative_groups.h>

#include <algorithm>
#include <cmath>
#include <vector>

#include "clfft.cuh"
#include "device_plan.hpp"

namespace cg = cooperative_groups;

namespace qtam {

extern __shared__ __align__(16) unsigned char qtam_cl_smem[];

constexpr int kClLog2P = 12;

// Cluster barrier.  release / acquire (the default pair) orders memory across the cluster: the arrive waits
// until the CTA's earlier writes -- global ones too -- are performed, the wait invalidates L1.  The relaxed
// arrive only counts the CTA in: enough where the barrier says "I have finished READING your shared memory".
__device__ __forceinline__ void cl_arrive() { asm volatile("barrier.cluster.arrive.release.aligned;" ::: "memory"); }
__device__ __forceinline__ void cl_arrive_relaxed() { asm volatile("barrier.cluster.arrive.relaxed.aligned;" ::: "memory"); }
__device__ __forceinline__ void cl_wait() { asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory"); }

// Predicated loads as volatile asm: a batch of them stays a batch (issued back to back, in program order), instead
// of being interleaved with their uses by the scheduler when registers are tight -- every load of the batch then
// waits out its latency at the same time.  The value is zero when the predicate is off.
__device__ __forceinline__ float2 ld_nc_f2(const float2 *p, bool ok) {
  float2 v;
  asm volatile("{\n .reg .pred q;\n setp.ne.s32 q, %3, 0;\n mov.f32 %0, 0f00000000;\n mov.f32 %1, 0f00000000;\n"
               " @q ld.global.nc.v2.f32 {%0, %1}, [%2];\n}" : "=f"(v.x), "=f"(v.y) : "l"(p), "r"((int)ok));
  return v;
}
__device__ __forceinline__ float ld_nc_f1(const float *p, bool ok) {
  float v;
  asm volatile("{\n .reg .pred q;\n setp.ne.s32 q, %2, 0;\n mov.f32 %0, 0f00000000;\n"
               " @q ld.global.nc.f32 %0, [%1];\n}" : "=f"(v) : "l"(p), "r"((int)ok));
  return v;
}
__device__ __forceinline__ float2 ld_cg_f2(const float2 *p, bool ok) {
  float2 v;
  asm volatile("{\n .reg .pred q;\n setp.ne.s32 q, %3, 0;\n mov.f32 %0, 0f00000000;\n mov.f32 %1, 0f00000000;\n"
               " @q ld.global.cg.v2.f32 {%0, %1}, [%2];\n}" : "=f"(v.x), "=f"(v.y) : "l"(p), "r"((int)ok) : "memory");
  return v;
}
__device__ __forceinline__ float2 ld_cs_f2(const float2 *p) {
  float2 v;
  asm volatile("ld.global.cs.v2.f32 {%0, %1}, [%2];" : "=f"(v.x), "=f"(v.y) : "l"(p));
  return v;
}

struct ClArgs {
  const ClLeader *lead; const int2 *mem; int nlead;         // leaders of this class (ascending centre bin), members
  const ClGroup *groups; int ngroups;                       // inverse: groups of consecutive leaders
  const float *win;
  const float2 *spec; long long xstride; int nbins;
  float2 *coef; long long ctot;
  float2 *part; long long part_stride;
  const float2 *ptw, *ftw;                                  // sub-transform pass tables; radix-F twiddles (rows 1, 4)
  int batch, plane;
};

// Pass 1 of the forward's sub-transforms, straight from the spectrum: B[j] = X[kc + jj] W_k[jj] s at
// j = q + F jc (R6), zero off the support and off the one-sided spectrum (R8).  A butterfly's inputs sit at
// compile-time distances from its first one (jc = i + r P/R, and jc >= P/2 -- the negative offsets -- exactly for
// r >= R/2), so a load is one compare against a per-butterfly bound and one address with an immediate offset;
// all 2 R loads of a butterfly are issued before the first multiply.
template <int LOG2P, int F, class Mid>
__device__ __forceinline__ void cl_pass1_gather(float2 *s, const float2 *__restrict__ X, const float *__restrict__ W,
                                                int kc, int dk, int nbins, int q0, float scale, const Mid &mid) {
  typedef ClFft<LOG2P> PL;
  constexpr int P = PL::P, R = PL::R0, NBF = P / R, TPS = PL::NT / 4, BPT = NBF / TPS;
  const int ja = threadIdx.x & 3, ib = threadIdx.x >> 2;
  const int hi = min(dk, nbins - 1 - kc), lo = max(-dk, -kc);      // offsets jj kept: lo <= jj <= hi
  float2 v[BPT][R];
#pragma unroll
  for (int u = 0; u < BPT; ++u) {
    const int jj0 = q0 + ja + F * (ib + TPS * u);                  // offset of the butterfly's first input (r = 0)
    const float2 *Xp = X + kc + jj0;
    const float *Wp = W + jj0;
    const int a = hi - jj0, b = lo - jj0;
    float w[R];
#pragma unroll
    for (int r = 0; r < R; ++r) {
      constexpr int dummy = 0; (void)dummy;
      const int c = r * F * NBF - (r >= R / 2 ? F * P : 0);        // compile-time distance from the first input
      const bool ok = r < R / 2 ? c <= a : c >= b;
      v[u][r] = ld_nc_f2(Xp + c, ok);
      w[r] = ld_nc_f1(Wp + c, ok);
    }
#pragma unroll
    for (int r = 0; r < R; ++r) v[u][r] = pscale(v[u][r], w[r] * scale);
    RegFFT<R, +1>::run(v[u]);
  }
  mid();
#pragma unroll
  for (int u = 0; u < BPT; ++u) {
    const int i = ib + TPS * u;
#pragma unroll
    for (int r = 0; r < R; ++r) {
      const int a = i * R + r;
      s[4 * (a + (a >> 4)) + ja] = v[u][r];
    }
  }
}

template <int LOG2P, int LOG2CL, bool FWD>
__global__ void __launch_bounds__(ClFft<LOG2P>::NT, 1)
k_rows_cluster(const ClArgs A) {
  typedef ClFft<LOG2P> PL;
  constexpr int P = PL::P, NT = PL::NT, CL = 1 << LOG2CL, F = 4 * CL;
  constexpr int NCQ = P / CL;            // values of nc one CTA takes in the radix-F stage
  constexpr int BPTF = NCQ / NT;         // ... per thread
  static_assert(NCQ % NT == 0 && BPTF >= 1, "radix-F stage must divide among the threads");
  static_assert(PL::R0 == 16, "pass 1 writes the skew of radix 16");
  cg::cluster_group cluster = cg::this_cluster();
  const int crank = (int)cluster.block_rank();
  const int cid = blockIdx.x >> LOG2CL, ncl = gridDim.x >> LOG2CL;
  const int tid = threadIdx.x;
  float2 *s = reinterpret_cast<float2 *>(qtam_cl_smem);
  // the pass tables of the sub-transforms live in shared memory: the cluster barrier's acquire invalidates L1, so
  // table reads from global memory would go to L2 in every pass of every row
  float2 *stw = s + PL::SMEM_ELEMS;
  for (int i = tid; i < PL::PTW_ELEMS; i += NT) stw[i] = A.ptw[i];
  __syncthreads();
  float2 *rs[CL];
#pragma unroll
  for (int jb = 0; jb < CL; ++jb) rs[jb] = cluster.map_shared_rank(s, jb);
  __shared__ int s_nm;
  __shared__ int s_off[kCtaMaxMembers];
  bool pending = false;                  // a cluster-barrier arrive without its wait

  if constexpr (FWD) {
    const long long total = (long long)A.nlead * A.batch;
    for (long long item = cid; item < total; item += ncl) {
      const int seg = (int)(item / A.nlead);
      const ClLeader L = A.lead[item - (long long)seg * A.nlead];
      __syncthreads();                   // the previous item's stores have read s_off
      if (tid < L.nmem) s_off[tid] = A.mem[L.mem0 + tid].x;
      // sub-transforms: pass 1 straight from the spectrum
      auto before_write = [&]() { if (pending) { cl_wait(); pending = false; } };   // the others have read my last result
      cl_pass1_gather<LOG2P, F>(s, A.spec + (size_t)seg * A.xstride, A.win + L.woff + L.dk, L.kc, L.dk, A.nbins,
                                4 * crank, L.fwd_scale, before_write);
      __syncthreads();
      cl_passes_23<LOG2P, +1>(s, stw);
      cl_arrive();
      // radix-F stage for nc = crank NCQ .. + NCQ
      float2 *Yseg = A.coef + (size_t)seg * A.ctot;
      const int nm = L.nmem;
#pragma unroll 1
      for (int u = 0; u < BPTF; ++u) {
        const int nc = crank * NCQ + tid + NT * u;
        const float2 w1 = __ldg(A.ftw + nc), w4 = __ldg(A.ftw + P + nc);
        if (u == 0) cl_wait();           // every CTA's sub-transforms are in its shared memory
        float2 v[F];
#pragma unroll
        for (int jb = 0; jb < CL; ++jb) {
          const float4 *src = reinterpret_cast<const float4 *>(rs[jb] + 4 * nc);
          const float4 a = src[0], b = src[1];
          v[4 * jb] = make_float2(a.x, a.y); v[4 * jb + 1] = make_float2(a.z, a.w);
          v[4 * jb + 2] = make_float2(b.x, b.y); v[4 * jb + 3] = make_float2(b.z, b.w);
        }
        cl_twiddle<F>(v, w1, w4);
        RegFFT<F, +1>::run(v);
        for (int m = 0; m < nm; ++m) {
          float2 *Y = Yseg + s_off[m] + nc;
#pragma unroll
          for (int mm = 0; mm < F; ++mm) __stcs(Y + mm * P, v[mm]);
        }
      }
      cl_arrive_relaxed(); pending = true;   // done reading the others' shared memory; the stores drain on their own
    }
  } else {
    const long long total = (long long)A.ngroups * A.batch;
    for (long long item = cid; item < total; item += ncl) {
      const int seg = (int)(item / A.ngroups);
      const ClGroup Gp = A.groups[item - (long long)seg * A.ngroups];
      float2 *pg = A.part + (size_t)seg * A.part_stride + Gp.part_off;
      // the group's partial sum starts at zero (float4 stores: part_off and the padded length are even)
      {
        float4 *z = reinterpret_cast<float4 *>(pg);
        const int n4 = ((Gp.nb + 1) & ~1) / 2;
        for (int i = crank * NT + tid; i < n4; i += CL * NT) z[i] = make_float4(0.f, 0.f, 0.f, 0.f);
      }
      const float2 *Yseg = A.coef + (size_t)seg * A.ctot;
#pragma unroll 1
      for (int l = 0; l < Gp.nlead; ++l) {
        const ClLeader L = A.lead[Gp.lead0 + l];
        __syncthreads();
        if (tid < 32) {
          // members that take part (all of them, or those of the requested plane), compacted in order
          const bool ok = tid < L.nmem && (A.plane < 0 || A.mem[L.mem0 + tid].y == A.plane);
          const unsigned b = __ballot_sync(0xffffffffu, ok);
          if (ok) s_off[__popc(b & ((1u << tid) - 1u))] = A.mem[L.mem0 + tid].x;
          if (tid == 0) s_nm = __popc(b);
        }
        __syncthreads();
        const int nm = s_nm;
        if (nm == 0) continue;           // the same decision in every CTA of the cluster
        // radix-F stage on the sum of the members' rows, scattered to the CTA that owns the residue
#pragma unroll 1
        for (int u = 0; u < BPTF; ++u) {
          const int nc = crank * NCQ + tid + NT * u;
          float2 w1 = __ldg(A.ftw + nc), w4 = __ldg(A.ftw + P + nc);
          float2 v[F];
          {
            const float2 *Y = Yseg + s_off[0] + nc;
#pragma unroll
            for (int mm = 0; mm < F; ++mm) v[mm] = ld_cs_f2(Y + mm * P);
          }
          for (int m = 1; m < nm; ++m) {
            const float2 *Y = Yseg + s_off[m] + nc;
            float2 y[F];
#pragma unroll
            for (int mm = 0; mm < F; ++mm) y[mm] = ld_cs_f2(Y + mm * P);
#pragma unroll
            for (int mm = 0; mm < F; ++mm) v[mm] = padd(v[mm], y[mm]);
          }
          RegFFT<F, -1>::run(v);
          w1.y = -w1.y; w4.y = -w4.y;
          cl_twiddle<F>(v, w1, w4);
          if (pending) { cl_wait(); pending = false; }     // every CTA is done with the previous row's result
#pragma unroll
          for (int jb = 0; jb < CL; ++jb) {
            float4 *dst = reinterpret_cast<float4 *>(rs[jb] + 4 * nc);
            dst[0] = make_float4(v[4 * jb].x, v[4 * jb].y, v[4 * jb + 1].x, v[4 * jb + 1].y);
            dst[1] = make_float4(v[4 * jb + 2].x, v[4 * jb + 2].y, v[4 * jb + 3].x, v[4 * jb + 3].y);
          }
        }
        cl_arrive(); cl_wait();
        // the four sub-transforms of this CTA's residues
        cl_pass<LOG2P, PL::R0, 0, -1, 0, true>(s, ClNoMid{}, ClSyncMid{}, stw);
        __syncthreads();
        cl_passes_23<LOG2P, -1>(s, stw);
        // G_k[jj] = sqrt(N/M) Bhat[jj] W_k[jj], added into the group's partial sum at bin kc + jj (R8 clip).
        // The loads of a batch are issued before its stores (a store may not be overtaken by a later load of
        // the same array, which would serialise the round trips to L2).
        {
          const int ja = tid & 3, ib = tid >> 2;
          const float *W = A.win + L.woff + L.dk;
          float2 *pb = pg + (L.kc - Gp.lo);
          constexpr int TPS = NT / 4, CH = 8;
          static_assert(P % (CH * TPS) == 0, "batches must tile the sub-transform");
#pragma unroll 1
          for (int jc0 = ib; jc0 < P; jc0 += CH * TPS) {
            float2 old[CH]; float w[CH]; int jjs[CH];
#pragma unroll
            for (int c = 0; c < CH; ++c) {
              const int jc = jc0 + c * TPS;
              const int jj = 4 * crank + ja + F * jc - (jc >= P / 2 ? F * P : 0);
              const int f = L.kc + jj;
              const bool ok = jj >= -L.dk && jj <= L.dk && (unsigned)f < (unsigned)A.nbins;
              jjs[c] = ok ? jj : (1 << 30);
              old[c] = ld_cg_f2(pb + jj, ok);
              w[c] = ld_nc_f1(W + jj, ok);
            }
#pragma unroll
            for (int c = 0; c < CH; ++c)
              if (jjs[c] != (1 << 30)) {
                const float a = L.inv_amp * w[c];
                pb[jjs[c]] = pfma(s[4 * (jc0 + c * TPS) + ja], make_float2(a, a), old[c]);
              }
          }
        }
        cl_arrive(); pending = true;     // release: the next row's updates of these bins may come from another CTA
      }
    }
  }
  if (pending) cl_wait();                // nobody leaves while a neighbour may still read its shared memory
}

// --------------------------------------------------------------------------------------------------
// host side
// --------------------------------------------------------------------------------------------------
// class c = log2 M - kClLog2Min = log2 CL: the sub-transforms have P = 2^kClLog2P points in every class
template <int LOG2P, int LOG2CL> static bool prepare_cl(qtam_plan *p, int c) {
  typedef ClFft<LOG2P> PL;
  const size_t smem = sizeof(float2) * (size_t)(PL::SMEM_ELEMS + PL::PTW_ELEMS);
  for (int fwd = 0; fwd < 2; ++fwd) {
    KernelCfg &cfg = p->cfg_rows_cl[c][fwd];
    cfg.smem = smem; cfg.occ = 0; cfg.ready = false;
    const void *kern = fwd ? (const void *)k_rows_cluster<LOG2P, LOG2CL, true> : (const void *)k_rows_cluster<LOG2P, LOG2CL, false>;
    if (!raise_dynamic_smem(kern, smem)) return false;
    cudaLaunchConfig_t lc = {};
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeClusterDimension;
    at[0].val.clusterDim.x = 1 << LOG2CL; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
    lc.gridDim = dim3((unsigned)(p->num_sms / (1 << LOG2CL)) << LOG2CL);
    lc.blockDim = dim3(PL::NT); lc.dynamicSmemBytes = smem; lc.attrs = at; lc.numAttrs = 1;
    int ncl = 0;
    if (cudaOccupancyMaxActiveClusters(&ncl, kern, &lc) != cudaSuccess || ncl < 1) return false;
    cfg.occ = ncl;                       // clusters that can be resident at once
    cfg.ready = true;
  }
  return true;
}

qtam_status build_rows_cluster(qtam_plan *p) {
  const HostPlan &hp = p->hp;
  p->cl_rows = false;
  if (!p->fast_rows) return QTAM_OK;
  auto up = [&](void **dst, const void *src, size_t bytes) -> bool {
    *dst = nullptr;
    if (cudaMalloc(dst, bytes ? bytes : 16) != cudaSuccess) return false;
    p->device_bytes += bytes;
    return bytes == 0 || cudaMemcpy(*dst, src, bytes, cudaMemcpyHostToDevice) == cudaSuccess;
  };
  for (int c = 0; c < kClClasses; ++c) {
    const int lm = kClLog2Min + c;
    const int64_t M = int64_t(1) << lm;
    std::vector<int> idx;
    for (size_t k = 0; k < hp.rows.size(); ++k)
      if (hp.rows[k].M == M) { idx.push_back((int)k); p->cl_sumM[c] += (double)M; p->cl_sumL[c] += (double)hp.rows[k].L; }
    p->n_cl_lead[c] = 0; p->n_cl_groups[c] = 0;
    if (idx.empty()) continue;
    std::vector<ClLeader> lead;
    std::vector<int2> mem;
    std::vector<ClGroup> groups;
    // about ten groups per class: (groups x segments) spreads over the resident clusters while the partial sums
    // stay a fraction of the band values
    // the classes of 2^15 and 2^16 points run as the dataflow of rows_split.cu (partial sums sorted by residue)
    // when their tables fit its shared memory; one CTA holds a 2^14-point row, and the 2^17-point rows stay here
    bool by_residue = false;
    const bool want = c == 1 || c == 2;
    build_leaders_and_groups(p, idx, want ? 6 : 10, lead, mem, groups, want ? split_max_leaders() : 0,
                             want ? split_max_members() : 0, &by_residue);
    p->n_cl_lead[c] = (int)lead.size(); p->n_cl_groups[c] = (int)groups.size();
    if (!up(reinterpret_cast<void **>(&p->d_cl_lead[c]), lead.data(), lead.size() * sizeof(ClLeader))) return QTAM_ERR_ALLOC;
    if (!up(reinterpret_cast<void **>(&p->d_cl_mem[c]), mem.data(), mem.size() * sizeof(int2))) return QTAM_ERR_ALLOC;
    if (!up(reinterpret_cast<void **>(&p->d_cl_groups[c]), groups.data(), groups.size() * sizeof(ClGroup))) return QTAM_ERR_ALLOC;
    std::vector<float> t;
    fill_clfft_final(t, ClFft<kClLog2P>::P, M);
    if (!up(&p->d_cl_ftw[c], t.data(), t.size() * sizeof(float))) return QTAM_ERR_ALLOC;

    bool ok = false;
    switch (c) {
      case 0: ok = prepare_cl<kClLog2P, 0>(p, c); break;
      case 1: ok = prepare_cl<kClLog2P, 1>(p, c); break;
      case 2: ok = prepare_cl<kClLog2P, 2>(p, c); break;
      default: ok = prepare_cl<kClLog2P, 3>(p, c); break;
    }
    if (!ok) return QTAM_ERR_CUDA;
    p->cl_rows = true;
    if (by_residue) {
      const qtam_status ss = build_rows_split(p, c, lead, mem, groups);
      if (ss != QTAM_OK) return ss;
    }
  }
  if (p->cl_rows) {
    std::vector<float> t;
    fill_clfft_tables<kClLog2P>(t);
    if (!up(&p->d_cl_ptw, t.data(), t.size() * sizeof(float))) return QTAM_ERR_ALLOC;
  }
  return QTAM_OK;
}

template <int LOG2P, int LOG2CL, bool FWD>
static qtam_status cl_launch(qtam_plan *p, int c, int batch, void *d_coef, int plane, cudaStream_t st) {
  typedef ClFft<LOG2P> PL;
  if (p->n_cl_lead[c] == 0) return QTAM_OK;
  const KernelCfg &cfg = p->cfg_rows_cl[c][FWD ? 1 : 0];
  if (!cfg.ready) return QTAM_ERR_CUDA;
  ClArgs A{};
  A.lead = p->d_cl_lead[c]; A.mem = p->d_cl_mem[c]; A.nlead = p->n_cl_lead[c];
  A.groups = p->d_cl_groups[c]; A.ngroups = p->n_cl_groups[c];
  A.win = static_cast<const float *>(p->d_win);
  A.spec = static_cast<const float2 *>(p->d_spec); A.xstride = p->xstride; A.nbins = (int)p->hp.nb;
  A.coef = static_cast<float2 *>(d_coef); A.ctot = p->hp.ctot;
  A.part = static_cast<float2 *>(p->d_part); A.part_stride = p->part_stride;
  A.ptw = static_cast<const float2 *>(p->d_cl_ptw);
  A.ftw = static_cast<const float2 *>(p->d_cl_ftw[c]);
  A.batch = batch; A.plane = plane;
  const long long items = (long long)(FWD ? A.nlead : A.ngroups) * batch;
  const long long ncl = std::min<long long>(items, cfg.occ);
  cudaLaunchConfig_t lc = {};
  cudaLaunchAttribute at[1];
  at[0].id = cudaLaunchAttributeClusterDimension;
  at[0].val.clusterDim.x = 1 << LOG2CL; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
  lc.gridDim = dim3((unsigned)(ncl << LOG2CL)); lc.blockDim = dim3(PL::NT);
  lc.dynamicSmemBytes = cfg.smem; lc.stream = st; lc.attrs = at; lc.numAttrs = 1;
  const double bytes = (double)batch * 8.0 * p->cl_sumM[c];       // compulsory: the coefficients
  {
    LaunchScope ls(p, st, (KernelId)((FWD ? K_ROWS_L14_FWD : K_ROWS_L14_INV) + c), bytes, bytes + (double)batch * 8.0 * p->cl_sumL[c]);
    if (cudaLaunchKernelEx(&lc, k_rows_cluster<LOG2P, LOG2CL, FWD>, A) != cudaSuccess) return QTAM_ERR_CUDA;
  }
  QTAM_LAUNCH_CHECK();
  return QTAM_OK;
}

// every class on a stream of its own, the longest rows first (the classes write disjoint coefficients / partial sums)
template <bool FWD>
static qtam_status cl_all(qtam_plan *p, int batch, void *d_coef, int plane, Fork &fk) {
  qtam_status s = QTAM_OK;
  if (p->n_cl_lead[3]) s = cl_launch<kClLog2P, 3, FWD>(p, 3, batch, d_coef, plane, fk.next());
  // the dataflow classes share one stream: the forward's residue-sorted copy of the spectrum (k_spec_residues) goes
  // first on it, so that only they wait for it -- every other row kernel of the call starts right after the long FFT
  cudaStream_t sx = nullptr;
  bool have_sx = false;
  auto split_stream = [&]() -> cudaStream_t {
    if (!have_sx) {
      sx = fk.next(); have_sx = true;
      if (FWD && s == QTAM_OK) s = split_spectrum(p, batch, sx);
    }
    return sx;
  };
  if (s == QTAM_OK && p->n_cl_lead[2]) {
    if (p->sp_ok[2]) { cudaStream_t t = split_stream(); if (s == QTAM_OK) s = split_rows(p, 2, FWD, batch, d_coef, plane, t); }
    else s = cl_launch<kClLog2P, 2, FWD>(p, 2, batch, d_coef, plane, fk.next());
  }
  if (s == QTAM_OK && p->n_cl_lead[1]) {
    if (p->sp_ok[1]) { cudaStream_t t = split_stream(); if (s == QTAM_OK) s = split_rows(p, 1, FWD, batch, d_coef, plane, t); }
    else s = cl_launch<kClLog2P, 1, FWD>(p, 1, batch, d_coef, plane, fk.next());
  }
  if (s == QTAM_OK && p->n_cl_lead[0]) s = cl_launch<kClLog2P, 0, FWD>(p, 0, batch, d_coef, plane, fk.next());
  return s;
}

qtam_status cluster_forward_rows(qtam_plan *p, int batch, void *d_coef, Fork &fk) {
  return cl_all<true>(p, batch, d_coef, -1, fk);
}
qtam_status cluster_inverse_rows(qtam_plan *p, const void *d_coef, int batch, int plane, Fork &fk) {
  return cl_all<false>(p, batch, const_cast<void *>(d_coef), plane, fk);
}

}  // namespace qtam
