// threshold_fast.cu -- a4, the row-median threshold of BASELINE.json config 5 (R11), for rows
// of up to 1024 points: the row lives in registers, the median is found by a radix select over the bit
// patterns of the magnitudes inside a warp (no shared memory, no block barrier).
//
// A row of M = 32 G points is held by G lanes (32 magnitudes per lane, 32/G rows per warp); rows of
// 4, 8 or 16 points by one lane each (32 rows per warp).  The select walks the bits from the most
// significant one down; per bit every lane counts its candidates with a 0 there and the G lanes add
// their counts with shuffles.  The two middle order statistics, their mean, the threshold and the
// comparison use the correctly rounded, unfused operations of thrbits.cuh, so the decisions are those
// of the oracle bit for bit.  One read and one (predicated) write of the coefficients.
#include <algorithm>
#include <vector>

#include "cplx.cuh"
#include "device_plan.hpp"
#include "thrselect.cuh"

namespace qtam {

static int ilog2(long long v) { int l = 0; while ((1LL << l) < v) ++l; return l; }

qtam_status build_thr_fast(qtam_plan *p) {
  const HostPlan &hp = p->hp;
  std::vector<int> offs;
  std::vector<ThrTask> tasks;
  // offsets are kept as 32-bit integers: a plan with more coefficients per segment stays on the generic kernel
  const bool fits = hp.ctot < (int64_t(1) << 31);
  for (int lm = 0; lm <= kThrFastLog2Max; ++lm) { p->thr_first[lm] = 0; p->thr_count[lm] = 0; }
  for (int lm = kThrFastLog2Max; fits && lm >= 2; --lm) {
    const int M = 1 << lm, G = M >= 32 ? M / 32 : 1, per = 32 / G;
    p->thr_first[lm] = (int)tasks.size();
    std::vector<int> mine;
    for (const HostRow &h : hp.rows) if (h.M == M) mine.push_back((int)h.offset);
    for (size_t i = 0; i < mine.size(); i += (size_t)per) {
      ThrTask t{};
      t.log2M = lm; t.row0 = (int)offs.size(); t.nrows = (int)std::min(mine.size() - i, (size_t)per);
      for (int r = 0; r < t.nrows; ++r) offs.push_back(mine[i + (size_t)r]);
      tasks.push_back(t);
    }
    p->thr_count[lm] = (int)tasks.size() - p->thr_first[lm];
  }
  p->n_thr_tasks = (int)tasks.size();
  p->thr_has_big = false;
  for (const HostRow &h : hp.rows) if (!fits || ilog2(h.M) > kThrFastLog2Max) p->thr_has_big = true;
  auto up = [&](void **dst, const void *src, size_t bytes) -> bool {
    *dst = nullptr;
    if (cudaMalloc(dst, bytes ? bytes : 16) != cudaSuccess) return false;
    p->device_bytes += bytes;
    return cudaMemcpy(*dst, src, bytes, cudaMemcpyHostToDevice) == cudaSuccess || bytes == 0;
  };
  if (!up(reinterpret_cast<void **>(&p->d_thr_tasks), tasks.data(), tasks.size() * sizeof(ThrTask))) return QTAM_ERR_ALLOC;
  if (!up(reinterpret_cast<void **>(&p->d_thr_offs), offs.data(), offs.size() * sizeof(int))) return QTAM_ERR_ALLOC;
  return QTAM_OK;
}

// One group of G lanes, E values per lane (M = E G): the row lives in registers (thrselect.cuh).
template <typename T, int E>
__device__ __forceinline__ void thr_group(C2<T> *__restrict__ Y, int G, int t, T kappa) {
  typedef typename Bits<T>::U U;
  typedef C2<T> V;
  U x[E];
  U vor = 0, vand = ~(U)0;
#pragma unroll
  for (int e = 0; e < E; ++e) {
    V y = cmk<T>(0, 0);
    if (Y) y = Y[t + G * e];
    x[e] = Bits<T>::of(Bits<T>::add(Bits<T>::mul(y.x, y.x), Bits<T>::mul(y.y, y.y)));
    if (Y) { vor |= x[e]; vand &= x[e]; }
  }
  U prefix;
  const U cut = thr_select<T, E>(x, vor, vand, G, kappa, prefix);
  if (Y) {
#pragma unroll
    for (int e = 0; e < E; ++e)
      if ((x[e] ^ prefix) < cut) Y[t + G * e] = cmk<T>(0, 0);
  }
}

// One kernel per row length: the select of one length is a few thousand fully unrolled instructions (more in double
// precision), and a kernel that switched between all lengths ran out of instruction cache (ncu: "no instruction" was
// the first stall reason of the double-precision kernel, 424 us at config 5).
template <typename T, int NW, int LM>
__global__ void __launch_bounds__(NW * 32)
k_threshold_fast(const ThrTask *__restrict__ tasks, int n_tasks, const int *__restrict__ offs,
                 C2<T> *__restrict__ coef, long long ctot, int batch, T kappa) {
  const int lane = threadIdx.x & 31;
  const long long item = (long long)blockIdx.x * NW + (threadIdx.x >> 5);
  if (item >= (long long)n_tasks * batch) return;
  const int seg = (int)(item / n_tasks);
  const ThrTask tk = tasks[item - (long long)seg * n_tasks];
  constexpr int M = 1 << LM;
  constexpr int G = M >= 32 ? M >> 5 : 1;
  const int t = lane & (G - 1), rw = lane / G;
  C2<T> *Y = nullptr;
  if (rw < tk.nrows) Y = coef + (size_t)seg * ctot + offs[tk.row0 + rw];
  if constexpr (LM < 5) thr_group<T, M>(Y, 1, 0, kappa);           // rows of 4, 8, 16 points: one lane each
  else thr_group<T, 32>(Y, G, t, kappa);                           // (the lanes-per-row count is a literal)
}

template <typename T>
static qtam_status thr_launch(qtam_plan *p, void *d_coef, int batch, double kappa, cudaStream_t st) {
  constexpr int NW = 4;
  const long long total = (long long)p->n_thr_tasks * batch;
  if (total == 0) return QTAM_OK;
  double elems = 0;
  for (const HostRow &h : p->hp.rows) if (ilog2(h.M) <= kThrFastLog2Max) elems += (double)h.M;
  {
    // a separate threshold pass moves no compulsory bytes (zero extra when fused)
    LaunchScope ls(p, st, K_THRESHOLD_FAST, 0.0, 2.0 * sizeof(C2<T>) * (double)batch * elems);
    C2<T> *Y = static_cast<C2<T> *>(d_coef);
    int launched = 0;
#define QTAM_THR_LM(LM)                                                                                        \
    if (p->thr_count[LM] > 0) {                                                                                \
      const long long n = (long long)p->thr_count[LM] * batch;                                                 \
      k_threshold_fast<T, NW, LM><<<(unsigned)((n + NW - 1) / NW), NW * 32, 0, st>>>(                          \
          p->d_thr_tasks + p->thr_first[LM], p->thr_count[LM], p->d_thr_offs, Y, p->hp.ctot, batch, (T)kappa); \
      ++launched;                                                                                              \
    }
    QTAM_THR_LM(10) QTAM_THR_LM(9) QTAM_THR_LM(8) QTAM_THR_LM(7) QTAM_THR_LM(6) QTAM_THR_LM(5)
    QTAM_THR_LM(4) QTAM_THR_LM(3) QTAM_THR_LM(2)
#undef QTAM_THR_LM
    if (launched > 1) p->last_launches += launched - 1;      // (the scope counted one)
  }
  QTAM_LAUNCH_CHECK();
  return QTAM_OK;
}

qtam_status fast_threshold(qtam_plan *p, void *d_coef, int batch, double kappa, cudaStream_t st) {
  return p->esz == 4 ? thr_launch<float>(p, d_coef, batch, kappa, st)
                     : thr_launch<double>(p, d_coef, batch, kappa, st);
}

}  // namespace qtam
