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
#include "thrbits.cuh"

namespace qtam {

#define QTAM_LAUNCH_CHECK()                                         \
  do {                                                              \
    if (cudaPeekAtLastError() != cudaSuccess) return QTAM_ERR_CUDA; \
  } while (0)

static int ilog2(long long v) { int l = 0; while ((1LL << l) < v) ++l; return l; }

qtam_status build_thr_fast(qtam_plan *p) {
  const HostPlan &hp = p->hp;
  std::vector<int> offs;
  std::vector<ThrTask> tasks;
  // offsets are kept as 32-bit integers: a plan with more coefficients per segment stays on the generic kernel
  const bool fits = hp.ctot < (int64_t(1) << 31);
  for (int lm = kThrFastLog2Max; fits && lm >= 2; --lm) {
    const int M = 1 << lm, G = M >= 32 ? M / 32 : 1, per = 32 / G;
    std::vector<int> mine;
    for (const HostRow &h : hp.rows) if (h.M == M) mine.push_back((int)h.offset);
    for (size_t i = 0; i < mine.size(); i += (size_t)per) {
      ThrTask t{};
      t.log2M = lm; t.row0 = (int)offs.size(); t.nrows = (int)std::min(mine.size() - i, (size_t)per);
      for (int r = 0; r < t.nrows; ++r) offs.push_back(mine[i + (size_t)r]);
      tasks.push_back(t);
    }
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

// One group of G lanes, E values per lane (M = E G).  `Y`: the lane's row (nullptr: no row).
//
// The select runs on a = fl(fl(re re) + fl(im im)) instead of mag = fl(sqrt(a)): the correctly rounded
// square root is non-decreasing, so the k-th smallest magnitude is fl(sqrt(k-th smallest a)), and
// "mag < thr" holds exactly for a < a*, a* the smallest value whose rounded root reaches thr (found by
// stepping through neighbouring bit patterns).  One square root per order statistic instead of one
// per coefficient; every decision is still the one DESIGN.md's threshold arithmetic defines.
template <typename T, int E>
__device__ __forceinline__ void thr_group(C2<T> *__restrict__ Y, int G, int t, T kappa) {
  typedef typename Bits<T>::U U;
  typedef C2<T> V;
  const int M = E * G;
  U x[E];          // a ^ prefix: a value is still a candidate at `bit` iff x < 2^(bit+1)
  U vor = 0, vand = ~(U)0;
#pragma unroll
  for (int e = 0; e < E; ++e) {
    V y = cmk<T>(0, 0);
    if (Y) y = Y[t + G * e];
    x[e] = Bits<T>::of(Bits<T>::add(Bits<T>::mul(y.x, y.x), Bits<T>::mul(y.y, y.y)));
    if (Y) { vor |= x[e]; vand &= x[e]; }
  }
  for (int o = G >> 1; o > 0; o >>= 1) {
    vor |= __shfl_xor_sync(0xffffffffu, vor, o);
    vand &= __shfl_xor_sync(0xffffffffu, vand, o);
  }
  // bits on which every value of the row agrees belong to every order statistic
  const U diff = vor ^ vand;
  U prefix = vand & ~diff;
  int top = Bits<T>::nbits - 1;
  while (top >= 0 && !((diff >> top) & 1)) --top;
  {
    const U hi_mask = top >= Bits<T>::nbits - 1 ? (U)0 : ~((((U)1) << (top + 1)) - 1);
    prefix &= hi_mask;
  }
  int kk = M / 2 - 1;
  int alive = M;
  // Short cut: the squared magnitudes of a noise row are close to exponentially distributed, so the
  // median sits near ln 2 times their mean.  The aligned block of bit patterns that contains
  // mean ln2 (1 -+ 2.5/sqrt(M)) is tested with one exact counting pass; when the wanted order statistic
  // lies inside it (it nearly always does), the select starts at the block's prefix and needs about
  // log2(block population) steps instead of one per undecided exponent and mantissa bit.  A wrong guess
  // costs the counting pass and nothing else: every decision below is still exact.
  {
    float sum = 0.f;
#pragma unroll
    for (int e = 0; e < E; ++e) sum += (float)Bits<T>::from(x[e]);
    for (int o = G >> 1; o > 0; o >>= 1) sum += __shfl_xor_sync(0xffffffffu, sum, o);
    const float est = 0.6931472f * sum / (float)M;
    const float dl = fminf(0.9f, 2.5f * rsqrtf((float)M));
    const U blo = Bits<T>::of((T)(est * (1.f - dl))), bhi = Bits<T>::of((T)(est * (1.f + dl)));
    int sb = 0;
    U P = 0, Pend = 0;
    const bool sane = blo > 0 && blo <= bhi && bhi < Bits<T>::inf_bits();
    if (sane) {
      const U d = blo ^ bhi;
      sb = d == 0 ? 0 : Bits<T>::nbits - (sizeof(U) == 8 ? __clzll((long long)d) : __clz((int)d));
      P = (blo >> sb) << sb;
      Pend = P + (((U)1) << sb);
    }
    int c_lo = 0, c_hi = 0;
#pragma unroll
    for (int e = 0; e < E; ++e) {
      c_lo += (x[e] < P) ? 1 : 0;
      c_hi += (x[e] < Pend) ? 1 : 0;
    }
    for (int o = G >> 1; o > 0; o >>= 1) {
      c_lo += __shfl_xor_sync(0xffffffffu, c_lo, o);
      c_hi += __shfl_xor_sync(0xffffffffu, c_hi, o);
    }
    if (sane && c_lo <= kk && kk < c_hi && sb - 1 < top) {
      prefix = P; top = sb - 1; kk -= c_lo; alive = c_hi - c_lo;
    }
  }
#pragma unroll
  for (int e = 0; e < E; ++e) x[e] ^= prefix;
  // rank kk among the candidates, most significant undecided bit first; stops when one candidate is left
  int bit = top;
  // (the groups of a warp sit at different bits and stop at different times, but all lanes take the
  // shuffles together: a finished group counts against a zero limit and changes nothing)
#pragma unroll 1
  for (;;) {
    const bool active = bit >= 0 && alive > 1;
    if (!__any_sync(0xffffffffu, active)) break;
    const U lim = active ? ((U)1) << bit : (U)0;
    int c0 = 0;
#pragma unroll
    for (int e = 0; e < E; ++e) c0 += (x[e] < lim) ? 1 : 0;
    for (int o = G >> 1; o > 0; o >>= 1) c0 += __shfl_xor_sync(0xffffffffu, c0, o);
    if (active) {
      if (kk >= c0) {
        kk -= c0; alive -= c0; prefix |= lim;
#pragma unroll
        for (int e = 0; e < E; ++e) x[e] ^= lim;
      } else {
        alive = c0;
      }
      --bit;
    }
  }
  {
    // a single candidate left: the one value whose undecided bits are still below 2^(bit+1)
    const U lim2 = bit >= 0 ? ((U)2) << bit : (U)0;     // bit + 1 <= nbits - 1
    U low = 0;
#pragma unroll
    for (int e = 0; e < E; ++e) if (x[e] < lim2) low = x[e];
    for (int o = G >> 1; o > 0; o >>= 1) low |= __shfl_xor_sync(0xffffffffu, low, o);
    prefix |= low;
#pragma unroll
    for (int e = 0; e < E; ++e) x[e] ^= low;
  }
  // now x = a ^ a_lo.  Next order statistic: a_lo again if enough values are <= a_lo, else the
  // smallest value above it
  int cle = 0;
  U mn = ~(U)0;
#pragma unroll
  for (int e = 0; e < E; ++e) {
    const U a = x[e] ^ prefix;
    if (a <= prefix) ++cle;
    else if (a < mn) mn = a;
  }
  for (int o = G >> 1; o > 0; o >>= 1) {
    cle += __shfl_xor_sync(0xffffffffu, cle, o);
    const U other = __shfl_xor_sync(0xffffffffu, mn, o);
    if (other < mn) mn = other;
  }
  const T lo = Bits<T>::root(Bits<T>::from(prefix));
  const T hi = (cle >= M / 2 + 1) ? lo : Bits<T>::root(Bits<T>::from(mn));
  const T med = Bits<T>::mul((T)0.5, Bits<T>::add(lo, hi));
  const T thr = Bits<T>::mul(kappa, med);
  // a* = the smallest non-negative value with root(a*) >= thr (bit patterns of non-negative values are
  // ordered); thr = 0 or NaN: nothing is below it
  U cut = 0;
  if (thr > (T)0) {
    cut = Bits<T>::of(Bits<T>::mul(thr, thr));
    const U infbits = Bits<T>::inf_bits();
    if (cut > infbits) cut = infbits;
    while (cut > 0 && !(Bits<T>::root(Bits<T>::from(cut - 1)) < thr)) --cut;
    while (cut < infbits && Bits<T>::root(Bits<T>::from(cut)) < thr) ++cut;
  }
  if (Y) {
#pragma unroll
    for (int e = 0; e < E; ++e)
      if ((x[e] ^ prefix) < cut) Y[t + G * e] = cmk<T>(0, 0);
  }
}

template <typename T, int NW>
__global__ void __launch_bounds__(NW * 32)
k_threshold_fast(const ThrTask *__restrict__ tasks, int n_tasks, const int *__restrict__ offs,
                 C2<T> *__restrict__ coef, long long ctot, int batch, T kappa) {
  const int lane = threadIdx.x & 31;
  const long long item = (long long)blockIdx.x * NW + (threadIdx.x >> 5);
  if (item >= (long long)n_tasks * batch) return;
  const int seg = (int)(item / n_tasks);
  const ThrTask tk = tasks[item - (long long)seg * n_tasks];
  const int M = 1 << tk.log2M;
  const int G = M >= 32 ? M >> 5 : 1;
  const int t = lane & (G - 1), rw = lane / G;
  C2<T> *Y = nullptr;
  if (rw < tk.nrows) Y = coef + (size_t)seg * ctot + offs[tk.row0 + rw];
  switch (tk.log2M) {
    case 2: thr_group<T, 4>(Y, 1, 0, kappa); break;
    case 3: thr_group<T, 8>(Y, 1, 0, kappa); break;
    case 4: thr_group<T, 16>(Y, 1, 0, kappa); break;
    default: thr_group<T, 32>(Y, G, t, kappa); break;
  }
}

template <typename T>
static qtam_status thr_launch(qtam_plan *p, void *d_coef, int batch, double kappa, cudaStream_t st) {
  constexpr int NW = 4;
  const long long total = (long long)p->n_thr_tasks * batch;
  if (total == 0) return QTAM_OK;
  double elems = 0;
  for (const HostRow &h : p->hp.rows) if (ilog2(h.M) <= kThrFastLog2Max) elems += (double)h.M;
  {
    LaunchScope ls(p, st, K_THRESHOLD_FAST, 2.0 * sizeof(C2<T>) * (double)batch * elems);
    k_threshold_fast<T, NW><<<(unsigned)((total + NW - 1) / NW), NW * 32, 0, st>>>(
        p->d_thr_tasks, p->n_thr_tasks, p->d_thr_offs, static_cast<C2<T> *>(d_coef), p->hp.ctot, batch, (T)kappa);
  }
  QTAM_LAUNCH_CHECK();
  return QTAM_OK;
}

qtam_status fast_threshold(qtam_plan *p, void *d_coef, int batch, double kappa, cudaStream_t st) {
  return p->esz == 4 ? thr_launch<float>(p, d_coef, batch, kappa, st)
                     : thr_launch<double>(p, d_coef, batch, kappa, st);
}

}  // namespace qtam
