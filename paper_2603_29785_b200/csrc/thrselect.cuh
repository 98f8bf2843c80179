// thrselect.cuh -- the row-median threshold's order-statistic select on values held in registers
// (R11): shared by k_threshold_fast and the fused forward + threshold.
#pragma once
#include "thrbits.cuh"

namespace qtam {

// One group of G lanes, E values per lane (M = E G).  `has_row`: the lane holds a row.
//
// The select runs on a = fl(fl(re re) + fl(im im)) instead of mag = fl(sqrt(a)): the correctly rounded
// square root is non-decreasing, so the k-th smallest magnitude is fl(sqrt(k-th smallest a)), and
// "mag < thr" holds exactly for a < a*, a* the smallest value whose rounded root reaches thr (found by
// stepping through neighbouring bit patterns).  One square root per order statistic instead of one
// per coefficient; every decision is still the one DESIGN.md's threshold arithmetic defines.
// In: x[e] = bit pattern of a = fl(fl(re re) + fl(im im)) of the lane's E values (0 without a row), vor / vand
// = OR / AND of the lane's patterns.  Out: x[e] = a ^ prefix; returns the cut a* (zero iff (x[e] ^ prefix) < cut).
// All 32 lanes of the warp must call it together (the G lanes of a row exchange counts with shuffles).
template <typename T, int E>
__device__ __forceinline__ typename Bits<T>::U thr_select(typename Bits<T>::U (&x)[E], typename Bits<T>::U vor,
                                                           typename Bits<T>::U vand, int G, T kappa,
                                                           typename Bits<T>::U &prefix_out) {
  typedef typename Bits<T>::U U;
  const int M = E * G;
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
  prefix_out = prefix;
  return cut;
}

}  // namespace qtam
