// tinyrow.cuh -- rows shorter than 32 points (M = 4, 8, 16): the whole row in one thread's registers.
// Forward: B[j] = X[kc + jj] W[jj] at j = jj mod M (R6; the spectrum's zero pads implement R8),
// Y = (N M)^{-1/2} IFFT_M(B) (C47).  Inverse: G[jj] = sqrt(N/M) FFT_M(Y)[jj mod M] W[jj] (C49), written to
// Gb[jj] for the offsets that fall on the one-sided spectrum.
#pragma once
#include "device_plan.hpp"
#include "fftreg.cuh"
#include "thrbits.cuh"

namespace qtam {

// Row-median threshold (R11 and "threshold arithmetic") of a row held by one thread: the two middle
// order statistics by rank counting (M <= 16), every operation correctly rounded and unfused as in the oracle.
template <int M>
__device__ __forceinline__ void tiny_threshold(float2 (&v)[M], float kappa) {
  float mag[M];
#pragma unroll
  for (int e = 0; e < M; ++e) mag[e] = Bits<float>::mag(v[e].x, v[e].y);
  float lo = 0.f, hi = 0.f;
#pragma unroll
  for (int e = 0; e < M; ++e) {
    int less = 0, equal = 0;
#pragma unroll
    for (int j = 0; j < M; ++j) { less += mag[j] < mag[e] ? 1 : 0; equal += mag[j] == mag[e] ? 1 : 0; }
    if (less <= M / 2 - 1 && M / 2 - 1 < less + equal) lo = mag[e];
    if (less <= M / 2 && M / 2 < less + equal) hi = mag[e];
  }
  const float thr = Bits<float>::mul(kappa, Bits<float>::mul(0.5f, Bits<float>::add(lo, hi)));
#pragma unroll
  for (int e = 0; e < M; ++e) if (mag[e] < thr) v[e] = make_float2(0.f, 0.f);
}

template <int M, bool FORWARD, bool THRESH = false>
__device__ __forceinline__ void tiny_row(const FastRow &row, const float2 *__restrict__ X, const float *__restrict__ fwin,
                                         float2 *__restrict__ Y, float2 *__restrict__ Gb, int nbins, float scale,
                                         float kappa = 0.f) {
  float2 v[M];
  const float *W = fwin + row.woff + row.dk;
  if constexpr (FORWARD) {
#pragma unroll
    for (int j = 0; j < M; ++j) {
      const int jj = j < M / 2 ? j : j - M;
      v[j] = make_float2(0.f, 0.f);
      if (jj >= -row.dk && jj <= row.dk) v[j] = pscale(X[row.kc + jj], __ldg(W + jj) * scale);
    }
    RegFFT<M, +1>::run(v);
    if constexpr (THRESH) tiny_threshold<M>(v, kappa);
    float4 *dst = reinterpret_cast<float4 *>(Y);
#pragma unroll
    for (int j = 0; j < M / 2; ++j) __stcs(dst + j, make_float4(v[2 * j].x, v[2 * j].y, v[2 * j + 1].x, v[2 * j + 1].y));
  } else {
    const float4 *src = reinterpret_cast<const float4 *>(Y);
#pragma unroll
    for (int j = 0; j < M / 2; ++j) {
      const float4 q = __ldcs(src + j);
      v[2 * j] = make_float2(q.x, q.y); v[2 * j + 1] = make_float2(q.z, q.w);
    }
    RegFFT<M, -1>::run(v);
#pragma unroll
    for (int j = 0; j < M; ++j) {
      const int jj = j < M / 2 ? j : j - M;
      const int f = row.kc + jj;
      if (jj >= -row.dk && jj <= row.dk && (unsigned)f < (unsigned)nbins) Gb[jj] = pscale(v[j], __ldg(W + jj) * scale);
    }
  }
}

}  // namespace qtam
