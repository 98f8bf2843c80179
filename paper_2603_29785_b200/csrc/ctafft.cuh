// ctafft.cuh -- one long complex FFT per CTA in shared memory (the half-length FFT behind the long
// real transforms a1 / a8), float, Nc = 2^11 .. 2^14 points.
// Stockham autosort in place: every pass loads its butterflies into registers, the CTA synchronises,
// and the results go back to their autosorted positions; 2-3 passes of radix 8/16/32 done with the
// in-register FFTs of fftreg.cuh.  Pass 1 writes with stride R, so it writes a skewed layout
// phys(a) = a + (a >> log2 R1) that the second pass reads back; later passes use the natural layout.
#pragma once
#include <cmath>
#include <vector>

#include "fftreg.cuh"

namespace qtam {

// radices per (log2 Nc, threads per CTA); every pass has Nc/R butterflies spread over NT threads
template <int LOG2NC, int NT> struct CtaFftRadix;
template <> struct CtaFftRadix<11, 128> { static constexpr int R0 = 16, R1 = 16, R2 = 8; };
template <> struct CtaFftRadix<11, 256> { static constexpr int R0 = 16, R1 = 16, R2 = 8; };
template <> struct CtaFftRadix<11, 512> { static constexpr int R0 = 16, R1 = 16, R2 = 8; };
template <> struct CtaFftRadix<11, 384> { static constexpr int R0 = 16, R1 = 16, R2 = 8; };
template <> struct CtaFftRadix<12, 384> { static constexpr int R0 = 16, R1 = 16, R2 = 16; };
template <> struct CtaFftRadix<13, 384> { static constexpr int R0 = 16, R1 = 16, R2 = 32; };
template <> struct CtaFftRadix<12, 256> { static constexpr int R0 = 16, R1 = 16, R2 = 16; };
template <> struct CtaFftRadix<12, 512> { static constexpr int R0 = 16, R1 = 16, R2 = 16; };
template <> struct CtaFftRadix<13, 256> { static constexpr int R0 = 32, R1 = 16, R2 = 16; };
template <> struct CtaFftRadix<13, 512> { static constexpr int R0 = 16, R1 = 16, R2 = 32; };
template <> struct CtaFftRadix<14, 512> { static constexpr int R0 = 32, R1 = 32, R2 = 16; };
// default thread count of the stand-alone long-FFT kernels
template <int LOG2NC> struct CtaFftPlan;
template <> struct CtaFftPlan<11> { static constexpr int NT = 128; };
template <> struct CtaFftPlan<12> { static constexpr int NT = 256; };
template <> struct CtaFftPlan<13> { static constexpr int NT = 256; };
template <> struct CtaFftPlan<14> { static constexpr int NT = 512; };

template <int V> struct ILog2 { static constexpr int value = 1 + ILog2<V / 2>::value; };
template <> struct ILog2<1> { static constexpr int value = 0; };

// shared-memory elements the transform needs (skew padding included)
template <int LOG2NC> __host__ __device__ constexpr int cta_fft_smem_elems() {
  return (1 << LOG2NC) + ((1 << LOG2NC) >> 4) + 2;   // the smallest first radix is 16
}

// sources / sinks of the transform's first / last pass (natural order index a)
struct CtaFftGlobalIn {
  const float2 *__restrict__ p;
  __device__ __forceinline__ float2 operator()(int a) const { return p[a]; }
};
struct CtaFftGlobalOut {
  float2 *__restrict__ p; float scale;
  __device__ __forceinline__ void operator()(int a, float2 v) const { p[a] = pscale(v, scale); }
};
struct CtaFftNone {
  __device__ __forceinline__ float2 operator()(int) const { return make_float2(0.f, 0.f); }
  __device__ __forceinline__ void operator()(int, float2) const {}
};

// One Stockham pass.  IN_MODE / OUT_MODE: 0 natural smem, 1 skewed smem, 2 the functor `in` / `out`.
template <int LOG2NC, int NT, int R, int LOG2NS, int DIR, int IN_MODE, int OUT_MODE, int SKEW, class In, class Out>
__device__ __forceinline__ void cta_fft_pass(float2 *s, const In &in, const Out &out,
                                             const float2 *__restrict__ ptw) {
  constexpr int NC = 1 << LOG2NC;
  constexpr int NBF = NC / R;                 // butterflies
  constexpr int BPT = (NBF + NT - 1) / NT;    // per thread
  constexpr int NS = 1 << LOG2NS;
  float2 v[BPT][R];
#pragma unroll
  for (int u = 0; u < BPT; ++u) {
    const int i = threadIdx.x + NT * u;
    if (NBF % NT == 0 || i < NBF) {
#pragma unroll
      for (int r = 0; r < R; ++r) {
        const int a = i + r * NBF;
        if constexpr (IN_MODE == 2) v[u][r] = in(a);
        else if constexpr (IN_MODE == 1) v[u][r] = s[a + (a >> SKEW)];
        else v[u][r] = s[a];
      }
      if constexpr (LOG2NS > 0) {
        const int k = i & (NS - 1);
        // r = 4a + b: w_{NS R}^{kr} = w^{4ka} w^{kb} from R/4 - 1 + 3 table values and one product each.
        // ptw: the pass's table [m][k] = e^{2 pi i k m/(NS R)}, m = 1, 2, 3, 4, 8, .. (coalesced over k)
        constexpr int RA = R / 4;
        float2 wb[4], wa[RA];
#pragma unroll
        for (int b = 1; b < 4; ++b) {
          wb[b] = __ldg(ptw + (b - 1) * NS + k);
          if (DIR < 0) wb[b].y = -wb[b].y;
        }
#pragma unroll
        for (int a = 1; a < RA; ++a) {
          wa[a] = __ldg(ptw + (2 + a) * NS + k);
          if (DIR < 0) wa[a].y = -wa[a].y;
        }
#pragma unroll
        for (int r = 1; r < R; ++r) {
          const int a = r >> 2, b = r & 3;
          const float2 w = a == 0 ? wb[b] : (b == 0 ? wa[a] : pcmul(wa[a], wb[b]));
          v[u][r] = pcmul(v[u][r], w);
        }
      }
      RegFFT<R, DIR>::run(v[u]);
    }
  }
  if constexpr (IN_MODE != 2 && OUT_MODE != 2) __syncthreads();   // all reads done before in-place writes
#pragma unroll
  for (int u = 0; u < BPT; ++u) {
    const int i = threadIdx.x + NT * u;
    if (NBF % NT == 0 || i < NBF) {
      const int k = i & (NS - 1);
      const int base = ((i - k) * R) + k;
#pragma unroll
      for (int r = 0; r < R; ++r) {
        const int a = base + r * NS;
        if constexpr (OUT_MODE == 2) out(a, v[u][r]);
        else if constexpr (OUT_MODE == 1) s[a + (a >> SKEW)] = v[u][r];
        else s[a] = v[u][r];
      }
    }
  }
  if constexpr (OUT_MODE != 2) __syncthreads();
}

// entries of the pass tables of one transform (passes 2 and 3), and the offset of pass 3's
template <int LOG2NC, int NT> __host__ __device__ constexpr int cta_fft_ptw_off3() {
  return (2 + CtaFftRadix<LOG2NC, NT>::R1 / 4) * CtaFftRadix<LOG2NC, NT>::R0;
}
template <int LOG2NC, int NT> __host__ __device__ constexpr int cta_fft_ptw_elems() {
  return cta_fft_ptw_off3<LOG2NC, NT>() +
         (2 + CtaFftRadix<LOG2NC, NT>::R2 / 4) * CtaFftRadix<LOG2NC, NT>::R0 * CtaFftRadix<LOG2NC, NT>::R1;
}

// host: the pass tables (interleaved re, im), long double evaluation with the index reduced mod the period
template <int LOG2NC, int NT> inline void fill_cta_fft_tables(std::vector<float> &out) {
  typedef CtaFftRadix<LOG2NC, NT> PL;
  out.clear();
  const long double tau = 6.283185307179586476925286766559005768L;
  auto pass = [&](int R, int NS) {
    const long long period = (long long)NS * R;
    for (int row = 0; row < 2 + R / 4; ++row) {
      const int m = row < 3 ? row + 1 : 4 * (row - 2);
      for (int k = 0; k < NS; ++k) {
        const long long e = ((long long)k * m) % period;
        const long double a = tau * (long double)e / (long double)period;
        out.push_back((float)cosl(a));
        out.push_back((float)sinl(a));
      }
    }
  };
  pass(PL::R1, PL::R0);
  pass(PL::R2, PL::R0 * PL::R1);
}

// Whole transform with NT threads (all threads of the CTA must call it).
// FROM_GLOBAL: pass 1 takes its inputs from in(a), a = natural-order index, instead of s (natural layout).
// TO_GLOBAL: the last pass hands its results to out(a, value) instead of writing s (natural layout).
// ptw: the pass tables built by fill_cta_fft_tables (host) for this (LOG2NC, NT)'s radices.
template <int LOG2NC, int NT, int DIR, bool FROM_GLOBAL, bool TO_GLOBAL, class In, class Out>
__device__ __forceinline__ void cta_fft_io(float2 *s, const In &in, const Out &out, const float2 *__restrict__ ptw) {
  typedef CtaFftRadix<LOG2NC, NT> PL;
  constexpr int L0 = ILog2<PL::R0>::value, L1 = ILog2<PL::R1>::value;
  static_assert(L0 + L1 + ILog2<PL::R2>::value == LOG2NC, "radices must multiply to Nc");
  cta_fft_pass<LOG2NC, NT, PL::R0, 0, DIR, FROM_GLOBAL ? 2 : 0, 1, L0>(s, in, out, ptw);
  cta_fft_pass<LOG2NC, NT, PL::R1, L0, DIR, 1, 0, L0>(s, in, out, ptw);
  cta_fft_pass<LOG2NC, NT, PL::R2, L0 + L1, DIR, 0, TO_GLOBAL ? 2 : 0, L0>(
      s, in, out, ptw + cta_fft_ptw_off3<LOG2NC, NT>());
}

// the same with plain global pointers: gin read in natural order, gout written in natural order x out_scale
template <int LOG2NC, int NT, int DIR, bool FROM_GLOBAL, bool TO_GLOBAL>
__device__ __forceinline__ void cta_fft(float2 *s, const float2 *__restrict__ gin, float2 *__restrict__ gout,
                                        const float2 *__restrict__ ptw, float out_scale) {
  cta_fft_io<LOG2NC, NT, DIR, FROM_GLOBAL, TO_GLOBAL>(s, CtaFftGlobalIn{gin}, CtaFftGlobalOut{gout, out_scale}, ptw);
}

}  // namespace qtam
