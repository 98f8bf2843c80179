// clfft.cuh -- one complex FFT of M = F * P points spread over a thread-block cluster (float), for the rows of
// 2^13 .. 2^17 points of rows_cluster.cu.
//
// Cooley-Tukey with the cluster split in the MIDDLE, so that each side of the transform touches global memory
// in whole 32-byte sectors and only one all-to-all goes through distributed shared memory:
//   M = F * P,  F = 4 * CL (CL = CTAs per cluster, F <= 32),  P = 2^LOG2P points per sub-transform.
//   index on the "band" side   j = q + F * jc,   q = ja + 4 * jb  (ja = 0..3, jb = the CTA's rank, jc < P)
//   index on the "time" side   n = nc + P * m,   m < F, nc < P
//   DIR = +1 (forward rows, C47):  Z[q][nc] = sum_jc B[q + F jc] w_P^{+jc nc}          (P-point sub-FFTs, local)
//                                  Y[nc + P m] = sum_q w_M^{+q nc} Z[q][nc] w_F^{+q m}  (radix F across the cluster)
//   DIR = -1 (inverse rows, C49):  u[q][nc] = w_M^{-q nc} sum_m Y[nc + P m] w_F^{-q m}  (radix F, then scattered)
//                                  Bhat[q + F jc] = sum_nc u[q][nc] w_P^{-jc nc}        (P-point sub-FFTs, local)
// CTA jb owns the four sub-transforms q = 4 jb .. 4 jb + 3: on the band side four CONSECUTIVE bins (one sector)
// every F bins.  They sit interleaved in its shared memory, element (ja, p) at 4 * phys(p) + ja, and run as one
// batched Stockham transform (radix 16, 16, P/256) in which thread t works on sub-transform ja = t & 3: a warp
// reads 8 sectors of the band, and every shared-memory access is a contiguous 256-byte run.  The radix-F stage
// takes its F inputs for one nc from the F/4 CTAs (32 contiguous bytes each) and owns P/CL consecutive nc, so
// the time side is CL... F contiguous runs of P/CL points.
#pragma once
#include <vector>

#include "fftreg.cuh"

namespace qtam {

template <int LOG2P> struct ClFft {
  static constexpr int P = 1 << LOG2P;
  static constexpr int NT = P / 8;               // threads per CTA: every pass holds 64 values per thread
  static constexpr int R0 = 16, R1 = 16, R2 = P / 256;
  static constexpr int SMEM_ELEMS = 4 * (P + P / 16);      // pass 1 writes a skewed layout phys(a) = a + (a >> 4)
  static constexpr int PTW_OFF2 = (2 + R1 / 4) * R0;       // entries of pass 2's table before pass 3's
  static constexpr int PTW_ELEMS = PTW_OFF2 + (2 + R2 / 4) * R0 * R1;
};

// host: pass tables of the batched sub-transforms, [m][k] = e^{2 pi i k m / (NS R)}, m = 1, 2, 3, 4, 8, ..
// (long double, index reduced mod the period; same layout as ctafft.cuh)
template <int LOG2P> inline void fill_clfft_tables(std::vector<float> &out) {
  typedef ClFft<LOG2P> PL;
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

// host: the radix-F stage's twiddles, rows m = 1 and m = 4 of e^{2 pi i m nc / M}, nc < P
inline void fill_clfft_final(std::vector<float> &out, int P, long long M) {
  out.clear();
  const long double tau = 6.283185307179586476925286766559005768L;
  for (int m = 1; m <= 4; m += 3)
    for (int nc = 0; nc < P; ++nc) {
      const long double a = tau * (long double)(((long long)nc * m) % M) / (long double)M;
      out.push_back((float)cosl(a));
      out.push_back((float)sinl(a));
    }
}

struct ClNoMid { __device__ __forceinline__ void operator()() const {} };
struct ClSyncMid { __device__ __forceinline__ void operator()() const { __syncthreads(); } };

// One pass of the four interleaved sub-transforms.  IN_MODE: 0 natural layout, 1 skewed layout, 2 the functor
// in(ja, a) (a = natural index of the sub-transform's input).  The results go to shared memory (natural or
// skewed); mid() runs between the last read and the first write (a barrier when the pass works in place).
template <int LOG2P, int R, int LOG2NS, int DIR, int IN_MODE, bool OUT_SKEW, class In, class Mid>
__device__ __forceinline__ void cl_pass(float2 *s, const In &in, const Mid &mid, const float2 *ptw) {
  typedef ClFft<LOG2P> PL;
  constexpr int NBF = PL::P / R;            // butterflies per sub-transform
  constexpr int TPS = PL::NT / 4;           // threads per sub-transform
  constexpr int BPT = NBF / TPS;
  constexpr int NS = 1 << LOG2NS;
  static_assert(NBF % TPS == 0 && BPT >= 1, "butterflies must divide among the threads");
  const int ja = threadIdx.x & 3, ib = threadIdx.x >> 2;
  float2 v[BPT][R];
#pragma unroll
  for (int u = 0; u < BPT; ++u) {
    const int i = ib + TPS * u;
#pragma unroll
    for (int r = 0; r < R; ++r) {
      const int a = i + r * NBF;
      if constexpr (IN_MODE == 2) v[u][r] = in(ja, a);
      else if constexpr (IN_MODE == 1) v[u][r] = s[4 * (a + (a >> 4)) + ja];
      else v[u][r] = s[4 * a + ja];
    }
    if constexpr (LOG2NS > 0) {
      // r = 4a + b: w^{kr} = w^{4ka} w^{kb} from R/4 - 1 + 3 table values and one product each
      const int k = i & (NS - 1);
      constexpr int RA = R / 4;
      float2 wb[4], wa[RA];
#pragma unroll
      for (int b = 1; b < 4; ++b) {
        wb[b] = ptw[(b - 1) * NS + k];
        if (DIR < 0) wb[b].y = -wb[b].y;
      }
#pragma unroll
      for (int a = 1; a < RA; ++a) {
        wa[a] = ptw[(2 + a) * NS + k];
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
  mid();
#pragma unroll
  for (int u = 0; u < BPT; ++u) {
    const int i = ib + TPS * u;
    const int k = i & (NS - 1);
    const int base = ((i - k) * R) + k;
#pragma unroll
    for (int r = 0; r < R; ++r) {
      const int a = base + r * NS;
      s[4 * (OUT_SKEW ? a + (a >> 4) : a) + ja] = v[u][r];
    }
  }
}

// passes 2 and 3 of the batched sub-transforms (pass 1 is written out by the caller: its input or the barrier
// before its writes differs between the forward and the inverse); natural layout on exit, ends with a barrier
template <int LOG2P, int DIR>
__device__ __forceinline__ void cl_passes_23(float2 *s, const float2 *ptw) {
  typedef ClFft<LOG2P> PL;
  cl_pass<LOG2P, PL::R1, 4, DIR, 1, false>(s, ClNoMid{}, ClSyncMid{}, ptw);
  __syncthreads();
  cl_pass<LOG2P, PL::R2, 8, DIR, 0, false>(s, ClNoMid{}, ClSyncMid{}, ptw + PL::PTW_OFF2);
  __syncthreads();
}

// the F twiddles w^q, q = 4a + b, of one nc, applied in place: w1 = w_M^{dir nc}, w4 = w_M^{dir 4 nc}
template <int F> __device__ __forceinline__ void cl_twiddle(float2 (&v)[F], float2 w1, float2 w4) {
  const float2 w2 = pcmul(w1, w1), w3 = pcmul(w2, w1);
  v[1] = pcmul(v[1], w1); v[2] = pcmul(v[2], w2); v[3] = pcmul(v[3], w3);
  float2 wa = w4;
#pragma unroll
  for (int a = 1; a < F / 4; ++a) {
    if (a > 1) wa = pcmul(wa, w4);
    v[4 * a] = pcmul(v[4 * a], wa);
    v[4 * a + 1] = pcmul(v[4 * a + 1], pcmul(wa, w1));
    v[4 * a + 2] = pcmul(v[4 * a + 2], pcmul(wa, w2));
    v[4 * a + 3] = pcmul(v[4 * a + 3], pcmul(wa, w3));
  }
}

}  // namespace qtam
