// rowfft.cuh -- warp-level row FFT engine: one row of M = 32*G points per group of G lanes
// (G = 1..32, so 32/G rows per warp), 32 points per thread in registers, two passes:
//   pass 1  in-thread radix-32 over j1 (inputs B[t + G*j1]), twiddle w_M^{dir t n1} (x scale) from a
//           shared-memory table laid out [n1][t] (conflict free)
//   exchange through the warp's private shared-memory buffer EX[row][j2][n1] with a 33-element
//           pitch (conflict-free 64-bit stores and loads; no block barrier, only __syncwarp)
//   pass 2  32/G in-thread FFTs of size G over j2; thread t ends with Y[(t + G*i) + 32*n2] in
//           v[i*G + n2], so that for a fixed register the G lanes of a row hold G consecutive outputs
#pragma once
#include "fftreg.cuh"

namespace qtam {

constexpr int kExPitch = 33;
constexpr int kExPerWarp = 32 * kExPitch;   // float2 elements of exchange buffer per warp

template <int LOG2G, int DIR> struct RowFFT {
  static constexpr int G = 1 << LOG2G;
  static constexpr int F = 32 / G;
  static constexpr int M = 32 * G;

  static __device__ __forceinline__ float2 twmulx(float2 a, float2 w) {
    return pcmul(a, w);      // FMUL2 + FFMA2 (swap/negate and the broadcasts are operand modifiers)
  }
  static __device__ __forceinline__ float scale_of(float2 w) { return w.x; }

  // tw1: [n1][t] entries (wx, wy) of w_M^{dir t n1} x scale, in shared or global memory (64-bit loads:
  // half the shared-memory wavefronts of a pre-duplicated (wx, wx, wy, wy) table, measured faster)
  template <typename TW>
  static __device__ __forceinline__ void run(float2 (&v)[32], float2 *ex, const TW *tw1, int lane) {
    const int t = lane & (G - 1), rw = lane >> LOG2G;
    RegFFT<32, DIR>::run(v);
    if constexpr (G > 1) {
      float2 *exw = ex + rw * (G * kExPitch) + t * kExPitch;
      // twiddles in batches of 8, one batch ahead of the multiplies: the shared-memory latency is paid
      // four times per row instead of once per element
      TW w[2][8];
#pragma unroll
      for (int k = 0; k < 8; ++k) w[0][k] = tw1[k * G + t];
#pragma unroll
      for (int c = 0; c < 4; ++c) {
        if (c < 3) {
#pragma unroll
          for (int k = 0; k < 8; ++k) w[(c + 1) & 1][k] = tw1[(8 * (c + 1) + k) * G + t];
        }
#pragma unroll
        for (int k = 0; k < 8; ++k) exw[8 * c + k] = twmulx(v[8 * c + k], w[c & 1][k]);
      }
      __syncwarp();
      const float2 *exr = ex + rw * (G * kExPitch) + t;
#pragma unroll
      for (int i = 0; i < F; ++i) {
        float2 u[G];
#pragma unroll
        for (int j2 = 0; j2 < G; ++j2) u[j2] = exr[j2 * kExPitch + G * i];
        RegFFT<G, DIR>::run(u);
#pragma unroll
        for (int n2 = 0; n2 < G; ++n2) v[i * G + n2] = u[n2];
      }
      __syncwarp();
    } else {
      // M = 32: one thread per row, only the scale remains
#pragma unroll
      for (int n1 = 0; n1 < 32; ++n1) v[n1] = pscale(v[n1], scale_of(tw1[0]));
    }
  }
};

}  // namespace qtam
