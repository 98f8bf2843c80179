// fftreg.cuh -- in-register complex FFTs of size 2..64 on float2 for sm_100a.
// Complex add/sub go through Blackwell's packed add.f32x2 / sub.f32x2 (SASS FADD2: one issue slot
// for both halves; a multiply by +-i folds into the FADD2 operand modifiers).  Twiddle constants
// are compile-time, so the multiplies become FMUL/FFMA with immediates.
#pragma once
#include <cuda_runtime.h>

namespace qtam {

typedef unsigned long long u64_t;

__device__ __forceinline__ float2 padd(float2 a, float2 b) {
  float2 r;
  asm("add.rn.f32x2 %0, %1, %2;" : "=l"(*reinterpret_cast<u64_t *>(&r))
      : "l"(*reinterpret_cast<u64_t *>(&a)), "l"(*reinterpret_cast<u64_t *>(&b)));
  return r;
}
__device__ __forceinline__ float2 psub(float2 a, float2 b) {
  float2 r;
  asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(*reinterpret_cast<u64_t *>(&r))
      : "l"(*reinterpret_cast<u64_t *>(&a)), "l"(*reinterpret_cast<u64_t *>(&b)));
  return r;
}
__device__ __forceinline__ float2 pmul(float2 a, float2 b) {
  float2 r;
  asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(*reinterpret_cast<u64_t *>(&r))
      : "l"(*reinterpret_cast<u64_t *>(&a)), "l"(*reinterpret_cast<u64_t *>(&b)));
  return r;
}
__device__ __forceinline__ float2 pfma(float2 a, float2 b, float2 c) {
  float2 r;
  asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(*reinterpret_cast<u64_t *>(&r))
      : "l"(*reinterpret_cast<u64_t *>(&a)), "l"(*reinterpret_cast<u64_t *>(&b)),
        "l"(*reinterpret_cast<u64_t *>(&c)));
  return r;
}
// a * w for a run-time twiddle w: (ax wx - ay wy, ax wy + ay wx) = a*(wx,wx) + (-ay,ax)*(wy,wy)
__device__ __forceinline__ float2 pcmul(float2 a, float2 w) {
  return pfma(a, make_float2(w.x, w.x), pmul(make_float2(-a.y, a.x), make_float2(w.y, w.y)));
}
// same with the twiddle stored pre-duplicated as (wx, wx, wy, wy): no pair-building moves
__device__ __forceinline__ float2 pcmul4(float2 a, float4 w) {
  return pfma(a, make_float2(w.x, w.y), pmul(make_float2(-a.y, a.x), make_float2(w.z, w.w)));
}
__device__ __forceinline__ float2 pscale(float2 a, float s) { return pmul(a, make_float2(s, s)); }

// cos / sin of 2 pi k/64, exact on the axes
__host__ __device__ constexpr float cos64(int k) {
  constexpr float c[17] = {1.0f, 9.951847267e-01f, 9.807852804e-01f, 9.569403357e-01f, 9.238795325e-01f,
                           8.819212643e-01f, 8.314696123e-01f, 7.730104534e-01f, 7.071067812e-01f,
                           6.343932842e-01f, 5.555702330e-01f, 4.713967368e-01f, 3.826834324e-01f,
                           2.902846773e-01f, 1.950903220e-01f, 9.801714033e-02f, 0.0f};
  k &= 63;
  return k <= 16 ? c[k] : k <= 32 ? -c[32 - k] : k <= 48 ? -c[k - 32] : c[64 - k];
}
__host__ __device__ constexpr float sin64(int k) { return cos64(k - 16); }

// o * e^{DIR 2 pi i Q/R} with compile-time Q, R (R | 64)
template <int Q, int R, int DIR>
__device__ __forceinline__ float2 twmul(float2 o) {
  constexpr int k = (Q * (64 / R)) & 63;
  if constexpr (k == 0) return o;
  else if constexpr (k == 16) return DIR > 0 ? make_float2(-o.y, o.x) : make_float2(o.y, -o.x);
  else if constexpr (k == 32) return make_float2(-o.x, -o.y);
  else if constexpr (k == 48) return DIR > 0 ? make_float2(o.y, -o.x) : make_float2(-o.y, o.x);
  else {
    // o (c + i s) = o (c, c) + (-o.y, o.x) (s, s): two packed instructions -- the swap and the sign of the
    // second factor fold into FMUL2's operand modifiers, (c, c) and (s, s) are scalar-broadcast operands
    constexpr float c = cos64(k);
    constexpr float s = DIR > 0 ? sin64(k) : -sin64(k);
    return pfma(o, make_float2(c, c), pmul(make_float2(-o.y, o.x), make_float2(s, s)));
  }
}

// In-register FFT of size R (power of two <= 64), natural order in and out, on v[0..R).
// out[n] = sum_j v[j] e^{DIR 2 pi i jn/R}.  Recursive decimation in time; everything unrolls.
template <int R, int DIR> struct RegFFT {
  template <int Q> static __device__ __forceinline__ void combine(float2 (&v)[R], const float2 (&e)[R / 2],
                                                                 const float2 (&o)[R / 2]) {
    if constexpr (Q < R / 2) {
      const float2 t = twmul<Q, R, DIR>(o[Q]);
      v[Q] = padd(e[Q], t);
      v[Q + R / 2] = psub(e[Q], t);
      combine<Q + 1>(v, e, o);
    }
  }
  static __device__ __forceinline__ void run(float2 (&v)[R]) {
    float2 e[R / 2], o[R / 2];
#pragma unroll
    for (int q = 0; q < R / 2; ++q) { e[q] = v[2 * q]; o[q] = v[2 * q + 1]; }
    RegFFT<R / 2, DIR>::run(e);
    RegFFT<R / 2, DIR>::run(o);
    combine<0>(v, e, o);
  }
};
template <int DIR> struct RegFFT<1, DIR> {
  static __device__ __forceinline__ void run(float2 (&)[1]) {}
};

}  // namespace qtam
