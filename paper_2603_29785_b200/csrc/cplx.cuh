// cplx.cuh -- tiny complex helpers on float2 / double2 for the libqtam kernels.
#pragma once
#include <cuda_runtime.h>

namespace qtam {

template <typename T> struct Vec2;
template <> struct Vec2<float> { typedef float2 type; };
template <> struct Vec2<double> { typedef double2 type; };
template <typename T> using C2 = typename Vec2<T>::type;

template <typename T> __host__ __device__ __forceinline__ C2<T> cmk(T x, T y) { C2<T> r; r.x = x; r.y = y; return r; }
template <typename V> __host__ __device__ __forceinline__ V cadd(V a, V b) { a.x += b.x; a.y += b.y; return a; }
template <typename V> __host__ __device__ __forceinline__ V csub(V a, V b) { a.x -= b.x; a.y -= b.y; return a; }
template <typename V> __host__ __device__ __forceinline__ V cmul(V a, V b) {
  V r; r.x = a.x * b.x - a.y * b.y; r.y = a.x * b.y + a.y * b.x; return r;
}
template <typename V> __host__ __device__ __forceinline__ V cconj(V a) { a.y = -a.y; return a; }
template <typename V, typename T> __host__ __device__ __forceinline__ V cscale(V a, T s) { a.x *= s; a.y *= s; return a; }
// multiply by +i (dir>0) or -i (dir<0)
template <typename V> __host__ __device__ __forceinline__ V cmul_i(V a, int dir) {
  V r;
  if (dir > 0) { r.x = -a.y; r.y = a.x; } else { r.x = a.y; r.y = -a.x; }
  return r;
}
// e^{dir * 2 pi i idx / twn} from the table tw[k] = e^{+2 pi i k / twn}
template <typename V> __device__ __forceinline__ V tw_get(const V *__restrict__ tw, long long idx, int dir) {
  V w = tw[idx];
  if (dir < 0) w.y = -w.y;
  return w;
}

}  // namespace qtam
