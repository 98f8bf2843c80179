// thrbits.cuh -- the row-median threshold's arithmetic: every operation
// correctly rounded in T, no fused multiply-add, magnitudes compared through their bit patterns.
#pragma once
#include <cuda_runtime.h>

namespace qtam {

template <typename T> struct Bits;
template <> struct Bits<float> {
  typedef unsigned int U; static const int nbits = 32;
  static __device__ __forceinline__ U of(float v) { return __float_as_uint(v); }
  static __device__ __forceinline__ float from(U u) { return __uint_as_float(u); }
  static __device__ __forceinline__ float mag(float re, float im) {
    return __fsqrt_rn(__fadd_rn(__fmul_rn(re, re), __fmul_rn(im, im)));
  }
  static __device__ __forceinline__ float root(float a) { return __fsqrt_rn(a); }
  static __device__ __forceinline__ U inf_bits() { return 0x7f800000u; }
  static __device__ __forceinline__ float mul(float a, float b) { return __fmul_rn(a, b); }
  static __device__ __forceinline__ float add(float a, float b) { return __fadd_rn(a, b); }
};
template <> struct Bits<double> {
  typedef unsigned long long U; static const int nbits = 64;
  static __device__ __forceinline__ U of(double v) { return (U)__double_as_longlong(v); }
  static __device__ __forceinline__ double from(U u) { return __longlong_as_double((long long)u); }
  static __device__ __forceinline__ double mag(double re, double im) {
    return __dsqrt_rn(__dadd_rn(__dmul_rn(re, re), __dmul_rn(im, im)));
  }
  static __device__ __forceinline__ double root(double a) { return __dsqrt_rn(a); }
  static __device__ __forceinline__ U inf_bits() { return 0x7ff0000000000000ull; }
  static __device__ __forceinline__ double mul(double a, double b) { return __dmul_rn(a, b); }
  static __device__ __forceinline__ double add(double a, double b) { return __dadd_rn(a, b); }
};

}  // namespace qtam
