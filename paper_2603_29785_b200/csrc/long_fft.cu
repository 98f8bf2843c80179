// long_fft.cu -- batched complex FFTs of 2^15 .. 2^19 points (float): the half-length transform behind
// the long real FFTs a1 / a8 when the segment does not fit one CTA's shared memory (N = 2^16 .. 2^20,
// BASELINE config 4).  Two kernels, each reading and writing its data once:
//   A  k_long_a  n = j1 N2 + j2, N2 = 2^14, R = n/N2 = 2 .. 32: one thread per j2 takes the R points
//                z[j1 N2 + j2] (coalesced over j2), transforms them in registers and multiplies by
//                w_n^{dir j2 n1}; result A[n1][j2] to the workspace
//   B  k_long_b  one CTA per (n1, sequence): the 2^14-point transform over j2 in shared memory
//                (ctafft.cuh), written to Z[n1 + R n2] (stride R; the 32-byte sectors are completed in L2
//                by the CTAs of the neighbouring n1)
#include "ctafft.cuh"
#include "device_plan.hpp"

namespace qtam {

extern __shared__ __align__(16) unsigned char qtam_long_smem[];

constexpr int kLongLog2N2 = 14;

template <int LOG2R, int DIR>
__global__ void __launch_bounds__(256)
k_long_a(const float2 *in, long long in_stride, float2 *out, long long out_stride,
         const float2 *__restrict__ tw, int tw_shift) {   // in may equal out: a thread loads its R points, then stores to the same R addresses
  constexpr int R = 1 << LOG2R, N2 = 1 << kLongLog2N2;
  const int j2 = blockIdx.x * 256 + threadIdx.x;
  const float2 *src = in + (size_t)blockIdx.y * in_stride + j2;
  float2 v[R];
#pragma unroll
  for (int j1 = 0; j1 < R; ++j1) v[j1] = __ldcs(src + (size_t)j1 * N2);
  RegFFT<R, DIR>::run(v);
  // w^{n1}, w = e^{dir 2 pi i j2/n}: the powers of two from the table (tw[k] = e^{+2 pi i k/twn}),
  // every other one a product of at most LOG2R of them
  float2 pw[R];
  pw[0] = make_float2(1.f, 0.f);
#pragma unroll
  for (int b = 0; b < LOG2R; ++b) {
    float2 w = __ldg(tw + ((size_t)(j2 << b) << tw_shift));
    if (DIR < 0) w.y = -w.y;
    pw[1 << b] = w;
  }
#pragma unroll
  for (int k = 3; k < R; ++k)
    if (k & (k - 1)) pw[k] = pcmul(pw[k & (k - 1)], pw[k & -k]);
  float2 *dst = out + (size_t)blockIdx.y * out_stride + j2;
  dst[0] = v[0];
#pragma unroll
  for (int n1 = 1; n1 < R; ++n1) dst[(size_t)n1 * N2] = pcmul(v[n1], pw[n1]);
}

struct LongStridedOut {
  float2 *__restrict__ p; int log2R; float scale;
  __device__ __forceinline__ void operator()(int a, float2 v) const { p[(size_t)a << log2R] = pscale(v, scale); }
};

template <int DIR>
__global__ void __launch_bounds__(CtaFftPlan<kLongLog2N2>::NT)
k_long_b(const float2 *__restrict__ in, long long in_stride, float2 *__restrict__ out, long long out_stride,
         int log2R, const float2 *__restrict__ ptw, float scale) {
  constexpr int NT = CtaFftPlan<kLongLog2N2>::NT;
  float2 *s = reinterpret_cast<float2 *>(qtam_long_smem);
  const int n1 = blockIdx.x;
  const CtaFftGlobalIn gin{in + (size_t)blockIdx.y * in_stride + ((size_t)n1 << kLongLog2N2)};
  const LongStridedOut gout{out + (size_t)blockIdx.y * out_stride + n1, log2R, scale};
  cta_fft_io<kLongLog2N2, NT, DIR, true, true>(s, gin, gout, ptw);
}

template <int LOG2R>
static qtam_status long_launch(qtam_plan *p, const float2 *in, long long in_stride, float2 *out,
                               long long out_stride, float2 *tmp, long long tmp_stride, int count, int dir,
                               float scale, cudaStream_t st, double algo_in, double algo_out) {
  constexpr int NT = CtaFftPlan<kLongLog2N2>::NT;
  const int log2n = kLongLog2N2 + LOG2R;
  int log2twn = 0;
  while ((int64_t(1) << log2twn) < p->twn) ++log2twn;
  const int tw_shift = log2twn - log2n;
  if (tw_shift < 0) return QTAM_ERR_UNSUPPORTED;
  const double pass_bytes = 16.0 * (double)count * (double)(1LL << log2n);
  const float2 *tw = static_cast<const float2 *>(p->d_tw);
  const float2 *ptw = static_cast<const float2 *>(p->d_ptw_long);
  const size_t smem = sizeof(float2) * (size_t)cta_fft_smem_elems<kLongLog2N2>();
  dim3 ga((1 << kLongLog2N2) / 256, count), gb(1 << LOG2R, count);
  {
    LaunchScope ls(p, st, K_LONG_A, algo_in, pass_bytes);
    if (dir < 0) k_long_a<LOG2R, -1><<<ga, 256, 0, st>>>(in, in_stride, tmp, tmp_stride, tw, tw_shift);
    else k_long_a<LOG2R, +1><<<ga, 256, 0, st>>>(in, in_stride, tmp, tmp_stride, tw, tw_shift);
  }
  QTAM_LAUNCH_CHECK();
  {
    LaunchScope ls(p, st, K_LONG_B, algo_out, pass_bytes);
    if (dir < 0) k_long_b<-1><<<gb, NT, smem, st>>>(tmp, tmp_stride, out, out_stride, LOG2R, ptw, scale);
    else k_long_b<+1><<<gb, NT, smem, st>>>(tmp, tmp_stride, out, out_stride, LOG2R, ptw, scale);
  }
  QTAM_LAUNCH_CHECK();
  return QTAM_OK;
}

bool fast_cfft_long_ok(const qtam_plan *p, int log2n) {
  return p->d_ptw_long != nullptr && log2n > kLongLog2N2 && log2n <= kLongLog2N2 + 5;
}

qtam_status fast_cfft_long(qtam_plan *p, const void *in, long long in_stride, void *out, long long out_stride,
                           void *tmp, long long tmp_stride, int log2n, int count, int dir, float scale,
                           cudaStream_t st, double algo_in, double algo_out) {
  const float2 *i = static_cast<const float2 *>(in);
  float2 *o = static_cast<float2 *>(out), *t = static_cast<float2 *>(tmp);
  switch (log2n - kLongLog2N2) {
    case 1: return long_launch<1>(p, i, in_stride, o, out_stride, t, tmp_stride, count, dir, scale, st, algo_in, algo_out);
    case 2: return long_launch<2>(p, i, in_stride, o, out_stride, t, tmp_stride, count, dir, scale, st, algo_in, algo_out);
    case 3: return long_launch<3>(p, i, in_stride, o, out_stride, t, tmp_stride, count, dir, scale, st, algo_in, algo_out);
    case 4: return long_launch<4>(p, i, in_stride, o, out_stride, t, tmp_stride, count, dir, scale, st, algo_in, algo_out);
    case 5: return long_launch<5>(p, i, in_stride, o, out_stride, t, tmp_stride, count, dir, scale, st, algo_in, algo_out);
    default: return QTAM_ERR_UNSUPPORTED;
  }
}

qtam_status build_long_fft(qtam_plan *p) {
  int lnc = 0;
  while ((int64_t(1) << lnc) < p->sub_n) ++lnc;    // log2 of the power-of-two complex FFT behind the long transform
  if (p->esz != 4 || lnc <= kLongLog2N2 || lnc > kLongLog2N2 + 5) return QTAM_OK;
  std::vector<float> t;
  fill_cta_fft_tables<kLongLog2N2, CtaFftPlan<kLongLog2N2>::NT>(t);
  if (cudaMalloc(&p->d_ptw_long, t.size() * sizeof(float)) != cudaSuccess) return QTAM_ERR_ALLOC;
  p->device_bytes += t.size() * sizeof(float);
  if (cudaMemcpy(p->d_ptw_long, t.data(), t.size() * sizeof(float), cudaMemcpyHostToDevice) != cudaSuccess)
    return QTAM_ERR_CUDA;
  const size_t smem = sizeof(float2) * (size_t)cta_fft_smem_elems<kLongLog2N2>();
  if (cudaFuncSetAttribute(k_long_b<-1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess ||
      cudaFuncSetAttribute(k_long_b<+1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess)
    return QTAM_ERR_CUDA;
  return QTAM_OK;
}

}  // namespace qtam
