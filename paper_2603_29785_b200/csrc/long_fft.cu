// long_fft.cu -- batched complex FFTs of 2^14 .. 2^19 points (float): the half-length transform behind
// the long real FFTs a1 / a8 when the segment does not fit one CTA's shared memory (N = 2^16 .. 2^20,
// BASELINE config 4).  Two kernels, each reading and writing its data once:
//   A  k_long_a  n = j1 N2 + j2, N2 = 2^13, R = n/N2 = 2 .. 64: one thread per j2 takes the R points
//                z[j1 N2 + j2] (coalesced over j2), transforms them in registers and multiplies by
//                w_n^{dir j2 n1}; result A[n1][j2] to the workspace
//   B  k_long_b  one CTA per (n1, sequence), three CTAs per SM: the 2^13-point transform over j2 in shared
//                memory (ctafft.cuh), written to Z[n1 + R n2] (stride R; the 32-byte sectors are completed in L2
//                by the CTAs of the neighbouring n1).  (2^14-point transforms, one 512-thread CTA per SM, with
//                R <= 32: 241 us per cfg4 step for the two directions instead of 220.)
#include "ctafft.cuh"
#include "device_plan.hpp"

namespace qtam {

extern __shared__ __align__(16) unsigned char qtam_long_smem[];

constexpr int kLongLog2N2 = 13;

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

// --------------------------------------------------------------------------------------------------
// The long transform with the spectrum in RESIDUE ORDER (N = 2^20: n = 2^19 = 64 * 2^13), for plans whose long rows
// read the spectrum sorted by residue mod 64 anyway (rows_split.cu: bin f at [f mod 64][f div 64]).  With
// f = f1 + 64 f2 and n = 2^13 n1 + n2 the two passes are contiguous on both sides:
//   forward  k_long_a (radix 64 over n1, twiddle)  ->  k_long_b_res: Z[f1 + 64 f2] = FFT over n2, written to
//            row f1 of the residue-sorted buffer  ->  k_post_residues: the real post-processing in that buffer, in
//            place, and the spectrum in bin order for the other row kernels through shared-memory tiles
//   inverse  k_combine_runs writes the pre-processed spectrum in residue order  ->  k_long_b_res (FFT over f2 for
//            every f1)  ->  k_long_a_pre (twiddle, radix 64 over f1) straight to x_out
// instead of a second pass whose output has stride 64 (8 bytes every 512).
// --------------------------------------------------------------------------------------------------
template <int DIR>
__global__ void __launch_bounds__(CtaFftPlan<kLongLog2N2>::NT)
k_long_b_res(const float2 *__restrict__ in, long long in_seg, long long in_row, float2 *__restrict__ out,
             long long out_seg, long long out_row, const float2 *__restrict__ ptw) {
  constexpr int NT = CtaFftPlan<kLongLog2N2>::NT;
  float2 *s = reinterpret_cast<float2 *>(qtam_long_smem);
  cta_fft<kLongLog2N2, NT, DIR, true, true>(s, in + (size_t)blockIdx.y * in_seg + (size_t)blockIdx.x * in_row,
                                            out + (size_t)blockIdx.y * out_seg + (size_t)blockIdx.x * out_row, ptw, 1.f);
}

// x[N2 n1 + n2] = sum_f1 w_R^{dir f1 n1} (w_n^{dir f1 n2} A[f1][n2]): the twiddle BEFORE the radix-R transform
template <int LOG2R, int DIR>
__global__ void __launch_bounds__(256)
k_long_a_pre(const float2 *__restrict__ in, long long in_stride, float2 *__restrict__ out, long long out_stride,
             const float2 *__restrict__ tw, int tw_shift) {
  constexpr int R = 1 << LOG2R, N2 = 1 << kLongLog2N2;
  const int j2 = blockIdx.x * 256 + threadIdx.x;
  const float2 *src = in + (size_t)blockIdx.y * in_stride + j2;
  float2 v[R];
#pragma unroll
  for (int j1 = 0; j1 < R; ++j1) v[j1] = __ldcs(src + (size_t)j1 * N2);
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
#pragma unroll
  for (int k = 1; k < R; ++k) v[k] = pcmul(v[k], pw[k]);
  RegFFT<R, DIR>::run(v);
  float2 *dst = out + (size_t)blockIdx.y * out_stride + j2;
#pragma unroll
  for (int n1 = 0; n1 < R; ++n1) __stcs(dst + (size_t)n1 * N2, v[n1]);
}

// Real post-processing (k_r2c_post, row a1) on the residue-sorted half-length transform, in place, plus the spectrum
// in bin order.  A CTA takes the 4096 bins f = 4096 t .. (64 of every residue) and their mirrors g = Nc - f (bins
// G0 + 1 .. G0 + 4096, G0 = Nc - 4096 t - 4096): both tiles are read in runs of 64 elements per residue, paired in
// shared memory (static: two tiles), and written back to the same places and, in bin order, to `spec`.  rt: [64][rt_len] per segment,
// bin f at [f mod 64][pad + f div 64].
template <int TI>                                 // TI elements of every residue per tile: 64 TI bins
__global__ void __launch_bounds__(256)
k_post_residues(float2 *__restrict__ rt, long long rt_stride, int rt_len, int pad, float2 *__restrict__ spec,
                long long xstride, int Nc, const float2 *__restrict__ twN) {
  constexpr int TB = 64 * TI;                        // bins per tile
  __shared__ float2 tf[TI][65];                      // [f2 - TI t][residue]
  __shared__ float2 tg[TI + 1][65];                  // [u div 64][u mod 64], u = g - G0 = 1 .. TB
  const int seg = blockIdx.y, t = blockIdx.x, f0 = TB * t, G0 = Nc - f0 - TB;
  float2 *R = rt + (size_t)seg * rt_stride + pad;
  float2 *S = spec + (size_t)seg * xstride;
  if (f0 == Nc / 2) {
    // the middle bin alone (its own mirror); the rest of this block of bins belongs to the last tile's mirror
    if (threadIdx.x == 0) {
      const float2 A = R[f0 >> 6];                       // residue 0
      float2 w = __ldg(twN + f0); w.y = -w.y;
      const float2 D = make_float2(0.f, A.y);            // B = A: E = (Ax, 0), D = (0, Ay)
      const float2 tt = make_float2(w.x * D.x - w.y * D.y, w.x * D.y + w.y * D.x);
      const float2 xf = make_float2(A.x + tt.y, -tt.x);
      R[f0 >> 6] = xf; S[f0] = xf;
    }
    return;
  }
  for (int i = threadIdx.x; i < TB; i += 256) {
    const int res = i / TI, di = i - res * TI;
    tf[di][res] = R[(size_t)res * rt_len + (f0 >> 6) + di];
  }
  for (int i = threadIdx.x; i < (TI + 1) * 64; i += 256) {
    const int res = i / (TI + 1), di = i - res * (TI + 1);
    const int u = 64 * di + res;
    // (bin Nc itself -- u = TB of the first tile -- is not part of the half-length transform)
    if (u >= 1 && u <= TB && G0 + u < Nc) tg[di][res] = R[(size_t)res * rt_len + (G0 >> 6) + di];
  }
  __syncthreads();
  for (int j = threadIdx.x; j < TB; j += 256) {
    const int f = f0 + j, u = TB - j;                    // g = Nc - f = G0 + u
    const float2 A = tf[j >> 6][j & 63];
    const float2 B = (f == 0) ? A : tg[u >> 6][u & 63];
    const float2 E = make_float2(0.5f * (A.x + B.x), 0.5f * (A.y - B.y));
    const float2 D = make_float2(0.5f * (A.x - B.x), 0.5f * (A.y + B.y));
    float2 w = __ldg(twN + f); w.y = -w.y;               // e^{-2 pi i f/N}
    const float2 tt = make_float2(w.x * D.x - w.y * D.y, w.x * D.y + w.y * D.x);
    const float2 xf = make_float2(E.x + tt.y, E.y - tt.x), xg = make_float2(E.x - tt.y, -E.y - tt.x);
    tf[j >> 6][j & 63] = xf; tg[u >> 6][u & 63] = xg;
    S[f] = xf; S[Nc - f] = xg;
  }
  __syncthreads();
  for (int i = threadIdx.x; i < TB; i += 256) {
    const int res = i / TI, di = i - res * TI;
    R[(size_t)res * rt_len + (f0 >> 6) + di] = tf[di][res];
  }
  for (int i = threadIdx.x; i < (TI + 1) * 64; i += 256) {
    const int res = i / (TI + 1), di = i - res * (TI + 1);
    const int u = 64 * di + res;
    if (u >= 1 && u <= TB) R[(size_t)res * rt_len + (G0 >> 6) + di] = tg[di][res];
  }
}

constexpr int kPostTI = 16;

bool long_residues_ok(const qtam_plan *p) {
  return p->esz == 4 && p->n_pow2 && p->d_sp_xt != nullptr && p->d_ptw_long != nullptr &&
         p->hp.N == (int64_t(1) << (kLongLog2N2 + 7));     // n = N/2 = 64 * 2^13
}

static int long_tw_shift(const qtam_plan *p, int log2n) {
  int log2twn = 0;
  while ((int64_t(1) << log2twn) < p->twn) ++log2twn;
  return log2twn - log2n;
}

// forward: x -> the residue-sorted spectrum (p->d_sp_xt) and the spectrum in bin order (p->d_spec)
qtam_status long_forward_residues(qtam_plan *p, const void *d_x, int batch, cudaStream_t st) {
  constexpr int NT = CtaFftPlan<kLongLog2N2>::NT, LOG2R = 6;
  const int Nc = (int)(p->hp.N / 2);
  const int tw_shift = long_tw_shift(p, kLongLog2N2 + LOG2R);
  if (tw_shift < 0) return QTAM_ERR_UNSUPPORTED;
  const float2 *tw = static_cast<const float2 *>(p->d_tw);
  const float2 *ptw = static_cast<const float2 *>(p->d_ptw_long);
  float2 *ws = static_cast<float2 *>(p->d_ws), *rt = static_cast<float2 *>(p->d_sp_xt);
  const long long rt_stride = 64LL * p->sp_xt_len;
  const size_t smem = sizeof(float2) * (size_t)cta_fft_smem_elems<kLongLog2N2>();
  const double pass_bytes = 16.0 * (double)batch * (double)Nc;
  dim3 ga((1 << kLongLog2N2) / 256, batch), gb(1 << LOG2R, batch);
  {
    LaunchScope ls(p, st, K_LONG_A, (double)batch * 4.0 * (double)p->hp.N, pass_bytes);
    k_long_a<LOG2R, -1><<<ga, 256, 0, st>>>(static_cast<const float2 *>(d_x), Nc, ws, p->hp.N, tw, tw_shift);
  }
  QTAM_LAUNCH_CHECK();
  {
    LaunchScope ls(p, st, K_LONG_B, 0.0, pass_bytes);
    k_long_b_res<-1><<<gb, NT, smem, st>>>(ws, p->hp.N, 1 << kLongLog2N2, rt + p->sp_xt_pad, rt_stride, p->sp_xt_len, ptw);
  }
  QTAM_LAUNCH_CHECK();
  {
    dim3 gp((unsigned)(Nc / 2 / (64 * kPostTI) + 1), batch);
    LaunchScope ls(p, st, K_R2C_POST, 0.0, 3.0 * 8.0 * (double)batch * (double)Nc);
    k_post_residues<kPostTI><<<gp, 256, 0, st>>>(rt, rt_stride, p->sp_xt_len, p->sp_xt_pad, static_cast<float2 *>(p->d_spec),
                                            p->xstride, Nc, static_cast<const float2 *>(p->d_twN));
  }
  QTAM_LAUNCH_CHECK();
  return QTAM_OK;
}

// inverse: the pre-processed spectrum in residue order (p->d_sp_xt, written by k_combine_runs) -> x_out
qtam_status long_inverse_residues(qtam_plan *p, void *d_x_out, int batch, cudaStream_t st) {
  constexpr int NT = CtaFftPlan<kLongLog2N2>::NT, LOG2R = 6;
  const int Nc = (int)(p->hp.N / 2);
  const int tw_shift = long_tw_shift(p, kLongLog2N2 + LOG2R);
  if (tw_shift < 0) return QTAM_ERR_UNSUPPORTED;
  const float2 *tw = static_cast<const float2 *>(p->d_tw);
  const float2 *ptw = static_cast<const float2 *>(p->d_ptw_long);
  float2 *ws = static_cast<float2 *>(p->d_ws), *rt = static_cast<float2 *>(p->d_sp_xt);
  const long long rt_stride = 64LL * p->sp_xt_len;
  const size_t smem = sizeof(float2) * (size_t)cta_fft_smem_elems<kLongLog2N2>();
  const double pass_bytes = 16.0 * (double)batch * (double)Nc;
  dim3 ga((1 << kLongLog2N2) / 256, batch), gb(1 << LOG2R, batch);
  {
    LaunchScope ls(p, st, K_LONG_B, 0.0, pass_bytes);
    k_long_b_res<+1><<<gb, NT, smem, st>>>(rt + p->sp_xt_pad, rt_stride, p->sp_xt_len, ws, p->hp.N, 1 << kLongLog2N2, ptw);
  }
  QTAM_LAUNCH_CHECK();
  {
    LaunchScope ls(p, st, K_LONG_A, (double)batch * 4.0 * (double)p->hp.N, pass_bytes);
    k_long_a_pre<LOG2R, +1><<<ga, 256, 0, st>>>(ws, p->hp.N, static_cast<float2 *>(d_x_out), Nc, tw, tw_shift);
  }
  QTAM_LAUNCH_CHECK();
  return QTAM_OK;
}

// Batched complex FFTs of 2^11 .. 2^14 points, one CTA per sequence in shared memory (ctafft.cuh): the power-of-two
// transforms inside the radix-3 step of the segment lengths N = 3 * 2^k (the paper's 6 s at 4096 Hz = 3 * 2^13).
template <int LOG2N, int DIR>
__global__ void __launch_bounds__(CtaFftPlan<LOG2N>::NT)
k_cfft_cta(const float2 *__restrict__ in, long long in_stride, float2 *__restrict__ out, long long out_stride,
           const float2 *__restrict__ ptw, float scale) {
  float2 *s = reinterpret_cast<float2 *>(qtam_long_smem);
  cta_fft<LOG2N, CtaFftPlan<LOG2N>::NT, DIR, true, true>(s, in + (size_t)blockIdx.x * in_stride,
                                                         out + (size_t)blockIdx.x * out_stride, ptw, scale);
}

template <int LOG2N> static bool mid_prepare(qtam_plan *p) {
  std::vector<float> t;
  fill_cta_fft_tables<LOG2N, CtaFftPlan<LOG2N>::NT>(t);
  if (cudaMalloc(&p->d_ptw_mid, t.size() * sizeof(float)) != cudaSuccess) return false;
  p->device_bytes += t.size() * sizeof(float);
  if (cudaMemcpy(p->d_ptw_mid, t.data(), t.size() * sizeof(float), cudaMemcpyHostToDevice) != cudaSuccess) return false;
  const size_t smem = sizeof(float2) * (size_t)cta_fft_smem_elems<LOG2N>();
  return kernel_prepare(p->cfg_cfft_mid[0], k_cfft_cta<LOG2N, -1>, CtaFftPlan<LOG2N>::NT, smem) &&
         kernel_prepare(p->cfg_cfft_mid[1], k_cfft_cta<LOG2N, +1>, CtaFftPlan<LOG2N>::NT, smem);
}

template <int LOG2N>
static qtam_status mid_launch(qtam_plan *p, const float2 *in, long long in_stride, float2 *out, long long out_stride,
                              int count, int dir, float scale, cudaStream_t st, double algo) {
  const KernelCfg &cfg = p->cfg_cfft_mid[dir < 0 ? 0 : 1];
  if (!cfg.ready) return QTAM_ERR_CUDA;
  const float2 *ptw = static_cast<const float2 *>(p->d_ptw_mid);
  {
    LaunchScope ls(p, st, K_CFFT_SEQ, algo, 16.0 * (double)count * (double)(1 << LOG2N));
    if (dir < 0) k_cfft_cta<LOG2N, -1><<<(unsigned)count, CtaFftPlan<LOG2N>::NT, cfg.smem, st>>>(in, in_stride, out, out_stride, ptw, scale);
    else k_cfft_cta<LOG2N, +1><<<(unsigned)count, CtaFftPlan<LOG2N>::NT, cfg.smem, st>>>(in, in_stride, out, out_stride, ptw, scale);
  }
  QTAM_LAUNCH_CHECK();
  return QTAM_OK;
}

// The whole long real FFT / inverse FFT of a segment of N = 3 * 2^k samples in ONE CTA (n = N/2 = 3 Np complex
// points, Np = 2^11 .. 2^13): the three decimated sequences z[3 a + r] are gathered straight from global memory into
// three shared-memory transforms F_r = DFT_Np; the radix-3 butterfly Z[f] = sum_r w_n^{dir r f} F_r[f mod Np] and the
// real post-processing of row a1 (k_r2c_post) / the store of row a8 read them from shared memory.  One pass over
// the data instead of four (split, transforms, butterfly, post-processing).
struct Strided3In {
  const float2 *__restrict__ p;
  __device__ __forceinline__ float2 operator()(int a) const { return p[3 * a]; }
};
template <int LOG2NP> constexpr int r3_smem_elems() { return 3 * cta_fft_smem_elems<LOG2NP>(); }

template <int LOG2NP, int DIR>
__device__ __forceinline__ float2 r3_point(const float2 *s0, const float2 *s1, const float2 *s2, int f,
                                           const float2 *__restrict__ twN) {
  // Z[f] = F0[k] + w F1[k] + w^2 F2[k], k = f mod Np, w = e^{DIR 2 pi i f/n} = twN[2 f] (twN[j] = e^{2 pi i j/N})
  constexpr int NP = 1 << LOG2NP, N = 6 * NP;
  const int k = f & (NP - 1);
  float2 w1 = __ldg(twN + (2 * f) % N), w2 = __ldg(twN + (4 * f) % N);
  if (DIR < 0) { w1.y = -w1.y; w2.y = -w2.y; }
  return padd(s0[k], padd(pcmul(s1[k], w1), pcmul(s2[k], w2)));
}

template <int LOG2NP>
__global__ void __launch_bounds__(CtaFftPlan<LOG2NP>::NT)
k_r2c3(const float *__restrict__ x, float2 *__restrict__ spec, long long xstride, const float2 *__restrict__ twN,
       const float2 *__restrict__ ptw) {
  constexpr int NP = 1 << LOG2NP, NC = 3 * NP, NT = CtaFftPlan<LOG2NP>::NT, SE = cta_fft_smem_elems<LOG2NP>();
  float2 *s = reinterpret_cast<float2 *>(qtam_long_smem);
  const float2 *z = reinterpret_cast<const float2 *>(x) + (size_t)blockIdx.x * NC;
#pragma unroll 1
  for (int r = 0; r < 3; ++r) {
    cta_fft_io<LOG2NP, NT, -1, true, false>(s + r * SE, Strided3In{z + r}, CtaFftNone{}, ptw);
    __syncthreads();
  }
  float2 *X = spec + (size_t)blockIdx.x * xstride;
  for (int f = threadIdx.x; f <= NC / 2; f += NT) {
    const int g = NC - f;
    const float2 A = r3_point<LOG2NP, -1>(s, s + SE, s + 2 * SE, f, twN);
    const float2 B = (f == 0) ? A : r3_point<LOG2NP, -1>(s, s + SE, s + 2 * SE, g, twN);
    const float2 E = make_float2(0.5f * (A.x + B.x), 0.5f * (A.y - B.y));
    const float2 D = make_float2(0.5f * (A.x - B.x), 0.5f * (A.y + B.y));
    float2 w = __ldg(twN + f);                   // e^{+2 pi i f/N}
    w.y = -w.y;
    const float2 t = make_float2(w.x * D.x - w.y * D.y, w.x * D.y + w.y * D.x);
    X[f] = make_float2(E.x + t.y, E.y - t.x);
    if (g != f) X[g] = make_float2(E.x - t.y, -E.y - t.x);
  }
}

template <int LOG2NP>
__global__ void __launch_bounds__(CtaFftPlan<LOG2NP>::NT)
k_c2c3(const float2 *__restrict__ spec, long long xstride, const float2 *__restrict__ twN,
       const float2 *__restrict__ ptw, float *__restrict__ x_out) {
  constexpr int NP = 1 << LOG2NP, NC = 3 * NP, NT = CtaFftPlan<LOG2NP>::NT, SE = cta_fft_smem_elems<LOG2NP>();
  float2 *s = reinterpret_cast<float2 *>(qtam_long_smem);
  const float2 *z = spec + (size_t)blockIdx.x * xstride;
#pragma unroll 1
  for (int r = 0; r < 3; ++r) {
    cta_fft_io<LOG2NP, NT, +1, true, false>(s + r * SE, Strided3In{z + r}, CtaFftNone{}, ptw);
    __syncthreads();
  }
  float2 *out = reinterpret_cast<float2 *>(x_out) + (size_t)blockIdx.x * NC;
  for (int f = threadIdx.x; f < NC; f += NT) out[f] = r3_point<LOG2NP, +1>(s, s + SE, s + 2 * SE, f, twN);
}

template <int LOG2NP> static bool r3_prepare(qtam_plan *p) {
  const size_t smem = sizeof(float2) * (size_t)r3_smem_elems<LOG2NP>();
  return kernel_prepare(p->cfg_r3[0], k_r2c3<LOG2NP>, CtaFftPlan<LOG2NP>::NT, smem) &&
         kernel_prepare(p->cfg_r3[1], k_c2c3<LOG2NP>, CtaFftPlan<LOG2NP>::NT, smem);
}

bool fast_r3_ok(const qtam_plan *p) { return p->cfg_r3[0].ready && p->cfg_r3[1].ready; }

template <int LOG2NP> static qtam_status r3_launch(qtam_plan *p, bool fwd, const void *d_in, void *d_out, int batch,
                                                   cudaStream_t st) {
  const float2 *twN = static_cast<const float2 *>(p->d_twN), *ptw = static_cast<const float2 *>(p->d_ptw_mid);
  const double nbytes = (double)batch * 4.0 * (double)p->hp.N;
  if (fwd) {
    LaunchScope ls(p, st, K_R2C_FAST, nbytes, nbytes + (double)batch * 8.0 * (double)p->hp.nb);
    k_r2c3<LOG2NP><<<(unsigned)batch, CtaFftPlan<LOG2NP>::NT, p->cfg_r3[0].smem, st>>>(
        static_cast<const float *>(d_in), static_cast<float2 *>(p->d_spec), p->xstride, twN, ptw);
  } else {
    LaunchScope ls(p, st, K_C2C_FAST, nbytes, 2.0 * nbytes);
    k_c2c3<LOG2NP><<<(unsigned)batch, CtaFftPlan<LOG2NP>::NT, p->cfg_r3[1].smem, st>>>(
        static_cast<const float2 *>(p->d_spec), p->xstride, twN, ptw, static_cast<float *>(d_out));
  }
  QTAM_LAUNCH_CHECK();
  return QTAM_OK;
}

// fwd: x -> spectrum buffer (rows a1); else: pre-processed spectrum buffer (k_combine_runs) -> x_out (row a8)
qtam_status fast_r3(qtam_plan *p, bool fwd, const void *d_in, void *d_out, int batch, cudaStream_t st) {
  switch (p->mid_log2n) {
    case 11: return r3_launch<11>(p, fwd, d_in, d_out, batch, st);
    case 12: return r3_launch<12>(p, fwd, d_in, d_out, batch, st);
    case 13: return r3_launch<13>(p, fwd, d_in, d_out, batch, st);
    default: return QTAM_ERR_UNSUPPORTED;
  }
}

bool fast_cfft_mid_ok(const qtam_plan *p, int log2n) { return p->d_ptw_mid != nullptr && log2n == p->mid_log2n; }

qtam_status fast_cfft_mid(qtam_plan *p, const void *in, long long in_stride, void *out, long long out_stride,
                          int log2n, int count, int dir, float scale, cudaStream_t st, double algo) {
  const float2 *i = static_cast<const float2 *>(in);
  float2 *o = static_cast<float2 *>(out);
  switch (log2n) {
    case 11: return mid_launch<11>(p, i, in_stride, o, out_stride, count, dir, scale, st, algo);
    case 12: return mid_launch<12>(p, i, in_stride, o, out_stride, count, dir, scale, st, algo);
    case 13: return mid_launch<13>(p, i, in_stride, o, out_stride, count, dir, scale, st, algo);
    case 14: return mid_launch<14>(p, i, in_stride, o, out_stride, count, dir, scale, st, algo);
    default: return QTAM_ERR_UNSUPPORTED;
  }
}

bool fast_cfft_long_ok(const qtam_plan *p, int log2n) {
  return p->d_ptw_long != nullptr && log2n > kLongLog2N2 && log2n <= kLongLog2N2 + 6;
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
    case 6: return long_launch<6>(p, i, in_stride, o, out_stride, t, tmp_stride, count, dir, scale, st, algo_in, algo_out);
    default: return QTAM_ERR_UNSUPPORTED;
  }
}

qtam_status build_long_fft(qtam_plan *p) {
  int lnc = 0;
  while ((int64_t(1) << lnc) < p->sub_n) ++lnc;    // log2 of the power-of-two complex FFT behind the long transform
  if (p->esz == 4 && !p->n_pow2 && lnc >= 11 && lnc <= 14) {
    // N = 3 * 2^k: the three transforms of N/6 points per segment run one CTA each
    bool ok = false;
    switch (lnc) {
      case 11: ok = mid_prepare<11>(p); break;
      case 12: ok = mid_prepare<12>(p); break;
      case 13: ok = mid_prepare<13>(p); break;
      default: ok = mid_prepare<14>(p); break;
    }
    if (!ok) return QTAM_ERR_CUDA;
    p->mid_log2n = lnc;
    // ... or, when three of them fit one CTA's shared memory, the whole long transform does
    ok = true;
    switch (lnc) {
      case 11: ok = r3_prepare<11>(p); break;
      case 12: ok = r3_prepare<12>(p); break;
      case 13: ok = r3_prepare<13>(p); break;
      default: break;
    }
    if (!ok) return QTAM_ERR_CUDA;
    return QTAM_OK;
  }
  if (p->esz != 4 || lnc <= kLongLog2N2 || lnc > kLongLog2N2 + 6) return QTAM_OK;
  std::vector<float> t;
  fill_cta_fft_tables<kLongLog2N2, CtaFftPlan<kLongLog2N2>::NT>(t);
  if (cudaMalloc(&p->d_ptw_long, t.size() * sizeof(float)) != cudaSuccess) return QTAM_ERR_ALLOC;
  p->device_bytes += t.size() * sizeof(float);
  if (cudaMemcpy(p->d_ptw_long, t.data(), t.size() * sizeof(float), cudaMemcpyHostToDevice) != cudaSuccess)
    return QTAM_ERR_CUDA;
  const size_t smem = sizeof(float2) * (size_t)cta_fft_smem_elems<kLongLog2N2>();
  if (!raise_dynamic_smem(reinterpret_cast<const void *>(k_long_b<-1>), smem) ||
      !raise_dynamic_smem(reinterpret_cast<const void *>(k_long_b<+1>), smem) ||
      !raise_dynamic_smem(reinterpret_cast<const void *>(k_long_b_res<-1>), smem) ||
      !raise_dynamic_smem(reinterpret_cast<const void *>(k_long_b_res<+1>), smem))
    return QTAM_ERR_CUDA;
  return QTAM_OK;
}

}  // namespace qtam
