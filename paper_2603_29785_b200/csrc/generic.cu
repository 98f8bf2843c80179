// generic.cu -- the "correct for everything" CUDA path of libqtam: any power-of-two N, any row
// length M, float and double.  Shared-memory Stockham radix-4 (radix-2 first pass when log2 M is
// odd) with ping-pong buffers; FFTs larger than the shared-memory cap are split
//   - long FFT:   four-step  Nc = N1 x N2 (column FFTs + twiddle, then row FFTs)
//   - long rows:  M = R1 x M2, decimation over the input residue (forward) or redundant first
//                 butterfly (inverse), R1 <= 16
// The tuned kernels (fast.cu, inv_tiled.cu, threshold_fast.cu) take over the shapes they cover; everything else runs here.
//
// Hot-path steps: a1 long R2C, a2 window gather + baseband shift (PAPER.md:323-325,
// C46 :583), a3 short inverse FFT scaled (N*M)^(-1/2) (C47 :589), a4 row-median threshold
// (BASELINE.json cfg 5), a5 per-row FFT + window + sqrt(N/M) (C49 :598), a6 sum over rows as a
// segmented reduction over bins, a7 division by P (Eq. 11 :135), a8 long C2R, a9 dense tiles (C3 :377).

#include "cplx.cuh"
#include "device_plan.hpp"
#include "thrbits.cuh"

namespace qtam {

// ---------------------------------------------------------------------------------------------------
// Block-level Stockham FFT on `total` = S*M points in shared memory; S sequences of length
// M = 2^log2M, each contiguous.  dir = +1: e^{+2 pi i jk/M} (unscaled inverse), -1: forward.
// Returns the buffer that holds the result (natural order).  Ends with a __syncthreads().
// ---------------------------------------------------------------------------------------------------
template <typename T>
__device__ C2<T> *block_fft(C2<T> *a, C2<T> *b, int log2M, int total, int dir,
                            const C2<T> *__restrict__ tw, int log2twn) {
  typedef C2<T> V;
  int log2Ns = 0;
  int rem = log2M;
  __syncthreads();
  while (rem > 0) {
    const int lr = (rem & 1) ? 1 : 2;         // radix 2 only as the first pass of an odd log2M
    const int nbf = total >> lr;              // butterflies over all sequences
    const int MR = (1 << log2M) >> lr;        // butterflies per sequence
    const int Ns = 1 << log2Ns;
    const int tshift = log2twn - log2Ns - lr; // w_{Ns*R}^k = tw[k << tshift]
    for (int idx = threadIdx.x; idx < nbf; idx += blockDim.x) {
      const int t = idx >> (log2M - lr);
      const int i = idx & (MR - 1);
      const int k = i & (Ns - 1);
      const V *src = a + ((size_t)t << log2M) + i;
      V *dst = b + ((size_t)t << log2M) + ((i - k) << lr) + k;
      if (lr == 1) {
        V v0 = src[0], v1 = src[MR];
        if (log2Ns > 0) v1 = cmul(v1, tw_get(tw, (long long)k << tshift, dir));
        dst[0] = cadd(v0, v1);
        dst[Ns] = csub(v0, v1);
      } else {
        V v0 = src[0], v1 = src[MR], v2 = src[2 * MR], v3 = src[3 * MR];
        if (log2Ns > 0) {
          v1 = cmul(v1, tw_get(tw, (long long)k << tshift, dir));
          v2 = cmul(v2, tw_get(tw, (long long)(2 * k) << tshift, dir));
          v3 = cmul(v3, tw_get(tw, (long long)(3 * k) << tshift, dir));
        }
        V a0 = cadd(v0, v2), a1 = csub(v0, v2), a2 = cadd(v1, v3), a3 = cmul_i(csub(v1, v3), dir);
        dst[0] = cadd(a0, a2);
        dst[Ns] = cadd(a1, a3);
        dst[2 * Ns] = csub(a0, a2);
        dst[3 * Ns] = csub(a1, a3);
      }
    }
    __syncthreads();
    V *tmp = a; a = b; b = tmp;
    log2Ns += lr;
    rem -= lr;
  }
  return a;
}

extern __shared__ __align__(16) unsigned char qtam_smem[];

// ---------------------------------------------------------------------------------------------------
// a2 + a3: window gather, baseband shift, short inverse FFT.  One CTA per (work item, segment).
// ---------------------------------------------------------------------------------------------------
template <typename T>
__global__ void k_fwd_rows(const RowDev *__restrict__ rows, const WorkItem *__restrict__ items,
                           const C2<T> *__restrict__ spec, long long xstride, int nbins,
                           const T *__restrict__ win, const C2<T> *__restrict__ tw, int log2twn,
                           C2<T> *__restrict__ coef, long long ctot, int bufpts,
                           const int *__restrict__ fol_ptr, const long long *__restrict__ fol_off) {
  typedef C2<T> V;
  V *a = reinterpret_cast<V *>(qtam_smem);
  V *bb = a + bufpts;
  const WorkItem it = items[blockIdx.x];
  const RowDev r = rows[it.row];
  const int M2 = 1 << it.log2M2;
  const V *X = spec + (long long)blockIdx.y * xstride;
  for (int i = threadIdx.x; i < M2; i += blockDim.x) {
    const int j = it.j1 + it.R1 * i;                 // index in the M-array, 0..M-1
    const int jj = (j < (r.M >> 1)) ? j : j - r.M;   // signed offset from the window centre (R6)
    const int f = r.kc + jj;
    V v = cmk<T>(0, 0);
    if (jj >= -r.dk && jj <= r.dk && f >= 0 && f < nbins) {   // clip at DC / Nyquist (R8)
      const T w = win[r.woff + jj + r.dk];
      const V x = X[f];
      v = cmk<T>(x.x * w, x.y * w);
    }
    a[i] = v;
  }
  V *res = block_fft<T>(a, bb, it.log2M2, M2, +1, tw, log2twn);
  const T sc = (T)r.fwd_scale;
  V *out = coef + (long long)blockIdx.y * ctot + r.offset + (long long)it.j1 * M2;
  for (int i = threadIdx.x; i < M2; i += blockDim.x) {
    V v = res[i];
    if (it.R1 > 1) v = cmul(v, tw_get(tw, (long long)(it.j1 * i) << (log2twn - r.log2M), +1));
    v = cscale(v, sc);
    out[i] = v;
    // rows with the same centre bin and half-width (other Q-planes under the clamp) have these very values
    for (int e = fol_ptr[it.row]; e < fol_ptr[it.row + 1]; ++e)
      coef[(long long)blockIdx.y * ctot + fol_off[e] + i] = v;
  }
}

// long rows: Y[n1*M2+n2] = sum_j1 z_j1[n2] e^{+2 pi i j1 n1/R1}, in place over the row's coefficients
template <typename T>
__global__ void k_fwd_combine(const RowDev *__restrict__ rows, const int *__restrict__ bigrows,
                              int cap_log2, const C2<T> *__restrict__ tw, int log2twn,
                              C2<T> *__restrict__ coef, long long ctot) {
  typedef C2<T> V;
  const RowDev r = rows[bigrows[blockIdx.y]];
  const int log2R1 = r.log2M - cap_log2;
  const int R1 = 1 << log2R1;
  const int M2 = 1 << cap_log2;
  const int n2 = blockIdx.x * blockDim.x + threadIdx.x;
  if (n2 >= M2) return;
  V *base = coef + (long long)blockIdx.z * ctot + r.offset + n2;
  V z[16], y[16];
  for (int j1 = 0; j1 < R1; ++j1) z[j1] = base[(long long)j1 * M2];
  for (int n1 = 0; n1 < R1; ++n1) {
    V acc = z[0];
    for (int j1 = 1; j1 < R1; ++j1)
      acc = cadd(acc, cmul(z[j1], tw_get(tw, (long long)((j1 * n1) & (R1 - 1)) << (log2twn - log2R1), +1)));
    y[n1] = acc;
  }
  for (int n1 = 0; n1 < R1; ++n1) base[(long long)n1 * M2] = y[n1];
}

// ---------------------------------------------------------------------------------------------------
// complex FFT building blocks (long FFT a1/a8, dense a9)
// ---------------------------------------------------------------------------------------------------
// contiguous sequences of n = 2^log2n <= cap points, one CTA each
template <typename T>
__global__ void k_cfft_seq(const C2<T> *__restrict__ in, long long in_stride, C2<T> *__restrict__ out,
                           long long out_stride, int log2n, int dir, const C2<T> *__restrict__ tw,
                           int log2twn, T scale, int bufpts) {
  typedef C2<T> V;
  V *a = reinterpret_cast<V *>(qtam_smem);
  V *bb = a + bufpts;
  const int n = 1 << log2n;
  const V *src = in + (long long)blockIdx.x * in_stride;
  for (int i = threadIdx.x; i < n; i += blockDim.x) a[i] = src[i];
  V *res = block_fft<T>(a, bb, log2n, n, dir, tw, log2twn);
  V *dst = out + (long long)blockIdx.x * out_stride;
  for (int i = threadIdx.x; i < n; i += blockDim.x) dst[i] = cscale(res[i], scale);
}

// four-step, step A: for a tile of Tc columns j2, FFT over j1 (stride N2), times w_Nc^{dir n1 j2}.
// `in` may equal `out` (the dense path runs it in place: a CTA reads its whole address set into shared memory
// before it stores to the same set, and CTAs touch disjoint sets), so neither pointer is __restrict__.
template <typename T>
__global__ void k_cfft_cols(const C2<T> *in, long long in_stride, C2<T> *out,
                            long long out_stride, int log2N1, int log2N2, int log2Tc, int dir,
                            const C2<T> *__restrict__ tw, int log2twn, int bufpts) {
  typedef C2<T> V;
  V *a = reinterpret_cast<V *>(qtam_smem);
  V *bb = a + bufpts;
  const int Tc = 1 << log2Tc;
  const int total = Tc << log2N1;
  const int j20 = blockIdx.x << log2Tc;
  const V *src = in + (long long)blockIdx.y * in_stride;
  for (int idx = threadIdx.x; idx < total; idx += blockDim.x) {
    const int t = idx & (Tc - 1), j1 = idx >> log2Tc;
    a[(t << log2N1) + j1] = src[((long long)j1 << log2N2) + j20 + t];
  }
  V *res = block_fft<T>(a, bb, log2N1, total, dir, tw, log2twn);
  V *dst = out + (long long)blockIdx.y * out_stride;
  const int tsh = log2twn - log2N1 - log2N2;
  for (int idx = threadIdx.x; idx < total; idx += blockDim.x) {
    const int t = idx & (Tc - 1), n1 = idx >> log2Tc;
    const long long j2 = j20 + t;
    V v = cmul(res[(t << log2N1) + n1], tw_get(tw, ((long long)n1 * j2) << tsh, dir));
    dst[((long long)n1 << log2N2) + j2] = v;
  }
}

// four-step, step B: for a tile of Tr rows n1, FFT over j2 (contiguous); Z[n1 + N1*n2]
template <typename T>
__global__ void k_cfft_rows(const C2<T> *__restrict__ in, long long in_stride, C2<T> *__restrict__ out,
                            long long out_stride, int log2N1, int log2N2, int log2Tr, int dir,
                            const C2<T> *__restrict__ tw, int log2twn, T scale, int bufpts) {
  typedef C2<T> V;
  V *a = reinterpret_cast<V *>(qtam_smem);
  V *bb = a + bufpts;
  const int Tr = 1 << log2Tr;
  const int total = Tr << log2N2;
  const int n10 = blockIdx.x << log2Tr;
  const V *src = in + (long long)blockIdx.y * in_stride + ((long long)n10 << log2N2);
  for (int idx = threadIdx.x; idx < total; idx += blockDim.x) a[idx] = src[idx];
  V *res = block_fft<T>(a, bb, log2N2, total, dir, tw, log2twn);
  V *dst = out + (long long)blockIdx.y * out_stride + n10;
  for (int idx = threadIdx.x; idx < total; idx += blockDim.x) {
    const int t = idx & (Tr - 1), n2 = idx >> log2Tr;
    dst[((long long)n2 << log2N1) + t] = cscale(res[(t << log2N2) + n2], scale);
  }
}

// Radix-3 step of a complex FFT of n = 3 Np points (segment lengths N = 3 * 2^k: the paper's 6 s at 4096 Hz,
// :178, :339), decimation in time: F_r = DFT_Np of z[3 n2 + r], Z[k + Np m] = sum_r w_3^{r m} w_n^{r k} F_r[k].
// k_split3 separates the three decimated sequences, the power-of-two transform runs on them, k_combine3 is the
// butterfly.  tw: e^{+2 pi i k/N} (period N = tw_mul * n).
template <typename T>
__global__ void k_split3(const C2<T> *__restrict__ in, long long in_stride, C2<T> *__restrict__ a, int Np) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= 3 * Np) return;
  a[(long long)blockIdx.y * 3 * Np + (long long)(i % 3) * Np + i / 3] = in[(long long)blockIdx.y * in_stride + i];
}

template <typename T>
__global__ void k_combine3(const C2<T> *__restrict__ b, C2<T> *__restrict__ out, long long out_stride, int Np,
                           int dir, const C2<T> *__restrict__ tw, long long tw_mul, long long N, T scale) {
  typedef C2<T> V;
  const int k = blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= Np) return;
  const V *B = b + (long long)blockIdx.y * 3 * Np;
  const V f0 = B[k];
  const V a1 = cmul(B[Np + k], tw_get(tw, ((long long)k * tw_mul) % N, dir));
  const V a2 = cmul(B[2 * (long long)Np + k], tw_get(tw, (2LL * k * tw_mul) % N, dir));
  // w_3 = -1/2 + dir i sqrt(3)/2:  w_3 a1 + w_3^2 a2 = -(a1 + a2)/2 + dir i (sqrt(3)/2) (a1 - a2)
  const V s = cadd(a1, a2), d = csub(a1, a2);
  const T h = (T)0.86602540378443864676 * (T)dir;
  const V m = cmk<T>(f0.x - (T)0.5 * s.x, f0.y - (T)0.5 * s.y), r = cmk<T>(-h * d.y, h * d.x);
  V *O = out + (long long)blockIdx.y * out_stride;
  O[k] = cscale(cadd(f0, s), scale);
  O[Np + k] = cscale(cadd(m, r), scale);
  O[2 * (long long)Np + k] = cscale(csub(m, r), scale);
}

// a1 tail: X[f] from the half-length complex FFT Z of z[m] = x[2m] + i x[2m+1]; in place in `spec`
//   X[f] = (Z[f] + conj Z[Nc-f])/2 - (i/2) e^{-2 pi i f/N} (Z[f] - conj Z[Nc-f]),  f = 0..Nc
template <typename T>
__global__ void k_r2c_post(C2<T> *__restrict__ spec, long long xstride, int Nc,
                           const C2<T> *__restrict__ tw) {
  typedef C2<T> V;
  const int f = blockIdx.x * blockDim.x + threadIdx.x;
  if (f > Nc / 2) return;
  V *S = spec + (long long)blockIdx.y * xstride;
  const int g = Nc - f;
  const V A = S[f];
  const V B = (f == 0) ? A : S[g];
  const T h = (T)0.5;
  const V E = cmk<T>(h * (A.x + B.x), h * (A.y - B.y));
  const V D = cmk<T>(h * (A.x - B.x), h * (A.y + B.y));
  const V w = tw_get(tw, f, -1);       // twn == N
  const V t = cmul(w, D);
  S[f] = cmk<T>(E.x + t.y, E.y - t.x);
  if (g != f) S[g] = cmk<T>(E.x - t.y, -E.y - t.x);
}

// a8 head: Z[f] = E + i O, E = (X[f] + conj X[Nc-f])/2, O = (X[f] - conj X[Nc-f])/2 e^{+2 pi i f/N},
// scaled by 1/Nc; DC and Nyquist take their real parts (row a8); in place in `spec`
template <typename T>
__global__ void k_c2r_pre(C2<T> *__restrict__ spec, long long xstride, int Nc,
                          const C2<T> *__restrict__ tw) {
  typedef C2<T> V;
  const int f = blockIdx.x * blockDim.x + threadIdx.x;
  if (f > Nc / 2) return;
  V *S = spec + (long long)blockIdx.y * xstride;
  const int g = Nc - f;
  V A = S[f], B = S[g];
  if (f == 0) { A.y = 0; B.y = 0; }
  const T h = (T)0.5 / (T)Nc;
  const V E = cmk<T>(h * (A.x + B.x), h * (A.y - B.y));
  const V D = cmk<T>(h * (A.x - B.x), h * (A.y + B.y));
  const V O = cmul(D, tw_get(tw, f, +1));
  S[f] = cmk<T>(E.x - O.y, E.y + O.x);                 // E + i O
  if (g != f && f != 0) S[g] = cmk<T>(E.x + O.y, -E.y + O.x);   // conj(E) + i conj(O)
}

// ---------------------------------------------------------------------------------------------------
// a5: per-row forward FFT, window, sqrt(N/M); band values to the band workspace
// ---------------------------------------------------------------------------------------------------
template <typename T>
__global__ void k_inv_rows(const RowDev *__restrict__ rows, const WorkItem *__restrict__ items,
                           const C2<T> *__restrict__ coef, long long ctot, const T *__restrict__ win,
                           const C2<T> *__restrict__ tw, int log2twn, C2<T> *__restrict__ band,
                           long long sumL, int nbins, int plane, int bufpts,
                           const int *__restrict__ fol_ptr, const long long *__restrict__ fol_off,
                           const long long *__restrict__ fol_woff) {
  typedef C2<T> V;
  V *a = reinterpret_cast<V *>(qtam_smem);
  V *bb = a + bufpts;
  const WorkItem it = items[blockIdx.x];
  const RowDev r = rows[it.row];
  if (plane >= 0 && r.plane != plane) return;
  const int M2 = 1 << it.log2M2;
  const V *Y = coef + (long long)blockIdx.y * ctot + r.offset;
  // joint inverse (fol_ptr != nullptr): the item list holds one leader per set of identical rows; the
  // followers' coefficient rows are added before the transform (linearity) and their band slots are zeroed
  const int e0 = fol_ptr ? fol_ptr[it.row] : 0, e1 = fol_ptr ? fol_ptr[it.row + 1] : 0;
  if (it.R1 == 1) {
    for (int i = threadIdx.x; i < M2; i += blockDim.x) {
      V acc = Y[i];
      for (int e = e0; e < e1; ++e) acc = cadd(acc, coef[(long long)blockIdx.y * ctot + fol_off[e] + i]);
      a[i] = acc;
    }
  } else {
    const int log2R1 = r.log2M - it.log2M2;
    for (int i = threadIdx.x; i < M2; i += blockDim.x) {
      V acc = Y[i];
      for (int n1 = 1; n1 < it.R1; ++n1)
        acc = cadd(acc, cmul(Y[(long long)n1 * M2 + i],
                             tw_get(tw, (long long)((it.j1 * n1) & (it.R1 - 1)) << (log2twn - log2R1), -1)));
      a[i] = cmul(acc, tw_get(tw, (long long)(it.j1 * i) << (log2twn - r.log2M), -1));
    }
  }
  V *res = block_fft<T>(a, bb, it.log2M2, M2, -1, tw, log2twn);
  const T amp = (T)r.inv_amp;
  V *G = band + (long long)blockIdx.y * sumL + r.woff;
  for (int i = threadIdx.x; i < M2; i += blockDim.x) {
    const int j = it.j1 + it.R1 * i;
    const int jj = (j < (r.M >> 1)) ? j : j - r.M;
    const int f = r.kc + jj;
    if (jj >= -r.dk && jj <= r.dk && f >= 0 && f < nbins) {
      const T w = win[r.woff + jj + r.dk] * amp;
      G[jj + r.dk] = cscale(res[i], w);
      for (int e = e0; e < e1; ++e) band[(long long)blockIdx.y * sumL + fol_woff[e] + jj + r.dk] = cmk<T>(0, 0);
    }
  }
}

// a6 + a7: S[f] = sum over the bin's CSR entries (ascending row order), Xhat = S * (1/P) on the cover
template <typename T>
__global__ void k_inv_reduce(const C2<T> *__restrict__ band, long long sumL,
                             const int32_t *__restrict__ ptr, const int32_t *__restrict__ idx,
                             const T *__restrict__ invP, int nbins, int nsets, int plo, int phi, int plane,
                             C2<T> *__restrict__ spec, long long xstride) {
  typedef C2<T> V;
  const int f = blockIdx.x * blockDim.x + threadIdx.x;
  if (f >= nbins) return;
  // the bin's entries: sets plo .. phi-1 of the CSR's nsets per bin (see csr_select)
  const int lo = ptr[(long long)f * nsets + plo];
  const int hi = ptr[(long long)f * nsets + phi];
  const V *G = band + (long long)blockIdx.y * sumL;
  V s = cmk<T>(0, 0);
  for (int e = lo; e < hi; ++e) s = cadd(s, G[idx[e]]);
  const T ip = invP[(long long)(plane + 1) * nbins + f];
  spec[(long long)blockIdx.y * xstride + f] = cscale(s, ip);
}

// a9: place the windowed band of one row at its own bins of a length-N spectrum (scaled 1/N)
template <typename T>
__global__ void k_dense_place(const RowDev *__restrict__ rows, int row, const C2<T> *__restrict__ spec,
                              long long xstride, int nbins, const T *__restrict__ win,
                              C2<T> *__restrict__ ws, int N, T eps_norm) {
  typedef C2<T> V;
  const int f = blockIdx.x * blockDim.x + threadIdx.x;
  if (f >= N) return;
  const RowDev r = rows[row];
  const int jj = f - r.kc;
  V v = cmk<T>(0, 0);
  // eps_norm = epsilon x the row's norm (Eq. 12 :143, R17): the window is floored there on the support and
  // equals it on the rest of the one-sided spectrum; 0 = the plain window
  if (jj >= -r.dk && jj <= r.dk && f < nbins) {
    T w = win[r.woff + jj + r.dk];
    if (w < eps_norm) w = eps_norm;
    v = cscale(spec[(long long)blockIdx.y * xstride + f], w / (T)N);
  } else if (eps_norm > (T)0 && f < nbins) {
    v = cscale(spec[(long long)blockIdx.y * xstride + f], eps_norm / (T)N);
  }
  ws[(long long)blockIdx.y * N + f] = v;
}

// Eq. 13 (:148): Xhat[f] = F[T_k][f] / W_k[f], f = 0..N/2, with the window of Eq. 12
template <typename T>
__global__ void k_dense_divide(const RowDev *__restrict__ rows, int row, const C2<T> *__restrict__ ft, int N,
                               const T *__restrict__ win, T eps_norm, int nbins, C2<T> *__restrict__ spec,
                               long long xstride) {
  const int f = blockIdx.x * blockDim.x + threadIdx.x;
  if (f >= nbins) return;
  const RowDev r = rows[row];
  const int jj = f - r.kc;
  T w = eps_norm;
  if (jj >= -r.dk && jj <= r.dk) {
    w = win[r.woff + jj + r.dk];
    if (w < eps_norm) w = eps_norm;
  }
  spec[(long long)blockIdx.y * xstride + f] = cscale(ft[(long long)blockIdx.y * N + f], (T)1 / w);
}

// ---------------------------------------------------------------------------------------------------
// a4: row-median threshold.  Selection by radix-select on the bit patterns of the (non-negative)
// magnitudes; every operation correctly rounded in T, no fused multiply-add (DESIGN.md "threshold
// arithmetic"), so the decisions equal the oracle's bit for bit on identical inputs.
// ---------------------------------------------------------------------------------------------------
__device__ __forceinline__ int block_sum(int v, int *sm) {
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  const int w = threadIdx.x >> 5, nw = (blockDim.x + 31) >> 5;
  __syncthreads();
  if ((threadIdx.x & 31) == 0) sm[w] = v;
  __syncthreads();
  int t = 0;
  for (int i = 0; i < nw; ++i) t += sm[i];
  return t;
}

template <typename T>
__global__ void k_threshold(const RowDev *__restrict__ rows, C2<T> *__restrict__ coef, long long ctot,
                            T kappa, int cache_pts, int min_log2M) {
  typedef C2<T> V;
  typedef typename Bits<T>::U U;
  __shared__ int red[32];
  __shared__ U red_min[32];
  T *cache = reinterpret_cast<T *>(qtam_smem);
  const RowDev r = rows[blockIdx.x];
  if (r.log2M < min_log2M) return;   // shorter rows run in threshold_fast.cu
  V *Y = coef + (long long)blockIdx.y * ctot + r.offset;
  const int M = r.M;
  const bool cached = M <= cache_pts;
  if (cached) {
    for (int i = threadIdx.x; i < M; i += blockDim.x) { const V y = Y[i]; cache[i] = Bits<T>::mag(y.x, y.y); }
    __syncthreads();
  }
  auto magat = [&](int i) -> T {
    if (cached) return cache[i];
    const V y = Y[i];
    return Bits<T>::mag(y.x, y.y);
  };
  // rank M/2-1 (0-based) by radix select, most significant bit first (sign bit is 0)
  U prefix = 0;
  int kk = M / 2 - 1;
  for (int bit = Bits<T>::nbits - 2; bit >= 0; --bit) {
    const U himask = ~((((U)1) << (bit + 1)) - 1);
    int c0 = 0;
    for (int i = threadIdx.x; i < M; i += blockDim.x) {
      const U u = Bits<T>::of(magat(i));
      if ((u & himask) == prefix && ((u >> bit) & 1) == 0) ++c0;
    }
    c0 = block_sum(c0, red);
    if (kk >= c0) { kk -= c0; prefix |= ((U)1) << bit; }
  }
  const U lo_bits = prefix;
  // next order statistic: equal to lo if enough values are <= lo, else the smallest value > lo
  int cle = 0;
  U mn = ~(U)0;
  for (int i = threadIdx.x; i < M; i += blockDim.x) {
    const U u = Bits<T>::of(magat(i));
    if (u <= lo_bits) ++cle; else if (u < mn) mn = u;
  }
  cle = block_sum(cle, red);
  for (int o = 16; o > 0; o >>= 1) { const U other = __shfl_xor_sync(0xffffffffu, mn, o); if (other < mn) mn = other; }
  __syncthreads();
  if ((threadIdx.x & 31) == 0) red_min[threadIdx.x >> 5] = mn;
  __syncthreads();
  mn = ~(U)0;
  for (int i = 0; i < (int)((blockDim.x + 31) >> 5); ++i) if (red_min[i] < mn) mn = red_min[i];
  const T lo = Bits<T>::from(lo_bits);
  const T hi = (cle >= M / 2 + 1) ? lo : Bits<T>::from(mn);
  const T med = Bits<T>::mul((T)0.5, Bits<T>::add(lo, hi));
  const T thr = Bits<T>::mul(kappa, med);
  for (int i = threadIdx.x; i < M; i += blockDim.x)
    if (magat(i) < thr) Y[i] = cmk<T>(0, 0);
}

// ---------------------------------------------------------------------------------------------------
// host launchers
// ---------------------------------------------------------------------------------------------------
static int ilog2(long long v) { int l = 0; while ((1LL << l) < v) ++l; return l; }

template <typename K> static bool set_smem(K kernel, size_t bytes) {
  return raise_dynamic_smem(reinterpret_cast<const void *>(kernel), bytes);
}

constexpr int kThrCachePts = 8192;   // magnitudes k_threshold keeps in shared memory

// dynamic shared-memory limits of this file's kernels, set once at plan creation (the largest any launch asks for)
template <typename T> static bool prepare_t(const qtam_plan *p) {
  const size_t fft = 2 * sizeof(C2<T>) * ((size_t)1 << p->cap_log2);
  return set_smem(k_cfft_seq<T>, fft) && set_smem(k_cfft_cols<T>, fft) && set_smem(k_cfft_rows<T>, fft) &&
         set_smem(k_fwd_rows<T>, fft) && set_smem(k_inv_rows<T>, fft) &&
         set_smem(k_threshold<T>, sizeof(T) * (size_t)kThrCachePts);
}

// class c of the row kernels handles sub-transforms of up to 2^kClassLog2[c] points
static const int kClassLog2[qtam_plan::kClasses] = {8, 10, 12, 13};
static const int kClassThreads[qtam_plan::kClasses] = {64, 128, 256, 512};

int generic_class_of(int log2M2) {
  for (int c = 0; c < qtam_plan::kClasses; ++c)
    if (log2M2 <= kClassLog2[c]) return c;
  return -1;
}

// complex FFT of `count` sequences of n = 2^log2n points: in -> out (tmp used when n > cap; tmp may
// alias in, never out).  Strides in complex elements.  Unscaled times `scale`.
// algo_in / algo_out: compulsory bytes the first pass reads / the last pass writes, for the
// launch profile: the time series of the long R2C (in) or C2R (out); 0 for transforms of intermediates.
template <typename T>
static qtam_status cfft(qtam_plan *p, const C2<T> *in, long long in_stride, C2<T> *out,
                        long long out_stride, C2<T> *tmp, long long tmp_stride, int log2n, int count,
                        int dir, T scale, cudaStream_t st, double algo_in = 0.0, double algo_out = 0.0) {
  if constexpr (sizeof(T) == 4) {
    if (fast_cfft_long_ok(p, log2n) && tmp != out)
      return fast_cfft_long(p, in, in_stride, out, out_stride, tmp, tmp_stride, log2n, count, dir, scale, st,
                            algo_in, algo_out);
    if (fast_cfft_mid_ok(p, log2n) && in != out)
      return fast_cfft_mid(p, in, in_stride, out, out_stride, log2n, count, dir, scale, st, algo_in + algo_out);
  }
  const int cap = p->cap_log2;
  const C2<T> *tw = static_cast<const C2<T> *>(p->d_tw);
  const int log2twn = ilog2(p->twn);
  const int bufpts = 1 << cap;
  const size_t smem = 2 * sizeof(C2<T>) * (size_t)bufpts;
  if (log2n <= cap) {
    const int thr = log2n >= 10 ? 512 : (log2n >= 8 ? 128 : 64);
    {
      LaunchScope ls(p, st, K_CFFT_SEQ, algo_in + algo_out, 2.0 * sizeof(C2<T>) * (double)count * (double)(1 << log2n));
      k_cfft_seq<T><<<count, thr, smem, st>>>(in, in_stride, out, out_stride, log2n, dir, tw, log2twn, scale, bufpts);
    }
    QTAM_LAUNCH_CHECK();
    return QTAM_OK;
  }
  const int l1 = log2n / 2, l2 = log2n - l1;
  if (l2 > cap) return QTAM_ERR_UNSUPPORTED;
  int ltc = cap - l1; if (ltc > l2) ltc = l2;
  int ltr = cap - l2; if (ltr > l1) ltr = l1;
  dim3 ga((1 << l2) >> ltc, count), gb((1 << l1) >> ltr, count);
  const double pass_bytes = 2.0 * sizeof(C2<T>) * (double)count * (double)(1LL << log2n);
  {
    LaunchScope ls(p, st, K_CFFT_COLS, algo_in, pass_bytes);
    k_cfft_cols<T><<<ga, 512, smem, st>>>(in, in_stride, tmp, tmp_stride, l1, l2, ltc, dir, tw, log2twn, bufpts);
  }
  QTAM_LAUNCH_CHECK();
  {
    LaunchScope ls(p, st, K_CFFT_ROWS, algo_out, pass_bytes);
    k_cfft_rows<T><<<gb, 512, smem, st>>>(tmp, tmp_stride, out, out_stride, l1, l2, ltr, dir, tw, log2twn, scale, bufpts);
  }
  QTAM_LAUNCH_CHECK();
  return QTAM_OK;
}

// complex FFT of n = 2^a or 3 * 2^a points (the latter through the plan's radix-3 scratch: in and out are free
// to alias, tmp is not used)
template <typename T>
static qtam_status cfft_any(qtam_plan *p, const C2<T> *in, long long in_stride, C2<T> *out, long long out_stride,
                            C2<T> *tmp, long long tmp_stride, long long n, int count, int dir, T scale,
                            cudaStream_t st, double algo_in = 0.0, double algo_out = 0.0) {
  if ((n & (n - 1)) == 0)
    return cfft<T>(p, in, in_stride, out, out_stride, tmp, tmp_stride, ilog2(n), count, dir, scale, st, algo_in, algo_out);
  if (n % 3 != 0 || !p->d_ws3 || p->hp.N % n != 0 || n > p->hp.N) return QTAM_ERR_UNSUPPORTED;
  const int Np = (int)(n / 3);
  C2<T> *A = static_cast<C2<T> *>(p->d_ws3), *B = A + (size_t)p->max_batch * (size_t)p->hp.N;
  dim3 g3((unsigned)((3 * Np + 255) / 256), (unsigned)count), g1((unsigned)((Np + 255) / 256), (unsigned)count);
  const double bytes = 2.0 * sizeof(C2<T>) * (double)count * (double)n;
  {
    LaunchScope ls(p, st, K_SPLIT3, algo_in, bytes);
    k_split3<T><<<g3, 256, 0, st>>>(in, in_stride, A, Np);
  }
  QTAM_LAUNCH_CHECK();
  qtam_status s = cfft<T>(p, A, Np, B, Np, A, Np, ilog2(Np), 3 * count, dir, (T)1, st);
  if (s != QTAM_OK) return s;
  {
    LaunchScope ls(p, st, K_COMBINE3, algo_out, bytes);
    k_combine3<T><<<g1, 256, 0, st>>>(B, out, out_stride, Np, dir, static_cast<const C2<T> *>(p->d_twN),
                                      p->hp.N / n, p->hp.N, scale);
  }
  QTAM_LAUNCH_CHECK();
  return QTAM_OK;
}

template <typename T>
static qtam_status r2c_t(qtam_plan *p, const void *d_x, int batch, cudaStream_t st) {
  if (sizeof(T) == 4 && !p->n_pow2 && fast_r3_ok(p)) return fast_r3(p, true, d_x, nullptr, batch, st);
  p->sp_xt_fresh = false;
  if (sizeof(T) == 4 && long_residues_ok(p)) {
    const qtam_status sr = long_forward_residues(p, d_x, batch, st);
    p->sp_xt_fresh = sr == QTAM_OK;
    return sr;
  }
  const int Nc = (int)(p->hp.N / 2);
  C2<T> *spec = static_cast<C2<T> *>(p->d_spec);
  C2<T> *ws = static_cast<C2<T> *>(p->d_ws);
  qtam_status s = cfft_any<T>(p, static_cast<const C2<T> *>(d_x), Nc, spec, p->xstride, ws, p->hp.N,
                              Nc, batch, -1, (T)1, st, (double)batch * sizeof(T) * (double)p->hp.N, 0.0);
  if (s != QTAM_OK) return s;
  dim3 g((Nc / 2 + 1 + 255) / 256, batch);
  {
    LaunchScope ls(p, st, K_R2C_POST, 0.0, 2.0 * sizeof(C2<T>) * (double)batch * (double)Nc);
    k_r2c_post<T><<<g, 256, 0, st>>>(spec, p->xstride, Nc, static_cast<const C2<T> *>(p->d_twN));
  }
  QTAM_LAUNCH_CHECK();
  return QTAM_OK;
}

qtam_status generic_r2c(qtam_plan *p, const void *d_x, int batch, cudaStream_t st) {
  return p->esz == 4 ? r2c_t<float>(p, d_x, batch, st) : r2c_t<double>(p, d_x, batch, st);
}

template <typename T>
static qtam_status fwd_rows_t(qtam_plan *p, int batch, void *d_coef, cudaStream_t st) {
  const C2<T> *tw = static_cast<const C2<T> *>(p->d_tw);
  const int log2twn = ilog2(p->twn);
  for (int c = 0; c < qtam_plan::kClasses; ++c) {
    if (p->n_items_fwd[c] == 0) continue;
    const int bufpts = 1 << kClassLog2[c];
    const size_t smem = 2 * sizeof(C2<T>) * (size_t)bufpts;
    dim3 g(p->n_items_fwd[c], batch);
    {
      // reads the bands (L values per row), writes M coefficients per row
      LaunchScope ls(p, st, K_FWD_ROWS, sizeof(C2<T>) * (double)batch * p->class_M[c],
                     sizeof(C2<T>) * (double)batch * (p->class_L[c] + p->class_M[c]));
      k_fwd_rows<T><<<g, kClassThreads[c], smem, st>>>(
          p->d_rows, p->d_items_fwd[c], static_cast<const C2<T> *>(p->d_spec), p->xstride, (int)p->hp.nb,
          static_cast<const T *>(p->d_win), tw, log2twn, static_cast<C2<T> *>(d_coef), p->hp.ctot, bufpts,
          p->d_gfol_ptr, p->d_gfol_off);
    }
    QTAM_LAUNCH_CHECK();
  }
  if (p->n_bigrows > 0) {
    dim3 g(((1 << p->cap_log2) + 255) / 256, p->n_bigrows, batch);
    {
      LaunchScope ls(p, st, K_FWD_COMBINE, 0.0, 2.0 * sizeof(C2<T>) * (double)batch * p->big_M);
      k_fwd_combine<T><<<g, 256, 0, st>>>(p->d_rows, p->d_bigrows, p->cap_log2, tw, log2twn,
                                          static_cast<C2<T> *>(d_coef), p->hp.ctot);
    }
    QTAM_LAUNCH_CHECK();
  }
  return QTAM_OK;
}

qtam_status generic_forward_rows(qtam_plan *p, int batch, void *d_coef, cudaStream_t st) {
  return p->esz == 4 ? fwd_rows_t<float>(p, batch, d_coef, st) : fwd_rows_t<double>(p, batch, d_coef, st);
}

template <typename T>
static qtam_status inv_rows_t(qtam_plan *p, const void *d_coef, int batch, int plane, cudaStream_t st) {
  const C2<T> *tw = static_cast<const C2<T> *>(p->d_tw);
  const int log2twn = ilog2(p->twn);
  for (int c = 0; c < qtam_plan::kClasses; ++c) {
    // the joint inverse takes the leader lists (identical rows added first), one plane alone every row
    const bool lead = plane < 0;
    const int n_it = lead ? p->n_items_fwd[c] : p->n_items[c];
    if (n_it == 0) continue;
    const int bufpts = 1 << kClassLog2[c];
    const size_t smem = 2 * sizeof(C2<T>) * (size_t)bufpts;
    dim3 g(n_it, batch);
    {
      LaunchScope ls(p, st, K_INV_ROWS, sizeof(C2<T>) * (double)batch * p->class_M[c],
                     sizeof(C2<T>) * (double)batch * (p->class_L[c] + p->class_M[c]));
      k_inv_rows<T><<<g, kClassThreads[c], smem, st>>>(
          p->d_rows, lead ? p->d_items_fwd[c] : p->d_items[c], static_cast<const C2<T> *>(d_coef), p->hp.ctot,
          static_cast<const T *>(p->d_win), tw, log2twn, static_cast<C2<T> *>(p->d_band), p->hp.sumL,
          (int)p->hp.nb, plane, bufpts, lead ? p->d_gfol_ptr : nullptr, p->d_gfol_off, p->d_gfol_woff);
    }
    QTAM_LAUNCH_CHECK();
  }
  return QTAM_OK;
}

qtam_status generic_inverse_rows(qtam_plan *p, const void *d_coef, int batch, int plane, cudaStream_t st) {
  return p->esz == 4 ? inv_rows_t<float>(p, d_coef, batch, plane, st)
                     : inv_rows_t<double>(p, d_coef, batch, plane, st);
}

template <typename T>
static qtam_status inv_reduce_t(qtam_plan *p, int batch, int plane, cudaStream_t st) {
  dim3 g((unsigned)((p->hp.nb + 255) / 256), batch);
  {
    LaunchScope ls(p, st, K_INV_REDUCE, 0.0,
                   (double)batch * (sizeof(C2<T>) * ((double)p->hp.sumL + (double)p->hp.nb)));
    const CsrSel cs = csr_select(p, plane);
    k_inv_reduce<T><<<g, 256, 0, st>>>(static_cast<const C2<T> *>(p->d_band), p->hp.sumL, cs.ptr, cs.idx,
                                       static_cast<const T *>(p->d_invP), (int)p->hp.nb, cs.nsets, cs.plo,
                                       cs.phi, plane, static_cast<C2<T> *>(p->d_spec), p->xstride);
  }
  QTAM_LAUNCH_CHECK();
  return QTAM_OK;
}

qtam_status generic_inverse_reduce(qtam_plan *p, int batch, int plane, cudaStream_t st) {
  return p->esz == 4 ? inv_reduce_t<float>(p, batch, plane, st) : inv_reduce_t<double>(p, batch, plane, st);
}

template <typename T>
static qtam_status c2r_t(qtam_plan *p, int batch, void *d_x_out, cudaStream_t st) {
  const int Nc = (int)(p->hp.N / 2);
  C2<T> *spec = static_cast<C2<T> *>(p->d_spec);
  dim3 g((Nc / 2 + 1 + 255) / 256, batch);
  {
    LaunchScope ls(p, st, K_C2R_PRE, 0.0, 2.0 * sizeof(C2<T>) * (double)batch * (double)Nc);
    k_c2r_pre<T><<<g, 256, 0, st>>>(spec, p->xstride, Nc, static_cast<const C2<T> *>(p->d_twN));
  }
  QTAM_LAUNCH_CHECK();
  return cfft_any<T>(p, spec, p->xstride, static_cast<C2<T> *>(d_x_out), Nc, static_cast<C2<T> *>(p->d_ws),
                     p->hp.N, Nc, batch, +1, (T)1, st, 0.0, (double)batch * sizeof(T) * (double)p->hp.N);
}

// the complex FFT alone, for a spectrum buffer that already holds the pre-processed Z (k_combine_runs)
qtam_status generic_c2c_out(qtam_plan *p, int batch, void *d_x_out, cudaStream_t st) {
  if (!p->n_pow2 && fast_r3_ok(p)) return fast_r3(p, false, nullptr, d_x_out, batch, st);
  if (long_residues_ok(p)) return long_inverse_residues(p, d_x_out, batch, st);
  const int Nc = (int)(p->hp.N / 2);
  return cfft_any<float>(p, static_cast<const float2 *>(p->d_spec), p->xstride, static_cast<float2 *>(d_x_out), Nc,
                         static_cast<float2 *>(p->d_ws), p->hp.N, Nc, batch, +1, 1.f, st, 0.0,
                         (double)batch * 4.0 * (double)p->hp.N);
}

qtam_status generic_c2r(qtam_plan *p, int batch, void *d_x_out, cudaStream_t st) {
  return p->esz == 4 ? c2r_t<float>(p, batch, d_x_out, st) : c2r_t<double>(p, batch, d_x_out, st);
}

template <typename T>
static qtam_status dense_t(qtam_plan *p, int batch, int row_begin, int row_end, void *d_out, cudaStream_t st) {
  const int N = (int)p->hp.N;
  const int nr = row_end - row_begin;
  C2<T> *ws = static_cast<C2<T> *>(p->d_ws);
  C2<T> *out = static_cast<C2<T> *>(d_out);
  for (int k = row_begin; k < row_end; ++k) {
    dim3 g((N + 255) / 256, batch);
    {
      LaunchScope ls(p, st, K_DENSE_PLACE, sizeof(C2<T>) * (double)batch * (double)N);
      k_dense_place<T><<<g, 256, 0, st>>>(p->d_rows, k, static_cast<const C2<T> *>(p->d_spec), p->xstride,
                                          (int)p->hp.nb, static_cast<const T *>(p->d_win), ws, N,
                                          (T)(p->hp.opt.epsilon * p->hp.rows[(size_t)k].norm));
    }
    QTAM_LAUNCH_CHECK();
    qtam_status s = cfft_any<T>(p, ws, N, out + (long long)(k - row_begin) * N, (long long)nr * N, ws, N,
                                N, batch, +1, (T)1, st);
    if (s != QTAM_OK) return s;
  }
  return QTAM_OK;
}

template <typename T>
static qtam_status dense_invert_t(qtam_plan *p, const void *d_tile, int batch, int row, void *d_x_out, cudaStream_t st) {
  const int N = (int)p->hp.N;
  // the forward transform of the tile needs no scratch only while it fits one CTA (this is a check path
  // for small configurations, like qtam_dense)
  if (ilog2(N) > p->cap_log2) return QTAM_ERR_UNSUPPORTED;
  C2<T> *ws = static_cast<C2<T> *>(p->d_ws);
  qtam_status s = cfft_any<T>(p, static_cast<const C2<T> *>(d_tile), N, ws, N, ws, N, N, batch, -1, (T)1, st);
  if (s != QTAM_OK) return s;
  dim3 g((unsigned)((p->hp.nb + 255) / 256), batch);
  {
    LaunchScope ls(p, st, K_DENSE_PLACE, sizeof(C2<T>) * (double)batch * (double)p->hp.nb * 2.0);
    k_dense_divide<T><<<g, 256, 0, st>>>(p->d_rows, row, ws, N, static_cast<const T *>(p->d_win),
                                         (T)(p->hp.opt.epsilon * p->hp.rows[(size_t)row].norm), (int)p->hp.nb,
                                         static_cast<C2<T> *>(p->d_spec), p->xstride);
  }
  QTAM_LAUNCH_CHECK();
  return c2r_t<T>(p, batch, d_x_out, st);
}

qtam_status generic_dense_invert(qtam_plan *p, const void *d_tile, int batch, int row, void *d_x_out, cudaStream_t st) {
  return p->esz == 4 ? dense_invert_t<float>(p, d_tile, batch, row, d_x_out, st)
                     : dense_invert_t<double>(p, d_tile, batch, row, d_x_out, st);
}

qtam_status generic_dense(qtam_plan *p, int batch, int row_begin, int row_end, void *d_out, cudaStream_t st) {
  return p->esz == 4 ? dense_t<float>(p, batch, row_begin, row_end, d_out, st)
                     : dense_t<double>(p, batch, row_begin, row_end, d_out, st);
}

template <typename T>
static qtam_status threshold_t(qtam_plan *p, void *d_coef, int batch, double kappa, int min_log2M, cudaStream_t st) {
  const int cache_pts = kThrCachePts;
  const size_t smem = sizeof(T) * (size_t)cache_pts;
  dim3 g((unsigned)p->hp.rows.size(), batch);
  {
    LaunchScope ls(p, st, K_THRESHOLD, 0.0, 2.0 * sizeof(C2<T>) * (double)batch * (double)p->hp.ctot);
    k_threshold<T><<<g, 256, smem, st>>>(p->d_rows, static_cast<C2<T> *>(d_coef), p->hp.ctot, (T)kappa, cache_pts, min_log2M);
  }
  QTAM_LAUNCH_CHECK();
  return QTAM_OK;
}

qtam_status prepare_generic(qtam_plan *p) {
  return (p->esz == 4 ? prepare_t<float>(p) : prepare_t<double>(p)) ? QTAM_OK : QTAM_ERR_CUDA;
}

qtam_status generic_threshold(qtam_plan *p, void *d_coef, int batch, double kappa, int min_log2M, cudaStream_t st) {
  return p->esz == 4 ? threshold_t<float>(p, d_coef, batch, kappa, min_log2M, st)
                     : threshold_t<double>(p, d_coef, batch, kappa, min_log2M, st);
}

}  // namespace qtam
