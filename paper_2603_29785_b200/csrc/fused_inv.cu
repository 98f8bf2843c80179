// fused_inv.cu -- the whole inverse (rows a5-a8) in ONE kernel, one CTA per segment, float.
//
//   for every round of NW*F rows of one length bucket (F = 32/G rows per warp):
//     phase A  each warp: coefficients of its rows -> registers -> forward FFT (rowfft.cuh, the
//              sqrt(N/M) of C49 folded into the twiddles) -> times the window -> the rows' bands,
//              in natural bin order, into the warp's own exchange buffer ("staging")
//     phase B  the CTA adds the staged bands into the segment's spectrum S[f] held in shared memory.
//              Thread t owns the bins f = t (mod NT): it alone ever touches S[f], and it takes the
//              rows in ascending order, so the sum over rows (Eq. 11 numerator) is a segmented
//              reduction over bins with a fixed order -- no atomics, no band workspace in HBM.
//   rows shorter than 32 points are done by direct summation in one last round;
//   then Xhat = S/P on the cover set (C50, R9), Hermitian pre-processing and the long inverse FFT in
//   the same shared memory (ctafft.cuh), written straight to x_out.
// HBM traffic = the coefficients in, the time series out: the compulsory bytes of SURVEY.md 8(d).
#include <cstdlib>

#include "ctafft.cuh"
#include "device_plan.hpp"
#include "rowfft.cuh"

namespace qtam {

#define QTAM_LAUNCH_CHECK()                                         \
  do {                                                              \
    if (cudaPeekAtLastError() != cudaSuccess) return QTAM_ERR_CUDA; \
  } while (0)

extern __shared__ __align__(16) unsigned char qtam_fused_smem[];

struct RoundRow { int lo, L, stage, active; };   // band start bin, length, offset into the staging area

template <int LOG2G>
__device__ __noinline__ void inv_stage(const FastBucket &B, const FastRow *__restrict__ frows, int base, int warp,
                                       int lane, float2 *ex, const float2 *__restrict__ tw1,
                                       const float2 *__restrict__ Yseg, const float *__restrict__ fwinp,
                                       int plane) {
  constexpr int G = 1 << LOG2G, F = 32 / G, M = 32 * G;
  const int t = lane & (G - 1), rw = lane >> LOG2G;
  const int r = base + warp * F + rw;
  const bool inb = r < B.nrows;
  const FastRow row = frows[B.row_base + (inb ? r : 0)];
  const bool valid = inb && (plane < 0 || row.plane == plane);
  if (__ballot_sync(0xffffffffu, valid) == 0u) return;
  const float2 *Y = Yseg + row.offset + t;
  float2 v[32];
#pragma unroll
  for (int j1 = 0; j1 < 32; ++j1) v[j1] = __ldcs(Y + G * j1);
  RowFFT<LOG2G, -1>::run(v, ex, tw1, lane);
  if (valid) {
    // windowed band values G_k[jj] = Bhat_k[jj] W_k[jj] in natural bin order jj = -dk..dk; the window
    // table is stored at the M-array index, the same index the FFT output has
    float2 *stage = ex + rw * M + row.dk;
    const float *W = fwinp + row.wpad + t;
#pragma unroll
    for (int i = 0; i < F; ++i)
#pragma unroll
      for (int n2 = 0; n2 < G; ++n2) {
        const int j = (t + G * i) + 32 * n2;
        const int jj = (G == 1) ? (j < 16 ? j : j - M) : (n2 < G / 2 ? j : j - M);
        if (jj <= row.dk && jj >= -row.dk) stage[jj] = pscale(v[i * G + n2], W[G * i + 32 * n2]);
      }
  }
}

template <int LOG2NC, int NW>
__global__ void __launch_bounds__(NW * 32, NW <= 8 ? 2 : 1)
k_inv_fused(FastParams P, const FastRow *__restrict__ frows, const FastRow *__restrict__ tiny, int n_tiny,
            const float2 *__restrict__ tw1g, const float *__restrict__ fwin, const float *__restrict__ fwinp,
            const float2 *__restrict__ coef,
            long long ctot, const float *__restrict__ invP, int nbins, int plane,
            const float2 *__restrict__ tw, int log2twn, float *__restrict__ x_out) {
  constexpr int NC = 1 << LOG2NC, NT = NW * 32;
  float2 *S = reinterpret_cast<float2 *>(qtam_fused_smem);
  float2 *exall = S + cta_fft_smem_elems<LOG2NC>();
  RoundRow *rr = reinterpret_cast<RoundRow *>(exall + NW * kExPerWarp);
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  float2 *ex = exall + warp * kExPerWarp;
  const float2 *Yseg = coef + (size_t)blockIdx.x * ctot;

  for (int f = tid; f <= NC; f += NT) S[f] = make_float2(0.f, 0.f);

  for (int q = 0; q < P.nbuckets; ++q) {
    const FastBucket B = P.b[q];
    const int Fr = 32 >> B.log2G, Mr = 32 << B.log2G;
    const int per_round = NW * Fr;
    for (int base = 0; base < B.nrows; base += per_round) {
      const int nr = min(per_round, B.nrows - base);
      __syncthreads();            // previous round's reduction is done with the staging area and rr[]
      for (int s = tid; s < nr; s += NT) {
        const FastRow row = frows[B.row_base + base + s];
        RoundRow o;
        o.lo = row.kc - row.dk; o.L = 2 * row.dk + 1;
        o.stage = (s >> (5 - B.log2G)) * kExPerWarp + (s & (Fr - 1)) * Mr;
        o.active = (plane < 0 || row.plane == plane) ? 1 : 0;
        rr[s] = o;
      }
      const float2 *tw1 = tw1g + B.tw_base;
      switch (B.log2G) {
        case 5: inv_stage<5>(B, frows, base, warp, lane, ex, tw1, Yseg, fwinp, plane); break;
        case 4: inv_stage<4>(B, frows, base, warp, lane, ex, tw1, Yseg, fwinp, plane); break;
        case 3: inv_stage<3>(B, frows, base, warp, lane, ex, tw1, Yseg, fwinp, plane); break;
        case 2: inv_stage<2>(B, frows, base, warp, lane, ex, tw1, Yseg, fwinp, plane); break;
        case 1: inv_stage<1>(B, frows, base, warp, lane, ex, tw1, Yseg, fwinp, plane); break;
        default: inv_stage<0>(B, frows, base, warp, lane, ex, tw1, Yseg, fwinp, plane); break;
      }
      __syncthreads();
      for (int s = 0; s < nr; ++s) {
        const RoundRow o = rr[s];
        if (!o.active) continue;
        const float2 *stage = exall + o.stage;
        for (int j = (tid - o.lo) & (NT - 1); j < o.L; j += NT) {
          const int f = o.lo + j;
          if ((unsigned)f < (unsigned)nbins) S[f] = padd(S[f], stage[j]);
        }
      }
    }
  }

  // rows shorter than 32 points: Bhat[jj] = sqrt(N/M) sum_n Y[n] e^{-2 pi i jj n/M} by direct summation
  if (n_tiny > 0) {
    __syncthreads();
    for (int s = tid; s < n_tiny; s += NT) {
      const FastRow row = tiny[s];
      RoundRow o;
      o.lo = row.kc - row.dk; o.L = 2 * row.dk + 1;
      o.stage = (s % NW) * kExPerWarp + (s / NW) * 16;
      o.active = (plane < 0 || row.plane == plane) ? 1 : 0;
      rr[s] = o;
    }
    for (int s = warp; s < n_tiny; s += NW) {
      const FastRow row = tiny[s];            // goff holds log2 M for tiny rows
      if (plane >= 0 && row.plane != plane) continue;
      const int lm = row.goff, M = 1 << lm;
      const int jj = lane - row.dk;
      if (lane <= 2 * row.dk) {
        const float2 *Y = Yseg + row.offset;
        float2 acc = make_float2(0.f, 0.f);
        for (int n = 0; n < M; ++n) {
          const int m = (jj * n) & (M - 1);
          float2 w = __ldg(tw + ((size_t)m << (log2twn - lm)));
          w.y = -w.y;
          acc = padd(acc, pcmul(Y[n], w));
        }
        const float amp = sqrtf((float)(2 * NC) / (float)M);
        ex[(s / NW) * 16 + lane] = pscale(acc, amp * fwin[row.woff + lane]);
      }
    }
    __syncthreads();
    for (int s = 0; s < n_tiny; ++s) {
      const RoundRow o = rr[s];
      if (!o.active) continue;
      const int j = (tid - o.lo) & (NT - 1);
      const int f = o.lo + j;
      if (j < o.L && (unsigned)f < (unsigned)nbins) S[f] = padd(S[f], exall[o.stage + j]);
    }
  }
  __syncthreads();

  // Xhat = S/P on the cover set (0 elsewhere), Z[f] = E + i O scaled 1/Nc (row a8), in place
  const float *ip = invP + (size_t)(plane + 1) * nbins;
  const float h = 0.5f / (float)NC;
  for (int f = tid; f <= NC / 2; f += NT) {
    const int g = NC - f;
    float2 A = pscale(S[f], ip[f]), Bv = pscale(S[g], ip[g]);
    if (f == 0) { A.y = 0.f; Bv.y = 0.f; }
    const float2 E = make_float2(h * (A.x + Bv.x), h * (A.y - Bv.y));
    const float2 D = make_float2(h * (A.x - Bv.x), h * (A.y + Bv.y));
    const float2 w = __ldg(tw + ((size_t)f << (log2twn - LOG2NC - 1)));
    const float2 O = make_float2(D.x * w.x - D.y * w.y, D.x * w.y + D.y * w.x);
    S[f] = make_float2(E.x - O.y, E.y + O.x);
    if (g != f && f != 0) S[g] = make_float2(E.x + O.y, -E.y + O.x);
  }
  __syncthreads();
  float2 *gout = reinterpret_cast<float2 *>(x_out) + (size_t)blockIdx.x * NC;
  cta_fft<LOG2NC, NT, +1, false, true>(S, nullptr, gout, tw, log2twn, 1.f);
}

// --------------------------------------------------------------------------------------------------
static int ilog2(long long v) { int l = 0; while ((1LL << l) < v) ++l; return l; }

template <int LOG2NC, int NW>
static qtam_status launch(qtam_plan *p, const void *d_coef, int batch, int plane, void *d_x_out, cudaStream_t st) {
  const size_t smem = sizeof(float2) * ((size_t)cta_fft_smem_elems<LOG2NC>() + (size_t)NW * kExPerWarp) +
                      sizeof(RoundRow) * (size_t)NW * 32;
  auto kern = k_inv_fused<LOG2NC, NW>;
  if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess)
    return QTAM_ERR_CUDA;
  {
    LaunchScope ls(p, st, K_INV_FUSED, (double)batch * (8.0 * (double)p->hp.ctot + 4.0 * (double)p->hp.N));
    kern<<<batch, NW * 32, smem, st>>>(
        p->fast, p->d_frows, p->d_tiny, p->n_tiny, static_cast<const float2 *>(p->d_ftw_inv),
        static_cast<const float *>(p->d_fwin), static_cast<const float *>(p->d_fwinp),
        static_cast<const float2 *>(d_coef), p->hp.ctot,
        static_cast<const float *>(p->d_invP), (int)p->hp.nb, plane, static_cast<const float2 *>(p->d_tw),
        ilog2(p->twn), static_cast<float *>(d_x_out));
  }
  QTAM_LAUNCH_CHECK();
  return QTAM_OK;
}

qtam_status fused_inverse(qtam_plan *p, const void *d_coef, int batch, int plane, void *d_x_out, cudaStream_t st) {
  switch (ilog2(p->hp.N) - 1) {
    case 11: return launch<11, 8>(p, d_coef, batch, plane, d_x_out, st);
    case 12: return launch<12, 8>(p, d_coef, batch, plane, d_x_out, st);
    case 13: return launch<13, 16>(p, d_coef, batch, plane, d_x_out, st);
    default: return QTAM_ERR_UNSUPPORTED;
  }
}

}  // namespace qtam
