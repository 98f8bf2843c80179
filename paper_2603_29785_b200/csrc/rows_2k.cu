// rows_2k.cu -- forward rows of 2048 points (float), one WARP per (segment, row): the largest bucket of plans like
// BASELINE config 2 (8 s segments: 78 of 144 rows), which the one-CTA-per-row kernel of rows_cta.cu served at 41 %
// of the HBM roofline on its coefficients.
//
// M = 2 * 1024, decimation in time:  Y[n] = sum_j B[j] e^{+2 pi i j n / M}  (C47 :589)  with  j = q + 2 jc:
//   Z_q[nc] = sum_jc B[q + 2 jc] w_1024^{jc nc}            two 1024-point transforms in the warp's registers
//                                                           (rowfft.cuh: 32 values per lane, private exchange buffer)
//   Y[nc] = Z_0[nc] + w_M^{nc} Z_1[nc],  Y[nc + 1024] = Z_0[nc] - w_M^{nc} Z_1[nc]
// Z_0 waits in a second private buffer (8 KB) while Z_1 is computed; no block barrier, nothing but the spectrum is
// read and nothing but the coefficients written.  B[j] = X[kc + jj] W_k[jj] (N M)^{-1/2} at j = jj mod M (A9 :323,
// R6), zero off the support and off the one-sided spectrum (R8); identical rows are transformed once and stored to
// every member of the leader's set.
#include <algorithm>
#include <cmath>
#include <vector>

#include "device_plan.hpp"
#include "rowfft.cuh"

namespace qtam {

extern __shared__ __align__(16) unsigned char qtam_2k_smem[];

constexpr int k2kWarps = 12;                       // one CTA per SM: 12 x (8.25 + 8) KB + 16 KB of tables
constexpr int k2kPerWarp = kExPerWarp + 1024;      // exchange buffer + the stash for Z_0 (float2 elements)

__global__ void __launch_bounds__(k2kWarps * 32, 1)
k_rows_2k(const ClLeader *__restrict__ lead, const int2 *__restrict__ mem, int nlead, const float *__restrict__ win,
          const float2 *__restrict__ spec, long long xstride, int nbins, float2 *__restrict__ coef, long long ctot,
          const float2 *__restrict__ tw1g, const float2 *__restrict__ tw2g, int batch) {
  constexpr int M = 2048;
  float2 *tw1 = reinterpret_cast<float2 *>(qtam_2k_smem);          // [n1][t]: w_1024^{t n1} (N M)^-1/2
  float2 *tw2 = tw1 + 1024;                                        // w_M^{nc}, nc < 1024
  for (int i = threadIdx.x; i < 1024; i += k2kWarps * 32) { tw1[i] = tw1g[i]; tw2[i] = tw2g[i]; }
  __syncthreads();
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  float2 *ex = tw2 + 1024 + (size_t)warp * k2kPerWarp;
  float2 *stash = ex + kExPerWarp;
  const long long total = (long long)nlead * batch;
  const long long nwarps = (long long)gridDim.x * k2kWarps;
  for (long long item = (long long)blockIdx.x * k2kWarps + warp; item < total; item += nwarps) {
    const int seg = (int)(item / nlead);
    const ClLeader L = lead[item - (long long)seg * nlead];
    const float2 *X = spec + (size_t)seg * xstride + L.kc;
    const float *W = win + L.woff + L.dk;
    const int hi = min(L.dk, nbins - 1 - L.kc), lo = max(-L.dk, -L.kc);     // offsets jj kept (R8 clip)
    float2 v[32];
#pragma unroll 1
    for (int q = 0; q < 2; ++q) {
      // element jc = lane + 32 j1 of sub-transform q: j = q + 2 jc, jj = j (j < M/2) or j - M
#pragma unroll
      for (int j1 = 0; j1 < 32; ++j1) {
        const int j = q + 2 * (lane + 32 * j1);
        const int jj = j1 < 16 ? j : j - M;
        v[j1] = make_float2(0.f, 0.f);
        if (jj >= lo && jj <= hi) {
          const float2 x = __ldg(X + jj);
          const float w = __ldg(W + jj);
          v[j1] = make_float2(x.x * w, x.y * w);
        }
      }
      RowFFT<5, +1>::run(v, ex, tw1, lane);                          // v[n2] = Z_q[lane + 32 n2] (scaled)
      if (q == 0) {
#pragma unroll
        for (int n2 = 0; n2 < 32; ++n2) stash[32 * n2 + lane] = v[n2];
      }
    }
    float2 y0[32];
#pragma unroll
    for (int n2 = 0; n2 < 32; ++n2) {
      const float2 a = pcmul(v[n2], tw2[32 * n2 + lane]);
      const float2 z0 = stash[32 * n2 + lane];
      y0[n2] = padd(z0, a);
      v[n2] = psub(z0, a);
    }
    __syncwarp();
    float2 *Yseg = coef + (size_t)seg * ctot + lane;
    for (int m = 0; m < L.nmem; ++m) {
      float2 *Y = Yseg + __ldg(&mem[L.mem0 + m].x);
#pragma unroll
      for (int n2 = 0; n2 < 32; ++n2) __stcs(Y + 32 * n2, y0[n2]);
#pragma unroll
      for (int n2 = 0; n2 < 32; ++n2) __stcs(Y + 1024 + 32 * n2, v[n2]);
    }
  }
}

qtam_status build_rows_2k(qtam_plan *p) {
  p->rows2k_ok = false;
  if (!p->cta_rows || p->n_cta_rows[0] == 0) return QTAM_OK;        // class 0 of rows_cta.cu = 2^11 points
  const long double tau = 6.283185307179586476925286766559005768L;
  const double scale = 1.0 / std::sqrt((double)p->hp.N * 2048.0);
  std::vector<float> t;
  for (int n1 = 0; n1 < 32; ++n1)
    for (int tt = 0; tt < 32; ++tt) {
      const long double a = tau * (long double)((tt * n1) % 1024) / 1024.0L;
      t.push_back((float)(cosl(a) * scale)); t.push_back((float)(sinl(a) * scale));
    }
  for (int nc = 0; nc < 1024; ++nc) {
    const long double a = tau * (long double)nc / 2048.0L;
    t.push_back((float)cosl(a)); t.push_back((float)sinl(a));
  }
  if (cudaMalloc(&p->d_tw_2k, t.size() * sizeof(float)) != cudaSuccess) return QTAM_ERR_ALLOC;
  p->device_bytes += t.size() * sizeof(float);
  if (cudaMemcpy(p->d_tw_2k, t.data(), t.size() * sizeof(float), cudaMemcpyHostToDevice) != cudaSuccess)
    return QTAM_ERR_CUDA;
  const size_t smem = sizeof(float2) * (size_t)(2048 + k2kWarps * k2kPerWarp);
  if (!kernel_prepare(p->cfg_rows_2k, k_rows_2k, k2kWarps * 32, smem)) return QTAM_ERR_CUDA;
  p->rows2k_ok = true;
  return QTAM_OK;
}

qtam_status rows_2k_forward(qtam_plan *p, int batch, void *d_coef, cudaStream_t st) {
  const KernelCfg &cfg = p->cfg_rows_2k;
  if (!cfg.ready) return QTAM_ERR_CUDA;
  const long long total = (long long)p->n_cta_rows[0] * batch;
  const long long grid = std::min<long long>((total + k2kWarps - 1) / k2kWarps, (long long)p->num_sms * cfg.occ);
  const double bytes = (double)batch * 8.0 * p->cta_sumM[0];        // compulsory: the coefficients
  const float2 *tw = static_cast<const float2 *>(p->d_tw_2k);
  {
    LaunchScope ls(p, st, K_ROWS_CTA_FWD, bytes, bytes + (double)batch * 8.0 * p->cta_sumL[0]);
    k_rows_2k<<<(unsigned)grid, k2kWarps * 32, cfg.smem, st>>>(
        p->d_cta_lead[0], p->d_cta_mem[0], p->n_cta_rows[0], static_cast<const float *>(p->d_win),
        static_cast<const float2 *>(p->d_spec), p->xstride, (int)p->hp.nb, static_cast<float2 *>(d_coef), p->hp.ctot,
        tw, tw + 1024, batch);
  }
  QTAM_LAUNCH_CHECK();
  return QTAM_OK;
}

}  // namespace qtam
