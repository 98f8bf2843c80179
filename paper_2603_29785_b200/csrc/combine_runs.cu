// combine_runs.cu -- a6 (last step) + a7 + the head of a8 for every float plan that is not on the tiled path:
// the spectrum as the sum of RUNS.  The row kernels leave the inverse's contributions as contiguous pieces of
// spectrum -- the tiles' partial sums (inv_tiled.cu), the groups' partial sums (rows_cta.cu, rows_cluster.cu) and
// the band slots of the few rows that still write the band workspace (rows shorter than 32 points).  One pass
// adds, for every bin, the runs that cover it in a fixed order (Eq. 11's sum over k, :135), multiplies by 1/P on
// the cover set (C41 :558, C50 :602, R9) and applies the Hermitian pre-processing of the long C2R (row a8):
//   Z[f] = E + i O,  E = (Xhat[f] + conj Xhat[Nc-f])/2,  O = (Xhat[f] - conj Xhat[Nc-f])/2 e^{+2 pi i f/N},
// scaled 1/Nc, written to the spectrum buffer, from which the half-length complex FFT produces x.
// A CTA takes a block of bins f and the mirrored block Nc - f; the runs that touch either are listed per block.
#include <algorithm>
#include <vector>

#include "cplx.cuh"
#include "device_plan.hpp"
#include "fftreg.cuh"

namespace qtam {

constexpr int kRunBlock = 256;

static int ilog2(long long v) { int l = 0; while ((1LL << l) < v) ++l; return l; }

constexpr int kRunChunk = 128;     // run records staged in shared memory at a time

__global__ void __launch_bounds__(kRunBlock)
k_combine_runs(const int4 *__restrict__ runs, const int *__restrict__ ptr, const int *__restrict__ idx,
               const float2 *__restrict__ part, long long part_stride, const float2 *__restrict__ band,
               long long sumL, const float *__restrict__ invP, int Nc, int plane, const float2 *__restrict__ tw,
               int tw_shift, float2 *__restrict__ spec, long long xstride, float2 *__restrict__ rt,
               long long rt_stride, int rt_len, int rt_pad) {
  __shared__ int4 s_runs[kRunChunk];
  // hand-over buffers between the bin-ordered and the residue-ordered thread maps.  The residue-ordered index
  // tq = 64 a + b puts the four values of a (lanes 4 b .. 4 b + 3) on one bank; xi() shifts every block of 64 by four
  // elements, which spreads a half-warp's 8-byte accesses (and the flags' bytes) over distinct banks in both maps
  __shared__ float2 s_xch[2][kRunBlock + 16];
  __shared__ unsigned char s_ok[2][kRunBlock + 16];
  auto xi = [](int i) { return i + 4 * (i >> 6); };
  const int b = blockIdx.x, seg = blockIdx.y;
  const int f = b * kRunBlock + threadIdx.x;
  const int g = Nc - f;
  // Runs sorted by residue (src 2, rows_split.cu) hold the block's 256 bins as 64 residues x 4 consecutive
  // elements: they are read with a second thread -> bin map that follows that order (tf for the block's bins, tg
  // for the mirrored ones) and handed to the bins' own threads through shared memory at the end.
  const int tq = 64 * (threadIdx.x & 3) + (threadIdx.x >> 2);
  const int tf = b * kRunBlock + tq;
  const int tg = Nc - b * kRunBlock - (kRunBlock - 1) + tq;
  float2 At = make_float2(0.f, 0.f), Bt = make_float2(0.f, 0.f);
  const float2 *ps = part + (size_t)seg * part_stride;
  const float2 *bs = band + (size_t)seg * sumL;
  // lists 2b (runs that touch the block's bins f) and 2b + 1 (its mirror bins g) are adjacent in idx
  const int e0 = ptr[2 * b], e1 = ptr[2 * b + 1], e2 = ptr[2 * b + 2];
  float2 A = make_float2(0.f, 0.f), B = make_float2(0.f, 0.f);
  for (int c0 = e0; c0 < e2; c0 += kRunChunk) {
    const int n = min(kRunChunk, e2 - c0);
    __syncthreads();
    for (int i = threadIdx.x; i < n; i += kRunBlock) s_runs[i] = __ldg(runs + __ldg(idx + c0 + i));
    __syncthreads();
    // the runs are added in list order (a fixed order); the loads of four runs are in flight together
    for (int i0 = 0; i0 < n; i0 += 4) {
      float2 v[4]; bool forA[4], byres[4];
#pragma unroll
      for (int k = 0; k < 4; ++k) {
        v[k] = make_float2(0.f, 0.f);
        forA[k] = c0 + i0 + k < e1;
        byres[k] = false;
        if (i0 + k < n) {
          const int4 r = s_runs[i0 + k];           // lo, nb, off, src | (plane + 1) << 2
          const int rp = (r.w >> 2) - 1;
          const int src = r.w & 3;
          byres[k] = src == 2;
          const int x = byres[k] ? (forA[k] ? tf : tg) : (forA[k] ? f : g);
          const unsigned d = (unsigned)(x - r.x);
          if (d < (unsigned)r.y && !(rp >= 0 && plane >= 0 && rp != plane)) {
            if (byres[k]) {
              const int len64 = ((r.x + r.y - 1) >> 6) - (r.x >> 6) + 1;
              v[k] = __ldcs(ps + (size_t)r.z + (size_t)(x & 63) * len64 + ((x >> 6) - (r.x >> 6)));
            } else {
              v[k] = __ldcs((src == 1 ? ps : bs) + (size_t)r.z + d);
            }
          }
        }
      }
#pragma unroll
      for (int k = 0; k < 4; ++k) {
        if (byres[k]) { if (forA[k]) At = padd(At, v[k]); else Bt = padd(Bt, v[k]); }
        else { if (forA[k]) A = padd(A, v[k]); else B = padd(B, v[k]); }
      }
    }
  }
  s_xch[0][xi(tq)] = At;
  s_xch[1][xi(kRunBlock - 1 - tq)] = Bt;
  __syncthreads();
  A = padd(A, s_xch[0][xi(threadIdx.x)]);
  B = padd(B, s_xch[1][xi(threadIdx.x)]);
  const bool okf = f <= Nc / 2, okg = okf && g != f && f != 0;
  float2 vf = make_float2(0.f, 0.f), vg = vf;
  if (okf) {
    A = pscale(A, __ldg(invP + f));
    B = pscale(B, __ldg(invP + g));
    if (f == 0) { A.y = 0.f; B.y = 0.f; }
    const float h = 0.5f / (float)Nc;
    const float2 E = make_float2(h * (A.x + B.x), h * (A.y - B.y));
    const float2 D = make_float2(h * (A.x - B.x), h * (A.y + B.y));
    const float2 w = __ldg(tw + ((size_t)f << tw_shift));      // e^{+2 pi i f/N}
    const float2 O = make_float2(D.x * w.x - D.y * w.y, D.x * w.y + D.y * w.x);
    vf = make_float2(E.x - O.y, E.y + O.x);                    // E + i O
    vg = make_float2(E.x + O.y, -E.y + O.x);                   // conj(E) + i conj(O)
  }
  if (rt == nullptr) {
    float2 *S = spec + (size_t)seg * xstride;
    if (okf) S[f] = vf;
    if (okg) S[g] = vg;
    return;
  }
  // the spectrum in residue order for the long inverse FFT of long_fft.cu (bin x at [x mod 64][pad + x div 64]):
  // handed to the threads of the residue-ordered map, which write 4 consecutive elements of a residue each
  __syncthreads();
  s_xch[0][xi(threadIdx.x)] = vf; s_ok[0][xi(threadIdx.x)] = okf;
  s_xch[1][xi(threadIdx.x)] = vg; s_ok[1][xi(threadIdx.x)] = okg;
  __syncthreads();
  float2 *R = rt + (size_t)seg * rt_stride + rt_pad;
  if (s_ok[0][xi(tq)]) R[(size_t)(tf & 63) * rt_len + (tf >> 6)] = s_xch[0][xi(tq)];
  if (s_ok[1][xi(kRunBlock - 1 - tq)]) R[(size_t)(tg & 63) * rt_len + (tg >> 6)] = s_xch[1][xi(kRunBlock - 1 - tq)];
}

// Run lists, the band-slot runs of the rows that no tile or group covers, and the partial-sum buffer (the tiles'
// and the groups' pieces have been laid out by build_inv_tiled / build_rows_cta / build_rows_cluster).
qtam_status build_runs(qtam_plan *p) {
  const HostPlan &hp = p->hp;
  p->use_runs = false;
  auto up = [&](void **dst, const void *src, size_t bytes) -> bool {
    *dst = nullptr;
    if (cudaMalloc(dst, bytes ? bytes : 16) != cudaSuccess) return false;
    p->device_bytes += bytes;
    return !src || bytes == 0 || cudaMemcpy(*dst, src, bytes, cudaMemcpyHostToDevice) == cudaSuccess;
  };
  if (!p->fast_rows) return QTAM_OK;
  if (p->part_stride >= (int64_t(1) << 31)) return QTAM_ERR_UNSUPPORTED;
  if (!up(&p->d_part, nullptr, sizeof(float2) * (size_t)p->max_batch * (size_t)std::max<int64_t>(p->part_stride, 1)))
    return QTAM_ERR_ALLOC;
  if (p->tiled_inv) return QTAM_OK;
  // band slots: rows shorter than 32 points (k_tiny_rows), and the rows of 32 .. 1024 points when no tiles exist
  for (const HostRow &h : hp.rows) {
    const int lm = ilog2(h.M);
    if (!(lm < 5 || (lm <= 10 && !p->tiles_ok))) continue;
    const int64_t lo = std::max<int64_t>(h.kc - h.dk, 0), hi = std::min<int64_t>(h.kc + h.dk, hp.nb - 1);
    if (hi < lo) continue;
    p->runs.push_back(HostRun{(int)lo, (int)(hi - lo + 1), h.goff + (lo - (h.kc - h.dk)), 0, h.plane});
  }
  const int Nc = (int)(hp.N / 2);
  const int nblk = (Nc / 2 + 1 + kRunBlock - 1) / kRunBlock;
  std::vector<int4> dev(p->runs.size());
  for (size_t i = 0; i < p->runs.size(); ++i) {
    const HostRun &r = p->runs[i];
    dev[i] = make_int4(r.lo, r.nb, (int)r.off, r.src | ((r.plane + 1) << 2));
  }
  std::vector<int> ptr(2 * (size_t)nblk + 1, 0), idx;
  for (int b = 0; b < nblk; ++b) {
    const int f0 = b * kRunBlock, f1 = std::min(f0 + kRunBlock - 1, Nc / 2);    // bins f of the block
    const int g0 = Nc - f1, g1 = Nc - f0;                                       // their mirrors
    ptr[2 * (size_t)b] = (int)idx.size();
    for (size_t i = 0; i < p->runs.size(); ++i)
      if (p->runs[i].nb > 0 && p->runs[i].lo <= f1 && p->runs[i].lo + p->runs[i].nb - 1 >= f0) idx.push_back((int)i);
    ptr[2 * (size_t)b + 1] = (int)idx.size();
    for (size_t i = 0; i < p->runs.size(); ++i)
      if (p->runs[i].nb > 0 && p->runs[i].lo <= g1 && p->runs[i].lo + p->runs[i].nb - 1 >= g0) idx.push_back((int)i);
  }
  ptr[2 * (size_t)nblk] = (int)idx.size();
  p->n_run_blocks = nblk;
  if (!up(reinterpret_cast<void **>(&p->d_runs), dev.data(), dev.size() * sizeof(int4))) return QTAM_ERR_ALLOC;
  if (!up(reinterpret_cast<void **>(&p->d_run_ptr), ptr.data(), ptr.size() * sizeof(int))) return QTAM_ERR_ALLOC;
  if (!up(reinterpret_cast<void **>(&p->d_run_idx), idx.data(), idx.size() * sizeof(int))) return QTAM_ERR_ALLOC;
  p->use_runs = true;
  return QTAM_OK;
}

qtam_status combine_runs(qtam_plan *p, int batch, int plane, cudaStream_t st) {
  const int Nc = (int)(p->hp.N / 2);
  const int tw_shift = 0;            // d_twN[f] = e^{2 pi i f/N}
  double run_bins = 0;
  for (const HostRun &r : p->runs) run_bins += (double)r.nb;
  dim3 g((unsigned)p->n_run_blocks, (unsigned)batch);
  const bool res = long_residues_ok(p);      // the long inverse FFT takes the spectrum in residue order
  {
    LaunchScope ls(p, st, K_COMBINE_RUNS, 0.0, (double)batch * 8.0 * (run_bins + (double)p->hp.nb));
    k_combine_runs<<<g, kRunBlock, 0, st>>>(
        p->d_runs, p->d_run_ptr, p->d_run_idx, static_cast<const float2 *>(p->d_part), p->part_stride,
        static_cast<const float2 *>(p->d_band), p->hp.sumL,
        static_cast<const float *>(p->d_invP) + (size_t)(plane + 1) * (size_t)p->hp.nb, Nc, plane,
        static_cast<const float2 *>(p->d_twN), tw_shift, static_cast<float2 *>(p->d_spec), p->xstride,
        res ? static_cast<float2 *>(p->d_sp_xt) : nullptr, 64LL * p->sp_xt_len, p->sp_xt_len, p->sp_xt_pad);
  }
  QTAM_LAUNCH_CHECK();
  return QTAM_OK;
}

}  // namespace qtam
