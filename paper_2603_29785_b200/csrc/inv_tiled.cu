// inv_tiled.cu -- the float inverse (rows a5-a8) as two kernels with no band workspace and no atomics.
//
//   K1 k_inv_tiles   a5 + a6   persistent warps.  A work item = (segment, tile); a tile = a run of leaders
//                              (one per set of identical rows: their coefficient rows are added before the
//                              one transform)
//                              of one length bucket, consecutive in centre bin, whose bands fit a
//                              warp-private accumulator of kAccBins bins in shared memory.  The warp takes
//                              the tile's rows pass by pass (32/G rows of M = 32 G points per pass):
//                              coefficients -> registers -> forward FFT (rowfft.cuh, sqrt(N/M) of C49 in
//                              the twiddles) -> times the window -> added into the accumulator at bin
//                              kc + jj (Eq. 11 numerator).  One warp owns the accumulator and takes its
//                              rows in a fixed order, so the overlap-add is a segmented reduction with
//                              a fixed summation order: no atomics on data, no block barrier.  The
//                              finished partial sum (<= kAccBins bins) goes to the partial buffer.
//   K2 k_combine_c2r a6-a8     one CTA per segment: S[f] = sum of the tiles' partial sums in tile order
//                              (thread t owns the bins f = t mod NT), rows shorter than 32 points one per
//                              thread (tinyrow.cuh), Xhat = S/P on the cover set (C50, R9), Hermitian
//                              pre-processing and the long inverse FFT in shared memory (ctafft.cuh).
// HBM traffic = coefficients in, time series out; the partial sums (about ΣL/3 values per segment) are
// written and read back once and are meant to stay in L2.
#include <algorithm>
#include <vector>

#include "ctafft.cuh"
#include "device_plan.hpp"
#include "rowfft.cuh"
#include "tinyrow.cuh"

namespace qtam {

extern __shared__ __align__(16) unsigned char qtam_tiled_smem[];

static int ilog2(long long v) { int l = 0; while ((1LL << l) < v) ++l; return l; }
static bool prepare_tiled(qtam_plan *p);   // launch configurations of the two kernels (end of this file)
constexpr int kTileWarps = 11;   // warps per CTA of k_inv_tiles: 18 KB of shared memory each, one CTA per SM

// --------------------------------------------------------------------------------------------------
// host: tiles
// --------------------------------------------------------------------------------------------------
qtam_status build_inv_tiled(qtam_plan *p) {
  const HostPlan &hp = p->hp;
  const FastParams &F = p->fast;
  p->tiled_inv = false;
  p->tiles_ok = false;
  if (!p->fast_rows || F.nbuckets == 0) return QTAM_OK;
  // the whole inverse runs as tiles + k_combine_c2r when the long transform fits one CTA and no row is longer
  // than 1024 points; otherwise the tiles are one of the sources of k_combine_runs (combine_runs.cu)
  bool whole = p->fast_long && ilog2(hp.N) - 1 <= 14 && p->n_tiny <= 256;
  for (const HostRow &h : hp.rows) if (h.M > 1024) whole = false;
  std::vector<TileRow> trows;
  std::vector<TileItem> items;
  std::vector<int2> tmem;                 // (coefficient offset, plane) of every member
  std::vector<int> item_members;          // members per item, for the schedule
  // Passes per tile: long tiles mean few partial sums (less traffic for the combine pass), short tiles a finer
  // schedule.  12 at the batch sizes of configs 3 and 5; fewer when (tiles x max_batch) would not give every
  // resident warp several items (config 4: 16 segments).
  auto make_tiles = [&](int max_pass) -> bool {
    trows.clear(); items.clear(); tmem.clear(); item_members.clear();
    for (int q = 0; q < F.nbuckets; ++q) {
      const FastBucket &B = F.b[q];
      const int G = 1 << B.log2G, Fr = 32 / G;
      std::vector<FastRow> all(p->h_frows.begin() + B.row_base, p->h_frows.begin() + B.row_base + B.nrows);
      std::stable_sort(all.begin(), all.end(), [](const FastRow &a, const FastRow &b) {
        return a.kc != b.kc ? a.kc < b.kc : (a.dk != b.dk ? a.dk < b.dk : a.woff < b.woff);
      });
      // rows with the same centre bin and half-width (the clamped rows of different Q-planes) share their
      // window and their place in the spectrum: by linearity their coefficient rows are added before ONE
      // transform.  `rows` = one leader per such set; pad0 / pad1 = first member / number of members.
      std::vector<FastRow> rows;
      for (size_t i = 0; i < all.size(); ++i) {
        if (rows.empty() || rows.back().kc != all[i].kc || rows.back().dk != all[i].dk || rows.back().woff != all[i].woff) {
          rows.push_back(all[i]);
          rows.back().pad = (int)tmem.size();
          rows.back().goff = 0;            // member count
        }
        tmem.push_back(make_int2(all[i].offset, all[i].plane));
        rows.back().goff += 1;
      }
      size_t i = 0;
      while (i < rows.size()) {
        TileItem it{};
        it.row0 = (int)trows.size(); it.log2G = B.log2G; it.tw_base = B.tw_base;
        int lo = 1 << 30, hi = -(1 << 30), nmem = 0;
        while (i < rows.size() && it.npass < max_pass) {
          const size_t e = std::min(rows.size(), i + (size_t)Fr);
          int lo2 = lo, hi2 = hi;
          for (size_t r = i; r < e; ++r) {
            const int jlo = std::max(-rows[r].dk, -rows[r].kc);
            const int jhi = std::min(rows[r].dk, (int)hp.nb - 1 - rows[r].kc);
            if (jlo > jhi) continue;
            lo2 = std::min(lo2, rows[r].kc + jlo); hi2 = std::max(hi2, rows[r].kc + jhi);
          }
          if (hi2 >= lo2 && hi2 - lo2 + 1 > kAccBins) {
            if (it.npass == 0) return false;     // one pass does not fit: leave the plan to the other paths
            break;
          }
          lo = lo2; hi = hi2;
          for (size_t r = i; r < e; ++r) {
            TileRow t{};
            t.kc = rows[r].kc; t.offset = rows[r].offset; t.wpad = rows[r].wpad; t.plane = rows[r].plane;
            t.jlo = std::max(-rows[r].dk, -rows[r].kc);
            t.jhi = std::min(rows[r].dk, (int)hp.nb - 1 - rows[r].kc);
            t.pad0 = rows[r].pad; t.pad1 = rows[r].goff;
            nmem += rows[r].goff;
            trows.push_back(t);
          }
          it.npass += 1; it.nrows += (int)(e - i);
          i = e;
        }
        if (hi < lo) { lo = 0; hi = -1; }
        it.lo = lo; it.nb = hi - lo + 1;
        items.push_back(it);
        item_members.push_back(nmem);
      }
    }
    return true;
  };
  {
    static const int tries[] = {12, 8, 6, 4, 3, 2, 1};
    bool ok = false;
    for (int mp : tries) {
      ok = make_tiles(mp);
      if (!ok || (long long)items.size() * p->max_batch >= 4LL * p->num_sms * kTileWarps) break;
    }
    if (!ok) return QTAM_OK;
  }
  // heaviest items first: the dynamic schedule then ends on the short ones
  {
    // weight = transforms + member rows to load (both in units of one pass of the bucket)
    std::vector<size_t> order(items.size());
    for (size_t i = 0; i < order.size(); ++i) order[i] = i;
    auto weight = [&](size_t i) {
      const int Fr = 32 >> items[i].log2G;
      return items[i].npass * (10 + items[i].log2G) + 6 * ((item_members[i] + Fr - 1) / Fr);
    };
    std::stable_sort(order.begin(), order.end(), [&](size_t a, size_t b) { return weight(a) > weight(b); });
    std::vector<TileItem> sorted;
    for (size_t i : order) sorted.push_back(items[i]);
    items.swap(sorted);
  }
  int64_t off = p->part_stride;      // the tiles' partial sums open the per-segment partial-sum layout
  for (TileItem &it : items) {
    it.part_off = (int)off; off += (it.nb + 1) & ~1;                                // 16-byte aligned slots
    p->runs.push_back(HostRun{it.lo, it.nb, it.part_off, 1, -1});
  }
  p->part_stride = off;
  p->n_titems = (int)items.size();
  size_t *tot = &p->device_bytes;
  auto up = [&](void **dst, const void *src, size_t bytes) -> bool {
    *dst = nullptr;
    if (cudaMalloc(dst, bytes ? bytes : 16) != cudaSuccess) return false;
    *tot += bytes;
    return !src || cudaMemcpy(*dst, src, bytes, cudaMemcpyHostToDevice) == cudaSuccess;
  };
  if (!up(reinterpret_cast<void **>(&p->d_trows), trows.data(), trows.size() * sizeof(TileRow))) return QTAM_ERR_ALLOC;
  if (!up(reinterpret_cast<void **>(&p->d_titems), items.data(), items.size() * sizeof(TileItem))) return QTAM_ERR_ALLOC;
  if (!up(reinterpret_cast<void **>(&p->d_tmem), tmem.data(), tmem.size() * sizeof(int2))) return QTAM_ERR_ALLOC;
  if (!up(reinterpret_cast<void **>(&p->d_counter), nullptr, 256)) return QTAM_ERR_ALLOC;
  p->tiled_inv = whole;
  if (!prepare_tiled(p)) return QTAM_ERR_CUDA;
  p->tiles_ok = true;
  return QTAM_OK;
}

// --------------------------------------------------------------------------------------------------
// K1: tiles
// --------------------------------------------------------------------------------------------------
// One pass of a tile: F = 32/G rows of M = 32 G points.  acc[0] is bin it.lo.
template <int LOG2G>
__device__ __forceinline__ void tile_pass(const TileItem &it, const TileRow *__restrict__ trows, int pass, int lane,
                                          float2 *ex, const float2 *tw1, const float2 *__restrict__ Yseg,
                                          const float *__restrict__ fwinp, int plane, float2 *acc,
                                          const int2 *__restrict__ tmem) {
  constexpr int G = 1 << LOG2G, F = 32 / G, M = 32 * G;
  const int t = lane & (G - 1), rw = lane >> LOG2G;
  const int r = pass * F + rw;
  const bool inb = r < it.nrows;
  // lanes past the end of the tile recompute its last row and contribute nothing
  TileRow row = trows[it.row0 + (inb ? r : it.nrows - 1)];
  // members of the leader's set that take part (all of them, or those of the requested plane)
  int nmatch = 0;
  if (inb && row.jlo <= row.jhi) {
    if (plane < 0) nmatch = row.pad1;
    else for (int m = 0; m < row.pad1; ++m) nmatch += (__ldg(&tmem[row.pad0 + m].y) == plane) ? 1 : 0;
  }
  const bool active = nmatch > 0;
  if (__ballot_sync(0xffffffffu, active) == 0u) return;
  if (!active) { row.jlo = 1; row.jhi = 0; row.pad1 = 0; }
  float2 v[32];
#pragma unroll
  for (int j1 = 0; j1 < 32; ++j1) v[j1] = make_float2(0.f, 0.f);
  // sum of the members' coefficient rows (linearity of the transform; Eq. 11's sum over k)
#pragma unroll 1
  for (int m = 0; m < row.pad1; ++m) {
    const int2 mb = __ldg(tmem + row.pad0 + m);
    if (plane >= 0 && mb.y != plane) continue;
    const float2 *Y = Yseg + mb.x + t;
    float2 y[32];
#pragma unroll
    for (int j1 = 0; j1 < 32; ++j1) y[j1] = __ldcs(Y + G * j1);
#pragma unroll
    for (int j1 = 0; j1 < 32; ++j1) v[j1] = padd(v[j1], y[j1]);
  }
  RowFFT<LOG2G, -1>::run(v, ex, tw1, lane);
  // G_k[jj] = Bhat_k[jj] W_k[jj] (C49); the window table is stored at the M-array index of the FFT output
  const float *W = fwinp + row.wpad + t;
  const unsigned span = (unsigned)(row.jhi - row.jlo);
  if constexpr (G == 32) {
    // one row per warp: straight from the registers into the accumulator
    float2 *a = acc + (row.kc - it.lo);
#pragma unroll
    for (int n2 = 0; n2 < 32; ++n2) {
      const int j = t + 32 * n2;
      const int jj = n2 < 16 ? j : j - M;
      if (active && (unsigned)(jj - row.jlo) <= span) {
        const float w = __ldg(W + 32 * n2);
        a[jj] = pfma(v[n2], make_float2(w, w), a[jj]);
      }
    }
  } else {
    // several rows per warp: their bands overlap, so they are staged in natural order in the exchange
    // buffer and added one row at a time by the whole warp
    float2 *stage = ex + rw * M + M / 2;
#pragma unroll
    for (int i = 0; i < F; ++i)
#pragma unroll
      for (int n2 = 0; n2 < G; ++n2) {
        const int j = (t + G * i) + 32 * n2;
        const int jj = (G == 1) ? (j < 16 ? j : j - M) : (n2 < G / 2 ? j : j - M);
        if ((unsigned)(jj - row.jlo) <= span) stage[jj] = pscale(v[i * G + n2], __ldg(W + G * i + 32 * n2));
      }
    __syncwarp();
#pragma unroll 1
    for (int rr = 0; rr < F; ++rr) {
      const int kc = __shfl_sync(0xffffffffu, row.kc, rr * G);
      const int jlo = __shfl_sync(0xffffffffu, row.jlo, rr * G);
      const int jhi = __shfl_sync(0xffffffffu, row.jhi, rr * G);
      const float2 *sr = ex + rr * M + M / 2;
      float2 *a = acc + (kc - it.lo);
      for (int jj = jlo + lane; jj <= jhi; jj += 32) a[jj] = padd(a[jj], sr[jj]);
    }
    __syncwarp();
  }
}

template <int NW>
__global__ void __launch_bounds__(NW * 32, 1)
k_inv_tiles(const TileItem *__restrict__ items, int n_items, const TileRow *__restrict__ trows,
            const float2 *__restrict__ tw1g, int tw_total, const float *__restrict__ fwinp,
            const float2 *__restrict__ coef, long long ctot, int batch, int plane,
            float2 *__restrict__ part, long long part_stride, unsigned int *__restrict__ counter,
            const int2 *__restrict__ tmem) {
  float2 *tw1s = reinterpret_cast<float2 *>(qtam_tiled_smem);
  float2 *warp_base = tw1s + ((tw_total + 1) & ~1);
  for (int i = threadIdx.x; i < tw_total; i += NW * 32) tw1s[i] = tw1g[i];
  __syncthreads();
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  float2 *ex = warp_base + (size_t)warp * (kExPerWarp + kAccBins);
  float2 *acc = ex + kExPerWarp;
  const unsigned int total = (unsigned int)n_items * (unsigned int)batch;
  for (;;) {
    unsigned int id = 0;
    if (lane == 0) id = atomicAdd(counter, 1u);
    id = __shfl_sync(0xffffffffu, id, 0);
    if (id >= total) break;
    const unsigned int ii = id / (unsigned int)batch;
    const int seg = (int)(id - ii * (unsigned int)batch);
    TileItem it;
    {
      const int4 a = __ldg(reinterpret_cast<const int4 *>(items + ii));
      const int4 b = __ldg(reinterpret_cast<const int4 *>(items + ii) + 1);
      it.row0 = a.x; it.nrows = a.y; it.log2G = a.z; it.tw_base = a.w;
      it.lo = b.x; it.nb = b.y; it.part_off = b.z; it.npass = b.w;
    }
    const int nbe = (it.nb + 1) & ~1;
    for (int i = lane; i < nbe; i += 32) acc[i] = make_float2(0.f, 0.f);
    __syncwarp();
    const float2 *Yseg = coef + (size_t)seg * ctot;
    const float2 *tw1 = tw1s + it.tw_base;
#define QTAM_TILE_CASE(L)                                                                      \
  case L:                                                                                      \
    _Pragma("unroll 1") for (int pass = 0; pass < it.npass; ++pass)                            \
        tile_pass<L>(it, trows, pass, lane, ex, tw1, Yseg, fwinp, plane, acc, tmem);           \
    break;
    switch (it.log2G) {
      QTAM_TILE_CASE(5) QTAM_TILE_CASE(4) QTAM_TILE_CASE(3) QTAM_TILE_CASE(2) QTAM_TILE_CASE(1) QTAM_TILE_CASE(0)
      default: break;
    }
#undef QTAM_TILE_CASE
    __syncwarp();
    float4 *dst = reinterpret_cast<float4 *>(part + (size_t)seg * part_stride + it.part_off);
    const float4 *src = reinterpret_cast<const float4 *>(acc);
    for (int i = lane; i < nbe / 2; i += 32) dst[i] = src[i];
    __syncwarp();
  }
}

// --------------------------------------------------------------------------------------------------
// K2: combine + tiny rows + 1/P + long C2R
// --------------------------------------------------------------------------------------------------
template <int LOG2NC, int NT>
__global__ void __launch_bounds__(NT)
k_combine_c2r(const TileItem *__restrict__ items, int n_items, const float2 *__restrict__ part,
              long long part_stride, const FastRow *__restrict__ tiny, int n_tiny,
              const float *__restrict__ fwin, const float2 *__restrict__ coef, long long ctot,
              const float *__restrict__ invP, int nbins, int plane, const float2 *__restrict__ tw,
              int log2twn, const float2 *__restrict__ ptw, float *__restrict__ x_out) {
  typedef CtaFftRadix<LOG2NC, NT> PL;
  typedef CtaFftRadix<LOG2NC, CtaFftPlan<LOG2NC>::NT> PL0;
  static_assert(PL::R0 == PL0::R0 && PL::R1 == PL0::R1 && PL::R2 == PL0::R2, "pass tables are built for PL0");
  constexpr int NC = 1 << LOG2NC;
  float2 *S = reinterpret_cast<float2 *>(qtam_tiled_smem);
  float2 *tbuf = S + cta_fft_smem_elems<LOG2NC>();      // 32 band values per tiny row
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const float2 *Yseg = coef + (size_t)blockIdx.x * ctot;

  // rows shorter than 32 points: one thread per row, transform in registers (tinyrow.cuh); the windowed
  // band (at most 31 values) goes to tbuf[s][jj + dk], zero where the offset leaves the spectrum (R8)
  for (int s = tid; s < n_tiny; s += NT) {
    const FastRow row = tiny[s];              // goff holds log2 M for tiny rows
    float2 *tb = tbuf + s * 32;
#pragma unroll
    for (int j = 0; j < 32; ++j) tb[j] = make_float2(0.f, 0.f);
    if (plane < 0 || row.plane == plane) {
      const float amp = sqrtf((float)(2 * NC) / (float)(1 << row.goff));
      float2 *Y = const_cast<float2 *>(Yseg) + row.offset;
      switch (row.goff) {
        case 2: tiny_row<4, false>(row, nullptr, fwin, Y, tb + row.dk, nbins, amp); break;
        case 3: tiny_row<8, false>(row, nullptr, fwin, Y, tb + row.dk, nbins, amp); break;
        case 4: tiny_row<16, false>(row, nullptr, fwin, Y, tb + row.dk, nbins, amp); break;
        default: break;
      }
    }
  }

  // S[f] = sum over the tiles' partial sums in tile order.  Thread t owns the bins f = t (mod NT): for
  // every tile it adds the tile's values at its bins into S (shared memory), so each bin is updated by one
  // thread, in tile order (fixed summation order, no atomics), and every thread has the same amount of work.
  for (int f = tid; f <= NC; f += NT) S[f] = make_float2(0.f, 0.f);
  const float2 *pseg = part + (size_t)blockIdx.x * part_stride;
  constexpr int KMAX = (kAccBins + NT - 1) / NT;
#pragma unroll 4
  for (int i = 0; i < n_items; ++i) {
    const int4 b = __ldg(reinterpret_cast<const int4 *>(items + i) + 1);   // lo, nb, part_off, npass
    const int f0 = b.x + ((tid - b.x) & (NT - 1));
    const float2 *src = pseg + b.z - b.x;
    float2 pv[KMAX];
#pragma unroll
    for (int k = 0; k < KMAX; ++k) {
      const int f = f0 + k * NT;
      pv[k] = (f < b.x + b.y) ? __ldcg(src + f) : make_float2(0.f, 0.f);
    }
#pragma unroll
    for (int k = 0; k < KMAX; ++k) {
      const int f = f0 + k * NT;
      if (f < b.x + b.y) S[f] = padd(S[f], pv[k]);
    }
  }
  __syncthreads();
  for (int s = 0; s < n_tiny; ++s) {
    const FastRow row = tiny[s];
    if (plane >= 0 && row.plane != plane) continue;
    const int lo = row.kc - row.dk;
    const int j = (tid - lo) & (NT - 1);
    const int f = lo + j;
    if (j <= 2 * row.dk && (unsigned)f < (unsigned)nbins) S[f] = padd(S[f], tbuf[s * 32 + j]);
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
  cta_fft<LOG2NC, NT, +1, false, true>(S, nullptr, gout, ptw, 1.f);
}

// --------------------------------------------------------------------------------------------------
// host side
// --------------------------------------------------------------------------------------------------
template <int NW>
static qtam_status tiles_launch(qtam_plan *p, const void *d_coef, int batch, int plane, cudaStream_t st) {
  const int twt = p->fast.tw_total;
  if (!p->cfg_tiles.ready) return QTAM_ERR_CUDA;
  const size_t smem = p->cfg_tiles.smem;
  auto kern = k_inv_tiles<NW>;
  const long long total = (long long)p->n_titems * batch;
  long long grid = (long long)p->num_sms * p->cfg_tiles.occ;
  if (grid * NW > total) grid = (total + NW - 1) / NW;
  if (grid < 1) grid = 1;
  if (cudaMemsetAsync(p->d_counter, 0, sizeof(unsigned int), st) != cudaSuccess) return QTAM_ERR_CUDA;
  {
    LaunchScope ls(p, st, K_INV_TILES, (double)batch * 8.0 * p->fast.sum_M,
                   (double)batch * 8.0 * (p->fast.sum_M + (double)p->part_stride));
    kern<<<(int)grid, NW * 32, smem, st>>>(
        p->d_titems, p->n_titems, p->d_trows, static_cast<const float2 *>(p->d_ftw_inv), twt,
        static_cast<const float *>(p->d_fwinp), static_cast<const float2 *>(d_coef), p->hp.ctot, batch, plane,
        static_cast<float2 *>(p->d_part), p->part_stride, p->d_counter, p->d_tmem);
  }
  QTAM_LAUNCH_CHECK();
  return QTAM_OK;
}

template <int LOG2NC, int NT>
static qtam_status combine_launch(qtam_plan *p, const void *d_coef, int batch, int plane, void *d_x_out,
                                  cudaStream_t st) {
  if (!p->cfg_combine.ready) return QTAM_ERR_CUDA;
  const size_t smem = p->cfg_combine.smem;
  auto kern = k_combine_c2r<LOG2NC, NT>;
  {
    LaunchScope ls(p, st, K_COMBINE_C2R, (double)batch * (4.0 * (double)p->hp.N + 8.0 * p->tiny_sumM),
                   (double)batch * (8.0 * ((double)p->part_stride + p->tiny_sumM) + 4.0 * (double)p->hp.N));
    kern<<<batch, NT, smem, st>>>(
        p->d_titems, p->n_titems, static_cast<const float2 *>(p->d_part), p->part_stride, p->d_tiny, p->n_tiny,
        static_cast<const float *>(p->d_fwin), static_cast<const float2 *>(d_coef), p->hp.ctot,
        static_cast<const float *>(p->d_invP), (int)p->hp.nb, plane, static_cast<const float2 *>(p->d_tw),
        ilog2(p->twn), static_cast<const float2 *>(p->d_ptw), static_cast<float *>(d_x_out));
  }
  QTAM_LAUNCH_CHECK();
  return QTAM_OK;
}

template <int LOG2NC, int NT> static bool prepare_combine(qtam_plan *p) {
  const size_t smem = sizeof(float2) * ((size_t)cta_fft_smem_elems<LOG2NC>() + 32 * (size_t)p->n_tiny);
  return kernel_prepare(p->cfg_combine, k_combine_c2r<LOG2NC, NT>, NT, smem);
}

static bool prepare_tiled(qtam_plan *p) {
  const size_t smem = sizeof(float2) * ((size_t)((p->fast.tw_total + 1) & ~1) + (size_t)kTileWarps * (kExPerWarp + kAccBins));
  if (!kernel_prepare(p->cfg_tiles, k_inv_tiles<kTileWarps>, kTileWarps * 32, smem)) return false;
  if (!p->tiled_inv) return true;
  switch (ilog2(p->hp.N) - 1) {
    case 11: return prepare_combine<11, 256>(p);
    case 12: return prepare_combine<12, 256>(p);
    case 13: return prepare_combine<13, 256>(p);
    case 14: return prepare_combine<14, 512>(p);
    default: return false;
  }
}

// the tiles alone: partial sums for k_combine_runs
qtam_status tiles_only(qtam_plan *p, const void *d_coef, int batch, int plane, cudaStream_t st) {
  return tiles_launch<kTileWarps>(p, d_coef, batch, plane, st);
}

qtam_status tiled_inverse(qtam_plan *p, const void *d_coef, int batch, int plane, void *d_x_out, cudaStream_t st) {
  const qtam_status s = tiles_launch<kTileWarps>(p, d_coef, batch, plane, st);
  if (s != QTAM_OK) return s;
  switch (ilog2(p->hp.N) - 1) {
    case 11: return combine_launch<11, 256>(p, d_coef, batch, plane, d_x_out, st);
    case 12: return combine_launch<12, 256>(p, d_coef, batch, plane, d_x_out, st);
    case 13: return combine_launch<13, 256>(p, d_coef, batch, plane, d_x_out, st);
    case 14: return combine_launch<14, 512>(p, d_coef, batch, plane, d_x_out, st);
    default: return QTAM_ERR_UNSUPPORTED;
  }
}

}  // namespace qtam
