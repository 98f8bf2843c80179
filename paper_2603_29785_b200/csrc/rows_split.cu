// rows_split.cu -- rows of 2^15 and 2^16 points (float) as a DATAFLOW of warp-sized work items in one persistent
// kernel: the row's short FFT of M = F * P points (P = 1024, F = 32, 64) is split
// Cooley-Tukey-wise into
//   sub-transform items (row, residue q):        one P-point FFT in ONE WARP's registers (32 values per lane, two
//                                                radix-32 passes around the warp's private piece of shared memory)
//   radix-F items       (row, 32 or 16 values of nc):  the radix-F stage in registers (F = 64: a pair of lanes per nc)
// and the intermediate Z[q][nc] crosses between them through a small ring of row-sized slots that stays in L2
// (the items of a row run on different SMs).  Index split:
//   band side   j = q + F jc   (q < F, jc < P),     time side   n = nc + P m   (m < F, nc < P)
//   forward (a2 + a3, C47 :589)  Z[q][nc] = sum_jc B[q + F jc] w_P^{+jc nc},   B[j] = X[kc + jj] W_k[jj]
//                                Y[nc + P m] = (N M)^-1/2 sum_q w_M^{+q nc} Z[q][nc] w_F^{+q m}
//   inverse (a5 + a6, C49 :598)  u[q][nc] = sqrt(N/M) w_M^{-q nc} sum_m (sum over members Y[nc + P m]) w_F^{-q m}
//                                Bhat[q + F jc] = sum_nc u[q][nc] w_P^{-jc nc},  G = Bhat W_k  added into the partial
//                                spectrum of the leader's group by plain read-modify-write; the leaders of a group
//                                follow each other through a completion count, so every bin is updated in a fixed
//                                order: a segmented reduction without atomics on data and without a band workspace
//                                (Eq. 11 :135).  k_combine_runs adds the groups' partial sums.
// Why not one CTA (or one cluster) per row: a 2^16-point row is 512 KB, more than one SM holds, and the phases of a
// cluster that owns a row (gather, sub-transforms, exchange through distributed shared memory, stores) run one
// after the other on all of its SMs -- measured on cfg4: 38.6 k cycles per row and SM where HBM needs 14 k, the
// exchange alone at 11 B/cycle/SM.  Here 16 warps per SM work on items of many rows in different phases and never
// meet (no block barrier after the tables are loaded); the price is one round trip of the intermediate through
// L2 (the ring holds a few dozen rows).
//
// Scheduling.  Items are popped in a fixed order from one counter (atomicAdd): block t of the order holds the
// first-stage items of row t followed by the second-stage items of row t - LAG.  A second-stage item needs the
// first-stage items of its row (a completion count per row, release / acquire); a first-stage item needs the slot,
// i.e. the second-stage items of row t - NSLOTS; an inverse sub-transform item also needs the previous leader of
// its group.  Every wait is on items EARLIER in the order, and only running warps hold items, so the earliest
// unfinished item can always run: no deadlock, whatever the number of resident CTAs and whatever else runs on
// the GPU (NSLOTS > LAG is all it takes).  See the kernel for how lane 0 keeps the schedule's latencies (pop, counts,
// release) out of the warp's way.
#include <algorithm>
#include <cmath>
#include <cstdint>
#include <vector>

#include "device_plan.hpp"
#include "fftreg.cuh"

namespace qtam {

extern __shared__ __align__(16) unsigned char qtam_sp_smem[];

constexpr int kSpP = 1024, kSpNT = 128, kSpR = 32;
constexpr int kSpSmemElems = 4 * (kSpP + kSpP / 32);      // four interleaved sub-transforms, skew a + (a >> 5)
constexpr int kSpTwRows = 2 + kSpR / 4;                   // pass-2 table rows m = 1, 2, 3, 4, 8, .., 28
constexpr int kSpTwElems = kSpTwRows * 32;
constexpr int kSpMaxLead = 96, kSpMaxMem = 384;           // leaders / members of a class kept in shared memory
// The sub-transform of residue q reads the band at bins kc + q + F jc: every F-th bin.  k_spec_residues keeps a
// second copy of the spectrum sorted by residue, XT[f mod 64][f div 64] (64 = the largest F), in which those bins
// are consecutive (F = 64) or two interleaved runs (F = 32), so that a warp reads whole lines; kSpPad zero
// entries on both sides of every residue stand for the bins outside 0 .. N/2 (R8) -- no bounds test anywhere.
// The windows of these rows are kept the same way, WT[q][jc] = W_k[q + F jc'] (zero off the support).
constexpr int kSpRes = 64, kSpPad = 520;

// position oi of the row order: leader, position of the previous leader of its group (-1: none), and the group's
// partial sum, sorted by residue: bin f at element pbase + (f mod 64) len64 + f div 64
struct SpOrder { int lead, prev, pbase, len64; };

struct SpArgs {
  const ClLeader *lead; const int2 *mem; int nlead, nmem;
  const SpOrder *order;
  const float *wt; const int *wt_off;      // windows by residue, first element per leader
  const float2 *xt; long long xt_stride; int xt_len;   // spectrum by residue: [segment][64][xt_len]
  int nbins;
  float2 *coef; long long ctot;
  float2 *part; long long part_stride;
  const float2 *tw2;                       // pass-2 table of the sub-transforms
  const float2 *ftw;                       // radix-F twiddles: rows m = 1, 4, 32 of e^{2 pi i m nc / M}, nc < P
  float2 *scratch; int nslots, lag;        // ring of row slots, M elements each
  int *cnt1, *cnt2;                        // per row: first-stage / second-stage items finished
  unsigned int *queue;
  int batch, plane, nrows;
};

__device__ __forceinline__ int ld_acquire(const int *p) {
  int v;
  asm volatile("ld.acquire.gpu.global.s32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
  return v;
}
__device__ __forceinline__ float2 ldg_cg_f2(const float2 *p, bool ok) {
  float2 v;
  asm volatile("{\n .reg .pred q;\n setp.ne.s32 q, %3, 0;\n mov.f32 %0, 0f00000000;\n mov.f32 %1, 0f00000000;\n"
               " @q ld.global.cg.v2.f32 {%0, %1}, [%2];\n}" : "=f"(v.x), "=f"(v.y) : "l"(p), "r"((int)ok) : "memory");
  return v;
}

// pass-2 twiddles of one thread: w^{k r}, r = 4 a + b, from the table rows (see kSpTwRows) and one product each
template <int DIR>
__device__ __forceinline__ void sp_twiddle32(float2 (&v)[32], const float2 *tw2, int k) {
  float2 wb[4], wa[8];
#pragma unroll
  for (int b = 1; b < 4; ++b) { wb[b] = tw2[(b - 1) * 32 + k]; if (DIR < 0) wb[b].y = -wb[b].y; }
#pragma unroll
  for (int a = 1; a < 8; ++a) { wa[a] = tw2[(2 + a) * 32 + k]; if (DIR < 0) wa[a].y = -wa[a].y; }
#pragma unroll
  for (int r = 1; r < 32; ++r) {
    const int a = r >> 2, b = r & 3;
    const float2 w = a == 0 ? wb[b] : (b == 0 ? wa[a] : pcmul(wa[a], wb[b]));
    v[r] = pcmul(v[r], w);
  }
}

// the F twiddles w^{q}, q = 4 a + b, times w0, applied in place: w1 = w_M^{dir nc}, w4 = w_M^{dir 4 nc}
template <int F> __device__ __forceinline__ void sp_twiddleF(float2 (&v)[F], float2 w0, float2 w1, float2 w4) {
  float2 wb[4];
  wb[0] = w0; wb[1] = pcmul(w0, w1); wb[2] = pcmul(wb[1], w1); wb[3] = pcmul(wb[2], w1);
#pragma unroll
  for (int b = 0; b < 4; ++b) v[b] = pcmul(v[b], wb[b]);
  float2 wa = w4;
#pragma unroll
  for (int a = 1; a < F / 4; ++a) {
    if (a > 1) wa = pcmul(wa, w4);
#pragma unroll
    for (int b = 0; b < 4; ++b) v[4 * a + b] = pcmul(v[4 * a + b], pcmul(wa, wb[b]));
  }
}

// v[i] *= w_64^{DIR i}, i < N (compile-time twiddles)
template <int I, int N, int DIR> struct SpTw64 {
  static __device__ __forceinline__ void run(float2 (&v)[N]) {
    constexpr float c = cos64(I);
    constexpr float sn = DIR > 0 ? sin64(I) : -sin64(I);
    if constexpr (I != 0) v[I] = pfma(v[I], make_float2(c, c), pmul(make_float2(-v[I].y, v[I].x), make_float2(sn, sn)));
    if constexpr (I + 1 < N) SpTw64<I + 1, N, DIR>::run(v);
  }
};

// Radix-2 step across a pair of lanes (l and l ^ 16; h says which of the two I am) around the 32-point transforms
// of a 64-point stage; the values cross through the warp's private shared memory (one store and one load per
// value: shuffles under a lane-dependent mask cost three instructions each).  DIF (forward: the lane holds
// t[32 h + i]): h = 0 keeps v + o, h = 1 keeps (o - v) w_64^{+i}, o being the partner's value.  DIT (inverse: the
// lane holds U_h[i]): h = 1 first multiplies its values by w_64^{-i}; then h = 0 keeps v + o, h = 1 keeps o - v.
template <int N, bool DIF>
__device__ __forceinline__ void sp_pair(float2 (&v)[N], bool h, float2 *sw) {
  const int lane = threadIdx.x & 31;
  if (!DIF && h) SpTw64<0, N, -1>::run(v);
  __syncwarp();
#pragma unroll
  for (int i = 0; i < N; ++i) sw[i * 32 + lane] = v[i];
  __syncwarp();
  const float2 *o = sw + (lane ^ 16);
  if (h) {
#pragma unroll
    for (int i = 0; i < N; ++i) v[i] = psub(o[i * 32], v[i]);
    if (DIF) SpTw64<0, N, +1>::run(v);
  } else {
#pragma unroll
    for (int i = 0; i < N; ++i) v[i] = padd(v[i], o[i * 32]);
  }
  __syncwarp();
}

// Work items are warp-sized: a sub-transform item is one residue q of one row (a P-point transform in the warp's
// registers and private shared memory), a radix-F item 32 values of nc (16 when a pair of lanes shares an nc).
// A warp pops kSpChunk consecutive items of one row and stage at a time.
constexpr int kSpChunk = 1;
template <int F> struct SpGeo {
  static constexpr int PAIR = F > 32 ? F / 32 : 1;          // lanes that share one nc in the radix-F stage (1, 2)
  static constexpr int FT = F / PAIR;                       // values per lane there
  static constexpr int NC_ITEM = 32 / PAIR;                 // values of nc per radix-F item
  static constexpr int NSUB = F;                            // sub-transform items per row
  static constexpr int NRAD = kSpP / NC_ITEM;               // radix-F items per row
  static constexpr int PER = (NSUB + NRAD) / kSpChunk;      // chunks per block of the item order
  static_assert(PAIR <= 2, "rows longer than 2^16 points need a wider pair split");
  static_assert(NSUB % kSpChunk == 0 && NRAD % kSpChunk == 0, "chunks must not straddle stages");
};

// shared state of a CTA: the class's tables (read only) and the warps' private pieces
struct SpShared {
  ClLeader lead[kSpMaxLead];
  int2 mem[kSpMaxMem];
  SpOrder order[kSpMaxLead];
  int wt[kSpMaxLead];
  int off[kSpNT / 32][kCtaMaxMembers];
};

// members of a leader's set that take part in the inverse (all of them, or those of the requested plane),
// compacted in order into the warp's list; returns how many
__device__ __forceinline__ int sp_members(const SpArgs &A, const SpShared &sh, const ClLeader &L, int *off) {
  const int lane = threadIdx.x & 31;
  const bool ok = lane < L.nmem && (A.plane < 0 || sh.mem[L.mem0 + lane].y == A.plane);
  const unsigned b = __ballot_sync(0xffffffffu, ok);
  __syncwarp();
  if (off && ok) off[__popc(b & ((1u << lane) - 1u))] = sh.mem[L.mem0 + lane].x;
  __syncwarp();
  return __popc(b);
}

// --------------------------------------------------------------------------------------------------
// forward items
// --------------------------------------------------------------------------------------------------
// One warp = one residue q: its P-point transform lives in the warp's registers (32 values per lane) and its
// private piece of shared memory; no block barrier.
template <int F, class Sched>
__device__ __forceinline__ void sp_fwd_sub(const SpArgs &A, const SpShared &sh, float2 *sw, const float2 *stw,
                                           int row, int q, const Sched &sc) {
  constexpr int P = kSpP, M = F * P, S = kSpRes / F;      // S interleaved runs of the residue-sorted spectrum
  const int lane = threadIdx.x & 31;
  const int seg = row / A.nlead, li = row - seg * A.nlead;
  const ClLeader &L = sh.lead[li];
  float2 v[32];
  {
    // B[q + F jc] = X[kc + q + F jc'] W_k[q + F jc'], jc = lane + 32 r, jc' = jc (r < 16) or jc - P (R6)
    const int e = lane % S;
    const int f0 = L.kc + q + F * e;                       // bin of jc' = e
    const int res = f0 & (kSpRes - 1), idx = (f0 >> 6) + kSpPad;   // floor semantics for negative bins
    const float2 *Xp = A.xt + (size_t)seg * A.xt_stride + (size_t)res * A.xt_len + idx + (lane - e) / S;
    const float *Wp = A.wt + sh.wt[li] + q * P + lane;
    float w[32];
#pragma unroll
    for (int r = 0; r < 32; ++r) {
      v[r] = __ldg(Xp + (32 / S) * r - (r >= 16 ? P / S : 0));
      w[r] = __ldg(Wp + 32 * r);
    }
#pragma unroll
    for (int r = 0; r < 32; ++r) v[r] = pscale(v[r], w[r]);        // (N M)^-1/2 rides on the radix-F twiddles
  }
  RegFFT<32, +1>::run(v);
#pragma unroll
  for (int r = 0; r < 32; ++r) sw[33 * lane + r] = v[r];                    // a' = 32 lane + r, skewed
  __syncwarp();
#pragma unroll
  for (int r = 0; r < 32; ++r) v[r] = sw[lane + 33 * r];                    // a = lane + 32 r, skewed
  __syncwarp();
  sp_twiddle32<+1>(v, stw, lane);
  RegFFT<32, +1>::run(v);
  float2 *Z = A.scratch + (size_t)(row % A.nslots) * M + (size_t)q * P;
  sc.wait0();                              // the slot's previous row has been read
  sc.mid();
#pragma unroll
  for (int r = 0; r < 32; ++r) __stcg(Z + lane + 32 * r, v[r]);             // nc = lane + 32 r
}

template <int F, class Sched>
__device__ __forceinline__ void sp_fwd_radix(const SpArgs &A, const SpShared &sh, float2 *sw, int row, int ncb,
                                             const Sched &sc) {
  typedef SpGeo<F> G;
  constexpr int P = kSpP, M = F * P, FT = G::FT;
  const int lane = threadIdx.x & 31;
  const int seg = row / A.nlead;
  const ClLeader &L = sh.lead[row - seg * A.nlead];
  // lanes l and l ^ 16 share their nc when the stage is split over a pair
  const int h = G::PAIR == 2 ? (lane >> 4) : 0;
  const int nc = ncb * G::NC_ITEM + (G::PAIR == 2 ? (lane & 15) : lane);
  const float2 *Z = A.scratch + (size_t)(row % A.nslots) * M;
  const float2 w1 = __ldg(A.ftw + nc), w4 = __ldg(A.ftw + P + nc);
  float2 w0 = make_float2(1.f, 0.f);
  if (G::PAIR == 2 && h) w0 = __ldg(A.ftw + 2 * P + nc);
  sc.wait0();                              // the row's sub-transforms are in the slot
  float2 v[FT];
#pragma unroll
  for (int i = 0; i < FT; ++i) v[i] = __ldcg(Z + (size_t)(h * FT + i) * P + nc);
  w0 = pscale(w0, L.fwd_scale);            // C47's (N M)^-1/2
  sp_twiddleF<FT>(v, w0, w1, w4);
  if constexpr (G::PAIR == 2) sp_pair<FT, true>(v, h != 0, sw);
  RegFFT<FT, +1>::run(v);
  // Y[nc + P m], m = PAIR mm + h, to every member of the leader's set (identical rows are transformed once)
  float2 *Yseg = A.coef + (size_t)seg * A.ctot + nc + (size_t)h * P;
  const int nm = L.nmem;
  sc.mid();
  for (int m = 0; m < nm; ++m) {
    float2 *Y = Yseg + sh.mem[L.mem0 + m].x;
#pragma unroll
    for (int mm = 0; mm < FT; ++mm) __stcs(Y + (size_t)mm * (G::PAIR * P), v[mm]);
  }
}

// --------------------------------------------------------------------------------------------------
// inverse items (row t of the order: position oi = t / batch of the order table, segment t % batch)
// --------------------------------------------------------------------------------------------------
template <int F, class Sched>
__device__ __forceinline__ void sp_inv_radix(const SpArgs &A, const SpShared &sh, float2 *sw, const int *off, int nm,
                                             int row, int ncb, const Sched &sc) {
  typedef SpGeo<F> G;
  constexpr int P = kSpP, M = F * P, FT = G::FT;
  const int lane = threadIdx.x & 31;
  const int oi = row / A.batch, seg = row - oi * A.batch;
  const float amp = sh.lead[sh.order[oi].lead].inv_amp;
  const int h = G::PAIR == 2 ? (lane >> 4) : 0;
  const int nc = ncb * G::NC_ITEM + (G::PAIR == 2 ? (lane & 15) : lane);
  const float2 *Yseg = A.coef + (size_t)seg * A.ctot + nc + (size_t)h * P;
  float2 v[FT];
  {
    const float2 *Y = Yseg + off[0];
#pragma unroll
    for (int mm = 0; mm < FT; ++mm) v[mm] = __ldcs(Y + (size_t)mm * (G::PAIR * P));
  }
  for (int m = 1; m < nm; ++m) {           // Eq. 11's sum over identical rows, by linearity before the transform
    const float2 *Y = Yseg + off[m];
    float2 y[FT];
#pragma unroll
    for (int mm = 0; mm < FT; ++mm) y[mm] = __ldcs(Y + (size_t)mm * (G::PAIR * P));
#pragma unroll
    for (int mm = 0; mm < FT; ++mm) v[mm] = padd(v[mm], y[mm]);
  }
  float2 w1 = __ldg(A.ftw + nc), w4 = __ldg(A.ftw + P + nc);
  float2 w0 = make_float2(1.f, 0.f);
  if (G::PAIR == 2 && h) w0 = __ldg(A.ftw + 2 * P + nc);
  w1.y = -w1.y; w4.y = -w4.y; w0.y = -w0.y;
  w0 = pscale(w0, amp);                    // C49's sqrt(N/M)
  RegFFT<FT, -1>::run(v);
  if constexpr (G::PAIR == 2) sp_pair<FT, false>(v, h != 0, sw);
  sp_twiddleF<FT>(v, w0, w1, w4);          // lane h now holds u[q = FT h + i][nc]
  float2 *Z = A.scratch + (size_t)(row % A.nslots) * M;
  sc.wait0();                              // the slot's previous row has been read
  sc.mid();
#pragma unroll
  for (int i = 0; i < FT; ++i) __stcg(Z + (size_t)(h * FT + i) * P + nc, v[i]);
}

template <int F, class Sched>
__device__ __forceinline__ void sp_inv_sub(const SpArgs &A, const SpShared &sh, float2 *sw, const float2 *stw,
                                           int row, int q, const Sched &sc) {
  constexpr int P = kSpP, M = F * P, S = kSpRes / F;
  const int lane = threadIdx.x & 31;
  const int oi = row / A.batch, seg = row - oi * A.batch;
  const SpOrder O = sh.order[oi];
  const ClLeader &L = sh.lead[O.lead];
  const float2 *Z = A.scratch + (size_t)(row % A.nslots) * M + (size_t)q * P;
  sc.wait0();                              // the row's radix-F stage is in the slot
  float2 v[32];
#pragma unroll
  for (int r = 0; r < 32; ++r) v[r] = __ldcg(Z + lane + 32 * r);            // nc = lane + 32 r
  RegFFT<32, -1>::run(v);
#pragma unroll
  for (int r = 0; r < 32; ++r) sw[33 * lane + r] = v[r];
  __syncwarp();
#pragma unroll
  for (int r = 0; r < 32; ++r) v[r] = sw[lane + 33 * r];
  __syncwarp();
  sp_twiddle32<-1>(v, stw, lane);
  RegFFT<32, -1>::run(v);                  // v[r] = Bhat[q + F jc], jc = lane + 32 r
  sc.wait1();                              // the previous leader of the group has added its bands
  sc.mid();
  // G_k[jj] = sqrt(N/M) Bhat[jj] W_k[jj], added into the group's partial sum at bin kc + jj (R8 clip).  The
  // partial sum is sorted by residue like the spectrum copy (element of bin f: (f mod 64) len64 + f div 64),
  // so a warp's updates are whole lines.  The loads of a batch are issued before its stores.
  const float *Wp = A.wt + sh.wt[O.lead] + q * P + lane;
  const int e = lane % S;
  const int f0 = L.kc + q + F * e;
  const int res = f0 & (kSpRes - 1);
  float2 *pp = A.part + (size_t)seg * A.part_stride + O.pbase + (size_t)res * O.len64 + (f0 >> 6) + (lane - e) / S;
  const int hi = min(L.dk, A.nbins - 1 - L.kc), lo = max(-L.dk, -L.kc);
  const int jj0 = q + F * lane;
  const int a = hi - jj0, b = lo - jj0;
#pragma unroll
  for (int r0 = 0; r0 < 32; r0 += 16) {
    float2 old[16]; float w[16];
#pragma unroll
    for (int u = 0; u < 16; ++u) {
      const int r = r0 + u;
      const int c = r * 32 * F - (r >= 16 ? M : 0);
      const bool ok = r < 16 ? c <= a : c >= b;
      old[u] = ldg_cg_f2(pp + (32 / S) * r - (r >= 16 ? P / S : 0), ok);
      w[u] = __ldg(Wp + 32 * r);
    }
#pragma unroll
    for (int u = 0; u < 16; ++u) {
      const int r = r0 + u;
      const int c = r * 32 * F - (r >= 16 ? M : 0);
      const bool ok = r < 16 ? c <= a : c >= b;
      const float g = w[u];                // sqrt(N/M) rode on the radix-F twiddles
      if (ok) __stcg(pp + (32 / S) * r - (r >= 16 ? P / S : 0), pfma(v[r], make_float2(g, g), old[u]));
    }
  }
}

// Copy of the spectrum sorted by residue (see kSpRes): a CTA takes 4096 consecutive bins, 64 of every residue.
__global__ void __launch_bounds__(256)
k_spec_residues(const float2 *__restrict__ spec, long long xstride, int nbins, float2 *__restrict__ xt,
                long long xt_stride, int xt_len) {
  __shared__ float2 tile[64][65];
  const int seg = blockIdx.y, f0 = blockIdx.x * 4096;
  const float2 *X = spec + (size_t)seg * xstride;
  for (int i = threadIdx.x; i < 4096; i += 256) {
    const int f = f0 + i;
    tile[i >> 6][i & 63] = f < nbins ? __ldg(X + f) : make_float2(0.f, 0.f);    // [idx][res]
  }
  __syncthreads();
  float2 *T = xt + (size_t)seg * xt_stride + kSpPad + (f0 >> 6);
  for (int i = threadIdx.x; i < 4096; i += 256) {
    const int res = i >> 6, di = i & 63;
    if (f0 + 64 * di < ((nbins + 63) & ~63)) T[(size_t)res * xt_len + di] = tile[di][res];
  }
}

// --------------------------------------------------------------------------------------------------
// the kernel: item order, dependencies, signals (everything per warp)
// --------------------------------------------------------------------------------------------------
// the schedule's hooks inside an item: wait0 / wait1 before the first access that depends on the chunk's first /
// second count, mid just before the item's stores
template <class W0, class W1, class M> struct SpSched { const W0 &wait0; const W1 &wait1; const M &mid; };

// what a chunk waits for (up to two counts) and what it signals
struct SpDeps { const int *p0; int n0; const int *p1; int n1; int *sig; };

template <int F, bool FWD>
__device__ __forceinline__ bool sp_decode(const SpArgs &A, const SpShared &sh, unsigned int chunk, int &row, int &id,
                                          bool &first, SpDeps &D) {
  typedef SpGeo<F> G;
  constexpr int N1 = FWD ? G::NSUB : G::NRAD;      // items of the first stage per row, of the second
  constexpr int N2 = FWD ? G::NRAD : G::NSUB;
  const int t = (int)(chunk / G::PER);
  id = (int)(chunk - (unsigned int)t * G::PER) * kSpChunk;       // first item of the chunk
  first = id < N1;
  D.p0 = D.p1 = nullptr; D.n0 = D.n1 = 0; D.sig = nullptr;
  if (first) {
    row = t;
    if (row >= A.nrows) return false;
    if (row >= A.nslots) { D.p0 = A.cnt2 + (row - A.nslots); D.n0 = N2; }   // the slot's previous row is done
    D.sig = A.cnt1 + row;
  } else {
    id -= N1;
    row = t - A.lag;
    if (row < 0) return false;
    D.p0 = A.cnt1 + row; D.n0 = N1;
    if (!FWD) {
      const int oi = row / A.batch;
      const int prev = sh.order[oi].prev;
      if (prev >= 0) { D.p1 = A.cnt2 + (prev * A.batch + (row - oi * A.batch)); D.n1 = N2; }
    }
    D.sig = A.cnt2 + row;
  }
  return true;
}

template <int F, bool FWD>
__global__ void __launch_bounds__(kSpNT, 4)
k_rows_split(const SpArgs A) {
  typedef SpGeo<F> G;
  float2 *s = reinterpret_cast<float2 *>(qtam_sp_smem);
  float2 *stw = s + kSpSmemElems;
  SpShared &sh = *reinterpret_cast<SpShared *>(stw + kSpTwElems);
  const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
  for (int i = tid; i < kSpTwElems; i += kSpNT) stw[i] = A.tw2[i];
  for (int i = tid; i < A.nlead; i += kSpNT) {
    sh.lead[i] = A.lead[i]; sh.wt[i] = A.wt_off[i];
    if (!FWD) sh.order[i] = A.order[i];
  }
  for (int i = tid; i < A.nmem; i += kSpNT) sh.mem[i] = A.mem[i];
  __syncthreads();                         // the only block barrier: from here on every warp is on its own
  float2 *sw = s + wid * (kSpP + kSpP / 32);
  int *off = sh.off[wid];
  const unsigned int total = (unsigned int)(A.nrows + A.lag) * G::PER;

  // Lane 0 looks after the schedule, with no latency in the warp's way in the steady state:
  //  - the counts a chunk depends on are read (relaxed loads) at its top and looked at only where the dependent
  //    access starts -- for first-stage chunks that is just before their stores into the slot, at the very end;
  //    a count that was not there yet is polled with acquire loads;
  //  - the next chunk is popped in the middle of the running one, just before its stores (the number is needed
  //    at the top of the next iteration: an atomicAdd whose result is used at once costs a round trip to L2);
  //  - the completion signal of a chunk (fence + atomicAdd) is sent from that same point of the NEXT chunk: by
  //    then the signalled stores have been performed and the fence is cheap.  A pending signal is sent first
  //    whenever the warp has to wait.
  int *pend = nullptr;
  unsigned int chunk = 0, popped_val = 0; bool popped = false;
  int v0 = 0, v1 = 0; SpDeps D;
  D.p0 = D.p1 = nullptr; D.n0 = D.n1 = 0; D.sig = nullptr;
  auto flush = [&]() {
    // release only: a fence (acq_rel) would also invalidate L1
    if (lane == 0 && pend) {
      asm volatile("red.release.gpu.global.add.s32 [%0], %1;" :: "l"(pend), "r"(kSpChunk) : "memory");
      pend = nullptr;
    }
  };
  auto wait_on = [&](const int *p, int n, int v) {
    if (lane == 0 && p && v < n) { flush(); while (ld_acquire(p) < n) __nanosleep(64); }
    __syncwarp();
  };
  auto wait0 = [&]() { wait_on(D.p0, D.n0, v0); };
  auto wait1 = [&]() { wait_on(D.p1, D.n1, v1); };
  auto mid = [&]() {
    flush();
    if (lane == 0 && !popped) { popped_val = atomicAdd(A.queue, 1u); popped = true; }
  };
  const SpSched<decltype(wait0), decltype(wait1), decltype(mid)> sc{wait0, wait1, mid};
  if (lane == 0) chunk = atomicAdd(A.queue, 1u);
  for (;;) {
    chunk = __shfl_sync(0xffffffffu, chunk, 0);
    if (chunk >= total) break;
    int row, id; bool first;
    const bool valid = sp_decode<F, FWD>(A, sh, chunk, row, id, first, D);
    popped = false; v0 = 0; v1 = 0;
    if (lane == 0 && valid) {
      // (acquire loads: a count that is already there when it is first read is the common case, and a relaxed load
      // that observes the signalling warp's red.release does not synchronise with it under the PTX memory model --
      // the lanes' reads of the guarded slot after the __syncwarp need this load to be the acquire side)
      if (D.p0) v0 = ld_acquire(D.p0);
      if (D.p1) v1 = ld_acquire(D.p1);
    }
    if (valid) {
      if constexpr (FWD) {
        if (first) {
          for (int i = 0; i < kSpChunk; ++i) sp_fwd_sub<F>(A, sh, sw, stw, row, id + i, sc);
        } else {
          for (int i = 0; i < kSpChunk; ++i) sp_fwd_radix<F>(A, sh, sw, row, id + i, sc);
        }
      } else {
        // the members that take part: none -> the row contributes nothing (the same decision in all its items);
        // its place in the order of the group's leaders is kept all the same
        const int oi = row / A.batch;
        const ClLeader &L = sh.lead[sh.order[oi].lead];
        const int nm = sp_members(A, sh, L, first ? off : nullptr);
        if (nm > 0) {
          if (first) {
            for (int i = 0; i < kSpChunk; ++i) sp_inv_radix<F>(A, sh, sw, off, nm, row, id + i, sc);
          } else {
            for (int i = 0; i < kSpChunk; ++i) sp_inv_sub<F>(A, sh, sw, stw, row, id + i, sc);
          }
        } else if (!first) {
          wait1();
        }
      }
    }
    mid();
    if (lane == 0) {
      if (valid) pend = D.sig;
      chunk = popped_val;
    }
    __syncwarp();
  }
  flush();
}

// --------------------------------------------------------------------------------------------------
// host side
// --------------------------------------------------------------------------------------------------
int split_max_leaders() { return kSpMaxLead; }
int split_max_members() { return kSpMaxMem; }

static size_t sp_smem_bytes() { return sizeof(float2) * (size_t)(kSpSmemElems + kSpTwElems) + sizeof(SpShared); }

template <int F> static bool sp_prepare(qtam_plan *p, int c) {
  return kernel_prepare(p->cfg_rows_sp[c][1], k_rows_split<F, true>, kSpNT, sp_smem_bytes()) &&
         kernel_prepare(p->cfg_rows_sp[c][0], k_rows_split<F, false>, kSpNT, sp_smem_bytes());
}

qtam_status build_rows_split(qtam_plan *p, int c, const std::vector<ClLeader> &lead, const std::vector<int2> &mem,
                             const std::vector<ClGroup> &groups) {
  auto up = [&](void **dst, const void *src, size_t bytes) -> bool {
    *dst = nullptr;
    if (cudaMalloc(dst, bytes ? bytes : 16) != cudaSuccess) return false;
    p->device_bytes += bytes;
    return !src || bytes == 0 || cudaMemcpy(*dst, src, bytes, cudaMemcpyHostToDevice) == cudaSuccess;
  };
  const long double tau = 6.283185307179586476925286766559005768L;
  p->sp_ok[c] = false;
  if (lead.empty()) return QTAM_OK;
  const long long M = 1LL << (kClLog2Min + c);
  const int F = (int)(M / kSpP);
  bool ok = false;
  switch (F) {
    case 32: ok = sp_prepare<32>(p, c); break;
    case 64: ok = sp_prepare<64>(p, c); break;
    default: break;
  }
  if (!ok) return QTAM_ERR_CUDA;
  // radix-F twiddles: rows m = 1, 4, 32 of e^{2 pi i m nc / M}, nc < P (long double, index reduced mod M)
  {
    std::vector<float> t;
    for (int m : {1, 4, 32})
      for (int nc = 0; nc < kSpP; ++nc) {
        const long double a = tau * (long double)(((long long)nc * m) % M) / (long double)M;
        t.push_back((float)cosl(a)); t.push_back((float)sinl(a));
      }
    if (!up(&p->d_sp_ftw[c], t.data(), t.size() * sizeof(float))) return QTAM_ERR_ALLOC;
  }
  // inverse row order: round robin over the groups, so that the leaders of one group -- whose updates of the
  // group's partial sum follow each other -- lie a whole round apart
  {
    std::vector<SpOrder> order;
    std::vector<int> pos(lead.size(), -1);
    int lmax = 0;
    for (const ClGroup &g : groups) lmax = std::max(lmax, g.nlead);
    for (int l = 0; l < lmax; ++l)
      for (const ClGroup &g : groups)
        if (l < g.nlead) {
          const int li = g.lead0 + l;
          SpOrder o{};
          o.lead = li; o.prev = l > 0 ? pos[(size_t)li - 1] : -1;
          o.len64 = (int)(((g.lo + g.nb - 1) >> 6) - (g.lo >> 6) + 1);
          o.pbase = (int)(g.part_off - (g.lo >> 6));
          pos[(size_t)li] = (int)order.size();
          order.push_back(o);
        }
    if (!up(&p->d_sp_order[c], order.data(), order.size() * sizeof(SpOrder))) return QTAM_ERR_ALLOC;
    p->sp_part_lo[c] = groups.front().part_off;
    const ClGroup &gl = groups.back();
    p->sp_part_len[c] = gl.part_off + kSpRes * (((gl.lo + gl.nb - 1) >> 6) - (gl.lo >> 6) + 1) - groups.front().part_off;
  }
  // windows by residue: WT[q][jc] = W_k[q + F jc'] (jc' = jc or jc - P), zero off the support; one table per
  // distinct window of the class
  {
    const HostPlan &hp = p->hp;
    std::vector<float> wt;
    std::vector<int> wt_off(lead.size(), 0);
    // keyed on (half-width, window identity) like build_fast: a row's woff is its private offset into hp.win, so
    // keying on it would give every leader (the clamped rows of every plane) a table of its own
    std::vector<std::pair<std::pair<long long, int>, int>> seen;   // ((dk, wid), first element)
    for (size_t li = 0; li < lead.size(); ++li) {
      const ClLeader &L = lead[li];
      const std::pair<long long, int> key((long long)L.dk, hp.rows[(size_t)L.row].wid);
      int at = -1;
      for (const auto &e : seen) if (e.first == key) at = e.second;
      if (at < 0) {
        at = (int)wt.size();
        seen.push_back(std::make_pair(key, at));
        wt.resize(wt.size() + (size_t)M, 0.f);
        for (int q = 0; q < F; ++q)
          for (int jc = 0; jc < kSpP; ++jc) {
            const long long jj = q + (long long)F * (jc < kSpP / 2 ? jc : jc - kSpP);
            if (jj >= -L.dk && jj <= L.dk) wt[(size_t)at + (size_t)q * kSpP + jc] = (float)hp.win[(size_t)(L.woff + L.dk + jj)];
          }
      }
      wt_off[li] = at;
    }
    if (!up(&p->d_sp_wt[c], wt.data(), wt.size() * sizeof(float))) return QTAM_ERR_ALLOC;
    if (!up(&p->d_sp_wtoff[c], wt_off.data(), wt_off.size() * sizeof(int))) return QTAM_ERR_ALLOC;
  }
  if (!p->d_sp_xt) {
    p->sp_xt_len = 2 * kSpPad + (int)((p->hp.nb + kSpRes - 1) / kSpRes);
    p->sp_xt_pad = kSpPad;
    const size_t bytes = sizeof(float2) * (size_t)p->max_batch * kSpRes * (size_t)p->sp_xt_len;
    if (!up(&p->d_sp_xt, nullptr, bytes)) return QTAM_ERR_ALLOC;
    if (cudaMemset(p->d_sp_xt, 0, bytes) != cudaSuccess) return QTAM_ERR_CUDA;   // the pads stay zero for good
  }
  p->sp_nmem[c] = (int)mem.size();
  // the ring: LAG = twice the rows in flight (a second-stage item finds its row finished when it is popped),
  // and as many slots again plus the rows in flight
  const int per = (F + kSpP / (F > 32 ? 16 : 32)) / kSpChunk;           // chunks per row
  const int occ = std::max(std::min(p->cfg_rows_sp[c][0].occ, p->cfg_rows_sp[c][1].occ), 1);
  const int inflight = (p->num_sms * occ * (kSpNT / 32) + per - 1) / per;   // rows in flight: one chunk per warp
  p->sp_lag[c] = 2 * inflight + 1;
  p->sp_nslots[c] = p->sp_lag[c] + 2 * inflight + 4;
  if (!up(&p->d_sp_scratch[c], nullptr, sizeof(float2) * (size_t)p->sp_nslots[c] * (size_t)M)) return QTAM_ERR_ALLOC;
  const size_t nrows = lead.size() * (size_t)p->max_batch;
  if (!up(reinterpret_cast<void **>(&p->d_sp_ctl[c]), nullptr, sizeof(int) * (2 * nrows + 4))) return QTAM_ERR_ALLOC;
  if (!p->d_sp_tw2) {
    // pass-2 table of the sub-transforms: rows m = 1, 2, 3, 4, 8, .., 28 of e^{2 pi i m k / 1024}, k < 32
    std::vector<float> t;
    for (int row = 0; row < kSpTwRows; ++row) {
      const int m = row < 3 ? row + 1 : 4 * (row - 2);
      for (int k = 0; k < 32; ++k) {
        const long double a = tau * (long double)((k * m) % kSpP) / (long double)kSpP;
        t.push_back((float)cosl(a)); t.push_back((float)sinl(a));
      }
    }
    if (!up(&p->d_sp_tw2, t.data(), t.size() * sizeof(float))) return QTAM_ERR_ALLOC;
  }
  p->sp_ok[c] = true;
  return QTAM_OK;
}

template <int F, bool FWD>
static qtam_status sp_launch(qtam_plan *p, int c, int batch, void *d_coef, int plane, cudaStream_t st) {
  typedef SpGeo<F> G;
  const KernelCfg &cfg = p->cfg_rows_sp[c][FWD ? 1 : 0];
  if (!cfg.ready) return QTAM_ERR_CUDA;
  const size_t nrows = (size_t)p->n_cl_lead[c] * (size_t)batch;
  SpArgs A{};
  A.lead = p->d_cl_lead[c]; A.mem = p->d_cl_mem[c]; A.nlead = p->n_cl_lead[c]; A.nmem = p->sp_nmem[c];
  A.order = static_cast<const SpOrder *>(p->d_sp_order[c]);
  A.wt = static_cast<const float *>(p->d_sp_wt[c]); A.wt_off = static_cast<const int *>(p->d_sp_wtoff[c]);
  A.xt = static_cast<const float2 *>(p->d_sp_xt); A.xt_len = p->sp_xt_len;
  A.xt_stride = (long long)kSpRes * p->sp_xt_len;
  A.nbins = (int)p->hp.nb;
  A.coef = static_cast<float2 *>(d_coef); A.ctot = p->hp.ctot;
  A.part = static_cast<float2 *>(p->d_part); A.part_stride = p->part_stride;
  A.tw2 = static_cast<const float2 *>(p->d_sp_tw2);
  A.ftw = static_cast<const float2 *>(p->d_sp_ftw[c]);
  A.scratch = static_cast<float2 *>(p->d_sp_scratch[c]); A.nslots = p->sp_nslots[c]; A.lag = p->sp_lag[c];
  A.cnt1 = p->d_sp_ctl[c] + 4; A.cnt2 = A.cnt1 + nrows;
  A.queue = reinterpret_cast<unsigned int *>(p->d_sp_ctl[c]);
  A.batch = batch; A.plane = plane; A.nrows = (int)nrows;
  const long long chunks = (long long)(nrows + (size_t)A.lag) * G::PER;
  const long long grid = std::min<long long>((chunks + kSpNT / 32 - 1) / (kSpNT / 32), (long long)p->num_sms * cfg.occ);
  const double bytes = (double)batch * 8.0 * p->cl_sumM[c];       // compulsory: the coefficients
  {
    LaunchScope ls(p, st, (KernelId)((FWD ? K_ROWS_L14_FWD : K_ROWS_L14_INV) + c), bytes, bytes + (double)batch * 8.0 * p->cl_sumL[c]);
    if (cudaMemsetAsync(p->d_sp_ctl[c], 0, sizeof(int) * (2 * nrows + 4), st) != cudaSuccess) return QTAM_ERR_CUDA;
    if (!FWD) {
      // the groups' partial sums start at zero
      if (cudaMemset2DAsync(static_cast<float2 *>(p->d_part) + p->sp_part_lo[c], sizeof(float2) * (size_t)p->part_stride,
                            0, sizeof(float2) * (size_t)p->sp_part_len[c], (size_t)batch, st) != cudaSuccess)
        return QTAM_ERR_CUDA;
    }
    k_rows_split<F, FWD><<<(unsigned)grid, kSpNT, cfg.smem, st>>>(A);
  }
  QTAM_LAUNCH_CHECK();
  return QTAM_OK;
}

// the residue-sorted copy of the spectrum the forward sub-transforms read (after the long R2C, before the rows)
qtam_status split_spectrum(qtam_plan *p, int batch, cudaStream_t st) {
  if (!p->d_sp_xt) return QTAM_OK;
  if (p->sp_xt_fresh) { p->sp_xt_fresh = false; return QTAM_OK; }   // the long FFT has left it there
  const int nb = (int)p->hp.nb;
  const dim3 grid((unsigned)((nb + 4095) / 4096), (unsigned)batch);
  const double bytes = (double)batch * 8.0 * (double)nb;
  {
    LaunchScope ls(p, st, K_SPEC_RES, 0.0, 2.0 * bytes);
    k_spec_residues<<<grid, 256, 0, st>>>(static_cast<const float2 *>(p->d_spec), p->xstride, nb,
                                          static_cast<float2 *>(p->d_sp_xt), (long long)kSpRes * p->sp_xt_len,
                                          p->sp_xt_len);
  }
  QTAM_LAUNCH_CHECK();
  return QTAM_OK;
}

qtam_status split_rows(qtam_plan *p, int c, bool fwd, int batch, void *d_coef, int plane, cudaStream_t st) {
  const int F = (int)((1LL << (kClLog2Min + c)) / kSpP);
  switch (F) {
    case 32: return fwd ? sp_launch<32, true>(p, c, batch, d_coef, plane, st) : sp_launch<32, false>(p, c, batch, d_coef, plane, st);
    case 64: return fwd ? sp_launch<64, true>(p, c, batch, d_coef, plane, st) : sp_launch<64, false>(p, c, batch, d_coef, plane, st);
    default: break;
  }
  return QTAM_ERR_UNSUPPORTED;
}

}  // namespace qtam
