// device_plan.hpp -- the plan object behind the C ABI: host plan + device tables + workspace,
// and the launcher entry points implemented in the .cu files.
#pragma once
#include <cuda_runtime.h>

#include <map>
#include <mutex>
#include <utility>
#include <vector>

#include "qtam_internal.hpp"

namespace qtam {
// kernel ids for the launch profile (names in profile.cu)
enum KernelId {
  K_CFFT_SEQ = 0, K_CFFT_COLS, K_CFFT_ROWS, K_R2C_POST, K_C2R_PRE, K_FWD_ROWS, K_FWD_COMBINE,
  K_INV_ROWS, K_INV_REDUCE, K_DENSE_PLACE, K_THRESHOLD, K_R2C_FAST, K_FWD_ROWS_FAST, K_INV_ROWS_FAST,
  K_REDUCE_C2R_FAST, K_INV_FUSED, K_INV_TILES, K_COMBINE_C2R, K_THRESHOLD_FAST, K_ROWS_CTA_FWD, K_ROWS_CTA_INV,
  K_TINY_FWD, K_TINY_INV, K_LONG_A, K_LONG_B, K_PLANE_METRIC, K_BEST_PLANE, K_REMODULATE, K_INST_FREQ, K_FWD_ROWS_THR, K_GATHER_PLANE,
  K_ROWS_CL_FWD, K_ROWS_CL_INV, K_COMBINE_RUNS, K_C2C_FAST, K_SPLIT3, K_COMBINE3, K_LEN_BAND, K_LEN_SYNTH, K_LEN_ANALYSIS,
  K_CLUSTER, K_MASK, K_SPEC_RES,
  // rows of 2^14 .. 2^17 points, one name per length class (rows_cluster.cu, rows_split.cu): index + class
  K_ROWS_L14_FWD, K_ROWS_L15_FWD, K_ROWS_L16_FWD, K_ROWS_L17_FWD, K_ROWS_L14_INV, K_ROWS_L15_INV, K_ROWS_L16_INV, K_ROWS_L17_INV,
  K_COUNT
};
// fast float path (fast.cu): rows with 32 <= M <= 1024, grouped by G = M/32 lanes per row
struct FastRow { int kc, dk, woff, goff, offset, plane, wpad, pad; };   // wpad: offset into the padded window table
struct FastBucket { int log2G, nrows, ngroups, row_base, tw_base, pad; };
struct FastParams {
  int nbuckets, groups_per_seg, tw_total;
  int rows_smem;                // rows staged in shared memory by k_rows_fast (0: table too long, read from global)
  double sum_M, sum_L;          // coefficients / band values per segment the fast rows cover
  FastBucket b[6];
};
// tiled inverse (inv_tiled.cu): a work item = consecutive rows (sorted by centre bin) of one length bucket
// whose bands fit one warp-private accumulator of kAccBins bins
struct __align__(16) TileRow { int kc, offset, wpad, jlo, jhi, plane, pad0, pad1; };   // jlo..jhi: band offsets kept (R8 clip)
struct __align__(16) TileItem { int row0, nrows, log2G, tw_base, lo, nb, part_off, npass; };
constexpr int kAccBins = 1280;
// fast threshold (threshold_fast.cu): a warp task = up to 32/G rows of one length M = 32 G (or 32 rows of M < 32)
struct ThrTask { int log2M, row0, nrows, pad; };
constexpr int kThrFastLog2Max = 10;
// CTA-level rows (rows_cta.cu): 2^11 .. 2^13 points, one shared-memory transform per CTA;
// cluster-level rows (rows_cluster.cu): 2^14 .. 2^17 points, one transform per thread-block cluster
constexpr int kCtaLog2Min = 11, kCtaClasses = 3;
constexpr int kClLog2Min = 14, kClClasses = 4;
static_assert(kClLog2Min == 14 && kClClasses == 4, "K_ROWS_L14_FWD .. K_ROWS_L17_INV name these classes");
constexpr int kCtaLog2Max = kClLog2Min + kClClasses - 1;   // longest row of the tuned float kernels
constexpr int kCtaMaxMembers = 32;   // rows per leader (same centre bin and half-width)
// a leader = one set of identical rows (same centre bin and half-width: transformed once); a group = consecutive
// leaders whose inverse contributions one CTA / cluster adds into one partial spectrum, in order
// (the leader's record carries what the row kernels need, so that an item costs one table read: centre bin,
// half-width, window offset, (N M)^{-1/2} and sqrt(N/M); members are (coefficient offset, plane) pairs)
struct __align__(16) ClLeader { int kc, dk, woff, mem0; int nmem, row; float fwd_scale, inv_amp; };
struct ClGroup { int lead0, nlead, lo, nb; long long part_off; };
// a run = a contiguous piece of the spectrum held somewhere: `nb` bins from bin `lo` at element `off` of a
// segment's partial-sum buffer (src 1) or band workspace (src 0); plane >= 0: only for the joint inverse and for
// that plane's own (a band slot of one row); src 2: a partial sum sorted by residue, bin f at element
// off - lo div 64 + (f mod 64) len64 + f div 64 (rows_split.cu).  k_combine_runs adds the runs that cover a bin
// in list order.
struct HostRun { int lo, nb; long long off; int src, plane; };
struct ProfRec { int kid; double bytes, design; cudaEvent_t e0, e1; };
}  // namespace qtam

namespace qtam { constexpr int kSpecPad = 512; }

// A failed launch is reported once and cleared (cudaGetLastError), so that one bad call does not poison every
// later call on any plan; the compute entry points also clear whatever an earlier library left behind.
#define QTAM_LAUNCH_CHECK()                                        \
  do {                                                             \
    if (cudaGetLastError() != cudaSuccess) return QTAM_ERR_CUDA;   \
  } while (0)

namespace qtam {
// Launch configuration of one kernel instantiation, fixed when the plan is created (qtam_plan_create sets the
// dynamic shared-memory limit and asks the occupancy calculator once; the compute calls only read this).
struct KernelCfg { int occ = 0; size_t smem = 0; bool ready = false; };
// cudaFuncAttributeMaxDynamicSharedMemorySize belongs to the kernel (per device, for the whole process), not to a
// plan, and several kernels ask for a plan-dependent amount: a second plan that needs less must not lower the limit
// under a live plan that needs more (its next launch would fail).  So the limit is only ever raised: the high-water
// mark per (device, kernel) is kept here, and every plan's launches fit under it.
inline bool raise_dynamic_smem(const void *kernel, size_t smem) {
  static std::mutex mu;
  static std::map<std::pair<int, const void *>, size_t> high;
  if (smem <= 48 * 1024) return true;
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess) return false;
  std::lock_guard<std::mutex> lock(mu);
  size_t &h = high[std::make_pair(dev, kernel)];
  if (smem <= h) return true;
  if (cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess) return false;
  h = smem;
  return true;
}
template <typename K> inline bool kernel_prepare(KernelCfg &c, K kernel, int threads, size_t smem) {
  c.smem = smem; c.occ = 1; c.ready = false;
  if (!raise_dynamic_smem(reinterpret_cast<const void *>(kernel), smem)) return false;
  int occ = 0;
  if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kernel, threads, smem) != cudaSuccess) return false;
  c.occ = occ < 1 ? 1 : occ;
  c.ready = true;
  return true;
}
}  // namespace qtam   // zero bins kept on both sides of every segment's spectrum

struct qtam_plan {
  qtam::HostPlan hp;
  int esz = 4;                 // sizeof real: 4 or 8
  int max_batch = 1;
  int64_t xstride = 0;         // spectrum segment stride in complex elements (>= N/2+1, padded)
  int64_t twn = 0;             // twiddle table length, a power of two: tw[k] = e^{+2 pi i k/twn} (= N when N = 2^k)
  bool n_pow2 = true;          // N = 2^k; otherwise N = 3 * 2^k and the long transform takes a radix-3 step
  int64_t sub_n = 0;           // points of the power-of-two complex FFT behind the long real transform (N/2 or N/6)
  int cap_log2 = 0;            // generic path: largest in-smem FFT is 2^cap_log2 points

  // device tables
  qtam::RowDev *d_rows = nullptr;
  void *d_win = nullptr;       // real[sumL]
  void *d_tw = nullptr;        // complex[twn]
  void *d_twN = nullptr;       // complex[N]: e^{+2 pi i k/N} (the same table when N is a power of two)
  void *d_ws3 = nullptr;       // complex[2][max_batch][N]: scratch of the radix-3 step (N = 3 * 2^k only)
  void *d_invP = nullptr;      // real[(nP+1)*nb], 0 outside the cover set
  int32_t *d_csr_ptr = nullptr;
  int32_t *d_csr_idx = nullptr;
  long long max_plane_coeffs = 0;     // largest plane (coefficients), the row length of qtam_gather_plane's output
  long long *d_plane_off = nullptr;   // [nP+1] first coefficient of every plane (planes are contiguous)
  // generic-path work lists, one per smem size class
  static const int kClasses = 4;
  qtam::WorkItem *d_items[kClasses] = {nullptr, nullptr, nullptr, nullptr};
  int n_items[kClasses] = {0, 0, 0, 0};
  // forward lists: one leader per set of identical rows (same kc, dk; single-transform rows only); the
  // followers' coefficient offsets per leader row: d_gfol_off[d_gfol_ptr[row] .. d_gfol_ptr[row+1])
  qtam::WorkItem *d_items_fwd[kClasses] = {nullptr, nullptr, nullptr, nullptr};
  int n_items_fwd[kClasses] = {0, 0, 0, 0};
  int *d_gfol_ptr = nullptr;
  long long *d_gfol_off = nullptr;
  long long *d_gfol_woff = nullptr;   // the followers' band-workspace offsets (joint inverse zeroes their slots)
  double class_L[kClasses] = {0, 0, 0, 0};   // sum of band lengths / output lengths of a class's
  double class_M[kClasses] = {0, 0, 0, 0};   // items (for the launch profile's byte counts)
  double big_M = 0;                          // sum of M over the rows that need the combine pass
  int *d_bigrows = nullptr;    // rows with R1 > 1 (need the combine pass)
  int n_bigrows = 0;
  int big_R1max = 1;

  // workspace (sized for max_batch)
  void *d_spec = nullptr;      // complex[max_batch][xstride]   spectrum X / Xhat
  void *d_ws = nullptr;        // complex[max_batch][N]         four-step scratch, dense scratch
  void *d_band = nullptr;      // complex[max_batch][sumL]      inverse band values G_k[j]
  size_t device_bytes = 0;

  // fast float path
  bool fast_rows = false;      // rows 32..1024 points run in fast.cu
  bool fast_long = false;      // long FFTs run in fast.cu (float, N = 2^12..2^15)
  int num_sms = 148;
  qtam::FastParams fast{};
  qtam::FastRow *d_frows = nullptr;
  qtam::FastParams fast_fwd{};        // forward: one leader per set of identical rows (same kc, dk)
  qtam::FastRow *d_frows_fwd = nullptr;   // leaders: plane = number of members, pad = first entry in d_fmem
  int *d_fmem = nullptr;              // coefficient offsets of the members
  int2 *d_tmem = nullptr;             // tiled inverse: (coefficient offset, plane) of the members
  void *d_fwin = nullptr;      // float windows, one per distinct half-width
  void *d_fwinp = nullptr;     // float windows zero-padded to M points in M-array order (index j mod M)
  int4 *d_red = nullptr;       // per fast row (frows order): first bin, bins, first band index (R8 clip), plane
  void *d_spec_alloc = nullptr;   // allocation behind d_spec (zero pads of kSpecPad bins on both sides)
  void *d_ftw_fwd = nullptr;   // float2 pass-1 twiddles [bucket][n1][t], forward (x (N M)^-1/2)
  void *d_ftw_inv = nullptr;   // same, inverse (conjugate, x sqrt(N/M))
  void *d_ptw = nullptr;       // pass tables of the long FFT (ctafft.cuh)
  void *d_ptw_mid = nullptr;   // pass tables of k_cfft_cta (N = 3 * 2^k: transforms of N/6 = 2^11 .. 2^14 points)
  int mid_log2n = 0;
  void *d_ptw_long = nullptr;  // pass tables of the 2^14-point stage of long_fft.cu (N = 2^16 .. 2^20)
  qtam::FastRow *d_tiny = nullptr;   // rows shorter than 32 points (goff holds log2 M), for the combine kernel of inv_tiled.cu
  int n_tiny = 0;
  double tiny_sumM = 0, tiny_sumL = 0;   // coefficients / band values per segment of those rows
  // tiled inverse (inv_tiled.cu)
  std::vector<qtam::FastRow> h_frows;   // host copy of d_frows (bucket-major), for build_inv_tiled
  bool tiled_inv = false;
  qtam::TileRow *d_trows = nullptr;
  qtam::TileItem *d_titems = nullptr;
  int n_titems = 0;
  int64_t part_stride = 0;     // partial sums per segment (complex elements)
  void *d_part = nullptr;      // complex[max_batch][part_stride]
  unsigned int *d_counter = nullptr;   // work counter of the persistent tile kernel

  // fast threshold (threshold_fast.cu)
  qtam::ThrTask *d_thr_tasks = nullptr;
  int *d_thr_offs = nullptr;      // coefficient offsets of the tasks' rows
  int n_thr_tasks = 0;
  int thr_first[qtam::kThrFastLog2Max + 1] = {}, thr_count[qtam::kThrFastLog2Max + 1] = {};   // tasks per row length
  bool thr_has_big = false;       // some row is longer than 2^kThrFastLog2Max points (generic kernel)

  // CTA-level rows (rows_cta.cu), one class per transform length 2^11 .. 2^13
  bool cta_rows = false;
  qtam::ClLeader *d_cta_lead[qtam::kCtaClasses] = {};   // one leader per set of identical rows, ascending centre bin
  int2 *d_cta_mem[qtam::kCtaClasses] = {};              // members of the leaders: (coefficient offset, plane)
  qtam::ClGroup *d_cta_groups[qtam::kCtaClasses] = {};  // inverse: groups of consecutive leaders
  int n_cta_rows[qtam::kCtaClasses] = {}, n_cta_groups[qtam::kCtaClasses] = {};
  double cta_sumM[qtam::kCtaClasses] = {}, cta_sumL[qtam::kCtaClasses] = {};
  void *d_ptw_rows[qtam::kCtaClasses] = {};             // pass tables per class
  bool rows2k_ok = false;                               // forward rows of 2^11 points run one warp each (rows_2k.cu)
  void *d_tw_2k = nullptr;
  // cluster-level rows (rows_cluster.cu), one class per transform length 2^14 .. 2^17
  bool cl_rows = false;
  qtam::ClLeader *d_cl_lead[qtam::kClClasses] = {};
  int2 *d_cl_mem[qtam::kClClasses] = {};
  qtam::ClGroup *d_cl_groups[qtam::kClClasses] = {};
  int n_cl_lead[qtam::kClClasses] = {}, n_cl_groups[qtam::kClClasses] = {};
  double cl_sumM[qtam::kClClasses] = {}, cl_sumL[qtam::kClClasses] = {};
  void *d_cl_ptw = nullptr;                             // pass tables of the 4096-point sub-transforms
  void *d_cl_ftw[qtam::kClClasses] = {};                // radix-F twiddles per class
  // dataflow rows (rows_split.cu): the classes of 2^14 .. 2^16 points as sub-transform and radix-F items
  bool sp_ok[qtam::kClClasses] = {};
  int sp_lag[qtam::kClClasses] = {}, sp_nslots[qtam::kClClasses] = {};
  void *d_sp_tw2 = nullptr;                             // pass-2 table of the 1024-point sub-transforms
  void *d_sp_ftw[qtam::kClClasses] = {};                // radix-F twiddles per class
  void *d_sp_scratch[qtam::kClClasses] = {};            // ring of row slots (the intermediate; stays in L2)
  int *d_sp_ctl[qtam::kClClasses] = {};                 // item counter + per-row completion counts
  void *d_sp_order[qtam::kClClasses] = {};              // inverse row order (SpOrder records)
  long long sp_part_lo[qtam::kClClasses] = {}, sp_part_len[qtam::kClClasses] = {};   // the class's partial sums
  int sp_nmem[qtam::kClClasses] = {};
  void *d_sp_wt[qtam::kClClasses] = {}, *d_sp_wtoff[qtam::kClClasses] = {};   // windows by residue, first element per leader
  void *d_sp_xt = nullptr;                              // spectrum by residue [max_batch][64][sp_xt_len]
  int sp_xt_len = 0, sp_xt_pad = 0;
  bool sp_xt_fresh = false;                             // the long FFT has just written d_sp_xt (forward)
  // run-based combine (combine_runs.cu): the inverse of every float plan that is not on the tiled path
  bool use_runs = false;
  std::vector<qtam::HostRun> runs;                      // in summation order (tiles, CTA groups, cluster groups, band slots)
  int4 *d_runs = nullptr;                               // (lo, nb, off, src | (plane + 1) << 2)
  int *d_run_ptr = nullptr, *d_run_idx = nullptr;       // lists 2b (bins f) and 2b + 1 (mirror bins Nc - f) of block b
  int n_run_blocks = 0;
  bool tiles_ok = false;                                // rows of 32 .. 1024 points have tiles (k_inv_tiles)

  // launch configurations fixed at plan creation (see KernelCfg)
  qtam::KernelCfg cfg_r2c, cfg_rows_fwd, cfg_rows_thr, cfg_rows_inv, cfg_tiles, cfg_combine,
      cfg_rows_cta[qtam::kCtaClasses][2], cfg_rows_cl[qtam::kClClasses][2], cfg_rows_sp[qtam::kClClasses][2], cfg_c2c, cfg_cfft_mid[2], cfg_r3[2], cfg_rows_2k;

  // output-length options (length.cu): the plan's uniform length n, the standard one, e^{2 pi i m/n} for both
  long long len_n = 0, len_std = 0;
  void *d_len_tw[2] = {nullptr, nullptr};

  int *d_ccl_area = nullptr;    // cluster.cu: pixel counts per component root, [max_batch][ccl_pixels]
  long long ccl_pixels = 0;

  // side streams: the row launches of one call are independent of each other (disjoint outputs), so they are
  // forked onto these and joined back (events; nothing waits on the host): short classes fill the SMs the long
  // ones leave idle
  static const int kSide = 8;
  cudaStream_t side[kSide] = {};
  cudaEvent_t ev_fork = nullptr, ev_join[kSide] = {};
  int n_side = 0;

  int last_launches = 0;
  // launch profile (qtam_profile_enable / qtam_profile_read)
  bool prof_on = false;
  std::vector<qtam::ProfRec> prof_pool;   // pre-created event pairs
  int prof_used = 0;
  int prof_dropped = 0;
  bool host_only = false;      // built by qtam_plan_create_host: tables on the host only
};

namespace qtam {

// Brackets one kernel launch: counts it and, when profiling is on, records CUDA events around it on
// the launch stream.  `bytes` = the COMPULSORY bytes of SURVEY.md 8(d) this launch moves (input samples read,
// coefficients written / read, output samples written: what the method itself must move); `design` = everything
// the launch moves by design (compulsory + spectrum, partial sums, band workspace, scratch); < 0: same as bytes.
struct LaunchScope {
  qtam_plan *p; cudaStream_t st; int slot;
  LaunchScope(qtam_plan *plan, cudaStream_t stream, int kid, double bytes, double design = -1.0)
      : p(plan), st(stream), slot(-1) {
    p->last_launches += 1;
    if (!p->prof_on) return;
    if (p->prof_used >= (int)p->prof_pool.size()) { p->prof_dropped += 1; return; }
    slot = p->prof_used++;
    p->prof_pool[(size_t)slot].kid = kid;
    p->prof_pool[(size_t)slot].bytes = bytes;
    p->prof_pool[(size_t)slot].design = design < 0.0 ? bytes : design;
    cudaEventRecord(p->prof_pool[(size_t)slot].e0, st);
  }
  ~LaunchScope() { if (slot >= 0) cudaEventRecord(p->prof_pool[(size_t)slot].e1, st); }
};

// Fork-join over the plan's side streams.  next() hands out a stream that starts after everything issued on the
// caller's stream before the fork; join() makes the caller's stream wait for all of them.  Capturable in a CUDA
// graph (every forked stream joins back), never touches the host.  While the launch profile is on everything stays
// on the caller's stream, so that the profile's events bracket one kernel at a time (qtam_profile_enable).
struct Fork {
  qtam_plan *p; cudaStream_t main; int used, avail;
  Fork(qtam_plan *plan, cudaStream_t st) : p(plan), main(st), used(0), avail(plan->prof_on ? 0 : plan->n_side) {
    if (avail > 0) cudaEventRecord(p->ev_fork, main);
  }
  cudaStream_t next() {
    if (used >= avail) return main;
    cudaStream_t s = p->side[used++];
    cudaStreamWaitEvent(s, p->ev_fork, 0);
    return s;
  }
  void join() {
    for (int i = 0; i < used; ++i) {
      cudaEventRecord(p->ev_join[i], p->side[i]);
      cudaStreamWaitEvent(main, p->ev_join[i], 0);
    }
    used = 0;
  }
};

// which part of the CSR a reduction over the band workspace walks: sets plo .. phi-1 of nsets per bin
struct CsrSel { const int32_t *ptr, *idx; int nsets, plo, phi; };
inline CsrSel csr_select(const qtam_plan *p, int plane) {
  return CsrSel{p->d_csr_ptr, p->d_csr_idx, p->hp.nP + 1, plane < 0 ? 0 : plane, plane < 0 ? p->hp.nP : plane + 1};
}

// generic.cu : correct-for-everything kernels (any N, any M, float and double)
qtam_status generic_r2c(qtam_plan *p, const void *d_x, int batch, cudaStream_t st);
qtam_status generic_forward_rows(qtam_plan *p, int batch, void *d_coef, cudaStream_t st);
qtam_status generic_inverse_rows(qtam_plan *p, const void *d_coef, int batch, int plane, cudaStream_t st);
qtam_status generic_inverse_reduce(qtam_plan *p, int batch, int plane, cudaStream_t st);
qtam_status generic_c2r(qtam_plan *p, int batch, void *d_x_out, cudaStream_t st);
qtam_status generic_c2c_out(qtam_plan *p, int batch, void *d_x_out, cudaStream_t st);
qtam_status generic_dense(qtam_plan *p, int batch, int row_begin, int row_end, void *d_out, cudaStream_t st);
qtam_status generic_dense_invert(qtam_plan *p, const void *d_tile, int batch, int row, void *d_x_out, cudaStream_t st);
qtam_status generic_threshold(qtam_plan *p, void *d_coef, int batch, double kappa, int min_log2M, cudaStream_t st);

// fast.cu
qtam_status build_long_tables(qtam_plan *p);
qtam_status prepare_fast(qtam_plan *p);
qtam_status prepare_generic(qtam_plan *p);
qtam_status fast_r2c(qtam_plan *p, const void *d_x, int batch, cudaStream_t st);
qtam_status fast_forward_rows(qtam_plan *p, int batch, void *d_coef, cudaStream_t st);
qtam_status fast_inverse_rows(qtam_plan *p, const void *d_coef, int batch, int plane, cudaStream_t st);
qtam_status fast_forward_rows_threshold(qtam_plan *p, int batch, void *d_coef, float kappa, cudaStream_t st,
                                        bool *done);
qtam_status fast_tiny_inverse(qtam_plan *p, const void *d_coef, int batch, int plane, cudaStream_t st);
qtam_status fast_c2c_out(qtam_plan *p, int batch, void *d_x_out, cudaStream_t st);
// long_fft.cu
qtam_status build_long_fft(qtam_plan *p);
bool fast_cfft_long_ok(const qtam_plan *p, int log2n);
bool long_residues_ok(const qtam_plan *p);
qtam_status long_forward_residues(qtam_plan *p, const void *d_x, int batch, cudaStream_t st);
qtam_status long_inverse_residues(qtam_plan *p, void *d_x_out, int batch, cudaStream_t st);
bool fast_cfft_mid_ok(const qtam_plan *p, int log2n);
bool fast_r3_ok(const qtam_plan *p);
qtam_status fast_r3(qtam_plan *p, bool fwd, const void *d_in, void *d_out, int batch, cudaStream_t st);
qtam_status fast_cfft_mid(qtam_plan *p, const void *in, long long in_stride, void *out, long long out_stride,
                          int log2n, int count, int dir, float scale, cudaStream_t st, double algo);
qtam_status fast_cfft_long(qtam_plan *p, const void *in, long long in_stride, void *out, long long out_stride,
                           void *tmp, long long tmp_stride, int log2n, int count, int dir, float scale,
                           cudaStream_t st, double algo_in, double algo_out);
// scan.cu
qtam_status plane_metric(qtam_plan *p, const void *d_coef, int batch, int metric, void *d_metric, int32_t *d_best,
                         cudaStream_t st);
qtam_status gather_plane(qtam_plan *p, const void *d_coef, int batch, const int32_t *d_best, void *d_out,
                         cudaStream_t st);
qtam_status remodulate(qtam_plan *p, const void *d_coef, int batch, void *d_out, cudaStream_t st);
qtam_status instantaneous_frequency(qtam_plan *p, const void *d_coef, int batch, void *d_out, cudaStream_t st);
// rows_cta.cu
void build_leaders_and_groups(qtam_plan *p, const std::vector<int> &rows_in, int groups_wanted,
                              std::vector<ClLeader> &lead, std::vector<int2> &mem, std::vector<ClGroup> &groups,
                              int by_residue_max_lead, int by_residue_max_mem, bool *by_residue);
qtam_status build_rows_cta(qtam_plan *p);
qtam_status cta_forward_rows(qtam_plan *p, int batch, void *d_coef, Fork &fk);
qtam_status cta_inverse_rows(qtam_plan *p, const void *d_coef, int batch, int plane, Fork &fk);
// rows_2k.cu
qtam_status build_rows_2k(qtam_plan *p);
qtam_status rows_2k_forward(qtam_plan *p, int batch, void *d_coef, cudaStream_t st);
// rows_cluster.cu
qtam_status build_rows_cluster(qtam_plan *p);
qtam_status cluster_forward_rows(qtam_plan *p, int batch, void *d_coef, Fork &fk);
qtam_status cluster_inverse_rows(qtam_plan *p, const void *d_coef, int batch, int plane, Fork &fk);
// rows_split.cu
qtam_status build_rows_split(qtam_plan *p, int c, const std::vector<ClLeader> &lead, const std::vector<int2> &mem,
                             const std::vector<ClGroup> &groups);
int split_max_leaders();
int split_max_members();
qtam_status split_rows(qtam_plan *p, int c, bool fwd, int batch, void *d_coef, int plane, cudaStream_t st);
qtam_status split_spectrum(qtam_plan *p, int batch, cudaStream_t st);
// combine_runs.cu
qtam_status build_runs(qtam_plan *p);
qtam_status combine_runs(qtam_plan *p, int batch, int plane, cudaStream_t st);
// length.cu
long long length_resolve(const HostPlan &hp, long long mode);
qtam_status build_length(qtam_plan *p);
qtam_status length_forward(qtam_plan *p, int batch, void *d_out, cudaStream_t st);
qtam_status length_inverse_bands(qtam_plan *p, const void *d_in, int batch, int plane, cudaStream_t st);
qtam_status length_resample(qtam_plan *p, const void *d_in, int batch, int to_standard, void *d_out, cudaStream_t st);
// cluster.cu
bool plane_image(const qtam_plan *p, int plane, long long *off, int *R, int *M);
qtam_status build_cluster(qtam_plan *p);
qtam_status cluster_labels(qtam_plan *p, const void *d_coef, int batch, int plane, int min_area, int32_t *d_labels,
                           int32_t *d_count, cudaStream_t st);
qtam_status cluster_mask(qtam_plan *p, const void *d_coef, int batch, int plane, const int32_t *d_labels, int label,
                         void *d_out, cudaStream_t st);
// threshold_fast.cu
qtam_status build_thr_fast(qtam_plan *p);
qtam_status fast_threshold(qtam_plan *p, void *d_coef, int batch, double kappa, cudaStream_t st);
// inv_tiled.cu
qtam_status build_inv_tiled(qtam_plan *p);
qtam_status tiled_inverse(qtam_plan *p, const void *d_coef, int batch, int plane, void *d_x_out, cudaStream_t st);
qtam_status tiles_only(qtam_plan *p, const void *d_coef, int batch, int plane, cudaStream_t st);

}  // namespace qtam
