// qtam_internal.hpp -- shared declarations of libqtam (host plan + device tables).
// Product code: shares nothing with oracle/.
#pragma once
#include <cstddef>
#include <cstdint>
#include <vector>

#include "../../include/qtam.h"

namespace qtam {

// ---- host-side plan (built once by build_host_plan, plan.cpp) -------------------------------------
struct HostRow {
  int plane, row;
  double q, f_request, f_center;
  int64_t kc, dk, L, M, offset;   // offset into a segment's coefficient vector
  int64_t woff;                   // offset of W_k[-dk] in the window table
  int64_t goff;                   // offset of the row's band in the band workspace (== woff)
  double norm;
  int wid;                        // window identity: rows with the same (kc, dk, wid) are identical rows
};

struct HostPlan {
  double fs = 0;
  int64_t N = 0, nb = 0;            // samples, one-sided bins N/2+1
  int nP = 0, nR = 0;               // planes, rows per plane
  qtam_dtype dtype = QTAM_F32;
  qtam_options opt{};
  std::vector<HostRow> rows;
  std::vector<double> win;          // concatenated normalised windows, sum_L values
  int64_t ctot = 0, sumL = 0, Mmax = 0;
  // frame operator / cover sets: index 0 joint, 1+p plane p; each nb long
  std::vector<std::vector<double>> P;
  std::vector<std::vector<uint8_t>> cover;
  int64_t cover_lo = -1, cover_hi = -1, holes = 0;
  double frame_A = 0, frame_B = 0;
  // CSR bin -> band-workspace index, entries ordered by (bin, row); csr_ptr has (nP+1) entries per bin
  // plus a final sentinel: plane p of bin f spans [csr_ptr[f*(nP+1)+p], csr_ptr[f*(nP+1)+p+1])
  std::vector<int32_t> csr_ptr;
  std::vector<int32_t> csr_idx;
};

// returns QTAM_OK or an error; fills `hp`
qtam_status build_host_plan(HostPlan &hp, double fs, int64_t N, const double *Q, int nQ, double fmin,
                            double fmax, double spacing, qtam_dtype dtype, const qtam_options *opt);

// ---- device-side tables -----------------------------------------------------------------------------
struct RowDev {          // one per row, in global memory
  int kc, dk, M, log2M;
  int plane, pad0;
  long long offset;      // into coef segment
  long long woff;        // into window table / band workspace segment
  double fwd_scale;      // (N*M)^(-1/2)      (C47, R4)
  double inv_amp;        // sqrt(N/M)         (C49)
};

struct WorkItem {        // one sub-transform of a row: M = R1 * M2, residue j1 (generic path)
  int row, j1, R1, log2M2;
};

}  // namespace qtam
