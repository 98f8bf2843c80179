// cluster.cu -- clusters of active pixels and their binary masks ("a clustering algorithm to identify
// contiguous energetic regions based on a tunable normalized threshold and minimum area.  For each identified
// cluster, we generated a binary mask applied to the complex CQT, which was subsequently inverted").
// The image is one Q-plane in the uniform-tile layout (qtam_options.tile_length != 0): R rows x M time samples,
// contiguous in the coefficient array.  A pixel is active where its coefficient is non-zero -- the row-median
// threshold (a4) is the "normalized threshold" and runs first.  Clusters = connected components under
// 4-connectivity, the time axis circular like the transform, the frequency axis not (R19).
// Labelling: lock-free union-find over the pixels (roots are the smallest pixel index of a component, so the result
// does not depend on the order in which threads merge), then areas, then the minimum-area filter.  The atomics
// here are on labels and counters, never on data sums.  labels[pixel] = 0 (background / dropped) or 1 + the smallest
// pixel index of its cluster: a canonical numbering, equal to the oracle's flood fill label by label.
#include <algorithm>

#include "cplx.cuh"
#include "device_plan.hpp"

namespace qtam {

// (volatile reads: other threads relink parent[] with atomicMin and plain stores while this thread walks it, so a
// link must be fetched from memory every time it is followed, never kept in a register or taken from the read-only path)
__device__ __forceinline__ int ccl_find(const int *parent, int x) {
  const volatile int *p = parent;
  int px = p[x];
  while (px != x) { x = px; px = p[x]; }
  return x;
}

// unite the components of a and b; the smaller root wins
__device__ __forceinline__ void ccl_union(int *parent, int a, int b) {
  for (;;) {
    a = ccl_find(parent, a); b = ccl_find(parent, b);
    if (a == b) return;
    if (a > b) { const int t = a; a = b; b = t; }
    const int old = atomicMin(parent + b, a);
    if (old == b) return;
    b = old;
  }
}

template <typename T>
__global__ void k_ccl_init(const C2<T> *__restrict__ coef, long long ctot, long long plane_off, int npx,
                           int *__restrict__ parent, int *__restrict__ area, int *__restrict__ count) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i == 0) count[blockIdx.y] = 0;
  if (i >= npx) return;
  const C2<T> y = coef[(long long)blockIdx.y * ctot + plane_off + i];
  parent[(long long)blockIdx.y * npx + i] = (y.x != (T)0 || y.y != (T)0) ? i : -1;
  area[(long long)blockIdx.y * npx + i] = 0;
}

__global__ void k_ccl_merge(int *parent_all, int R, int M) {
  const int npx = R * M;
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= npx) return;
  int *parent = parent_all + (long long)blockIdx.y * npx;
  if (parent[i] < 0) return;
  const int r = i / M, n = i - r * M;
  const int right = r * M + (n + 1 == M ? 0 : n + 1);     // circular in time
  if (right != i && parent[right] >= 0) ccl_union(parent, i, right);
  if (r + 1 < R && parent[i + M] >= 0) ccl_union(parent, i, i + M);
}

__global__ void k_ccl_compress(int *parent_all, int *area_all, int npx) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= npx) return;
  int *parent = parent_all + (long long)blockIdx.y * npx;
  if (parent[i] < 0) return;
  const int root = ccl_find(parent, i);
  parent[i] = root;                       // other threads passing through i still reach the same root
  atomicAdd(area_all + (long long)blockIdx.y * npx + root, 1);
}

__global__ void k_ccl_filter(int *__restrict__ parent_all, const int *__restrict__ area_all, int npx, int min_area,
                             int *__restrict__ count) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= npx) return;
  int *parent = parent_all + (long long)blockIdx.y * npx;
  const int root = parent[i];             // after k_ccl_compress: the root itself
  int label = 0;
  if (root >= 0 && area_all[(long long)blockIdx.y * npx + root] >= min_area) {
    label = root + 1;
    if (root == i) atomicAdd(count + blockIdx.y, 1);
  }
  parent[i] = label;
}

// (coef and out are not __restrict__: qtam.h allows d_out == d_coef, masking in place)
template <typename T>
__global__ void k_apply_mask(const C2<T> *coef, long long ctot, long long plane_off, int npx,
                             const int *__restrict__ labels, int label, C2<T> *out) {
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= ctot) return;
  const long long j = i - plane_off;
  C2<T> v = cmk<T>(0, 0);
  if (j >= 0 && j < npx) {
    const int l = labels[(long long)blockIdx.y * npx + j];
    if (label > 0 ? l == label : l > 0) v = coef[(long long)blockIdx.y * ctot + i];
  }
  out[(long long)blockIdx.y * ctot + i] = v;
}

// the plane's image: first coefficient, rows, row length; false unless every row of the plane has the same length
bool plane_image(const qtam_plan *p, int plane, long long *off, int *R, int *M) {
  long long first = -1, m = 0; int rows = 0;
  for (const HostRow &h : p->hp.rows) {
    if (h.plane != plane) continue;
    if (first < 0) { first = h.offset; m = h.M; }
    if (h.M != m) return false;
    ++rows;
  }
  if (rows == 0 || m * rows >= (1LL << 31)) return false;
  *off = first; *R = rows; *M = (int)m;
  return true;
}

qtam_status cluster_labels(qtam_plan *p, const void *d_coef, int batch, int plane, int min_area, int32_t *d_labels,
                           int32_t *d_count, cudaStream_t st) {
  long long off; int R, M;
  if (!plane_image(p, plane, &off, &R, &M) || !p->d_ccl_area) return QTAM_ERR_INVALID_ARG;
  const int npx = R * M;
  dim3 g((unsigned)((npx + 255) / 256), (unsigned)batch);
  const double bytes = (double)batch * (double)npx;
  {
    LaunchScope ls(p, st, K_CLUSTER, 2.0 * p->esz * bytes, (2.0 * p->esz + 8.0) * bytes);
    if (p->esz == 4)
      k_ccl_init<float><<<g, 256, 0, st>>>(static_cast<const float2 *>(d_coef), p->hp.ctot, off, npx, d_labels, p->d_ccl_area, d_count);
    else
      k_ccl_init<double><<<g, 256, 0, st>>>(static_cast<const double2 *>(d_coef), p->hp.ctot, off, npx, d_labels, p->d_ccl_area, d_count);
  }
  QTAM_LAUNCH_CHECK();
  { LaunchScope ls(p, st, K_CLUSTER, 0.0, 8.0 * bytes); k_ccl_merge<<<g, 256, 0, st>>>(d_labels, R, M); }
  QTAM_LAUNCH_CHECK();
  { LaunchScope ls(p, st, K_CLUSTER, 0.0, 12.0 * bytes); k_ccl_compress<<<g, 256, 0, st>>>(d_labels, p->d_ccl_area, npx); }
  QTAM_LAUNCH_CHECK();
  { LaunchScope ls(p, st, K_CLUSTER, 4.0 * bytes, 12.0 * bytes); k_ccl_filter<<<g, 256, 0, st>>>(d_labels, p->d_ccl_area, npx, min_area, d_count); }
  QTAM_LAUNCH_CHECK();
  return QTAM_OK;
}

qtam_status cluster_mask(qtam_plan *p, const void *d_coef, int batch, int plane, const int32_t *d_labels, int label,
                         void *d_out, cudaStream_t st) {
  long long off; int R, M;
  if (!plane_image(p, plane, &off, &R, &M)) return QTAM_ERR_INVALID_ARG;
  dim3 g((unsigned)((p->hp.ctot + 255) / 256), (unsigned)batch);
  {
    LaunchScope ls(p, st, K_MASK, 4.0 * p->esz * (double)batch * (double)p->hp.ctot);
    if (p->esz == 4)
      k_apply_mask<float><<<g, 256, 0, st>>>(static_cast<const float2 *>(d_coef), p->hp.ctot, off, R * M, d_labels, label,
                                            static_cast<float2 *>(d_out));
    else
      k_apply_mask<double><<<g, 256, 0, st>>>(static_cast<const double2 *>(d_coef), p->hp.ctot, off, R * M, d_labels, label,
                                             static_cast<double2 *>(d_out));
  }
  QTAM_LAUNCH_CHECK();
  return QTAM_OK;
}

// the areas' scratch: [max_batch][largest plane] counters, only for plans in the uniform-tile layout
qtam_status build_cluster(qtam_plan *p) {
  if (p->hp.opt.tile_length == 0) return QTAM_OK;
  long long biggest = 0;
  for (int q = 0; q < p->hp.nP; ++q) {
    long long off; int R, M;
    if (plane_image(p, q, &off, &R, &M)) biggest = std::max<long long>(biggest, (long long)R * M);
  }
  if (biggest == 0) return QTAM_OK;
  const size_t bytes = sizeof(int) * (size_t)p->max_batch * (size_t)biggest;
  if (cudaMalloc(reinterpret_cast<void **>(&p->d_ccl_area), bytes) != cudaSuccess) return QTAM_ERR_ALLOC;
  p->device_bytes += bytes;
  p->ccl_pixels = biggest;
  return QTAM_OK;
}

}  // namespace qtam
