// cluster_noalloc.cu -- qtam_cluster_noalloc: the cluster labelling of cluster.cu (R19) for
// callers that are not in a position to allocate device memory.
//
// Who that is.  Every other compute call of this library needs a qtam_plan, and qtam_plan_create obtains the plan's
// tables and workspace with cudaMalloc.  Some users of the labelling step cannot do that:
//   - a stage of a low-latency pipeline (the paper's Sec. V is such a search) that runs after start-up, where a
//     cudaMalloc / cudaFree would synchronise the whole device and stall every other stream for an unbounded time;
//   - a plug-in inside a host application that has given all free device memory to its own pool (a framework's caching
//     allocator): a raw cudaMalloc from a plug-in fails there, or eats into memory the host counts as its own;
//   - code that is handed its buffers by somebody else and is simply not allowed to own device memory.
// They already hold an image of coefficients (theirs) and room for the labels (theirs); the only thing the labelling
// needs beyond that is one pixel counter per component root.  qtam_cluster keeps those counters in the plan's
// workspace; here they live in a file-scope __device__ array of fixed size, which the CUDA runtime places on every
// device that loads libqtam.so when the module is loaded and keeps until the process ends (4 MiB per device, used or
// not).  The call itself allocates and frees nothing, on the device or on the host, and needs no plan.
//
// What follows from one shared array:
//   - the problem size is bounded: batch * rows * samples <= QTAM_CLUSTER_NOALLOC_MAX_PIXELS, else
//     QTAM_ERR_TOO_LARGE and nothing is launched;
//   - the array keeps what the previous call left in it, so the first kernel of a call sets the counters it is going
//     to use to zero before any of them is incremented;
//   - two calls that overlap on one GPU (different streams, different host threads) count into the same memory and
//     give wrong areas.  Issue the calls on one stream, or order them with events.
//
// Set-up.  In host code the array's name stands for the symbol, it is not a device address.  The first call on a
// device (with that device current) asks the runtime for the address (cudaGetSymbolAddress) and keeps it per device;
// that query may load the module and is not a stream operation, so let a first call happen during start-up, before
// any stream capture.  Later calls only launch kernels.
//
// The kernels are written for this entry point (a union-find like cluster.cu's, but the image is addressed directly by
// pointer and segment stride, the counters are cleared here, and the parent links are read through volatile loads,
// because other threads relink them while a thread walks them).  Nothing in cluster.cu is used or changed.
#include <cuda_runtime.h>

#include <mutex>

#include "../../include/qtam.h"
#include "cplx.cuh"

namespace qtam {
namespace {

constexpr long long kNoAllocPixels = QTAM_CLUSTER_NOALLOC_MAX_PIXELS;
constexpr int kNoAllocDevices = 64;

// pixel counters of the component roots, [batch][rows * samples] of the running call
static __device__ __align__(256) int g_noalloc_area[kNoAllocPixels];

std::mutex g_noalloc_mu;
int *g_noalloc_area_ptr[kNoAllocDevices];      // device address of g_noalloc_area on device d, null until asked for

// the device address of the counters on the current device: asked for once per device
qtam_status noalloc_area(int **out) {
  int dev = -1;
  if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= kNoAllocDevices) { cudaGetLastError(); return QTAM_ERR_CUDA; }
  std::lock_guard<std::mutex> lock(g_noalloc_mu);
  if (!g_noalloc_area_ptr[dev]) {
    int *ptr = nullptr;
    if (cudaGetSymbolAddress(reinterpret_cast<void **>(&ptr), g_noalloc_area) != cudaSuccess || !ptr) {
      cudaGetLastError();
      return QTAM_ERR_CUDA;
    }
    g_noalloc_area_ptr[dev] = ptr;
  }
  *out = g_noalloc_area_ptr[dev];
  return QTAM_OK;
}

__device__ __forceinline__ int na_find(const int *parent, int x) {
  const volatile int *p = parent;
  int px = p[x];
  while (px != x) { x = px; px = p[x]; }
  return x;
}

// unite the components of a and b; the smaller root wins, so the final roots do not depend on the merge order
__device__ __forceinline__ void na_union(int *parent, int a, int b) {
  for (;;) {
    a = na_find(parent, a); b = na_find(parent, b);
    if (a == b) return;
    if (a > b) { const int t = a; a = b; b = t; }
    const int old = atomicMin(parent + b, a);
    if (old == b) return;
    b = old;
  }
}

// active pixels point at themselves, the others at -1; the counters and the cluster count of this call start at zero
template <typename T>
__global__ void __launch_bounds__(256)
k_na_init(const C2<T> *img, long long stride, int npx, int *parent, int *area, int *count) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i == 0) count[blockIdx.y] = 0;
  if (i >= npx) return;
  const C2<T> y = img[(long long)blockIdx.y * stride + i];
  parent[(long long)blockIdx.y * npx + i] = (y.x != (T)0 || y.y != (T)0) ? i : -1;
  area[(long long)blockIdx.y * npx + i] = 0;
}

// 4-connectivity: the right neighbour (circular in time) and the row above (not circular in frequency)
__global__ void __launch_bounds__(256) k_na_merge(int *parent_all, int R, int M) {
  const int npx = R * M;
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= npx) return;
  int *parent = parent_all + (long long)blockIdx.y * npx;
  const volatile int *pv = parent;
  if (pv[i] < 0) return;
  const int r = i / M, n = i - r * M;
  const int right = r * M + (n + 1 == M ? 0 : n + 1);
  if (right != i && pv[right] >= 0) na_union(parent, i, right);
  if (r + 1 < R && pv[i + M] >= 0) na_union(parent, i, i + M);
}

__global__ void __launch_bounds__(256) k_na_compress(int *parent_all, int *area_all, int npx) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= npx) return;
  int *parent = parent_all + (long long)blockIdx.y * npx;
  if (*(const volatile int *)(parent + i) < 0) return;
  const int root = na_find(parent, i);
  *(volatile int *)(parent + i) = root;      // a thread that passes through i afterwards still ends at the same root
  atomicAdd(area_all + (long long)blockIdx.y * npx + root, 1);
}

__global__ void __launch_bounds__(256)
k_na_filter(int *parent_all, const int *area_all, int npx, int min_area, int *count) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= npx) return;
  int *parent = parent_all + (long long)blockIdx.y * npx;
  const int root = parent[i];                // after k_na_compress: the root itself
  int label = 0;
  if (root >= 0 && area_all[(long long)blockIdx.y * npx + root] >= min_area) {
    label = root + 1;
    if (root == i) atomicAdd(count + blockIdx.y, 1);
  }
  parent[i] = label;
}

}  // namespace
}  // namespace qtam

extern "C" qtam_status qtam_cluster_noalloc(qtam_dtype dtype, const void *d_img, int64_t segment_stride, int batch,
                                            int rows, int samples, int min_area, int32_t *d_labels, int32_t *d_count,
                                            void *stream) {
  using namespace qtam;
  if (!d_img || !d_labels || !d_count || (dtype != QTAM_F32 && dtype != QTAM_F64) || batch < 0 || batch > 65535 ||
      rows < 1 || samples < 1 || min_area < 1 || segment_stride < (int64_t)rows * samples)
    return QTAM_ERR_INVALID_ARG;
  const long long npx = (long long)rows * samples;
  if (npx > kNoAllocPixels || npx * batch > kNoAllocPixels) return QTAM_ERR_TOO_LARGE;   // before any CUDA call
  if (batch == 0) return QTAM_OK;
  int *area = nullptr;
  const qtam_status s = noalloc_area(&area);
  if (s != QTAM_OK) return s;
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  cudaGetLastError();                        // an error somebody else left behind is not this call's
  const dim3 g((unsigned)((npx + 255) / 256), (unsigned)batch);
  if (dtype == QTAM_F32)
    k_na_init<float><<<g, 256, 0, st>>>(static_cast<const float2 *>(d_img), segment_stride, (int)npx, d_labels, area, d_count);
  else
    k_na_init<double><<<g, 256, 0, st>>>(static_cast<const double2 *>(d_img), segment_stride, (int)npx, d_labels, area, d_count);
  k_na_merge<<<g, 256, 0, st>>>(d_labels, rows, samples);
  k_na_compress<<<g, 256, 0, st>>>(d_labels, area, (int)npx);
  k_na_filter<<<g, 256, 0, st>>>(d_labels, area, (int)npx, min_area, d_count);
  return cudaGetLastError() == cudaSuccess ? QTAM_OK : QTAM_ERR_CUDA;
}
