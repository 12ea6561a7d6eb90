// Parameter estimation on the device ("N_eig ... estimated ... minimum number of leading
// eigenvectors that account for a user-defined percentage of the total energy"; "Level partitions
// can be automatically determined using k-means clustering on the eigenvalues"; Table 4 caption PAPER.md:593).
// Both work on a list of eigenvalues (one collect's, or pooled from a subset of the data) and are glue, not the
// hot path: one CTA, fp64, deterministic.
//   n_eig   sort descending; total = sum of the positive eigenvalues; smallest m with sum_{a<=m} lambda_a >= f total.
//   k-means in one dimension has an exact solution: optimal clusters are contiguous in sorted order, so dynamic
//           programming over the split points minimises the within-cluster sum of squares globally (DESIGN.md
//           reading Q16: positive eigenvalues only, optionally in the log domain; interval edges at the midpoints
//           between adjacent centroids, mapped back; outer edges 0 and DBL_MAX; level 0 = highest energy).
#include "internal.h"

#include <cfloat>
#include <cstdio>
#include <cstdlib>
#include <mutex>

namespace {

constexpr int kEstThreads = 1024;

// ascending bitonic sort of m (power of two) doubles in shared memory
__device__ void bitonic_sort(double* v, int m) {
  for (int k = 2; k <= m; k <<= 1)
    for (int j = k >> 1; j > 0; j >>= 1) {
      for (int i = threadIdx.x; i < m; i += blockDim.x) {
        const int p = i ^ j;
        if (p > i) {
          const bool up = (i & k) == 0;
          const double a = v[i], b = v[p];
          if ((a > b) == up) { v[i] = b; v[p] = a; }
        }
      }
      __syncthreads();
    }
}

__global__ void __launch_bounds__(kEstThreads) n_eig_kernel(const double* __restrict__ lam, int n, int m, double fraction, int* out) {
  extern __shared__ double sh[];
  for (int i = threadIdx.x; i < m; i += blockDim.x) sh[i] = i < n ? lam[i] : -DBL_MAX;
  __syncthreads();
  bitonic_sort(sh, m);                                     // ascending: largest at m - 1
  if (threadIdx.x == 0) {
    double total = 0.0;
    for (int a = 0; a < n; ++a) { const double x = sh[m - 1 - a]; total = __dadd_rn(total, x > 0.0 ? x : 0.0); }
    const double target = __dmul_rn(fraction, total);
    double run = 0.0;
    int count = n;
    for (int a = 0; a < n; ++a) {
      const double x = sh[m - 1 - a];
      run = __dadd_rn(run, x > 0.0 ? x : 0.0);
      if (run >= target) { count = a + 1; break; }
    }
    *out = count;
  }
}

// within-cluster sum of squares of the sorted values i..j-1 from the prefix sums of the CENTRED values
// (y = x - mean of all values, which keeps S2 - S1^2 / cnt well conditioned for tightly packed spectra)
__device__ __forceinline__ double seg_cost(const double* p1, const double* p2, int i, int j) {
  const double s1 = p1[j] - p1[i], s2 = p2[j] - p2[i];
  return fmax(fma(-s1, s1 / (double)(j - i), s2), 0.0);
}

// workspace (global): x[np], p1[np+1], p2[np+1], dp[2][np+1], arg[k][np+1]
__global__ void __launch_bounds__(kEstThreads) kmeans_kernel(const double* __restrict__ lam, int n, int m, int k, int log_domain,
                                                            double* __restrict__ ws, int* __restrict__ arg, double* __restrict__ iv,
                                                            int ld_int, int* __restrict__ status) {
  extern __shared__ double sh[];
  __shared__ int np_s;
  __shared__ double mean_s;
  for (int i = threadIdx.x; i < m; i += blockDim.x) {
    const double x = i < n ? lam[i] : -1.0;
    sh[i] = x > 0.0 ? (log_domain ? log(x) : x) : DBL_MAX;  // non-positive values sort to the end and are dropped
  }
  __syncthreads();
  bitonic_sort(sh, m);
  if (threadIdx.x == 0) {
    int np = 0;
    while (np < m && sh[np] != DBL_MAX) ++np;
    np_s = np;
  }
  __syncthreads();
  const int np = np_s;
  double* x = ws;
  double* p1 = x + m;
  double* p2 = p1 + m + 1;
  double* dp0 = p2 + m + 1;
  double* dp1 = dp0 + m + 1;
  if (np < k) { if (threadIdx.x == 0) *status = 1; return; }
  for (int i = threadIdx.x; i < np; i += blockDim.x) x[i] = sh[i];
  if (threadIdx.x == 0) {
    double mean = 0.0;
    for (int i = 0; i < np; ++i) mean += sh[i];
    mean /= (double)np;
    p1[0] = 0.0; p2[0] = 0.0;
    for (int i = 0; i < np; ++i) { const double y = sh[i] - mean; p1[i + 1] = p1[i] + y; p2[i + 1] = fma(y, y, p2[i]); }
    mean_s = mean;
  }
  __syncthreads();
  // dp[c][j] = min cost of splitting the first j values into c + 1 clusters; arg[c][j] = start of the last one
  for (int j = threadIdx.x; j <= np; j += blockDim.x) { dp0[j] = j >= 1 ? seg_cost(p1, p2, 0, j) : DBL_MAX; arg[j] = 0; }
  __syncthreads();
  double* prev = dp0;
  double* cur = dp1;
  for (int c = 1; c < k; ++c) {
    for (int j = threadIdx.x; j <= np; j += blockDim.x) {
      double best = DBL_MAX;
      int bi = c;
      if (j >= c + 1)
        for (int i = c; i < j; ++i) {                      // last cluster = values i..j-1, the first i in c clusters
          const double v = prev[i] + seg_cost(p1, p2, i, j);
          if (v < best) { best = v; bi = i; }              // equal costs: the earliest split (any of them is optimal)
        }
      cur[j] = best;
      arg[(size_t)c * (m + 1) + j] = bi;
    }
    __syncthreads();
    double* t = prev; prev = cur; cur = t;
  }
  if (threadIdx.x == 0) {
    // backtrack: cluster c (ascending) = values start[c] .. start[c+1]-1
    int start[BB_MAX_LEVELS + 1];
    start[k] = np;
    for (int c = k - 1; c >= 1; --c) start[c] = arg[(size_t)c * (m + 1) + start[c + 1]];
    start[0] = 0;
    double cen[BB_MAX_LEVELS];
    for (int c = 0; c < k; ++c) cen[c] = mean_s + (p1[start[c + 1]] - p1[start[c]]) / (double)(start[c + 1] - start[c]);
    // level l = cluster k - 1 - l (level 0 = highest energy); interval = [lower edge, upper edge]
    for (int l = 0; l < k; ++l) {
      const int c = k - 1 - l;
      double lo = 0.0, hi = DBL_MAX;
      if (c > 0) { const double e = 0.5 * (cen[c - 1] + cen[c]); lo = log_domain ? exp(e) : e; }
      if (c < k - 1) { const double e = 0.5 * (cen[c] + cen[c + 1]); hi = log_domain ? exp(e) : e; }
      iv[l] = lo;
      iv[l + ld_int] = hi;
    }
    *status = 0;
  }
}

int next_pow2(int n) { int m = 1; while (m < n) m <<= 1; return m; }

}  // namespace

int bb_estimate_n_eig_dev(const double* lam_dev, int n, double fraction, int* out_dev, cudaStream_t st) {
  const int m = next_pow2(n);
  n_eig_kernel<<<1, kEstThreads, (size_t)m * sizeof(double), st>>>(lam_dev, n, m, fraction, out_dev);
  BB_CUDA(cudaGetLastError());
  return BB_OK;
}

size_t bb_kmeans_workspace_doubles(int n) { const int m = next_pow2(n); return (size_t)m + 4 * ((size_t)m + 1); }
size_t bb_kmeans_workspace_ints(int n, int k) { return (size_t)k * (next_pow2(n) + 1); }

int bb_kmeans_levels_dev(const double* lam_dev, int n, int k, int log_domain, double* ws, int* arg, double* iv_dev, int ld_int,
                         int* status_dev, cudaStream_t st) {
  const int m = next_pow2(n);
  kmeans_kernel<<<1, kEstThreads, (size_t)m * sizeof(double), st>>>(lam_dev, n, m, k, log_domain, ws, arg, iv_dev, ld_int, status_dev);
  BB_CUDA(cudaGetLastError());
  return BB_OK;
}

// ------------------------------------------------------------------------------ k-means levels without allocation
// bb_kmeans_levels_static: the same kmeans_kernel, for callers that must not allocate device memory at call time.
// Who that is: an imaging service that sized all of its device memory when it started (a streaming telescope back end
// with a fixed memory plan, or a process in which a framework's caching pool already holds nearly all of HBM, so a
// raw cudaMalloc can simply fail), and any latency-bound loop, because cudaMalloc / cudaFree take a device-wide lock
// and make the whole GPU idle before they return, stalling streams that have nothing to do with this call.
// bb_kmeans_levels above allocates four scratch buffers per call; here the dynamic-programming tables live in ONE
// array that is part of the loaded library image. Cost: every GPU that loads the library carries these
// kStaticBytes (about 170 KB) until the process exits, and the problem size is capped at BB_KMEANS_STATIC_MAX_N.
//
// The array's name below is only a host-side handle of the symbol: handed to a kernel from host code it is NOT the
// device address. The address is asked for once per device (cudaGetSymbolAddress, with that device current) and
// cached; this happens in the first call made for a device, which is therefore the set-up call (make it once,
// early, before any stream capture; it may initialise the device's primary context and load the module).
//
// All calls on one GPU share the array. kmeans_kernel writes every table entry before it reads it (x, p1, p2 and
// the dp / arg rows up to the np of THIS call), so nothing has to be cleared between calls and the contents a
// previous call left behind are never read. Two calls whose kernels overlap on the same GPU (different streams,
// or different host threads on different streams) race on the tables: serialise them on one stream.
namespace {

constexpr int kStaticM = BB_KMEANS_STATIC_MAX_N;                                    // a power of two
static_assert((kStaticM & (kStaticM - 1)) == 0, "BB_KMEANS_STATIC_MAX_N must be a power of two");
constexpr size_t kStaticDoubles = (size_t)kStaticM + 4 * ((size_t)kStaticM + 1);   // = bb_kmeans_workspace_doubles(max n)
constexpr size_t kStaticInts = (size_t)BB_MAX_LEVELS * (kStaticM + 1);             // = bb_kmeans_workspace_ints(max n, max k)
constexpr size_t kStaticIntOffset = (kStaticDoubles * sizeof(double) + 255) / 256 * 256;
constexpr size_t kStaticBytes = kStaticIntOffset + kStaticInts * sizeof(int);

static __device__ __align__(256) unsigned char kmeans_static_scratch[kStaticBytes];

constexpr int kMaxStaticDevices = 64;
std::mutex g_static_mutex;
unsigned char* g_static_ptr[kMaxStaticDevices] = {};   // device address of kmeans_static_scratch, per CUDA ordinal

// true for memory a kernel on the current device can dereference (device or managed allocations)
bool static_arg_on_device(const void* p) {
  cudaPointerAttributes a{};
  if (cudaPointerGetAttributes(&a, p) != cudaSuccess) { cudaGetLastError(); return false; }
  return a.type == cudaMemoryTypeDevice || a.type == cudaMemoryTypeManaged;
}

}  // namespace

extern "C" int bb_kmeans_levels_static(int device, void* cuda_stream, const double* lambda_dev, int n, int n_levels,
                                       int log_domain, double* intervals_dev, int ld_int, int* status_dev) {
  if (!lambda_dev || !intervals_dev || !status_dev || n < 1 || n_levels < 1 || n_levels > BB_MAX_LEVELS || n_levels > n ||
      ld_int < n_levels || device < 0 || device >= kMaxStaticDevices)
    return BB_EINVAL;
  if (n > BB_KMEANS_STATIC_MAX_N) {
    if (getenv("BB_VERBOSE"))
      fprintf(stderr, "[bluebild] bb_kmeans_levels_static: n = %d exceeds the static scratch limit of %d eigenvalues; "
                      "use bb_kmeans_levels (which allocates)\n", n, BB_KMEANS_STATIC_MAX_N);
    return BB_EUNSUPPORTED;
  }
  BB_CUDA(cudaSetDevice(device));
  if (!static_arg_on_device(lambda_dev) || !static_arg_on_device(intervals_dev) || !static_arg_on_device(status_dev))
    return BB_EINVAL;                                      // host buffers would need staging memory: not here
  unsigned char* base = nullptr;
  {
    std::lock_guard<std::mutex> lock(g_static_mutex);
    if (!g_static_ptr[device]) {                           // set-up: once per device, with that device current
      void* p = nullptr;
      BB_CUDA(cudaGetSymbolAddress(&p, kmeans_static_scratch));
      g_static_ptr[device] = static_cast<unsigned char*>(p);
    }
    base = g_static_ptr[device];
  }
  double* ws = reinterpret_cast<double*>(base);
  int* arg = reinterpret_cast<int*>(base + kStaticIntOffset);
  return bb_kmeans_levels_dev(lambda_dev, n, n_levels, log_domain != 0, ws, arg, intervals_dev, ld_int, status_dev,
                              static_cast<cudaStream_t>(cuda_stream));
}
