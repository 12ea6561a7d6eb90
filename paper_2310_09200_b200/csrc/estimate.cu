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
