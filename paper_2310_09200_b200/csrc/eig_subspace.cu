// Leading eigenpairs of a batch of Hermitian matrices by block subspace iteration with Rayleigh-Ritz.
//
// Why: Algorithm 1 keeps only the N_eig largest eigenpairs (l.4; N_eig = 64 of 512 on the wide-field
// configs), the eigenproblem "must be repeated for each timestep t and frequency band f", and a full
// batched fp64 eigensolve of 20 matrices of order 512 costs ~31 ms on a B200 whatever the batch size below ~20
// (tridiagonalisation is a chain of small dependent kernels) while a strided-batched ZGEMM of the same 20 matrices
// runs at 34 TFLOP/s (0.16 ms for C X with 128 columns). So the leading invariant subspace is found with GEMMs:
//     X <- orth(C^2 X) repeated, X of p = N_eig + guard columns; then H = X^H C X (p x p), H = Q Theta Q^H, X <- X Q
//   converging like (lambda_{p+1} / lambda_{N_eig})^(2 steps); visibility matrices are sums of a few hundred
//   sources over a noise floor, so their spectra decay fast and a dozen products suffice. Orthonormalisation is
//   Cholesky-QR (Gram matrix, potrfBatched, trsmBatched), done twice before a Rayleigh-Ritz step.
// Safety: the residuals |C x - theta x| of the N_eig wanted pairs are computed on the device after each
// Rayleigh-Ritz step; unless every matrix of the batch meets 1e-11 |theta|_max (or will after a bounded number of
// further products, estimated from the Ritz values), the caller falls back to the full eigensolve. It also falls
// back, converged or not, when the block holds a negative Ritz value at least as large in magnitude as the smallest
// wanted one (powers of C^2 rank by |lambda|, so wanted pairs may then lie outside the block: uniform weighting and
// other indefinite S). Indefinite or flat spectra, breakdown of a Cholesky-QR and small problems therefore take the
// library path, not a wrong answer.
// One host synchronisation of the glue stream per Rayleigh-Ritz step (verdicts of the whole batch in 16 bytes per
// matrix); the synthesizer stream is not involved.
#include "glue_internal.h"

#include <cmath>

typedef cuDoubleComplex Z;

struct SubspaceWork {
  double* verdict_host = nullptr;        // pinned: [nb][2] = {worst relative residual, convergence ratio}
  int* info_host = nullptr;              // pinned: [nb] Cholesky-QR / Rayleigh-Ritz verdicts, OR-ed
  int cap = 0;
};

void bb_subspace_destroy(SubspaceWork* w) {
  if (!w) return;
  if (w->verdict_host) cudaFreeHost(w->verdict_host);
  if (w->info_host) cudaFreeHost(w->info_host);
  cudaGetLastError();
  delete w;
}

namespace {

constexpr double kResidualTol = 1e-11;   // |C x - theta x|_2 <= tol * theta_max for every wanted pair
constexpr int kMaxExtraSteps = 24;       // further C^2 products after the first Rayleigh-Ritz step before giving up

// deterministic start block: uniform in (-1, 1) from a counter hash (any full-rank block works)
__global__ void start_block_kernel(Z* __restrict__ x, size_t count) {
  const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= count) return;
  uint64_t h = i * 0x9E3779B97F4A7C15ull + 0x632BE59BD9B4E019ull;
  h ^= h >> 32; h *= 0xD6E8FEB86659FD93ull; h ^= h >> 32; h *= 0xD6E8FEB86659FD93ull; h ^= h >> 32;
  const double re = (double)(uint32_t)h * (2.0 / 4294967296.0) - 1.0;
  const double im = (double)(uint32_t)(h >> 32) * (2.0 / 4294967296.0) - 1.0;
  x[i] = make_cuDoubleComplex(re, im);
}

__global__ void hermitize_kernel(Z* __restrict__ a, int n) {   // in place: both triangles <- Hermitian part
  const int r = blockIdx.x * blockDim.x + threadIdx.x, c = blockIdx.y;
  if (r >= n || r < c) return;
  Z* m = a + (size_t)blockIdx.z * n * n;
  const Z x = m[r + (size_t)c * n], y = m[c + (size_t)r * n];
  const double re = 0.5 * (x.x + y.x), im = (r == c) ? 0.0 : 0.5 * (x.y - y.y);
  m[r + (size_t)c * n] = make_cuDoubleComplex(re, im);
  m[c + (size_t)r * n] = make_cuDoubleComplex(re, -im);
}

__global__ void pointers_kernel(Z** arr, Z* base, size_t stride, int n) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) arr[i] = base + (size_t)i * stride;
}

__global__ void or_ints_kernel(int* __restrict__ acc, const int* __restrict__ v, int n) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n && v[i] != 0) acc[i] = 1;
}

// res2[b][k] = | Y[:, col] - theta[col] X[:, col] |^2 for the k-th largest Ritz pair (col = p - 1 - k; ascending order)
__global__ void __launch_bounds__(256) residual_kernel(const Z* __restrict__ x, const Z* __restrict__ y, const double* __restrict__ theta,
                                                      int n, int p, double* __restrict__ res2, int m) {
  __shared__ double red[256];
  const int k = blockIdx.x, b = blockIdx.y, col = p - 1 - k;
  const Z* xc = x + ((size_t)b * p + col) * n;
  const Z* yc = y + ((size_t)b * p + col) * n;
  const double th = theta[(size_t)b * p + col];
  double acc = 0.0;
  for (int i = threadIdx.x; i < n; i += 256) {
    const double dr = yc[i].x - th * xc[i].x, di = yc[i].y - th * xc[i].y;
    acc += dr * dr + di * di;
  }
  red[threadIdx.x] = acc;
  __syncthreads();
  for (int w = 128; w > 0; w >>= 1) {
    if ((int)threadIdx.x < w) red[threadIdx.x] += red[threadIdx.x + w];
    __syncthreads();
  }
  if (threadIdx.x == 0) res2[(size_t)b * m + k] = red[0];
}

// verdict[b] = { max_k sqrt(res2) / theta_max , theta_min_of_block / theta_m }  (theta ascending: block minimum first)
__global__ void verdict_kernel(const double* __restrict__ res2, const double* __restrict__ theta, int p, int m, double* __restrict__ verdict) {
  const int b = blockIdx.x * blockDim.x + threadIdx.x;
  if (b >= (int)gridDim.x * (int)blockDim.x) return;
  const double* th = theta + (size_t)b * p;
  double worst = 0.0;
  for (int k = 0; k < m; ++k) worst = fmax(worst, res2[(size_t)b * m + k]);
  const double top = fmax(fabs(th[p - 1]), fabs(th[0]));
  const double th_m = th[p - m];                           // the smallest wanted Ritz value
  verdict[2 * b] = top > 0.0 ? sqrt(worst) / top : 0.0;
  // Powers of C^2 find the largest |lambda|, Algorithm 1 l.4 wants the largest lambda. The two agree only while no
  // negative eigenvalue is as large in magnitude as the smallest wanted one: otherwise the block fills with negative
  // pairs, wanted positive ones may lie outside it, and small residuals prove nothing (they show that the Ritz pairs
  // are eigenpairs, not that they are the m largest). th is ascending, so th[0] is the most negative value.
  // Verdict -1 = "not this solver's problem": the host hands the batch to the full eigensolve whatever the residuals.
  const bool negative_competes = !(th_m > 0.0) || (th[0] < 0.0 && -th[0] >= th_m);
  // otherwise: convergence ratio of the wanted pairs against the block's smallest Ritz value; >= 1 (or a slightly
  // negative spectrum end) means plain powers of C do not separate them
  verdict[2 * b + 1] = negative_competes ? -1.0 : (th[0] >= 0.0 ? th[0] / th_m : 2.0);
}

struct Ctx {
  GlueWork* g; cudaStream_t st; cublasHandle_t blas; cusolverDnHandle_t solver; cusolverDnParams_t params;
  int nb, n, p, m;
  Z *C, *X, *Y, *T, *Gm, *H;
  double* theta; double* res2; double* verdict;
  Z **pGm, **pX;
  int *info, *info_acc;
  int* launches;
};

const Z kOne = {1.0, 0.0}, kZero = {0.0, 0.0};

bool gemm(Ctx& c, cublasOperation_t ta, cublasOperation_t tb, int M, int N, int K, const Z* A, int lda, long long sa, const Z* B, int ldb,
          long long sb, Z* Cm, int ldc, long long sc) {
  return cublasZgemmStridedBatched(c.blas, ta, tb, M, N, K, &kOne, A, lda, sa, B, ldb, sb, &kZero, Cm, ldc, sc, c.nb) == CUBLAS_STATUS_SUCCESS;
}

// X <- X R^-1 with X^H X = R^H R (Cholesky-QR), in place
bool chol_qr(Ctx& c) {
  const int n = c.n, p = c.p;
  bool ok = gemm(c, CUBLAS_OP_C, CUBLAS_OP_N, p, p, n, c.X, n, (long long)n * p, c.X, n, (long long)n * p, c.Gm, p, (long long)p * p);
  hermitize_kernel<<<dim3((p + 127) / 128, p, c.nb), 128, 0, c.st>>>(c.Gm, p);
  ok = ok && cusolverDnZpotrfBatched(c.solver, CUBLAS_FILL_MODE_LOWER, p, c.pGm, p, c.info, c.nb) == CUSOLVER_STATUS_SUCCESS;
  or_ints_kernel<<<(c.nb + 127) / 128, 128, 0, c.st>>>(c.info_acc, c.info, c.nb);
  ok = ok && cublasZtrsmBatched(c.blas, CUBLAS_SIDE_RIGHT, CUBLAS_FILL_MODE_LOWER, CUBLAS_OP_C, CUBLAS_DIAG_NON_UNIT, n, p, &kOne, c.pGm, p,
                                c.pX, n, c.nb) == CUBLAS_STATUS_SUCCESS;
  *c.launches += 2;
  return ok;
}

// X <- orth(C^2 X)
bool power_block(Ctx& c) {
  const int n = c.n, p = c.p;
  const long long sC = (long long)n * n, sX = (long long)n * p;
  return gemm(c, CUBLAS_OP_N, CUBLAS_OP_N, n, p, n, c.C, n, sC, c.X, n, sX, c.Y, n, sX) &&
         gemm(c, CUBLAS_OP_N, CUBLAS_OP_N, n, p, n, c.C, n, sC, c.Y, n, sX, c.X, n, sX) && chol_qr(c);
}

// Rayleigh-Ritz on span(X) (X re-orthonormalised first): X <- Ritz vectors (ascending), Y <- C X, theta, residual verdicts
int rayleigh_ritz(Ctx& c) {
  const int n = c.n, p = c.p, m = c.m;
  const long long sC = (long long)n * n, sX = (long long)n * p, sH = (long long)p * p;
  bool ok = chol_qr(c);                                    // second pass: orthonormal to rounding
  ok = ok && gemm(c, CUBLAS_OP_N, CUBLAS_OP_N, n, p, n, c.C, n, sC, c.X, n, sX, c.Y, n, sX);
  ok = ok && gemm(c, CUBLAS_OP_C, CUBLAS_OP_N, p, p, n, c.X, n, sX, c.Y, n, sX, c.H, p, sH);
  if (!ok) return BB_ECUDA;
  hermitize_kernel<<<dim3((p + 127) / 128, p, c.nb), 128, 0, c.st>>>(c.H, p);
  size_t wdev = 0, whost = 0;
  if (cusolverDnXsyevBatched_bufferSize(c.solver, c.params, CUSOLVER_EIG_MODE_VECTOR, CUBLAS_FILL_MODE_LOWER, p, CUDA_C_64F, nullptr, p,
                                        CUDA_R_64F, nullptr, CUDA_C_64F, &wdev, &whost, c.nb) != CUSOLVER_STATUS_SUCCESS) return BB_ECUDA;
  int rc = bb_glue_grow(c.g, GB_WORK, wdev ? wdev : 16, c.st);
  if (rc != BB_OK) return rc;
  std::vector<char> hw(whost + 1);
  if (cusolverDnXsyevBatched(c.solver, c.params, CUSOLVER_EIG_MODE_VECTOR, CUBLAS_FILL_MODE_LOWER, p, CUDA_C_64F, c.H, p, CUDA_R_64F, c.theta,
                             CUDA_C_64F, bb_glue_buffer(c.g, GB_WORK), wdev, hw.data(), whost, c.info, c.nb) != CUSOLVER_STATUS_SUCCESS)
    return BB_ECUDA;
  or_ints_kernel<<<(c.nb + 127) / 128, 128, 0, c.st>>>(c.info_acc, c.info, c.nb);
  // X <- X Q, Y <- Y Q (T as scratch)
  ok = gemm(c, CUBLAS_OP_N, CUBLAS_OP_N, n, p, p, c.X, n, sX, c.H, p, sH, c.T, n, sX);
  BB_CUDA(cudaMemcpyAsync(c.X, c.T, (size_t)sX * c.nb * sizeof(Z), cudaMemcpyDeviceToDevice, c.st));
  ok = ok && gemm(c, CUBLAS_OP_N, CUBLAS_OP_N, n, p, p, c.Y, n, sX, c.H, p, sH, c.T, n, sX);
  if (!ok) return BB_ECUDA;
  residual_kernel<<<dim3(m, c.nb), 256, 0, c.st>>>(c.X, c.T, c.theta, n, p, c.res2, m);
  verdict_kernel<<<1, c.nb, 0, c.st>>>(c.res2, c.theta, p, m, c.verdict);
  *c.launches += 5;
  return BB_OK;
}

}  // namespace

int bb_subspace_top_eigs(GlueWork* g, cudaStream_t st, int nb, int n, int m, Z* C, const Z** vecs, int64_t* stride_v, const double** lams,
                         int64_t* stride_l, int* n_vec, int* used, int* launches) {
  *used = 0;
  const int p = m + (m > 32 ? m : 32);                     // block width: wanted pairs + as many guard vectors (>= 32)
  if (n < 256 || 2 * p > n || nb > 1024) return BB_OK;     // small problems: the full solve is cheap enough
  SubspaceWork** slot = bb_glue_subspace_slot(g);
  if (!*slot) { *slot = new (std::nothrow) SubspaceWork; if (!*slot) return BB_EALLOC; }
  SubspaceWork* w = *slot;
  if (w->cap < nb) {
    if (w->verdict_host) cudaFreeHost(w->verdict_host);
    if (w->info_host) cudaFreeHost(w->info_host);
    w->verdict_host = nullptr; w->info_host = nullptr; w->cap = 0;
    if (cudaMallocHost(&w->verdict_host, (size_t)2 * nb * sizeof(double)) != cudaSuccess ||
        cudaMallocHost(&w->info_host, (size_t)nb * sizeof(int)) != cudaSuccess) { cudaGetLastError(); return BB_EALLOC; }
    w->cap = nb;
  }
  const size_t zb = sizeof(Z), blk = (size_t)n * p * nb * zb;
  int rc;
  if ((rc = bb_glue_grow(g, GB_SUB0, blk, st)) || (rc = bb_glue_grow(g, GB_SUB1, blk, st)) || (rc = bb_glue_grow(g, GB_SUB2, blk, st)) ||
      (rc = bb_glue_grow(g, GB_SUB3, (size_t)2 * p * p * nb * zb, st)) ||
      (rc = bb_glue_grow(g, GB_SUB4, ((size_t)p * nb + (size_t)m * nb + 2 * (size_t)nb) * sizeof(double), st)) ||
      (rc = bb_glue_grow(g, GB_SUB5, (size_t)2 * nb * sizeof(void*) + (size_t)2 * nb * sizeof(int), st)))
    return rc;
  int nl = 0;
  Ctx c{};
  c.g = g; c.st = st; c.blas = bb_glue_blas(g); c.solver = bb_glue_solver(g); c.params = bb_glue_params(g);
  c.nb = nb; c.n = n; c.p = p; c.m = m; c.C = C;
  c.X = (Z*)bb_glue_buffer(g, GB_SUB0); c.Y = (Z*)bb_glue_buffer(g, GB_SUB1); c.T = (Z*)bb_glue_buffer(g, GB_SUB2);
  c.Gm = (Z*)bb_glue_buffer(g, GB_SUB3); c.H = c.Gm + (size_t)p * p * nb;
  c.theta = (double*)bb_glue_buffer(g, GB_SUB4); c.res2 = c.theta + (size_t)p * nb; c.verdict = c.res2 + (size_t)m * nb;
  c.pGm = (Z**)bb_glue_buffer(g, GB_SUB5); c.pX = c.pGm + nb;
  c.info = (int*)(c.pX + nb); c.info_acc = c.info + nb;
  c.launches = &nl;
  BB_CUDA(cudaMemsetAsync(c.info_acc, 0, (size_t)nb * sizeof(int), st));
  pointers_kernel<<<(nb + 127) / 128, 128, 0, st>>>(c.pGm, c.Gm, (size_t)p * p, nb);
  pointers_kernel<<<(nb + 127) / 128, 128, 0, st>>>(c.pX, c.X, (size_t)n * p, nb);
  const size_t count = (size_t)n * p * nb;
  start_block_kernel<<<(unsigned)((count + 255) / 256), 256, 0, st>>>(c.X, count);
  nl += 3;
  bool ok = chol_qr(c);
  // C^12 on the start block: enough for a decay of ~0.1 between the wanted pairs and the block's end (the wide-field
  // configs), so that the first Rayleigh-Ritz step usually is the last (each costs a 128 x 128 batched eigensolve)
  for (int s = 0; ok && s < 6; ++s) ok = power_block(c);
  if (!ok) { bb_note_cuda_error(cudaErrorUnknown, "subspace iteration (cuBLAS/cuSOLVER call)", __FILE__, __LINE__); return BB_ECUDA; }
  for (int round = 0; round < 2; ++round) {
    if ((rc = rayleigh_ritz(c)) != BB_OK) return rc;
    BB_CUDA(cudaMemcpyAsync(w->verdict_host, c.verdict, (size_t)2 * nb * sizeof(double), cudaMemcpyDeviceToHost, st));
    BB_CUDA(cudaMemcpyAsync(w->info_host, c.info_acc, (size_t)nb * sizeof(int), cudaMemcpyDeviceToHost, st));
    BB_CUDA(cudaStreamSynchronize(st));
    bool all = true, hopeless = false;
    int extra = 0;
    for (int b = 0; b < nb; ++b) {
      const double res = w->verdict_host[2 * b], rho = w->verdict_host[2 * b + 1];
      if (w->info_host[b] != 0 || !(res == res) || rho < 0.0) { hopeless = true; break; }   // rho < 0: indefinite, see verdict_kernel
      if (res <= kResidualTol) continue;
      all = false;
      if (!(rho < 0.95)) { hopeless = true; break; }
      // every C^2 block multiplies the error of the wanted pairs by about rho^2
      const int need = (int)std::ceil(std::log(0.1 * kResidualTol / res) / (2.0 * std::log(rho)));
      extra = need > extra ? need : extra;
    }
    if (hopeless || (!all && (round == 1 || extra > kMaxExtraSteps))) { if (launches) *launches += nl; return BB_OK; }   // *used = 0: full solve
    if (all) break;
    for (int s = 0; ok && s < extra; ++s) ok = power_block(c);
    if (!ok) { bb_note_cuda_error(cudaErrorUnknown, "subspace iteration (cuBLAS/cuSOLVER call)", __FILE__, __LINE__); return BB_ECUDA; }
  }
  *vecs = c.X; *stride_v = (int64_t)n * p; *lams = c.theta; *stride_l = p; *n_vec = p; *used = 1;
  if (launches) *launches += nl;
  return BB_OK;
}
