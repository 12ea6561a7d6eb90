// Device-side glue of Algorithm 1 lines 2-4, fp64, timed separately:
//   a0   Gram:   Psi_pq = sinc(2 |x_p - x_q| / lambda_w) (Eq. 11, normalized sinc), G = W^H Psi W (Eq. 24)
//   a0'  S v = lambda G v with V^H G V = I (Eq. 13): cusolverDnZhegvd, itype 1 (Cholesky of G,
//        reduction to standard form, Hermitian eigensolve, back-transform - the library primitive)
//   a0'' keep the n_eig largest (Alg. 1 l.4), B = W V (Eq. 22-24), cast to complex64;
//        level weights D[l,k] = lambda_k [min_l <= lambda_k <= max_l] (Alg. 1 l.7-8, closed intervals).
// fp64 rather than the paper's single precision: an fp32 eigensolve cannot
// reproduce level images when near-degenerate eigenvalues straddle the N_eig cut (Q14).
#include "internal.h"

#include <cublas_v2.h>
#include <cusolverDn.h>

struct GlueWork {
  cublasHandle_t blas = nullptr;
  cusolverDnHandle_t solver = nullptr;
  // scratch, grown on demand
  cuDoubleComplex *psi = nullptr, *w128 = nullptr, *t = nullptr, *g = nullptr, *s128 = nullptr, *vsel = nullptr, *b128 = nullptr;
  double* lam_all = nullptr;
  cuDoubleComplex* work = nullptr; int lwork = 0;
  int* info = nullptr; int* info_host = nullptr;
  int cap_ant = 0, cap_beam = 0;
  // batched path (bb_glue_eig_batch): one allocation per array, grown on demand
  cusolverDnParams_t params = nullptr;
  void* bat[10] = {nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr};
  size_t bat_bytes[10] = {0, 0, 0, 0, 0, 0, 0, 0, 0, 0};
};

namespace {

__global__ void gram_psi_kernel(const double* __restrict__ xyz, int ld, int n_ant, double wavelength,
                                cuDoubleComplex* __restrict__ psi) {
  const int p = blockIdx.x * blockDim.x + threadIdx.x, q = blockIdx.y;
  if (p >= n_ant) return;
  const double dx = xyz[p] - xyz[q], dy = xyz[p + ld] - xyz[q + ld], dz = xyz[p + 2 * (size_t)ld] - xyz[q + 2 * (size_t)ld];
  const double x = 2.0 * sqrt(dx * dx + dy * dy + dz * dz) / wavelength;   // 2 |b_pq|
  const double v = (x == 0.0) ? 1.0 : sinpi(x) / (M_PI * x);               // sin(pi x)/(pi x)
  psi[p + (size_t)q * n_ant] = make_cuDoubleComplex(v, 0.0);
}

__global__ void widen_kernel(const bb_c32* __restrict__ src, int ld, int rows, int cols, cuDoubleComplex* __restrict__ dst) {
  const int r = blockIdx.x * blockDim.x + threadIdx.x, c = blockIdx.y;
  if (r < rows && c < cols) dst[r + (size_t)c * rows] = make_cuDoubleComplex(src[r + (size_t)c * ld].re, src[r + (size_t)c * ld].im);
}

// dst = (src + src^H)/2 widened to complex128 (reading Q10: S is used as its Hermitian part)
__global__ void hermitian_part_kernel(const bb_c32* __restrict__ src, int ld, int n, cuDoubleComplex* __restrict__ dst) {
  const int r = blockIdx.x * blockDim.x + threadIdx.x, c = blockIdx.y;
  if (r >= n) return;
  const bb_c32 a = src[r + (size_t)c * ld], b = src[c + (size_t)r * ld];
  dst[r + (size_t)c * n] = make_cuDoubleComplex(0.5 * ((double)a.re + (double)b.re), 0.5 * ((double)a.im - (double)b.im));
}

__global__ void hermitian_fix_kernel(cuDoubleComplex* __restrict__ a, int n) {  // in place, lower -> both
  const int r = blockIdx.x * blockDim.x + threadIdx.x, c = blockIdx.y;
  if (r >= n || r < c) return;
  const cuDoubleComplex x = a[r + (size_t)c * n], y = a[c + (size_t)r * n];
  const double re = 0.5 * (x.x + y.x), im = (r == c) ? 0.0 : 0.5 * (x.y - y.y);
  a[r + (size_t)c * n] = make_cuDoubleComplex(re, im);
  a[c + (size_t)r * n] = make_cuDoubleComplex(re, -im);
}

// eigenvalues come out ascending: column k of the selection is eigenpair n_beam-1-k (largest first)
__global__ void select_kernel(const cuDoubleComplex* __restrict__ v, const double* __restrict__ lam_all, int n_beam,
                              int n_eig, cuDoubleComplex* __restrict__ vsel, double* __restrict__ lam) {
  const int r = blockIdx.x * blockDim.x + threadIdx.x, k = blockIdx.y;
  if (r < n_beam) vsel[r + (size_t)k * n_beam] = v[r + (size_t)(n_beam - 1 - k) * n_beam];
  if (r == 0) lam[k] = lam_all[n_beam - 1 - k];
}

__global__ void narrow_kernel(const cuDoubleComplex* __restrict__ src, int rows, int cols, bb_c32* __restrict__ dst) {
  const int r = blockIdx.x * blockDim.x + threadIdx.x, c = blockIdx.y;
  if (r < rows && c < cols) {
    const cuDoubleComplex x = src[r + (size_t)c * rows];
    dst[r + (size_t)c * rows] = bb_c32{(float)x.x, (float)x.y};
  }
}

__global__ void level_weights_kernel(const double* __restrict__ lam, int n_eig, const double* __restrict__ iv, int ld_int,
                                     int n_intervals, FilterList filters, float* __restrict__ D, int ldd) {
  const int k = blockIdx.x * blockDim.x + threadIdx.x, l = blockIdx.y;
  if (k < n_eig && l < n_intervals * filters.n) {
    const int f = l / n_intervals, i = l - f * n_intervals;
    const double x = lam[k];
    const float d = filters.kind[f] == BB_FILTER_STD ? 1.f : (float)x;      // Alg. 1 l.7: LSQ d = lambda, STD d = 1
    D[l + (size_t)k * ldd] = (x >= iv[i] && x <= iv[i + ld_int]) ? d : 0.f;
  }
}

__global__ void identity_kernel(cuDoubleComplex* __restrict__ a, int n) {
  const int r = blockIdx.x * blockDim.x + threadIdx.x, c = blockIdx.y;
  if (r < n) a[r + (size_t)c * n] = make_cuDoubleComplex(r == c ? 1.0 : 0.0, 0.0);
}

template <class T> int grow(T** p, size_t n) {
  cudaFree(*p); *p = nullptr;
  return cudaMalloc(p, n * sizeof(T)) == cudaSuccess ? BB_OK : BB_EALLOC;
}

}  // namespace

int bb_glue_create(GlueWork** out) {
  GlueWork* g = new (std::nothrow) GlueWork;
  if (!g) return BB_EALLOC;
  if (cublasCreate(&g->blas) != CUBLAS_STATUS_SUCCESS || cusolverDnCreate(&g->solver) != CUSOLVER_STATUS_SUCCESS ||
      cudaMalloc(&g->info, sizeof(int)) != cudaSuccess || cudaMallocHost(&g->info_host, sizeof(int)) != cudaSuccess) {
    bb_glue_destroy(g);
    bb_note_cuda_error(cudaErrorUnknown, "cuBLAS/cuSOLVER handle creation", __FILE__, __LINE__);
    return BB_ECUDA;
  }
  *out = g;
  return BB_OK;
}

void bb_glue_destroy(GlueWork* g) {
  if (!g) return;
  if (g->blas) cublasDestroy(g->blas);
  if (g->solver) cusolverDnDestroy(g->solver);
  cudaFree(g->psi); cudaFree(g->w128); cudaFree(g->t); cudaFree(g->g); cudaFree(g->s128); cudaFree(g->vsel);
  cudaFree(g->b128); cudaFree(g->lam_all); cudaFree(g->work); cudaFree(g->info);
  for (void* b : g->bat) cudaFree(b);
  if (g->params) cusolverDnDestroyParams(g->params);
  if (g->info_host) cudaFreeHost(g->info_host);
  cudaGetLastError();
  delete g;
}

int bb_glue_eig(GlueWork* g, cudaStream_t st, int n_ant, int n_beam, int n_eig, double wavelength, const bb_c32* W,
                int ldw, const bb_c32* S, int lds, const double* xyz, int ldxyz, double* lambda_dev, bb_c32* B_dev,
                cudaEvent_t ev_gram0, cudaEvent_t ev_gram1, cudaEvent_t ev_eig0, cudaEvent_t ev_eig1, int gram_mode) {
  cublasSetStream(g->blas, st);
  cusolverDnSetStream(g->solver, st);
  if (n_ant > g->cap_ant || n_beam > g->cap_beam) {
    BB_CUDA(cudaStreamSynchronize(st));
    const int ca = n_ant > g->cap_ant ? n_ant : g->cap_ant, cb = n_beam > g->cap_beam ? n_beam : g->cap_beam;
    if (grow(&g->psi, (size_t)ca * ca) || grow(&g->w128, (size_t)ca * cb) || grow(&g->t, (size_t)ca * cb) ||
        grow(&g->g, (size_t)cb * cb) || grow(&g->s128, (size_t)cb * cb) || grow(&g->vsel, (size_t)cb * cb) ||
        grow(&g->b128, (size_t)ca * cb) || grow(&g->lam_all, (size_t)cb)) { g->cap_ant = g->cap_beam = 0; return BB_EALLOC; }
    int lwork = 0;
    if (cusolverDnZhegvd_bufferSize(g->solver, CUSOLVER_EIG_TYPE_1, CUSOLVER_EIG_MODE_VECTOR, CUBLAS_FILL_MODE_LOWER, cb,
                                    g->s128, cb, g->g, cb, g->lam_all, &lwork) != CUSOLVER_STATUS_SUCCESS) return BB_ECUDA;
    if (grow(&g->work, (size_t)lwork)) return BB_EALLOC;
    g->lwork = lwork; g->cap_ant = ca; g->cap_beam = cb;
  }
  const dim3 blk(128);
  const cuDoubleComplex one = make_cuDoubleComplex(1, 0), zero = make_cuDoubleComplex(0, 0);

  // ---- a0: Gram
  if (ev_gram0) cudaEventRecord(ev_gram0, st);
  if (W) widen_kernel<<<dim3((n_ant + 127) / 128, n_beam), blk, 0, st>>>(W, ldw, n_ant, n_beam, g->w128);
  if (gram_mode == BB_GRAM_IDENTITY) {                    // G := I: eigendecomposition of the dirty image (Eq. 38-40)
    identity_kernel<<<dim3((n_beam + 127) / 128, n_beam), blk, 0, st>>>(g->g, n_beam);
  } else {
    gram_psi_kernel<<<dim3((n_ant + 127) / 128, n_ant), blk, 0, st>>>(xyz, ldxyz, n_ant, wavelength, W ? g->psi : g->g);
  }
  if (W && gram_mode != BB_GRAM_IDENTITY) {
    if (cublasZgemm(g->blas, CUBLAS_OP_N, CUBLAS_OP_N, n_ant, n_beam, n_ant, &one, g->psi, n_ant, g->w128, n_ant, &zero,
                    g->t, n_ant) != CUBLAS_STATUS_SUCCESS ||
        cublasZgemm(g->blas, CUBLAS_OP_C, CUBLAS_OP_N, n_beam, n_beam, n_ant, &one, g->w128, n_ant, g->t, n_ant, &zero,
                    g->g, n_beam) != CUBLAS_STATUS_SUCCESS) {
      bb_note_cuda_error(cudaErrorUnknown, "cublasZgemm (Gram)", __FILE__, __LINE__);
      return BB_ECUDA;
    }
    hermitian_fix_kernel<<<dim3((n_beam + 127) / 128, n_beam), blk, 0, st>>>(g->g, n_beam);
  }
  if (ev_gram1) cudaEventRecord(ev_gram1, st);

  // ---- a0': generalized Hermitian eigenproblem
  if (ev_eig0) cudaEventRecord(ev_eig0, st);
  hermitian_part_kernel<<<dim3((n_beam + 127) / 128, n_beam), blk, 0, st>>>(S, lds, n_beam, g->s128);
  int lwork = 0;
  cusolverDnZhegvd_bufferSize(g->solver, CUSOLVER_EIG_TYPE_1, CUSOLVER_EIG_MODE_VECTOR, CUBLAS_FILL_MODE_LOWER, n_beam,
                              g->s128, n_beam, g->g, n_beam, g->lam_all, &lwork);
  if (lwork > g->lwork) {
    BB_CUDA(cudaStreamSynchronize(st));
    if (grow(&g->work, (size_t)lwork)) return BB_EALLOC;
    g->lwork = lwork;
  }
  if (cusolverDnZhegvd(g->solver, CUSOLVER_EIG_TYPE_1, CUSOLVER_EIG_MODE_VECTOR, CUBLAS_FILL_MODE_LOWER, n_beam, g->s128,
                       n_beam, g->g, n_beam, g->lam_all, g->work, g->lwork, g->info) != CUSOLVER_STATUS_SUCCESS) {
    bb_note_cuda_error(cudaErrorUnknown, "cusolverDnZhegvd", __FILE__, __LINE__);
    return BB_ECUDA;
  }
  // ---- a0'': select, beamform, cast
  select_kernel<<<dim3((n_beam + 127) / 128, n_eig), blk, 0, st>>>(g->s128, g->lam_all, n_beam, n_eig, g->vsel, lambda_dev);
  if (W) {
    if (cublasZgemm(g->blas, CUBLAS_OP_N, CUBLAS_OP_N, n_ant, n_eig, n_beam, &one, g->w128, n_ant, g->vsel, n_beam, &zero,
                    g->b128, n_ant) != CUBLAS_STATUS_SUCCESS) {
      bb_note_cuda_error(cudaErrorUnknown, "cublasZgemm (B = W V)", __FILE__, __LINE__);
      return BB_ECUDA;
    }
    narrow_kernel<<<dim3((n_ant + 127) / 128, n_eig), blk, 0, st>>>(g->b128, n_ant, n_eig, B_dev);
  } else {
    narrow_kernel<<<dim3((n_ant + 127) / 128, n_eig), blk, 0, st>>>(g->vsel, n_ant, n_eig, B_dev);
  }
  if (ev_eig1) cudaEventRecord(ev_eig1, st);
  BB_CUDA(cudaGetLastError());
  // the solver's verdict decides whether this collect may touch the images: read it now
  BB_CUDA(cudaMemcpyAsync(g->info_host, g->info, sizeof(int), cudaMemcpyDeviceToHost, st));
  BB_CUDA(cudaStreamSynchronize(st));
  if (*g->info_host > n_beam) return BB_ENOTPOSDEF;   // leading minor of G not positive definite
  if (*g->info_host != 0) return BB_ENOCONV;
  return BB_OK;
}


// ---------------------------------------------------------------------------------------------------------
// Batched glue: the same steps for nb collects at once (blockIdx.z = collect). The Hermitian eigensolves run as
// ONE cusolverDnXsyevBatched call (measured on B200: 20 x 512^2 complex128 in 33.7 ms against 128.6 ms for 20
// Zheevd calls), the Cholesky factorisations as one potrfBatched, the reductions as trsmBatched.
namespace {

__global__ void gram_psi_batch_kernel(const double* __restrict__ xyz, int ld, int64_t stride, int n_ant,
                                      const double* __restrict__ wavelength, cuDoubleComplex* __restrict__ psi) {
  const int p = blockIdx.x * blockDim.x + threadIdx.x, q = blockIdx.y, b = blockIdx.z;
  if (p >= n_ant) return;
  const double* x = xyz + (size_t)b * stride;
  const double dx = x[p] - x[q], dy = x[p + ld] - x[q + ld], dz = x[p + 2 * (size_t)ld] - x[q + 2 * (size_t)ld];
  const double u = 2.0 * sqrt(dx * dx + dy * dy + dz * dz) / wavelength[b];
  const double v = (u == 0.0) ? 1.0 : sinpi(u) / (M_PI * u);
  psi[(size_t)b * n_ant * n_ant + p + (size_t)q * n_ant] = make_cuDoubleComplex(v, 0.0);
}

__global__ void widen_batch_kernel(const bb_c32* __restrict__ src, int ld, int64_t stride, int rows, int cols,
                                   cuDoubleComplex* __restrict__ dst) {
  const int r = blockIdx.x * blockDim.x + threadIdx.x, c = blockIdx.y, b = blockIdx.z;
  if (r >= rows) return;
  const bb_c32 x = src[(size_t)b * stride + r + (size_t)c * ld];
  dst[(size_t)b * rows * cols + r + (size_t)c * rows] = make_cuDoubleComplex(x.re, x.im);
}

__global__ void hermitian_part_batch_kernel(const bb_c32* __restrict__ src, int ld, int64_t stride, int n,
                                            cuDoubleComplex* __restrict__ dst) {
  const int r = blockIdx.x * blockDim.x + threadIdx.x, c = blockIdx.y, b = blockIdx.z;
  if (r >= n) return;
  const bb_c32* s = src + (size_t)b * stride;
  const bb_c32 x = s[r + (size_t)c * ld], y = s[c + (size_t)r * ld];
  dst[(size_t)b * n * n + r + (size_t)c * n] = make_cuDoubleComplex(0.5 * ((double)x.re + (double)y.re), 0.5 * ((double)x.im - (double)y.im));
}

__global__ void hermitian_fix_batch_kernel(cuDoubleComplex* __restrict__ a, int n) {
  const int r = blockIdx.x * blockDim.x + threadIdx.x, c = blockIdx.y;
  if (r >= n || r < c) return;
  cuDoubleComplex* m = a + (size_t)blockIdx.z * n * n;
  const cuDoubleComplex x = m[r + (size_t)c * n], y = m[c + (size_t)r * n];
  const double re = 0.5 * (x.x + y.x), im = (r == c) ? 0.0 : 0.5 * (x.y - y.y);
  m[r + (size_t)c * n] = make_cuDoubleComplex(re, im);
  m[c + (size_t)r * n] = make_cuDoubleComplex(re, -im);
}

__global__ void select_batch_kernel(const cuDoubleComplex* __restrict__ v, const double* __restrict__ lam_all, int n_beam, int n_eig,
                                    cuDoubleComplex* __restrict__ vsel, double* __restrict__ lam) {
  const int r = blockIdx.x * blockDim.x + threadIdx.x, k = blockIdx.y, b = blockIdx.z;
  if (r < n_beam)
    vsel[(size_t)b * n_beam * n_eig + r + (size_t)k * n_beam] = v[(size_t)b * n_beam * n_beam + r + (size_t)(n_beam - 1 - k) * n_beam];
  if (r == 0) lam[(size_t)b * n_eig + k] = lam_all[(size_t)b * n_beam + n_beam - 1 - k];
}

__global__ void narrow_batch_kernel(const cuDoubleComplex* __restrict__ src, int rows, int cols, bb_c32* __restrict__ dst) {
  const int r = blockIdx.x * blockDim.x + threadIdx.x, c = blockIdx.y;
  const size_t o = (size_t)blockIdx.z * rows * cols + r + (size_t)c * rows;
  if (r < rows) dst[o] = bb_c32{(float)src[o].x, (float)src[o].y};
}

__global__ void pointer_array_kernel(cuDoubleComplex** arr, cuDoubleComplex* base, size_t stride, int n) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) arr[i] = base + (size_t)i * stride;
}

int grow_bytes(GlueWork* g, int slot, size_t bytes) {
  if (bytes <= g->bat_bytes[slot]) return BB_OK;
  cudaFree(g->bat[slot]); g->bat[slot] = nullptr; g->bat_bytes[slot] = 0;
  if (cudaMalloc(&g->bat[slot], bytes) != cudaSuccess) { cudaGetLastError(); return BB_EALLOC; }
  g->bat_bytes[slot] = bytes;
  return BB_OK;
}

}  // namespace

// nb collects; W/S/xyz device pointers with element strides between collects (stride_w == 0: one W for all);
// wavelength_dev: nb doubles on the device. Outputs: lambda_dev [nb][n_eig] (descending), B_dev [nb][n_ant x n_eig].
int bb_glue_eig_batch(GlueWork* g, cudaStream_t st, int nb, int n_ant, int n_beam, int n_eig, const double* wavelength_dev,
                      const bb_c32* W, int ldw, int64_t stride_w, const bb_c32* S, int lds, int64_t stride_s, const double* xyz,
                      int ldxyz, int64_t stride_xyz, double* lambda_dev, bb_c32* B_dev, cudaEvent_t ev_gram0, cudaEvent_t ev_gram1,
                      cudaEvent_t ev_eig0, cudaEvent_t ev_eig1) {
  cublasSetStream(g->blas, st);
  cusolverDnSetStream(g->solver, st);
  if (!g->params && cusolverDnCreateParams(&g->params) != CUSOLVER_STATUS_SUCCESS) return BB_ECUDA;
  enum { PSI = 0, G = 1, W128 = 2, T = 3, S128 = 4, LAM = 5, VSEL = 6, B128 = 7, PTRS = 8, WORK = 9 };
  const size_t zb = sizeof(cuDoubleComplex), bb2 = (size_t)n_beam * n_beam, ab = (size_t)n_ant * n_beam;
  size_t wdev = 0, whost = 0;
  if (cusolverDnXsyevBatched_bufferSize(g->solver, g->params, CUSOLVER_EIG_MODE_VECTOR, CUBLAS_FILL_MODE_LOWER, n_beam, CUDA_C_64F,
                                        nullptr, n_beam, CUDA_R_64F, nullptr, CUDA_C_64F, &wdev, &whost, nb) != CUSOLVER_STATUS_SUCCESS) {
    bb_note_cuda_error(cudaErrorUnknown, "cusolverDnXsyevBatched_bufferSize", __FILE__, __LINE__);
    return BB_ECUDA;
  }
  BB_CUDA(cudaStreamSynchronize(st));                      // scratch may be regrown below
  if (grow_bytes(g, G, bb2 * nb * zb) || grow_bytes(g, S128, bb2 * nb * zb) || grow_bytes(g, LAM, (size_t)n_beam * nb * sizeof(double)) ||
      grow_bytes(g, VSEL, (size_t)n_beam * n_eig * nb * zb) || grow_bytes(g, PTRS, (size_t)2 * nb * sizeof(void*) + (size_t)2 * nb * sizeof(int)) ||
      grow_bytes(g, WORK, wdev ? wdev : 16) ||
      (W && (grow_bytes(g, PSI, (size_t)n_ant * n_ant * nb * zb) || grow_bytes(g, W128, ab * nb * zb) || grow_bytes(g, T, ab * nb * zb) ||
             grow_bytes(g, B128, (size_t)n_ant * n_eig * nb * zb))))
    return BB_EALLOC;
  std::vector<char> host_work(whost + 1);
  cuDoubleComplex* gG = (cuDoubleComplex*)g->bat[G];
  cuDoubleComplex* gS = (cuDoubleComplex*)g->bat[S128];
  cuDoubleComplex* gPsi = (cuDoubleComplex*)g->bat[PSI];
  cuDoubleComplex* gW = (cuDoubleComplex*)g->bat[W128];
  cuDoubleComplex* gT = (cuDoubleComplex*)g->bat[T];
  cuDoubleComplex* gV = (cuDoubleComplex*)g->bat[VSEL];
  cuDoubleComplex* gB = (cuDoubleComplex*)g->bat[B128];
  double* gLam = (double*)g->bat[LAM];
  cuDoubleComplex** pG = (cuDoubleComplex**)g->bat[PTRS];
  cuDoubleComplex** pS = pG + nb;
  int* info_potrf = (int*)(pS + nb);
  int* info_syev = info_potrf + nb;
  const dim3 blk(128);
  const cuDoubleComplex one = make_cuDoubleComplex(1, 0), zero = make_cuDoubleComplex(0, 0);
  const int wb = stride_w ? nb : 1;                        // number of distinct W matrices

  // ---- a0: Gram
  if (ev_gram0) cudaEventRecord(ev_gram0, st);
  gram_psi_batch_kernel<<<dim3((n_ant + 127) / 128, n_ant, nb), blk, 0, st>>>(xyz, ldxyz, stride_xyz, n_ant, wavelength_dev, W ? gPsi : gG);
  if (W) {
    widen_batch_kernel<<<dim3((n_ant + 127) / 128, n_beam, wb), blk, 0, st>>>(W, ldw, stride_w, n_ant, n_beam, gW);
    const long long sW = stride_w ? (long long)ab : 0;
    if (cublasZgemmStridedBatched(g->blas, CUBLAS_OP_N, CUBLAS_OP_N, n_ant, n_beam, n_ant, &one, gPsi, n_ant, (long long)n_ant * n_ant,
                                  gW, n_ant, sW, &zero, gT, n_ant, (long long)ab, nb) != CUBLAS_STATUS_SUCCESS ||
        cublasZgemmStridedBatched(g->blas, CUBLAS_OP_C, CUBLAS_OP_N, n_beam, n_beam, n_ant, &one, gW, n_ant, sW, gT, n_ant, (long long)ab,
                                  &zero, gG, n_beam, (long long)bb2, nb) != CUBLAS_STATUS_SUCCESS) {
      bb_note_cuda_error(cudaErrorUnknown, "cublasZgemmStridedBatched (Gram)", __FILE__, __LINE__);
      return BB_ECUDA;
    }
    hermitian_fix_batch_kernel<<<dim3((n_beam + 127) / 128, n_beam, nb), blk, 0, st>>>(gG, n_beam);
  }
  if (ev_gram1) cudaEventRecord(ev_gram1, st);

  // ---- a0': G = L L^H, C = L^-1 S L^-H, C = Q diag(lambda) Q^H, V = L^-H Q
  if (ev_eig0) cudaEventRecord(ev_eig0, st);
  hermitian_part_batch_kernel<<<dim3((n_beam + 127) / 128, n_beam, nb), blk, 0, st>>>(S, lds, stride_s, n_beam, gS);
  pointer_array_kernel<<<(nb + 127) / 128, 128, 0, st>>>(pG, gG, bb2, nb);
  pointer_array_kernel<<<(nb + 127) / 128, 128, 0, st>>>(pS, gS, bb2, nb);
  bool ok = cusolverDnZpotrfBatched(g->solver, CUBLAS_FILL_MODE_LOWER, n_beam, pG, n_beam, info_potrf, nb) == CUSOLVER_STATUS_SUCCESS;
  ok = ok && cublasZtrsmBatched(g->blas, CUBLAS_SIDE_LEFT, CUBLAS_FILL_MODE_LOWER, CUBLAS_OP_N, CUBLAS_DIAG_NON_UNIT, n_beam, n_beam, &one,
                                pG, n_beam, pS, n_beam, nb) == CUBLAS_STATUS_SUCCESS;
  ok = ok && cublasZtrsmBatched(g->blas, CUBLAS_SIDE_RIGHT, CUBLAS_FILL_MODE_LOWER, CUBLAS_OP_C, CUBLAS_DIAG_NON_UNIT, n_beam, n_beam, &one,
                                pG, n_beam, pS, n_beam, nb) == CUBLAS_STATUS_SUCCESS;
  if (ok) hermitian_fix_batch_kernel<<<dim3((n_beam + 127) / 128, n_beam, nb), blk, 0, st>>>(gS, n_beam);
  ok = ok && cusolverDnXsyevBatched(g->solver, g->params, CUSOLVER_EIG_MODE_VECTOR, CUBLAS_FILL_MODE_LOWER, n_beam, CUDA_C_64F, gS, n_beam,
                                    CUDA_R_64F, gLam, CUDA_C_64F, g->bat[WORK], wdev, host_work.data(), whost, info_syev, nb) ==
                 CUSOLVER_STATUS_SUCCESS;
  ok = ok && cublasZtrsmBatched(g->blas, CUBLAS_SIDE_LEFT, CUBLAS_FILL_MODE_LOWER, CUBLAS_OP_C, CUBLAS_DIAG_NON_UNIT, n_beam, n_beam, &one,
                                pG, n_beam, pS, n_beam, nb) == CUBLAS_STATUS_SUCCESS;
  if (!ok) { bb_note_cuda_error(cudaErrorUnknown, "batched Cholesky / trsm / syev", __FILE__, __LINE__); return BB_ECUDA; }
  // ---- a0'': select, beamform, cast
  select_batch_kernel<<<dim3((n_beam + 127) / 128, n_eig, nb), blk, 0, st>>>(gS, gLam, n_beam, n_eig, gV, lambda_dev);
  if (W) {
    if (cublasZgemmStridedBatched(g->blas, CUBLAS_OP_N, CUBLAS_OP_N, n_ant, n_eig, n_beam, &one, gW, n_ant, stride_w ? (long long)ab : 0, gV,
                                  n_beam, (long long)n_beam * n_eig, &zero, gB, n_ant, (long long)n_ant * n_eig, nb) != CUBLAS_STATUS_SUCCESS) {
      bb_note_cuda_error(cudaErrorUnknown, "cublasZgemmStridedBatched (B = W V)", __FILE__, __LINE__);
      return BB_ECUDA;
    }
    narrow_batch_kernel<<<dim3((n_ant + 127) / 128, n_eig, nb), blk, 0, st>>>(gB, n_ant, n_eig, B_dev);
  } else {
    narrow_batch_kernel<<<dim3((n_ant + 127) / 128, n_eig, nb), blk, 0, st>>>(gV, n_ant, n_eig, B_dev);
  }
  if (ev_eig1) cudaEventRecord(ev_eig1, st);
  BB_CUDA(cudaGetLastError());
  std::vector<int> info_host(2 * (size_t)nb);
  BB_CUDA(cudaMemcpyAsync(info_host.data(), info_potrf, 2 * (size_t)nb * sizeof(int), cudaMemcpyDeviceToHost, st));
  BB_CUDA(cudaStreamSynchronize(st));
  for (int b = 0; b < nb; ++b) {
    if (info_host[b] != 0) return BB_ENOTPOSDEF;
    if (info_host[nb + b] != 0) return BB_ENOCONV;
  }
  return BB_OK;
}

int bb_launch_level_weights(const double* lambda_dev, int n_eig, const double* intervals_dev, int ld_int, int n_intervals,
                            FilterList filters, float* D_dev, int ldd, cudaStream_t st) {
  level_weights_kernel<<<dim3((n_eig + 127) / 128, n_intervals * filters.n), 128, 0, st>>>(lambda_dev, n_eig, intervals_dev,
                                                                                          ld_int, n_intervals, filters, D_dev, ldd);
  BB_CUDA(cudaGetLastError());
  return BB_OK;
}
