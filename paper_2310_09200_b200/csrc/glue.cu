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

int bb_launch_level_weights(const double* lambda_dev, int n_eig, const double* intervals_dev, int ld_int, int n_intervals,
                            FilterList filters, float* D_dev, int ldd, cudaStream_t st) {
  level_weights_kernel<<<dim3((n_eig + 127) / 128, n_intervals * filters.n), 128, 0, st>>>(lambda_dev, n_eig, intervals_dev,
                                                                                          ld_int, n_intervals, filters, D_dev, ldd);
  BB_CUDA(cudaGetLastError());
  return BB_OK;
}
