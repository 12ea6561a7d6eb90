// Device-side glue of Algorithm 1 lines 2-4, fp64, batched over collects, timed separately:
//   a0   Gram:   Psi_pq = sinc(2 |x_p - x_q| / lambda_w) (Eq. 11, normalized sinc), G = W^H Psi W (Eq. 24)
//   a0'  S v = lambda G v with V^H G V = I (Eq. 13): G = L L^H (potrfBatched), C = L^-1 S L^-H (trsmBatched),
//        Hermitian eigensolve of C, V = L^-H Q
//   a0'' keep the n_eig largest (Alg. 1 l.4), B = W V (Eq. 22-24), cast to complex64;
//        level weights D[l,k] = d_f(lambda_k) [min_l <= lambda_k <= max_l] (Alg. 1 l.7-8, closed intervals).
// Every step takes nb collects at once (blockIdx.z = collect, strided-batched cuBLAS, batched cuSOLVER): the
// eigenproblem "must be repeated for each timestep t and frequency band f" and a single 512 x 512
// solve leaves most of the GPU idle. Nothing here synchronises with the host: solver verdicts stay on the device
// (info words), a failed collect gets all-zero level weights (so it leaves the images unchanged) and raises a
// sticky flag that bb_synth_get reports.
// fp64 rather than the paper's single precision: an fp32 eigensolve cannot reproduce level images
// when near-degenerate eigenvalues straddle the N_eig cut (Q14).
#include "glue_internal.h"

struct GlueWork {
  cublasHandle_t blas = nullptr;
  cusolverDnHandle_t solver = nullptr;
  cusolverDnParams_t params = nullptr;
  void* bat[kGlueBuffers] = {};          // scratch, one allocation per array, grown on demand
  size_t bat_bytes[kGlueBuffers] = {};
  std::vector<char> host_work;
  SubspaceWork* sub = nullptr;           // leading-eigenpair solver (eig_subspace.cu)
};

namespace {

typedef cuDoubleComplex Z;

__global__ void gram_psi_kernel(const double* __restrict__ xyz, int ld, int64_t stride, int n_ant,
                                const double* __restrict__ wavelength, int64_t stride_wl, Z* __restrict__ psi) {
  const int p = blockIdx.x * blockDim.x + threadIdx.x, q = blockIdx.y, b = blockIdx.z;
  if (p >= n_ant) return;
  const double* x = xyz + (size_t)b * stride;
  const double dx = x[p] - x[q], dy = x[p + ld] - x[q + ld], dz = x[p + 2 * (size_t)ld] - x[q + 2 * (size_t)ld];
  const double u = 2.0 * sqrt(dx * dx + dy * dy + dz * dz) / wavelength[(size_t)b * stride_wl];   // 2 |b_pq|
  const double v = (u == 0.0) ? 1.0 : sinpi(u) / (M_PI * u);                                       // sin(pi u)/(pi u)
  psi[(size_t)b * n_ant * n_ant + p + (size_t)q * n_ant] = make_cuDoubleComplex(v, 0.0);
}

__global__ void widen_kernel(const bb_c32* __restrict__ src, int ld, int64_t stride, int rows, int cols, Z* __restrict__ dst) {
  const int r = blockIdx.x * blockDim.x + threadIdx.x, c = blockIdx.y, b = blockIdx.z;
  if (r >= rows) return;
  const bb_c32 x = src[(size_t)b * stride + r + (size_t)c * ld];
  dst[(size_t)b * rows * cols + r + (size_t)c * rows] = make_cuDoubleComplex(x.re, x.im);
}

// dst = (src + src^H)/2 widened to complex128 (reading Q10: S is used as its Hermitian part); with uniform weighting
// (Section 3.5) every visibility is divided by the sampling density of its uv cell
struct UvArgs { UvGridView g; const double* xyz; int ldxyz; int64_t stride_xyz; const double* wavelength; int64_t stride_wl; int on; };
__global__ void hermitian_part_kernel(const bb_c32* __restrict__ src, int ld, int64_t stride, int n, Z* __restrict__ dst, UvArgs uv) {
  const int r = blockIdx.x * blockDim.x + threadIdx.x, c = blockIdx.y, b = blockIdx.z;
  if (r >= n) return;
  const bb_c32* s = src + (size_t)b * stride;
  const bb_c32 x = s[r + (size_t)c * ld], y = s[c + (size_t)r * ld];
  double w = 0.5;
  if (uv.on) {
    const int d = uv.g.count[bb_uv_cell(uv.g, uv.xyz + (size_t)b * uv.stride_xyz, uv.ldxyz, r, c, uv.wavelength[(size_t)b * uv.stride_wl])];
    w = 0.5 / (double)(d > 0 ? d : 1);
  }
  dst[(size_t)b * n * n + r + (size_t)c * n] = make_cuDoubleComplex(w * ((double)x.re + (double)y.re), w * ((double)x.im - (double)y.im));
}

__global__ void hermitian_fix_kernel(Z* __restrict__ a, int n) {  // in place: both triangles <- Hermitian part
  const int r = blockIdx.x * blockDim.x + threadIdx.x, c = blockIdx.y;
  if (r >= n || r < c) return;
  Z* m = a + (size_t)blockIdx.z * n * n;
  const Z x = m[r + (size_t)c * n], y = m[c + (size_t)r * n];
  const double re = 0.5 * (x.x + y.x), im = (r == c) ? 0.0 : 0.5 * (x.y - y.y);
  m[r + (size_t)c * n] = make_cuDoubleComplex(re, im);
  m[c + (size_t)r * n] = make_cuDoubleComplex(re, -im);
}

// Column k of the selection is the k-th largest eigenpair (Alg. 1 l.4) of the solver's output, n_vec pairs in
// ascending order (the full spectrum, or the Ritz pairs of the leading block): source column n_vec - 1 - k.
__global__ void select_kernel(const Z* __restrict__ v, int64_t stride_v, const double* __restrict__ lam_all, int64_t stride_l,
                              int n_beam, int n_vec, int ascending, int n_eig, Z* __restrict__ vsel, double* __restrict__ lam,
                              int64_t stride_lam) {
  const int r = blockIdx.x * blockDim.x + threadIdx.x, k = blockIdx.y, b = blockIdx.z;
  const int src = ascending ? n_vec - 1 - k : k;
  if (r < n_beam) vsel[(size_t)b * n_beam * n_eig + r + (size_t)k * n_beam] = v[(size_t)b * stride_v + r + (size_t)src * n_beam];
  if (r == 0) lam[(size_t)b * stride_lam + k] = lam_all[(size_t)b * stride_l + src];
}

// cast to complex64; a collect whose factorisation or eigensolve failed gets B = 0 (its eigenvectors may hold NaN, and
// 0 weight x NaN would still poison the images)
__global__ void narrow_kernel(const Z* __restrict__ src, int rows, int cols, bb_c32* __restrict__ dst, int64_t stride_dst,
                              const int* __restrict__ info_chol, const int* __restrict__ info_eig) {
  const int r = blockIdx.x * blockDim.x + threadIdx.x, c = blockIdx.y, b = blockIdx.z;
  if (r >= rows) return;
  const bool bad = info_chol[b] != 0 || info_eig[b] != 0;
  const Z x = src[(size_t)b * rows * cols + r + (size_t)c * rows];
  dst[(size_t)b * stride_dst + r + (size_t)c * rows] = bad ? bb_c32{0.f, 0.f} : bb_c32{(float)x.x, (float)x.y};
}

__global__ void pointer_array_kernel(Z** arr, Z* base, size_t stride, int n) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) arr[i] = base + (size_t)i * stride;
}

__global__ void zero_ints_kernel(int* p, int n) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) p[i] = 0;
}

// D[f * n_intervals + i, k] = d_f(lambda_k) [min_i <= lambda_k <= max_i]; all zero (and a sticky status flag) when
// the Cholesky factorisation or the eigensolve of this collect failed.
__global__ void level_weights_kernel(const double* __restrict__ lam, int n_eig, const double* __restrict__ iv, int ld_int,
                                     int n_intervals, FilterList filters, float* __restrict__ D, int ldd,
                                     const int* __restrict__ info_chol, const int* __restrict__ info_eig, int* __restrict__ status) {
  const int k = blockIdx.x * blockDim.x + threadIdx.x, l = blockIdx.y;
  const int bad_chol = info_chol ? *info_chol : 0, bad_eig = info_eig ? *info_eig : 0;
  if (k == 0 && l == 0 && status && (bad_chol || bad_eig)) atomicOr(status, bad_chol ? BB_FLAG_NOTPOSDEF : BB_FLAG_NOCONV);
  if (k < n_eig && l < n_intervals * filters.n) {
    const int f = l / n_intervals, i = l - f * n_intervals;
    const double x = lam[k];
    const float d = filters.kind[f] == BB_FILTER_STD ? 1.f : (float)x;      // Alg. 1 l.7: LSQ d = lambda, STD d = 1
    D[l + (size_t)k * ldd] = (!bad_chol && !bad_eig && x >= iv[i] && x <= iv[i + ld_int]) ? d : 0.f;
  }
}

}  // namespace

int bb_glue_grow(GlueWork* g, int slot, size_t bytes, cudaStream_t st) {
  if (bytes <= g->bat_bytes[slot]) return BB_OK;
  BB_CUDA(cudaStreamSynchronize(st));                      // work in flight may still use the old buffer
  cudaFree(g->bat[slot]); g->bat[slot] = nullptr; g->bat_bytes[slot] = 0;
  if (cudaMalloc(&g->bat[slot], bytes) != cudaSuccess) { cudaGetLastError(); return BB_EALLOC; }
  g->bat_bytes[slot] = bytes;
  return BB_OK;
}
void* bb_glue_buffer(GlueWork* g, int slot) { return g->bat[slot]; }
cublasHandle_t bb_glue_blas(GlueWork* g) { return g->blas; }
cusolverDnHandle_t bb_glue_solver(GlueWork* g) { return g->solver; }
cusolverDnParams_t bb_glue_params(GlueWork* g) { return g->params; }
SubspaceWork** bb_glue_subspace_slot(GlueWork* g) { return &g->sub; }

int bb_glue_create(GlueWork** out) {
  GlueWork* g = new (std::nothrow) GlueWork;
  if (!g) return BB_EALLOC;
  if (cublasCreate(&g->blas) != CUBLAS_STATUS_SUCCESS || cusolverDnCreate(&g->solver) != CUSOLVER_STATUS_SUCCESS ||
      cusolverDnCreateParams(&g->params) != CUSOLVER_STATUS_SUCCESS) {
    bb_glue_destroy(g);
    bb_note_cuda_error(cudaErrorUnknown, "cuBLAS/cuSOLVER handle creation", __FILE__, __LINE__);
    return BB_ECUDA;
  }
  *out = g;
  return BB_OK;
}

void bb_glue_destroy(GlueWork* g) {
  if (!g) return;
  bb_subspace_destroy(g->sub);
  if (g->blas) cublasDestroy(g->blas);
  if (g->solver) cusolverDnDestroy(g->solver);
  if (g->params) cusolverDnDestroyParams(g->params);
  for (void* b : g->bat) cudaFree(b);
  cudaGetLastError();
  delete g;
}

// Full Hermitian eigensolve of nb matrices (n x n, complex128, contiguous, overwritten by the eigenvectors);
// eigenvalues ascending in lam [nb][n]; info [nb] on the device.
static int eig_full(GlueWork* g, cudaStream_t st, int nb, int n, Z* C, double* lam, int* info) {
  size_t wdev = 0, whost = 0;
  if (cusolverDnXsyevBatched_bufferSize(g->solver, g->params, CUSOLVER_EIG_MODE_VECTOR, CUBLAS_FILL_MODE_LOWER, n, CUDA_C_64F, nullptr, n,
                                        CUDA_R_64F, nullptr, CUDA_C_64F, &wdev, &whost, nb) != CUSOLVER_STATUS_SUCCESS) {
    bb_note_cuda_error(cudaErrorUnknown, "cusolverDnXsyevBatched_bufferSize", __FILE__, __LINE__);
    return BB_ECUDA;
  }
  int rc = bb_glue_grow(g, GB_WORK, wdev ? wdev : 16, st);
  if (rc != BB_OK) return rc;
  if (g->host_work.size() < whost + 1) g->host_work.resize(whost + 1);
  if (cusolverDnXsyevBatched(g->solver, g->params, CUSOLVER_EIG_MODE_VECTOR, CUBLAS_FILL_MODE_LOWER, n, CUDA_C_64F, C, n, CUDA_R_64F, lam,
                             CUDA_C_64F, g->bat[GB_WORK], wdev, g->host_work.data(), whost, info, nb) != CUSOLVER_STATUS_SUCCESS) {
    bb_note_cuda_error(cudaErrorUnknown, "cusolverDnXsyevBatched", __FILE__, __LINE__);
    return BB_ECUDA;
  }
  return BB_OK;
}

// nb collects; W/S/xyz/wavelength device pointers with element strides between collects (stride_w == 0: one W for
// all). Outputs: lambda_dev [nb] (stride_lam, descending), B_dev [nb] (stride_b, n_ant x n_eig complex64, ld n_ant),
// info_dev [2 nb]: Cholesky verdicts then eigensolver verdicts (0 = fine). Asynchronous on st.
int bb_glue_eig_batch(GlueWork* g, cudaStream_t st, const GlueBatch& a, int* launches) {
  const int nb = a.nb, n_ant = a.n_ant, n_beam = a.n_beam, n_eig = a.n_eig;
  cublasSetStream(g->blas, st);
  cusolverDnSetStream(g->solver, st);
  const size_t zb = sizeof(Z), bb2 = (size_t)n_beam * n_beam, ab = (size_t)n_ant * n_beam;
  const bool sinc = a.gram_mode != BB_GRAM_IDENTITY;
  const bool has_w = a.W != nullptr;
  int rc;
  if ((rc = bb_glue_grow(g, GB_S, bb2 * nb * zb, st)) || (rc = bb_glue_grow(g, GB_LAM, (size_t)n_beam * nb * sizeof(double), st)) ||
      (rc = bb_glue_grow(g, GB_VSEL, (size_t)n_beam * n_eig * nb * zb, st)) ||
      (rc = bb_glue_grow(g, GB_PTRS, (size_t)2 * nb * sizeof(void*), st)))
    return rc;
  if (sinc && (rc = bb_glue_grow(g, GB_G, bb2 * nb * zb, st))) return rc;
  if (has_w && ((rc = bb_glue_grow(g, GB_W, ab * nb * zb, st)) || (rc = bb_glue_grow(g, GB_B, (size_t)n_ant * n_eig * nb * zb, st)))) return rc;
  if (has_w && sinc && ((rc = bb_glue_grow(g, GB_PSI, (size_t)n_ant * n_ant * nb * zb, st)) || (rc = bb_glue_grow(g, GB_T, ab * nb * zb, st)))) return rc;
  Z* gG = (Z*)g->bat[GB_G];
  Z* gS = (Z*)g->bat[GB_S];
  Z* gPsi = (Z*)g->bat[GB_PSI];
  Z* gW = (Z*)g->bat[GB_W];
  Z* gT = (Z*)g->bat[GB_T];
  Z* gV = (Z*)g->bat[GB_VSEL];
  Z* gB = (Z*)g->bat[GB_B];
  double* gLam = (double*)g->bat[GB_LAM];
  Z** pG = (Z**)g->bat[GB_PTRS];
  Z** pS = pG + nb;
  int* info_chol = a.info_dev;
  int* info_eig = a.info_dev + nb;
  const dim3 blk(128);
  const Z one = make_cuDoubleComplex(1, 0), zero = make_cuDoubleComplex(0, 0);
  const int wb = a.stride_w ? nb : 1;                      // number of distinct W matrices
  const long long sW = a.stride_w ? (long long)ab : 0;
  int nl = 0;

  // ---- a0: Gram
  if (a.ev_gram0) cudaEventRecord(a.ev_gram0, st);
  zero_ints_kernel<<<(2 * nb + 127) / 128, 128, 0, st>>>(a.info_dev, 2 * nb); ++nl;
  if (has_w) { widen_kernel<<<dim3((n_ant + 127) / 128, n_beam, wb), blk, 0, st>>>(a.W, a.ldw, a.stride_w, n_ant, n_beam, gW); ++nl; }
  if (sinc) {
    gram_psi_kernel<<<dim3((n_ant + 127) / 128, n_ant, nb), blk, 0, st>>>(a.xyz, a.ldxyz, a.stride_xyz, n_ant, a.wavelength, a.stride_wl,
                                                                         has_w ? gPsi : gG); ++nl;
    if (has_w) {
      if (cublasZgemmStridedBatched(g->blas, CUBLAS_OP_N, CUBLAS_OP_N, n_ant, n_beam, n_ant, &one, gPsi, n_ant, (long long)n_ant * n_ant,
                                    gW, n_ant, sW, &zero, gT, n_ant, (long long)ab, nb) != CUBLAS_STATUS_SUCCESS ||
          cublasZgemmStridedBatched(g->blas, CUBLAS_OP_C, CUBLAS_OP_N, n_beam, n_beam, n_ant, &one, gW, n_ant, sW, gT, n_ant, (long long)ab,
                                    &zero, gG, n_beam, (long long)bb2, nb) != CUBLAS_STATUS_SUCCESS) {
        bb_note_cuda_error(cudaErrorUnknown, "cublasZgemmStridedBatched (Gram)", __FILE__, __LINE__);
        return BB_ECUDA;
      }
      hermitian_fix_kernel<<<dim3((n_beam + 127) / 128, n_beam, nb), blk, 0, st>>>(gG, n_beam); ++nl;
    }
  }
  if (a.ev_gram1) cudaEventRecord(a.ev_gram1, st);

  // ---- a0': G = L L^H, C = L^-1 S L^-H, C = Q diag(lambda) Q^H, V = L^-H Q   (G := I: C = S, V = Q, Eq. 38-40)
  if (a.ev_eig0) cudaEventRecord(a.ev_eig0, st);
  UvArgs uv{};
  if (a.uv) { uv.g = *a.uv; uv.xyz = a.xyz; uv.ldxyz = a.ldxyz; uv.stride_xyz = a.stride_xyz; uv.wavelength = a.wavelength; uv.stride_wl = a.stride_wl; uv.on = 1; }
  hermitian_part_kernel<<<dim3((n_beam + 127) / 128, n_beam, nb), blk, 0, st>>>(a.S, a.lds, a.stride_s, n_beam, gS, uv); ++nl;
  bool ok = true;
  if (sinc) {
    pointer_array_kernel<<<(nb + 127) / 128, 128, 0, st>>>(pG, gG, bb2, nb);
    pointer_array_kernel<<<(nb + 127) / 128, 128, 0, st>>>(pS, gS, bb2, nb);
    nl += 2;
    ok = cusolverDnZpotrfBatched(g->solver, CUBLAS_FILL_MODE_LOWER, n_beam, pG, n_beam, info_chol, nb) == CUSOLVER_STATUS_SUCCESS;
    ok = ok && cublasZtrsmBatched(g->blas, CUBLAS_SIDE_LEFT, CUBLAS_FILL_MODE_LOWER, CUBLAS_OP_N, CUBLAS_DIAG_NON_UNIT, n_beam, n_beam, &one,
                                  pG, n_beam, pS, n_beam, nb) == CUBLAS_STATUS_SUCCESS;
    ok = ok && cublasZtrsmBatched(g->blas, CUBLAS_SIDE_RIGHT, CUBLAS_FILL_MODE_LOWER, CUBLAS_OP_C, CUBLAS_DIAG_NON_UNIT, n_beam, n_beam, &one,
                                  pG, n_beam, pS, n_beam, nb) == CUBLAS_STATUS_SUCCESS;
    if (ok) { hermitian_fix_kernel<<<dim3((n_beam + 127) / 128, n_beam, nb), blk, 0, st>>>(gS, n_beam); ++nl; }
  }
  if (!ok) { bb_note_cuda_error(cudaErrorUnknown, "batched Cholesky / trsm", __FILE__, __LINE__); return BB_ECUDA; }
  // leading n_eig pairs by block subspace iteration where that pays (large n_beam, n_eig << n_beam, decaying
  // spectrum); otherwise, or when it does not converge, the full batched eigensolve
  int n_vec = n_beam;
  const int ascending = 1;                                 // both solvers return eigenvalues in ascending order
  const Z* vecs = gS;
  const double* lams = gLam;
  int64_t stride_v = (int64_t)bb2, stride_l = n_beam;
  int used_subspace = 0;
  if ((rc = bb_subspace_top_eigs(g, st, nb, n_beam, n_eig, gS, &vecs, &stride_v, &lams, &stride_l, &n_vec, &used_subspace, &nl)) != BB_OK) return rc;
  if (!used_subspace && (rc = eig_full(g, st, nb, n_beam, gS, gLam, info_eig)) != BB_OK) return rc;
  // ---- a0'': select, back-transform, beamform, cast
  select_kernel<<<dim3((n_beam + 127) / 128, n_eig, nb), blk, 0, st>>>(vecs, stride_v, lams, stride_l, n_beam, n_vec, ascending, n_eig, gV,
                                                                      a.lambda_dev, a.stride_lam); ++nl;
  if (sinc) {
    pointer_array_kernel<<<(nb + 127) / 128, 128, 0, st>>>(pS, gV, (size_t)n_beam * n_eig, nb); ++nl;
    if (cublasZtrsmBatched(g->blas, CUBLAS_SIDE_LEFT, CUBLAS_FILL_MODE_LOWER, CUBLAS_OP_C, CUBLAS_DIAG_NON_UNIT, n_beam, n_eig, &one, pG, n_beam,
                           pS, n_beam, nb) != CUBLAS_STATUS_SUCCESS) {
      bb_note_cuda_error(cudaErrorUnknown, "cublasZtrsmBatched (V = L^-H Q)", __FILE__, __LINE__);
      return BB_ECUDA;
    }
  }
  if (has_w) {
    if (cublasZgemmStridedBatched(g->blas, CUBLAS_OP_N, CUBLAS_OP_N, n_ant, n_eig, n_beam, &one, gW, n_ant, sW, gV, n_beam,
                                  (long long)n_beam * n_eig, &zero, gB, n_ant, (long long)n_ant * n_eig, nb) != CUBLAS_STATUS_SUCCESS) {
      bb_note_cuda_error(cudaErrorUnknown, "cublasZgemmStridedBatched (B = W V)", __FILE__, __LINE__);
      return BB_ECUDA;
    }
    narrow_kernel<<<dim3((n_ant + 127) / 128, n_eig, nb), blk, 0, st>>>(gB, n_ant, n_eig, a.B_dev, a.stride_b, info_chol, info_eig);
  } else {
    narrow_kernel<<<dim3((n_ant + 127) / 128, n_eig, nb), blk, 0, st>>>(gV, n_ant, n_eig, a.B_dev, a.stride_b, info_chol, info_eig);
  }
  ++nl;
  if (a.ev_eig1) cudaEventRecord(a.ev_eig1, st);
  BB_CUDA(cudaGetLastError());
  if (launches) *launches += nl;
  return BB_OK;
}

int bb_launch_level_weights(const double* lambda_dev, int n_eig, const double* intervals_dev, int ld_int, int n_intervals,
                            FilterList filters, float* D_dev, int ldd, const int* info_chol, const int* info_eig, int* status_dev,
                            cudaStream_t st) {
  level_weights_kernel<<<dim3((n_eig + 127) / 128, n_intervals * filters.n), 128, 0, st>>>(lambda_dev, n_eig, intervals_dev, ld_int,
                                                                                          n_intervals, filters, D_dev, ldd, info_chol,
                                                                                          info_eig, status_dev);
  BB_CUDA(cudaGetLastError());
  return BB_OK;
}
