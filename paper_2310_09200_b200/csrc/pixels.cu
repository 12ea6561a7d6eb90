// Pixel preparation (once per imaging handle): field centre r_c and centred directions r' = r - r_c.
//
// Centring identity (exact): <p_i, r_j> = <p_i - pbar, r_j - r_c> + <p_i - pbar, r_c> + <pbar, r_j>.
// The last term is common to all antennas of a pixel and vanishes in |E|^2; the middle one is a
// per-antenna constant folded into B by the prep kernels. r_c is the centre of the bounding box
// of the pixel vectors (any r_c is exact; this one minimises max |r'|), found with a
// fixed-shape two-pass min/max reduction, so it is deterministic.
#include "internal.h"
#include <cfloat>

namespace {

constexpr int kBlocks = 256, kThreads = 256;

__global__ void __launch_bounds__(kThreads)
minmax_partial(const double* __restrict__ pix, int64_t n_pix, int64_t ld, double* __restrict__ part) {
  __shared__ double sm[6][kThreads];
  double lo[3] = {DBL_MAX, DBL_MAX, DBL_MAX}, hi[3] = {-DBL_MAX, -DBL_MAX, -DBL_MAX};
  for (int64_t j = (int64_t)blockIdx.x * kThreads + threadIdx.x; j < n_pix; j += (int64_t)kBlocks * kThreads)
    for (int c = 0; c < 3; ++c) {
      const double v = pix[j + c * ld];
      lo[c] = fmin(lo[c], v);
      hi[c] = fmax(hi[c], v);
    }
  for (int c = 0; c < 3; ++c) { sm[c][threadIdx.x] = lo[c]; sm[3 + c][threadIdx.x] = hi[c]; }
  __syncthreads();
  for (int w = kThreads / 2; w > 0; w >>= 1) {
    if ((int)threadIdx.x < w)
      for (int c = 0; c < 3; ++c) {
        sm[c][threadIdx.x] = fmin(sm[c][threadIdx.x], sm[c][threadIdx.x + w]);
        sm[3 + c][threadIdx.x] = fmax(sm[3 + c][threadIdx.x], sm[3 + c][threadIdx.x + w]);
      }
    __syncthreads();
  }
  if (threadIdx.x < 6) part[blockIdx.x * 6 + threadIdx.x] = sm[threadIdx.x][0];
}

// rc[0..2] = centre of the bounding box, rc[3] = half its diagonal (>= max |r - r_c|)
__global__ void minmax_final(const double* __restrict__ part, double* __restrict__ rc) {
  __shared__ double half[3];
  if (threadIdx.x < 3) {
    double lo = DBL_MAX, hi = -DBL_MAX;
    for (int b = 0; b < kBlocks; ++b) {
      lo = fmin(lo, part[b * 6 + threadIdx.x]);
      hi = fmax(hi, part[b * 6 + 3 + threadIdx.x]);
    }
    rc[threadIdx.x] = 0.5 * (lo + hi);
    half[threadIdx.x] = 0.5 * (hi - lo);
  }
  __syncthreads();
  if (threadIdx.x == 0) rc[3] = sqrt(half[0] * half[0] + half[1] * half[1] + half[2] * half[2]);
}

__global__ void __launch_bounds__(kThreads)
centre_pixels(const double* __restrict__ pix, int64_t n_pix, int64_t ld, const double* __restrict__ rc,
              double* __restrict__ rprime, int64_t stride) {
  const int64_t j = (int64_t)blockIdx.x * kThreads + threadIdx.x;
  if (j < stride)
    for (int c = 0; c < 3; ++c) rprime[c * stride + j] = (j < n_pix) ? pix[j + c * ld] - rc[c] : 0.0;
}

}  // namespace

int bb_pixels_prepare(const double* pix_dev, int64_t n_pix, int64_t ld_pix, double* rprime, int64_t pix_stride,
                      double rc_out[3], double* rmax_out, cudaStream_t st) {
  double* scratch = nullptr;
  double host[4] = {0, 0, 0, 0};
  BB_CUDA(cudaMalloc(&scratch, (kBlocks * 6 + 4) * sizeof(double)));
  minmax_partial<<<kBlocks, kThreads, 0, st>>>(pix_dev, n_pix, ld_pix, scratch);
  minmax_final<<<1, 32, 0, st>>>(scratch, scratch + kBlocks * 6);
  centre_pixels<<<(unsigned)((pix_stride + kThreads - 1) / kThreads), kThreads, 0, st>>>(
      pix_dev, n_pix, ld_pix, scratch + kBlocks * 6, rprime, pix_stride);
  cudaError_t e = cudaGetLastError();
  if (e == cudaSuccess) e = cudaMemcpyAsync(host, scratch + kBlocks * 6, 4 * sizeof(double), cudaMemcpyDeviceToHost, st);
  if (e == cudaSuccess) e = cudaStreamSynchronize(st);
  cudaFree(scratch);
  rc_out[0] = host[0]; rc_out[1] = host[1]; rc_out[2] = host[2];
  *rmax_out = host[3];
  if (e != cudaSuccess) { bb_note_cuda_error(e, "bb_pixels_prepare", __FILE__, __LINE__); return BB_ECUDA; }
  return BB_OK;
}
