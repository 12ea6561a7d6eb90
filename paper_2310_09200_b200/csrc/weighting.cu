// "Uniform" image weighting (Section 3.5): "we calculate the sampling density function on a grid in uv
// space with Delta u = Delta v = 1/FoV. Each visibility is then weighted with the inverse of its sampling density
// function" — applied to the visibility matrix before the eigendecomposition. Readings (Q17): a
// visibility is an antenna pair (p, q), p = q included; its uv point is the baseline (x_p - x_q) / lambda_w
// projected on the image-plane axes e_u, e_v; cell index = nearest integer of u / cell; the density is
// accumulated over all collects the caller adds (all time steps and channels of the observation); beamformed
// visibilities (W != I) have no single baseline and are not supported.
#include "internal.h"

#include <new>

struct bb_uvgrid {
  bb_ctx* ctx = nullptr;
  UvGridView view{};
  double* xyz_tmp = nullptr; size_t xyz_cap = 0;
};

namespace {

__global__ void density_add_kernel(const double* __restrict__ xyz, int ld, int n_ant, double wavelength, UvGridView g) {
  const int p = blockIdx.x * blockDim.x + threadIdx.x;
  if (p >= n_ant) return;
  for (int q = blockIdx.y; q < n_ant; q += gridDim.y)      // gridDim.y is capped at 65535: stride over the second antenna
    atomicAdd(&g.count[bb_uv_cell(g, xyz, ld, p, q, wavelength)], 1);
}

}  // namespace

cudaStream_t bb_ctx_glue_stream(bb_ctx* ctx);
int bb_ctx_device(bb_ctx* ctx);
cudaStream_t bb_ctx_user_stream(bb_ctx* ctx);

extern "C" int bb_uvgrid_create(bb_ctx* ctx, double cell, const double* e_u, const double* e_v, double max_uv, bb_uvgrid** out) {
  if (!out) return BB_EINVAL;
  *out = nullptr;
  if (!ctx || !e_u || !e_v || !(cell > 0.0) || !(max_uv >= 0.0)) return BB_EINVAL;
  const double half_d = ceil(max_uv / cell) + 1.0;
  if (!(half_d < 32000.0)) return BB_EUNSUPPORTED;          // (2 half + 1)^2 counters must stay below ~16 GB
  BB_CUDA(cudaSetDevice(bb_ctx_device(ctx)));
  bb_uvgrid* g = new (std::nothrow) bb_uvgrid;
  if (!g) return BB_EALLOC;
  g->ctx = ctx;
  g->view.half = (int)half_d;
  g->view.cell = cell;
  for (int d = 0; d < 3; ++d) { g->view.eu[d] = e_u[d]; g->view.ev[d] = e_v[d]; }
  const size_t side = 2 * (size_t)g->view.half + 1;
  if (cudaMalloc(&g->view.count, side * side * sizeof(int)) != cudaSuccess) { cudaGetLastError(); delete g; return BB_EALLOC; }
  cudaStream_t st = bb_ctx_glue_stream(ctx);
  if (cudaMemsetAsync(g->view.count, 0, side * side * sizeof(int), st) != cudaSuccess) {
    bb_note_cuda_error(cudaGetLastError(), "bb_uvgrid_create", __FILE__, __LINE__);
    cudaFree(g->view.count); delete g; return BB_ECUDA;
  }
  *out = g;
  return BB_OK;
}

extern "C" int bb_uvgrid_add(bb_uvgrid* g, int n_ant, double wavelength, const double* xyz, int ldxyz) {
  if (!g || !xyz || n_ant < 1 || ldxyz < n_ant || !(wavelength > 0.0)) return BB_EINVAL;
  BB_CUDA(cudaSetDevice(bb_ctx_device(g->ctx)));
  cudaStream_t st = bb_ctx_glue_stream(g->ctx);
  cudaPointerAttributes at;
  const bool dev = cudaPointerGetAttributes(&at, xyz) == cudaSuccess && (at.type == cudaMemoryTypeDevice || at.type == cudaMemoryTypeManaged);
  cudaGetLastError();
  const double* x = xyz;
  int ld = ldxyz;
  if (!dev) {
    if (g->xyz_cap < (size_t)n_ant * 3) {
      BB_CUDA(cudaStreamSynchronize(st));
      cudaFree(g->xyz_tmp); g->xyz_tmp = nullptr; g->xyz_cap = 0;
      if (cudaMalloc(&g->xyz_tmp, (size_t)n_ant * 3 * sizeof(double)) != cudaSuccess) { cudaGetLastError(); return BB_EALLOC; }
      g->xyz_cap = (size_t)n_ant * 3;
    }
    BB_CUDA(cudaMemcpy2DAsync(g->xyz_tmp, (size_t)n_ant * 8, xyz, (size_t)ldxyz * 8, (size_t)n_ant * 8, 3, cudaMemcpyHostToDevice, st));
    BB_CUDA(cudaStreamSynchronize(st));                     // host buffers are snapshotted before the call returns
    x = g->xyz_tmp; ld = n_ant;
  } else {
    BB_CUDA(cudaStreamSynchronize(bb_ctx_user_stream(g->ctx)));   // device input: the caller's work on the context stream is done
  }
  density_add_kernel<<<dim3((n_ant + 127) / 128, n_ant < 65535 ? n_ant : 65535), 128, 0, st>>>(x, ld, n_ant, wavelength, g->view);
  BB_CUDA(cudaGetLastError());
  if (!dev) BB_CUDA(cudaStreamSynchronize(st));             // xyz_tmp is reused by the next call
  return BB_OK;
}

extern "C" int bb_uvgrid_destroy(bb_uvgrid* g) {
  if (!g) return BB_EINVAL;
  cudaSetDevice(bb_ctx_device(g->ctx));
  cudaStreamSynchronize(bb_ctx_glue_stream(g->ctx));
  cudaFree(g->view.count);
  cudaFree(g->xyz_tmp);
  cudaGetLastError();
  delete g;
  return BB_OK;
}

const UvGridView* bb_uvgrid_view(const bb_uvgrid* g) { return g ? &g->view : nullptr; }
