// Peak probes: register-only loops that saturate one pipe on every SM, timed with CUDA events.
// They give the measured denominators of the compute roofline:
//   kind 0  FFMA   (fma.rn.f32)            ops = lane-FMAs
//   kind 1  FFMA2  (fma.rn.f32x2)          ops = lane-FMAs (2 per lane-instruction)
//   kind 2  MUFU   (sin.approx+cos.approx) ops = MUFU lane-ops
//   kind 3  DFMA   (fma.rn.f64)            ops = lane-FMAs
#include "internal.h"

namespace {

constexpr int kIters = 4096, kThreads = 256, kCtasPerSm = 4;

__global__ void __launch_bounds__(kThreads) probe_ffma(float* out, float a, float b) {
  float x[16];
#pragma unroll
  for (int i = 0; i < 16; ++i) x[i] = (float)threadIdx.x + i;
  for (int it = 0; it < kIters; ++it)
#pragma unroll
    for (int i = 0; i < 16; ++i) x[i] = fmaf(x[i], a, b);
  float s = 0.f;
#pragma unroll
  for (int i = 0; i < 16; ++i) s += x[i];
  out[blockIdx.x * kThreads + threadIdx.x] = s;
}

__global__ void __launch_bounds__(kThreads) probe_ffma2(float* out, float a, float b) {
  float2 x[16];
#pragma unroll
  for (int i = 0; i < 16; ++i) x[i] = make_float2((float)threadIdx.x + i, (float)i);
  const float2 aa = make_float2(a, a * 0.5f), bb = make_float2(b, b + 1.f);
  for (int it = 0; it < kIters; ++it)
#pragma unroll
    for (int i = 0; i < 16; ++i) x[i] = __ffma2_rn(x[i], aa, bb);
  float s = 0.f;
#pragma unroll
  for (int i = 0; i < 16; ++i) s += x[i].x + x[i].y;
  out[blockIdx.x * kThreads + threadIdx.x] = s;
}

__global__ void __launch_bounds__(kThreads) probe_mufu(float* out, float a) {
  float x[8];
#pragma unroll
  for (int i = 0; i < 8; ++i) x[i] = a * (float)(threadIdx.x + i);
  for (int it = 0; it < kIters; ++it)
#pragma unroll
    for (int i = 0; i < 8; ++i) x[i] = __sinf(x[i]) + __cosf(x[i]);
  float s = 0.f;
#pragma unroll
  for (int i = 0; i < 8; ++i) s += x[i];
  out[blockIdx.x * kThreads + threadIdx.x] = s;
}

__global__ void __launch_bounds__(kThreads) probe_dfma(float* out, double a, double b) {
  double x[16];
#pragma unroll
  for (int i = 0; i < 16; ++i) x[i] = (double)threadIdx.x + i;
  for (int it = 0; it < kIters; ++it)
#pragma unroll
    for (int i = 0; i < 16; ++i) x[i] = fma(x[i], a, b);
  double s = 0.0;
#pragma unroll
  for (int i = 0; i < 16; ++i) s += x[i];
  out[blockIdx.x * kThreads + threadIdx.x] = (float)s;
}

}  // namespace

int bb_probe_run(int kind, int sm_count, cudaStream_t st, double* ops_per_s, double* ms_out) {
  const int grid = sm_count * kCtasPerSm * 4;
  float* out = nullptr;
  BB_CUDA(cudaMalloc(&out, (size_t)grid * kThreads * sizeof(float)));
  cudaEvent_t e0, e1;
  cudaEventCreate(&e0);
  cudaEventCreate(&e1);
  float best = 1e30f;
  double per_thread = 0;
  for (int rep = 0; rep < 4; ++rep) {
    cudaEventRecord(e0, st);
    switch (kind) {
      case 0: probe_ffma<<<grid, kThreads, 0, st>>>(out, 0.999f, 0.001f); per_thread = 16.0 * kIters; break;
      case 1: probe_ffma2<<<grid, kThreads, 0, st>>>(out, 0.999f, 0.001f); per_thread = 32.0 * kIters; break;
      case 2: probe_mufu<<<grid, kThreads, 0, st>>>(out, 0.001f); per_thread = 16.0 * kIters; break;
      case 3: probe_dfma<<<grid, kThreads, 0, st>>>(out, 0.999, 0.001); per_thread = 16.0 * kIters; break;
      default: cudaFree(out); return BB_EINVAL;
    }
    cudaEventRecord(e1, st);
    cudaError_t e = cudaEventSynchronize(e1);
    if (e != cudaSuccess) { cudaFree(out); bb_note_cuda_error(e, "probe", __FILE__, __LINE__); return BB_ECUDA; }
    float ms = 0.f;
    cudaEventElapsedTime(&ms, e0, e1);
    if (rep > 0 && ms < best) best = ms;
  }
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  cudaFree(out);
  *ms_out = best;
  *ops_per_s = per_thread * (double)grid * kThreads / (best * 1e-3);
  return BB_OK;
}
