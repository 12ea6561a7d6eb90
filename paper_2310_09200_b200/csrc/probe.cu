// Peak probes: register-only loops that saturate one pipe on every SM, timed with CUDA events.
// They give the measured denominators of the compute roofline:
//   kind 0  FFMA   (fma.rn.f32)            ops = lane-FMAs
//   kind 1  FFMA2  (fma.rn.f32x2)          ops = lane-FMAs (2 per lane-instruction)
//   kind 2  MUFU   (sin.approx+cos.approx) ops = MUFU lane-ops
//   kind 3  DFMA   (fma.rn.f64)            ops = lane-FMAs
// Interference probes (why the tensor variants reduce phases without fp64):
// 8 warps per SM run independent FMA chains while, for the odd kinds, one thread streams tcgen05.mma
// (kind::f16, 128x128x16, operands zero) on the same SM; time is the slowest warp's clock64 span.
//   kind 4 / 5  DFMA without / with the MMA stream
//   kind 6 / 7  IMAD without / with the MMA stream
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

// ---- interference probe ------------------------------------------------------------------------------
constexpr int kMixIters = 512, kMixMmas = 3072;

__global__ void __launch_bounds__(288, 1) probe_mix(long long* cycles, float* sink, int use_imad, int with_mma, double a, double b) {
  extern __shared__ __align__(1024) unsigned char smem[];
  __shared__ uint64_t bar;
  __shared__ uint32_t tmem_slot;
  const int tid = threadIdx.x, warp = tid >> 5;
  const uint32_t bar_a = (uint32_t)__cvta_generic_to_shared(&bar);
  if (tid == 0) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(bar_a));
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  if (warp == 8) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], 256;" ::"r"((uint32_t)__cvta_generic_to_shared(&tmem_slot)));
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::);
  }
  for (int i = tid; i < 4096 / 4; i += blockDim.x) reinterpret_cast<uint32_t*>(smem)[i] = 0;   // B tile (zeros)
  asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
  asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
  __syncthreads();
  asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
  const uint32_t tb = tmem_slot;
  if (warp < 8) {
    long long t0, t1;
    asm volatile("mov.u64 %0, %%clock64;" : "=l"(t0));
    float r = 0.f;
    if (use_imad) {
      int x[8];
#pragma unroll
      for (int i = 0; i < 8; ++i) x[i] = tid + i;
      const int m = (int)a + 3, c = (int)b + 1;
      for (int it = 0; it < kMixIters; ++it)
#pragma unroll
        for (int i = 0; i < 8; ++i) x[i] = x[i] * m + c;
#pragma unroll
      for (int i = 0; i < 8; ++i) r += (float)x[i];
    } else {
      double x[8];
#pragma unroll
      for (int i = 0; i < 8; ++i) x[i] = (double)tid + i;
      for (int it = 0; it < kMixIters; ++it)
#pragma unroll
        for (int i = 0; i < 8; ++i) x[i] = fma(x[i], a, b);
#pragma unroll
      for (int i = 0; i < 8; ++i) r += (float)x[i];
    }
    asm volatile("mov.u64 %0, %%clock64;" : "=l"(t1));
    sink[blockIdx.x * 256 + tid] = r;
    if ((tid & 31) == 0) cycles[blockIdx.x * 8 + warp] = t1 - t0;
  } else if (with_mma && tid == 256) {
    // D[128 x 128] at TMEM column 0 (+)= A[128 x 16 halves] at column 128 (garbage is fine) x B (zeros, K-major no swizzle)
    const uint32_t idesc = (1u << 4) | ((128u >> 3) << 17) | ((128u >> 4) << 24);
    const uint32_t sa = (uint32_t)__cvta_generic_to_shared(smem);
    uint64_t bd = (uint64_t)((sa >> 4) & 0x3FFF) | ((uint64_t)(2048 >> 4) << 16) | ((uint64_t)(128 >> 4) << 32) | ((uint64_t)1 << 46);
    for (int i = 0; i < kMixMmas; ++i)
      asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\ttcgen05.mma.cta_group::1.kind::f16 [%0], [%1], %2, %3, p;\n\t}" ::"r"(tb),
                   "r"(tb + 128), "l"(bd), "r"(idesc), "r"(1) : "memory");
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(bar_a) : "memory");
    asm volatile("{\n\t.reg .pred p;\n\tW_%=:\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%0], 0;\n\t@p bra D_%=;\n\tbra W_%=;\n\tD_%=:\n\t}" ::"r"(bar_a) : "memory");
  }
  asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
  __syncthreads();
  if (warp == 8) {
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 256;" ::"r"(tb));
  }
}

int probe_mix_run(int kind, int sm_count, cudaStream_t st, double* ops_per_s, double* ms_out) {
  long long* cyc = nullptr;
  float* sink = nullptr;
  BB_CUDA(cudaMalloc(&cyc, (size_t)sm_count * 8 * sizeof(long long)));
  BB_CUDA(cudaMalloc(&sink, (size_t)sm_count * 256 * sizeof(float)));
  int khz = 0, dev = 0;
  cudaGetDevice(&dev);
  cudaDeviceGetAttribute(&khz, cudaDevAttrClockRate, dev);
  std::vector<long long> h((size_t)sm_count * 8);
  long long worst = 0;
  for (int rep = 0; rep < 3; ++rep) {
    probe_mix<<<sm_count, 288, 4096, st>>>(cyc, sink, kind >= 6, kind & 1, 0.999, 0.001);
    cudaError_t e = cudaStreamSynchronize(st);
    if (e != cudaSuccess) { cudaFree(cyc); cudaFree(sink); bb_note_cuda_error(e, "probe_mix", __FILE__, __LINE__); return BB_ECUDA; }
    cudaMemcpy(h.data(), cyc, h.size() * sizeof(long long), cudaMemcpyDeviceToHost);
    worst = 0;
    for (long long c : h) worst = c > worst ? c : worst;
  }
  cudaFree(cyc);
  cudaFree(sink);
  // slowest warp's span in SM cycles -> seconds at the nominal maximum clock
  const double sec = (double)worst / ((double)khz * 1e3);
  *ms_out = sec * 1e3;
  *ops_per_s = 8.0 * kMixIters * 256.0 * sm_count / sec;
  return BB_OK;
}

}  // namespace

int bb_probe_run(int kind, int sm_count, cudaStream_t st, double* ops_per_s, double* ms_out) {
  if (kind >= 4 && kind <= 7) return probe_mix_run(kind, sm_count, st, ops_per_s, ms_out);
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
