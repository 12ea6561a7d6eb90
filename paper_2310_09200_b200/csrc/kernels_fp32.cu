// FP32 CUDA-core variant of the fused Standard Synthesizer (sm_100a).
//
// One kernel does, per pixel tile and for every queued collect (time step / channel):
//   a1  phase generator   P_ij = exp(j 2 pi <p'_i, r'_j>)          PAPER.md:323 (Alg. 2 line 5)
//   a2  contraction       E_kj = sum_i conj(B_ik) P_ij             PAPER.md:123 (Eq. 15), :325
//   a3  epilogue          I_l(j) += sum_k D[l,k] |E_kj|^2          PAPER.md:332-336, :301, Eq. 20
//   a4  collect loop      over all queued collects
// E is never written to memory. Design notes:
//   * thread = PT pixels x KT eigenpairs; accumulators (Re, Im') for eigenpair PAIRS are packed
//     in float2 so that every FMA is an FFMA2 (fma.rn.f32x2) whose first operand is the scalar
//     cos / sin / -sin of the thread's pixel (SASS broadcasts it: "R.F32"), the second a pair
//     (b_2q, b_2q+1) read from shared memory by ONE uniform (broadcast) LDS.128 per eigen-pair.
//     Im' = -Im is accumulated; only |E|^2 is used, so the sign is irrelevant.
//   * phase: centred coordinates, t = fma(px,rx, fma(py,ry, fma(pz,rz, 1.5*2^20))) in fp64; the
//     low 32 bits of t are the phase in turns as a signed fixed-point fraction (ulp 2^-32 turn),
//     i.e. the fp64 range reduction costs 3 DFMA and nothing else; then I2F + MUFU.SIN/COS.
//   * B chunks (AC antennas) are staged global->shared with cp.async.bulk (UBLKCP) on mbarriers,
//     STAGES deep; p'_i rides in the same chunk.
//   * level sums live in shared memory across collects; the image is read-modified-written once
//     per launch (8*L bytes per pixel per launch).
#include "internal.h"
#include <cuda.h>

namespace {

constexpr int kThreads = 128;
constexpr int kStages = 3;
constexpr double kMagic = 1572864.0;  // 1.5 * 2^20: ulp = 2^-32, valid for |phase| < 2^19 turns

__host__ __device__ inline size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

// ---------------------------------------------------------------------------- PTX helpers
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
  asm volatile(
      "{\n\t.reg .pred p;\n\t"
      "WAIT_%=:\n\t"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
      "@p bra DONE_%=;\n\t"
      "bra WAIT_%=;\n\t"
      "DONE_%=:\n\t}" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}
__device__ __forceinline__ void bulk_g2s(void* dst, const void* src, uint32_t bytes, uint64_t* bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                   smem_u32(dst)),
               "l"(src), "r"(bytes), "r"(smem_u32(bar))
               : "memory");
}
__device__ __forceinline__ void fence_barrier_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

// a1: phase of (antenna, pixel) in turns -> (cos, sin) in fp32
__device__ __forceinline__ void phase_cs(double px, double py, double pz, double rx, double ry, double rz,
                                         float& c, float& s) {
  double t = fma(px, rx, kMagic);
  t = fma(py, ry, t);
  t = fma(pz, rz, t);
  const float x = (float)__double2loint(t) * (6.283185307179586f / 4294967296.0f);
  c = __cosf(x);  // FMUL.RZ by 1/(2 pi) + MUFU.COS
  s = __sinf(x);
}

// ---------------------------------------------------------------------------- synthesizer
template <int KT, int PT, int GC, int MINB>
__global__ void __launch_bounds__(kThreads, MINB)
synth_fp32_kernel(const double* __restrict__ rprime, int64_t n_pix, int64_t pix_stride,
                  const unsigned char* __restrict__ packed, size_t packed_stride, size_t slab_offset,
                  const float* __restrict__ weights, size_t weight_stride, int n_eig_pad, int eig_offset,
                  int n_collects_all, int n_chunks, int AC, int n_levels, float* __restrict__ img,
                  int64_t img_stride, int collects_per_split, float* __restrict__ scratch) {
  // gridDim.y > 1: collect-range split of a small image (kernels_tc.cu bb_collect_split): this CTA handles the collects
  // [e0, e0 + n_collects) and leaves its level sums in scratch[blockIdx.y]
  const int e0 = (int)blockIdx.y * collects_per_split;
  const int n_collects = min(collects_per_split, n_collects_all - e0);
  packed += (size_t)e0 * packed_stride;
  weights += (size_t)e0 * weight_stride;
  constexpr int TG = kThreads / GC;       // threads per eigen-group
  constexpr int NQ = KT / 2;              // eigen-pairs per thread
  constexpr int ROW4 = GC * NQ;           // float4 per antenna row in a chunk
  extern __shared__ __align__(128) unsigned char smem_raw[];

  const uint32_t chunk_bytes = (uint32_t)AC * (ROW4 * 16 + 32);
  unsigned char* stage_base = smem_raw;                                   // kStages * chunk_bytes
  float* lev = reinterpret_cast<float*>(smem_raw + align_up((size_t)kStages * chunk_bytes, 128));  // [L][PT][128]
  float* dsm = lev + (size_t)n_levels * PT * kThreads;                    // [2][L][GC*KT]
  uint64_t* full = reinterpret_cast<uint64_t*>(dsm + 2 * (size_t)n_levels * GC * KT);

  const int tid = threadIdx.x;
  const int g = tid / TG, t = tid % TG;
  const int64_t tile_base = (int64_t)blockIdx.x * (TG * PT);

  if (tid == 0) {
    for (int s = 0; s < kStages; ++s) mbar_init(&full[s], 1);
    fence_barrier_init();
  }
  for (int i = tid; i < n_levels * PT * kThreads; i += kThreads) lev[i] = 0.f;

  double rx[PT], ry[PT], rz[PT];
#pragma unroll
  for (int p = 0; p < PT; ++p) {
    const int64_t j = tile_base + t + (int64_t)p * TG;
    const bool ok = j < n_pix;
    rx[p] = ok ? rprime[j] : 0.0;
    ry[p] = ok ? rprime[pix_stride + j] : 0.0;
    rz[p] = ok ? rprime[2 * pix_stride + j] : 0.0;
  }
  __syncthreads();

  const int total = n_collects * n_chunks;
  auto issue = [&](int n) {  // thread 0: stage chunk n (global order) into stage n % kStages
    const int e = n / n_chunks, c = n - e * n_chunks;
    const unsigned char* src = packed + (size_t)e * packed_stride + slab_offset + (size_t)c * chunk_bytes;
    uint64_t* bar = &full[n % kStages];
    mbar_expect_tx(bar, chunk_bytes);
    bulk_g2s(stage_base + (size_t)(n % kStages) * chunk_bytes, src, chunk_bytes, bar);
  };
  if (tid == 0)
    for (int n = 0; n < kStages && n < total; ++n) issue(n);

  int n = 0;
  for (int e = 0; e < n_collects; ++e) {
    // weights of this collect -> shared (double-buffered by collect parity)
    float* dcur = dsm + (size_t)(e & 1) * n_levels * GC * KT;
    for (int i = tid; i < n_levels * GC * KT; i += kThreads) {
      const int l = i / (GC * KT), k = i - l * (GC * KT);
      dcur[i] = weights[(size_t)e * weight_stride + (size_t)l * n_eig_pad + eig_offset + k];
    }

    float2 re[PT][NQ], im[PT][NQ];
#pragma unroll
    for (int p = 0; p < PT; ++p)
#pragma unroll
      for (int q = 0; q < NQ; ++q) re[p][q] = im[p][q] = make_float2(0.f, 0.f);

    for (int c = 0; c < n_chunks; ++c, ++n) {
      const int st = n % kStages;
      mbar_wait(&full[st], (uint32_t)((n / kStages) & 1));
      const float4* brow = reinterpret_cast<const float4*>(stage_base + (size_t)st * chunk_bytes) + g * NQ;
      const double4* prow = reinterpret_cast<const double4*>(stage_base + (size_t)st * chunk_bytes + (size_t)AC * ROW4 * 16);

      float cs[PT], sn[PT];
      {
        const double4 pp = prow[0];
#pragma unroll
        for (int p = 0; p < PT; ++p) phase_cs(pp.x, pp.y, pp.z, rx[p], ry[p], rz[p], cs[p], sn[p]);
      }
#pragma unroll 2
      for (int i = 0; i < AC; ++i) {
        float cn[PT], snn[PT];
        {  // a1 for the NEXT antenna, overlapped with this antenna's FMAs (last one is a dummy)
          const double4 pp = prow[(i + 1 < AC) ? i + 1 : i];
#pragma unroll
          for (int p = 0; p < PT; ++p) phase_cs(pp.x, pp.y, pp.z, rx[p], ry[p], rz[p], cn[p], snn[p]);
        }
        // a2: 4 FFMA2 per (pixel, eigen-pair). Order matters: an FFMA2 reads 5 registers (scalar, pair,
        // accumulator pair) and the register file delivers 2 per bank per FFMA2 slot, so consecutive
        // FFMA2 must share an operand through the operand-reuse cache.
#pragma unroll
        for (int q = 0; q < NQ; ++q) {
          const float4 b = brow[(size_t)i * ROW4 + q];
          const float2 br = make_float2(b.x, b.y), bi = make_float2(b.z, b.w);
#pragma unroll
          for (int p = 0; p < PT; ++p) re[p][q] = __ffma2_rn(make_float2(cs[p], cs[p]), br, re[p][q]);
#pragma unroll
          for (int p = 0; p < PT; ++p) im[p][q] = __ffma2_rn(make_float2(-sn[p], -sn[p]), br, im[p][q]);
#pragma unroll
          for (int p = 0; p < PT; ++p) re[p][q] = __ffma2_rn(make_float2(sn[p], sn[p]), bi, re[p][q]);
#pragma unroll
          for (int p = 0; p < PT; ++p) im[p][q] = __ffma2_rn(make_float2(cs[p], cs[p]), bi, im[p][q]);
        }
#pragma unroll
        for (int p = 0; p < PT; ++p) { cs[p] = cn[p]; sn[p] = snn[p]; }
      }
      __syncthreads();  // every thread is done with stage st
      if (tid == 0 && n + kStages < total) issue(n + kStages);
    }

    // a3: square, weight, reduce over this thread's eigenpairs into the level sums
#pragma unroll
    for (int p = 0; p < PT; ++p) {
      float pw[KT];
#pragma unroll
      for (int q = 0; q < NQ; ++q) {
        pw[2 * q] = re[p][q].x * re[p][q].x + im[p][q].x * im[p][q].x;
        pw[2 * q + 1] = re[p][q].y * re[p][q].y + im[p][q].y * im[p][q].y;
      }
      for (int l = 0; l < n_levels; ++l) {
        const float* dl = dcur + (size_t)l * (GC * KT) + g * KT;
        float sacc = 0.f;
#pragma unroll
        for (int k = 0; k < KT; ++k) sacc = fmaf(dl[k], pw[k], sacc);
        lev[((size_t)l * PT + p) * kThreads + tid] += sacc;
      }
    }
  }
  __syncthreads();
  // image read-modify-write: sum the GC eigen-groups in a fixed order (deterministic)
  for (int idx = tid; idx < n_levels * PT * TG; idx += kThreads) {
    const int l = idx / (PT * TG), r = idx - l * (PT * TG);
    const int p = r / TG, tt = r - p * TG;
    const int64_t j = tile_base + tt + (int64_t)p * TG;
    if (j < n_pix) {
      float v = 0.f;
#pragma unroll
      for (int gg = 0; gg < GC; ++gg) v += lev[((size_t)l * PT + p) * kThreads + gg * TG + tt];
      if (gridDim.y > 1) scratch[((size_t)blockIdx.y * n_levels + l) * img_stride + j] = v;
      else img[(size_t)l * img_stride + j] += v;
    }
  }
}

// ---------------------------------------------------------------------------- preparation (a0'')
// One thread per (antenna, eigenpair) of the padded operand; every block recomputes the antenna
// centroid with a fixed-order reduction (deterministic, identical in all blocks).
__global__ void __launch_bounds__(256)
prep_fp32_kernel(PrepArgs a, int KT, int GC, int AC, int n_slabs, int n_chunks, int n_eig_pad, int n_ant_pad,
                 size_t chunk_bytes) {
  __shared__ double red[3][256];
  __shared__ double cen[3];
  const int tid = threadIdx.x;
  double sx = 0, sy = 0, sz = 0;
  for (int i = tid; i < a.n_ant; i += 256) {
    sx += a.xyz[i]; sy += a.xyz[i + a.ldxyz]; sz += a.xyz[i + 2 * (size_t)a.ldxyz];
  }
  red[0][tid] = sx; red[1][tid] = sy; red[2][tid] = sz;
  __syncthreads();
  for (int w = 128; w > 0; w >>= 1) {
    if (tid < w) { red[0][tid] += red[0][tid + w]; red[1][tid] += red[1][tid + w]; red[2][tid] += red[2][tid + w]; }
    __syncthreads();
  }
  if (tid < 3) cen[tid] = red[tid][0] / (double)a.n_ant;
  __syncthreads();
  // range of the fixed-point phase reduction: |<p', r'>| <= |p'| rmax must stay below 2^19 turns; every block
  // reaches the same verdict, and a collect that fails it (NaN / Inf coordinates included) contributes nothing
  // (zero weights, zero B, zero positions) and raises the flag
  double far2 = 0.0;
  for (int i = tid; i < a.n_ant; i += 256) {
    const double dx = a.xyz[i] - cen[0], dy = a.xyz[i + a.ldxyz] - cen[1], dz = a.xyz[i + 2 * (size_t)a.ldxyz] - cen[2];
    const double d2 = dx * dx + dy * dy + dz * dz;
    if (!(d2 <= far2)) far2 = (d2 == d2) ? d2 : INFINITY;    // fmax would DROP a NaN: a non-finite coordinate must fail the test
  }
  red[0][tid] = far2;
  __syncthreads();
  for (int w = 128; w > 0; w >>= 1) {
    if (tid < w) red[0][tid] = fmax(red[0][tid], red[0][tid + w]);
    __syncthreads();
  }
  const bool in_range = sqrt(red[0][0]) / a.wavelength * a.rmax < kFp32PhaseLimit;
  if (!in_range && blockIdx.x == 0 && tid == 0) atomicOr(a.status, BB_FLAG_RANGE);

  const int64_t gid = (int64_t)blockIdx.x * 256 + tid;
  const int64_t n_elem = (int64_t)n_ant_pad * n_eig_pad;
  if (gid < n_elem) {
    const int i = (int)(gid / n_eig_pad), k = (int)(gid - (int64_t)i * n_eig_pad);
    double px = 0, py = 0, pz = 0;
    float br = 0.f, bi = 0.f;
    if (i < a.n_ant && in_range) {                            // a refused collect is packed as zeros: 0 weight x NaN |E|^2 would be NaN
      px = (a.xyz[i] - cen[0]) / a.wavelength;
      py = (a.xyz[i + a.ldxyz] - cen[1]) / a.wavelength;
      pz = (a.xyz[i + 2 * (size_t)a.ldxyz] - cen[2]) / a.wavelength;
      if (k < a.n_eig) {
        // fold the per-antenna constant phase exp(-j 2 pi <p'_i, r_c>) into B (fp64)
        double th = px * a.rc[0] + py * a.rc[1] + pz * a.rc[2];
        th -= rint(th);
        double sn, cs;
        sincospi(2.0 * th, &sn, &cs);
        const bb_c32 b = a.B[i + (size_t)k * a.ldb];
        br = (float)((double)b.re * cs + (double)b.im * sn);
        bi = (float)((double)b.im * cs - (double)b.re * sn);
      }
    }
    const int per_slab = GC * KT;
    const int slab = k / per_slab, kk = k - slab * per_slab;
    const int c = i / AC, ii = i - c * AC;
    unsigned char* chunk = a.packed + ((size_t)slab * n_chunks + c) * chunk_bytes;
    float* bf = reinterpret_cast<float*>(chunk) + ((size_t)ii * (per_slab / 2) + kk / 2) * 4 + (kk & 1);
    bf[0] = br;
    bf[2] = bi;
    if (kk == 0) {
      double* pp = reinterpret_cast<double*>(chunk + (size_t)AC * per_slab * 8) + (size_t)ii * 4;
      pp[0] = px; pp[1] = py; pp[2] = pz; pp[3] = 0.0;
    }
  }
  // weights D[l,k] -> [level][n_eig_pad], zero padded
  const int64_t n_w = (int64_t)a.n_levels * n_eig_pad;
  if (gid < n_w) {
    const int l = (int)(gid / n_eig_pad), k = (int)(gid - (int64_t)l * n_eig_pad);
    a.weights[gid] = (k < a.n_eig && in_range) ? a.D[l + (size_t)k * a.ldd] : 0.f;
  }
}

template <int KT, int PT, int GC, int MINB>
int launch_variant(const Fp32Plan& plan, const SynthArgs& a, cudaStream_t st, int* launches) {
  constexpr int TG = kThreads / GC;
  const size_t smem = align_up((size_t)kStages * plan.chunk_bytes, 128) +
                      (size_t)a.n_levels * PT * kThreads * 4 + 2 * (size_t)a.n_levels * GC * KT * 4 + kStages * 8 + 16;
  auto kern = synth_fp32_kernel<KT, PT, GC, MINB>;
  BB_CUDA(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  const int64_t tiles = (a.n_pix + TG * PT - 1) / (TG * PT);
  const int cps = (a.n_collects + (a.scratch ? a.n_split : 1) - 1) / (a.scratch ? a.n_split : 1);
  const int n_split = (a.n_collects + cps - 1) / cps;      // ranges of cps collects that are not empty (<= a.n_split)
  for (int slab = 0; slab < plan.n_slabs; ++slab) {
    kern<<<dim3((unsigned)tiles, (unsigned)n_split), kThreads, smem, st>>>(a.rprime, a.n_pix, a.pix_stride, a.packed, a.packed_stride,
                                                   (size_t)slab * plan.n_chunks * plan.chunk_bytes, a.weights,
                                                   a.weight_stride, plan.n_eig_pad, slab * GC * KT, a.n_collects,
                                                   plan.n_chunks, plan.AC, a.n_levels, a.img, a.img_stride, cps, a.scratch);
    BB_CUDA(cudaGetLastError());
    ++*launches;
    if (n_split > 1) {
      const int rc = bb_launch_reduce_splits(a.scratch, n_split, a.n_levels, a.n_pix, a.img_stride, a.img, st);
      if (rc != BB_OK) return rc;
      ++*launches;
    }
  }
  return BB_OK;
}

}  // namespace

Fp32Plan bb_fp32_plan(int n_ant, int n_eig, int n_levels) {
  Fp32Plan p{};
  if (n_eig <= 8) { p.KT = 8; p.PT = 4; p.GC = 1; }
  else if (n_eig <= 12) { p.KT = 12; p.PT = 4; p.GC = 1; }
  else if (n_eig <= 16) { p.KT = 16; p.PT = 4; p.GC = 1; }
  else if (n_eig <= 32) { p.KT = 32; p.PT = 2; p.GC = 1; }
  else if (n_eig <= 64) { p.KT = 32; p.PT = 2; p.GC = 2; }
  else { p.KT = 32; p.PT = 2; p.GC = 4; }
  p.MINB = 2;
  p.AC = 32;
  const int per_slab = p.GC * p.KT;
  p.n_slabs = (n_eig + per_slab - 1) / per_slab;
  p.n_chunks = (n_ant + p.AC - 1) / p.AC;
  p.n_eig_pad = p.n_slabs * per_slab;
  p.n_ant_pad = p.n_chunks * p.AC;
  p.chunk_bytes = (size_t)p.AC * ((size_t)per_slab * 8 + 32);
  p.collect_bytes = (size_t)p.n_slabs * p.n_chunks * p.chunk_bytes;
  p.weight_floats = (size_t)n_levels * p.n_eig_pad;
  return p;
}

int bb_fp32_split(const Fp32Plan& plan, int64_t n_pix, int n_collects, int sm_count) {
  const int tile = (kThreads / plan.GC) * plan.PT;                   // pixels per CTA; MINB CTAs are resident per SM
  return bb_collect_split((n_pix + tile - 1) / tile, n_collects, sm_count * plan.MINB);
}

int bb_launch_prep_fp32(const Fp32Plan& plan, const PrepArgs& a, cudaStream_t st) {
  const int64_t n_elem = (int64_t)plan.n_ant_pad * plan.n_eig_pad;
  const int64_t n_w = (int64_t)a.n_levels * plan.n_eig_pad;
  const int64_t n = n_elem > n_w ? n_elem : n_w;
  prep_fp32_kernel<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(a, plan.KT, plan.GC, plan.AC, plan.n_slabs,
                                                                plan.n_chunks, plan.n_eig_pad, plan.n_ant_pad,
                                                                plan.chunk_bytes);
  BB_CUDA(cudaGetLastError());
  return BB_OK;
}

int bb_launch_synth_fp32(const Fp32Plan& plan, const SynthArgs& a, int /*sm_count*/, cudaStream_t st, int* launches) {
  *launches = 0;
  if (a.n_collects <= 0 || a.n_pix <= 0) return BB_OK;
#define BB_CASE(kt, pt, gc, mb) \
  if (plan.KT == kt && plan.PT == pt && plan.GC == gc && plan.MINB == mb) return launch_variant<kt, pt, gc, mb>(plan, a, st, launches);
  BB_CASE(8, 4, 1, 2) BB_CASE(12, 4, 1, 2) BB_CASE(16, 4, 1, 2)
  BB_CASE(32, 2, 1, 2) BB_CASE(32, 2, 2, 2) BB_CASE(32, 2, 4, 2)
#undef BB_CASE
  return BB_EUNSUPPORTED;
}
