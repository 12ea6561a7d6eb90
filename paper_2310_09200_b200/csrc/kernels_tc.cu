// tcgen05 (3xTF32) tensor-core variant of the fused Standard Synthesizer (sm_100a).
//
// Same rows a1-a4 as kernels_fp32.cu (Alg. 2, Eq. 15, Eq. 20, Alg. 1 l.9), but the
// contraction runs on the 5th-generation tensor cores as a REAL GEMM:
//     D[j, n] += A[j, kappa] * Bop[n, kappa]
//     j      pixel of the tile (M = 128 = TMEM lanes: one producer thread owns one pixel / lane)
//     kappa  (antenna i, {cos, sin})            K = 2 * N_ant
//     n      ({Re, Im'} x eigenpair k)          N = 2 * NE,  NE = eigenpairs per slab (<= 64)
//     A[j,(i,cos)] = cos phi_ij, A[j,(i,sin)] = sin phi_ij
//     Bop[(Re,k),(i,cos)] = b_re, Bop[(Re,k),(i,sin)] = b_im, Bop[(Im',k),(i,cos)] = b_im, Bop[(Im',k),(i,sin)] = -b_re
//   so Re E_kj = sum_i (c b_re + s b_im), Im' E_kj = sum_i (c b_im - s b_re): 8 real flops per term.
// Split precision: x = hi + lo, hi = x with the 13 low mantissa bits cleared (exactly a TF32), lo = x - hi
// (exact); D += A_hi B_hi + A_lo B_hi + A_hi B_lo with fp32 accumulation in TMEM (lo*lo ~ 2^-22 dropped).
//
// CTA = 2 pixel tiles of 128 (256 pixels), 320 threads, 1 CTA per SM, all 512 TMEM columns:
//   warps 0-7  producers + epilogue: phase generator (fp64 fixed-point reduction, MUFU), hi/lo split,
//              tcgen05.st of their A rows straight into TMEM (A operand from TMEM: no smem round trip);
//              after the last chunk of a collect: tcgen05.ld of D, |E|^2, level weights, level sums.
//   warp 8     one elected thread issues tcgen05.mma.cta_group::1.kind::tf32 (A from TMEM, B from smem
//              descriptors) and tcgen05.commit to the stage / accumulator mbarriers; owns TMEM alloc.
//   warp 9     one elected thread streams the pre-tiled B chunks (UMMA canonical K-major no-swizzle
//              layout, written by prep_tc_kernel) global -> shared with cp.async.bulk on mbarriers.
#include "internal.h"
#include <cstdio>
#include <cstdlib>

namespace {

constexpr int kProducerThreads = 256;
constexpr int kThreadsTC = 320;
constexpr int kAC = 16;                 // antennas per chunk
constexpr int kK = 2 * kAC;             // tf32 K-columns per chunk and pass
constexpr int kSA = 2;                  // A stages (TMEM)
constexpr int kSB = 4;                  // B stages (shared memory)
constexpr int kMaxNE = 64;              // eigenpairs per slab
constexpr uint32_t kTmemCols = 512;
constexpr uint32_t kColD = 0;           // D of tile t at kColD + 128 t
constexpr uint32_t kColA = 256;         // A of stage s, tile t at kColA + 128 s + 64 t (+0 hi, +32 lo)
constexpr double kMagic = 1572864.0;    // 1.5 * 2^20 (see kernels_fp32.cu)

__host__ __device__ inline size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

// ---------------------------------------------------------------------------- PTX helpers
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_arrive(uint64_t* bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
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
                   smem_u32(dst)), "l"(src), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void fence_barrier_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_commit(uint64_t* bar) {
  asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void tc_commit_mc(uint64_t* bar, uint16_t mask) {   // same barrier offset in every CTA of the mask
  asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.multicast::cluster.b64 [%0], %1;" ::"r"(smem_u32(bar)), "h"(mask) : "memory");
}
__device__ __forceinline__ void bulk_g2s_mc(void* dst, const void* src, uint32_t bytes, uint64_t* bar, uint16_t mask) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.multicast::cluster [%0], [%1], %2, [%3], %4;" ::"r"(
                   smem_u32(dst)), "l"(src), "r"(bytes), "r"(smem_u32(bar)), "h"(mask) : "memory");
}
__device__ __forceinline__ void cluster_sync_all() {
  asm volatile("barrier.cluster.arrive.release.aligned;\n\tbarrier.cluster.wait.acquire.aligned;" ::: "memory");
}
__device__ __forceinline__ uint32_t cluster_rank() { uint32_t r; asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r)); return r; }
__device__ __forceinline__ void named_bar_sync(int id, int n) { asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(n) : "memory"); }

// D[tmem] (+)= A[tmem] * B[smem desc]; kind::tf32, cta_group::1
__device__ __forceinline__ void mma_tf32_ts(uint32_t d_tmem, uint32_t a_tmem, uint64_t b_desc, uint32_t idesc, uint32_t accumulate) {
  asm volatile(
      "{\n\t.reg .pred p;\n\t"
      "setp.ne.b32 p, %4, 0;\n\t"
      "tcgen05.mma.cta_group::1.kind::tf32 [%0], [%1], %2, %3, p;\n\t}" ::"r"(d_tmem), "r"(a_tmem), "l"(b_desc), "r"(idesc), "r"(accumulate)
      : "memory");
}
// shared-memory matrix descriptor: K-major, no swizzle; core matrix = 8 rows x 16 bytes, contiguous 128 B
__device__ __forceinline__ uint64_t make_b_desc(uint32_t saddr, uint32_t lbo_bytes, uint32_t sbo_bytes) {
  uint64_t d = 0;
  d |= (uint64_t)((saddr >> 4) & 0x3FFF);
  d |= (uint64_t)((lbo_bytes >> 4) & 0x3FFF) << 16;
  d |= (uint64_t)((sbo_bytes >> 4) & 0x3FFF) << 32;
  d |= (uint64_t)1 << 46;  // descriptor version (Blackwell)
  return d;                // base_offset 0, lbo_mode 0, layout_type 0 = SWIZZLE_NONE
}
__device__ __forceinline__ void tmem_st16(uint32_t addr, const uint32_t (&v)[16]) {
  asm volatile("tcgen05.st.sync.aligned.32x32b.x16.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16};" ::"r"(addr),
               "r"(v[0]), "r"(v[1]), "r"(v[2]), "r"(v[3]), "r"(v[4]), "r"(v[5]), "r"(v[6]), "r"(v[7]), "r"(v[8]), "r"(v[9]),
               "r"(v[10]), "r"(v[11]), "r"(v[12]), "r"(v[13]), "r"(v[14]), "r"(v[15]) : "memory");
}
__device__ __forceinline__ void tmem_ld8(uint32_t addr, float (&v)[8]) {
  uint32_t r[8];
  asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
               : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]) : "r"(addr));
#pragma unroll
  for (int i = 0; i < 8; ++i) v[i] = __uint_as_float(r[i]);
}
__device__ __forceinline__ void tmem_wait_ld() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }
__device__ __forceinline__ void tmem_wait_st() { asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory"); }

__device__ __forceinline__ void phase_cs(double px, double py, double pz, double rx, double ry, double rz, float& c, float& s) {
  double t = fma(px, rx, kMagic);
  t = fma(py, ry, t);
  t = fma(pz, rz, t);
  const float x = (float)__double2loint(t) * (6.283185307179586f / 4294967296.0f);
  c = __cosf(x);
  s = __sinf(x);
}
__device__ __forceinline__ void split_tf32(float x, uint32_t& hi, uint32_t& lo) {
  hi = __float_as_uint(x) & 0xFFFFE000u;
  lo = __float_as_uint(x - __uint_as_float(hi));
}

// ---------------------------------------------------------------------------- synthesizer
// Chunk in global/shared memory (N = 2 NE rows, kK columns):
//   [ B_hi : (kK/4) core columns x (N/8) row groups x (8 rows x 16 B) ][ B_lo : same ][ p' : kAC x 4 double ]
// With CS > 1 the CTAs of a cluster consume the same B chunks: each CTA fetches 1/CS of every chunk and
// multicasts it to all CTAs of the cluster (L2 -> SM traffic / CS); a stage is reused only after the MMAs of
// ALL CTAs of the cluster have read it (tcgen05.commit multicast onto every CTA's b_empty, count CS).
template <int CS>
__global__ void __launch_bounds__(kThreadsTC, 1)
synth_tc_kernel(const double* __restrict__ rprime, int64_t n_pix, int64_t pix_stride,
                const unsigned char* __restrict__ packed, size_t packed_stride, size_t slab_offset,
                const float* __restrict__ weights, size_t weight_stride, int n_eig_pad, int eig_offset, int NE,
                int n_collects, int n_chunks, int n_levels, float* __restrict__ img, int64_t img_stride, int dbg) {
  extern __shared__ __align__(1024) unsigned char smem_raw[];
  const int N = 2 * NE;
  const uint32_t half_bytes = (uint32_t)kK * N * 4;                 // one of B_hi / B_lo
  const uint32_t chunk_bytes = 2 * half_bytes + kAC * 32;
  const uint32_t lbo = (uint32_t)(N / 8) * 128, sbo = 128;

  unsigned char* stage_base = smem_raw;
  float* lev = reinterpret_cast<float*>(smem_raw + align_up((size_t)kSB * chunk_bytes, 1024));   // [L][256]
  float* dsm = lev + (size_t)n_levels * kProducerThreads;                                        // [2][L][NE]
  uint64_t* bars = reinterpret_cast<uint64_t*>(dsm + 2 * (size_t)n_levels * NE);
  uint64_t* b_full = bars;                 // [kSB]
  uint64_t* b_empty = bars + kSB;          // [kSB]
  uint64_t* a_full = bars + 2 * kSB;       // [kSA]
  uint64_t* a_empty = a_full + kSA;        // [kSA]
  uint64_t* d_full = a_empty + kSA;
  uint64_t* d_empty = d_full + 1;
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(d_empty + 1);

  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;

  if (tid == 0) {
    for (int s = 0; s < kSB; ++s) { mbar_init(&b_full[s], 1); mbar_init(&b_empty[s], CS); }
    for (int s = 0; s < kSA; ++s) { mbar_init(&a_full[s], kProducerThreads / 32); mbar_init(&a_empty[s], 1); }
    mbar_init(d_full, 1);
    mbar_init(d_empty, kProducerThreads / 32);
    fence_barrier_init();
  }
  if (warp == 8) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(tmem_slot)), "r"(kTmemCols));
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::);
  }
  for (int i = tid; i < n_levels * kProducerThreads; i += kThreadsTC) lev[i] = 0.f;
  tc_fence_before();
  __syncthreads();
  if (CS > 1) cluster_sync_all();          // every CTA's barriers are initialised before any remote arrive / copy
  tc_fence_after();
  const uint32_t tmem_base = *tmem_slot;
  const int total = n_collects * n_chunks;

  if (warp < 8) {
    // ===================== producers / epilogue: one pixel (TMEM lane) per thread =====================
    const int tile = warp >> 2;
    const uint32_t lane_field = (uint32_t)((warp & 3) * 32) << 16;
    const int64_t j = (int64_t)blockIdx.x * kProducerThreads + tid;
    const bool ok = j < n_pix;
    const double rx = ok ? rprime[j] : 0.0, ry = ok ? rprime[pix_stride + j] : 0.0, rz = ok ? rprime[2 * pix_stride + j] : 0.0;
    int n = 0;
    for (int e = 0; e < n_collects; ++e) {
      float* dcur = dsm + (size_t)(e & 1) * n_levels * NE;
      for (int i = tid; i < n_levels * NE; i += kProducerThreads) {
        const int l = i / NE, k = i - l * NE;
        dcur[i] = weights[(size_t)e * weight_stride + (size_t)l * n_eig_pad + eig_offset + k];
      }
      for (int c = 0; c < n_chunks; ++c, ++n) {
        const int sa = n % kSA, sb = n % kSB;
        mbar_wait(&a_empty[sa], (uint32_t)(((n / kSA) & 1) ^ 1));
        mbar_wait(&b_full[sb], (uint32_t)((n / kSB) & 1));
        tc_fence_after();
        const double4* prow = reinterpret_cast<const double4*>(stage_base + (size_t)sb * chunk_bytes + 2 * half_bytes);
        const uint32_t a_col = tmem_base + lane_field + kColA + (uint32_t)(sa * 128 + tile * 64);
#pragma unroll
        for (int h = 0; h < 2; ++h) {                      // 8 antennas -> 16 K-columns (cos, sin interleaved)
          uint32_t hi[16], lo[16];
#pragma unroll
          for (int a = 0; a < 8; ++a) {
            const double4 pp = prow[h * 8 + a];
            float cs = 0.5f, sn = 0.25f;
            if (!(dbg & 1)) phase_cs(pp.x, pp.y, pp.z, rx, ry, rz, cs, sn);
            split_tf32(cs, hi[2 * a], lo[2 * a]);
            split_tf32(sn, hi[2 * a + 1], lo[2 * a + 1]);
          }
          tmem_st16(a_col + h * 16, hi);
          tmem_st16(a_col + 32 + h * 16, lo);
        }
        tmem_wait_st();
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive(&a_full[sa]);
      }
      // ---- a3: epilogue of this collect -------------------------------------------------------------
      mbar_wait(d_full, (uint32_t)(e & 1));
      tc_fence_after();
      named_bar_sync(1, kProducerThreads);                 // weights of this collect are in shared memory
      const uint32_t d_col = tmem_base + lane_field + kColD + (uint32_t)(tile * 128);
      float pw[kMaxNE];
#pragma unroll
      for (int g = 0; g < kMaxNE / 8; ++g) {
        if (g * 8 < NE) {
          float re[8], im[8];
          tmem_ld8(d_col + g * 8, re);
          tmem_ld8(d_col + NE + g * 8, im);
          tmem_wait_ld();
#pragma unroll
          for (int t = 0; t < 8; ++t) pw[g * 8 + t] = re[t] * re[t] + im[t] * im[t];
        } else {
#pragma unroll
          for (int t = 0; t < 8; ++t) pw[g * 8 + t] = 0.f;
        }
      }
      tc_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive(d_empty);                 // D may be overwritten by the next collect
      for (int l = 0; l < n_levels; ++l) {
        const float4* dl = reinterpret_cast<const float4*>(dcur + (size_t)l * NE);
        float sacc = 0.f;
#pragma unroll
        for (int g = 0; g < kMaxNE / 4; ++g)
          if (g * 4 < NE) {
            const float4 w = dl[g];
            sacc = fmaf(w.x, pw[4 * g], sacc);
            sacc = fmaf(w.y, pw[4 * g + 1], sacc);
            sacc = fmaf(w.z, pw[4 * g + 2], sacc);
            sacc = fmaf(w.w, pw[4 * g + 3], sacc);
          }
        lev[(size_t)l * kProducerThreads + tid] += sacc;
      }
    }
    if (ok)
      for (int l = 0; l < n_levels; ++l) img[(size_t)l * img_stride + j] += lev[(size_t)l * kProducerThreads + tid];
  } else if (warp == 8) {
    // ===================== MMA issuer =====================
    if (lane == 0) {
      const uint32_t idesc = (1u << 4) | (2u << 7) | (2u << 10) | ((uint32_t)(N >> 3) << 17) | ((128u >> 4) << 24);
      int n = 0;
      for (int e = 0; e < n_collects; ++e) {
        mbar_wait(d_empty, (uint32_t)((e & 1) ^ 1));
        tc_fence_after();
        for (int c = 0; c < n_chunks; ++c, ++n) {
          const int sa = n % kSA, sb = n % kSB;
          mbar_wait(&a_full[sa], (uint32_t)((n / kSA) & 1));
          mbar_wait(&b_full[sb], (uint32_t)((n / kSB) & 1));
          tc_fence_after();
          const uint32_t b_hi = smem_u32(stage_base + (size_t)sb * chunk_bytes), b_lo = b_hi + half_bytes;
#pragma unroll
          for (int t = 0; t < 2; ++t) {
            const uint32_t d = tmem_base + kColD + t * 128;
            const uint32_t a_hi = tmem_base + kColA + sa * 128 + t * 64, a_lo = a_hi + 32;
#pragma unroll
            for (int pass = 0; pass < 3; ++pass)
#pragma unroll
              for (int kk = 0; kk < kK / 8; ++kk) {
                const uint32_t a = (pass == 1 ? a_lo : a_hi) + kk * 8;
                const uint64_t bd = make_b_desc((pass == 2 ? b_lo : b_hi) + kk * 2 * lbo, lbo, sbo);
                if (!(dbg & 2)) mma_tf32_ts(d, a, bd, idesc, (c | pass | kk) != 0 ? 1u : 0u);
              }
          }
          tc_commit(&a_empty[sa]);
          if (CS > 1) tc_commit_mc(&b_empty[sb], (uint16_t)((1u << CS) - 1)); else tc_commit(&b_empty[sb]);
          if (c == n_chunks - 1) tc_commit(d_full);
        }
      }
    }
  } else {
    // ===================== B / p' loader =====================
    if (lane == 0) {
      for (int n = 0; n < total; ++n) {
        const int sb = n % kSB;
        mbar_wait(&b_empty[sb], (uint32_t)(((n / kSB) & 1) ^ 1));
        const int e = n / n_chunks, c = n - e * n_chunks;
        const unsigned char* src = packed + (size_t)e * packed_stride + slab_offset + (size_t)c * chunk_bytes;
        mbar_expect_tx(&b_full[sb], chunk_bytes);
        if (CS > 1) {
          const uint32_t part = chunk_bytes / CS, off = cluster_rank() * part;
          bulk_g2s_mc(stage_base + (size_t)sb * chunk_bytes + off, src + off, part, &b_full[sb], (uint16_t)((1u << CS) - 1));
        } else {
          bulk_g2s(stage_base + (size_t)sb * chunk_bytes, src, chunk_bytes, &b_full[sb]);
        }
      }
    }
  }
  tc_fence_before();
  __syncthreads();
  if (CS > 1) cluster_sync_all();          // no CTA exits while a peer may still multicast into it
  if (warp == 8) {
    tc_fence_after();
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "r"(kTmemCols));
  }
}

// ---------------------------------------------------------------------------- preparation (a0'')
// One thread per (antenna, eigenpair) of the padded operand: centre, fold the constant phase into B in fp64
// (as prep_fp32_kernel), split hi/lo and scatter the four real entries into the UMMA canonical tiles.
__global__ void __launch_bounds__(256)
prep_tc_kernel(PrepArgs a, int NE, int n_slabs, int n_chunks, int n_eig_pad, int n_ant_pad, size_t chunk_bytes) {
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

  const int N = 2 * NE;
  const size_t half_bytes = (size_t)kK * N * 4;
  const int64_t gid = (int64_t)blockIdx.x * 256 + tid;
  const int64_t n_elem = (int64_t)n_ant_pad * n_eig_pad;
  if (gid < n_elem) {
    const int i = (int)(gid / n_eig_pad), k = (int)(gid - (int64_t)i * n_eig_pad);
    double px = 0, py = 0, pz = 0;
    float br = 0.f, bi = 0.f;
    if (i < a.n_ant) {
      px = (a.xyz[i] - cen[0]) / a.wavelength;
      py = (a.xyz[i + a.ldxyz] - cen[1]) / a.wavelength;
      pz = (a.xyz[i + 2 * (size_t)a.ldxyz] - cen[2]) / a.wavelength;
      if (k < a.n_eig) {
        double th = px * a.rc[0] + py * a.rc[1] + pz * a.rc[2];
        th -= rint(th);
        double sn, cs;
        sincospi(2.0 * th, &sn, &cs);
        const bb_c32 b = a.B[i + (size_t)k * a.ldb];
        br = (float)((double)b.re * cs + (double)b.im * sn);
        bi = (float)((double)b.im * cs - (double)b.re * sn);
      }
    }
    const int slab = k / NE, kk = k - slab * NE;
    const int c = i / kAC, ii = i - c * kAC;
    unsigned char* chunk = a.packed + ((size_t)slab * n_chunks + c) * chunk_bytes;
    auto put = [&](int n, int kidx, float v) {
      const size_t off = (size_t)(kidx >> 2) * ((size_t)(N / 8) * 128) + (size_t)(n >> 3) * 128 + (size_t)(n & 7) * 16 + (size_t)(kidx & 3) * 4;
      uint32_t hi, lo;
      split_tf32(v, hi, lo);
      *reinterpret_cast<uint32_t*>(chunk + off) = hi;
      *reinterpret_cast<uint32_t*>(chunk + half_bytes + off) = lo;
    };
    put(kk, 2 * ii, br);            // (Re,k)  x (i,cos)
    put(kk, 2 * ii + 1, bi);        // (Re,k)  x (i,sin)
    put(NE + kk, 2 * ii, bi);       // (Im',k) x (i,cos)
    put(NE + kk, 2 * ii + 1, -br);  // (Im',k) x (i,sin)
    if (kk == 0) {
      double* pp = reinterpret_cast<double*>(chunk + 2 * half_bytes) + (size_t)ii * 4;
      pp[0] = px; pp[1] = py; pp[2] = pz; pp[3] = 0.0;
    }
  }
  const int64_t n_w = (int64_t)a.n_levels * n_eig_pad;
  if (gid < n_w) {
    const int l = (int)(gid / n_eig_pad), k = (int)(gid - (int64_t)l * n_eig_pad);
    a.weights[gid] = (k < a.n_eig) ? a.D[l + (size_t)k * a.ldd] : 0.f;
  }
}

}  // namespace

TcPlan bb_tc_plan(int n_ant, int n_eig, int n_levels) {
  TcPlan p{};
  p.AC = kAC;
  int ne = (n_eig + 7) / 8 * 8;
  if (ne > kMaxNE) ne = kMaxNE;
  p.eig_per_slab = ne;
  p.NB = 2 * ne;
  p.n_slabs = (n_eig + ne - 1) / ne;
  p.n_chunks = (n_ant + kAC - 1) / kAC;
  p.n_eig_pad = p.n_slabs * ne;
  p.n_ant_pad = p.n_chunks * kAC;
  p.chunk_bytes = 2 * (size_t)kK * p.NB * 4 + (size_t)kAC * 32;
  p.collect_bytes = (size_t)p.n_slabs * p.n_chunks * p.chunk_bytes;
  p.weight_floats = (size_t)n_levels * p.n_eig_pad;
  return p;
}

int bb_launch_prep_tc(const TcPlan& plan, const PrepArgs& a, cudaStream_t st) {
  const int64_t n_elem = (int64_t)plan.n_ant_pad * plan.n_eig_pad;
  const int64_t n_w = (int64_t)a.n_levels * plan.n_eig_pad;
  const int64_t n = n_elem > n_w ? n_elem : n_w;
  prep_tc_kernel<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(a, plan.eig_per_slab, plan.n_slabs, plan.n_chunks,
                                                              plan.n_eig_pad, plan.n_ant_pad, plan.chunk_bytes);
  BB_CUDA(cudaGetLastError());
  return BB_OK;
}

template <int CS>
static int launch_tc(const TcPlan& plan, const SynthArgs& a, cudaStream_t st, int* launches, int dbg) {
  const int NE = plan.eig_per_slab;
  const size_t smem = align_up((size_t)kSB * plan.chunk_bytes, 1024) + (size_t)a.n_levels * kProducerThreads * 4 +
                      2 * (size_t)a.n_levels * NE * 4 + (2 * kSB + 2 * kSA + 2) * 8 + 16 + 1024;
  auto kern = synth_tc_kernel<CS>;
  BB_CUDA(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  int64_t tiles = (a.n_pix + kProducerThreads - 1) / kProducerThreads;
  tiles = (tiles + CS - 1) / CS * CS;     // whole clusters; surplus CTAs own no pixel but take part in the B exchange
  cudaLaunchConfig_t cfg{};
  cfg.gridDim = dim3((unsigned)tiles);
  cfg.blockDim = dim3(kThreadsTC);
  cfg.dynamicSmemBytes = smem;
  cfg.stream = st;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeClusterDimension;
  attr[0].val.clusterDim.x = CS; attr[0].val.clusterDim.y = 1; attr[0].val.clusterDim.z = 1;
  cfg.attrs = attr; cfg.numAttrs = 1;
  for (int slab = 0; slab < plan.n_slabs; ++slab) {
    BB_CUDA(cudaLaunchKernelEx(&cfg, kern, a.rprime, a.n_pix, a.pix_stride, a.packed, a.packed_stride,
                               (size_t)slab * plan.n_chunks * plan.chunk_bytes, a.weights, a.weight_stride, plan.n_eig_pad,
                               slab * NE, NE, a.n_collects, plan.n_chunks, a.n_levels, a.img, a.img_stride, dbg));
    ++*launches;
  }
  return BB_OK;
}

int bb_launch_synth_tc(const TcPlan& plan, const SynthArgs& a, int /*sm_count*/, cudaStream_t st, int* launches) {
  *launches = 0;
  if (a.n_collects <= 0 || a.n_pix <= 0) return BB_OK;
  const int dbg = getenv("BB_TC_DEBUG") ? atoi(getenv("BB_TC_DEBUG")) : 0;        // timing experiments only
  const int cs = getenv("BB_TC_CLUSTER") ? atoi(getenv("BB_TC_CLUSTER")) : 2;
  if (cs == 1) return launch_tc<1>(plan, a, st, launches, dbg);
  if (cs == 4) return launch_tc<4>(plan, a, st, launches, dbg);
  return launch_tc<2>(plan, a, st, launches, dbg);
}
