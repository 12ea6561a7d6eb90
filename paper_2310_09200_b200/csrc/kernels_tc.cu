// tcgen05 tensor-core variants of the fused Standard Synthesizer (sm_100a): 3xTF32 and 3xFP16 split precision.
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
// Split precision: x = hi + lo with hi, lo in the 11-bit-significand tensor format (TF32, or FP16 with the
// B columns pre-scaled by a power of two into FP16's range and the weights D[l,k] divided by its square);
// D += A_hi B_hi + A_lo B_hi + A_hi B_lo with fp32 accumulation in TMEM (lo*lo ~ 2^-22 dropped).
// FP16 carries the same significand as TF32 at twice the tensor rate and half the operand bytes.
// A third mode (F16F8) keeps the FP16 main pass and runs BOTH cross terms as one FP8 pass at twice the FP16 rate:
//     D += A_hi16 B_hi16  +  [ e5m2(A_lo) | e5m2(A) ] . [ e5m2(B) ; e5m2(B_lo) ]      (K doubled, kind::f8f6f4)
//   2 FP16-pass units instead of 3; the cross terms are 2^-11 of the result, so their 3-bit significands cost
//   ~2^-14 (measured rel-L2 < 1e-5).
//
// Phase generator (a1) WITHOUT fp64: DFMA shares hardware with the tensor pipe on B200 (round-1 probe: a dependent
// DFMA chain runs 2.6x slower, independent DFMAs 13x lower throughput, while tcgen05.mma is streaming),
// and the 3-DFMA reduction of kernels_fp32.cu made
// the producers serialise with the MMAs), so the range reduction is done in exact integer arithmetic:
//     p'_d = IH_d 2^-8 + PL_d      (IH = rint(p' 2^8) int32, |PL| <= 2^-9; per antenna, written by prep)
//     r'_d = JH_d 2^-24 + RL_d     (JH = rint(r' 2^24) int32, |RL| <= 2^-25; per pixel, once per thread)
//     frac(<p', r'>) = [ sum_d IH_d * JH_d mod 2^32 ] 2^-32  +  sum_d ( PH_d RL_d + PL_d r'_d )      (turns)
//   three wrapping 32-bit IMADs give the large part exactly; the small part (< 2^-6 turns) is bilinear of rank 6:
//   TF32 mode evaluates it with 6 fp32 FMAs per (antenna, pixel); FP16 mode runs it as a K = 16 mini-GEMM on the
//   tensor core (pixels x 16 antennas per chunk, hi/lo of both sides folded into K) whose result lands in the
//   lo half of the A stage the producers fill next. The 32-bit fraction becomes a float by an integer add onto
//   an exponent pattern (no I2F on the MUFU pipe), then one FFMA and MUFU.SIN/COS.
//
// CTA = 2 pixel tiles of 128 (256 pixels), 1 CTA per SM, all 512 TMEM columns; G producer groups (FP16 modes: 3 groups,
// 864 threads at 72 registers; TF32 mode: 2 groups, 608 threads):
//   warps 0 .. 8G-1  producers + epilogue (groups take chunks in turn): phase generator, hi/lo split,
//              tcgen05.st of their A rows straight into TMEM (A operand from TMEM: no smem round trip);
//              per collect: tcgen05.ld of D, |E|^2, level weights, level sums.
//   warps 8G, 8G+1   one elected thread per pixel tile issues tcgen05.mma.cta_group::1 (A from TMEM, B from smem
//              descriptors) and tcgen05.commit to the stage / accumulator mbarriers; warp 8G owns TMEM alloc.
//   warp 8G+2  one elected thread streams the pre-tiled B chunks (UMMA canonical K-major no-swizzle
//              layout, written by prep_tc_kernel) global -> shared with cp.async.bulk on mbarriers.
// Small images: grid.y splits every tile's collects into ranges so that the CTA count fills whole waves of SMs
// (bb_tc_split); the ranges' level sums are added in a fixed order by reduce_splits_kernel.
#include "internal.h"
#include <cuda_fp16.h>
#include <cuda_fp8.h>

namespace {

constexpr int kTilePixels = 256;        // pixels per CTA (2 tiles of 128 TMEM lanes)
constexpr int kAC = 16;                 // antennas per chunk
constexpr int kK = 2 * kAC;             // K-columns (cos, sin per antenna) per chunk and pass
constexpr int kRec = 48;                // bytes of one antenna record {IH[3],0 | 2pi PH[3],0 | 2pi PL[3],0}
constexpr int kMaxNE = 64;              // eigenpairs per slab
constexpr uint32_t kTmemCols = 512;
constexpr uint32_t kColD = 0;           // D of tile t at kColD + 128 t (+ 64 for the second buffer when N <= 64)
constexpr int kLsTile = 512;            // bytes of one mini-GEMM B operand tile (16 antennas x 16 halves)
constexpr float kTwoPi = 6.283185307179586f;

template <int MODE> struct Cfg;
template <> struct Cfg<BB_TC_TF32> {    // 4-byte operands: 32 A columns per (tile, hi|lo); small phase part on CUDA cores
  static constexpr int kElem = 4, kSA = 2, kSB = 4, kColsHalf = kK, kMmaPerPass = kK / 8;
  static constexpr int kGroups = 2;     // producer groups taking chunks in turn
  static constexpr uint32_t kFmt = 2;   // instruction-descriptor operand format: TF32
  static constexpr bool kLsOnTensor = false;
  static constexpr uint32_t kColLs = 0;                  // unused
  static constexpr uint32_t kColA = 256;                 // A stages start
  static constexpr int kTail = kAC * kRec;               // chunk tail: antenna records
};
template <> struct Cfg<BB_TC_FP16> {    // 2-byte operands: (cos, sin) of one antenna share a 32-bit column
  static constexpr int kElem = 2, kSA = 3, kSB = 6, kColsHalf = kK / 2, kMmaPerPass = kK / 16;
  static constexpr int kGroups = 3;     // one producer group per A stage
  static constexpr uint32_t kFmt = 0;   // F16
  static constexpr bool kLsOnTensor = true;              // small phase part as a K=16 mini-GEMM (see below)
  static constexpr uint32_t kColLs = 256;                // mini-GEMM A operand (per-pixel constants): 8 columns per tile
  static constexpr uint32_t kColA = 272;                 // A stages start (the mini-GEMM writes ls into a stage's lo half)
  static constexpr int kTail = 2 * kLsTile + kAC * 16;   // chunk tail: B1 | B2 (mini-GEMM operands) | IH records
};

template <> struct Cfg<BB_TC_F16F8> : Cfg<BB_TC_FP16> {};   // same tiles and TMEM plan; the lo half holds the FP8 cross-term operand

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
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1, %2;\n\t"
      "@p bra DONE_%=;\n\t"
      "bra WAIT_%=;\n\t"
      "DONE_%=:\n\t}" ::"r"(smem_u32(bar)), "r"(parity), "r"(0x989680u) : "memory");   // suspend-time hint: sleep, do not poll
}
// Wait for two barriers at once: both try_waits are in flight together, so the common "both already complete"
// case costs one barrier latency. Safe only when neither barrier can complete a further phase before this
// thread acts (true for every pair used below).
__device__ __forceinline__ void mbar_wait2(uint64_t* bar_a, uint32_t parity_a, uint64_t* bar_b, uint32_t parity_b) {
  asm volatile(
      "{\n\t.reg .pred p, q;\n\t"
      "WAIT_%=:\n\t"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1, %4;\n\t"
      "mbarrier.try_wait.parity.shared::cta.b64 q, [%2], %3, %4;\n\t"
      "and.pred p, p, q;\n\t"
      "@p bra DONE_%=;\n\t"
      "bra WAIT_%=;\n\t"
      "DONE_%=:\n\t}" ::"r"(smem_u32(bar_a)), "r"(parity_a), "r"(smem_u32(bar_b)), "r"(parity_b), "r"(0x989680u) : "memory");
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
__device__ __forceinline__ bool elect_one() {           // one lane of a converged warp
  uint32_t pred;
  asm volatile("{\n\t.reg .pred p;\n\telect.sync _|p, 0xffffffff;\n\tselp.u32 %0, 1, 0, p;\n\t}" : "=r"(pred));
  return pred != 0;
}
__device__ __forceinline__ void named_bar_sync(int id, int n) { asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(n) : "memory"); }

// D[tmem] (+)= A[tmem] * B[smem desc]; cta_group::1
template <int MODE>
__device__ __forceinline__ void mma_ts(uint32_t d_tmem, uint32_t a_tmem, uint64_t b_desc, uint32_t idesc, uint32_t accumulate) {
  if (MODE == BB_TC_TF32)
    asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
                 "tcgen05.mma.cta_group::1.kind::tf32 [%0], [%1], %2, %3, p;\n\t}" ::"r"(d_tmem), "r"(a_tmem), "l"(b_desc), "r"(idesc), "r"(accumulate) : "memory");
  else
    asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
                 "tcgen05.mma.cta_group::1.kind::f16 [%0], [%1], %2, %3, p;\n\t}" ::"r"(d_tmem), "r"(a_tmem), "l"(b_desc), "r"(idesc), "r"(accumulate) : "memory");
}
// D[tmem] (+)= A[tmem] * B[smem desc]; kind::f8f6f4 (the FP8 cross-term pass of F16F8 mode), K = 32 per instruction
__device__ __forceinline__ void mma_ts_f8(uint32_t d_tmem, uint32_t a_tmem, uint64_t b_desc, uint32_t idesc, uint32_t accumulate) {
  asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
               "tcgen05.mma.cta_group::1.kind::f8f6f4 [%0], [%1], %2, %3, p;\n\t}" ::"r"(d_tmem), "r"(a_tmem), "l"(b_desc), "r"(idesc), "r"(accumulate) : "memory");
}
// D[tmem] (+)= A[smem desc] * B[smem desc]; kind::f16 (the mini-GEMM of the small phase part)
__device__ __forceinline__ void mma_ss_f16(uint32_t d_tmem, uint64_t a_desc, uint64_t b_desc, uint32_t idesc, uint32_t accumulate) {
  asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
               "tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n\t}" ::"r"(d_tmem), "l"(a_desc), "l"(b_desc), "r"(idesc), "r"(accumulate) : "memory");
}
__device__ __forceinline__ void fence_proxy_async_smem() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
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
__device__ __forceinline__ void tmem_st8(uint32_t addr, uint32_t v0, uint32_t v1, uint32_t v2, uint32_t v3, uint32_t v4, uint32_t v5,
                                         uint32_t v6, uint32_t v7) {
  asm volatile("tcgen05.st.sync.aligned.32x32b.x8.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8};" ::"r"(addr), "r"(v0), "r"(v1), "r"(v2), "r"(v3),
               "r"(v4), "r"(v5), "r"(v6), "r"(v7) : "memory");
}
__device__ __forceinline__ void tmem_ld8(uint32_t addr, float (&v)[8]) {
  uint32_t r[8];
  asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
               : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]) : "r"(addr));
#pragma unroll
  for (int i = 0; i < 8; ++i) v[i] = __uint_as_float(r[i]);
}
__device__ __forceinline__ void tmem_ld16(uint32_t addr, float (&v)[16]) {
  uint32_t r[16];
  asm volatile("tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];"
               : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]), "=r"(r[9]),
                 "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15]) : "r"(addr));
#pragma unroll
  for (int i = 0; i < 16; ++i) v[i] = __uint_as_float(r[i]);
}
__device__ __forceinline__ void tmem_wait_ld() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }
__device__ __forceinline__ void tmem_wait_st() { asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory"); }

// Per-pixel constants of the integer phase generator.
struct PixelSplit {
  int jx, jy, jz;        // JH = rint(r' 2^24)
  float lx, ly, lz;      // RL = r' - JH 2^-24
  float fx, fy, fz;      // r' rounded to fp32
};
__device__ __forceinline__ void split_pixel(double r, int& j, float& l, float& f) {
  const double s = rint(r * 16777216.0);
  j = (int)s;
  l = (float)(r - s * (1.0 / 16777216.0));
  f = (float)r;
}
// cos / sin of 2 pi <p', r'> from one antenna record (three 16-byte words in shared memory).
__device__ __forceinline__ void phase_cs(const int4& ih, const float4& ph, const float4& pl, const PixelSplit& q, float& c, float& s) {
  const uint32_t fr = (uint32_t)ih.x * (uint32_t)q.jx + (uint32_t)ih.y * (uint32_t)q.jy + (uint32_t)ih.z * (uint32_t)q.jz;
  float ls = ph.x * q.lx;
  ls = fmaf(ph.y, q.ly, ls);
  ls = fmaf(ph.z, q.lz, ls);
  ls = fmaf(pl.x, q.fx, ls);
  ls = fmaf(pl.y, q.fy, ls);
  ls = fmaf(pl.z, q.fz, ls);
  // signed fraction of a turn, top 23 bits, as an exactly representable float (magic add, no I2F)
  const float f = __int_as_float(0x4B400000 + ((int)fr >> 9)) - 12582912.0f;
  const float x = fmaf(f, kTwoPi / 8388608.0f, ls);        // radians in (-pi - eps, pi + eps)
  c = __cosf(x);
  s = __sinf(x);
}
// Same with the small part taken from the mini-GEMM, which also carries the constant -2 pi: lsm = ls - 2 pi.
// One 16-byte word {IH_x, IH_y, IH_z, 0} per antenna. F = 1 + frac in [1, 2) is built by an integer add on the
// exponent pattern of 1.0f, so x = 2 pi F + lsm = 2 pi frac + ls lies in [0, 2 pi): 3 IMAD, LEA.HI, FFMA, then MUFU.
__device__ __forceinline__ void phase_cs_ls(const int4& ih, float lsm, int jx, int jy, int jz, float& c, float& s) {
  const uint32_t fr = (uint32_t)ih.x * (uint32_t)jx + (uint32_t)ih.y * (uint32_t)jy + (uint32_t)ih.z * (uint32_t)jz;
  const float F = __uint_as_float(0x3F800000u + (fr >> 9));
  const float x = fmaf(F, kTwoPi, lsm);
  c = __cosf(x);
  s = __sinf(x);
}
// hi = x rounded to nearest at TF32's 10-bit mantissa (add half an ulp, then clear the 13 low bits), lo = x - hi exactly;
// the tensor core truncates lo to TF32 itself (error 2^-11 of a 2^-11 term).
__device__ __forceinline__ void split_tf32(float x, uint32_t& hi, uint32_t& lo) {
  hi = (__float_as_uint(x) + 0x1000u) & 0xFFFFE000u;
  lo = __float_as_uint(x - __uint_as_float(hi));
}
// (cos, sin) -> packed FP16 pairs: hi = rn16(x), lo = rn16(x - hi); K order (cos, sin) = (low, high) half.
// x - hi is one mixed-precision FMA per value (fma.rn.f32.f16: hi * -1 + x, SASS FHFMA).
__device__ __forceinline__ void split_f16(float c, float s, uint32_t& hi, uint32_t& lo) {
  const __half2 h = __floats2half2_rn(c, s);
  hi = *reinterpret_cast<const uint32_t*>(&h);
  float lc, lsn;
  asm("{\n\t.reg .f16 a, b, m;\n\tmov.b32 {a, b}, %2;\n\tmov.b16 m, 0xBC00;\n\t"
      "fma.rn.f32.f16 %0, a, m, %3;\n\tfma.rn.f32.f16 %1, b, m, %4;\n\t}" : "=f"(lc), "=f"(lsn) : "r"(hi), "f"(c), "f"(s));
  const __half2 l = __floats2half2_rn(lc, lsn);
  lo = *reinterpret_cast<const uint32_t*>(&l);
}

// (cos, sin) -> FP16 pair hi = rn16(x) and the FP8 cross-term word {e5m2(c - hi_c), e5m2(s - hi_s), e5m2(c), e5m2(s)}
// (bytes 0..3 = the four K elements of this antenna in the FP8 pass).
__device__ __forceinline__ void split_f16f8(float c, float s, uint32_t& hi, uint32_t& x8) {
  const __half2 h = __floats2half2_rn(c, s);
  hi = *reinterpret_cast<const uint32_t*>(&h);
  float lc, lsn;
  asm("{\n\t.reg .f16 a, b, m;\n\tmov.b32 {a, b}, %2;\n\tmov.b16 m, 0xBC00;\n\t"
      "fma.rn.f32.f16 %0, a, m, %3;\n\tfma.rn.f32.f16 %1, b, m, %4;\n\t}" : "=f"(lc), "=f"(lsn) : "r"(hi), "f"(c), "f"(s));
  asm("{\n\t.reg .b16 l, a;\n\t"
      "cvt.rn.satfinite.e5m2x2.f32 l, %2, %1;\n\t"
      "cvt.rn.satfinite.e5m2x2.f32 a, %4, %3;\n\t"
      "mov.b32 %0, {l, a};\n\t}" : "=r"(x8) : "f"(lc), "f"(lsn), "f"(c), "f"(s));
}

// ---------------------------------------------------------------------------- synthesizer
// Chunk in global/shared memory (N = 2 NE rows, kK columns of kElem bytes):
//   [ B_hi : (kK*kElem/16) core columns x (N/8) row groups x (8 rows x 16 B) ][ B_lo : same ][ kAC antenna records ]
//
// Producer warps: w = 0 .. 8 G - 1; lane quadrant w & 3 (the TMEM lanes a warp may touch), tile (w >> 2) & 1,
// group w >> 3. Group g produces the chunks n = g, g + G, ..., so each SM sub-partition always holds producer
// warps in different phases of their chunk (latency hiding) while per-chunk fixed costs stay amortised over
// 16 antennas. The epilogue of collect e is deferred until a group has produced its first chunk of collect
// e + 1, so the tensor pipe restarts on ready operands as soon as D is released; the groups split the eigenpair
// columns of D between them.
//
// What paces the FP16 modes (per-warp clock64 traces) is a LOOP three chunks long, not a pipe: the A rows
// of chunk n feed MMAs behind which the mini-GEMM of chunk n + 3 writes its ls into the same A stage, and that ls is
// what the producers of chunk n + 3 need first. Hence: one producer group per A stage (a group never waits for
// another group's stage), the mini-GEMM issued straight behind the MMAs that free its columns, and the operands of
// chunk n + 3 waited for together with the A rows of chunk n.
template <int MODE>
__global__ void __launch_bounds__((8 * Cfg<MODE>::kGroups + 3) * 32, 1)
synth_tc_kernel(const double* __restrict__ rprime, int64_t n_pix, int64_t pix_stride,
                const unsigned char* __restrict__ packed, size_t packed_stride, size_t slab_offset,
                const float* __restrict__ weights, size_t weight_stride, int n_eig_pad, int eig_offset, int NE,
                int n_collects_all, int n_chunks, int n_levels, float* __restrict__ img, int64_t img_stride,
                int collects_per_split, float* __restrict__ scratch) {
  using C = Cfg<MODE>;
  // gridDim.y > 1: this CTA handles the collects [e0, e0 + n_collects) of its pixel tile and leaves its level sums in
  // scratch[blockIdx.y] (summed into the images, in a fixed order, by reduce_splits_kernel)
  const int e0 = (int)blockIdx.y * collects_per_split;
  const int n_collects = min(collects_per_split, n_collects_all - e0);
  packed += (size_t)e0 * packed_stride;
  weights += (size_t)e0 * weight_stride;
  constexpr int kGroups = C::kGroups;
  constexpr int kProducerWarps = 8 * kGroups;              // groups x 2 tiles x 4 lane quadrants
  constexpr int kThreadsTC = (kProducerWarps + 3) * 32;    // + one MMA issuer per tile + the loader
  constexpr int kOctPerGroup = (kMaxNE / 8 + kGroups - 1) / kGroups;   // eigenpair octets of D one group reduces
  constexpr int kSA = C::kSA, kSB = C::kSB;
  constexpr uint32_t kColA = C::kColA;
  constexpr uint32_t kColsStage = 4 * C::kColsHalf;                 // 2 tiles x (hi | lo)
  static_assert(kColA + kSA * kColsStage <= kTmemCols, "TMEM budget");
  extern __shared__ __align__(1024) unsigned char smem_raw[];
  const int N = 2 * NE;
  const uint32_t half_bytes = (uint32_t)kK * N * C::kElem;          // one of B_hi / B_lo
  const uint32_t chunk_bytes = 2 * half_bytes + C::kTail;
  const uint32_t lbo = (uint32_t)(N / 8) * 128, sbo = 128;

  unsigned char* stage_base = smem_raw;
  float* lev = reinterpret_cast<float*>(smem_raw + align_up((size_t)kSB * chunk_bytes, 1024));   // [2 groups][L][256]
  float* dsm = lev + kGroups * (size_t)n_levels * kTilePixels;                                         // [2][L][NE]
  uint64_t* bars = reinterpret_cast<uint64_t*>(dsm + 2 * (size_t)n_levels * NE);
  uint64_t* b_full = bars;                 // [kSB]
  uint64_t* b_empty = b_full + kSB;        // [kSB]
  uint64_t* a_full = b_empty + kSB;        // [kSA][2 tiles]
  uint64_t* a_empty = a_full + 2 * kSA;    // [kSA]
  uint64_t* d_full = a_empty + kSA;        // [2 buffers]
  uint64_t* d_empty = d_full + 2;          // [2 buffers]
  uint64_t* ls_full = d_empty + 2;         // [kSA][2 tiles]
  uint64_t* apix_full = ls_full + 2 * kSA; // [2 tiles]
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(apix_full + 2);

  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;

  if (tid == 0) {
    for (int s = 0; s < kSB; ++s) { mbar_init(&b_full[s], 1); mbar_init(&b_empty[s], 2); }      // 2: one commit per tile issuer
    for (int s = 0; s < kSA; ++s) { mbar_init(&a_full[2 * s], 4); mbar_init(&a_full[2 * s + 1], 4); mbar_init(&a_empty[s], 2); }
    mbar_init(&d_full[0], 2); mbar_init(&d_full[1], 2);
    mbar_init(&d_empty[0], kProducerWarps); mbar_init(&d_empty[1], kProducerWarps);
    for (int b = 0; b < 2 * kSA; ++b) mbar_init(&ls_full[b], 1);
    mbar_init(&apix_full[0], 4); mbar_init(&apix_full[1], 4);
    fence_barrier_init();
  }
  if (warp == kProducerWarps) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(tmem_slot)), "r"(kTmemCols));
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::);
  }
  for (int i = tid; i < kGroups * n_levels * kTilePixels; i += kThreadsTC) lev[i] = 0.f;
  for (int i = tid; i < n_levels * NE; i += kThreadsTC) {          // weights of collect 0
    const int l = i / NE, k = i - l * NE;
    dsm[i] = weights[(size_t)l * n_eig_pad + eig_offset + k];
  }
  // per-pixel constants of the phase generator (producer threads; all groups own the same 256 pixels)
  const int slot = tid & (kTilePixels - 1);                // pixel of the CTA: tile * 128 + quadrant * 32 + lane
  const int64_t j = (int64_t)blockIdx.x * kTilePixels + slot;
  const bool ok = warp < kProducerWarps && j < n_pix;
  PixelSplit q;
  split_pixel(ok ? rprime[j] : 0.0, q.jx, q.lx, q.fx);
  split_pixel(ok ? rprime[pix_stride + j] : 0.0, q.jy, q.ly, q.fy);
  split_pixel(ok ? rprime[2 * pix_stride + j] : 0.0, q.jz, q.lz, q.fz);
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = *tmem_slot;
  const int total = n_collects * n_chunks;
  // N <= 64 accumulator columns per tile: the 128 columns of a tile hold TWO accumulators, so the MMAs of collect
  // e + 1 run while the producers still read collect e (the epilogue is 8 % of a 20-collect launch otherwise)
  const bool dbuf = N <= 64;

  if (warp < kProducerWarps) {
    // ===================== producers / epilogue: one pixel (TMEM lane) per thread =====================
    const int group = warp >> 3, tile = (warp >> 2) & 1;
    const int ptid = tid;                                  // 0 .. 256 G - 1 over all groups
    const uint32_t lane_field = (uint32_t)((warp & 3) * 32) << 16;
    if (C::kLsOnTensor && group == 0) {
      // A operand of the mini-GEMM in TMEM, row = pixel, K = 16 halves in 8 columns:
      //   columns 0-3 = hi of {RL 2^24 (x,y,z), r' (x,y,z), 1, 0}, columns 4-7 = lo of the same.
      const float v[7] = {q.lx * 16777216.0f, q.ly * 16777216.0f, q.lz * 16777216.0f, q.fx, q.fy, q.fz, 1.0f};
      __align__(16) __half hi[8], lo[8];
#pragma unroll
      for (int u = 0; u < 8; ++u) {
        const float x = u < 7 ? v[u] : 0.f;
        hi[u] = __float2half_rn(x);
        lo[u] = __float2half_rn(x - __half2float(hi[u]));
      }
      const uint32_t* hw = reinterpret_cast<const uint32_t*>(hi);
      const uint32_t* lw = reinterpret_cast<const uint32_t*>(lo);
      tmem_st8(tmem_base + lane_field + C::kColLs + (uint32_t)tile * 8, hw[0], hw[1], hw[2], hw[3], lw[0], lw[1], lw[2], lw[3]);
      tmem_wait_st();
      tc_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive(&apix_full[tile]);
    }
    float* mylev = lev + (size_t)group * n_levels * kTilePixels + slot;
    int woff[4];                                           // this thread's share of a collect's [level][NE] weight block
#pragma unroll
    for (int u = 0; u < 4; ++u) {
      const int i = ptid + u * kProducerWarps * 32;
      const int l = i / NE, k = i - l * NE;
      woff[u] = i < n_levels * NE ? l * n_eig_pad + eig_offset + k : -1;
    }
    int next_epi = 0, next_due = n_chunks;                 // epilogue e is due once this group produced a chunk of collect e + 1
    int sa = group % kSA, sb = group % kSB;                // this group's chunks: n = group, group + kGroups, ...
    uint32_t pa = (uint32_t)(group / kSA) & 1u, pb = 0;    // phase parities of the A / B stage rings
    for (int n = group;; n += kGroups) {
      const bool have = n < total;
      if (have) {
        if constexpr (C::kLsOnTensor) {
          // ls_full(n) also implies that the MMAs which last read this A stage have completed (same issuer, in order)
          // Two waits, not a paired one: the chunk's B stage landed long ago (the ring is kSB deep), so its check costs one
          // barrier round trip that runs under the wait for ls; the ls loop then polls ONE barrier — the polls of waiting
          // producer warps were 14 % of all issued instructions with the paired wait (ncu source page, round 2b).
          mbar_wait(&b_full[sb], pb);
          mbar_wait(&ls_full[2 * sa + tile], pa);
        } else {
          mbar_wait2(&a_empty[sa], pa ^ 1, &b_full[sb], pb);
        }
        tc_fence_after();
        const int4* rec = reinterpret_cast<const int4*>(stage_base + (size_t)sb * chunk_bytes + 2 * half_bytes);
        const uint32_t a_col = tmem_base + lane_field + kColA + (uint32_t)sa * kColsStage + (uint32_t)tile * 2 * C::kColsHalf;
        if constexpr (MODE == BB_TC_TF32) {
#pragma unroll
          for (int h = 0; h < 2; ++h) {                    // 8 antennas -> 16 K-columns (cos, sin interleaved)
            uint32_t hi[16], lo[16];
#pragma unroll
            for (int a = 0; a < 8; ++a) {
              const int4* r3 = rec + 3 * (h * 8 + a);
              float cs, sn;
              phase_cs(r3[0], *reinterpret_cast<const float4*>(r3 + 1), *reinterpret_cast<const float4*>(r3 + 2), q, cs, sn);
              split_tf32(cs, hi[2 * a], lo[2 * a]);
              split_tf32(sn, hi[2 * a + 1], lo[2 * a + 1]);
            }
            tmem_st16(a_col + h * 16, hi);
            tmem_st16(a_col + C::kColsHalf + h * 16, lo);
          }
        } else {
          // small phase part of this chunk (minus 2 pi): the mini-GEMM left it in the lo half of this A stage
          const int4* ihrec = reinterpret_cast<const int4*>(stage_base + (size_t)sb * chunk_bytes + 2 * half_bytes + 2 * kLsTile);
#pragma unroll
          for (int h = 0; h < 2; ++h) {                    // 8 antennas at a time (registers: three groups run at 72 per thread)
            float ls[8];
            tmem_ld8(a_col + C::kColsHalf + 8 * h, ls);
            tmem_wait_ld();
            uint32_t hi[8], lo[8];                         // 8 antennas -> 8 packed (cos, sin) columns
#pragma unroll
            for (int a = 0; a < 8; ++a) {
              float cs, sn;
              phase_cs_ls(ihrec[8 * h + a], ls[a], q.jx, q.jy, q.jz, cs, sn);
              if constexpr (MODE == BB_TC_F16F8) split_f16f8(cs, sn, hi[a], lo[a]);
              else split_f16(cs, sn, hi[a], lo[a]);
            }
            tmem_st8(a_col + 8 * h, hi[0], hi[1], hi[2], hi[3], hi[4], hi[5], hi[6], hi[7]);
            tmem_st8(a_col + C::kColsHalf + 8 * h, lo[0], lo[1], lo[2], lo[3], lo[4], lo[5], lo[6], lo[7]);
          }
        }
        tmem_wait_st();
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive(&a_full[2 * sa + tile]);
      }
      sa += kGroups; while (sa >= kSA) { sa -= kSA; pa ^= 1; }
      sb += kGroups; if (sb >= kSB) { sb -= kSB; pb ^= 1; }
      // ---- a3: deferred epilogues (collect e once this group had a go at collect e + 1, or at the end) ----
      while (next_epi < n_collects && (next_due <= n || !have)) {
        const int e = next_epi;
        ++next_epi;
        next_due += n_chunks;
        const float* dcur = dsm + (size_t)(e & 1) * n_levels * NE;
        const int db = dbuf ? (e & 1) : 0;                   // accumulator buffer of collect e and the parity of its use
        const uint32_t dph = dbuf ? (uint32_t)((e >> 1) & 1) : (uint32_t)(e & 1);
        mbar_wait(&d_full[db], dph);
        tc_fence_after();
        named_bar_sync(1, kProducerWarps * 32);            // weights of collect e are in shared memory; buffer (e+1)&1 is free
        float wnext[4];                                    // prefetch the weights of collect e + 1 (<= 2048 floats)
        if (e + 1 < n_collects) {
#pragma unroll
          for (int u = 0; u < 4; ++u)
            if (woff[u] >= 0) wnext[u] = weights[(size_t)(e + 1) * weight_stride + woff[u]];
        }
        const uint32_t d_col = tmem_base + lane_field + kColD + (uint32_t)(tile * 128 + db * 64);
        float2 pw[kOctPerGroup * 4];                       // |E|^2 of this group's eigenpair octets g = group, group + kGroups, ...
#pragma unroll
        for (int gg = 0; gg < kOctPerGroup; ++gg) {
          const int g = kGroups * gg + group;
          if (g * 8 < NE) {
            float re[8], im[8];
            tmem_ld8(d_col + g * 8, re);
            tmem_ld8(d_col + NE + g * 8, im);
            tmem_wait_ld();
#pragma unroll
            for (int t = 0; t < 4; ++t) {
              const float2 r2 = make_float2(re[2 * t], re[2 * t + 1]), i2 = make_float2(im[2 * t], im[2 * t + 1]);
              pw[gg * 4 + t] = __ffma2_rn(i2, i2, __fmul2_rn(r2, r2));
            }
          } else {
#pragma unroll
            for (int t = 0; t < 4; ++t) pw[gg * 4 + t] = make_float2(0.f, 0.f);
          }
        }
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive(&d_empty[db]);          // this accumulator may be overwritten by a later collect
        for (int l = 0; l < n_levels; ++l) {               // a3: I_l += sum_k D[l,k] |E_k|^2 (packed pairs over k)
          float2 sacc = make_float2(0.f, 0.f);
#pragma unroll
          for (int gg = 0; gg < kOctPerGroup; ++gg) {
            const int g = kGroups * gg + group;
            if (g * 8 < NE) {
              const float4* dl = reinterpret_cast<const float4*>(dcur + (size_t)l * NE + g * 8);
              const float4 w0 = dl[0], w1 = dl[1];
              sacc = __ffma2_rn(make_float2(w0.x, w0.y), pw[gg * 4], sacc);
              sacc = __ffma2_rn(make_float2(w0.z, w0.w), pw[gg * 4 + 1], sacc);
              sacc = __ffma2_rn(make_float2(w1.x, w1.y), pw[gg * 4 + 2], sacc);
              sacc = __ffma2_rn(make_float2(w1.z, w1.w), pw[gg * 4 + 3], sacc);
            }
          }
          mylev[(size_t)l * kTilePixels] += sacc.x + sacc.y;
        }
        if (e + 1 < n_collects) {
          float* dnext = dsm + (size_t)((e + 1) & 1) * n_levels * NE;
#pragma unroll
          for (int u = 0; u < 4; ++u)
            if (woff[u] >= 0) dnext[ptid + u * kProducerWarps * 32] = wnext[u];
        }
      }
      if (!have) break;
    }
    named_bar_sync(1, kProducerWarps * 32);                // all groups' level sums are complete
    if (ok && group == 0)
      for (int l = 0; l < n_levels; ++l) {                 // fixed order: bit-identical run to run
        float acc = lev[(size_t)l * kTilePixels + slot];
#pragma unroll
        for (int g = 1; g < kGroups; ++g) acc += lev[(size_t)(g * n_levels + l) * kTilePixels + slot];
        if (gridDim.y > 1) scratch[((size_t)blockIdx.y * n_levels + l) * img_stride + j] = acc;
        else img[(size_t)l * img_stride + j] += acc;
      }
  } else if (warp < kProducerWarps + 2) {
    // ===================== MMA issuers: one warp per pixel tile =====================
    // One elected thread each; every operand is warp-uniform (the TMEM base is broadcast by shuffle and the
    // thread is chosen by elect.sync) so that each tcgen05.mma costs a handful of uniform-datapath
    // instructions. A blocking mbarrier wait costs ~90 cycles even when already complete and the issuer is a
    // single serial instruction stream, so the two tiles get independent issuers and waits are paired.
    const int t = warp - kProducerWarps;                   // tile of this issuer
    const uint32_t tb = __shfl_sync(0xffffffffu, tmem_base, 0);
    if (elect_one()) {
      const uint32_t idesc = (1u << 4) | (C::kFmt << 7) | (C::kFmt << 10) | ((uint32_t)(N >> 3) << 17) | ((128u >> 4) << 24);
      const uint32_t idesc8 = (1u << 4) | (1u << 7) | (1u << 10) | ((uint32_t)(N >> 3) << 17) | ((128u >> 4) << 24);   // A, B = E5M2
      const uint64_t desc0 = make_b_desc(smem_u32(stage_base), lbo, sbo);
      const uint32_t step16 = (2 * lbo) >> 4;              // one MMA consumes two 16-byte core columns of B
      const uint32_t chunk16 = chunk_bytes >> 4, half16 = half_bytes >> 4;
      const uint32_t d0 = tb + kColD + t * 128;
      int n = 0;
      int sa = 0, sb = 0;
      uint32_t pa = 0, pb = 0;                             // phase parities of the A / B stage rings
      // mini-GEMM (FP16 mode): ls[pixel, antenna] = sum_d (2 pi PH_d RL_d + 2 pi PL_d r'_d) - 2 pi for the 16
      // antennas of chunk m, written into the lo half of A stage m % kSA, kSA chunks ahead of the main MMAs of
      // chunk m. The stage was last read by the main MMAs of chunk m - kSA, issued just before by this same thread:
      // the tensor pipe executes one thread's MMAs in order, so no barrier is needed to reuse the columns, and
      // ls_full(m) tells the producers both "ls is there" and "the stage is free".
      const uint32_t idesc_ls = (1u << 4) | ((uint32_t)(kAC >> 3) << 17) | ((128u >> 4) << 24);
      const uint64_t desc_ls0 = make_b_desc(smem_u32(stage_base) + 2 * half_bytes, 2 * 128, 128);
      const uint32_t a_pix = tb + C::kColLs + (uint32_t)t * 8;
      int sbm = 0, sam = 0;
      uint32_t pbm = 0;
      auto issue_mini = [&](bool waited) {
        if (!waited) {
          mbar_wait(&b_full[sbm], pbm);
          tc_fence_after();
        }
        const uint64_t b1 = desc_ls0 + (uint64_t)((uint32_t)sbm * chunk16), b2 = b1 + (uint64_t)(kLsTile >> 4);
        const uint32_t dl = tb + kColA + (uint32_t)sam * kColsStage + (uint32_t)t * 2 * C::kColsHalf + C::kColsHalf;
        mma_ts<BB_TC_FP16>(dl, a_pix, b1, idesc_ls, 0u);   // A_hi B_hi + A_lo B_hi
        mma_ts<BB_TC_FP16>(dl, a_pix, b2, idesc_ls, 1u);   // A_hi B_lo
        tc_commit(&ls_full[2 * sam + t]);
        if (++sbm == kSB) { sbm = 0; pbm ^= 1; }
        if (++sam == kSA) sam = 0;
      };
      constexpr int kLA = kSA;                             // chunks the mini-GEMM runs ahead of the main MMAs
      if (C::kLsOnTensor) {
        static_assert(!C::kLsOnTensor || (kSA >= 3 && kGroups <= kSA), "every group's first chunk of a collect has its ls before the accumulator hand-over");
        mbar_wait(&apix_full[t], 0);
        tc_fence_after();
        for (int m = 0; m < kLA && m < total; ++m) issue_mini(false);
      }
      for (int e = 0; e < n_collects; ++e) {
        const int db = dbuf ? (e & 1) : 0;
        const uint32_t d = d0 + (uint32_t)db * 64;
        mbar_wait(&d_empty[db], (dbuf ? (uint32_t)((e >> 1) & 1) : (uint32_t)(e & 1)) ^ 1);
        tc_fence_after();
        for (int c = 0; c < n_chunks; ++c, ++n) {
          const bool more = n + kLA < total;
          if (C::kLsOnTensor) {
            if (more) {
              // the operands of chunk n + kSA (normally long there: the B ring is kSB deep) and the A rows of chunk n
              mbar_wait2(&b_full[sbm], pbm, &a_full[2 * sa + t], pa);
            } else {
              mbar_wait(&a_full[2 * sa + t], pa);
            }
          } else {
            mbar_wait2(&b_full[sb], pb, &a_full[2 * sa + t], pa);
          }
          tc_fence_after();
          const uint64_t b_hi = desc0 + (uint64_t)((uint32_t)sb * chunk16);
          const uint64_t b_lo = b_hi + (uint64_t)half16;
          const uint32_t a_hi = tb + kColA + (uint32_t)sa * kColsStage + (uint32_t)t * 2 * C::kColsHalf, a_lo = a_hi + C::kColsHalf;
          if constexpr (MODE == BB_TC_F16F8) {
            // FP16 main pass (K = 32 halves), then both cross terms as one FP8 pass (K = 64 bytes: 2 MMAs of K = 32)
#pragma unroll
            for (int kk = 0; kk < C::kMmaPerPass; ++kk)
              mma_ts<BB_TC_FP16>(d, a_hi + kk * 8, b_hi + (uint64_t)(kk * step16), idesc, (c | kk) != 0 ? 1u : 0u);
#pragma unroll
            for (int kk = 0; kk < 2; ++kk)
              mma_ts_f8(d, a_lo + kk * 8, b_lo + (uint64_t)(kk * step16), idesc8, 1u);
          } else {
#pragma unroll
            for (int pass = 0; pass < 3; ++pass)
#pragma unroll
              for (int kk = 0; kk < C::kMmaPerPass; ++kk) {
                const uint32_t a = (pass == 1 ? a_lo : a_hi) + kk * 8;
                const uint64_t bd = (pass == 2 ? b_lo : b_hi) + (uint64_t)(kk * step16);
                mma_ts<MODE>(d, a, bd, idesc, (c | pass | kk) != 0 ? 1u : 0u);
              }
          }
          // chunk n + kSA's small phase part goes into the lo half of THIS A stage, straight behind the MMAs that read
          // it (one thread's MMAs execute in order): the ls -> producers -> A rows -> ls loop, three chunks long, is
          // what paces the kernel, so nothing else may sit between the two
          if (C::kLsOnTensor && more) issue_mini(true);
          if (!C::kLsOnTensor) tc_commit(&a_empty[sa]);
          tc_commit(&b_empty[sb]);
          if (c == n_chunks - 1) tc_commit(&d_full[db]);
          if (++sa == kSA) { sa = 0; pa ^= 1; }
          if (++sb == kSB) { sb = 0; pb ^= 1; }
        }
      }
    }
  } else {
    // ===================== B / antenna-record loader =====================
    if (elect_one()) {
      int sb = 0, e = 0, c = 0;
      uint32_t pb = 1;
      for (int n = 0; n < total; ++n) {
        mbar_wait(&b_empty[sb], pb);
        const unsigned char* src = packed + (size_t)e * packed_stride + slab_offset + (size_t)c * chunk_bytes;
        mbar_expect_tx(&b_full[sb], chunk_bytes);
        bulk_g2s(stage_base + (size_t)sb * chunk_bytes, src, chunk_bytes, &b_full[sb]);
        if (++sb == kSB) { sb = 0; pb ^= 1; }
        if (++c == n_chunks) { c = 0; ++e; }
      }
    }
  }
  tc_fence_before();
  __syncthreads();
  if (warp == kProducerWarps) {
    tc_fence_after();
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "r"(kTmemCols));
  }
}

// ---------------------------------------------------------------------------- preparation (a0'')
// One block per padded eigenpair column k: centre the antennas, fold the constant phase into B in fp64
// (as prep_fp32_kernel), scale the column into FP16 range (FP16 mode), split hi/lo and scatter the four
// real entries per antenna into the UMMA canonical tiles. The first column of a slab also writes the
// antenna records of that slab's chunks.
template <int MODE>
__global__ void __launch_bounds__(256)
prep_tc_kernel(PrepArgs a, int NE, int n_chunks, int n_eig_pad, int n_ant_pad, size_t chunk_bytes) {
  using C = Cfg<MODE>;
  __shared__ double red[3][256];
  __shared__ float redf[256];
  __shared__ double cen[3];
  const int tid = threadIdx.x;
  const int k = blockIdx.x;
  double sx = 0, sy = 0, sz = 0;
  float amax = 0.f;
  for (int i = tid; i < a.n_ant; i += 256) {
    sx += a.xyz[i]; sy += a.xyz[i + a.ldxyz]; sz += a.xyz[i + 2 * (size_t)a.ldxyz];
    if (MODE != BB_TC_TF32 && k < a.n_eig) {
      const bb_c32 b = a.B[i + (size_t)k * a.ldb];
      amax = fmaxf(amax, fmaxf(fabsf(b.re), fabsf(b.im)));
    }
  }
  red[0][tid] = sx; red[1][tid] = sy; red[2][tid] = sz; redf[tid] = amax;
  __syncthreads();
  for (int w = 128; w > 0; w >>= 1) {
    if (tid < w) {
      red[0][tid] += red[0][tid + w]; red[1][tid] += red[1][tid + w]; red[2][tid] += red[2][tid + w];
      redf[tid] = fmaxf(redf[tid], redf[tid + w]);
    }
    __syncthreads();
  }
  if (tid < 3) cen[tid] = red[tid][0] / (double)a.n_ant;
  __syncthreads();
  // range of the integer phase reduction: IH = rint(p' 2^8) must fit an int32, i.e. |p'_d| < 2^23 wavelengths; every
  // block reaches the same verdict, and a collect that fails it (NaN / Inf coordinates included) contributes nothing
  // (zero weights, zero B, zero antenna records) and raises the flag
  double far = 0.0;
  for (int i = tid; i < a.n_ant; i += 256) {
    const double dx = fabs(a.xyz[i] - cen[0]), dy = fabs(a.xyz[i + a.ldxyz] - cen[1]), dz = fabs(a.xyz[i + 2 * (size_t)a.ldxyz] - cen[2]);
    const double d = (dx + dy + dz == dx + dy + dz) ? fmax(dx, fmax(dy, dz)) : INFINITY;   // fmax would DROP a NaN: non-finite input must fail
    far = fmax(far, d);
  }
  __shared__ double redm[256];
  redm[tid] = far;
  __syncthreads();
  for (int w = 128; w > 0; w >>= 1) {
    if (tid < w) redm[tid] = fmax(redm[tid], redm[tid + w]);
    __syncthreads();
  }
  const bool in_range = redm[0] / a.wavelength < kTcCoordLimit;
  if (!in_range && blockIdx.x == 0 && tid == 0) atomicOr(a.status, BB_FLAG_RANGE);
  // FP16 mode: the column scale 2^ex puts the largest input component in [2^12, 2^13) (the phase fold can
  // grow a component by sqrt 2; FP16 overflows at 65504); the weights absorb 2^(-2 ex) exactly.
  int ex = 0;
  if (MODE != BB_TC_TF32 && redf[0] > 0.f && isfinite(redf[0])) {
    ex = 12 - ilogbf(redf[0]);
    ex = ex > 40 ? 40 : (ex < -40 ? -40 : ex);
  }
  const double scale = ldexp(1.0, ex);

  const int N = 2 * NE;
  const size_t half_bytes = (size_t)kK * N * C::kElem;
  const int slab = k / NE, kk = k - slab * NE;
  constexpr int kEpc = 16 / C::kElem;                      // elements per 16-byte core-matrix row
  for (int i = tid; i < n_ant_pad; i += 256) {
    double px = 0, py = 0, pz = 0;
    float br = 0.f, bi = 0.f;
    if (i < a.n_ant && in_range) {                            // a refused collect is packed as zeros: 0 weight x NaN |E|^2 would be NaN
      px = (a.xyz[i] - cen[0]) / a.wavelength;
      py = (a.xyz[i + a.ldxyz] - cen[1]) / a.wavelength;
      pz = (a.xyz[i + 2 * (size_t)a.ldxyz] - cen[2]) / a.wavelength;
      if (k < a.n_eig) {
        double th = px * a.rc[0] + py * a.rc[1] + pz * a.rc[2];
        th -= rint(th);
        double sn, cs;
        sincospi(2.0 * th, &sn, &cs);
        const bb_c32 b = a.B[i + (size_t)k * a.ldb];
        br = (float)(((double)b.re * cs + (double)b.im * sn) * scale);
        bi = (float)(((double)b.im * cs - (double)b.re * sn) * scale);
      }
    }
    const int c = i / kAC, ii = i - c * kAC;
    unsigned char* chunk = a.packed + ((size_t)slab * n_chunks + c) * chunk_bytes;
    auto put = [&](int n, int kidx, float v) {
      const size_t off = (size_t)(kidx / kEpc) * ((size_t)(N / 8) * 128) + (size_t)(n >> 3) * 128 + (size_t)(n & 7) * 16 +
                         (size_t)(kidx % kEpc) * C::kElem;
      if (MODE == BB_TC_TF32) {
        uint32_t hi, lo;
        split_tf32(v, hi, lo);
        *reinterpret_cast<uint32_t*>(chunk + off) = hi;
        *reinterpret_cast<uint32_t*>(chunk + half_bytes + off) = lo;
      } else if (MODE == BB_TC_FP16) {
        const __half h = __float2half_rn(v);
        *reinterpret_cast<__half*>(chunk + off) = h;
        *reinterpret_cast<__half*>(chunk + half_bytes + off) = __float2half_rn(v - __half2float(h));
      } else {
        // F16F8: FP16 main operand as above; FP8 cross-term operand (K = 64 bytes per row, 16 per core column):
        // byte 4 ii + w pairs with e5m2(A_lo) and holds e5m2(v), byte 4 ii + 2 + w pairs with e5m2(A) and holds e5m2(v - hi)
        const __half h = __float2half_rn(v);
        *reinterpret_cast<__half*>(chunk + off) = h;
        const int w = kidx & 1, ant = kidx >> 1;
        const int k8 = 4 * ant + w;
        const size_t off8 = (size_t)(k8 / 16) * ((size_t)(N / 8) * 128) + (size_t)(n >> 3) * 128 + (size_t)(n & 7) * 16 + (size_t)(k8 % 16);
        chunk[half_bytes + off8] = (unsigned char)__nv_cvt_float_to_fp8(v, __NV_SATFINITE, __NV_E5M2);
        chunk[half_bytes + off8 + 2] = (unsigned char)__nv_cvt_float_to_fp8(v - __half2float(h), __NV_SATFINITE, __NV_E5M2);
      }
    };
    put(kk, 2 * ii, br);            // (Re,k)  x (i,cos)
    put(kk, 2 * ii + 1, bi);        // (Re,k)  x (i,sin)
    put(NE + kk, 2 * ii, bi);       // (Im',k) x (i,cos)
    put(NE + kk, 2 * ii + 1, -br);  // (Im',k) x (i,sin)
    if (kk == 0) {                  // per-antenna phase-generator data (zero for padding antennas)
      const double tp = 6.283185307179586;
      const double hx = rint(px * 256.0), hy = rint(py * 256.0), hz = rint(pz * 256.0);
      int4 ih;
      ih.x = (int)hx; ih.y = (int)hy; ih.z = (int)hz; ih.w = 0;
      unsigned char* tail = chunk + 2 * half_bytes;
      if (MODE == BB_TC_TF32) {
        float4 ph, pl;
        ph.x = (float)(tp * hx / 256.0); ph.y = (float)(tp * hy / 256.0); ph.z = (float)(tp * hz / 256.0); ph.w = 0.f;
        pl.x = (float)(tp * (px - hx / 256.0)); pl.y = (float)(tp * (py - hy / 256.0)); pl.z = (float)(tp * (pz - hz / 256.0)); pl.w = 0.f;
        int4* rec = reinterpret_cast<int4*>(tail + (size_t)ii * kRec);
        rec[0] = ih;
        rec[1] = *reinterpret_cast<int4*>(&ph);
        rec[2] = *reinterpret_cast<int4*>(&pl);
      } else {
        // mini-GEMM B operand rows (N = 16 antennas, K = 16 halves, UMMA K-major no swizzle, LBO 256, SBO 128):
        //   v = {2 pi PH 2^-24 (x,y,z), 2 pi PL (x,y,z), -2 pi, 0};  B1 = [hi(v) | hi(v)],  B2 = [lo(v) | 0]
        const double v[7] = {tp * hx / 256.0 / 16777216.0, tp * hy / 256.0 / 16777216.0, tp * hz / 256.0 / 16777216.0,
                             tp * (px - hx / 256.0), tp * (py - hy / 256.0), tp * (pz - hz / 256.0), -tp};
        __align__(16) __half hi[8], lo[8];
#pragma unroll
        for (int t = 0; t < 8; ++t) {
          const float x = t < 7 ? (float)v[t] : 0.f;
          hi[t] = __float2half_rn(x);
          lo[t] = __float2half_rn(x - __half2float(hi[t]));
        }
        unsigned char* row = tail + (size_t)(ii >> 3) * 128 + (size_t)(ii & 7) * 16;
        const int4 z = make_int4(0, 0, 0, 0);
        *reinterpret_cast<int4*>(row) = *reinterpret_cast<const int4*>(hi);                    // B1 core column 0
        *reinterpret_cast<int4*>(row + 256) = *reinterpret_cast<const int4*>(hi);              // B1 core column 1
        *reinterpret_cast<int4*>(row + kLsTile) = *reinterpret_cast<const int4*>(lo);          // B2 core column 0
        *reinterpret_cast<int4*>(row + kLsTile + 256) = z;                                     // B2 core column 1
        reinterpret_cast<int4*>(tail + 2 * kLsTile)[ii] = ih;
      }
    }
  }
  // weights [level][n_eig_pad]; FP16 mode: |E|^2 comes out scaled by 2^(2 ex)
  const float wscale = (float)ldexp(1.0, -2 * ex);
  for (int l = tid; l < a.n_levels; l += 256)
    a.weights[(size_t)l * n_eig_pad + k] = (k < a.n_eig && in_range) ? a.D[l + (size_t)k * a.ldd] * wscale : 0.f;
}

// img[l][j] += sum over splits of scratch[s][l][j], splits in ascending order (deterministic)
__global__ void reduce_splits_kernel(const float* __restrict__ scratch, int n_split, int n_levels, int64_t n_pix, int64_t stride,
                                     float* __restrict__ img) {
  const int64_t j = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  const int l = blockIdx.y;
  if (j >= n_pix) return;
  float acc = img[(size_t)l * stride + j];
  for (int s = 0; s < n_split; ++s) acc += scratch[((size_t)s * n_levels + l) * stride + j];
  img[(size_t)l * stride + j] = acc;
}

template <int MODE>
int launch_prep(const TcPlan& plan, const PrepArgs& a, cudaStream_t st) {
  prep_tc_kernel<MODE><<<(unsigned)plan.n_eig_pad, 256, 0, st>>>(a, plan.eig_per_slab, plan.n_chunks, plan.n_eig_pad,
                                                                 plan.n_ant_pad, plan.chunk_bytes);
  BB_CUDA(cudaGetLastError());
  return BB_OK;
}

template <int MODE>
int launch_tc(const TcPlan& plan, const SynthArgs& a, cudaStream_t st, int* launches) {
  using C = Cfg<MODE>;
  const int NE = plan.eig_per_slab;
  constexpr int kThreadsTC = (8 * C::kGroups + 3) * 32;
  const size_t smem = align_up((size_t)C::kSB * plan.chunk_bytes, 1024) + C::kGroups * (size_t)a.n_levels * kTilePixels * 4 +
                      2 * (size_t)a.n_levels * NE * 4 + (2 * C::kSB + 5 * C::kSA + 6) * 8 + 16 + 1024;
  auto kern = synth_tc_kernel<MODE>;
  BB_CUDA(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  const int64_t tiles = (a.n_pix + kTilePixels - 1) / kTilePixels;
  const int cps = (a.n_collects + (a.scratch ? a.n_split : 1) - 1) / (a.scratch ? a.n_split : 1);
  const int n_split = (a.n_collects + cps - 1) / cps;      // ranges of cps collects that are not empty (<= a.n_split)
  for (int slab = 0; slab < plan.n_slabs; ++slab) {
    kern<<<dim3((unsigned)tiles, (unsigned)n_split), kThreadsTC, smem, st>>>(
        a.rprime, a.n_pix, a.pix_stride, a.packed, a.packed_stride, (size_t)slab * plan.n_chunks * plan.chunk_bytes, a.weights,
        a.weight_stride, plan.n_eig_pad, slab * NE, NE, a.n_collects, plan.n_chunks, a.n_levels, a.img, a.img_stride, cps, a.scratch);
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

TcPlan bb_tc_plan(int n_ant, int n_eig, int n_levels, int mode) {
  TcPlan p{};
  p.mode = mode;
  p.AC = kAC;
  int ne = (n_eig + 7) / 8 * 8;
  if (ne > kMaxNE) ne = kMaxNE;
  p.eig_per_slab = ne;
  p.NB = 2 * ne;
  p.n_slabs = (n_eig + ne - 1) / ne;
  p.n_chunks = (n_ant + kAC - 1) / kAC;
  p.n_eig_pad = p.n_slabs * ne;
  p.n_ant_pad = p.n_chunks * kAC;
  const int elem = mode == BB_TC_TF32 ? 4 : 2;
  p.chunk_bytes = 2 * (size_t)kK * p.NB * elem + (size_t)(mode == BB_TC_TF32 ? Cfg<BB_TC_TF32>::kTail : Cfg<BB_TC_FP16>::kTail);
  p.collect_bytes = (size_t)p.n_slabs * p.n_chunks * p.chunk_bytes;
  p.weight_floats = (size_t)n_levels * p.n_eig_pad;
  return p;
}

// Collect-range split for small images: the grid is one CTA per pixel tile, so n_tiles / (resident CTA slots) far from an
// integer leaves SMs idle in the last wave (config 2, tensor variants: 256 tiles on 148 SMs = 1.73 waves). Splitting every tile's collects into
// n_split ranges multiplies the CTA count; the smallest split (each range >= 4 collects) that lifts the wave efficiency
// above 95 % is taken, or none if the unsplit grid is already within 5 % of the best.
int bb_collect_split(int64_t tiles, int n_collects, int cta_slots) {
  if (tiles <= 0 || cta_slots <= 0) return 1;
  auto eff = [&](int s) {
    const int64_t ctas = tiles * s, waves = (ctas + cta_slots - 1) / cta_slots;
    return (double)ctas / (double)(waves * cta_slots);
  };
  int best = 1;
  double best_eff = eff(1);
  for (int s = 2; s <= 8 && n_collects / s >= 4; ++s) {
    if (best_eff >= 0.95) break;
    // ranges are ceil(n / s) collects long; s such ranges must all be non-empty (25 collects in 6 ranges of 5 would
    // leave the sixth empty, 33 in 8 ranges of 5 the eighth with a negative length)
    const int cps = (n_collects + s - 1) / s;
    if ((s - 1) * cps >= n_collects) continue;
    if (eff(s) > best_eff + 0.05) { best = s; best_eff = eff(s); }
  }
  return best;
}
int bb_tc_split(int64_t n_pix, int n_collects, int sm_count) {      // tensor variants: 256-pixel tiles, one CTA per SM
  return bb_collect_split((n_pix + kTilePixels - 1) / kTilePixels, n_collects, sm_count);
}
int bb_launch_reduce_splits(const float* scratch, int n_split, int n_levels, int64_t n_pix, int64_t stride, float* img, cudaStream_t st) {
  reduce_splits_kernel<<<dim3((unsigned)((n_pix + 255) / 256), (unsigned)n_levels), 256, 0, st>>>(scratch, n_split, n_levels, n_pix, stride, img);
  BB_CUDA(cudaGetLastError());
  return BB_OK;
}

int bb_launch_prep_tc(const TcPlan& plan, const PrepArgs& a, cudaStream_t st) {
  return plan.mode == BB_TC_FP16 ? launch_prep<BB_TC_FP16>(plan, a, st)
         : plan.mode == BB_TC_F16F8 ? launch_prep<BB_TC_F16F8>(plan, a, st) : launch_prep<BB_TC_TF32>(plan, a, st);
}

int bb_launch_synth_tc(const TcPlan& plan, const SynthArgs& a, int /*sm_count*/, cudaStream_t st, int* launches) {
  *launches = 0;
  if (a.n_collects <= 0 || a.n_pix <= 0) return BB_OK;
  return plan.mode == BB_TC_FP16 ? launch_tc<BB_TC_FP16>(plan, a, st, launches)
         : plan.mode == BB_TC_F16F8 ? launch_tc<BB_TC_F16F8>(plan, a, st, launches) : launch_tc<BB_TC_TF32>(plan, a, st, launches);
}
