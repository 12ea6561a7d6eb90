// Internal declarations shared by the translation units of libbluebild_b200.so.
// Nothing here is part of the ABI (include/bluebild.h is) and nothing here is used by oracle/.
#pragma once
#include <cuda_runtime.h>
#include <cstdint>
#include <cstddef>
#include <vector>

#include "../../include/bluebild.h"

#define BB_CUDA(call)                                         \
  do {                                                        \
    cudaError_t err__ = (call);                               \
    if (err__ != cudaSuccess) { bb_note_cuda_error(err__, #call, __FILE__, __LINE__); return BB_ECUDA; } \
  } while (0)

void bb_note_cuda_error(cudaError_t err, const char* what, const char* file, int line);

// ------------------------------------------------------------------------------------------
// Packed per-collect operand layout of the FP32 synthesizer.
//   eigenpairs are padded to n_slabs * GC * KT; antennas to n_chunks * AC.
//   collect buffer = [slab][chunk]{ B part: AC x (GC*KT/2) float4 (br_2q, br_2q+1, bi_2q, bi_2q+1)
//                                   P part: AC x 4 double (p'_x, p'_y, p'_z, 0) }
//   weights        = [level][n_eig_pad] float
// B already carries the per-antenna constant phase exp(-j 2 pi <p'_i, r_c>) (centring identity).
struct Fp32Plan {
  int KT;        // eigenpairs per thread (template parameter of the kernel)
  int PT;        // pixels per thread
  int GC;        // eigen-groups per CTA (CTA = 128 threads = GC groups of 128/GC threads)
  int AC;        // antennas per staged chunk
  int MINB;      // __launch_bounds__ min CTAs per SM the kernel is compiled for
  int n_slabs;   // ceil(n_eig / (GC*KT))
  int n_chunks;  // ceil(n_ant / AC)
  int n_eig_pad; // n_slabs * GC * KT
  int n_ant_pad; // n_chunks * AC
  size_t chunk_bytes;    // AC * (GC*KT*8 + 32)
  size_t collect_bytes;  // n_slabs * n_chunks * chunk_bytes
  size_t weight_floats;  // n_levels * n_eig_pad
};

Fp32Plan bb_fp32_plan(int n_ant, int n_eig, int n_levels);

// Packed operand layout of the tensor-core (3xTF32 / 3xFP16) synthesizers; see kernels_tc.cu.
enum { BB_TC_TF32 = 0, BB_TC_FP16 = 1, BB_TC_F16F8 = 2 };
struct TcPlan {
  int mode;          // BB_TC_TF32, BB_TC_FP16 or BB_TC_F16F8
  int AC;            // antennas per K-chunk (K = 2*AC real columns per pass)
  int NB;            // N of the MMA = 2 * n_eig_pad_slab (Re | Im' halves)
  int n_slabs, n_chunks, n_eig_pad, n_ant_pad, eig_per_slab;
  size_t chunk_bytes;    // B_hi + B_lo tiles in UMMA canonical layout + antenna records
  size_t collect_bytes;
  size_t weight_floats;
};
TcPlan bb_tc_plan(int n_ant, int n_eig, int n_levels, int mode);

struct PrepArgs {
  const bb_c32* B; int ldb;           // device
  const float* D; int ldd;            // device
  const double* xyz; int ldxyz;       // device
  int n_ant, n_eig, n_levels;
  double wavelength;
  double rc[3];
  double rmax;                        // upper bound of |r'| over the handle's pixels (range check of the phase generator)
  unsigned char* packed;              // device: collect buffer
  float* weights;                     // device: [level][n_eig_pad]
  int* status;                        // device: sticky BB_FLAG_* word of the handle
};

// Sticky device-side verdicts of a handle (read back by bb_synth_get / bb_synth_status). A collect that raises one
// contributes nothing to the images: its level weights are written as zeros.
enum { BB_FLAG_RANGE = 1, BB_FLAG_NOTPOSDEF = 2, BB_FLAG_NOCONV = 4 };

// Phase-generator range limits, checked by the prep kernels against the centred antenna positions p' (wavelengths):
//   FP32 variant:  |<p', r'>| < 2^19 turns (the fixed-point fraction is read from an fp64 sum anchored at 1.5 * 2^20);
//                  enforced as |p'|_2 * rmax < 2^19
//   tensor variants: |p'_d| < 2^23 wavelengths (IH = rint(p' 2^8) must fit an int32)
constexpr double kFp32PhaseLimit = 524288.0;
constexpr double kTcCoordLimit = 8388608.0;

int bb_launch_prep_fp32(const Fp32Plan& plan, const PrepArgs& a, cudaStream_t st);
int bb_launch_prep_tc(const TcPlan& plan, const PrepArgs& a, cudaStream_t st);

struct SynthArgs {
  const double* rprime; int64_t n_pix; int64_t pix_stride;  // r' SoA: [3][pix_stride]
  const unsigned char* packed; size_t packed_stride;       // queued collects, contiguous slots
  const float* weights; size_t weight_stride;              // floats per slot
  int n_collects, n_levels;
  float* img; int64_t img_stride;                          // [level][img_stride]
  float* scratch; int n_split;                             // [n_split][level][img_stride] partial sums of a collect-range split (NULL / 1: none)
};
// number of collect ranges a launch over n_collects is split into (1 = one CTA per pixel tile handles them all):
// generic rule (tiles, resident CTA slots of the GPU), and per kernel family
int bb_collect_split(int64_t tiles, int n_collects, int cta_slots);
int bb_tc_split(int64_t n_pix, int n_collects, int sm_count);
int bb_fp32_split(const Fp32Plan& plan, int64_t n_pix, int n_collects, int sm_count);
// img[l][j] += sum_s scratch[s][l][j], s ascending (deterministic)
int bb_launch_reduce_splits(const float* scratch, int n_split, int n_levels, int64_t n_pix, int64_t stride, float* img, cudaStream_t st);
// returns number of kernels launched in *launches
int bb_launch_synth_fp32(const Fp32Plan& plan, const SynthArgs& a, int sm_count, cudaStream_t st, int* launches);
int bb_launch_synth_tc(const TcPlan& plan, const SynthArgs& a, int sm_count, cudaStream_t st, int* launches);

// pixel preparation: bounding-box centre r_c, r' = r - r_c (SoA fp64) and rmax = half the box diagonal >= max |r'|
int bb_pixels_prepare(const double* pix_dev, int64_t n_pix, int64_t ld_pix, double* rprime,
                      int64_t pix_stride, double rc_out[3], double* rmax_out, cudaStream_t st);

// uniform weighting (Section 3.5, weighting.cu): the uv sampling-density grid as the kernels see it
struct UvGridView {
  int* count;          // device: (2 half + 1)^2 counters, cell (cu, cv) at (cv + half) * (2 half + 1) + cu + half
  int half;
  double cell;         // 1 / FoV, wavelengths
  double eu[3], ev[3]; // image-plane axes
};
// cell of the visibility (p, q): baseline (x_p - x_q) / lambda_w projected on (e_u, e_v), nearest cell, clamped to the grid
__device__ __forceinline__ size_t bb_uv_cell(const UvGridView& g, const double* __restrict__ xyz, int ld, int p, int q, double wavelength) {
  const double px = xyz[p], py = xyz[p + ld], pz = xyz[p + 2 * (size_t)ld];
  const double qx = xyz[q], qy = xyz[q + ld], qz = xyz[q + 2 * (size_t)ld];
  const double up = (px * g.eu[0] + py * g.eu[1] + pz * g.eu[2]) / wavelength, uq = (qx * g.eu[0] + qy * g.eu[1] + qz * g.eu[2]) / wavelength;
  const double vp = (px * g.ev[0] + py * g.ev[1] + pz * g.ev[2]) / wavelength, vq = (qx * g.ev[0] + qy * g.ev[1] + qz * g.ev[2]) / wavelength;
  double cu = rint((up - uq) / g.cell), cv = rint((vp - vq) / g.cell);
  const double h = (double)g.half;
  cu = fmin(fmax(cu, -h), h); cv = fmin(fmax(cv, -h), h);
  return (size_t)((long long)cv + g.half) * (2 * (size_t)g.half + 1) + (size_t)((long long)cu + g.half);
}
struct bb_uvgrid;
const UvGridView* bb_uvgrid_view(const bb_uvgrid* g);

// glue (Alg. 1 lines 2-4) — glue.cu; everything is batched over collects and asynchronous on the given stream
struct GlueWork;
struct SubspaceWork;
enum { GB_PSI = 0, GB_G, GB_W, GB_T, GB_S, GB_LAM, GB_VSEL, GB_B, GB_PTRS, GB_WORK, GB_SUB0, GB_SUB1, GB_SUB2, GB_SUB3, GB_SUB4, GB_SUB5,
       kGlueBuffers };
int bb_glue_create(GlueWork** out);
void bb_glue_destroy(GlueWork* g);
int bb_glue_grow(GlueWork* g, int slot, size_t bytes, cudaStream_t st);   // scratch array `slot` of at least `bytes`
void* bb_glue_buffer(GlueWork* g, int slot);
struct GlueBatch {
  int nb, n_ant, n_beam, n_eig, gram_mode;
  const double* wavelength; int64_t stride_wl;       // device, one per collect
  const bb_c32* W; int ldw; int64_t stride_w;        // device or NULL; stride_w == 0: one W for all collects
  const bb_c32* S; int lds; int64_t stride_s;        // device
  const double* xyz; int ldxyz; int64_t stride_xyz;  // device
  double* lambda_dev; int64_t stride_lam;            // out: n_eig eigenvalues per collect, descending
  bb_c32* B_dev; int64_t stride_b;                   // out: B = W V, n_ant x n_eig complex64, ld n_ant
  const UvGridView* uv;                              // NULL = natural weighting; else S_pq is divided by the density of its uv cell
  int* info_dev;                                     // out: [2 nb] Cholesky verdicts, then eigensolver verdicts
  cudaEvent_t ev_gram0, ev_gram1, ev_eig0, ev_eig1;  // may be null
};
int bb_glue_eig_batch(GlueWork* g, cudaStream_t st, const GlueBatch& a, int* launches);
struct FilterList { int n; int kind[BB_MAX_FILTERS]; };
// D[f * n_intervals + i, k] = d_f(lambda_k) [min_i <= lambda_k <= max_i]; zeros + status flag when *info_* != 0
int bb_launch_level_weights(const double* lambda_dev, int n_eig, const double* intervals_dev, int ld_int,
                            int n_intervals, FilterList filters, float* D_dev, int ldd, const int* info_chol,
                            const int* info_eig, int* status_dev, cudaStream_t st);

// leading eigenpairs of nb Hermitian matrices by block subspace iteration (eig_subspace.cu). On return *used says
// whether the fast path produced the result (vectors / values descending in *vecs / *lams) or the caller must run
// the full eigensolve on C (left untouched in that case).
void bb_subspace_destroy(SubspaceWork* w);

// parameter estimation (estimate.cu); all pointers are device pointers
int bb_estimate_n_eig_dev(const double* lam_dev, int n, double fraction, int* out_dev, cudaStream_t st);
size_t bb_kmeans_workspace_doubles(int n);
size_t bb_kmeans_workspace_ints(int n, int k);
int bb_kmeans_levels_dev(const double* lam_dev, int n, int k, int log_domain, double* ws, int* arg, double* iv_dev, int ld_int,
                         int* status_dev, cudaStream_t st);
