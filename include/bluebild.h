/* bluebild.h — C ABI of the B200-native Bluebild Standard Synthesizer (libbluebild_b200.so).
 *
 * Method: arXiv 2310.09200 (BIPP), /root/reference/PAPER.md. Interface follows the paper's
 * "Context + imaging handle + collect per time step" design (Table 1
 * PAPER.md:250-258, Algorithm 1 line 1 PAPER.md:285): column-major inputs, host or device.
 *
 * Conventions for EVERY entry point
 *   - Every data pointer may be a HOST or a DEVICE pointer (classified with
 *     cudaPointerGetAttributes). Host buffers are snapshotted before the call returns. Device
 *     buffers are read in stream order with respect to the context stream: after all work that
 *     was enqueued on it when the call was made, and the context stream is made to wait for the
 *     kernel or copy that consumes them — so they may be overwritten or freed by later work on
 *     that stream, but not from the host or another stream before the context stream (or a later
 *     synchronising call: bb_synth_get / _status / _timings / _reset) has been synchronised.
 *     bb_synth_flush alone does NOT synchronise.
 *   - Work runs on streams the context owns (glue and synthesizer overlap); the
 *     context stream carries the ordering, also for results: after bb_synth_flush it waits for
 *     the synthesizer, so later work on it sees the images.
 *   - The caller owns all buffers; the library never frees or retains caller memory.
 *   - Return value: BB_OK or an error code; no exception crosses the ABI. All arguments are
 *     validated before any launch, so a failed call leaves the level images unchanged and the
 *     handle usable. Conditions only the device can see (Gram matrix not positive definite,
 *     eigensolver failure, antenna coordinates beyond the phase generator's range) do not stop
 *     the call: the offending collect contributes NOTHING to the images and a sticky flag is
 *     raised, which the next bb_synth_get / bb_synth_status returns as BB_ENOTPOSDEF /
 *     BB_ENOCONV / BB_EUNSUPPORTED (cleared by bb_synth_reset).
 *   - All matrices are column-major with an explicit leading dimension (in elements).
 *   - Complex single precision is interleaved (re, im) pairs of float (bb_c32).
 *   - There is no CPU fallback: without a CUDA device bb_ctx_create fails with BB_ECUDA.
 */
#ifndef BLUEBILD_B200_H
#define BLUEBILD_B200_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct bb_ctx bb_ctx;     /* device, stream, library handles, scratch ("Context") */
typedef struct bb_synth bb_synth; /* StandardSynthesis imaging handle                   */
typedef struct { float re, im; } bb_c32;

enum {
  BB_OK = 0,
  BB_EINVAL = 1,       /* bad argument (null pointer, non-positive size, ld too small, n_eig > n_beam ...) */
  BB_EALLOC = 2,       /* host or device allocation failed */
  BB_ECUDA = 3,        /* CUDA runtime / library error (no device, launch failure) */
  BB_ENOTPOSDEF = 4,   /* Gram matrix not positive definite (Cholesky failed) */
  BB_ENOCONV = 5,      /* eigensolver did not converge */
  BB_ESTATE = 6,       /* call not valid in the handle's state */
  BB_EUNSUPPORTED = 7  /* variant / size not supported by this build */
};

enum {
  BB_VARIANT_FP32 = 0,    /* FP32 CUDA-core synthesizer (FFMA2), fp64-reduced phases          */
  BB_VARIANT_TF32X3 = 1,  /* tcgen05 tensor-core synthesizer, 3xTF32 split, fp32 accumulation */
  BB_VARIANT_FP16X3 = 2,  /* same with the operands split into FP16 pairs (same 11-bit significand as TF32,
                             B columns pre-scaled by powers of two): twice the tensor rate            */
  BB_VARIANT_FP16_FP8 = 3 /* FP16 main pass + ONE FP8 (e5m2) pass for both cross terms (kind::f8f6f4, K doubled):
                             2 FP16-pass units instead of 3; rel-L2 ~ 8e-6 instead of ~5e-7  */
};

/* ---- context ------------------------------------------------------------------------------
 * device: CUDA ordinal. cuda_stream: a cudaStream_t (may be NULL = default stream) on which all
 * work of handles created from this context is enqueued. */
int bb_ctx_create(int device, void* cuda_stream, bb_ctx** out);
int bb_ctx_destroy(bb_ctx* ctx); /* BB_ESTATE while imaging handles created from it are alive */

/* ---- imaging handle -----------------------------------------------------------------------
 * pix: X_pix of Table 1: n_pix x 3 pixel unit vectors, column-major with leading
 * dimension ld_pix >= n_pix, float64, same sky-fixed frame as the antenna positions.
 * n_levels: number of eigenvalue intervals N_i (1..BB_MAX_LEVELS). Images start at zero. */
#define BB_MAX_LEVELS 32
#define BB_MAX_BEAMS 512
int bb_synth_create(bb_ctx* ctx, int64_t n_pix, const double* pix, int64_t ld_pix, int n_levels,
                    int variant, bb_synth** out);
int bb_synth_destroy(bb_synth* s);
int bb_synth_reset(bb_synth* s); /* drop pending collects and zero the level images */

/* ---- collect: Algorithm 1 for one time step / channel -------------------
 * G = W^H Psi W with Psi_pq = sinc(2 |x_p - x_q| / wavelength) (Eq. 11, 24; normalized sinc);
 * S v = lambda G v with V^H G V = I (Eq. 13); keep the n_eig largest lambda (Alg. 1 l.4);
 * B = W V; D[l,k] = lambda_k if intervals[l,0] <= lambda_k <= intervals[l,1] else 0 (closed
 * intervals, tested independently: overlap counts twice, uncovered eigenvalues are dropped);
 * then bb_synth_collect_eig. Glue runs in fp64 on the device.
 *   W   n_ant x n_beam complex64, ld ldw; NULL means identity (requires n_beam == n_ant)
 *   S   n_beam x n_beam complex64 Hermitian, full storage, ld lds (used as (S+S^H)/2)
 *   xyz n_ant x 3 float64 metres, ld ldxyz (P_icrs of Table 1)
 *   intervals n_levels x 2 float64, ld ld_int: column 0 = min, column 1 = max
 * Limits: 1 <= n_eig <= n_beam <= BB_MAX_BEAMS, n_ant >= 1, wavelength > 0; coordinate range as for
 * bb_synth_collect_eig. The call stages its inputs; the glue runs batched over up to 128 staged collects
 * (when 128 are staged, on bb_synth_flush, or on bb_synth_get) on the context's glue stream. */
int bb_synth_collect(bb_synth* s, int n_ant, int n_beam, int n_eig, double wavelength,
                     const bb_c32* W, int ldw, const bb_c32* S, int lds, const double* xyz,
                     int ldxyz, const double* intervals, int ld_int);

/* ---- collect_ex: Algorithm 1 with N_f filters (Alg. 1 l.6-7) and the Gram choice ----
 * filters: n_filters (1..BB_MAX_FILTERS) entries, HOST pointer, BB_FILTER_LSQ (d = lambda, Eq. 14/20) or
 * BB_FILTER_STD (d = 1, the "Standardized" image). The handle's n_levels must equal n_intervals * n_filters
 * with n_intervals = n_levels / n_filters rows in `intervals`; image index = filter * n_intervals + interval
 * (the B^(n_i, n_f) of Alg. 1 l.9). gram_mode BB_GRAM_SINC is Eq. 11/24; BB_GRAM_IDENTITY sets G := I, the
 * eigendecomposition of the dirty image (Eq. 38-40, App. A). All else as bb_synth_collect,
 * which is collect_ex with one LSQ filter and the sinc Gram. */
enum { BB_FILTER_LSQ = 0, BB_FILTER_STD = 1 };
enum { BB_GRAM_SINC = 0, BB_GRAM_IDENTITY = 1 };
#define BB_MAX_FILTERS 8
int bb_synth_collect_ex(bb_synth* s, int n_ant, int n_beam, int n_eig, double wavelength,
                        const bb_c32* W, int ldw, const bb_c32* S, int lds, const double* xyz,
                        int ldxyz, const double* intervals, int ld_int, int n_filters,
                        const int* filters, int gram_mode);

/* ---- collect_batch: Algorithm 1 for n_collects time steps / channels in one call (the
 * eigendecomposition is repeated for every time step and band). Same per-collect semantics as
 * bb_synth_collect (one LSQ filter, sinc Gram), applied in order c = 0 .. n_collects-1; the Gram matrices,
 * Cholesky factorisations and Hermitian eigensolves run as batched device calls (up to 128 collects at a time); the
 * synthesizer of one group runs while the glue of the next is in progress.
 *   wavelengths  n_collects float64, HOST pointer
 *   S, xyz       collect c starts at S + c * stride_s, xyz + c * stride_xyz (strides in elements)
 *   W            NULL (identity), or collect c at W + c * stride_w; stride_w == 0 shares one W
 * A collect whose Gram matrix is not positive definite or whose solve fails contributes nothing and raises the
 * sticky flag (see the conventions above). Does not synchronise. */
int bb_synth_collect_batch(bb_synth* s, int n_collects, int n_ant, int n_beam, int n_eig,
                           const double* wavelengths, const bb_c32* W, int ldw, int64_t stride_w,
                           const bb_c32* S, int lds, int64_t stride_s, const double* xyz, int ldxyz,
                           int64_t stride_xyz, const double* intervals, int ld_int);

/* ---- collect_eig: the hot path only (Algorithm 2 + Alg. 1 line 9, Eq. 15, 20) ---------------
 * I_l(r_j) += sum_k D[l,k] | sum_i conj(B_ik) exp(+j 2 pi <xyz_i, r_j> / wavelength) |^2
 *   B   n_ant x n_eig complex64 (= W V), ld ldb
 *   D   n_levels x n_eig float32 weights, ld ldd
 *   xyz n_ant x 3 float64, ld ldxyz
 * The call enqueues a small preparation kernel and queues the collect; the fused synthesizer
 * kernel runs when the queue is full, on bb_synth_flush, or on bb_synth_get, looping over all
 * queued collects inside one launch (every time step and band).
 * Coordinate range of the phase generator, with p' = (xyz - mean(xyz)) / wavelength and r' the pixel vectors
 * minus the centre of their bounding box: FP32 variant |p'| max|r'| < 2^19 turns; tensor variants
 * |p'_x|, |p'_y|, |p'_z| < 2^23 wavelengths. Checked on the device: a collect beyond it contributes nothing
 * and bb_synth_get / bb_synth_status return BB_EUNSUPPORTED.
 * Antenna-count limit of the tensor variants (every collect call; checked on the host, the call returns
 * BB_EUNSUPPORTED with nothing queued and the images unchanged): n_ant <= BB_MAX_ANT_TF32X3 / _FP16X3 / _FP16_FP8.
 * Reason: each tcgen05.mma that adds into the fp32 accumulator drops a fraction of an ulp, always towards zero, so
 * these variants' images are too small by a factor that grows with the number of instructions per accumulator,
 * n_ant / 16 x {12, 6, 4}: measured -2.45e-8, -1.24e-8, -0.82e-8 per antenna on one B200, i.e. -4.4e-5 for tf32x3 at
 * the 1776 antennas of BASELINE config 2 and -2.0e-4, twice the 1e-4 tolerance, at 8192 (profiles/r03_n_ant_bias.md).
 * The limits keep that shrink at or below 5.1e-5, half the tolerance, because the constant depends on how the sum
 * grows (up to 1.5x for an array whose first antennas dominate). The FP32 variant has no such term (n_ant <= 2^20):
 * arrays beamformed from more elements (Eq. 22-24) go through BB_VARIANT_FP32. */
#define BB_MAX_ANT_TF32X3 2048
#define BB_MAX_ANT_FP16X3 4096
#define BB_MAX_ANT_FP16_FP8 6144
int bb_synth_collect_eig(bb_synth* s, int n_ant, int n_eig, double wavelength, const bb_c32* B,
                         int ldb, const float* D, int ldd, const double* xyz, int ldxyz);

/* Launch the synthesizer over all queued collects now (asynchronous; does not synchronise). */
int bb_synth_flush(bb_synth* s);

/* Copy level image `level` (n_pix float32, pixel order of pix) to out (host or device).
 * Flushes pending collects and synchronises. Images are plain sums over collects (Alg. 1 line 9:
 * "+="; no division by the number of collects). The image is copied even when the return value
 * reports a sticky device-side condition (it then holds the sum of the collects that were fine). */
int bb_synth_get(bb_synth* s, int level, float* out);

/* Flush, synchronise and return the sticky device-side condition of the handle (BB_OK if none). */
int bb_synth_status(bb_synth* s);

/* Device-measured times (CUDA events, ms) accumulated since create/reset; any may be NULL. */
int bb_synth_timings(bb_synth* s, double* gram_ms, double* eig_ms, double* prep_ms, double* synth_ms);

/* Number of kernels this handle has launched since create/reset. */
int64_t bb_synth_launches(bb_synth* s);

/* ---- eigen stage alone (Alg. 1 lines 2-4), for parameter estimation ----
 * lambda_out: n_eig float64 eigenvalues, descending. B_out (may be NULL): n_ant x n_eig
 * complex64, ld ldb_out. Same argument rules as bb_synth_collect. Synchronises the stream. */
int bb_eig(bb_ctx* ctx, int n_ant, int n_beam, int n_eig, double wavelength, const bb_c32* W,
           int ldw, const bb_c32* S, int lds, const double* xyz, int ldxyz, double* lambda_out,
           bb_c32* B_out, int ldb_out);

/* ---- "uniform" image weighting (Section 3.5) ------------------------------------------------
 * "We calculate the sampling density function on a grid in uv space with Delta u = Delta v = 1/FoV. Each
 * visibility is then weighted with the inverse of its sampling density function", before the eigendecomposition.
 * A visibility is an antenna pair (p, q), p = q included; its uv point is (xyz_p - xyz_q) / wavelength projected on
 * the image-plane axes e_u, e_v (unit 3-vectors, HOST pointers); cell index = nearest integer of u / cell.
 *   bb_uvgrid_create   cell = 1 / FoV in wavelengths; max_uv = the largest |u|, |v| to resolve (baselines beyond are
 *                      counted in the border cells); (2 ceil(max_uv / cell) + 3)^2 int32 counters on the device.
 *   bb_uvgrid_add      adds the n_ant^2 visibilities of one collect (xyz n_ant x 3 float64, host or device) to the
 *                      density; call it for every time step and channel of the observation, then collect.
 *   bb_synth_set_weighting  collects made after this call divide S_pq by the density of its cell (cells never added
 *                      count as density 1); grid == NULL restores natural weighting. Only W == NULL collects (a
 *                      beamformed visibility has no single baseline): others return BB_EUNSUPPORTED. The grid must
 *                      outlive the handle's pending work (call bb_synth_status or bb_synth_get before destroying it).
 * Weighted visibility matrices may be indefinite; negative eigenvalues are handled as anywhere else. */
typedef struct bb_uvgrid bb_uvgrid;
int bb_uvgrid_create(bb_ctx* ctx, double cell, const double* e_u, const double* e_v, double max_uv, bb_uvgrid** out);
int bb_uvgrid_add(bb_uvgrid* g, int n_ant, double wavelength, const double* xyz, int ldxyz);
int bb_uvgrid_destroy(bb_uvgrid* g);
int bb_synth_set_weighting(bb_synth* s, bb_uvgrid* grid);

/* ---- level weights alone (Alg. 1 lines 7-8; filters PAPER.md:166) ----------------------
 * D_out[f * n_intervals + i, k] = d_f(lambda_k) if intervals[i,0] <= lambda_k <= intervals[i,1] else 0, with
 * d = lambda_k for BB_FILTER_LSQ and 1 for BB_FILTER_STD — the D that bb_synth_collect_eig takes, computed by the
 * same kernel bb_synth_collect uses. lambda: n_eig float64; intervals: n_intervals x 2, ld ld_int; filters:
 * n_filters entries, HOST pointer; D_out: (n_intervals * n_filters) x n_eig float32, ld ldd. Host or device
 * pointers; synchronises the context stream. */
int bb_level_weights(bb_ctx* ctx, const double* lambda, int n_eig, const double* intervals, int ld_int,
                     int n_intervals, int n_filters, const int* filters, float* D_out, int ldd);

/* ---- parameter estimation (Table 4 caption :593), device-side glue -------------
 * lambda: n (1..BB_MAX_ESTIMATE) eigenvalues in any order, host or device (one collect's, or pooled from a
 * subset of the data, e.g. from bb_eig). Both calls synchronise the context stream.
 * bb_estimate_n_eig: the smallest m such that the m largest eigenvalues hold at least energy_fraction
 *   (0 < f <= 1) of the sum of the positive eigenvalues; written to *n_eig_out (host).
 * bb_kmeans_levels: exact one-dimensional k-means (dynamic programming over the sorted values: the global
 *   minimum of the within-cluster sum of squares) of the positive eigenvalues, in the log domain if
 *   log_domain != 0. intervals_out (host or device, n_levels x 2, ld ld_int >= n_levels): level 0 = highest
 *   energy; edges at the midpoints between adjacent centroids (mapped back from the log domain), lowest
 *   edge 0, highest DBL_MAX. BB_EINVAL if fewer than n_levels positive values. */
#define BB_MAX_ESTIMATE 4096
int bb_estimate_n_eig(bb_ctx* ctx, const double* lambda, int n, double energy_fraction, int* n_eig_out);
int bb_kmeans_levels(bb_ctx* ctx, const double* lambda, int n, int n_levels, int log_domain,
                     double* intervals_out, int ld_int);

/* bb_kmeans_levels_static: bb_kmeans_levels (same kernel, same result) for callers that cannot
 * allocate device memory when they make the call: a service that laid out all of its GPU memory at start-up (a
 * streaming imager with a fixed memory plan; a process whose framework pool already owns nearly all of HBM, where
 * a raw cudaMalloc may simply fail), or a latency-bound loop, since cudaMalloc / cudaFree lock the whole device and
 * wait for it to go idle, stalling unrelated streams. It calls no cudaMalloc, cudaFree or allocating library
 * routine and needs no bb_ctx. Its dynamic-programming tables sit in a fixed array inside the library image instead:
 * about 170 KB that every GPU which loads the library holds until the process exits — hence the lower size limit.
 *   device, cuda_stream  CUDA ordinal (made current, as bb_ctx_create does; 0..63) and the cudaStream_t (NULL =
 *                        default stream) the kernel is enqueued on. The call does not synchronise.
 *   lambda_dev           n eigenvalues, any order, DEVICE memory, 1 <= n <= BB_KMEANS_STATIC_MAX_N.
 *   intervals_dev        out, DEVICE memory, n_levels x 2 column-major with ld_int >= n_levels, as bb_kmeans_levels.
 *   status_dev           out, DEVICE int: 0 = intervals written; 1 = fewer than n_levels positive eigenvalues,
 *                        intervals untouched (the case bb_kmeans_levels reports as BB_EINVAL). Read it in stream order.
 * All three buffers are the caller's, read and written in stream order on cuda_stream; host pointers are refused
 * with BB_EINVAL (staging them would take memory). n > BB_KMEANS_STATIC_MAX_N: BB_EUNSUPPORTED, nothing launched
 * (BB_VERBOSE=1 prints the limit) — use bb_kmeans_levels. Other bad arguments: BB_EINVAL.
 * First call per device = set-up: it looks up the device address of the built-in array (and may bring up the
 * device's primary context and load the module). Make that call once, early, before any stream capture begins.
 * Sharing: every call on a GPU uses the same array. Nothing in it needs clearing (the kernel writes each table
 * entry before reading it; what the previous call left is never read), but calls whose kernels OVERLAP on one GPU
 * — different streams, or threads using different streams — race on it. Keep them on one stream, or order them
 * with events. */
#define BB_KMEANS_STATIC_MAX_N 1024
int bb_kmeans_levels_static(int device, void* cuda_stream, const double* lambda_dev, int n, int n_levels,
                            int log_domain, double* intervals_dev, int ld_int, int* status_dev);

/* ---- NUFFT Synthesis (Section 2.5 Eq. 17-21, Section 3.4 Eq. 32-36, Algorithm 3), SURVEY 8(f) row 3 -----
 * Per collect: V'_l = B diag(D[l,:]) B^H (Eq. 17 with the level selection of Eq. 21; Alg. 3 l.8) on the n_ant^2
 * baselines b_pq = (x_p - x_q) / wavelength, then I_l(r_j) += sum_pq V'_l,pq exp(-2 pi i <b_pq, r_j>) (Eq. 18-19,
 * DESIGN.md reading Q18) by a type-3 (nonuniform to nonuniform) 3-D NUFFT: centring and pre-phase, spreading with
 * the "exponential of semicircle" kernel onto a fine grid (Eq. 33), a type-2 transform (deconvolve, zero-pad, FFT,
 * interpolate: Eq. 34) and the diagonal correction by the kernel's Fourier transform (Eq. 35). The baselines and the
 * pixels are partitioned into regular n_part_in x n_part_in x 1 and n_part_out x n_part_out x 1 cells along their two
 * widest axes (Section 3.4.1, Eq. 36); every non-empty (input cell, output cell) pair is one transform.
 * eps: requested relative tolerance (1e-2 .. 1e-7; sets the kernel width). pix as for bb_synth_create (host or
 * device). B, D, xyz: host or device, as bb_synth_collect_eig; the call snapshots them, forms V'_l on the device and
 * STAGES the collect (it synchronises the context stream). The transforms run in bb_nufft_get — ONE set over the
 * baselines of all staged collects, the paper's use of the NUFFT over all time steps — or earlier when 2^24 staged
 * baselines are reached or n_ant changes. BB_EUNSUPPORTED (from the call that runs the transforms): some pair's fine
 * grids (all levels, complex64) plus the FFT work area would exceed 32 GB: raise the partition counts. Every pair is
 * checked, and every buffer and FFT plan is set up, BEFORE the first transform runs, so BB_EUNSUPPORTED and BB_EALLOC
 * leave the level images exactly as they were (the staged collects are dropped; the handle stays usable). BB_ECUDA from
 * that call is a launch or execution failure part-way through: the images are then undefined, destroy the handle.
 * Same images as bb_synth_collect_eig up to eps; O(n_ant^2 L w^3 + grid log grid + n_pix L w^3) per pair. */
typedef struct bb_nufft bb_nufft;
int bb_nufft_create(bb_ctx* ctx, int64_t n_pix, const double* pix, int64_t ld_pix, int n_levels, double eps,
                    int n_part_in, int n_part_out, bb_nufft** out);
int bb_nufft_destroy(bb_nufft* h);
int bb_nufft_collect_eig(bb_nufft* h, int n_ant, int n_eig, double wavelength, const bb_c32* B, int ldb,
                         const float* D, int ldd, const double* xyz, int ldxyz);
/* Algorithm 3 from its own inputs: Gram matrix, generalized eigendecomposition, N_eig largest pairs
 * (l.2-4), interval selection and filters (l.5-7), V per level and the NUFFT (l.8-9). Arguments as bb_synth_collect_ex
 * (sinc Gram); the handle's n_levels must equal n_intervals * n_filters, image index = filter * n_intervals + interval.
 * n_ant <= 4096, n_beam <= BB_MAX_BEAMS. Synchronous up to the staging: BB_ENOTPOSDEF / BB_ENOCONV are returned by this
 * call and nothing is staged. Same images as bb_synth_collect_ex up to eps. */
int bb_nufft_collect(bb_nufft* h, int n_ant, int n_beam, int n_eig, double wavelength, const bb_c32* W, int ldw,
                     const bb_c32* S, int lds, const double* xyz, int ldxyz, const double* intervals, int ld_int,
                     int n_filters, const int* filters);
int bb_nufft_get(bb_nufft* h, int level, float* out);   /* n_pix floats, host or device; synchronises */
/* number of transforms run and the largest fine grid (points) so far: what Section 3.4.1 / Figure 1c is about */
int bb_nufft_stats(bb_nufft* h, int64_t* n_transforms, int64_t* max_grid_points);

/* Host-only planning query (no device needed; pix and xyz must be HOST pointers): the transforms ONE collect of this
 * array would need under an (n_part_in, n_part_out) partitioning — their number, the largest and the summed fine-grid
 * sizes (points, per level) and the fraction of non-empty input cells: the quantities of Section 3.4.1 / Figure 1c-d. */
int bb_nufft_plan(int64_t n_pix, const double* pix, int64_t ld_pix, int n_ant, const double* xyz, int ldxyz, double wavelength,
                  double eps, int n_part_in, int n_part_out, int64_t* n_transforms, int64_t* max_grid_points,
                  double* sum_grid_points, double* nonempty_input_cells);

/* ---- DIAGNOSTICS: launch-shape query (host only, no device needed). Like bb_synth_launches it follows no passage of
 * the paper: both exist so that tests and bench.py can check and count what the library launches. -------------------
 * Number of collect ranges a synthesizer launch over n_collects queued collects is split into on a GPU with sm_count
 * SMs: 1 = one CTA per pixel tile handles all collects; > 1 for small images whose tile count would leave most of a
 * wave of SMs empty (the ranges' level sums are added in a fixed order). Returns 0 on invalid arguments. */
int bb_plan_collect_split(int variant, int64_t n_pix, int n_ant, int n_eig, int n_levels, int n_collects, int sm_count);

const char* bb_status_string(int status);
const char* bb_version(void);

#ifdef __cplusplus
}
#endif
#endif /* BLUEBILD_B200_H */
