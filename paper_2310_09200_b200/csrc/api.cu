// C ABI of libbluebild_b200.so (include/bluebild.h): argument validation, host/device pointer handling, the
// queue of prepared collects and the stream choreography of Algorithm 1.
// All arithmetic of the method runs in the CUDA kernels of kernels_fp32.cu / kernels_tc.cu / glue.cu /
// eig_subspace.cu / pixels.cu / estimate.cu; nothing here computes on the host and there is no CPU fallback.
//
// Streams ("iteratively collect input data at each time step"):
//   user stream   the context stream: only ordering. Device inputs are read after an event recorded on it at call
//                 time, and it waits for the kernel / copy that consumes them, so the caller may reuse them in
//                 stream order; every synthesizer launch is followed by an event the user stream waits on, so
//                 work the caller enqueues after bb_synth_flush / get sees the updated images.
//   glue stream   (per context, high priority) staging copies of S / W / xyz / intervals, the batched Gram,
//                 Cholesky, eigensolve, selection and level weights of up to kGlueGroup collects at a time.
//   synth stream  (per context) per-collect prep kernels and the fused synthesizer launches.
// The glue of group n+1 therefore runs while the synthesizer of group n is busy; the only cross-stream edges are
// "prep of a collect waits for its glue" and "a slot's staging waits for the prep of its previous occupant".
// No call on this path synchronises the host with the device except get / timings / status / reset / destroy and
// a re-allocation when shapes grow: solver verdicts stay on the device (glue.cu) and surface as sticky flags.
#include "internal.h"

#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>

// ------------------------------------------------------------------------------ error notes
static thread_local char g_last_cuda[256];
void bb_note_cuda_error(cudaError_t err, const char* what, const char* file, int line) {
  snprintf(g_last_cuda, sizeof g_last_cuda, "%s at %s:%d: %s", what, file, line, cudaGetErrorString(err));
  if (getenv("BB_VERBOSE")) fprintf(stderr, "[bluebild] CUDA error: %s\n", g_last_cuda);
  cudaGetLastError();
}

extern "C" const char* bb_status_string(int status) {
  switch (status) {
    case BB_OK: return "ok";
    case BB_EINVAL: return "invalid argument";
    case BB_EALLOC: return "allocation failed";
    case BB_ECUDA: return g_last_cuda[0] ? g_last_cuda : "CUDA error";
    case BB_ENOTPOSDEF: return "Gram matrix not positive definite";
    case BB_ENOCONV: return "eigensolver did not converge";
    case BB_ESTATE: return "invalid handle state";
    case BB_EUNSUPPORTED: return "unsupported variant, size or coordinate range";
    default: return "unknown status";
  }
}

extern "C" const char* bb_version(void) { return "bluebild-b200 0.2 (sm_100a)"; }

// ------------------------------------------------------------------------------ handles
struct bb_ctx {
  int device = 0;
  cudaStream_t stream = nullptr;        // the caller's stream (ordering only)
  cudaStream_t glue_stream = nullptr;
  cudaStream_t synth_stream = nullptr;
  int sm_count = 0;
  GlueWork* glue = nullptr;
  int live_handles = 0;
};

constexpr int kGlueGroup = 128;         // collects per batched glue call = the deepest queue (scratch: ~30 MB per collect at n_beam 512)

enum { T_GRAM = 0, T_EIG = 1, T_PREP = 2, T_SYNTH = 3, T_KINDS = 4 };
struct Span { cudaEvent_t a, b; int kind; };

// layout of a full collect's inputs inside a staging slot (fixed per queue shape, so that the batched glue can
// address the collects of a group with one stride)
struct FullLayout { size_t off_w, off_s, off_x, off_iv, off_wl, bytes; };

struct PendingGlue { int n_filters; FilterList fl; };

struct bb_synth {
  bb_ctx* ctx = nullptr;
  int64_t n_pix = 0, pix_stride = 0;
  int n_levels = 0, variant = 0;
  double* rprime = nullptr;
  double rc[3] = {0, 0, 0};
  double rmax = 0;
  float* img = nullptr;
  float* split_scratch = nullptr;              // partial level sums of a collect-range split launch (small images)
  size_t split_cap = 0;                        // floats
  int* status_dev = nullptr;            // sticky BB_FLAG_* word
  int* status_pin = nullptr;
  cudaEvent_t ev_in = nullptr, ev_out = nullptr, ev_glue = nullptr;
  // queue of prepared collects (all with the same n_ant, n_eig)
  int q_cap = 0, q_len = 0, q_n_ant = 0, q_n_eig = 0, q_n_beam = 0;
  bool q_has_w = false;
  Fp32Plan fplan{};
  TcPlan tplan{};
  unsigned char* packed = nullptr; size_t packed_stride = 0;
  float* weights = nullptr; size_t weight_stride = 0;
  // staging of caller inputs, one slot per queue entry
  unsigned char* pin = nullptr; unsigned char* dev_in = nullptr; size_t in_slot_bytes = 0;
  FullLayout lay{};
  std::vector<cudaEvent_t> slot_ev, prep_done; std::vector<char> slot_busy, slot_prepped;
  // collects whose inputs are staged (slots q_len .. q_len + g_pending - 1) and whose glue has not been enqueued yet
  int g_pending = 0, g_gram_mode = 0;
  const bb_uvgrid* weighting = nullptr;   // uniform weighting (Section 3.5) of the collects staged from now on; NULL = natural
  std::vector<PendingGlue> pend;
  // glue outputs per slot
  bb_c32* glue_B = nullptr; double* glue_lambda = nullptr; float* glue_D = nullptr; int* glue_info = nullptr;
  // timing
  std::vector<Span> spans; std::vector<cudaEvent_t> free_ev;
  double acc_ms[T_KINDS] = {0, 0, 0, 0};
  int64_t launches = 0;
};

cudaStream_t bb_ctx_glue_stream(bb_ctx* ctx) { return ctx->glue_stream; }
cudaStream_t bb_ctx_user_stream(bb_ctx* ctx) { return ctx->stream; }
int bb_ctx_device(bb_ctx* ctx) { return ctx->device; }
void bb_ctx_ref(bb_ctx* ctx, int delta) { ctx->live_handles += delta; }   // handles of other translation units (bb_nufft)

static bool is_device_ptr(const void* p) {
  cudaPointerAttributes at;
  if (cudaPointerGetAttributes(&at, p) != cudaSuccess) { cudaGetLastError(); return false; }
  return at.type == cudaMemoryTypeDevice || at.type == cudaMemoryTypeManaged;
}

static size_t up16(size_t x) { return (x + 15) / 16 * 16; }

static cudaEvent_t get_event(bb_synth* s) {
  if (!s->free_ev.empty()) { cudaEvent_t e = s->free_ev.back(); s->free_ev.pop_back(); return e; }
  cudaEvent_t e = nullptr;
  cudaEventCreate(&e);
  return e;
}

static void fold_spans(bb_synth* s) {  // caller guarantees the streams are synchronised
  for (const Span& sp : s->spans) {
    float ms = 0.f;
    if (cudaEventSynchronize(sp.b) == cudaSuccess && cudaEventElapsedTime(&ms, sp.a, sp.b) == cudaSuccess)
      s->acc_ms[sp.kind] += ms;
    else
      cudaGetLastError();
    s->free_ev.push_back(sp.a);
    s->free_ev.push_back(sp.b);
  }
  s->spans.clear();
}

struct SpanGuard {  // records an event pair around a region of one stream
  bb_synth* s; Span sp; cudaStream_t st;
  SpanGuard(bb_synth* s_, int kind, cudaStream_t st_) : s(s_), st(st_) {
    sp.a = get_event(s); sp.b = get_event(s); sp.kind = kind;
    cudaEventRecord(sp.a, st);
  }
  ~SpanGuard() { cudaEventRecord(sp.b, st); s->spans.push_back(sp); }
};

static int sync_all(bb_synth* s) {
  BB_CUDA(cudaStreamSynchronize(s->ctx->glue_stream));
  BB_CUDA(cudaStreamSynchronize(s->ctx->synth_stream));
  BB_CUDA(cudaStreamSynchronize(s->ctx->stream));
  return BB_OK;
}

// ------------------------------------------------------------------------------ context
extern "C" int bb_ctx_create(int device, void* cuda_stream, bb_ctx** out) {
  if (!out) return BB_EINVAL;
  *out = nullptr;
  int n_dev = 0;
  if (cudaGetDeviceCount(&n_dev) != cudaSuccess || n_dev <= 0) {
    bb_note_cuda_error(cudaErrorNoDevice, "bb_ctx_create: no CUDA device (there is no CPU fallback)", __FILE__, __LINE__);
    return BB_ECUDA;
  }
  if (device < 0 || device >= n_dev) return BB_EINVAL;
  BB_CUDA(cudaSetDevice(device));
  cudaDeviceProp prop;
  BB_CUDA(cudaGetDeviceProperties(&prop, device));
  if (prop.major != 10) {
    bb_note_cuda_error(cudaErrorInvalidDevice, "bb_ctx_create: this library is built for sm_100a only", __FILE__, __LINE__);
    return BB_ECUDA;
  }
  bb_ctx* c = new (std::nothrow) bb_ctx;
  if (!c) return BB_EALLOC;
  c->device = device;
  c->stream = (cudaStream_t)cuda_stream;
  c->sm_count = prop.multiProcessorCount;
  int prio_lo = 0, prio_hi = 0;
  cudaDeviceGetStreamPriorityRange(&prio_lo, &prio_hi);
  if (cudaStreamCreateWithPriority(&c->glue_stream, cudaStreamNonBlocking, prio_hi) != cudaSuccess ||
      cudaStreamCreateWithPriority(&c->synth_stream, cudaStreamNonBlocking, prio_lo) != cudaSuccess) {
    bb_note_cuda_error(cudaGetLastError(), "bb_ctx_create: stream creation", __FILE__, __LINE__);
    if (c->glue_stream) cudaStreamDestroy(c->glue_stream);
    delete c;
    return BB_ECUDA;
  }
  *out = c;
  return BB_OK;
}

extern "C" int bb_ctx_destroy(bb_ctx* ctx) {
  if (!ctx) return BB_EINVAL;
  if (ctx->live_handles > 0) return BB_ESTATE;     // imaging handles still refer to this context
  cudaSetDevice(ctx->device);
  cudaStreamSynchronize(ctx->glue_stream);
  cudaStreamSynchronize(ctx->synth_stream);
  if (ctx->glue) bb_glue_destroy(ctx->glue);
  cudaStreamDestroy(ctx->glue_stream);
  cudaStreamDestroy(ctx->synth_stream);
  cudaGetLastError();
  delete ctx;
  return BB_OK;
}

// ------------------------------------------------------------------------------ imaging handle
static void free_queue(bb_synth* s) {
  cudaFree(s->packed); s->packed = nullptr;
  cudaFree(s->weights); s->weights = nullptr;
  cudaFree(s->dev_in); s->dev_in = nullptr;
  cudaFree(s->glue_B); s->glue_B = nullptr;
  cudaFree(s->glue_lambda); s->glue_lambda = nullptr;
  cudaFree(s->glue_D); s->glue_D = nullptr;
  cudaFree(s->glue_info); s->glue_info = nullptr;
  if (s->pin) { cudaFreeHost(s->pin); s->pin = nullptr; }
  for (cudaEvent_t e : s->slot_ev) cudaEventDestroy(e);
  for (cudaEvent_t e : s->prep_done) cudaEventDestroy(e);
  s->slot_ev.clear(); s->prep_done.clear(); s->slot_busy.clear(); s->slot_prepped.clear(); s->pend.clear();
  s->q_cap = s->q_len = s->q_n_ant = s->q_n_eig = s->q_n_beam = s->g_pending = 0;
  s->in_slot_bytes = 0;
}

extern "C" int bb_synth_destroy(bb_synth* s) {
  if (!s) return BB_EINVAL;
  cudaSetDevice(s->ctx->device);
  sync_all(s);
  fold_spans(s);
  for (cudaEvent_t e : s->free_ev) cudaEventDestroy(e);
  free_queue(s);
  if (s->ev_in) cudaEventDestroy(s->ev_in);
  if (s->ev_out) cudaEventDestroy(s->ev_out);
  if (s->ev_glue) cudaEventDestroy(s->ev_glue);
  cudaFree(s->rprime);
  cudaFree(s->img);
  cudaFree(s->split_scratch);
  cudaFree(s->status_dev);
  if (s->status_pin) cudaFreeHost(s->status_pin);
  cudaGetLastError();
  s->ctx->live_handles -= 1;
  delete s;
  return BB_OK;
}

extern "C" int bb_synth_create(bb_ctx* ctx, int64_t n_pix, const double* pix, int64_t ld_pix, int n_levels,
                               int variant, bb_synth** out) {
  if (!out) return BB_EINVAL;
  *out = nullptr;
  if (!ctx || n_pix < 0 || (n_pix > 0 && !pix) || ld_pix < n_pix || n_levels < 1 || n_levels > BB_MAX_LEVELS)
    return BB_EINVAL;
  if (variant != BB_VARIANT_FP32 && variant != BB_VARIANT_TF32X3 && variant != BB_VARIANT_FP16X3 && variant != BB_VARIANT_FP16_FP8) return BB_EUNSUPPORTED;
  BB_CUDA(cudaSetDevice(ctx->device));
  bb_synth* s = new (std::nothrow) bb_synth;
  if (!s) return BB_EALLOC;
  s->ctx = ctx; s->n_pix = n_pix; s->n_levels = n_levels; s->variant = variant;
  ctx->live_handles += 1;
  s->pix_stride = (n_pix + 511) / 512 * 512 + 512;   // whole tiles may be read past n_pix
  cudaStream_t st = ctx->synth_stream;
  int rc = BB_OK;
  double* tmp = nullptr;
  do {
    if (cudaMalloc(&s->rprime, 3 * (size_t)s->pix_stride * sizeof(double)) != cudaSuccess ||
        cudaMalloc(&s->img, (size_t)n_levels * s->pix_stride * sizeof(float)) != cudaSuccess ||
        cudaMalloc(&s->status_dev, sizeof(int)) != cudaSuccess ||
        cudaMallocHost(&s->status_pin, sizeof(int)) != cudaSuccess) { rc = BB_EALLOC; break; }
    if (cudaEventCreateWithFlags(&s->ev_in, cudaEventDisableTiming) != cudaSuccess ||
        cudaEventCreateWithFlags(&s->ev_out, cudaEventDisableTiming) != cudaSuccess ||
        cudaEventCreateWithFlags(&s->ev_glue, cudaEventDisableTiming) != cudaSuccess) { rc = BB_ECUDA; break; }
    if (cudaMemsetAsync(s->img, 0, (size_t)n_levels * s->pix_stride * sizeof(float), st) != cudaSuccess ||
        cudaMemsetAsync(s->status_dev, 0, sizeof(int), st) != cudaSuccess) { rc = BB_ECUDA; break; }
    const double* pix_dev = pix;
    int64_t ld = ld_pix;
    if (n_pix > 0 && !is_device_ptr(pix)) {
      if (cudaMalloc(&tmp, 3 * (size_t)n_pix * sizeof(double)) != cudaSuccess) { rc = BB_EALLOC; break; }
      if (cudaMemcpy2DAsync(tmp, n_pix * sizeof(double), pix, ld_pix * sizeof(double), n_pix * sizeof(double), 3,
                            cudaMemcpyHostToDevice, st) != cudaSuccess) { rc = BB_ECUDA; break; }
      pix_dev = tmp; ld = n_pix;
    } else if (n_pix > 0) {                          // device pixels: ordered after the caller's work on the context stream
      if (cudaEventRecord(s->ev_in, ctx->stream) != cudaSuccess || cudaStreamWaitEvent(st, s->ev_in, 0) != cudaSuccess) { rc = BB_ECUDA; break; }
    }
    if (n_pix > 0) rc = bb_pixels_prepare(pix_dev, n_pix, ld, s->rprime, s->pix_stride, s->rc, &s->rmax, st);   // synchronises st
    else if (cudaMemsetAsync(s->rprime, 0, 3 * (size_t)s->pix_stride * sizeof(double), st) != cudaSuccess) rc = BB_ECUDA;
  } while (0);
  cudaFree(tmp);
  if (rc != BB_OK) { cudaGetLastError(); bb_synth_destroy(s); return rc; }
  *out = s;
  return BB_OK;
}

extern "C" int bb_synth_reset(bb_synth* s) {
  if (!s) return BB_EINVAL;
  BB_CUDA(cudaSetDevice(s->ctx->device));
  s->q_len = 0; s->g_pending = 0; s->pend.clear();
  int rc = sync_all(s);
  if (rc != BB_OK) return rc;
  BB_CUDA(cudaMemsetAsync(s->img, 0, (size_t)s->n_levels * s->pix_stride * sizeof(float), s->ctx->synth_stream));
  BB_CUDA(cudaMemsetAsync(s->status_dev, 0, sizeof(int), s->ctx->synth_stream));
  BB_CUDA(cudaStreamSynchronize(s->ctx->synth_stream));
  fold_spans(s);
  for (int k = 0; k < T_KINDS; ++k) s->acc_ms[k] = 0;
  s->launches = 0;
  return BB_OK;
}

static int run_pending_glue(bb_synth* s);

// Launch the synthesizer over the prepared collects (synth stream); the user stream waits for it.
static int launch_queue(bb_synth* s) {
  if (s->q_len == 0) return BB_OK;
  SynthArgs a{};
  a.rprime = s->rprime; a.n_pix = s->n_pix; a.pix_stride = s->pix_stride;
  a.packed = s->packed; a.packed_stride = s->packed_stride;
  a.weights = s->weights; a.weight_stride = s->weight_stride;
  a.n_collects = s->q_len; a.n_levels = s->n_levels;
  a.img = s->img; a.img_stride = s->pix_stride;
  cudaStream_t st = s->ctx->synth_stream;
  {
    a.n_split = s->variant == BB_VARIANT_FP32 ? bb_fp32_split(s->fplan, s->n_pix, s->q_len, s->ctx->sm_count)
                                             : bb_tc_split(s->n_pix, s->q_len, s->ctx->sm_count);
    if (a.n_split > 1) {
      const size_t need = (size_t)a.n_split * s->n_levels * s->pix_stride;
      if (need > s->split_cap) {                 // grows only; earlier launches that read it are complete once the stream is
        BB_CUDA(cudaStreamSynchronize(st));
        cudaFree(s->split_scratch);
        s->split_scratch = nullptr; s->split_cap = 0;
        if (cudaMalloc(&s->split_scratch, need * sizeof(float)) != cudaSuccess) { cudaGetLastError(); return BB_EALLOC; }
        s->split_cap = need;
      }
      a.scratch = s->split_scratch;
    }
  }
  int launches = 0, rc;
  {
    SpanGuard g(s, T_SYNTH, st);
    rc = (s->variant == BB_VARIANT_FP32) ? bb_launch_synth_fp32(s->fplan, a, s->ctx->sm_count, st, &launches)
                                         : bb_launch_synth_tc(s->tplan, a, s->ctx->sm_count, st, &launches);
  }
  s->launches += launches;
  s->q_len = 0;
  if (rc != BB_OK) return rc;
  BB_CUDA(cudaEventRecord(s->ev_out, st));
  BB_CUDA(cudaStreamWaitEvent(s->ctx->stream, s->ev_out, 0));
  return BB_OK;
}

extern "C" int bb_plan_collect_split(int variant, int64_t n_pix, int n_ant, int n_eig, int n_levels, int n_collects, int sm_count) {
  if (n_pix < 1 || n_ant < 1 || n_eig < 1 || n_levels < 1 || n_collects < 1 || sm_count < 1) return 0;
  if (variant == BB_VARIANT_FP32) return bb_fp32_split(bb_fp32_plan(n_ant, n_eig, n_levels), n_pix, n_collects, sm_count);
  if (variant == BB_VARIANT_TF32X3 || variant == BB_VARIANT_FP16X3 || variant == BB_VARIANT_FP16_FP8) return bb_tc_split(n_pix, n_collects, sm_count);
  return 0;
}

extern "C" int bb_synth_flush(bb_synth* s) {
  if (!s) return BB_EINVAL;
  BB_CUDA(cudaSetDevice(s->ctx->device));
  int rc = run_pending_glue(s);
  if (rc != BB_OK) return rc;
  return launch_queue(s);
}

static FullLayout full_layout(int n_ant, int n_beam, int n_intervals, bool has_w) {
  FullLayout l{};
  size_t off = 0;
  l.off_w = off; off += has_w ? up16((size_t)n_ant * n_beam * 8) : 0;
  l.off_s = off; off += up16((size_t)n_beam * n_beam * 8);
  l.off_x = off; off += up16((size_t)n_ant * 24);
  l.off_iv = off; off += up16((size_t)n_intervals * 16);
  l.off_wl = off; off += 16;
  l.bytes = off;
  return l;
}

// (Re)size the queue for collects of shape (n_ant, n_eig) whose staged inputs need `need` bytes per slot; flushes
// pending work when the shape changes or the slots are too small (the slot size must follow n_beam).
static int ensure_queue(bb_synth* s, int n_ant, int n_eig, size_t need) {
  if (s->q_cap > 0 && s->q_n_ant == n_ant && s->q_n_eig == n_eig && need <= s->in_slot_bytes) return BB_OK;
  int rc = bb_synth_flush(s);
  if (rc != BB_OK) return rc;
  if ((rc = sync_all(s)) != BB_OK) return rc;
  fold_spans(s);
  free_queue(s);
  const int L = s->n_levels;
  if (s->variant == BB_VARIANT_FP32) {
    s->fplan = bb_fp32_plan(n_ant, n_eig, L);
    s->packed_stride = s->fplan.collect_bytes; s->weight_stride = s->fplan.weight_floats;
  } else {
    s->tplan = bb_tc_plan(n_ant, n_eig, L, s->variant == BB_VARIANT_FP16X3 ? BB_TC_FP16 : s->variant == BB_VARIANT_FP16_FP8 ? BB_TC_F16F8 : BB_TC_TF32);
    if (s->tplan.n_chunks == 0) return BB_EUNSUPPORTED;
    s->packed_stride = s->tplan.collect_bytes; s->weight_stride = s->tplan.weight_floats;
  }
  s->in_slot_bytes = (need + 255) / 256 * 256;
  // queue depth: enough collects per launch to amortise the image read-modify-write, bounded memory
  size_t per = s->packed_stride + s->weight_stride * 4 + 2 * s->in_slot_bytes + (size_t)n_ant * n_eig * 8;
  int cap = kGlueGroup;
  while (cap > 4 && per * cap > ((size_t)2 << 30)) cap /= 2;
  if (cudaMalloc(&s->packed, s->packed_stride * cap) != cudaSuccess ||
      cudaMalloc(&s->weights, s->weight_stride * 4 * cap) != cudaSuccess ||
      cudaMalloc(&s->dev_in, s->in_slot_bytes * cap) != cudaSuccess ||
      cudaMalloc(&s->glue_B, (size_t)n_ant * n_eig * 8 * cap) != cudaSuccess ||
      cudaMalloc(&s->glue_lambda, (size_t)n_eig * 8 * cap) != cudaSuccess ||
      cudaMalloc(&s->glue_D, (size_t)L * n_eig * 4 * cap) != cudaSuccess ||
      cudaMalloc(&s->glue_info, (size_t)2 * cap * sizeof(int)) != cudaSuccess ||
      cudaMallocHost(&s->pin, s->in_slot_bytes * cap) != cudaSuccess) {
    cudaGetLastError(); free_queue(s); return BB_EALLOC;
  }
  s->slot_ev.resize(cap); s->prep_done.resize(cap); s->slot_busy.assign(cap, 0); s->slot_prepped.assign(cap, 0);
  for (int i = 0; i < cap; ++i) {
    cudaEventCreateWithFlags(&s->slot_ev[i], cudaEventDisableTiming);
    cudaEventCreateWithFlags(&s->prep_done[i], cudaEventDisableTiming);
  }
  s->q_cap = cap; s->q_len = 0; s->q_n_ant = n_ant; s->q_n_eig = n_eig;
  return BB_OK;
}

// Copy a column-major host matrix (rows x cols, ld) compactly into dst.
static void pack_host(void* dst, const void* src, size_t elem, int rows, int cols, int ld) {
  if (ld == rows) { memcpy(dst, src, (size_t)rows * cols * elem); return; }   // already compact: one copy
  for (int c = 0; c < cols; ++c)
    memcpy((char*)dst + (size_t)c * rows * elem, (const char*)src + (size_t)c * ld * elem, (size_t)rows * elem);
}

// The pinned half of a slot may be rewritten once its previous host-to-device copy has completed.
static void wait_slot_copy(bb_synth* s, int slot) {
  if (s->slot_busy[slot]) { cudaEventSynchronize(s->slot_ev[slot]); s->slot_busy[slot] = 0; }
}

// Prep kernel of one collect on the synth stream (B, D, xyz: device pointers) -> slot q_len of the queue.
static int enqueue_prepared(bb_synth* s, int n_ant, int n_eig, double wavelength, const bb_c32* B, int ldb,
                            const float* D, int ldd, const double* xyz, int ldxyz) {
  PrepArgs a{};
  a.B = B; a.ldb = ldb; a.D = D; a.ldd = ldd; a.xyz = xyz; a.ldxyz = ldxyz;
  a.n_ant = n_ant; a.n_eig = n_eig; a.n_levels = s->n_levels; a.wavelength = wavelength;
  a.rc[0] = s->rc[0]; a.rc[1] = s->rc[1]; a.rc[2] = s->rc[2];
  a.rmax = s->rmax;
  a.status = s->status_dev;
  const int slot = s->q_len;
  a.packed = s->packed + (size_t)slot * s->packed_stride;
  a.weights = s->weights + (size_t)slot * s->weight_stride;
  cudaStream_t st = s->ctx->synth_stream;
  int rc;
  {
    SpanGuard g(s, T_PREP, st);
    rc = (s->variant == BB_VARIANT_FP32) ? bb_launch_prep_fp32(s->fplan, a, st) : bb_launch_prep_tc(s->tplan, a, st);
  }
  if (rc != BB_OK) return rc;
  BB_CUDA(cudaEventRecord(s->prep_done[slot], st));
  s->slot_prepped[slot] = 1;
  s->launches += 1;
  s->q_len += 1;
  if (s->spans.size() > 8192) { sync_all(s); fold_spans(s); }
  return BB_OK;
}

// Largest antenna count a variant takes (include/bluebild.h "Antenna-count limit"): the tensor variants' fp32
// accumulator loses a fraction of an ulp, always towards zero, with every tcgen05.mma that adds to it, so their images
// come out too small by a factor that grows with n_ant / 16 x {12, 6, 4} instructions (measured: profiles/r03_n_ant_bias.md).
static int max_antennas(int variant) {
  switch (variant) {
    case BB_VARIANT_TF32X3: return BB_MAX_ANT_TF32X3;
    case BB_VARIANT_FP16X3: return BB_MAX_ANT_FP16X3;
    case BB_VARIANT_FP16_FP8: return BB_MAX_ANT_FP16_FP8;
    default: return 1 << 20;
  }
}

extern "C" int bb_synth_collect_eig(bb_synth* s, int n_ant, int n_eig, double wavelength, const bb_c32* B, int ldb,
                                    const float* D, int ldd, const double* xyz, int ldxyz) {
  if (!s || !B || !D || !xyz || n_ant < 1 || n_eig < 1 || !(wavelength > 0.0) || ldb < n_ant ||
      ldd < s->n_levels || ldxyz < n_ant || n_eig > 4096 || n_ant > (1 << 20))
    return BB_EINVAL;
  if (n_ant > max_antennas(s->variant)) return BB_EUNSUPPORTED;    // nothing queued, images unchanged: use BB_VARIANT_FP32
  BB_CUDA(cudaSetDevice(s->ctx->device));
  const int L = s->n_levels;
  const size_t need = up16((size_t)n_ant * n_eig * 8) + up16((size_t)L * n_eig * 4) + up16((size_t)n_ant * 24);
  int rc = ensure_queue(s, n_ant, n_eig, need);
  if (rc == BB_OK) rc = run_pending_glue(s);                // keep the accumulation order = the call order
  if (rc == BB_OK && s->q_len == s->q_cap) rc = launch_queue(s);
  if (rc != BB_OK) return rc;
  cudaStream_t st = s->ctx->synth_stream;
  const int slot = s->q_len;
  const bool dB = is_device_ptr(B), dD = is_device_ptr(D), dX = is_device_ptr(xyz);
  if (dB || dD || dX) {                                     // device inputs: ordered after the caller's work on the context stream
    BB_CUDA(cudaEventRecord(s->ev_in, s->ctx->stream));
    BB_CUDA(cudaStreamWaitEvent(st, s->ev_in, 0));
  }
  const bb_c32* Bd = B; const float* Dd = D; const double* Xd = xyz;
  int ldb2 = ldb, ldd2 = ldd, ldx2 = ldxyz;
  if (!dB || !dD || !dX) {                                  // host inputs: snapshot into the pinned slot, one copy
    wait_slot_copy(s, slot);
    unsigned char* hp = s->pin + (size_t)slot * s->in_slot_bytes;
    unsigned char* dp = s->dev_in + (size_t)slot * s->in_slot_bytes;
    size_t off = 0;
    if (!dB) { pack_host(hp + off, B, 8, n_ant, n_eig, ldb); Bd = (const bb_c32*)(dp + off); ldb2 = n_ant; off += up16((size_t)n_ant * n_eig * 8); }
    if (!dD) { pack_host(hp + off, D, 4, L, n_eig, ldd); Dd = (const float*)(dp + off); ldd2 = L; off += up16((size_t)L * n_eig * 4); }
    if (!dX) { pack_host(hp + off, xyz, 8, n_ant, 3, ldxyz); Xd = (const double*)(dp + off); ldx2 = n_ant; off += up16((size_t)n_ant * 24); }
    BB_CUDA(cudaMemcpyAsync(dp, hp, off, cudaMemcpyHostToDevice, st));
    BB_CUDA(cudaEventRecord(s->slot_ev[slot], st));
    s->slot_busy[slot] = 1;
  }
  if ((rc = enqueue_prepared(s, n_ant, n_eig, wavelength, Bd, ldb2, Dd, ldd2, Xd, ldx2)) != BB_OK) return rc;
  if (dB || dD || dX) BB_CUDA(cudaStreamWaitEvent(s->ctx->stream, s->prep_done[slot], 0));   // the caller may reuse its device buffers in stream order
  if (s->q_len == s->q_cap) return launch_queue(s);
  return BB_OK;
}

// ------------------------------------------------------------------------------ Algorithm 1 (glue + hot path)
// Stage one full collect's inputs into slot q_len + g_pending: host -> pinned -> device, or device -> device,
// both on the glue stream. The glue itself is enqueued later, for the whole group at once.
static int stage_full(bb_synth* s, int n_ant, int n_beam, int n_eig, double wavelength, const bb_c32* W, int ldw,
                      const bb_c32* S, int lds, const double* xyz, int ldxyz, const double* intervals, int ld_int,
                      int n_intervals, const FilterList& fl, int gram_mode) {
  const FullLayout need = full_layout(n_ant, n_beam, n_intervals, W != nullptr);
  // a group shares one layout, one Gram mode and one "has W"; anything else closes the group first
  if (s->g_pending > 0 && (s->q_n_ant != n_ant || s->q_n_eig != n_eig || s->q_n_beam != n_beam || s->q_has_w != (W != nullptr) ||
                           s->g_gram_mode != gram_mode || need.bytes != s->lay.bytes)) {
    int rc = run_pending_glue(s);
    if (rc != BB_OK) return rc;
  }
  int rc = ensure_queue(s, n_ant, n_eig, need.bytes);
  if (rc != BB_OK) return rc;
  if (!s->ctx->glue && (rc = bb_glue_create(&s->ctx->glue)) != BB_OK) return rc;
  s->lay = need; s->q_n_beam = n_beam; s->q_has_w = W != nullptr; s->g_gram_mode = gram_mode;
  cudaStream_t gs = s->ctx->glue_stream;
  const int slot = s->q_len + s->g_pending;
  // the slot's previous occupant must have been consumed by its prep kernel before the slot is overwritten
  if (s->slot_prepped[slot]) { BB_CUDA(cudaStreamWaitEvent(gs, s->prep_done[slot], 0)); s->slot_prepped[slot] = 0; }
  wait_slot_copy(s, slot);
  unsigned char* hp = s->pin + (size_t)slot * s->in_slot_bytes;
  unsigned char* dp = s->dev_in + (size_t)slot * s->in_slot_bytes;
  bool any_dev = false;
  struct Item { const void* p; size_t off, elem; int rows, cols, ld; };
  const Item items[4] = {{W, need.off_w, 8, n_ant, n_beam, ldw}, {S, need.off_s, 8, n_beam, n_beam, lds},
                         {xyz, need.off_x, 8, n_ant, 3, ldxyz}, {intervals, need.off_iv, 8, n_intervals, 2, ld_int}};
  bool dev[4];
  for (int i = 0; i < 4; ++i) { dev[i] = items[i].p && is_device_ptr(items[i].p); any_dev = any_dev || dev[i]; }
  // host parts: one contiguous copy of the slot (the device parts are overwritten afterwards)
  for (int i = 0; i < 4; ++i)
    if (items[i].p && !dev[i]) pack_host(hp + items[i].off, items[i].p, items[i].elem, items[i].rows, items[i].cols, items[i].ld);
  memcpy(hp + need.off_wl, &wavelength, sizeof(double));
  BB_CUDA(cudaMemcpyAsync(dp, hp, need.bytes, cudaMemcpyHostToDevice, gs));
  BB_CUDA(cudaEventRecord(s->slot_ev[slot], gs));
  s->slot_busy[slot] = 1;
  if (any_dev) {
    BB_CUDA(cudaEventRecord(s->ev_in, s->ctx->stream));
    BB_CUDA(cudaStreamWaitEvent(gs, s->ev_in, 0));
    for (int i = 0; i < 4; ++i)
      if (dev[i])
        BB_CUDA(cudaMemcpy2DAsync(dp + items[i].off, (size_t)items[i].rows * items[i].elem, items[i].p, (size_t)items[i].ld * items[i].elem,
                                  (size_t)items[i].rows * items[i].elem, items[i].cols, cudaMemcpyDeviceToDevice, gs));
    BB_CUDA(cudaEventRecord(s->ev_in, gs));                 // the caller may reuse its device buffers in stream order
    BB_CUDA(cudaStreamWaitEvent(s->ctx->stream, s->ev_in, 0));
  }
  PendingGlue pg{};
  pg.n_filters = fl.n; pg.fl = fl;
  s->pend.push_back(pg);
  s->g_pending += 1;
  if (s->g_pending == kGlueGroup || s->q_len + s->g_pending == s->q_cap) {
    // a full group: its glue goes to the glue stream now and its synthesizer launch follows at once, so that the
    // next group's glue (and the host-side staging of its inputs) overlaps it. Groups are as large as the queue
    // allows: a batched glue pass costs ~8 ms + 0.12 ms per collect at n_beam 512 (measured: groups of 4, 8, 8
    // took 35 ms for config 4 where one group of 20 takes 28 ms).
    if ((rc = run_pending_glue(s)) != BB_OK) return rc;
    return launch_queue(s);
  }
  return BB_OK;
}

// Batched glue of the staged collects (glue stream), then their level weights, then — behind one event — their
// prep kernels on the synth stream.
static int run_pending_glue(bb_synth* s) {
  const int nb = s->g_pending;
  if (nb == 0) return BB_OK;
  s->g_pending = 0;
  bb_ctx* c = s->ctx;
  cudaStream_t gs = c->glue_stream;
  const int first = s->q_len, n_ant = s->q_n_ant, n_beam = s->q_n_beam, n_eig = s->q_n_eig, L = s->n_levels;
  const FullLayout& l = s->lay;
  unsigned char* base = s->dev_in + (size_t)first * s->in_slot_bytes;
  GlueBatch g{};
  g.nb = nb; g.n_ant = n_ant; g.n_beam = n_beam; g.n_eig = n_eig; g.gram_mode = s->g_gram_mode;
  g.wavelength = (const double*)(base + l.off_wl); g.stride_wl = (int64_t)(s->in_slot_bytes / 8);
  g.W = s->q_has_w ? (const bb_c32*)(base + l.off_w) : nullptr; g.ldw = n_ant; g.stride_w = (int64_t)(s->in_slot_bytes / 8);
  g.S = (const bb_c32*)(base + l.off_s); g.lds = n_beam; g.stride_s = (int64_t)(s->in_slot_bytes / 8);
  g.xyz = (const double*)(base + l.off_x); g.ldxyz = n_ant; g.stride_xyz = (int64_t)(s->in_slot_bytes / 8);
  g.lambda_dev = s->glue_lambda + (size_t)first * n_eig; g.stride_lam = n_eig;
  g.B_dev = s->glue_B + (size_t)first * n_ant * n_eig; g.stride_b = (int64_t)n_ant * n_eig;
  g.info_dev = s->glue_info + 2 * (size_t)first;
  g.uv = bb_uvgrid_view(s->weighting);
  g.ev_gram0 = get_event(s); g.ev_gram1 = get_event(s); g.ev_eig0 = get_event(s); g.ev_eig1 = get_event(s);
  int launches = 0;
  int rc = bb_glue_eig_batch(c->glue, gs, g, &launches);
  if (rc != BB_OK) {
    s->free_ev.push_back(g.ev_gram0); s->free_ev.push_back(g.ev_gram1); s->free_ev.push_back(g.ev_eig0); s->free_ev.push_back(g.ev_eig1);
    s->pend.clear();
    return rc;
  }
  s->spans.push_back(Span{g.ev_gram0, g.ev_gram1, T_GRAM});
  s->spans.push_back(Span{g.ev_eig0, g.ev_eig1, T_EIG});
  for (int b = 0; b < nb && rc == BB_OK; ++b) {
    const PendingGlue& pg = s->pend[b];
    const int n_intervals = L / pg.n_filters;
    rc = bb_launch_level_weights(g.lambda_dev + (size_t)b * n_eig, n_eig, (const double*)(base + (size_t)b * s->in_slot_bytes + l.off_iv),
                                 n_intervals, n_intervals, pg.fl, s->glue_D + (size_t)(first + b) * L * n_eig, L, g.info_dev + b,
                                 g.info_dev + nb + b, s->status_dev, gs);
    ++launches;
  }
  s->pend.clear();
  s->launches += launches;
  if (rc != BB_OK) return rc;
  BB_CUDA(cudaEventRecord(s->ev_glue, gs));
  BB_CUDA(cudaStreamWaitEvent(c->synth_stream, s->ev_glue, 0));
  // wavelengths are needed on the host by the prep launch: they were staged from the host side of the slot
  for (int b = 0; b < nb && rc == BB_OK; ++b) {
    double wl;
    memcpy(&wl, s->pin + (size_t)(first + b) * s->in_slot_bytes + l.off_wl, sizeof(double));
    rc = enqueue_prepared(s, n_ant, n_eig, wl, s->glue_B + (size_t)(first + b) * n_ant * n_eig, n_ant,
                          s->glue_D + (size_t)(first + b) * L * n_eig, L,
                          (const double*)(s->dev_in + (size_t)(first + b) * s->in_slot_bytes + l.off_x), n_ant);
  }
  return rc;
}

static int check_full_args(bb_synth* s, int n_ant, int n_beam, int n_eig, double wavelength, const bb_c32* W, int ldw,
                           const bb_c32* S, int lds, const double* xyz, int ldxyz, const double* intervals, int ld_int,
                           int n_intervals) {
  if (!s || !S || !xyz || !intervals) return BB_EINVAL;
  if (n_ant < 1 || n_beam < 1 || n_eig < 1 || n_eig > n_beam || n_beam > BB_MAX_BEAMS || !(wavelength > 0.0) || lds < n_beam ||
      ldxyz < n_ant || ld_int < n_intervals || (W && ldw < n_ant) || (!W && n_beam != n_ant) || n_ant > (1 << 20))
    return BB_EINVAL;
  if (n_ant > max_antennas(s->variant)) return BB_EUNSUPPORTED;    // nothing staged, images unchanged: use BB_VARIANT_FP32
  return BB_OK;
}

extern "C" int bb_synth_collect(bb_synth* s, int n_ant, int n_beam, int n_eig, double wavelength, const bb_c32* W,
                                int ldw, const bb_c32* S, int lds, const double* xyz, int ldxyz,
                                const double* intervals, int ld_int) {
  const int lsq = BB_FILTER_LSQ;
  return bb_synth_collect_ex(s, n_ant, n_beam, n_eig, wavelength, W, ldw, S, lds, xyz, ldxyz, intervals, ld_int, 1, &lsq,
                             BB_GRAM_SINC);
}

extern "C" int bb_synth_collect_ex(bb_synth* s, int n_ant, int n_beam, int n_eig, double wavelength, const bb_c32* W,
                                   int ldw, const bb_c32* S, int lds, const double* xyz, int ldxyz,
                                   const double* intervals, int ld_int, int n_filters, const int* filters, int gram_mode) {
  if (!s || !filters || n_filters < 1 || n_filters > BB_MAX_FILTERS || s->n_levels % n_filters != 0 ||
      (gram_mode != BB_GRAM_SINC && gram_mode != BB_GRAM_IDENTITY))
    return BB_EINVAL;
  const int n_intervals = s->n_levels / n_filters;
  FilterList fl{};
  fl.n = n_filters;
  for (int f = 0; f < n_filters; ++f) {
    if (filters[f] != BB_FILTER_LSQ && filters[f] != BB_FILTER_STD) return BB_EINVAL;
    fl.kind[f] = filters[f];
  }
  int rc = check_full_args(s, n_ant, n_beam, n_eig, wavelength, W, ldw, S, lds, xyz, ldxyz, intervals, ld_int, n_intervals);
  if (rc != BB_OK) return rc;
  if (s->weighting && W) return BB_EUNSUPPORTED;           // a beamformed visibility has no single baseline (Q17)
  BB_CUDA(cudaSetDevice(s->ctx->device));
  return stage_full(s, n_ant, n_beam, n_eig, wavelength, W, ldw, S, lds, xyz, ldxyz, intervals, ld_int, n_intervals, fl, gram_mode);
}

// Algorithm 1 for n_collects time steps / channels: the same staging, group after group.
extern "C" int bb_synth_collect_batch(bb_synth* s, int n_collects, int n_ant, int n_beam, int n_eig, const double* wavelengths,
                                      const bb_c32* W, int ldw, int64_t stride_w, const bb_c32* S, int lds, int64_t stride_s,
                                      const double* xyz, int ldxyz, int64_t stride_xyz, const double* intervals, int ld_int) {
  if (!s || !wavelengths || n_collects < 1 || is_device_ptr(wavelengths)) return BB_EINVAL;
  if (stride_s < (int64_t)lds * n_beam || stride_xyz < (int64_t)ldxyz * 3 || (W && stride_w != 0 && stride_w < (int64_t)ldw * n_beam))
    return BB_EINVAL;
  for (int c = 0; c < n_collects; ++c) {
    int rc = check_full_args(s, n_ant, n_beam, n_eig, wavelengths[c], W, ldw, S, lds, xyz, ldxyz, intervals, ld_int, s->n_levels);
    if (rc != BB_OK) return rc;
  }
  if (s->weighting && W) return BB_EUNSUPPORTED;
  BB_CUDA(cudaSetDevice(s->ctx->device));
  FilterList fl{};
  fl.n = 1; fl.kind[0] = BB_FILTER_LSQ;
  for (int c = 0; c < n_collects; ++c) {
    int rc = stage_full(s, n_ant, n_beam, n_eig, wavelengths[c], W ? W + (size_t)c * stride_w : nullptr, ldw, S + (size_t)c * stride_s, lds,
                        xyz + (size_t)c * stride_xyz, ldxyz, intervals, ld_int, s->n_levels, fl, BB_GRAM_SINC);
    if (rc != BB_OK) return rc;
  }
  return BB_OK;
}

extern "C" int bb_synth_set_weighting(bb_synth* s, bb_uvgrid* grid) {
  if (!s) return BB_EINVAL;
  BB_CUDA(cudaSetDevice(s->ctx->device));
  int rc = run_pending_glue(s);                            // collects staged so far keep the weighting they were staged under
  if (rc != BB_OK) return rc;
  s->weighting = grid;
  return BB_OK;
}

static int status_to_code(int flags) {
  if (flags & BB_FLAG_NOTPOSDEF) return BB_ENOTPOSDEF;
  if (flags & BB_FLAG_NOCONV) return BB_ENOCONV;
  if (flags & BB_FLAG_RANGE) return BB_EUNSUPPORTED;
  return BB_OK;
}

extern "C" int bb_synth_status(bb_synth* s) {
  if (!s) return BB_EINVAL;
  BB_CUDA(cudaSetDevice(s->ctx->device));
  int rc = bb_synth_flush(s);
  if (rc != BB_OK) return rc;
  BB_CUDA(cudaMemcpyAsync(s->status_pin, s->status_dev, sizeof(int), cudaMemcpyDeviceToHost, s->ctx->synth_stream));
  if ((rc = sync_all(s)) != BB_OK) return rc;
  fold_spans(s);
  return status_to_code(*s->status_pin);
}

extern "C" int bb_synth_get(bb_synth* s, int level, float* out) {
  if (!s || !out || level < 0 || level >= s->n_levels) return BB_EINVAL;
  BB_CUDA(cudaSetDevice(s->ctx->device));
  int rc = bb_synth_flush(s);
  if (rc != BB_OK) return rc;
  cudaStream_t st = s->ctx->synth_stream;
  BB_CUDA(cudaMemcpyAsync(out, s->img + (size_t)level * s->pix_stride, (size_t)s->n_pix * sizeof(float), cudaMemcpyDefault, st));
  BB_CUDA(cudaMemcpyAsync(s->status_pin, s->status_dev, sizeof(int), cudaMemcpyDeviceToHost, st));
  BB_CUDA(cudaStreamSynchronize(st));
  BB_CUDA(cudaStreamSynchronize(s->ctx->glue_stream));
  fold_spans(s);
  return status_to_code(*s->status_pin);
}

extern "C" int bb_synth_timings(bb_synth* s, double* gram_ms, double* eig_ms, double* prep_ms, double* synth_ms) {
  if (!s) return BB_EINVAL;
  BB_CUDA(cudaSetDevice(s->ctx->device));
  int rc = sync_all(s);
  if (rc != BB_OK) return rc;
  fold_spans(s);
  if (gram_ms) *gram_ms = s->acc_ms[T_GRAM];
  if (eig_ms) *eig_ms = s->acc_ms[T_EIG];
  if (prep_ms) *prep_ms = s->acc_ms[T_PREP];
  if (synth_ms) *synth_ms = s->acc_ms[T_SYNTH];
  return BB_OK;
}

extern "C" int64_t bb_synth_launches(bb_synth* s) { return s ? s->launches : -1; }

// ------------------------------------------------------------------------------ eigen stage alone
extern "C" int bb_eig(bb_ctx* ctx, int n_ant, int n_beam, int n_eig, double wavelength, const bb_c32* W, int ldw,
                      const bb_c32* S, int lds, const double* xyz, int ldxyz, double* lambda_out, bb_c32* B_out,
                      int ldb_out) {
  if (!ctx || !S || !xyz || !lambda_out || n_ant < 1 || n_beam < 1 || n_eig < 1 || n_eig > n_beam ||
      n_beam > BB_MAX_BEAMS || !(wavelength > 0.0) || lds < n_beam || ldxyz < n_ant || (W && ldw < n_ant) ||
      (!W && n_beam != n_ant) || (B_out && ldb_out < n_ant))
    return BB_EINVAL;
  BB_CUDA(cudaSetDevice(ctx->device));
  int rc;
  if (!ctx->glue && (rc = bb_glue_create(&ctx->glue)) != BB_OK) return rc;
  cudaStream_t gs = ctx->glue_stream;
  BB_CUDA(cudaStreamSynchronize(ctx->stream));             // device inputs: the caller's work on the context stream is done
  // device mirrors of host inputs (synchronous: this entry point is not on the hot path)
  std::vector<void*> tmp;
  auto mirror = [&](const void* p, size_t elem, int rows, int cols, int ld, int* ld_out) -> const void* {
    if (!p || is_device_ptr(p)) { *ld_out = ld; return p; }
    void* d = nullptr;
    if (cudaMalloc(&d, (size_t)rows * cols * elem) != cudaSuccess) return nullptr;
    tmp.push_back(d);
    if (cudaMemcpy2D(d, (size_t)rows * elem, p, (size_t)ld * elem, (size_t)rows * elem, cols, cudaMemcpyHostToDevice) != cudaSuccess)
      return nullptr;
    *ld_out = rows;
    return d;
  };
  int ldw2 = ldw, lds2, ldx2;
  const bb_c32* Wd = (const bb_c32*)mirror(W, 8, n_ant, n_beam, ldw, &ldw2);
  const bb_c32* Sd = (const bb_c32*)mirror(S, 8, n_beam, n_beam, lds, &lds2);
  const double* Xd = (const double*)mirror(xyz, 8, n_ant, 3, ldxyz, &ldx2);
  double* lam_d = nullptr; bb_c32* B_d = nullptr; double* wl_d = nullptr; int* info_d = nullptr;
  int info_h[2] = {0, 0};
  rc = BB_OK;
  if ((W && !Wd) || !Sd || !Xd || cudaMalloc(&lam_d, (size_t)n_eig * 8) != cudaSuccess || cudaMalloc(&wl_d, 8) != cudaSuccess ||
      cudaMalloc(&info_d, 2 * sizeof(int)) != cudaSuccess || cudaMalloc(&B_d, (size_t)n_ant * n_eig * 8) != cudaSuccess) rc = BB_EALLOC;
  if (rc == BB_OK && cudaMemcpy(wl_d, &wavelength, 8, cudaMemcpyHostToDevice) != cudaSuccess) rc = BB_ECUDA;
  if (rc == BB_OK) {
    GlueBatch g{};
    g.nb = 1; g.n_ant = n_ant; g.n_beam = n_beam; g.n_eig = n_eig; g.gram_mode = BB_GRAM_SINC;
    g.wavelength = wl_d; g.W = Wd; g.ldw = ldw2; g.S = Sd; g.lds = lds2; g.xyz = Xd; g.ldxyz = ldx2;
    g.lambda_dev = lam_d; g.stride_lam = n_eig; g.B_dev = B_d; g.stride_b = (int64_t)n_ant * n_eig; g.info_dev = info_d;
    rc = bb_glue_eig_batch(ctx->glue, gs, g, nullptr);
  }
  if (rc == BB_OK) {
    cudaError_t e = cudaMemcpyAsync(lambda_out, lam_d, (size_t)n_eig * 8, cudaMemcpyDefault, gs);
    if (e == cudaSuccess && B_out)
      e = cudaMemcpy2DAsync(B_out, (size_t)ldb_out * 8, B_d, (size_t)n_ant * 8, (size_t)n_ant * 8, n_eig, cudaMemcpyDefault, gs);
    if (e == cudaSuccess) e = cudaMemcpyAsync(info_h, info_d, 2 * sizeof(int), cudaMemcpyDeviceToHost, gs);
    if (e == cudaSuccess) e = cudaStreamSynchronize(gs);
    if (e != cudaSuccess) { bb_note_cuda_error(e, "bb_eig copy-out", __FILE__, __LINE__); rc = BB_ECUDA; }
    else if (info_h[0] != 0) rc = BB_ENOTPOSDEF;
    else if (info_h[1] != 0) rc = BB_ENOCONV;
  }
  cudaFree(lam_d); cudaFree(B_d); cudaFree(wl_d); cudaFree(info_d);
  for (void* d : tmp) cudaFree(d);
  cudaGetLastError();
  return rc;
}

// ------------------------------------------------------------------------------ level weights alone
extern "C" int bb_level_weights(bb_ctx* ctx, const double* lambda, int n_eig, const double* intervals, int ld_int,
                                int n_intervals, int n_filters, const int* filters, float* D_out, int ldd) {
  if (!ctx || !lambda || !intervals || !filters || !D_out || n_eig < 1 || n_intervals < 1 || ld_int < n_intervals ||
      n_filters < 1 || n_filters > BB_MAX_FILTERS || n_intervals * n_filters > BB_MAX_LEVELS || ldd < n_intervals * n_filters)
    return BB_EINVAL;
  FilterList fl{};
  fl.n = n_filters;
  for (int f = 0; f < n_filters; ++f) {
    if (filters[f] != BB_FILTER_LSQ && filters[f] != BB_FILTER_STD) return BB_EINVAL;
    fl.kind[f] = filters[f];
  }
  BB_CUDA(cudaSetDevice(ctx->device));
  const int L = n_intervals * n_filters;
  double* lam_d = nullptr; double* iv_d = nullptr; float* D_d = nullptr;
  int rc = BB_OK;
  if (cudaMalloc(&lam_d, (size_t)n_eig * 8) != cudaSuccess || cudaMalloc(&iv_d, (size_t)n_intervals * 16) != cudaSuccess ||
      cudaMalloc(&D_d, (size_t)L * n_eig * 4) != cudaSuccess) rc = BB_EALLOC;
  cudaStream_t st = ctx->stream;
  cudaError_t e = cudaSuccess;
  if (rc == BB_OK) e = cudaMemcpyAsync(lam_d, lambda, (size_t)n_eig * 8, cudaMemcpyDefault, st);
  if (rc == BB_OK && e == cudaSuccess)
    e = cudaMemcpy2DAsync(iv_d, (size_t)n_intervals * 8, intervals, (size_t)ld_int * 8, (size_t)n_intervals * 8, 2, cudaMemcpyDefault, st);
  if (rc == BB_OK && e == cudaSuccess) rc = bb_launch_level_weights(lam_d, n_eig, iv_d, n_intervals, n_intervals, fl, D_d, L, nullptr, nullptr, nullptr, st);
  if (rc == BB_OK && e == cudaSuccess)
    e = cudaMemcpy2DAsync(D_out, (size_t)ldd * 4, D_d, (size_t)L * 4, (size_t)L * 4, n_eig, cudaMemcpyDefault, st);
  if (rc == BB_OK && e == cudaSuccess) e = cudaStreamSynchronize(st);
  if (rc == BB_OK && e != cudaSuccess) { bb_note_cuda_error(e, "bb_level_weights", __FILE__, __LINE__); rc = BB_ECUDA; }
  cudaFree(lam_d); cudaFree(iv_d); cudaFree(D_d);
  cudaGetLastError();
  return rc;
}

// ------------------------------------------------------------------------------ parameter estimation
static int lambda_to_device(const double* lambda, int n, double** dev, bool* owned) {
  *owned = false;
  if (is_device_ptr(lambda)) { *dev = const_cast<double*>(lambda); return BB_OK; }
  if (cudaMalloc(dev, (size_t)n * sizeof(double)) != cudaSuccess) { cudaGetLastError(); return BB_EALLOC; }
  *owned = true;
  BB_CUDA(cudaMemcpy(*dev, lambda, (size_t)n * sizeof(double), cudaMemcpyHostToDevice));
  return BB_OK;
}

extern "C" int bb_estimate_n_eig(bb_ctx* ctx, const double* lambda, int n, double energy_fraction, int* n_eig_out) {
  if (!ctx || !lambda || !n_eig_out || n < 1 || n > BB_MAX_ESTIMATE || !(energy_fraction > 0.0) || energy_fraction > 1.0)
    return BB_EINVAL;
  BB_CUDA(cudaSetDevice(ctx->device));
  double* lam = nullptr; bool owned = false; int* out = nullptr;
  int rc = lambda_to_device(lambda, n, &lam, &owned);
  if (rc == BB_OK && cudaMalloc(&out, sizeof(int)) != cudaSuccess) rc = BB_EALLOC;
  if (rc == BB_OK) rc = bb_estimate_n_eig_dev(lam, n, energy_fraction, out, ctx->stream);
  if (rc == BB_OK) {
    cudaError_t e = cudaMemcpyAsync(n_eig_out, out, sizeof(int), cudaMemcpyDeviceToHost, ctx->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(ctx->stream);
    if (e != cudaSuccess) { bb_note_cuda_error(e, "bb_estimate_n_eig", __FILE__, __LINE__); rc = BB_ECUDA; }
  }
  if (owned) cudaFree(lam);
  cudaFree(out);
  cudaGetLastError();
  return rc;
}

extern "C" int bb_kmeans_levels(bb_ctx* ctx, const double* lambda, int n, int n_levels, int log_domain,
                                double* intervals_out, int ld_int) {
  if (!ctx || !lambda || !intervals_out || n < 1 || n > BB_MAX_ESTIMATE || n_levels < 1 || n_levels > BB_MAX_LEVELS ||
      n_levels > n || ld_int < n_levels)
    return BB_EINVAL;
  BB_CUDA(cudaSetDevice(ctx->device));
  double* lam = nullptr; bool owned = false;
  double* ws = nullptr; int* arg = nullptr; double* iv = nullptr; int* status = nullptr;
  int rc = lambda_to_device(lambda, n, &lam, &owned);
  if (rc == BB_OK && (cudaMalloc(&ws, bb_kmeans_workspace_doubles(n) * sizeof(double)) != cudaSuccess ||
                      cudaMalloc(&arg, bb_kmeans_workspace_ints(n, n_levels) * sizeof(int)) != cudaSuccess ||
                      cudaMalloc(&iv, (size_t)2 * n_levels * sizeof(double)) != cudaSuccess ||
                      cudaMalloc(&status, sizeof(int)) != cudaSuccess)) rc = BB_EALLOC;
  if (rc == BB_OK) rc = bb_kmeans_levels_dev(lam, n, n_levels, log_domain != 0, ws, arg, iv, n_levels, status, ctx->stream);
  if (rc == BB_OK) {
    int st_host = -1;
    cudaError_t e = cudaMemcpyAsync(&st_host, status, sizeof(int), cudaMemcpyDeviceToHost, ctx->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(ctx->stream);
    if (e == cudaSuccess && st_host == 0)
      e = cudaMemcpy2D(intervals_out, (size_t)ld_int * sizeof(double), iv, (size_t)n_levels * sizeof(double),
                       (size_t)n_levels * sizeof(double), 2, cudaMemcpyDefault);
    if (e != cudaSuccess) { bb_note_cuda_error(e, "bb_kmeans_levels", __FILE__, __LINE__); rc = BB_ECUDA; }
    else if (st_host != 0) rc = BB_EINVAL;                 // fewer positive eigenvalues than levels
  }
  if (owned) cudaFree(lam);
  cudaFree(ws); cudaFree(arg); cudaFree(iv); cudaFree(status);
  cudaGetLastError();
  return rc;
}
