// C ABI of libbluebild_b200.so (include/bluebild.h): argument validation, host/device pointer
// handling, the queue of prepared collects and the stream-ordered launch sequence.
// All arithmetic of the method runs in the CUDA kernels of kernels_fp32.cu / kernels_tc.cu /
// glue.cu / pixels.cu; nothing here computes on the host and there is no CPU fallback.
#include "internal.h"

#include <cstdio>
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
    case BB_EUNSUPPORTED: return "unsupported variant or size";
    default: return "unknown status";
  }
}

extern "C" const char* bb_version(void) { return "bluebild-b200 0.1 (sm_100a)"; }

// ------------------------------------------------------------------------------ handles
struct bb_ctx {
  int device = 0;
  cudaStream_t stream = nullptr;
  int sm_count = 0;
  GlueWork* glue = nullptr;
};

enum { T_GRAM = 0, T_EIG = 1, T_PREP = 2, T_SYNTH = 3, T_KINDS = 4 };
struct Span { cudaEvent_t a, b; int kind; };

struct bb_synth {
  bb_ctx* ctx = nullptr;
  int64_t n_pix = 0, pix_stride = 0;
  int n_levels = 0, variant = 0;
  double* rprime = nullptr;
  double rc[3] = {0, 0, 0};
  float* img = nullptr;
  // queue of prepared collects (all with the same n_ant, n_eig)
  int q_cap = 0, q_len = 0, q_n_ant = 0, q_n_eig = 0;
  Fp32Plan fplan{};
  TcPlan tplan{};
  unsigned char* packed = nullptr; size_t packed_stride = 0;
  float* weights = nullptr; size_t weight_stride = 0;
  // staging of caller inputs, one slot per queue entry
  unsigned char* pin = nullptr; unsigned char* dev_in = nullptr; size_t in_slot_bytes = 0;
  std::vector<cudaEvent_t> slot_ev; std::vector<char> slot_busy;
  // glue outputs per slot
  bb_c32* glue_B = nullptr; double* glue_lambda = nullptr; float* glue_D = nullptr;
  // timing
  std::vector<Span> spans; std::vector<cudaEvent_t> free_ev;
  double acc_ms[T_KINDS] = {0, 0, 0, 0};
  int64_t launches = 0;
};

static bool is_device_ptr(const void* p) {
  cudaPointerAttributes at;
  if (cudaPointerGetAttributes(&at, p) != cudaSuccess) { cudaGetLastError(); return false; }
  return at.type == cudaMemoryTypeDevice || at.type == cudaMemoryTypeManaged;
}

static cudaEvent_t get_event(bb_synth* s) {
  if (!s->free_ev.empty()) { cudaEvent_t e = s->free_ev.back(); s->free_ev.pop_back(); return e; }
  cudaEvent_t e = nullptr;
  cudaEventCreate(&e);
  return e;
}

static void fold_spans(bb_synth* s) {  // caller guarantees the stream is (or will be) synchronised
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

struct SpanGuard {  // records an event pair around a stream region
  bb_synth* s; Span sp;
  SpanGuard(bb_synth* s_, int kind) : s(s_) {
    sp.a = get_event(s); sp.b = get_event(s); sp.kind = kind;
    cudaEventRecord(sp.a, s->ctx->stream);
  }
  ~SpanGuard() { cudaEventRecord(sp.b, s->ctx->stream); s->spans.push_back(sp); }
};

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
  *out = c;
  return BB_OK;
}

extern "C" int bb_ctx_destroy(bb_ctx* ctx) {
  if (!ctx) return BB_EINVAL;
  if (ctx->glue) bb_glue_destroy(ctx->glue);
  delete ctx;
  return BB_OK;
}

extern "C" int bb_probe_peak(bb_ctx* ctx, int kind, double* ops_per_s, double* ms) {
  if (!ctx || !ops_per_s || !ms) return BB_EINVAL;
  BB_CUDA(cudaSetDevice(ctx->device));
  return bb_probe_run(kind, ctx->sm_count, ctx->stream, ops_per_s, ms);
}

// ------------------------------------------------------------------------------ imaging handle
static void free_queue(bb_synth* s) {
  cudaFree(s->packed); s->packed = nullptr;
  cudaFree(s->weights); s->weights = nullptr;
  cudaFree(s->dev_in); s->dev_in = nullptr;
  cudaFree(s->glue_B); s->glue_B = nullptr;
  cudaFree(s->glue_lambda); s->glue_lambda = nullptr;
  cudaFree(s->glue_D); s->glue_D = nullptr;
  if (s->pin) { cudaFreeHost(s->pin); s->pin = nullptr; }
  for (cudaEvent_t e : s->slot_ev) cudaEventDestroy(e);
  s->slot_ev.clear(); s->slot_busy.clear();
  s->q_cap = s->q_len = s->q_n_ant = s->q_n_eig = 0;
}

extern "C" int bb_synth_destroy(bb_synth* s) {
  if (!s) return BB_EINVAL;
  cudaSetDevice(s->ctx->device);
  cudaStreamSynchronize(s->ctx->stream);
  fold_spans(s);
  for (cudaEvent_t e : s->free_ev) cudaEventDestroy(e);
  free_queue(s);
  cudaFree(s->rprime);
  cudaFree(s->img);
  cudaGetLastError();
  delete s;
  return BB_OK;
}

extern "C" int bb_synth_create(bb_ctx* ctx, int64_t n_pix, const double* pix, int64_t ld_pix, int n_levels,
                               int variant, bb_synth** out) {
  if (!out) return BB_EINVAL;
  *out = nullptr;
  if (!ctx || n_pix < 0 || (n_pix > 0 && !pix) || ld_pix < n_pix || n_levels < 1 || n_levels > BB_MAX_LEVELS)
    return BB_EINVAL;
  if (variant != BB_VARIANT_FP32 && variant != BB_VARIANT_TF32X3 && variant != BB_VARIANT_FP16X3) return BB_EUNSUPPORTED;
  BB_CUDA(cudaSetDevice(ctx->device));
  bb_synth* s = new (std::nothrow) bb_synth;
  if (!s) return BB_EALLOC;
  s->ctx = ctx; s->n_pix = n_pix; s->n_levels = n_levels; s->variant = variant;
  s->pix_stride = (n_pix + 511) / 512 * 512 + 512;   // whole tiles may be read past n_pix
  int rc = BB_OK;
  double* tmp = nullptr;
  do {
    if (cudaMalloc(&s->rprime, 3 * (size_t)s->pix_stride * sizeof(double)) != cudaSuccess ||
        cudaMalloc(&s->img, (size_t)n_levels * s->pix_stride * sizeof(float)) != cudaSuccess) { rc = BB_EALLOC; break; }
    if (cudaMemsetAsync(s->img, 0, (size_t)n_levels * s->pix_stride * sizeof(float), ctx->stream) != cudaSuccess) { rc = BB_ECUDA; break; }
    const double* pix_dev = pix;
    int64_t ld = ld_pix;
    if (n_pix > 0 && !is_device_ptr(pix)) {
      if (cudaMalloc(&tmp, 3 * (size_t)n_pix * sizeof(double)) != cudaSuccess) { rc = BB_EALLOC; break; }
      if (cudaMemcpy2D(tmp, n_pix * sizeof(double), pix, ld_pix * sizeof(double), n_pix * sizeof(double), 3,
                       cudaMemcpyHostToDevice) != cudaSuccess) { rc = BB_ECUDA; break; }
      pix_dev = tmp; ld = n_pix;
    }
    if (n_pix > 0) rc = bb_pixels_prepare(pix_dev, n_pix, ld, s->rprime, s->pix_stride, s->rc, ctx->stream);
    else if (cudaMemsetAsync(s->rprime, 0, 3 * (size_t)s->pix_stride * sizeof(double), ctx->stream) != cudaSuccess) rc = BB_ECUDA;
  } while (0);
  cudaFree(tmp);
  if (rc != BB_OK) { cudaGetLastError(); bb_synth_destroy(s); return rc; }
  *out = s;
  return BB_OK;
}

extern "C" int bb_synth_reset(bb_synth* s) {
  if (!s) return BB_EINVAL;
  BB_CUDA(cudaSetDevice(s->ctx->device));
  s->q_len = 0;
  BB_CUDA(cudaMemsetAsync(s->img, 0, (size_t)s->n_levels * s->pix_stride * sizeof(float), s->ctx->stream));
  BB_CUDA(cudaStreamSynchronize(s->ctx->stream));
  fold_spans(s);
  for (int k = 0; k < T_KINDS; ++k) s->acc_ms[k] = 0;
  s->launches = 0;
  return BB_OK;
}

extern "C" int bb_synth_flush(bb_synth* s) {
  if (!s) return BB_EINVAL;
  if (s->q_len == 0) return BB_OK;
  BB_CUDA(cudaSetDevice(s->ctx->device));
  SynthArgs a{};
  a.rprime = s->rprime; a.n_pix = s->n_pix; a.pix_stride = s->pix_stride;
  a.packed = s->packed; a.packed_stride = s->packed_stride;
  a.weights = s->weights; a.weight_stride = s->weight_stride;
  a.n_collects = s->q_len; a.n_levels = s->n_levels;
  a.img = s->img; a.img_stride = s->pix_stride;
  int launches = 0, rc;
  {
    SpanGuard g(s, T_SYNTH);
    rc = (s->variant == BB_VARIANT_FP32) ? bb_launch_synth_fp32(s->fplan, a, s->ctx->sm_count, s->ctx->stream, &launches)
                                         : bb_launch_synth_tc(s->tplan, a, s->ctx->sm_count, s->ctx->stream, &launches);
  }
  s->launches += launches;
  s->q_len = 0;
  return rc;
}

// (Re)size the queue for collects of shape (n_ant, n_eig); flushes pending work of another shape.
static int ensure_queue(bb_synth* s, int n_ant, int n_beam, int n_eig) {
  if (s->q_cap > 0 && s->q_n_ant == n_ant && s->q_n_eig == n_eig) return BB_OK;
  int rc = bb_synth_flush(s);
  if (rc != BB_OK) return rc;
  BB_CUDA(cudaStreamSynchronize(s->ctx->stream));
  fold_spans(s);
  free_queue(s);
  const int L = s->n_levels;
  if (s->variant == BB_VARIANT_FP32) {
    s->fplan = bb_fp32_plan(n_ant, n_eig, L);
    s->packed_stride = s->fplan.collect_bytes; s->weight_stride = s->fplan.weight_floats;
  } else {
    s->tplan = bb_tc_plan(n_ant, n_eig, L, s->variant == BB_VARIANT_FP16X3 ? BB_TC_FP16 : BB_TC_TF32);
    if (s->tplan.n_chunks == 0) return BB_EUNSUPPORTED;
    s->packed_stride = s->tplan.collect_bytes; s->weight_stride = s->tplan.weight_floats;
  }
  // queue depth: enough collects per launch to amortise the image read-modify-write, bounded memory
  size_t per = s->packed_stride + s->weight_stride * 4;
  int cap = 32;
  while (cap > 4 && per * cap > ((size_t)256 << 20)) cap /= 2;
  // staging slot: B | D | xyz (collect_eig) or W | S | xyz | intervals (collect) — size for the larger
  size_t eig_bytes = (size_t)n_ant * n_eig * 8 + (size_t)L * n_eig * 4 + (size_t)n_ant * 24;
  size_t full_bytes = (size_t)n_ant * n_beam * 8 + (size_t)n_beam * n_beam * 8 + (size_t)n_ant * 24 + (size_t)L * 16;
  s->in_slot_bytes = ((eig_bytes > full_bytes ? eig_bytes : full_bytes) + 255) / 256 * 256;
  if (cudaMalloc(&s->packed, s->packed_stride * cap) != cudaSuccess ||
      cudaMalloc(&s->weights, s->weight_stride * 4 * cap) != cudaSuccess ||
      cudaMalloc(&s->dev_in, s->in_slot_bytes * cap) != cudaSuccess ||
      cudaMalloc(&s->glue_B, (size_t)n_ant * n_eig * 8 * cap) != cudaSuccess ||
      cudaMalloc(&s->glue_lambda, (size_t)n_eig * 8 * cap) != cudaSuccess ||
      cudaMalloc(&s->glue_D, (size_t)L * n_eig * 4 * cap) != cudaSuccess ||
      cudaMallocHost(&s->pin, s->in_slot_bytes * cap) != cudaSuccess) {
    cudaGetLastError(); free_queue(s); return BB_EALLOC;
  }
  s->slot_ev.resize(cap); s->slot_busy.assign(cap, 0);
  for (int i = 0; i < cap; ++i) cudaEventCreateWithFlags(&s->slot_ev[i], cudaEventDisableTiming);
  s->q_cap = cap; s->q_len = 0; s->q_n_ant = n_ant; s->q_n_eig = n_eig;
  return BB_OK;
}

// Copy a column-major host matrix (rows x cols, ld) compactly into dst; returns bytes written.
static size_t pack_host(void* dst, const void* src, size_t elem, int rows, int cols, int ld) {
  for (int c = 0; c < cols; ++c)
    memcpy((char*)dst + (size_t)c * rows * elem, (const char*)src + (size_t)c * ld * elem, (size_t)rows * elem);
  return (size_t)rows * cols * elem;
}

// Stage one input: host -> pinned slot (snapshot) with device mirror, or pass the device pointer through.
struct Stager {
  bb_synth* s; int slot; size_t off = 0; bool used = false;
  Stager(bb_synth* s_, int slot_) : s(s_), slot(slot_) {}
  template <class T>
  const T* put(const T* p, int rows, int cols, int ld, int* ld_out) {
    if (!p) { *ld_out = ld; return nullptr; }
    if (is_device_ptr(p)) { *ld_out = ld; return p; }
    if (!used) {  // the slot's previous H2D copy must have completed before its pinned memory is rewritten
      if (s->slot_busy[slot]) { cudaEventSynchronize(s->slot_ev[slot]); s->slot_busy[slot] = 0; }
      used = true;
    }
    unsigned char* hp = s->pin + (size_t)slot * s->in_slot_bytes + off;
    const T* dp = reinterpret_cast<const T*>(s->dev_in + (size_t)slot * s->in_slot_bytes + off);
    off += (pack_host(hp, p, sizeof(T), rows, cols, ld) + 15) / 16 * 16;
    *ld_out = rows;
    return dp;
  }
  int commit() {
    if (!used) return BB_OK;
    BB_CUDA(cudaMemcpyAsync(s->dev_in + (size_t)slot * s->in_slot_bytes, s->pin + (size_t)slot * s->in_slot_bytes, off,
                            cudaMemcpyHostToDevice, s->ctx->stream));
    BB_CUDA(cudaEventRecord(s->slot_ev[slot], s->ctx->stream));
    s->slot_busy[slot] = 1;
    return BB_OK;
  }
};

static int enqueue_prepared(bb_synth* s, int n_ant, int n_eig, double wavelength, const bb_c32* B, int ldb,
                            const float* D, int ldd, const double* xyz, int ldxyz) {
  PrepArgs a{};
  a.B = B; a.ldb = ldb; a.D = D; a.ldd = ldd; a.xyz = xyz; a.ldxyz = ldxyz;
  a.n_ant = n_ant; a.n_eig = n_eig; a.n_levels = s->n_levels; a.wavelength = wavelength;
  a.rc[0] = s->rc[0]; a.rc[1] = s->rc[1]; a.rc[2] = s->rc[2];
  a.packed = s->packed + (size_t)s->q_len * s->packed_stride;
  a.weights = s->weights + (size_t)s->q_len * s->weight_stride;
  int rc;
  {
    SpanGuard g(s, T_PREP);
    rc = (s->variant == BB_VARIANT_FP32) ? bb_launch_prep_fp32(s->fplan, a, s->ctx->stream)
                                         : bb_launch_prep_tc(s->tplan, a, s->ctx->stream);
  }
  if (rc != BB_OK) return rc;
  s->launches += 1;
  s->q_len += 1;
  if (s->spans.size() > 8192) { cudaStreamSynchronize(s->ctx->stream); fold_spans(s); }
  if (s->q_len == s->q_cap) return bb_synth_flush(s);
  return BB_OK;
}

extern "C" int bb_synth_collect_eig(bb_synth* s, int n_ant, int n_eig, double wavelength, const bb_c32* B, int ldb,
                                    const float* D, int ldd, const double* xyz, int ldxyz) {
  if (!s || !B || !D || !xyz || n_ant < 1 || n_eig < 1 || !(wavelength > 0.0) || ldb < n_ant ||
      ldd < s->n_levels || ldxyz < n_ant || n_eig > 4096 || n_ant > (1 << 20))
    return BB_EINVAL;
  BB_CUDA(cudaSetDevice(s->ctx->device));
  int rc = ensure_queue(s, n_ant, n_eig, n_eig);
  if (rc != BB_OK) return rc;
  Stager st(s, s->q_len);
  int ldb2, ldd2, ldx2;
  const bb_c32* Bd = st.put(B, n_ant, n_eig, ldb, &ldb2);
  const float* Dd = st.put(D, s->n_levels, n_eig, ldd, &ldd2);
  const double* Xd = st.put(xyz, n_ant, 3, ldxyz, &ldx2);
  if ((rc = st.commit()) != BB_OK) return rc;
  return enqueue_prepared(s, n_ant, n_eig, wavelength, Bd, ldb2, Dd, ldd2, Xd, ldx2);
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
  if (!s || !S || !xyz || !intervals || !filters || n_filters < 1 || n_filters > BB_MAX_FILTERS ||
      s->n_levels % n_filters != 0 || (gram_mode != BB_GRAM_SINC && gram_mode != BB_GRAM_IDENTITY))
    return BB_EINVAL;
  const int n_intervals = s->n_levels / n_filters;
  FilterList fl{};
  fl.n = n_filters;
  for (int f = 0; f < n_filters; ++f) {
    if (filters[f] != BB_FILTER_LSQ && filters[f] != BB_FILTER_STD) return BB_EINVAL;
    fl.kind[f] = filters[f];
  }
  if (n_ant < 1 || n_beam < 1 || n_eig < 1 || n_eig > n_beam ||
      n_beam > BB_MAX_BEAMS || !(wavelength > 0.0) || lds < n_beam || ldxyz < n_ant || ld_int < n_intervals ||
      (W && ldw < n_ant) || (!W && n_beam != n_ant) || n_ant > (1 << 20))
    return BB_EINVAL;
  BB_CUDA(cudaSetDevice(s->ctx->device));
  int rc = ensure_queue(s, n_ant, n_beam, n_eig);
  if (rc != BB_OK) return rc;
  if (!s->ctx->glue && (rc = bb_glue_create(&s->ctx->glue)) != BB_OK) return rc;
  const int slot = s->q_len;
  Stager st(s, slot);
  int ldw2, lds2, ldx2, ldi2;
  const bb_c32* Wd = st.put(W, n_ant, n_beam, ldw, &ldw2);
  const bb_c32* Sd = st.put(S, n_beam, n_beam, lds, &lds2);
  const double* Xd = st.put(xyz, n_ant, 3, ldxyz, &ldx2);
  const double* Id = st.put(intervals, n_intervals, 2, ld_int, &ldi2);
  if ((rc = st.commit()) != BB_OK) return rc;
  bb_c32* Bd = s->glue_B + (size_t)slot * n_ant * n_eig;
  double* lam = s->glue_lambda + (size_t)slot * n_eig;
  float* Dd = s->glue_D + (size_t)slot * s->n_levels * n_eig;
  cudaEvent_t e0 = get_event(s), e1 = get_event(s), e2 = get_event(s), e3 = get_event(s);
  rc = bb_glue_eig(s->ctx->glue, s->ctx->stream, n_ant, n_beam, n_eig, wavelength, Wd, ldw2, Sd, lds2, Xd, ldx2, lam,
                   Bd, e0, e1, e2, e3, gram_mode);
  if (rc != BB_OK) {
    s->free_ev.push_back(e0); s->free_ev.push_back(e1); s->free_ev.push_back(e2); s->free_ev.push_back(e3);
    return rc;
  }
  s->spans.push_back(Span{e0, e1, T_GRAM});
  s->spans.push_back(Span{e2, e3, T_EIG});
  s->launches += 6;  // gram, symmetrise/convert, select, cast kernels of glue.cu (library calls not counted)
  if ((rc = bb_launch_level_weights(lam, n_eig, Id, ldi2, n_intervals, fl, Dd, s->n_levels, s->ctx->stream)) != BB_OK) return rc;
  s->launches += 1;
  return enqueue_prepared(s, n_ant, n_eig, wavelength, Bd, n_ant, Dd, s->n_levels, Xd, ldx2);
}

// Algorithm 1 for n_collects time steps / channels at once: the eigenproblems are solved as one batch.
extern "C" int bb_synth_collect_batch(bb_synth* s, int n_collects, int n_ant, int n_beam, int n_eig, const double* wavelengths,
                                      const bb_c32* W, int ldw, int64_t stride_w, const bb_c32* S, int lds, int64_t stride_s,
                                      const double* xyz, int ldxyz, int64_t stride_xyz, const double* intervals, int ld_int) {
  if (!s || !S || !xyz || !intervals || !wavelengths || n_collects < 1 || n_ant < 1 || n_beam < 1 || n_eig < 1 || n_eig > n_beam ||
      n_beam > BB_MAX_BEAMS || lds < n_beam || ldxyz < n_ant || ld_int < s->n_levels || (W && ldw < n_ant) ||
      (!W && n_beam != n_ant) || n_ant > (1 << 20) || stride_s < (int64_t)lds * n_beam || stride_xyz < (int64_t)ldxyz * 3 ||
      (W && stride_w != 0 && stride_w < (int64_t)ldw * n_beam) || is_device_ptr(wavelengths))
    return BB_EINVAL;
  for (int c = 0; c < n_collects; ++c)
    if (!(wavelengths[c] > 0.0)) return BB_EINVAL;
  BB_CUDA(cudaSetDevice(s->ctx->device));
  int rc = ensure_queue(s, n_ant, n_beam, n_eig);
  if (rc != BB_OK) return rc;
  if (!s->ctx->glue && (rc = bb_glue_create(&s->ctx->glue)) != BB_OK) return rc;
  cudaStream_t st = s->ctx->stream;
  const int L = s->n_levels;
  // device mirrors of host inputs (synchronous copies: this is glue) and per-batch outputs
  std::vector<void*> tmp;
  auto dev_copy = [&](const void* p, size_t bytes) -> const void* {
    if (!p || is_device_ptr(p)) return p;
    void* d = nullptr;
    if (cudaMalloc(&d, bytes) != cudaSuccess) { cudaGetLastError(); return nullptr; }
    tmp.push_back(d);
    if (cudaMemcpy(d, p, bytes, cudaMemcpyHostToDevice) != cudaSuccess) { cudaGetLastError(); return nullptr; }
    return d;
  };
  auto dev_alloc = [&](size_t bytes) -> void* {
    void* d = nullptr;
    if (cudaMalloc(&d, bytes) != cudaSuccess) { cudaGetLastError(); return nullptr; }
    tmp.push_back(d);
    return d;
  };
  const size_t nS = (size_t)(n_collects - 1) * stride_s + (size_t)lds * n_beam;
  const size_t nX = (size_t)(n_collects - 1) * stride_xyz + (size_t)ldxyz * 3;
  const size_t nW = W ? (size_t)(stride_w ? n_collects - 1 : 0) * stride_w + (size_t)ldw * n_beam : 0;
  const bb_c32* Sd = (const bb_c32*)dev_copy(S, nS * sizeof(bb_c32));
  const double* Xd = (const double*)dev_copy(xyz, nX * sizeof(double));
  const bb_c32* Wd = W ? (const bb_c32*)dev_copy(W, nW * sizeof(bb_c32)) : nullptr;
  const double* wl_d = (const double*)dev_copy(wavelengths, (size_t)n_collects * sizeof(double));
  double* iv_d = (double*)dev_alloc((size_t)2 * L * sizeof(double));
  double* lam_d = (double*)dev_alloc((size_t)n_collects * n_eig * sizeof(double));
  bb_c32* B_d = (bb_c32*)dev_alloc((size_t)n_collects * n_ant * n_eig * sizeof(bb_c32));
  float* D_d = (float*)dev_alloc((size_t)n_collects * L * n_eig * sizeof(float));
  rc = BB_OK;
  if (!Sd || !Xd || (W && !Wd) || !wl_d || !iv_d || !lam_d || !B_d || !D_d) rc = BB_EALLOC;
  if (rc == BB_OK && cudaMemcpy2D(iv_d, (size_t)L * sizeof(double), intervals, (size_t)ld_int * sizeof(double), (size_t)L * sizeof(double),
                                  2, cudaMemcpyDefault) != cudaSuccess) { cudaGetLastError(); rc = BB_ECUDA; }
  FilterList fl{};
  fl.n = 1; fl.kind[0] = BB_FILTER_LSQ;
  const int group = 16;                                    // eigenproblems per batched solve (bounded workspace)
  for (int c0 = 0; rc == BB_OK && c0 < n_collects; c0 += group) {
    const int nb = n_collects - c0 < group ? n_collects - c0 : group;
    cudaEvent_t e0 = get_event(s), e1 = get_event(s), e2 = get_event(s), e3 = get_event(s);
    rc = bb_glue_eig_batch(s->ctx->glue, st, nb, n_ant, n_beam, n_eig, wl_d + c0, Wd ? Wd + (size_t)c0 * stride_w : nullptr, ldw,
                           stride_w, Sd + (size_t)c0 * stride_s, lds, stride_s, Xd + (size_t)c0 * stride_xyz, ldxyz, stride_xyz,
                           lam_d + (size_t)c0 * n_eig, B_d + (size_t)c0 * n_ant * n_eig, e0, e1, e2, e3);
    if (rc != BB_OK) {
      s->free_ev.push_back(e0); s->free_ev.push_back(e1); s->free_ev.push_back(e2); s->free_ev.push_back(e3);
      break;
    }
    s->spans.push_back(Span{e0, e1, T_GRAM});
    s->spans.push_back(Span{e2, e3, T_EIG});
    s->launches += 10;                                     // this file's batched kernels (library calls not counted)
    for (int c = c0; rc == BB_OK && c < c0 + nb; ++c) {
      float* Dc = D_d + (size_t)c * L * n_eig;
      rc = bb_launch_level_weights(lam_d + (size_t)c * n_eig, n_eig, iv_d, L, L, fl, Dc, L, st);
      if (rc != BB_OK) break;
      s->launches += 1;
      rc = enqueue_prepared(s, n_ant, n_eig, wavelengths[c], B_d + (size_t)c * n_ant * n_eig, n_ant, Dc, L,
                            Xd + (size_t)c * stride_xyz, ldxyz);
    }
  }
  cudaStreamSynchronize(st);                               // the prep kernels have consumed the temporaries
  for (void* d : tmp) cudaFree(d);
  cudaGetLastError();
  return rc;
}

extern "C" int bb_synth_get(bb_synth* s, int level, float* out) {
  if (!s || !out || level < 0 || level >= s->n_levels) return BB_EINVAL;
  BB_CUDA(cudaSetDevice(s->ctx->device));
  int rc = bb_synth_flush(s);
  if (rc != BB_OK) return rc;
  BB_CUDA(cudaMemcpyAsync(out, s->img + (size_t)level * s->pix_stride, (size_t)s->n_pix * sizeof(float),
                          cudaMemcpyDefault, s->ctx->stream));
  BB_CUDA(cudaStreamSynchronize(s->ctx->stream));
  fold_spans(s);
  return BB_OK;
}

extern "C" int bb_synth_timings(bb_synth* s, double* gram_ms, double* eig_ms, double* prep_ms, double* synth_ms) {
  if (!s) return BB_EINVAL;
  BB_CUDA(cudaSetDevice(s->ctx->device));
  BB_CUDA(cudaStreamSynchronize(s->ctx->stream));
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
  double* lam_d = nullptr; bb_c32* B_d = nullptr;
  rc = BB_OK;
  if ((W && !Wd) || !Sd || !Xd || cudaMalloc(&lam_d, (size_t)n_eig * 8) != cudaSuccess ||
      cudaMalloc(&B_d, (size_t)n_ant * n_eig * 8) != cudaSuccess) rc = BB_EALLOC;
  if (rc == BB_OK)
    rc = bb_glue_eig(ctx->glue, ctx->stream, n_ant, n_beam, n_eig, wavelength, Wd, ldw2, Sd, lds2, Xd, ldx2, lam_d, B_d,
                     nullptr, nullptr, nullptr, nullptr);
  if (rc == BB_OK) {
    cudaError_t e = cudaMemcpyAsync(lambda_out, lam_d, (size_t)n_eig * 8, cudaMemcpyDefault, ctx->stream);
    if (e == cudaSuccess && B_out)
      e = cudaMemcpy2DAsync(B_out, (size_t)ldb_out * 8, B_d, (size_t)n_ant * 8, (size_t)n_ant * 8, n_eig, cudaMemcpyDefault, ctx->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(ctx->stream);
    if (e != cudaSuccess) { bb_note_cuda_error(e, "bb_eig copy-out", __FILE__, __LINE__); rc = BB_ECUDA; }
  }
  cudaFree(lam_d); cudaFree(B_d);
  for (void* d : tmp) cudaFree(d);
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
