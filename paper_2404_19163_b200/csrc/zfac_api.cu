// C ABI of libzfac (see include/zfac.h).  Host-side sequencing only: every step of the
// path runs in the kernels of zfac_f64.cuh / zfac_umma.cuh / zfac_io.cuh.
#include <cuda.h>
#include <cuda_runtime.h>
#include <stdio.h>
#include <string.h>
#include <new>
#include <type_traits>

#include "zfac_common.cuh"
#include "zfac_io.cuh"
#include "zfac_f64.cuh"
#include "zfac_umma.cuh"
#include "zfac_f64_tma.cuh"
#include "zfac_mix.cuh"

using namespace zfac;

static thread_local char g_cuda_err[256] = "";

#define ZF_CUDA(call)                                                                     \
  do {                                                                                    \
    cudaError_t e_ = (call);                                                              \
    if (e_ != cudaSuccess) {                                                              \
      snprintf(g_cuda_err, sizeof(g_cuda_err), "%s:%d %s: %s", __FILE__, __LINE__, #call, \
               cudaGetErrorString(e_));                                                   \
      return ZFAC_E_CUDA;                                                                 \
    }                                                                                     \
  } while (0)

struct zfac_ctx {
  int64_t n, np;
  int mode;
  int batch = 1;   // zfac_create_batched: independent problems refined by one launch sequence (tcgen05 modes)
  int dev = 0;     // device the context was created on; every entry point checks that it is current
  Options opt;     // zfac_set_option
  char* ws;
  size_t ws_bytes;
  Layout L;
  int launches;
  int sm_count;
  int order;       // m of Eq. 13 (zfac_set_order): 2 (default), 3, 4
  UmmaPlan umma;   // tensor maps + launch geometry for the tcgen05 modes
  F64Plan f64p;    // tensor maps of the FP64 buffers (ZFAC_MODE_F64)
  MixPlan mix;     // FP64-master modes (ZFAC_MODE_F64_MIXED, ZFAC_MODE_F64_I8)
  cudaStream_t side = nullptr;                 // zfac_refine_host: stream of the chunked upload and the early download (lazy)
  cudaEvent_t ev_a5 = nullptr, ev_copy = nullptr;
  static constexpr int UP_CHUNKS = 8;            // zfac_refine_host: S is uploaded in at most this many row chunks
  cudaEvent_t ev_begin = nullptr, ev_up[1 + UP_CHUNKS] = {};
  Prof prof;
};

static bool valid_mode(int m) {
  return m == ZFAC_MODE_SPLIT16 || m == ZFAC_MODE_TF32 || m == ZFAC_MODE_F64 || m == ZFAC_MODE_HH16 ||
         m == ZFAC_MODE_F64_MIXED || m == ZFAC_MODE_F64_I8;
}
static bool mode_is_umma(int m) { return m == ZFAC_MODE_SPLIT16 || m == ZFAC_MODE_TF32 || m == ZFAC_MODE_HH16; }
// The context is bound to the device that was current at zfac_create (workspace, tensor maps, lazily created streams).
static bool on_own_device(const zfac_ctx* c) {
  int dev = -1;
  return cudaGetDevice(&dev) == cudaSuccess && dev == c->dev;
}
// precision rank of a mode for Alg. 3 ("enhanced precision"): one 11-bit pass < FP32-class split < FP64
static int mode_rank(int m) { return mode_is_f64_elt(m) ? 2 : (m == ZFAC_MODE_SPLIT16 ? 1 : 0); }

extern "C" {

size_t zfac_workspace_bytes(int64_t n, zfac_mode mode) {
  if (n <= 0 || n > (1 << 20) || !valid_mode(mode) || (mode == ZFAC_MODE_F64_I8 && n > 32768)) return 0;
  return make_layout(n, mode).total;
}

size_t zfac_workspace_bytes_batched(int64_t n, zfac_mode mode, int batch) {
  if (n <= 0 || n > (1 << 20) || !mode_is_umma(mode) || batch < 1 || batch > 4096) return 0;
  if ((int64_t)batch * padded_n(n, mode) > (int64_t)1 << 24) return 0;        // stacked rows must stay 32-bit TMA coordinates
  return make_layout(n, mode, batch).total;
}

int64_t zfac_padded_n(int64_t n, zfac_mode mode) {
  if (n <= 0 || !valid_mode(mode)) return 0;
  return padded_n(n, mode);
}

const char* zfac_status_string(zfac_status s) {
  switch (s) {
    case ZFAC_OK: return "ZFAC_OK";
    case ZFAC_E_INVALID: return "ZFAC_E_INVALID: invalid argument";
    case ZFAC_E_UNSUPPORTED: return "ZFAC_E_UNSUPPORTED: device is not sm_100 (no fallback path)";
    case ZFAC_E_WORKSPACE: return "ZFAC_E_WORKSPACE: workspace null, misaligned or too small";
    case ZFAC_E_CUDA: return "ZFAC_E_CUDA: CUDA call failed";
  }
  return "unknown zfac_status";
}

const char* zfac_last_cuda_error(void) { return g_cuda_err; }

static zfac_status create_impl(zfac_ctx** out, int64_t n, zfac_mode mode, int batch, void* d_workspace, size_t bytes) {
  if (!out) return ZFAC_E_INVALID;
  *out = nullptr;
  if (n <= 0 || n > (1 << 20) || !valid_mode(mode)) return ZFAC_E_INVALID;
  if (mode == ZFAC_MODE_F64_I8 && n > 32768) return ZFAC_E_INVALID;      // INT32 accumulation: 8 slice pairs x 2^12 x K < 2^31
  if (batch < 1 || batch > 4096 || (batch > 1 && !mode_is_umma(mode))) return ZFAC_E_INVALID;
  if ((int64_t)batch * padded_n(n, mode) > (int64_t)1 << 24) return ZFAC_E_INVALID;
  Layout L = make_layout(n, mode, batch);
  if (!d_workspace || (reinterpret_cast<uintptr_t>(d_workspace) & 255u) || bytes < L.total) return ZFAC_E_WORKSPACE;
  int dev = 0, major = 0, sms = 0;
  ZF_CUDA(cudaGetDevice(&dev));
  ZF_CUDA(cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev));
  ZF_CUDA(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
  if (major != 10) return ZFAC_E_UNSUPPORTED;
  zfac_ctx* c = new (std::nothrow) zfac_ctx();
  if (!c) return ZFAC_E_INVALID;
  c->n = n; c->np = L.np; c->mode = mode; c->ws = static_cast<char*>(d_workspace); c->ws_bytes = bytes;
  c->L = L; c->launches = 0; c->sm_count = sms; c->order = 2; c->dev = dev; c->batch = batch;
  if (mode == ZFAC_MODE_F64) {
    cudaError_t e = f64_plan_create(&c->f64p, L, c->ws);
    if (e == cudaSuccess) e = f64_tma_prepare<EPI_A1>();
    if (e == cudaSuccess) e = f64_tma_prepare<EPI_A2>();
    if (e == cudaSuccess) e = f64_tma_prepare<EPI_X3>();
    if (e == cudaSuccess) e = f64_tma_prepare<EPI_A4>();
    if (e == cudaSuccess) e = f64_tma_prepare<EPI_A5>();
    if (e == cudaSuccess) e = f64_tma_prepare<EPI_P2>();
    if (e != cudaSuccess) {
      snprintf(g_cuda_err, sizeof(g_cuda_err), "f64_plan_create: %s", cudaGetErrorString(e));
      delete c;
      return ZFAC_E_CUDA;
    }
  } else if (mode_is_mix(mode)) {
    cudaError_t e = mix_plan_create(&c->mix, L, c->ws, sms, &c->opt);
    if (e != cudaSuccess) {
      snprintf(g_cuda_err, sizeof(g_cuda_err), "mix_plan_create: %s", cudaGetErrorString(e));
      delete c;
      return ZFAC_E_CUDA;
    }
  } else {
    cudaError_t e = umma_plan_create(&c->umma, L, c->ws, sms, &c->opt);
    if (e != cudaSuccess) {
      snprintf(g_cuda_err, sizeof(g_cuda_err), "umma_plan_create: %s", cudaGetErrorString(e));
      delete c;
      return ZFAC_E_CUDA;
    }
  }
  *out = c;
  return ZFAC_OK;
}

zfac_status zfac_create(zfac_ctx** out, int64_t n, zfac_mode mode, void* d_workspace, size_t bytes) {
  return create_impl(out, n, mode, 1, d_workspace, bytes);
}

zfac_status zfac_create_batched(zfac_ctx** out, int64_t n, zfac_mode mode, int batch, void* d_workspace, size_t bytes) {
  return create_impl(out, n, mode, batch, d_workspace, bytes);
}

int zfac_get_batch(const zfac_ctx* c) { return c ? c->batch : 0; }

zfac_status zfac_destroy(zfac_ctx* ctx) {
  if (ctx) {
    if (ctx->ev_a5) cudaEventDestroy(ctx->ev_a5);
    if (ctx->ev_copy) cudaEventDestroy(ctx->ev_copy);
    if (ctx->ev_begin) cudaEventDestroy(ctx->ev_begin);
    for (cudaEvent_t e : ctx->ev_up) if (e) cudaEventDestroy(e);
    if (ctx->side) cudaStreamDestroy(ctx->side);
    for (int i = 0; i < ctx->prof.cap; ++i) cudaEventDestroy(ctx->prof.ev[i]);
    delete[] ctx->prof.ev;
    delete[] ctx->prof.tags;
  }
  delete ctx;
  return ZFAC_OK;
}

zfac_status zfac_set_profile(zfac_ctx* c, int enable) {
  if (!c) return ZFAC_E_INVALID;
  if (enable && c->prof.cap == 0) {
    const int cap = 1024;
    if (!c->prof.ev) c->prof.ev = new (std::nothrow) cudaEvent_t[cap];
    if (!c->prof.tags) c->prof.tags = new (std::nothrow) int[cap];
    if (!c->prof.ev || !c->prof.tags) return ZFAC_E_INVALID;
    int made = 0;
    for (; made < cap; ++made)
      if (cudaEventCreate(&c->prof.ev[made]) != cudaSuccess) break;
    if (made < cap) {                       // all or nothing: zfac_destroy only sees prof.cap events
      for (int i = 0; i < made; ++i) cudaEventDestroy(c->prof.ev[i]);
      snprintf(g_cuda_err, sizeof(g_cuda_err), "zfac_set_profile: cudaEventCreate failed after %d events", made);
      (void)cudaGetLastError();
      return ZFAC_E_CUDA;
    }
    c->prof.cap = cap;
  }
  c->prof.on = enable != 0;
  c->prof.count = 0;
  return ZFAC_OK;
}

int zfac_get_profile(zfac_ctx* c, int* tags, float* ms, int cap) {
  if (!c || !tags || !ms || c->prof.count < 2) return 0;
  int k = 0;
  for (int i = 0; i + 1 < c->prof.count && k < cap; ++i) {
    float t = 0.f;
    if (cudaEventElapsedTime(&t, c->prof.ev[i], c->prof.ev[i + 1]) != cudaSuccess) return k;
    tags[k] = c->prof.tags[i];
    ms[k] = t;
    ++k;
  }
  return k;
}

int zfac_last_launch_count(const zfac_ctx* ctx) { return ctx ? ctx->launches : 0; }

zfac_status zfac_set_order(zfac_ctx* c, int m) {
  if (!c || m < 2 || m > 4 || (mode_is_mix(c->mode) && m != 2)) return ZFAC_E_INVALID;
  c->order = m;
  return ZFAC_OK;
}

int zfac_get_order(const zfac_ctx* c) { return c ? c->order : 0; }

zfac_status zfac_set_option(zfac_ctx* c, zfac_option key, double v) {
  if (!c || !(v == v)) return ZFAC_E_INVALID;
  const long iv = (long)(v < 0 ? v - 0.5 : v + 0.5);
  Options& o = c->opt;
  switch (key) {
    case ZFAC_OPT_CHUNK_KB: if (iv < 1 || iv > 1024) return ZFAC_E_INVALID; o.chunk_kb = (int)iv; return ZFAC_OK;
    case ZFAC_OPT_CHUNK0_KB: if (iv < 1 || iv > 1024) return ZFAC_E_INVALID; o.chunk0_kb = (int)iv; return ZFAC_OK;
    case ZFAC_OPT_HH_SQUARE: if (iv != 0 && iv != 1) return ZFAC_E_INVALID; o.hh_square = (int)iv; return ZFAC_OK;
    case ZFAC_OPT_HH_SQUARE_ERR: if (!(v >= 0.0)) return ZFAC_E_INVALID; o.hh_square_err = v; return ZFAC_OK;
    case ZFAC_OPT_PROMOTE_UPDATE: if (iv != 0 && iv != 1) return ZFAC_E_INVALID; o.promote_update = (int)iv; return ZFAC_OK;
    case ZFAC_OPT_BAND: if (iv < 1 || iv > 4096) return ZFAC_E_INVALID; o.band = (int)iv; return ZFAC_OK;
    case ZFAC_OPT_MAX_PAIRS: if (iv < 0 || iv > 65536) return ZFAC_E_INVALID; o.max_pairs = (int)iv; return ZFAC_OK;
    case ZFAC_OPT_HOST_OVERLAP: if (iv != 0 && iv != 1) return ZFAC_E_INVALID; o.host_overlap = (int)iv; return ZFAC_OK;
    case ZFAC_OPT_HOST_UPLOAD_OVERLAP: if (iv != 0 && iv != 1) return ZFAC_E_INVALID; o.host_upload_overlap = (int)iv; return ZFAC_OK;
    case ZFAC_OPT_HOST_A5_BANDS: if (iv < 1 || iv > 64) return ZFAC_E_INVALID; o.host_a5_bands = (int)iv; return ZFAC_OK;
    case ZFAC_OPT_I8_SLICES: if (iv < 2 || iv > I8_MAX_SLICES) return ZFAC_E_INVALID; o.i8_slices = (int)iv; return ZFAC_OK;
    case ZFAC_OPT_INPUT_F32:
      if ((iv != 0 && iv != 1) || (iv == 1 && !mode_is_f64_elt(c->mode))) return ZFAC_E_INVALID;
      o.input_f32 = (int)iv; return ZFAC_OK;
    case ZFAC_OPT_I8_NARROW:
      if (iv < -1 || iv > 1 || (iv == 1 && c->mode != ZFAC_MODE_F64_I8)) return ZFAC_E_INVALID;
      o.i8_narrow = (int)iv; return ZFAC_OK;
    case ZFAC_OPT_PDL: if (iv < -1 || iv > 2) return ZFAC_E_INVALID; o.pdl = (int)iv; return ZFAC_OK;
    case ZFAC_OPT_NARROW_TILES:
      if ((iv < -1 || iv > 1) || (iv == 1 && !mode_is_umma(c->mode))) return ZFAC_E_INVALID;
      o.narrow_tiles = (int)iv; return ZFAC_OK;
    case ZFAC_OPT_I8_CLUSTER:
      if ((iv != 0 && iv != 1) || (iv == 1 && c->mode != ZFAC_MODE_F64_I8)) return ZFAC_E_INVALID;
      o.i8_cluster = (int)iv; return ZFAC_OK;
    case ZFAC_OPT_FINAL_CHECK:
      if ((iv != 0 && iv != 1) || (iv == 0 && !mode_is_mix(c->mode))) return ZFAC_E_INVALID;
      o.final_check = (int)iv; return ZFAC_OK;
    case ZFAC_OPT_EXTRA_UPDATE:
      if ((iv != 0 && iv != 1) || (iv == 1 && !mode_is_mix(c->mode))) return ZFAC_E_INVALID;
      o.extra_update = (int)iv; return ZFAC_OK;
  }
  return ZFAC_E_INVALID;
}

zfac_status zfac_get_option(const zfac_ctx* c, zfac_option key, double* v) {
  if (!c || !v) return ZFAC_E_INVALID;
  const Options& o = c->opt;
  switch (key) {
    case ZFAC_OPT_CHUNK_KB: *v = o.chunk_kb; return ZFAC_OK;
    case ZFAC_OPT_CHUNK0_KB: *v = o.chunk0_kb; return ZFAC_OK;
    case ZFAC_OPT_HH_SQUARE: *v = o.hh_square; return ZFAC_OK;
    case ZFAC_OPT_HH_SQUARE_ERR: *v = o.hh_square_err; return ZFAC_OK;
    case ZFAC_OPT_PROMOTE_UPDATE: *v = o.promote_update; return ZFAC_OK;
    case ZFAC_OPT_BAND: *v = o.band; return ZFAC_OK;
    case ZFAC_OPT_MAX_PAIRS: *v = o.max_pairs; return ZFAC_OK;
    case ZFAC_OPT_HOST_OVERLAP: *v = o.host_overlap; return ZFAC_OK;
    case ZFAC_OPT_HOST_UPLOAD_OVERLAP: *v = o.host_upload_overlap; return ZFAC_OK;
    case ZFAC_OPT_HOST_A5_BANDS: *v = o.host_a5_bands; return ZFAC_OK;
    case ZFAC_OPT_I8_SLICES: *v = o.i8_slices; return ZFAC_OK;
    case ZFAC_OPT_INPUT_F32: *v = o.input_f32; return ZFAC_OK;
    case ZFAC_OPT_EXTRA_UPDATE: *v = o.extra_update; return ZFAC_OK;
    case ZFAC_OPT_FINAL_CHECK: *v = o.final_check; return ZFAC_OK;
    case ZFAC_OPT_I8_CLUSTER: *v = o.i8_cluster; return ZFAC_OK;
    case ZFAC_OPT_NARROW_TILES: *v = o.narrow_tiles; return ZFAC_OK;
    case ZFAC_OPT_PDL: *v = o.pdl; return ZFAC_OK;
    case ZFAC_OPT_I8_NARROW: *v = o.i8_narrow; return ZFAC_OK;
  }
  return ZFAC_E_INVALID;
}

// FP64 mode: the two halves of one iteration (see UmmaSeq in zfac_umma.cuh for the contract of n_stop / par).
struct F64Seq {
  zfac_ctx* c;
  F64TParams P{};
  int full = 0, tri = 0;
  double *W, *T, *R, *Q, *Z[2];

  F64Seq(zfac_ctx* c_, int max_iter, zfac_stop stop, double* d_err, unsigned long long cond) : c(c_) {
    const Layout& L = c->L;
    char* ws = c->ws;
    State* st = reinterpret_cast<State*>(ws + L.off_state);
    W = reinterpret_cast<double*>(ws + L.off_W);          // epilogue pointers; the operands go through tensor maps
    T = reinterpret_cast<double*>(ws + L.off_T);
    R = reinterpret_cast<double*>(ws + L.off_R);
    Q = reinterpret_cast<double*>(ws + L.off_Q);
    Z[0] = reinterpret_cast<double*>(ws + L.off_Z[0]); Z[1] = reinterpret_cast<double*>(ws + L.off_Z[1]);
    const int tiles = (int)(L.np / F64_BM);
    full = tiles * tiles; tri = tiles * (tiles + 1) / 2;
    F64Params& p = P.q;
    p.ld = (int)L.np; p.K = (int)L.np; p.tiles = tiles; p.st = st;
    p.stop.st = st; p.stop.partials = reinterpret_cast<double*>(ws + L.off_partials);
    p.stop.num_partials = tri; p.stop.d_err = d_err; p.stop.max_iter = max_iter; p.stop.stop = stop;
    p.stop.order = c->order; p.stop.cond = cond;
    p.pc = poly_coef(c->order);
  }
  void residual(int n_stop, int tagn, cudaStream_t s, Prof* prof) {
    const F64Plan& fp = c->f64p;
    F64Params& p = P.q;
    P.mapA = fp.mW; P.mapB = fp.mS; p.out0 = T; p.out1 = nullptr; p.in0 = nullptr;          // a1: T = W S^T
    if (prof) prof->mark(s, EPI_A1 + 16 * tagn);
    f64_tma_launch(EPI_A1, full, s, P);
    P.mapA = fp.mW; P.mapB = fp.mT; p.out0 = R; p.stop.n_iter = n_stop;                      // a2: R = I - W T^T
    if (prof) prof->mark(s, EPI_A2 + 16 * tagn);
    f64_tma_launch(EPI_A2, tri, s, P);
    c->launches += 2;
    if (p.stop.cond) graph_cond_kernel<<<1, 1, 0, s>>>(p.st, p.stop.cond);       // zfac_graph_*: loop condition
  }
  void update(int par, int n_stop, int tagn, cudaStream_t s, Prof* prof) {
    const F64Plan& fp = c->f64p;
    F64Params& p = P.q;
    p.stop.n_iter = n_stop;
    if (c->order > 2) {
      // order m > 2: P = R R -> T buffer, G = 3/8 I + 5/16 R (+ 35/128 P) -> the Z buffer a5 overwrites next
      P.mapA = fp.mR; P.mapB = fp.mR; p.in0 = R; p.out0 = T; p.out1 = Z[(par + 1) & 1];
      if (prof) prof->mark(s, EPI_P2 + 16 * tagn);
      f64_tma_launch(EPI_P2, tri, s, P);
      c->launches += 1;
      P.mapA = fp.mT; P.mapB = fp.mZ[(par + 1) & 1]; p.in0 = R; p.out0 = Q; p.out1 = nullptr;  // Q = 1/2 R + P G
    } else {
      P.mapA = fp.mR; P.mapB = fp.mR; p.in0 = R; p.out0 = Q;
    }
    if (prof) prof->mark(s, EPI_A4 + 16 * tagn);
    f64_tma_launch(EPI_A4, tri, s, P);
    P.mapA = fp.mZ[par]; P.mapB = fp.mQ; p.in0 = Z[par]; p.out0 = Z[(par + 1) & 1]; p.out1 = W;   // a5
    if (prof) prof->mark(s, EPI_A5 + 16 * tagn);
    f64_tma_launch(EPI_A5, full, s, P);
    c->launches += 2;
  }
};

// skip_last: Alg. 3 as printed ends after the update, without evaluating the residual of the result.
static zfac_status refine_f64(zfac_ctx* c, int max_iter, zfac_stop stop, double* d_err, cudaStream_t s,
                              bool skip_last = false, const IterHook* hook = nullptr) {
  F64Seq q(c, max_iter, stop, d_err, 0ull);
  for (int n = 0; n <= max_iter; ++n) {
    if (n == max_iter && skip_last) break;
    q.residual(n, n, s, &c->prof);
    if (n == max_iter) break;
    q.update(n & 1, n, n, s, &c->prof);
    if (hook && hook->after_a5) hook->after_a5(hook->self, n, s);
  }
  c->prof.mark(s, 0);
  ZF_CUDA(cudaGetLastError());
  return ZFAC_OK;
}

// FP64-master modes: same loop, MixSeq's halves.
static zfac_status refine_mix(zfac_ctx* c, int max_iter, zfac_stop stop, double* d_err, cudaStream_t s, bool skip_last,
                              const IterHook* hook) {
  MixSeq q(c->mix, max_iter, (int)stop, d_err, 0ull);
  for (int n = 0; n <= max_iter; ++n) {
    if (n == max_iter && skip_last) break;
    // zfac_refine_host, I8 engine: slicing of S + a1 of the first residual band by band, behind the row chunks of the upload
    const bool banded = (n == 0) && hook && hook->first_a1 && hook->first_a1(hook->self, &q, s);
    q.residual(n, n, s, &c->prof, banded);
    if (n == max_iter) break;
    if (hook && hook->before_update) hook->before_update(hook->self, n, s);
    q.update(n & 1, n, n, s, &c->prof);
    if (hook && hook->after_a5) hook->after_a5(hook->self, n, s);
  }
  c->prof.mark(s, 0);
  c->launches += q.nl;
  ZF_CUDA(cudaGetLastError());
  return ZFAC_OK;
}

// Step a0: copy S and Z0 (element type float if in_f32, else the mode's own) into the padded buffers.
// what: 1 = S only, 2 = Z0 (W, State reset) only, 3 = both; tile rows [ty0, ty0 + tyn) of CI_TR rows each (tyn = 0: all).
// First operation of every call: clears State::range (set by any CTA of the copy-in and of the a1 / a5 kernels when an fp16
// conversion clamps, published as ZFAC_R_RANGE).  A memset node, not a kernel; capturable.
static cudaError_t clear_range(zfac_ctx* c, cudaStream_t s) {
  State* st = reinterpret_cast<State*>(c->ws + c->L.off_state);
  if (c->batch > 1) return cudaMemsetAsync(st, 0, (size_t)c->batch * sizeof(State), s);   // every problem's State (the copy-in sets the rest)
  return cudaMemsetAsync(&st->range, 0, sizeof(int), s);
}

static void launch_copy_in(zfac_ctx* c, const void* d_S, int64_t lds, const void* d_Z0, int64_t ldz0, bool in_f32,
                           cudaStream_t s, int what = 3, int ty0 = 0, int tyn = 0, const State* prev = nullptr,
                           const void* d_Z0_alt = nullptr, int64_t stride_S = 0, int64_t stride_Z0 = 0) {
  const Layout& L = c->L;
  char* ws = c->ws;
  CopyInArgs ci{};
  ci.prev = prev; ci.Z0_alt = d_Z0_alt;
  ci.stride_S = stride_S; ci.stride_Z0 = stride_Z0; ci.rows = (int)L.rows;
  ci.S = d_S; ci.lds = lds; ci.Z0 = d_Z0; ci.ldz0 = ldz0; ci.n = (int)c->n; ci.np = (int)L.np;
  ci.st = reinterpret_cast<State*>(ws + L.off_state);
  ci.oS = ws + L.off_S; ci.oZ = ws + L.off_Z[0]; ci.oW = ws + L.off_W; ci.oZb = ws + L.off_Zb[0];
  ci.what = what; ci.ty0 = ty0;
  dim3 gi((unsigned)(L.np / CI_TC), (unsigned)(tyn > 0 ? tyn : L.np / CI_TR), (unsigned)c->batch), bi(256);
  if (mode_is_mix(c->mode)) {
    // FP64 master Z (+ S, W in FP64 for the DMMA engine), then the FP32 operand pair of Z; I8 engine: int8 slices of S and W
    const bool i8 = (c->mode == ZFAC_MODE_F64_I8);
    const bool with_S = (what & 1) != 0;                       // what = 2: the host entry point slices S band by band (a1_band)
    ci.what = i8 ? (2 | 4) : 3;
    if (in_f32) copy_in_kernel<ZFAC_MODE_F64, float><<<gi, bi, 0, s>>>(ci);
    else copy_in_kernel<ZFAC_MODE_F64, double><<<gi, bi, 0, s>>>(ci);
    const size_t np2 = (size_t)L.np * (size_t)L.np;
    z_planes_kernel<<<(unsigned)((np2 / 8 + 255) / 256), 256, 0, s>>>(reinterpret_cast<const double*>(ws + L.off_Z[0]),
                                                                    reinterpret_cast<__half*>(ws + L.off_Zb[0]), np2, ci.st);
    c->launches += 2;
    if (i8) {
      int* eS = reinterpret_cast<int*>(ws + L.off_exp);
      int8_t* S8 = reinterpret_cast<int8_t*>(ws + L.off_S8);
      if (!with_S) {}
      else if (in_f32) slice_rows_kernel<float><<<small_grid((size_t)L.np), 256, 0, s>>>(static_cast<const float*>(d_S), lds, (int)c->n, (int)L.np, c->opt.i8_slices, S8, eS, ci.st);
      else slice_rows_kernel<double><<<small_grid((size_t)L.np), 256, 0, s>>>(static_cast<const double*>(d_S), lds, (int)c->n, (int)L.np, c->opt.i8_slices, S8, eS, ci.st);
      MixSeq q(c->mix, 0, 0, nullptr, 0ull);
      q.w_slices(s);
      c->launches += 1 + q.nl;
    }
    return;
  }
  switch (c->mode) {
    case ZFAC_MODE_F64:
      if (in_f32) copy_in_kernel<ZFAC_MODE_F64, float><<<gi, bi, 0, s>>>(ci);
      else copy_in_kernel<ZFAC_MODE_F64, double><<<gi, bi, 0, s>>>(ci);
      break;
    case ZFAC_MODE_TF32: copy_in_kernel<ZFAC_MODE_TF32, float><<<gi, bi, 0, s>>>(ci); break;
    case ZFAC_MODE_HH16: copy_in_kernel<ZFAC_MODE_HH16, float><<<gi, bi, 0, s>>>(ci); break;
    default: copy_in_kernel<ZFAC_MODE_SPLIT16, float><<<gi, bi, 0, s>>>(ci); break;
  }
  c->launches += 1;
}

static void launch_copy_out(zfac_ctx* c, const void* b0, const void* b1, int parity, void* d_Z, int64_t ldz,
                            int* d_iters, int* d_flags, cudaStream_t s, int64_t stride_Z = 0) {
  const Layout& L = c->L;
  if (!d_Z) {                                     // publish iters / flags only (the result stays in the workspace)
    publish_kernel<<<1, 32, 0, s>>>(reinterpret_cast<const State*>(c->ws + L.off_state), d_iters, d_flags);
    c->launches += 1;
    return;
  }
  CopyOutArgs co{};
  co.Zbuf[0] = b0; co.Zbuf[1] = b1; co.parity = parity;
  co.Z = d_Z; co.ldz = ldz; co.n = (int)c->n; co.np = (int)L.np; co.stride_Z = stride_Z;
  co.st = reinterpret_cast<State*>(c->ws + L.off_state); co.d_iters = d_iters; co.d_flags = d_flags;
  const int elt = (int)L.elt;
  const bool vec16 = ((size_t)c->n * elt) % 16 == 0 && ((size_t)ldz * elt) % 16 == 0 && ((size_t)L.np * elt) % 16 == 0 &&
                     ((size_t)stride_Z * elt) % 16 == 0 &&
                     (reinterpret_cast<uintptr_t>(d_Z) & 15u) == 0 && (reinterpret_cast<uintptr_t>(b0) & 15u) == 0 &&
                     (reinterpret_cast<uintptr_t>(b1) & 15u) == 0;
  if (vec16) {
    dim3 gv((unsigned)(((size_t)c->n * elt / 16 + 255) / 256), (unsigned)((c->n + 7) / 8), (unsigned)c->batch);
    copy_out_vec16_kernel<<<gv, 256, 0, s>>>(co, elt);
  } else {
    dim3 go((unsigned)((c->n + 255) / 256), (unsigned)((c->n + 7) / 8), (unsigned)c->batch);
    if (mode_is_f64_elt(c->mode)) copy_out_kernel<double><<<go, 256, 0, s>>>(co);
    else copy_out_kernel<float><<<go, 256, 0, s>>>(co);
  }
  c->launches += 1;
}

// The iteration proper (everything between copy-in and copy-out) in the context's mode.
static zfac_status run_iterations(zfac_ctx* c, int max_iter, zfac_stop stop, double* d_err, cudaStream_t s, bool skip_last,
                                  const IterHook* hook) {
  if (c->mode == ZFAC_MODE_F64) return refine_f64(c, max_iter, stop, d_err, s, skip_last, hook);
  if (mode_is_mix(c->mode)) return refine_mix(c, max_iter, stop, d_err, s, skip_last, hook);
  int nl = 0;
  cudaError_t e = umma_refine(c->umma, max_iter, (int)stop, c->order, d_err, s, &nl, &c->prof, hook, skip_last);
  c->launches += nl;
  if (e != cudaSuccess) {
    snprintf(g_cuda_err, sizeof(g_cuda_err), "umma_refine: %s", cudaGetErrorString(e));
    return ZFAC_E_CUDA;
  }
  return ZFAC_OK;
}

// d_Z == nullptr (zfac_refine_refi's low-precision stage): the result stays in the workspace, iters / flags are published.
static zfac_status refine_impl(zfac_ctx* c, const void* d_S, int64_t lds, const void* d_Z0, int64_t ldz0, void* d_Z,
                               int64_t ldz, int max_iter, zfac_stop stop, int* d_iters, double* d_err, int* d_flags,
                               void* stream, const IterHook* hook, int copy_what = 3, int64_t stride_S = 0,
                               int64_t stride_Z0 = 0, int64_t stride_Z = 0) {
  if (!c || !d_S || !d_Z0 || !d_iters || !d_err || !d_flags) return ZFAC_E_INVALID;
  if (lds < c->n || ldz0 < c->n || (d_Z && ldz < c->n) || max_iter < 0) return ZFAC_E_INVALID;
  if (stop != ZFAC_STOP_PAPER && stop != ZFAC_STOP_FIXED) return ZFAC_E_INVALID;
  if (!on_own_device(c)) return ZFAC_E_INVALID;
  cudaStream_t s = static_cast<cudaStream_t>(stream);
  const Layout& L = c->L;
  char* ws = c->ws;
  c->launches = 0;
  c->prof.count = 0;

  ZF_CUDA(clear_range(c, s));
  launch_copy_in(c, d_S, lds, d_Z0, ldz0, c->opt.input_f32 != 0, s, copy_what, 0, 0, nullptr, nullptr, stride_S, stride_Z0);   // copy_what = 2: the hook's first_a1 brings S in
  zfac_status rs = run_iterations(c, max_iter, stop, d_err, s, false, hook);
  if (rs != ZFAC_OK) return rs;
  launch_copy_out(c, ws + L.off_Z[0], ws + L.off_Z[1], -1, d_Z, ldz, d_iters, d_flags, s, stride_Z);
  ZF_CUDA(cudaGetLastError());
  return ZFAC_OK;
}

zfac_status zfac_refine(zfac_ctx* c, const void* d_S, int64_t lds, const void* d_Z0, int64_t ldz0, void* d_Z,
                        int64_t ldz, int max_iter, zfac_stop stop, int* d_iters, double* d_err, int* d_flags,
                        void* stream) {
  if (!d_Z || (c && c->batch != 1)) return ZFAC_E_INVALID;
  return refine_impl(c, d_S, lds, d_Z0, ldz0, d_Z, ldz, max_iter, stop, d_iters, d_err, d_flags, stream, nullptr);
}

zfac_status zfac_refine_batched(zfac_ctx* c, const void* d_S, int64_t lds, int64_t stride_S, const void* d_Z0, int64_t ldz0,
                                int64_t stride_Z0, void* d_Z, int64_t ldz, int64_t stride_Z, int max_iter, zfac_stop stop,
                                int* d_iters, double* d_err, int* d_flags, void* stream) {
  if (!c || !d_Z || !mode_is_umma(c->mode)) return ZFAC_E_INVALID;
  if (c->batch > 1 && (stride_S < c->n * lds - (lds - c->n) || stride_Z0 < c->n * ldz0 - (ldz0 - c->n) ||
                       stride_Z < c->n * ldz - (ldz - c->n))) return ZFAC_E_INVALID;      // problems must not overlap
  return refine_impl(c, d_S, lds, d_Z0, ldz0, d_Z, ldz, max_iter, stop, d_iters, d_err, d_flags, stream, nullptr, 3,
                     stride_S, stride_Z0, stride_Z);
}

// zfac_refine_host, pinned h_Z: the download of Z starts right after the FIRST update (a5 of iteration 0 always runs when
// max_iter >= 1) on a side stream, with the copy engine, straight from the internal buffer.  If that update turns out
// to be the only one -- the warm-start case -- the download has overlapped the final residual evaluation (a1 + a2), which
// the caller would otherwise wait for before the download even starts.  If more updates ran it is superseded by the
// normal download at the end; PCIe and the copy engine were idle anyway, so it cost nothing on the critical path.
// (A device-predicated copy KERNEL after every a5 was built and measured first: SM stores into mapped host memory reach
// ~31 GB/s where the copy engine reaches 54; it made the call slower.  DESIGN.md §7.)
struct HostOverlap {
  zfac_ctx* c;
  void* h_Z;
  int64_t ldz;
  const void* dS = nullptr;   // staged S (dense n x n), arriving in `chunks` row chunks; chunk k is complete at ev_up[1 + k]
  int chunks = 0;
  int early = 1;              // early downloads: after the updates 0 .. early - 1 (2 in the FP64-master modes, whose
                              // iteration is longer than the download; 1 elsewhere)
};

// Upload overlap (tcgen05 modes, pinned h_S): Z0 is uploaded first, then S in row chunks of whole macro-tile rows on
// the side stream.  Rows [r0, r1) of S are all step a1 needs for the columns [r0, r1) of T = W S^T, so the main stream
// converts each chunk (copy-in, S only) and runs a1 on that band while the next chunk is still on the bus; only the
// last band's a1 is exposed.  Bands are disjoint sets of whole tiles: bit-identical to the one-launch a1.
static void host_chunk_rows(const zfac_ctx* c, int chunks, int k, int* mc0, int* mcn) {
  const int T = (int)(c->L.np / UM_MACRO);
  *mc0 = (int)((int64_t)T * k / chunks);
  *mcn = (int)((int64_t)T * (k + 1) / chunks) - *mc0;
}
static bool host_first_a1(void* self, void* seq, cudaStream_t s) {
  HostOverlap* h = static_cast<HostOverlap*>(self);
  if (h->chunks <= 0) return false;
  zfac_ctx* c = h->c;
  UmmaSeq* q = static_cast<UmmaSeq*>(seq);
  for (int k = 0; k < h->chunks; ++k) {
    int mc0, mcn; host_chunk_rows(c, h->chunks, k, &mc0, &mcn);
    cudaStreamWaitEvent(s, c->ev_up[1 + k], 0);
    launch_copy_in(c, h->dS, c->n, nullptr, c->n, false, s, 1, mc0 * (UM_MACRO / CI_TR), mcn * (UM_MACRO / CI_TR));
    q->a1(mc0, mcn, s);
  }
  return true;
}
// ... and the same for the I8 engine of ZFAC_MODE_F64_I8 (seq is a MixSeq): slices of the S rows of a chunk, then the tile
// columns of T = W S^T that need exactly those rows.
static bool host_first_a1_i8(void* self, void* seq, cudaStream_t s) {
  HostOverlap* h = static_cast<HostOverlap*>(self);
  if (h->chunks <= 0) return false;
  zfac_ctx* c = h->c;
  MixSeq* q = static_cast<MixSeq*>(seq);
  for (int k = 0; k < h->chunks; ++k) {
    int mc0, mcn; host_chunk_rows(c, h->chunks, k, &mc0, &mcn);
    cudaStreamWaitEvent(s, c->ev_up[1 + k], 0);
    q->a1_band(h->dS, c->n, c->opt.input_f32 != 0, (int)c->n, mc0, mcn, s);
  }
  return true;
}
static void host_before_update(void* self, int n, cudaStream_t s) {
  HostOverlap* h = static_cast<HostOverlap*>(self);
  if (n >= 1 && n <= h->early) cudaStreamWaitEvent(s, h->c->ev_copy, 0);      // the download of Z_n has left the master buffer
}
static void host_after_a5(void* self, int n, cudaStream_t s) {
  HostOverlap* h = static_cast<HostOverlap*>(self);
  if (n >= h->early) return;
  zfac_ctx* c = h->c;
  const Layout& L = c->L;
  // Z_{n+1}: buffer (n + 1) & 1 (F64 / TF32); the 16-bit and the FP64-master modes update one master in place
  const char* src = c->ws + L.off_Z[(n + 1) & 1];
  cudaEventRecord(c->ev_a5, s);
  cudaStreamWaitEvent(c->side, c->ev_a5, 0);
  cudaMemcpy2DAsync(h->h_Z, (size_t)h->ldz * L.elt, src, (size_t)L.np * L.elt, (size_t)c->n * L.elt, (size_t)c->n,
                    cudaMemcpyDeviceToHost, c->side);
  cudaEventRecord(c->ev_copy, c->side);
}

// ... and in the tensor-core modes the first a5 itself runs in two row bands: the rows of the first band go out while the
// second band is still being computed, which hides the part of the download that a1 + a2 (3.8 ms) did not cover (4.8 ms).
static void host_after_a5_band(void* self, int r0, int r1, bool last, cudaStream_t s) {
  HostOverlap* h = static_cast<HostOverlap*>(self);
  zfac_ctx* c = h->c;
  const Layout& L = c->L;
  const int64_t a = r0 < c->n ? r0 : c->n, b = r1 < c->n ? r1 : c->n;
  cudaEventRecord(c->ev_a5, s);
  cudaStreamWaitEvent(c->side, c->ev_a5, 0);
  if (b > a)
    cudaMemcpy2DAsync(static_cast<char*>(h->h_Z) + (size_t)a * h->ldz * L.elt, (size_t)h->ldz * L.elt,
                      c->ws + L.off_Z[1] + (size_t)a * L.np * L.elt, (size_t)L.np * L.elt, (size_t)c->n * L.elt,
                      (size_t)(b - a), cudaMemcpyDeviceToHost, c->side);
  if (last) cudaEventRecord(c->ev_copy, c->side);
}

// Alg. 3.  low_hook / low_copy_what: the host entry point's upload overlap for the low-precision stage; high_hook: its
// early download.  d_upd (may be null): int[2] = refinement updates performed, Err entries written in total.
static zfac_status refi_impl(zfac_ctx* low, zfac_ctx* high, const void* d_S, int64_t lds, const void* d_Z0, int64_t ldz0,
                             void* d_Z, int64_t ldz, int max_iter, int refi_steps, int final_check, int* d_iters,
                             double* d_err, int* d_flags, int* d_upd, cudaStream_t s, const IterHook* low_hook,
                             int low_copy_what, const IterHook* high_hook) {
  if (!low || !high || !d_S || !d_Z0 || !d_Z || !d_iters || !d_err || !d_flags) return ZFAC_E_INVALID;
  if (low->batch != 1 || high->batch != 1) return ZFAC_E_INVALID;
  if (mode_rank(high->mode) <= mode_rank(low->mode) || low->n != high->n || low->order != high->order) return ZFAC_E_INVALID;
  if (lds < low->n || ldz0 < low->n || ldz < low->n || max_iter < 0 || refi_steps < 1 || refi_steps > 4000)
    return ZFAC_E_INVALID;
  if (!on_own_device(low) || low->dev != high->dev) return ZFAC_E_INVALID;
  const Layout& LL = low->L;
  const Layout& L = high->L;
  // 1. Alg. 2 in low precision; the result stays in `low`'s workspace (FP32 master Z; TF32: the buffer of parity iters & 1)
  zfac_status rs = refine_impl(low, d_S, lds, d_Z0, ldz0, nullptr, 0, max_iter, ZFAC_STOP_PAPER, d_iters, d_err, d_flags, s,
                               low_hook, low_copy_what);
  if (rs != ZFAC_OK) return rs;
  // 2. Z = FP32[Z] or FP64[Z], S converted exactly; X recomputed; 3. refi_steps updates in `high`'s kernels
  high->launches = 0;
  high->prof.count = 0;
  const State* lst = reinterpret_cast<const State*>(low->ws + LL.off_state);
  ZF_CUDA(clear_range(high, s));
  launch_copy_in(high, d_S, lds, low->ws + LL.off_Z[0], LL.np, true, s, 3, 0, 0, lst, low->ws + LL.off_Z[1]);
  double* err_hi = reinterpret_cast<double*>(high->ws + L.off_stage_out);
  rs = run_iterations(high, refi_steps, ZFAC_STOP_FIXED, err_hi, s, final_check == 0, high_hook);
  if (rs != ZFAC_OK) return rs;
  launch_copy_out(high, high->ws + L.off_Z[0], high->ws + L.off_Z[1], -2, d_Z, ldz, nullptr, nullptr, s);
  refi_merge_kernel<<<1, 32, 0, s>>>(reinterpret_cast<const State*>(high->ws + L.off_state), err_hi, d_err, d_iters, d_flags, d_upd);
  high->launches += 1;
  low->launches += high->launches;
  ZF_CUDA(cudaGetLastError());
  return ZFAC_OK;
}

zfac_status zfac_refine_refi(zfac_ctx* low, zfac_ctx* high, const void* d_S, int64_t lds, const void* d_Z0,
                             int64_t ldz0, void* d_Z, int64_t ldz, int max_iter, int refi_steps, int final_check,
                             int* d_iters, double* d_err, int* d_flags, void* stream) {
  return refi_impl(low, high, d_S, lds, d_Z0, ldz0, d_Z, ldz, max_iter, refi_steps, final_check, d_iters, d_err, d_flags,
                   nullptr, static_cast<cudaStream_t>(stream), nullptr, 3, nullptr);
}

zfac_status zfac_congruence(zfac_ctx* c, const void* d_H, int64_t ldh, const void* d_Z, int64_t ldz, void* d_out,
                            int64_t ldo, void* stream) {
  if (!c || !d_H || !d_Z || !d_out) return ZFAC_E_INVALID;
  if (ldh < c->n || ldz < c->n || ldo < c->n || !on_own_device(c) || mode_is_mix(c->mode) || c->batch != 1) return ZFAC_E_INVALID;
  cudaStream_t s = static_cast<cudaStream_t>(stream);
  const Layout& L = c->L;
  char* ws = c->ws;
  c->launches = 0;
  c->prof.count = 0;
  ZF_CUDA(clear_range(c, s));
  launch_copy_in(c, d_H, ldh, d_Z, ldz, false, s);        // H takes the place of S; W = Z^T
  if (c->mode == ZFAC_MODE_F64) {
    double* T = reinterpret_cast<double*>(ws + L.off_T);
    const int tiles = (int)(L.np / F64_BM);
    F64TParams P{};
    F64Params& p = P.q;
    p.ld = (int)L.np; p.K = (int)L.np; p.tiles = tiles; p.st = reinterpret_cast<State*>(ws + L.off_state);
    P.mapA = c->f64p.mW; P.mapB = c->f64p.mS; p.out0 = T;                                   // H sits in the S buffer
    f64_tma_launch(EPI_A1, tiles * tiles, s, P);
    P.mapA = c->f64p.mW; P.mapB = c->f64p.mT; p.out0 = reinterpret_cast<double*>(ws + L.off_R);
    f64_tma_launch(EPI_X3, tiles * (tiles + 1) / 2, s, P);
    c->launches += 2;
  } else {
    int nl = 0;
    cudaError_t e = umma_congruence(c->umma, s, &nl);
    c->launches += nl;
    if (e != cudaSuccess) {
      snprintf(g_cuda_err, sizeof(g_cuda_err), "umma_congruence: %s", cudaGetErrorString(e));
      return ZFAC_E_CUDA;
    }
  }
  launch_copy_out(c, ws + L.off_R, ws + L.off_R, 0, d_out, ldo, nullptr, nullptr, s);
  ZF_CUDA(cudaGetLastError());
  return ZFAC_OK;
}

// Upload of S and Z0 into the staging area for the host entry points.  With pinned inputs in a tensor-core mode
// (see host_first_a1) Z0 goes first and S follows in row chunks on the side stream; *chunks > 0 says so.
static zfac_status host_upload(zfac_ctx* c, const void* h_S, int64_t lds, const void* h_Z0, int64_t ldz0, cudaStream_t s,
                               int* chunks_out) {
  const Layout& L = c->L;
  char* dS = c->ws + L.off_stage_S;
  char* dZ = c->ws + L.off_stage_Z;
  const size_t elt = (mode_is_f64_elt(c->mode) && c->opt.input_f32) ? 4 : L.elt;      // element size of the INPUTS
  const size_t row = (size_t)c->n * elt;
  int chunks = 0;
  if ((mode_is_umma(c->mode) || c->mode == ZFAC_MODE_F64_I8) && L.np / UM_MACRO >= 4 && c->opt.host_upload_overlap) {
    cudaPointerAttributes pS{}, pZ{};
    if (cudaPointerGetAttributes(&pS, h_S) == cudaSuccess && pS.type == cudaMemoryTypeHost &&
        cudaPointerGetAttributes(&pZ, h_Z0) == cudaSuccess && pZ.type == cudaMemoryTypeHost) {
      const int T = (int)(L.np / UM_MACRO);
      chunks = T < zfac_ctx::UP_CHUNKS ? T : zfac_ctx::UP_CHUNKS;
    }
    (void)cudaGetLastError();
  }
  if (chunks > 0) {
    if (!c->side) ZF_CUDA(cudaStreamCreateWithFlags(&c->side, cudaStreamNonBlocking));
    if (!c->ev_begin) {
      ZF_CUDA(cudaEventCreateWithFlags(&c->ev_begin, cudaEventDisableTiming));
      for (cudaEvent_t& e : c->ev_up) ZF_CUDA(cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
    }
    ZF_CUDA(cudaEventRecord(c->ev_begin, s));                    // the uploads keep their place in the caller's stream order
    ZF_CUDA(cudaStreamWaitEvent(c->side, c->ev_begin, 0));
    ZF_CUDA(cudaMemcpy2DAsync(dZ, row, h_Z0, (size_t)ldz0 * elt, row, (size_t)c->n, cudaMemcpyHostToDevice, c->side));
    ZF_CUDA(cudaEventRecord(c->ev_up[0], c->side));
    for (int k = 0; k < chunks; ++k) {
      int mc0, mcn; host_chunk_rows(c, chunks, k, &mc0, &mcn);
      const int64_t r0 = (int64_t)mc0 * UM_MACRO < c->n ? (int64_t)mc0 * UM_MACRO : c->n;
      const int64_t r1 = (int64_t)(mc0 + mcn) * UM_MACRO < c->n ? (int64_t)(mc0 + mcn) * UM_MACRO : c->n;
      if (r1 > r0)
        ZF_CUDA(cudaMemcpy2DAsync(dS + (size_t)r0 * row, row, static_cast<const char*>(h_S) + (size_t)r0 * lds * elt,
                                  (size_t)lds * elt, row, (size_t)(r1 - r0), cudaMemcpyHostToDevice, c->side));
      ZF_CUDA(cudaEventRecord(c->ev_up[1 + k], c->side));
    }
    ZF_CUDA(cudaStreamWaitEvent(s, c->ev_up[0], 0));            // Z0 is there: copy-in of Z0 (W, operand planes) can start
  } else {
    ZF_CUDA(cudaMemcpy2DAsync(dS, row, h_S, (size_t)lds * elt, row, (size_t)c->n, cudaMemcpyHostToDevice, s));
    ZF_CUDA(cudaMemcpy2DAsync(dZ, row, h_Z0, (size_t)ldz0 * elt, row, (size_t)c->n, cudaMemcpyHostToDevice, s));
  }
  *chunks_out = chunks;
  return ZFAC_OK;
}

static bool host_pinned(const void* p) {
  cudaPointerAttributes pa{};
  const bool pinned = cudaPointerGetAttributes(&pa, p) == cudaSuccess && pa.type == cudaMemoryTypeHost;
  (void)cudaGetLastError();
  return pinned;
}

static zfac_status host_side_objects(zfac_ctx* c) {
  if (!c->side) ZF_CUDA(cudaStreamCreateWithFlags(&c->side, cudaStreamNonBlocking));
  if (!c->ev_a5) ZF_CUDA(cudaEventCreateWithFlags(&c->ev_a5, cudaEventDisableTiming));
  if (!c->ev_copy) ZF_CUDA(cudaEventCreateWithFlags(&c->ev_copy, cudaEventDisableTiming));
  return ZFAC_OK;
}

zfac_status zfac_refine_host(zfac_ctx* c, const void* h_S, int64_t lds, const void* h_Z0, int64_t ldz0, void* h_Z,
                             int64_t ldz, int max_iter, zfac_stop stop, int* h_iters, double* h_err, int* h_flags,
                             void* stream) {
  if (!c || !h_S || !h_Z0 || !h_Z || !h_iters || !h_err || !h_flags) return ZFAC_E_INVALID;
  if (lds < c->n || ldz0 < c->n || ldz < c->n || max_iter < 0 || max_iter > 4095) return ZFAC_E_INVALID;
  if (!on_own_device(c) || c->batch != 1) return ZFAC_E_INVALID;
  cudaStream_t s = static_cast<cudaStream_t>(stream);
  const Layout& L = c->L;
  char* dS = c->ws + L.off_stage_S;
  char* dZ = c->ws + L.off_stage_Z;
  double* dErr = reinterpret_cast<double*>(c->ws + L.off_stage_out);
  int* dInts = reinterpret_cast<int*>(c->ws + L.off_stage_out + 4096 * sizeof(double));
  const size_t row = (size_t)c->n * L.elt;
  int chunks = 0;
  zfac_status rs = host_upload(c, h_S, lds, h_Z0, ldz0, s, &chunks);
  if (rs != ZFAC_OK) return rs;
  // overlapped download: needs a pinned (device-visible) h_Z (an async copy to pageable memory is staged and may
  // block) and at least one possible update
  const bool z_dev = max_iter >= 1 && c->opt.host_overlap && host_pinned(h_Z);
  HostOverlap ho{c, h_Z, ldz};
  ho.dS = dS; ho.chunks = chunks;
  IterHook hook{z_dev ? host_after_a5 : nullptr, &ho};
  if (chunks > 0) hook.first_a1 = mode_is_mix(c->mode) ? host_first_a1_i8 : host_first_a1;
  if (z_dev && mode_is_mix(c->mode) && max_iter >= 2) {
    // one update of these modes (a full FP64-level residual) outlasts the download: the results of the first TWO updates
    // are sent early, each behind its update; the master is updated in place, so update n + 1 waits for the download of Z_n
    ho.early = 2;
    hook.before_update = host_before_update;
  }
  if (z_dev && mode_is_umma(c->mode) && L.np / UM_MACRO >= 4) {
    hook.a5_bands = c->opt.host_a5_bands;
    if (hook.a5_bands > (int)(L.np / UM_MACRO)) hook.a5_bands = (int)(L.np / UM_MACRO);
    hook.after_a5_band = host_after_a5_band;
  }
  if (z_dev && (rs = host_side_objects(c)) != ZFAC_OK) return rs;
  rs = refine_impl(c, dS, c->n, dZ, c->n, dZ, c->n, max_iter, stop, dInts, dErr, dInts + 1, s,
                   (z_dev || chunks > 0) ? &hook : nullptr, chunks > 0 ? 2 : 3);
  if (rs != ZFAC_OK) return rs;
  if (z_dev) ZF_CUDA(cudaStreamWaitEvent(s, c->ev_copy, 0));   // the early download is complete (and can no longer land late)
  else ZF_CUDA(cudaMemcpy2DAsync(h_Z, (size_t)ldz * L.elt, dZ, row, row, (size_t)c->n, cudaMemcpyDeviceToHost, s));
  int ints[2] = {0, 0};
  ZF_CUDA(cudaMemcpyAsync(ints, dInts, 2 * sizeof(int), cudaMemcpyDeviceToHost, s));
  ZF_CUDA(cudaStreamSynchronize(s));
  *h_iters = ints[0]; *h_flags = ints[1];
  // the early downloads hold Z_1 (.. Z_early): final if no later update ran.  In-place masters stay what they were once the
  // iteration has stopped, so the last early download is also right when FEWER updates ran (it re-sent the final Z).
  const bool early_final = (ho.early == 1) ? (ints[0] == 1) : (ints[0] >= 1 && ints[0] <= ho.early);
  if (z_dev && !early_final)
    ZF_CUDA(cudaMemcpy2DAsync(h_Z, (size_t)ldz * L.elt, dZ, row, row, (size_t)c->n, cudaMemcpyDeviceToHost, s));
  ZF_CUDA(cudaMemcpyAsync(h_err, dErr, (size_t)(ints[0] + 1) * sizeof(double), cudaMemcpyDeviceToHost, s));
  ZF_CUDA(cudaStreamSynchronize(s));
  return ZFAC_OK;
}

// zfac_refine_refi_host: the download of Z starts right after the LAST refinement update (straight from the internal
// buffer, on `high`'s side stream), so it overlaps the final check; if the refinement stage did not perform all its
// updates (non-finite residual) the normal download at the end supersedes it.
struct RefiDownload {
  zfac_ctx* high;
  void* h_Z;
  int64_t ldz;
  int last;            // index of the last refinement update (refi_steps - 1)
};
static void refi_after_a5(void* self, int n, cudaStream_t s) {
  RefiDownload* r = static_cast<RefiDownload*>(self);
  if (n != r->last) return;
  zfac_ctx* c = r->high;
  const Layout& L = c->L;
  // Z after update n sits in buffer (n + 1) & 1 (F64 / TF32); the 16-bit modes update one FP32 master in place
  const char* src = c->ws + L.off_Z[mode_is_h16(c->mode) ? 0 : ((n + 1) & 1)];
  cudaEventRecord(c->ev_a5, s);
  cudaStreamWaitEvent(c->side, c->ev_a5, 0);
  cudaMemcpy2DAsync(r->h_Z, (size_t)r->ldz * L.elt, src, (size_t)L.np * L.elt, (size_t)c->n * L.elt, (size_t)c->n,
                    cudaMemcpyDeviceToHost, c->side);
  cudaEventRecord(c->ev_copy, c->side);
}

zfac_status zfac_refine_refi_host(zfac_ctx* low, zfac_ctx* high, const void* h_S, int64_t lds, const void* h_Z0,
                                  int64_t ldz0, void* h_Z, int64_t ldz, int max_iter, int refi_steps, int final_check,
                                  int* h_iters, double* h_err, int* h_flags, void* stream) {
  if (!low || !high || !h_S || !h_Z0 || !h_Z || !h_iters || !h_err || !h_flags) return ZFAC_E_INVALID;
  if (!mode_is_umma(low->mode) || low->n != high->n) return ZFAC_E_INVALID;
  if (lds < low->n || ldz0 < low->n || ldz < low->n || max_iter < 0 || refi_steps < 1 || max_iter + refi_steps + 2 > 4096)
    return ZFAC_E_INVALID;
  if (!on_own_device(low) || low->dev != high->dev) return ZFAC_E_INVALID;
  cudaStream_t s = static_cast<cudaStream_t>(stream);
  const Layout& LL = low->L;
  const Layout& L = high->L;
  char* dS = low->ws + LL.off_stage_S;
  char* dZ0 = low->ws + LL.off_stage_Z;
  char* dZ = high->ws + L.off_stage_Z;                         // n x n of high's element type
  double* dErr = reinterpret_cast<double*>(low->ws + LL.off_stage_out);
  int* dInts = reinterpret_cast<int*>(low->ws + LL.off_stage_out + 4096 * sizeof(double));
  const size_t row = (size_t)high->n * L.elt;
  int chunks = 0;
  zfac_status rs = host_upload(low, h_S, lds, h_Z0, ldz0, s, &chunks);
  if (rs != ZFAC_OK) return rs;
  HostOverlap ho{low, nullptr, 0};
  ho.dS = dS; ho.chunks = chunks;
  IterHook low_hook{nullptr, &ho};
  low_hook.first_a1 = mode_is_mix(low->mode) ? host_first_a1_i8 : host_first_a1;
  const bool z_dev = high->opt.host_overlap && host_pinned(h_Z);
  RefiDownload rd{high, h_Z, ldz, refi_steps - 1};
  IterHook high_hook{refi_after_a5, &rd};
  if (z_dev && (rs = host_side_objects(high)) != ZFAC_OK) return rs;
  rs = refi_impl(low, high, dS, low->n, dZ0, low->n, dZ, high->n, max_iter, refi_steps, final_check, dInts, dErr, dInts + 1,
                 dInts + 2, s, chunks > 0 ? &low_hook : nullptr, chunks > 0 ? 2 : 3, z_dev ? &high_hook : nullptr);
  if (rs != ZFAC_OK) return rs;
  if (z_dev) ZF_CUDA(cudaStreamWaitEvent(s, high->ev_copy, 0));
  else ZF_CUDA(cudaMemcpy2DAsync(h_Z, (size_t)ldz * L.elt, dZ, row, row, (size_t)high->n, cudaMemcpyDeviceToHost, s));
  int ints[4] = {0, 0, 0, 0};
  ZF_CUDA(cudaMemcpyAsync(ints, dInts, 4 * sizeof(int), cudaMemcpyDeviceToHost, s));
  ZF_CUDA(cudaStreamSynchronize(s));
  *h_iters = ints[0]; *h_flags = ints[1];
  if (z_dev && ints[2] != refi_steps)      // the refinement stage stopped early: the early download is not the result
    ZF_CUDA(cudaMemcpy2DAsync(h_Z, (size_t)ldz * L.elt, dZ, row, row, (size_t)high->n, cudaMemcpyDeviceToHost, s));
  ZF_CUDA(cudaMemcpyAsync(h_err, dErr, (size_t)ints[3] * sizeof(double), cudaMemcpyDeviceToHost, s));
  ZF_CUDA(cudaStreamSynchronize(s));
  return ZFAC_OK;
}

// ------------------------------------------------------------------ zfac_graph: the call as a CUDA graph with a WHILE node
struct zfac_graph {
  zfac_ctx* c = nullptr;
  cudaGraph_t g = nullptr;
  cudaGraphExec_t ex = nullptr;
};

extern "C++" {
template <class Seq>
static void enqueue_loop_body(Seq& q, cudaStream_t s) {
  // two iterations (the Z operand buffers alternate with the parity of n); indices come from the device (n_stop = -1).
  // If the stop test fires in the first half, the second half's kernels return at once (State::done).
  q.update(0, -1, 0, s, nullptr); q.residual(-1, 0, s, nullptr);
  q.update(1, -1, 0, s, nullptr); q.residual(-1, 0, s, nullptr);
}
}

zfac_status zfac_graph_create(zfac_ctx* c, const void* d_S, int64_t lds, const void* d_Z0, int64_t ldz0, void* d_Z,
                              int64_t ldz, int max_iter, zfac_stop stop, int* d_iters, double* d_err, int* d_flags,
                              zfac_graph** out) {
  if (!out) return ZFAC_E_INVALID;
  *out = nullptr;
  if (!c || !d_S || !d_Z0 || !d_Z || !d_iters || !d_err || !d_flags) return ZFAC_E_INVALID;
  if (lds < c->n || ldz0 < c->n || ldz < c->n || max_iter < 0) return ZFAC_E_INVALID;
  if (stop != ZFAC_STOP_PAPER && stop != ZFAC_STOP_FIXED) return ZFAC_E_INVALID;
  if (!on_own_device(c) || c->batch != 1) return ZFAC_E_INVALID;
  const Layout& L = c->L;
  char* ws = c->ws;
  zfac_graph* zg = new (std::nothrow) zfac_graph();
  if (!zg) return ZFAC_E_INVALID;
  zg->c = c;
  cudaStream_t cs = nullptr, bs = nullptr;
  zfac_status rs = ZFAC_OK;
  bool capturing = false;
  auto fail = [&](const char* what, cudaError_t e) {
    snprintf(g_cuda_err, sizeof(g_cuda_err), "zfac_graph_create: %s: %s", what, cudaGetErrorString(e));
    rs = ZFAC_E_CUDA;
  };
  cudaError_t e;
  do {
    if ((e = cudaStreamCreateWithFlags(&cs, cudaStreamNonBlocking)) != cudaSuccess) { fail("stream", e); break; }
    if ((e = cudaStreamCreateWithFlags(&bs, cudaStreamNonBlocking)) != cudaSuccess) { fail("stream", e); break; }
    if ((e = cudaStreamBeginCapture(cs, cudaStreamCaptureModeRelaxed)) != cudaSuccess) { fail("begin capture", e); break; }
    capturing = true;
    cudaStreamCaptureStatus cst; unsigned long long cid = 0; cudaGraph_t g = nullptr;
    const cudaGraphNode_t* deps = nullptr; size_t ndeps = 0;
    if ((e = cudaStreamGetCaptureInfo_v2(cs, &cst, &cid, &g, &deps, &ndeps)) != cudaSuccess) { fail("capture info", e); break; }
    cudaGraphConditionalHandle h;
    if ((e = cudaGraphConditionalHandleCreate(&h, g, 1, cudaGraphCondAssignDefault)) != cudaSuccess) { fail("conditional handle", e); break; }
    // root: copy-in, first residual (its stop test already sets the condition: max_iter = 0 or a non-finite Err[0] skip the loop)
    const int saved_launches = c->launches;
    if ((e = clear_range(c, cs)) != cudaSuccess) { fail("memset", e); break; }
    launch_copy_in(c, d_S, lds, d_Z0, ldz0, c->opt.input_f32 != 0, cs);
    cudaGraphNodeParams np = {};
    np.type = cudaGraphNodeTypeConditional;
    np.conditional.handle = h; np.conditional.type = cudaGraphCondTypeWhile; np.conditional.size = 1;
    cudaGraphNode_t wnode = nullptr;
    auto splice_loop = [&]() -> bool {
      if ((e = cudaStreamGetCaptureInfo_v2(cs, &cst, &cid, &g, &deps, &ndeps)) != cudaSuccess) { fail("capture info", e); return false; }
      if ((e = cudaGraphAddNode(&wnode, g, deps, ndeps, &np)) != cudaSuccess) { fail("while node", e); return false; }
      if ((e = cudaStreamUpdateCaptureDependencies(cs, &wnode, 1, cudaStreamSetCaptureDependencies)) != cudaSuccess) { fail("capture deps", e); return false; }
      if ((e = cudaStreamBeginCaptureToGraph(bs, np.conditional.phGraph_out[0], nullptr, nullptr, 0, cudaStreamCaptureModeRelaxed)) != cudaSuccess) { fail("body capture", e); return false; }
      return true;
    };
    bool ok = true;
    if (c->mode == ZFAC_MODE_F64) {
      F64Seq q(c, max_iter, stop, d_err, (unsigned long long)h);
      q.residual(0, 0, cs, nullptr);
      if ((ok = splice_loop())) enqueue_loop_body(q, bs);
    } else if (mode_is_mix(c->mode)) {
      MixSeq q(c->mix, max_iter, (int)stop, d_err, (unsigned long long)h);
      q.residual(0, 0, cs, nullptr);
      if ((ok = splice_loop())) enqueue_loop_body(q, bs);
    } else {
      UmmaSeq q(c->umma, max_iter, (int)stop, c->order, d_err, (unsigned long long)h);
      q.residual(0, 0, cs, nullptr);
      if ((ok = splice_loop())) enqueue_loop_body(q, bs);
    }
    if (!ok) break;
    if ((e = cudaStreamEndCapture(bs, nullptr)) != cudaSuccess) { fail("end body capture", e); break; }
    launch_copy_out(c, ws + L.off_Z[0], ws + L.off_Z[1], -1, d_Z, ldz, d_iters, d_flags, cs);
    c->launches = saved_launches;
    capturing = false;
    if ((e = cudaStreamEndCapture(cs, &zg->g)) != cudaSuccess) { fail("end capture", e); break; }
    if ((e = cudaGetLastError()) != cudaSuccess) { fail("launch during capture", e); break; }
    if ((e = cudaGraphInstantiate(&zg->ex, zg->g, 0)) != cudaSuccess) { fail("instantiate", e); break; }
  } while (false);
  if (capturing) { cudaGraph_t junk = nullptr; cudaStreamEndCapture(cs, &junk); if (junk) cudaGraphDestroy(junk); }
  if (cs) cudaStreamDestroy(cs);
  if (bs) cudaStreamDestroy(bs);
  if (rs != ZFAC_OK) { zfac_graph_destroy(zg); return rs; }
  *out = zg;
  return ZFAC_OK;
}

zfac_status zfac_graph_launch(zfac_graph* zg, void* stream) {
  if (!zg || !zg->ex || !on_own_device(zg->c)) return ZFAC_E_INVALID;
  ZF_CUDA(cudaGraphLaunch(zg->ex, static_cast<cudaStream_t>(stream)));
  return ZFAC_OK;
}

zfac_status zfac_graph_destroy(zfac_graph* zg) {
  if (zg) {
    if (zg->ex) cudaGraphExecDestroy(zg->ex);
    if (zg->g) cudaGraphDestroy(zg->g);
    delete zg;
  }
  return ZFAC_OK;
}

zfac_status zfac_peek(zfac_ctx* c, zfac_buf which, void* d_out, int64_t ld, void* stream) {
  if (!c || !d_out || ld < c->n || !on_own_device(c) || c->batch != 1) return ZFAC_E_INVALID;
  cudaStream_t s = static_cast<cudaStream_t>(stream);
  const Layout& L = c->L;
  char* ws = c->ws;
  const int n = (int)c->n, np = (int)L.np;
  dim3 g((unsigned)((n + 255) / 256), (unsigned)n);
  // the current Z buffer index is only known on the device; read it (peek is a test hook, it may sync)
  State hst{};
  ZF_CUDA(cudaStreamSynchronize(s));
  ZF_CUDA(cudaMemcpy(&hst, ws + L.off_state, sizeof(State), cudaMemcpyDeviceToHost));
  if (mode_is_mix(c->mode)) {
    switch (which) {
      case ZFAC_BUF_T: peek_kernel<double, 0><<<g, 256, 0, s>>>(ws + L.off_T, d_out, ld, n, np); break;
      case ZFAC_BUF_R:
        if (c->mode == ZFAC_MODE_F64_MIXED) peek_kernel<double, 0><<<g, 256, 0, s>>>(ws + L.off_R, d_out, ld, n, np);
        else peek_kernel<double, 4><<<g, 256, 0, s>>>(ws + L.off_R, d_out, ld, n, np);
        break;
      case ZFAC_BUF_Z: peek_kernel<double, 0><<<g, 256, 0, s>>>(ws + L.off_Z[0], d_out, ld, n, np); break;
      default: return ZFAC_E_INVALID;               // Q exists only as the scaled operand pair in these modes
    }
  } else if (c->mode == ZFAC_MODE_F64 || c->mode == ZFAC_MODE_TF32) {
    size_t off;
    switch (which) {
      case ZFAC_BUF_T: off = L.off_T; break;
      case ZFAC_BUF_R: off = L.off_R; break;
      case ZFAC_BUF_Q: off = L.off_Q; break;
      case ZFAC_BUF_Z: off = L.off_Z[hst.iters & 1]; break;
      default: return ZFAC_E_INVALID;
    }
    if (c->mode == ZFAC_MODE_F64) peek_kernel<double, 0><<<g, 256, 0, s>>>(ws + off, d_out, ld, n, np);
    else peek_kernel<float, 0><<<g, 256, 0, s>>>(ws + off, d_out, ld, n, np);
  } else if (c->mode == ZFAC_MODE_SPLIT16) {
    switch (which) {
      case ZFAC_BUF_T: peek_kernel<float, 1><<<g, 256, 0, s>>>(ws + L.off_T, d_out, ld, n, np); break;
      case ZFAC_BUF_R: peek_kernel<float, 3><<<g, 256, 0, s>>>(ws + L.off_R, d_out, ld, n, np); break;
      case ZFAC_BUF_Q: peek_kernel<float, 1><<<g, 256, 0, s>>>(ws + L.off_Qb, d_out, ld, n, np); break;
      case ZFAC_BUF_Z: peek_kernel<float, 0><<<g, 256, 0, s>>>(ws + L.off_Z[0], d_out, ld, n, np); break;
      default: return ZFAC_E_INVALID;
    }
  } else {  // HH16
    switch (which) {
      case ZFAC_BUF_T: peek_kernel<float, 2><<<g, 256, 0, s>>>(ws + L.off_T, d_out, ld, n, np); break;
      case ZFAC_BUF_R: peek_kernel<float, 3><<<g, 256, 0, s>>>(ws + L.off_R, d_out, ld, n, np); break;
      case ZFAC_BUF_Q: peek_kernel<float, 2><<<g, 256, 0, s>>>(ws + L.off_Qb, d_out, ld, n, np); break;
      case ZFAC_BUF_Z: peek_kernel<float, 0><<<g, 256, 0, s>>>(ws + L.off_Z[0], d_out, ld, n, np); break;
      default: return ZFAC_E_INVALID;
    }
  }
  ZF_CUDA(cudaGetLastError());
  return ZFAC_OK;
}

}  // extern "C"
