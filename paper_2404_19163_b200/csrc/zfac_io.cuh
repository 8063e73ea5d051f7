// Workspace layout and the O(N^2) copy-in / copy-out kernels (steps a0 and a6).
//
// Padding (Sec. V.E, :398-400): the library works on internal buffers whose
// dimension Np is a multiple of the tile size.  The extra rows/columns of S and Z are
// filled with an IDENTITY block, S_pad = diag(S, I), Z_pad = diag(Z, I), which makes the
// padded problem exact: R is zero there, no epilogue needs a predicate and ||R||_F is
// unchanged (zero padding would add Np - N to ||R||_F^2).
//
// Operand splitting (Eq. 17-18, :143-149): A ~ A_hi + A_lo.
//   fp16 pair (SPLIT16, all four GEMMs):  hi = FP16[a],  lo' = FP16[(a - FP32[hi]) * 2^11]
//       -- the low half is stored SCALED by 2^11 so that it does not fall into the FP16
//       subnormal range; the products that contain one lo' are accumulated separately and
//       weighted by 2^-11 in the epilogue.  Error <= 2^-22 |a| as in PAPER.md:169.
//   R and Q shrink towards 0 as the iteration converges and their hi half underflows gradually
//   (fp16 subnormal spacing 2^-24); the remainder, scaled by 2^11, is then below 2^-14 and is
//   stored to 11 bits, so the ABSOLUTE error of the pair is <= 2^-36 -- far below the FP32
//   rounding of the sum Z + Z Q that these operands feed.
#pragma once
#include <cuda_fp16.h>
#include "zfac_common.cuh"

namespace zfac {

constexpr float LO_SCALE = 2048.0f;           // 2^11
constexpr float LO_UNSCALE = 1.0f / 2048.0f;  // 2^-11

__device__ __forceinline__ __half f2h_sat(float a) {
  unsigned short r;
  asm("cvt.rn.satfinite.f16.f32 %0, %1;" : "=h"(r) : "f"(a));
  return __ushort_as_half(r);
}
__device__ __forceinline__ void split_f16(float a, __half& hi, __half& lo) {
  hi = f2h_sat(a);
  lo = f2h_sat((a - __half2float(hi)) * LO_SCALE);
}

// Round-to-nearest FP32 -> TF32 (low 13 mantissa bits cleared).  The tensor core TRUNCATES FP32
// operands to TF32, which biases every product towards zero; operand buffers that are only ever
// read by the tensor core are therefore stored pre-rounded.
__device__ __forceinline__ float round_tf32(float a) {
  uint32_t r;
  asm("cvt.rna.tf32.f32 %0, %1;" : "=r"(r) : "f"(a));
  return __uint_as_float(r);
}

inline int64_t round_up(int64_t a, int64_t b) { return (a + b - 1) / b * b; }

struct Layout {
  int64_t n = 0, np = 0;
  int batch = 1;        // tcgen05 modes: `batch` independent problems stacked along the rows of every buffer
  int64_t rows = 0;     // = batch * np: rows of one plane of one buffer (problem b occupies rows [b np, (b + 1) np))
  int mode = 0;
  size_t elt = 0;  // user element size
  size_t off_state = 0, off_dbg = 0, off_partials = 0, num_partials = 0;
  size_t off_stage_S = 0, off_stage_Z = 0, off_stage_out = 0;
  // F64 / TF32: one buffer each of the mode's element type; Z double-buffered
  size_t off_S = 0, off_W = 0, off_T = 0, off_R = 0, off_Q = 0, off_Z[2] = {0, 0};
  // SPLIT16 / HH16: S, W, T, Rb, Qb, Zb[2] are fp16 [planes][Np][Np] (planes = 2: hi, lo'; HH16: 1);
  // R and the master Z (= off_Z[0]) are fp32
  size_t off_Rb = 0, off_Qb = 0, off_Zb[2] = {0, 0};
  // FP64-master modes (zfac_mix.cuh): S, W, T (F64_MIXED), Z in FP64; R in FP64 (F64_MIXED) or FP32 (F64_I8) at off_R;
  // R~ (FP32) at off_R32; fp16 pairs Rb, Qb, Zb[2]; F64_I8: int8 slices of S, W, T, row exponents, partial-sum scratch
  size_t off_R32 = 0, off_S8 = 0, off_W8 = 0, off_T8 = 0, off_exp = 0, off_scratch = 0;
  size_t total = 0;
};

inline int64_t padded_n(int64_t n, int mode) { return round_up(n, mode == ZFAC_MODE_F64 ? 128 : 256); }
inline bool mode_is_h16(int mode) { return mode == ZFAC_MODE_SPLIT16 || mode == ZFAC_MODE_HH16; }
inline bool mode_is_mix(int mode) { return mode == ZFAC_MODE_F64_MIXED || mode == ZFAC_MODE_F64_I8; }
inline bool mode_is_f64_elt(int mode) { return mode == ZFAC_MODE_F64 || mode_is_mix(mode); }

inline Layout make_layout(int64_t n, int mode, int batch = 1) {
  Layout L;
  L.n = n; L.mode = mode; L.np = padded_n(n, mode); L.batch = batch; L.rows = (int64_t)batch * L.np;
  L.elt = mode_is_f64_elt(mode) ? 8 : 4;
  const size_t np2 = (size_t)L.rows * (size_t)L.np, n2 = (size_t)n * (size_t)n;      // np2: one plane of one (stacked) buffer
  size_t off = 0;
  auto take = [&](size_t bytes) { size_t o = off; off += (bytes + 1023) / 1024 * 1024; return o; };
  L.off_state = take(sizeof(State));                             // State of problem 0 (the only one unless batched) ...
  L.off_dbg = take(8 * 148 * 8 * sizeof(unsigned long long));   // -DZFAC_TIMING counters (at a fixed offset: 1024)
  if (batch > 1) L.off_state = take((size_t)batch * sizeof(State));       // ... batched: an array of States
  // tcgen05 kernels: 16 partial sums per a2 tile (256 x 256), per problem; FP64 / INT8 kernels: one per CTA (<= (np / 128)^2)
  L.num_partials = (size_t)batch * 16 * (size_t)(L.np / 128) * (size_t)(L.np / 128);
  L.off_partials = take(L.num_partials * sizeof(double));
  L.off_stage_S = take(batch > 1 ? 0 : n2 * L.elt);              // staging of the host entry points (not batched)
  L.off_stage_Z = take(batch > 1 ? 0 : n2 * L.elt);
  L.off_stage_out = take((size_t)4096 * sizeof(double) + 64);
  if (mode_is_mix(mode)) {
    const size_t hb = np2 * 4;                                        // fp16 pair planes
    L.off_T = take(np2 * 8);
    L.off_Z[0] = take(np2 * 8); L.off_Z[1] = L.off_Z[0];              // FP64 master, updated in place
    L.off_R32 = take(np2 * 4); L.off_Rb = take(hb); L.off_Qb = take(hb);
    L.off_Zb[0] = take(hb); L.off_Zb[1] = take(hb);
    if (mode == ZFAC_MODE_F64_MIXED) {
      L.off_S = take(np2 * 8); L.off_W = take(np2 * 8); L.off_R = take(np2 * 8);
    } else {
      L.off_R = take(np2 * 4);
      L.off_S8 = take(np2 * 8); L.off_W8 = take(np2 * 8); L.off_T8 = take(np2 * 8);      // 8 slices of Np^2 int8 each
      L.off_exp = take(3 * (size_t)L.np * sizeof(int));
      L.off_scratch = take((size_t)192 * 128 * 256 * sizeof(double));
    }
  } else if (mode_is_h16(mode)) {
    const size_t hb = np2 * (mode == ZFAC_MODE_SPLIT16 ? 4 : 2);     // fp16 planes: (hi, lo') or hi only
    L.off_S = take(hb); L.off_W = take(hb); L.off_T = take(hb);
    L.off_R = take(np2 * 4); L.off_Rb = take(hb); L.off_Qb = take(hb);
    L.off_Z[0] = take(np2 * 4); L.off_Z[1] = L.off_Z[0];
    L.off_Zb[0] = take(hb); L.off_Zb[1] = take(hb);
  } else {
    L.off_S = take(np2 * L.elt); L.off_W = take(np2 * L.elt); L.off_T = take(np2 * L.elt);
    L.off_R = take(np2 * L.elt); L.off_Q = take(np2 * L.elt);
    L.off_Z[0] = take(np2 * L.elt); L.off_Z[1] = take(np2 * L.elt);
  }
  L.total = off;
  return L;
}

// ------------------------------------------------------------------ copy-in (step a0)
struct CopyInArgs {
  const void* S; int64_t lds;
  const void* Z0; int64_t ldz0;
  int n, np;
  State* st;
  void* oS;            // F64: double[Np][Np]; TF32: float; SPLIT16: half[2][Np][Np]
  void* oZ;            // F64/TF32: Z[0];  SPLIT16: float Z32
  void* oW;            // F64/TF32: W;     SPLIT16: half[2][Np][Np]
  void* oZb;           // SPLIT16 / HH16: half[planes][Np][Np] (Zb[0])
  int64_t stride_S, stride_Z0;   // batched: elements between consecutive problems in the caller's S and Z0 (grid.z = problem)
  int rows;            // batch * np
  int what;            // bit 0: S, bit 1: Z0 (and W, State reset); 0 is read as 3 (both); bit 2: no W (F64_I8: sliced later)
  int ty0;             // first tile row of this launch (grid.y counts from it): row chunks of S for zfac_refine_host
  // zfac_refine_refi: Z0 is the result of a low-precision run, taken straight from that context's workspace.
  const State* prev;   // State of the low-precision context (null: none)
  const void* Z0_alt;  // Z0 is this buffer instead when prev->iters is odd (modes whose Z buffers alternate); may be null
};

// One tile of CI_TR = 32 rows x CI_TC = 64 columns per CTA (256 threads).  Phase 1: coalesced loads of the S and Z0
// tiles (identity padding beyond n; the user's leading dimension need not be aligned) into shared memory.  Phase 2: every
// thread takes 8 consecutive columns of one row and writes S, Z (and the 16-bit operand planes) with 16-byte stores.
// Phase 3: every thread takes 8 consecutive ROWS of one column of the Z tile -- a conflict-free column read of the
// 65-wide tile -- and writes 8 consecutive elements of a row of W = Z^T, again as 16-byte stores.  (The first version
// wrote one element per thread, 2-byte stores to the fp16 planes: transaction-bound, i.e. as slow as the SM clock,
// which is 1.2-1.3 GHz inside a sustained run.)
// Tin = element type of the user's S and Z0: the mode's own type, or float for the FP64 refinement step of Alg. 3
// ("Z = FP64[Z]"; S is promoted exactly).
constexpr int CI_TR = 32, CI_TC = 64, CI_PITCH = CI_TC + 1;

template <int MODE>
__device__ __forceinline__ void ci_store8(void* buf, size_t np2, size_t o, const float (&v)[8], bool operand, State* st) {
  // 8 consecutive FP32 values -> the mode's representation at element offset o (o is a multiple of 8).
  // operand = true: a buffer only the tensor core reads (S, W; Zb): fp16 plane(s) / TF32-rounded FP32.
  if (MODE == ZFAC_MODE_SPLIT16 || MODE == ZFAC_MODE_HH16) {
    float mx = 0.0f;
#pragma unroll
    for (int j = 0; j < 8; ++j) mx = fmaxf(mx, fabsf(v[j]));
    if (mx >= H16_MAX) atomicOr(&st->range, 1);          // cvt.rn.satfinite is about to clamp: ZFAC_R_RANGE
    uint32_t hi[4], lo[4];
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      if (MODE == ZFAC_MODE_SPLIT16) {
        __half h0, l0, h1, l1;
        split_f16(v[2 * j], h0, l0); split_f16(v[2 * j + 1], h1, l1);
        hi[j] = (uint32_t)__half_as_ushort(h0) | ((uint32_t)__half_as_ushort(h1) << 16);
        lo[j] = (uint32_t)__half_as_ushort(l0) | ((uint32_t)__half_as_ushort(l1) << 16);
      } else {
        hi[j] = (uint32_t)__half_as_ushort(f2h_sat(v[2 * j])) | ((uint32_t)__half_as_ushort(f2h_sat(v[2 * j + 1])) << 16);
      }
    }
    __half* b = static_cast<__half*>(buf);
    *reinterpret_cast<uint4*>(b + o) = make_uint4(hi[0], hi[1], hi[2], hi[3]);
    if (MODE == ZFAC_MODE_SPLIT16) *reinterpret_cast<uint4*>(b + np2 + o) = make_uint4(lo[0], lo[1], lo[2], lo[3]);
  } else {                                   // TF32 operand buffers: FP32, rounded to nearest TF32
    float* b = static_cast<float*>(buf);
    (void)operand;
    *reinterpret_cast<float4*>(b + o) = make_float4(round_tf32(v[0]), round_tf32(v[1]), round_tf32(v[2]), round_tf32(v[3]));
    *reinterpret_cast<float4*>(b + o + 4) = make_float4(round_tf32(v[4]), round_tf32(v[5]), round_tf32(v[6]), round_tf32(v[7]));
  }
}

template <int MODE, typename Tin>
__global__ void __launch_bounds__(256) copy_in_kernel(const CopyInArgs a) {
  using Tw = typename std::conditional<MODE == ZFAC_MODE_F64, double, float>::type;   // internal element type
  __shared__ Tin sS[CI_TR * CI_PITCH];
  __shared__ Tin sZ[CI_TR * CI_PITCH];
  const int t = threadIdx.x;
  const bool doS = (a.what == 0) || (a.what & 1), doZ = (a.what == 0) || (a.what & 2), doW = doZ && !(a.what & 4);
  const int pb = blockIdx.z;                                   // problem of a batch (0 otherwise)
  State* st = a.st + pb;
  if (doZ && blockIdx.x == 0 && blockIdx.y == 0 && t == 0) {
    // refinement stage of Alg. 3 behind a low-precision run that ended non-finite: nothing to refine -- every later
    // kernel of this context exits at once (done = 1) and no Err entry exists (iters = -1)
    const bool dead = a.prev && (a.prev->flags & ZFAC_R_NONFINITE);
    st->done = dead ? 1 : 0; st->iters = dead ? -1 : 0; st->flags = 0; st->last = 0;
    st->arrive[0] = st->arrive[1] = st->arrive[2] = st->arrive[3] = 0u;
  }
  const int c0 = blockIdx.x * CI_TC, r0 = ((int)blockIdx.y + a.ty0) * CI_TR;
  const size_t np = (size_t)a.np, np2 = (size_t)(a.rows > 0 ? a.rows : a.np) * np;     // plane stride of the stacked buffers
  const size_t rb = (size_t)pb * np;                           // first row of this problem in the stacked buffers
  const Tin* S = static_cast<const Tin*>(a.S) + (size_t)pb * a.stride_S;
  const Tin* Z0 = static_cast<const Tin*>((a.prev && a.Z0_alt && (a.prev->iters & 1)) ? a.Z0_alt : a.Z0) + (size_t)pb * a.stride_Z0;
  // ---- phase 1: coalesced loads (64 consecutive columns per row), identity padding
#pragma unroll
  for (int i = 0; i < CI_TR * CI_TC / 256; ++i) {
    const int idx = t + 256 * i, lr = idx / CI_TC, lc = idx - lr * CI_TC;
    const int r = r0 + lr, c = c0 + lc;
    const bool in = (r < a.n && c < a.n);
    const Tin ident = (r == c) ? Tin(1) : Tin(0);
    if (doS) sS[lr * CI_PITCH + lc] = in ? S[(size_t)r * a.lds + c] : ident;
    if (doZ) sZ[lr * CI_PITCH + lc] = in ? Z0[(size_t)r * a.ldz0 + c] : ident;
  }
  __syncthreads();
  // ---- phase 2: S and Z, 8 consecutive columns of one row per thread
  {
    const int lr = t >> 3, lc = (t & 7) * 8;
    const size_t o = (rb + (size_t)(r0 + lr)) * np + (size_t)(c0 + lc);
    if (MODE == ZFAC_MODE_F64) {
      Tw* oS = static_cast<Tw*>(a.oS); Tw* oZ = static_cast<Tw*>(a.oZ);
#pragma unroll
      for (int j = 0; j < 8; j += 2) {
        if (doS) *reinterpret_cast<double2*>(reinterpret_cast<double*>(oS) + o + j) =
            make_double2((double)sS[lr * CI_PITCH + lc + j], (double)sS[lr * CI_PITCH + lc + j + 1]);
        if (doZ) *reinterpret_cast<double2*>(reinterpret_cast<double*>(oZ) + o + j) =
            make_double2((double)sZ[lr * CI_PITCH + lc + j], (double)sZ[lr * CI_PITCH + lc + j + 1]);
      }
    } else {
      if (doS) {
        float vs[8];
#pragma unroll
        for (int j = 0; j < 8; ++j) vs[j] = (float)sS[lr * CI_PITCH + lc + j];
        ci_store8<MODE>(a.oS, np2, o, vs, true, st);
      }
      if (doZ) {
        float vz[8];
#pragma unroll
        for (int j = 0; j < 8; ++j) vz[j] = (float)sZ[lr * CI_PITCH + lc + j];
        float* z32 = static_cast<float*>(a.oZ);                     // FP32 Z (the master copy in the 16-bit modes): not rounded
        *reinterpret_cast<float4*>(z32 + o) = make_float4(vz[0], vz[1], vz[2], vz[3]);
        *reinterpret_cast<float4*>(z32 + o + 4) = make_float4(vz[4], vz[5], vz[6], vz[7]);
        if (MODE == ZFAC_MODE_SPLIT16 || MODE == ZFAC_MODE_HH16) ci_store8<MODE>(a.oZb, np2, o, vz, true, st);
      }
    }
  }
  // ---- phase 3: W = Z^T, 8 consecutive rows of one column of the tile per thread -> 8 consecutive elements of a row of W
  if (doW) {
    const int wr = t >> 2, wc = (t & 3) * 8;                        // W tile: CI_TC rows x CI_TR columns
    const size_t o = (rb + (size_t)(c0 + wr)) * np + (size_t)(r0 + wc);
    if (MODE == ZFAC_MODE_F64) {
      double* oW = static_cast<double*>(a.oW);
#pragma unroll
      for (int j = 0; j < 8; j += 2)
        *reinterpret_cast<double2*>(oW + o + j) =
            make_double2((double)sZ[(wc + j) * CI_PITCH + wr], (double)sZ[(wc + j + 1) * CI_PITCH + wr]);
    } else {
      float vw[8];
#pragma unroll
      for (int j = 0; j < 8; ++j) vw[j] = (float)sZ[(wc + j) * CI_PITCH + wr];
      ci_store8<MODE>(a.oW, np2, o, vw, true, st);
    }
  }
}

// ------------------------------------------------------------------ copy-out (step a6)
struct CopyOutArgs {
  const void* Zbuf[2];   // internal Z buffers (selected by the parity of the update count; equal in the 16-bit modes)
  void* Z; int64_t ldz;
  int n, np;
  const State* st;
  int* d_iters; int* d_flags;   // may be null (refinement step, congruence)
  int parity;                   // >= 0: Zbuf[parity];  -1: Zbuf[st->iters & 1] (plain call);  -2: Zbuf[updates_done & 1]
  int64_t stride_Z;             // batched (grid.z = problem): elements between consecutive problems in the caller's Z
};
// Number of Z updates a call has performed.  State::iters is the index of the last Err written; it equals the update
// count unless the call ended with an update whose residual was not evaluated (Alg. 3 as printed: done stays 0).
__device__ __forceinline__ int updates_done(const State* st) {
  const int it = st->iters;
  return st->done ? (it > 0 ? it : 0) : it + 1;
}
__device__ __forceinline__ int published_flags(const State* st) { return st->flags | ((st->range & 1) ? ZFAC_R_RANGE : 0); }
// `plain`: the ordinary call (every residual evaluated): the update count is State::iters itself.
__device__ __forceinline__ void publish_and_select(const CopyOutArgs& a, bool first, const void*& src) {
  const int pb = blockIdx.z;
  const State* st = a.st + pb;
  const int iters = st->iters;
  if (a.d_iters && first) { a.d_iters[pb] = iters; a.d_flags[pb] = published_flags(st); }
  src = a.Zbuf[a.parity >= 0 ? a.parity : (a.parity == -1 ? (iters & 1) : (updates_done(st) & 1))];
}

template <typename T>
__global__ void __launch_bounds__(256) copy_out_kernel(const CopyOutArgs a) {
  const void* sel;
  publish_and_select(a, blockIdx.x == 0 && blockIdx.y == 0 && threadIdx.x == 0, sel);
  const T* src = static_cast<const T*>(sel) + (size_t)blockIdx.z * a.np * a.np;
  T* dst = static_cast<T*>(a.Z) + (size_t)blockIdx.z * a.stride_Z;
  const int c = blockIdx.x * 256 + threadIdx.x;
  const int r0 = blockIdx.y * 8;
  if (c >= a.n) return;
#pragma unroll
  for (int i = 0; i < 8; ++i) {
    const int r = r0 + i;
    if (r < a.n) dst[(size_t)r * a.ldz + c] = src[(size_t)r * a.np + c];
  }
}

// 16-byte-vector variant for the aligned case (N * sizeof(T), both pitches and both base pointers multiples of
// 16 bytes): one uint4 per thread and row, 8 rows per block row.
__global__ void __launch_bounds__(256) copy_out_vec16_kernel(const CopyOutArgs a, int elt) {
  const void* sel;
  publish_and_select(a, blockIdx.x == 0 && blockIdx.y == 0 && threadIdx.x == 0, sel);
  const char* src = static_cast<const char*>(sel) + (size_t)blockIdx.z * a.np * a.np * elt;
  char* dst = static_cast<char*>(a.Z) + (size_t)blockIdx.z * a.stride_Z * elt;
  const size_t row_bytes = (size_t)a.n * elt, spitch = (size_t)a.np * elt, dpitch = (size_t)a.ldz * elt;
  const size_t cb = ((size_t)blockIdx.x * 256 + threadIdx.x) * 16;
  if (cb >= row_bytes) return;
  const int r0 = blockIdx.y * 8;
  uint4 v[8];
#pragma unroll
  for (int i = 0; i < 8; ++i)
    if (r0 + i < a.n) v[i] = *reinterpret_cast<const uint4*>(src + (size_t)(r0 + i) * spitch + cb);
#pragma unroll
  for (int i = 0; i < 8; ++i)
    if (r0 + i < a.n) *reinterpret_cast<uint4*>(dst + (size_t)(r0 + i) * dpitch + cb) = v[i];
}

// ------------------------------------------------------------------ Alg. 3 bookkeeping
// Publishes iters / flags of a call without copying Z out (the low-precision stage of zfac_refine_refi, whose result
// the refinement stage takes straight from the workspace).
__global__ void publish_kernel(const State* st, int* d_iters, int* d_flags) {
  if (blockIdx.x == 0 && threadIdx.x == 0) { *d_iters = st->iters; *d_flags = published_flags(st); }
}
// Appends the history of the refinement stage (State `hi`, Err entries in err_hi) to the low-precision one and
// publishes iters / flags.  Everything is taken from the refinement stage's State, so a stage that stopped early
// (non-finite residual) or never ran (non-finite low-precision result) is reported as it happened.
__global__ void refi_merge_kernel(const State* hi, const double* err_hi, double* d_err, int* d_iters, int* d_flags, int* d_upd) {
  if (blockIdx.x == 0 && threadIdx.x == 0) {
    const int k = *d_iters;                       // stop index of the low-precision run
    const int entries = hi->iters + 1, upd = updates_done(hi);
    for (int i = 0; i < entries; ++i) d_err[k + 1 + i] = err_hi[i];
    *d_iters = k + upd;
    if (d_upd) { d_upd[0] = upd; d_upd[1] = k + 1 + entries; }     // refinement updates performed; Err entries in total
    *d_flags |= (upd > 0 ? ZFAC_R_REFINED : 0) | (hi->flags & ZFAC_R_NONFINITE) | ((hi->range & 1) ? ZFAC_R_RANGE : 0);
  }
}

// ------------------------------------------------------------------ peek (tests)
// kind 0: plain T buffer; 1: fp16 pair hi + lo' 2^-11; 2: fp16 (hi only); 3: plain T buffer of a SYMMETRIC matrix of
// which only the upper triangle of tiles is stored (the FP32 R of the 16-bit modes): element (r, c), r > c, is (c, r);
// 4: plain FLOAT buffer read into T (the FP32 R of ZFAC_MODE_F64_I8)
template <typename T, int KIND>
__global__ void __launch_bounds__(256) peek_kernel(const void* src, void* out, int64_t ld, int n, int np) {
  const int c = blockIdx.x * 256 + threadIdx.x, r = blockIdx.y;
  if (c >= n || r >= n) return;
  const size_t o = (KIND == 3 && r > c) ? (size_t)c * np + r : (size_t)r * np + c, np2 = (size_t)np * np;
  T v;
  if (KIND == 0 || KIND == 3) v = static_cast<const T*>(src)[o];
  else if (KIND == 4) v = (T) static_cast<const float*>(src)[o];
  else if (KIND == 1) {
    const __half* h = static_cast<const __half*>(src);
    v = (T)(__half2float(h[o]) + __half2float(h[np2 + o]) * LO_UNSCALE);
  } else {
    v = (T)__half2float(static_cast<const __half*>(src)[o]);
  }
  static_cast<T*>(out)[(size_t)r * ld + c] = v;
}

}  // namespace zfac
