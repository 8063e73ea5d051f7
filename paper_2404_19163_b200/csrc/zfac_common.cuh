// Shared device-side pieces of libzfac: the per-call state block, the on-device
// stopping test (step a3) and small helpers.  No oracle code is shared with this file.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include "../../include/zfac.h"

namespace zfac {

// Lives at the start of the workspace.  Reset by the first copy-in kernel of every call.
struct alignas(64) State {
  int done;                  // set by step a3; every later kernel of the call exits at once
  int iters;                 // number of Z updates performed so far (= index of the last Err)
  int flags;                 // ZFAC_R_* bits
  int last;                  // ZFAC_OPT_FINAL_CHECK = 0: the update now in flight is the last one, its residual is not evaluated
  unsigned int arrive[4];    // last-CTA counters (one per use site), self-resetting
  int range;                 // bit 0: a value of magnitude >= 65504 was clamped on its way into an fp16 operand (16-bit modes;
                             // bit 1: F64_I8 met a non-finite operand while slicing -> the next Err is NaN);
                             // cleared by a memset node BEFORE the copy-in of a call (every CTA of the copy-in may set it),
                             // merged into the published flags as ZFAC_R_RANGE
  // FP64-master modes (zfac_mix.cuh): R is handed to the FP32-class update GEMMs scaled by a power of two, R~ = rscale R,
  // chosen from ||R||_F by r_split_kernel so that the fp16 operand pairs of R~ and Q~ neither overflow nor underflow
  float rscale, rinv;        // rscale and 1 / rscale
  int pad1;
};
constexpr float H16_MAX = 65504.0f;   // largest finite fp16: cvt.rn.satfinite clamps beyond it

// Per-context tuning / behaviour options (zfac_set_option; defaults here).  Host-side state only.
struct Options {
  int chunk_kb = 1;          // SPLIT16 a1/a2: k-blocks (64 products each) per promoted-accumulation chunk
  int chunk0_kb = 1;         // ... of the first chunk of a tile
  int band = 8;              // full GEMMs: tile columns per rasterisation band
  int hh_square = 1;         // SPLIT16 a4/p2: (h)(h) pass only for updates taken from Err[n] <= hh_square_err
  double hh_square_err = 0.1;
  int promote_update = 0;    // SPLIT16: promoted accumulation in p2/a4/a5 too
  int max_pairs = 0;         // run on at most this many CTA pairs (0: all that are co-resident)
  int host_overlap = 1;      // zfac_refine_host: early download of Z after the first update
  int host_upload_overlap = 1;   // zfac_refine_host: chunked upload of S overlapped with copy-in + a1
  int host_a5_bands = 2;     // zfac_refine_host: row bands of the first a5 (each band downloaded as it completes)
  int narrow_tiles = -1;     // tcgen05 modes: 256 x 128 tiles (see umma_narrow): -1 auto, 0 never, 1 always (scheduling only)
  int pdl = -1;              // tcgen05 modes: programmatic dependent launch of the GEMM kernels: -1 auto, 0 off, 1 on, 2 on without the early set-up (scheduling only)
  int i8_narrow = -1;        // F64_I8: 256 x 128 tiles in the INT8 kernels: -1 auto (up to 6 x 6 macro tiles), 0 never, 1 always
  int i8_cluster = 0;        // F64_I8 a1: clusters of two CTA pairs sharing the B slices by TMA multicast (scheduling only)
  int i8_slices = 8;         // F64_I8: int8 slices per operand row (= orders i + j kept)
  int final_check = 1;       // FP64-master modes: 0 = skip a residual evaluation whose outcome is known beforehand (see stop_decide)
  int extra_update = 0;      // FP64-master modes: one more update after the paper's test has fired (see stop_decide)
  int input_f32 = 0;         // double-element modes: S and Z0 are float (promoted exactly), Z is returned as double
};

struct StopArgs {
  State* st;
  double* partials;          // one FP64 partial sum of squares per output tile
  int num_partials;
  double* d_err;             // user array, max_iter + 1 entries
  int n_iter;                // index n of the residual being evaluated
  int max_iter;
  int stop;                  // zfac_stop
  int order;                 // m of Eq. 13 (2, 3, 4): the test's exponent is nu_max = m + 1
  unsigned long long cond;   // zfac_graph_*: handle of the WHILE node's condition (0: none); set by graph_cond_kernel after a2
  // tcgen05 kernels (one launch may carry `batch` independent problems): `st` is an array of one State per problem, the
  // partials hold 16 sums per a2 tile (8 epilogue warps x 2 CTAs), tiles_pp a2 tiles per problem, and d_err is
  // [batch][err_stride]
  int extra;                 // FP64-master modes, ZFAC_OPT_EXTRA_UPDATE: when the test fires, perform ONE more update, then stop
  int nocheck;               // FP64-master modes, ZFAC_OPT_FINAL_CHECK = 0 (see stop_decide)
  double floor;              // ... the smallest Err worth iterating towards: 2^-53 sqrt(N)
  int tiles_pp;
  int slots_pt;              // partial sums per tile: 16 per 256 x 256 tile, 8 per 256 x 128 tile (one per warp and 128-column half)
  long long err_stride;
};
// n_iter < 0 (inside the loop body of a zfac_graph, whose kernel parameters are fixed): the index comes from the device,
// State::iters = index of the last Err written, so the residual being evaluated is iters + 1.
__device__ __forceinline__ int stop_index(const StopArgs& a) { return a.n_iter >= 0 ? a.n_iter : a.st->iters + 1; }

// Optional per-kernel timing (zfac_set_profile): an event is recorded on the launching stream
// before every GEMM kernel and one after the last; tags = step id (1,2,4,5) + 16 * iteration.
struct Prof {
  cudaEvent_t* ev = nullptr;
  int* tags = nullptr;
  int cap = 0, count = 0;
  bool on = false;
  inline void mark(cudaStream_t s, int tag) {
    if (!on || count >= cap) return;
    cudaEventRecord(ev[count], s);
    tags[count] = tag;
    ++count;
  }
};

// Host-side hook after step a5 of every statically enqueued iteration (zfac_refine_host starts the download of Z
// after the first update through it).
struct IterHook {
  void (*after_a5)(void* self, int n, cudaStream_t s);
  void* self;
  // tcgen05 modes: called once before the first residual with the sequencer (a zfac::UmmaSeq*); returns true if it has
  // enqueued the copy-in of S and step a1 itself (zfac_refine_host: band by band behind the upload of S)
  bool (*first_a1)(void* self, void* seq, cudaStream_t s) = nullptr;
  // tcgen05 modes, first update only: a5_bands > 1 runs a5 in that many row bands and calls after_a5_band after each
  // (rows [r0, r1) of the padded Z_1 are final; last = the whole of Z_1 is) INSTEAD of after_a5(0)
  int a5_bands = 1;
  void (*after_a5_band)(void* self, int r0, int r1, bool last, cudaStream_t s) = nullptr;
  // double-element modes: called before the update n is enqueued (an early download of the in-place FP64 master must have
  // finished before step a5 overwrites it)
  void (*before_update)(void* self, int n, cudaStream_t s) = nullptr;
};

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}

// The decision of step a3 for one problem, taken by ONE thread from Err[n] = err (Alg. 2, Eq. 38).
// Readings: strict '>' (Q9); test applied unconditionally as Alg. 2 prints it (Q10); non-finite Err stops with a flag
// (Q9); Err recorded for the final Z also at max_iter (Q7).
__device__ inline void stop_decide(const StopArgs& a, State* st, double* d_err, double err) {
  const int n = a.n_iter >= 0 ? a.n_iter : st->iters + 1;
  d_err[n] = err;
  st->iters = n;
  int flags = 0, done = 0;
  if (!isfinite(err)) {
    flags = ZFAC_R_NONFINITE; done = 1;
  } else if (a.stop == ZFAC_STOP_PAPER && n > 0) {
    const double prev = d_err[n - 1];
    double thr = prev * prev * prev;                         // m = 2: Err[n-1]^3 (Eq. 38)
    for (int k = 2; k < a.order; ++k) thr *= prev;           // m = 3, 4: Err[n-1]^(m+1)
    if (err > thr) { flags = ZFAC_R_STOPPED; done = 1; }
    // ZFAC_OPT_EXTRA_UPDATE (FP64-master modes): the correction of these modes is FP32-class, so the test also fires when the
    // residual has merely reached ~u32 sqrt(kappa) Err[n-1], one update short of the FP64 floor.  Like the refinement step of
    // Alg. 3 ("Typically we would only do one extra refinement step"), the first firing is answered by ONE
    // more update (marked ZFAC_R_REFINED); the evaluation after it ends the run.
    if (a.extra) {
      if (st->flags & ZFAC_R_REFINED) { flags = ZFAC_R_STOPPED; done = 1; }
      else if (done) { st->flags |= ZFAC_R_REFINED; flags = 0; done = 0; }
    }
  }
  if (!done && n == a.max_iter) { flags = ZFAC_R_MAXITER; done = 1; }
  // ZFAC_OPT_FINAL_CHECK = 0 (FP64-master modes, paper's rule): an evaluation whose outcome is known beforehand is not made.
  // That is the one after the extra update above (it ends the run whatever it finds), and, without that option, the one
  // after an update taken from Err[n]^3 < 2^-53 sqrt(N): the next Err cannot pass the test unless it is below anything the
  // arithmetic resolves, in which case there is nothing left to iterate for either.  The update in flight is then the last
  // (State::last); finish_kernel, at the head of the next residual, counts it and ends the run.
  if (!done && a.nocheck && a.stop == ZFAC_STOP_PAPER) {
    if (a.extra ? (st->flags & ZFAC_R_REFINED) != 0 : (err * err * err < a.floor)) st->last = 1;
  }
  if (done) { st->flags |= flags; __threadfence(); st->done = 1; }
}

// ZFAC_OPT_FINAL_CHECK = 0: first launch of every residual of the FP64-master modes.  If the update just performed was marked
// as the last one, count it, leave NaN in its Err entry and end the run: the residual kernels behind return at once.
__global__ void finish_kernel(State* st, double* d_err) {
  if (st->done || !st->last) return;
  const int n = st->iters + 1;
  st->iters = n;
  d_err[n] = nan("");
  st->flags |= ZFAC_R_STOPPED | ZFAC_R_NOCHECK;
  st->last = 0;
  __threadfence();
  st->done = 1;
}

// zfac_graph_*: the WHILE node's condition (another pass of the loop?) is set by this one-thread kernel right after every a2.
// It is a kernel of its own because cudaGraphSetConditional is a device-runtime CALL: a call anywhere in a kernel makes
// ptxas ignore setmaxnreg there (the a2 kernels ran all warps at the 168-register launch cap and spilled).
__global__ void graph_cond_kernel(const State* st, unsigned long long cond) {
  cudaGraphSetConditional((cudaGraphConditionalHandle)cond, st->done ? 0u : 1u);
}

// Step a3 in the tcgen05 kernels: every epilogue warp leaves the sum of squares of its 32 rows x 128 / 256 columns of an
// a2 tile in partials[(problem, tile)][slots_pt] and counts itself in; the warp that arrives LAST for a problem sums that
// problem's partials in index order (lane-strided, then a fixed shuffle tree) and takes the decision.  The order depends
// on the tile enumeration only, not on which CTA computed which tile: Err[] is run-to-run deterministic and the same
// whether a problem runs alone or as one of a batch.  Called by all 32 lanes of an epilogue warp after a tile.
// `lin` = position of this warp's sum among the tiles_pp * slots_pt sums of problem b.
__device__ inline void stop_test_index_warp(const StopArgs& a, int b, int lin, double tile_sumsq, int lane) {
  const double s = warp_sum(tile_sumsq);
  State* st = a.st + b;
  const int per = a.tiles_pp * a.slots_pt;
  double* part = a.partials + (size_t)b * per;
  int last = 0;
  if (lane == 0) {
    part[(size_t)lin] = s;
    __threadfence();
    last = (atomicAdd(&st->arrive[0], 1u) == (unsigned int)per - 1u);
    if (last) { st->arrive[0] = 0u; __threadfence(); }
  }
  last = __shfl_sync(0xffffffffu, last, 0);
  if (!last) return;
  double t = 0.0;
  for (int i = lane; i < per; i += 32) t += __ldcg(part + i);
  t = warp_sum(t);
  if (lane == 0) stop_decide(a, st, a.d_err + (size_t)b * a.err_stride, sqrt(t));
}

// Step a3 (Alg. 2, Eq. 38), FP64 / INT8 residual kernels.  Called by ALL threads of the CTA that
// finished last (blockDim.x <= 1024, multiple of 32).  Sums the per-CTA partials in a fixed
// order (thread-strided, then a fixed shuffle/smem tree), so Err[] is run-to-run deterministic.
__device__ inline void stop_test_last_cta(const StopArgs& a, double* smem_red /* >= 32 doubles */) {
  double s = 0.0;
  for (int i = threadIdx.x; i < a.num_partials; i += blockDim.x) s += __ldcg(a.partials + i);
  s = warp_sum(s);
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5, nw = (blockDim.x + 31) >> 5;
  if (lane == 0) smem_red[wid] = s;
  __syncthreads();
  if (threadIdx.x == 0) {
    double tot = 0.0;
    for (int w = 0; w < nw; ++w) tot += smem_red[w];
    stop_decide(a, a.st, a.d_err, sqrt(tot));
  }
}

// Returns true (to every thread of the CTA) if this CTA is the last of `total` to arrive.
__device__ inline bool arrive_is_last(unsigned int* counter, unsigned int total, int* smem_flag) {
  __syncthreads();
  if (threadIdx.x == 0) {
    __threadfence();
    const unsigned int prev = atomicAdd(counter, 1u);
    const int last = (prev == total - 1u);
    if (last) { *counter = 0u; __threadfence(); }
    *smem_flag = last;
  }
  __syncthreads();
  return *smem_flag != 0;
}

// Upper-triangle enumeration: t -> (i <= j), t = j (j + 1) / 2 + i.
__device__ __forceinline__ void tri_decode(int t, int& i, int& j) {
  int jj = (int)((sqrt(8.0 * (double)t + 1.0) - 1.0) * 0.5);
  while ((jj + 1) * (jj + 2) / 2 <= t) ++jj;
  while (jj * (jj + 1) / 2 > t) --jj;
  j = jj;
  i = t - jj * (jj + 1) / 2;
}

// Full-grid rasterisation in bands of `bw` tile-columns so that co-resident CTAs share
// operand rows/columns in L2.
__device__ __forceinline__ void band_decode(int t, int tiles_m, int tiles_n, int bw, int& mi, int& ni) {
  const int per_band = bw * tiles_m;
  const int band = t / per_band;
  const int r = t - band * per_band;
  int nb = tiles_n - band * bw;
  nb = nb < bw ? nb : bw;
  mi = r / nb;
  ni = band * bw + (r - mi * nb);
}

}  // namespace zfac
