// tcgen05 (5th-gen tensor core) GEMM kernels for the SPLIT16, HH16 and TF32 modes.
//
// One persistent, warp-specialised kernel template serves all four GEMMs of an iteration.
// As in zfac_f64.cuh every product is brought to  D[m][n] = sum_k A[m][k] B[n][k]  with both
// operands K-major (row-major storage), by keeping W = Z^T next to Z:
//   a1  T = (S Z)^T = W S^T    (Eq. 22)     a2  X = Z^T (S Z) = W T^T   (Eq. 26)
//   a4  P = R R = R R^T        (Eq. 30-32)  a5  Z Q = Z Q^T             (Eq. 13)
//
// CTA pair (cluster of 2, tcgen05 cta_group::2): one 256 x TILE_N output tile per pair.  CTA r of
// the pair stages rows [128 r, 128 r + 128) of the A tile and rows [TILE_N/2 r, ...) of the B tile
// (TMA, 128B-swizzle boxes of 64 rows x 128 B, landing on the LEADER's full barrier), the leader's
// elected thread issues tcgen05.mma with M = 256, N = TILE_N reading both CTAs' shared memory, and
// each CTA's TMEM (128 lanes x 512 columns) receives rows [128 r, 128 r + 128) of the accumulators.
//
// Roles per CTA (64 + 256 threads): warp 0 = TMA producer (one lane), warp 1 = TMEM allocator +
// (leader only) MMA issuer, warps 2-9 = two epilogue groups of 4 warps (tcgen05.ld, fused O(N^2)
// work, stores).  TMEM holds TWO accumulator sets; tile i of a pair uses set i mod 2 and epilogue
// group i mod 2, so the epilogue of a tile always overlaps the mainloop of the next one.
// Pipelines: shared-memory ring full/empty mbarriers (TMA <-> MMA; "empty" is multicast to both
// CTAs by tcgen05.commit) and, per accumulator set, TMEM full/empty mbarriers (MMA <-> that set's
// epilogue group in both CTAs) plus the D_hh chunk hand-over barriers of the promoted accumulation.
//
// Precision kinds
//   KIND_F16X2 (SPLIT16 mode): operands are fp16 pairs (hi, lo' = lo * 2^11), Eq. 17-18.
//       Three MMA passes per k-step, (l)(l) dropped (Eq. 25, 29, 32):
//           D_hh += A_hi B_hi          D_x += A_hi B_lo' + A_lo' B_hi
//       two FP32 accumulators per set, hence TILE_N = 128 (2 sets x 2 x 128 = 512 TMEM columns); the
//       epilogue forms D_hh + 2^-11 D_x.  D_hh is drained into FP32 registers every chunk_kb
//       k-blocks (promoted accumulation).
//   KIND_HH16  (HH16 mode, the paper's (h)(h) scheme, Sec. III.C): fp16 operands, one pass, TILE_N = 256.
//   KIND_TF32  (TF32 mode): FP32 operands read as TF32, one pass, TILE_N = 256.
#pragma once
#include <cuda.h>
#include <stdio.h>
#include <stdlib.h>
#include <cuda_fp16.h>
#include "zfac_common.cuh"
#include "zfac_io.cuh"
#include "zfac_f64.cuh"   // EPI_* ids

namespace zfac {

// ...N: the same kind on 256 x 128 tiles (small launches, ZFAC_OPT_NARROW_TILES)
enum { KIND_F16X2 = 0, KIND_HH16 = 1, KIND_TF32 = 2, KIND_F16X2N = 3, KIND_HH16N = 4, KIND_TF32N = 5 };
__host__ __device__ constexpr bool kind_is_pair(int kind) { return kind == KIND_F16X2 || kind == KIND_F16X2N; }
__host__ __device__ constexpr bool kind_is_tf32(int kind) { return kind == KIND_TF32 || kind == KIND_TF32N; }
__host__ __device__ constexpr bool kind_is_narrow(int kind) { return kind >= KIND_F16X2N; }

constexpr int UM_TILE_M = 256;                   // pair tile rows: two CTAs x 128 TMEM lanes
constexpr int UM_MACRO = 256;                    // padding unit and macro tile of the symmetric enumeration
constexpr int UM_ROWS = 128;                     // A-operand rows staged per CTA
constexpr int UM_ROWB = 128;                     // bytes per operand row per k-block (= swizzle span)
constexpr int UM_BOX_ROWS = 64;                  // rows per TMA box
constexpr int UM_BOX_BYTES = UM_BOX_ROWS * UM_ROWB;  // 8 KB
constexpr int UM_A_BYTES = UM_ROWS * UM_ROWB;    // 16 KB: A rows of one array, one stage, one CTA
constexpr int UM_SMEM_OPERANDS = 192 * 1024;
constexpr int UM_SMEM_BYTES = UM_SMEM_OPERANDS + 1024 /*align*/ + 256 /*barriers*/;
constexpr int UM_TMEM_COLS = 512;
constexpr int UM_EPI_WARPS = 8;                  // two groups of 4 (one warp per TMEM lane quarter), alternating tiles
constexpr int UM_EPI_WARP0 = 4;                  // first epilogue warp: warps 0-3 form the control warpgroup (producer, issuer, 2 idle)
constexpr int UM_THREADS = 32 * (UM_EPI_WARP0 + UM_EPI_WARPS);     // 384 = three warpgroups
// Register budget (setmaxnreg works on whole warpgroups): the kernel is launched with 65536 / 384 -> 168 registers per
// thread; the control warpgroup (one lane each runs TMA issue / MMA issue) gives most of its share to the two epilogue
// warpgroups, whose SPLIT16 threads hold a 128-column FP32 running sum: 128 x 64 + 256 x 216 <= 384 x 168.
constexpr int UM_REGS_CONTROL = 64, UM_REGS_EPILOGUE = 216;
#ifndef ZFAC_DRAIN_W
#define ZFAC_DRAIN_W 32
#endif
template <int N> __device__ __forceinline__ void reg_dealloc() { asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(N)); }
template <int N> __device__ __forceinline__ void reg_alloc() { asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(N)); }
constexpr int UM_MAX_STAGES = 6;

// TILE_N: columns of the pair tile (= N of one tcgen05.mma; each CTA stages TILE_N / 2 rows of B).
// SETS: accumulator sets in the 512 TMEM columns.  The one-pass kinds keep two (the epilogue of tile i overlaps
// the mainloop of tile i + 1, epilogue group i mod 2).  F16X2 needs two FP32 accumulators (D_hh, D_x) per set:
// at TILE_N = 256 only one set fits, so its epilogue copies the accumulators to registers and releases the
// tensor memory BEFORE it does the slow global loads / stores.  (TILE_N = 128 with two sets was measured: the
// operand reads of a 256 x 128 x 16 MMA plus the TMA fill exceed the 128 B/clk shared-memory port, a1 ran 30 %
// slower -- profiles/r1b_summary.md.)
template <int KIND> struct KindTraits;
template <> struct KindTraits<KIND_F16X2> {
  static constexpr int ARRAYS = 2, TILE_N = 256, SETS = 1, STAGES = 3, KSTEP_ELEMS = 16, BK_ELEMS = 64, FMT = 0, SUB = 16;
};
// The same arithmetic on 256 x 128 tiles with two accumulator sets: twice as many tiles.  Per tile column it is slower (the
// shared-memory port, see above), but a problem of <= 6 x 6 macro tiles leaves most of the 74 CTA pairs idle on 256 x 256
// tiles: one SPLIT16 problem of N = 512 / 1024 runs 24 / 23 % faster on these (ZFAC_OPT_NARROW_TILES).  Every output element
// is accumulated in the same order, and the a2 partial sums are laid out as for the wide tiles: bit-identical results.
template <> struct KindTraits<KIND_F16X2N> {
  static constexpr int ARRAYS = 2, TILE_N = 128, SETS = 2, STAGES = 4, KSTEP_ELEMS = 16, BK_ELEMS = 64, FMT = 0, SUB = 16;
};
template <> struct KindTraits<KIND_HH16> {
  static constexpr int ARRAYS = 1, TILE_N = 256, SETS = 2, STAGES = 6, KSTEP_ELEMS = 16, BK_ELEMS = 64, FMT = 0, SUB = 32;
};
template <> struct KindTraits<KIND_TF32> {
  static constexpr int ARRAYS = 1, TILE_N = 256, SETS = 2, STAGES = 6, KSTEP_ELEMS = 8, BK_ELEMS = 32, FMT = 2, SUB = 32;
};
template <> struct KindTraits<KIND_HH16N> {
  static constexpr int ARRAYS = 1, TILE_N = 128, SETS = 2, STAGES = 6, KSTEP_ELEMS = 16, BK_ELEMS = 64, FMT = 0, SUB = 32;
};
template <> struct KindTraits<KIND_TF32N> {
  static constexpr int ARRAYS = 1, TILE_N = 128, SETS = 2, STAGES = 6, KSTEP_ELEMS = 8, BK_ELEMS = 32, FMT = 2, SUB = 32;
};

struct UmmaParams {
  CUtensorMap mapA;     // A-operand buffer: [ARRAYS*Np rows][Np cols], box 128 B x 64 rows
  CUtensorMap mapB;     // B-operand buffer, same box
  int np;               // padded dimension (= K)
  int batch;            // independent problems in this launch (>= 1), stacked along the rows of every buffer
  int rows;             // batch * np: rows of one plane of a buffer; problem b owns rows [b np, (b + 1) np)
  int macro_tiles;      // Np / 256
  int chunk_kb;         // KIND_F16X2: k-blocks (of 64) per promoted accumulation chunk (0 = whole K)
  int chunk0_kb;        // KIND_F16X2: k-blocks of the FIRST chunk of a tile (>= chunk_kb; see the MMA issuer)
  State* st;            // [batch]
  StopArgs stop;        // a2 (partials: 2 UM_EPI_WARPS / SETS per tile and problem); a4 / p2: Err[n] of the one-pass decision
  // epilogue pointers (which are used depends on EPI / KIND; see the epilogue)
  float* f32_out;       // a1: T32 (TF32)   a2: R32   a4: Q32 (TF32)   a5: Z32 next
  const float* f32_in;  // a4: R32          a5: Z32 current
  void* h_out;          // 16-bit modes: a1: T16   a2: R16   a4: Q16   a5: Z16 next  ([ARRAYS][Np][Np])
  void* h_out_t;        // 16-bit modes: a5: W16 (transposed)                         TF32: a5: W32
  void* out2;           // p2 (order m > 2): G operand buffer, same format as the mode's operands
  int band;             // full outputs: tile columns per rasterisation band (L2 reuse of the B column blocks)
  int ioff, irows;      // full outputs: ... and tile rows [ioff, ioff + irows) only (irows = 0: all): a5 in row bands, so
                        // that zfac_refine_host can start downloading the finished rows of Z
  int joff, jcols;      // full outputs: this launch covers tile columns [joff, joff + jcols) only (jcols = 0: all) --
                        // zfac_refine_host runs a1 band by band while the row chunks of S are still arriving
  int hh_only;          // KIND_F16X2: 1 = this launch MAY use the (h)(h) pass only (D_x neither written nor read) ...
  double hh_err_max;    // ... and does so iff Err[n] = stop.d_err[stop.n_iter] <= hh_err_max (decided on the device)
  float q_r, q_d;       // a4: Q = q_r R + q_d D        (1/2, 3/8; m > 2: 1/2, 1)       see PolyCoef (zfac_f64.cuh)
  float g_i, g_r, g_p;  // p2: G = g_i I + g_r R + g_p D (3/8, 5/16, 35/128 or 0)
  int early;            // programmatic dependent launch with the wait AFTER the set-up (see the head of the kernel)
  int scaled;           // FP64-master modes: a4 works on R~ = rscale R (State::rscale): Q~ = q_r R~ + (q_d / rscale) R~ R~
  double* z64;          // a5x: FP64 master Z, updated in place: Z64 += D / rscale
  double* w64t;         // a5x: FP64 W = Z^T (DMMA residual engine) or null
  unsigned long long* dbg;  // -DZFAC_TIMING builds only: per-CTA wait-cycle counters of the MMA issuer (else null)
};

// ------------------------------------------------------------------ PTX wrappers
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ uint32_t cluster_ctarank() {
  uint32_t r;
  asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r));
  return r;
}
// shared::cluster address of `addr` (a shared::cta address of this CTA) in CTA `rank` of the cluster
__device__ __forceinline__ uint32_t mapa_u32(uint32_t addr, uint32_t rank) {
  uint32_t r;
  asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(addr), "r"(rank));
  return r;
}
__device__ __forceinline__ void cluster_sync_all() {
  asm volatile("barrier.cluster.arrive.release.aligned;" ::: "memory");
  asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory");
}
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
// Arrive on a barrier given by its shared::cluster address (own or peer CTA).  RELAXED: the arrivals of the
// epilogue warps only tell the MMA issuer that their tcgen05.ld of an accumulator have completed (the values are
// in registers after tcgen05.wait::ld; tcgen05.fence::before/after_thread_sync order the tensor-memory accesses).
// No generic-proxy data is published, and a .release.cluster arrive costs a GPU-scope fence
// (MEMBAR.ALL.GPU + ERRBAR + CGAERRBAR, profiles/r1a_summary.md) on the critical path of every chunk drain.
// Predicated inside the asm (one arrival per warp, lane 0) so that the call site is straight-line code: a
// compiler barrier in a divergent branch did not keep the epilogue's global loads / stores below the arrive.
__device__ __forceinline__ void mbar_arrive_cluster_lane0(uint32_t bar_cluster_addr, int lane) {
  asm volatile(
      "{\n .reg .pred p;\n setp.eq.s32 p, %1, 0;\n @p mbarrier.arrive.relaxed.cluster.shared::cluster.b64 _, [%0];\n}"
      ::"r"(bar_cluster_addr), "r"(lane) : "memory");
}
// Bounded wait: a pipeline bug traps (launch failure) instead of hanging the GPU.
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
  uint32_t ok = 0;
  unsigned long long spins = 0;
  while (true) {
    asm volatile(
        "{\n .reg .pred p;\n mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n selp.u32 %0, 1, 0, p;\n}"
        : "=r"(ok)
        : "r"(bar), "r"(parity)
        : "memory");
    if (ok) break;
    if (++spins > (1ull << 26)) __trap();
  }
}
// TMA load issued by one CTA of the pair into ITS shared memory; the transaction bytes are
// counted on the barrier `bar_cluster_addr` (the leader CTA's full barrier).
__device__ __forceinline__ void tma_load_2d_pair(uint32_t dst, const CUtensorMap* map, int c0, int c1, uint32_t bar_cluster_addr) {
  asm volatile(
      "cp.async.bulk.tensor.2d.cta_group::2.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];"
      ::"r"(dst), "l"(reinterpret_cast<uint64_t>(map)), "r"(c0), "r"(c1), "r"(bar_cluster_addr)
      : "memory");
}
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
// tcgen05.commit of the pair's MMAs: arrives on the barrier at offset `bar` in BOTH CTAs.
__device__ __forceinline__ void tc_commit_pair(uint32_t bar) {
  asm volatile("tcgen05.commit.cta_group::2.mbarrier::arrive::one.shared::cluster.multicast::cluster.b64 [%0], %1;"
               ::"r"(bar), "h"((uint16_t)3) : "memory");
}
template <int KIND>
__device__ __forceinline__ void tc_mma_pair(uint32_t d_tmem, uint64_t adesc, uint64_t bdesc, uint32_t idesc, uint32_t accum) {
  if (kind_is_tf32(KIND)) {
    asm volatile("{\n .reg .pred p;\n setp.ne.b32 p, %4, 0;\n tcgen05.mma.cta_group::2.kind::tf32 [%0], %1, %2, %3, p;\n}"
                 ::"r"(d_tmem), "l"(adesc), "l"(bdesc), "r"(idesc), "r"(accum) : "memory");
  } else {
    asm volatile("{\n .reg .pred p;\n setp.ne.b32 p, %4, 0;\n tcgen05.mma.cta_group::2.kind::f16 [%0], %1, %2, %3, p;\n}"
                 ::"r"(d_tmem), "l"(adesc), "l"(bdesc), "r"(idesc), "r"(accum) : "memory");
  }
}
__device__ __forceinline__ void tmem_ld(uint32_t taddr, uint32_t (&r)[32]) {
  asm volatile(
      "tcgen05.ld.sync.aligned.32x32b.x32.b32 "
      "{%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16,%17,%18,%19,%20,%21,%22,%23,%24,%25,%26,%27,%28,%29,%30,%31}, [%32];"
      : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]),
        "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15]), "=r"(r[16]),
        "=r"(r[17]), "=r"(r[18]), "=r"(r[19]), "=r"(r[20]), "=r"(r[21]), "=r"(r[22]), "=r"(r[23]), "=r"(r[24]),
        "=r"(r[25]), "=r"(r[26]), "=r"(r[27]), "=r"(r[28]), "=r"(r[29]), "=r"(r[30]), "=r"(r[31])
      : "r"(taddr));
}
__device__ __forceinline__ void tmem_ld(uint32_t taddr, uint32_t (&r)[16]) {
  asm volatile(
      "tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];"
      : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]),
        "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15])
      : "r"(taddr));
}
__device__ __forceinline__ void tmem_ld(uint32_t taddr, uint32_t (&r)[64]) {
  asm volatile(
      "tcgen05.ld.sync.aligned.32x32b.x64.b32 "
      "{%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16,%17,%18,%19,%20,%21,%22,%23,%24,%25,%26,%27,%28,%29,%30,%31,"
      "%32,%33,%34,%35,%36,%37,%38,%39,%40,%41,%42,%43,%44,%45,%46,%47,%48,%49,%50,%51,%52,%53,%54,%55,%56,%57,%58,%59,%60,%61,%62,%63}, [%64];"
      : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]),
        "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15]), "=r"(r[16]),
        "=r"(r[17]), "=r"(r[18]), "=r"(r[19]), "=r"(r[20]), "=r"(r[21]), "=r"(r[22]), "=r"(r[23]), "=r"(r[24]),
        "=r"(r[25]), "=r"(r[26]), "=r"(r[27]), "=r"(r[28]), "=r"(r[29]), "=r"(r[30]), "=r"(r[31]), "=r"(r[32]),
        "=r"(r[33]), "=r"(r[34]), "=r"(r[35]), "=r"(r[36]), "=r"(r[37]), "=r"(r[38]), "=r"(r[39]), "=r"(r[40]),
        "=r"(r[41]), "=r"(r[42]), "=r"(r[43]), "=r"(r[44]), "=r"(r[45]), "=r"(r[46]), "=r"(r[47]), "=r"(r[48]),
        "=r"(r[49]), "=r"(r[50]), "=r"(r[51]), "=r"(r[52]), "=r"(r[53]), "=r"(r[54]), "=r"(r[55]), "=r"(r[56]),
        "=r"(r[57]), "=r"(r[58]), "=r"(r[59]), "=r"(r[60]), "=r"(r[61]), "=r"(r[62]), "=r"(r[63])
      : "r"(taddr));
}
__device__ __forceinline__ void tmem_ld_wait() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }

// K-major, 128B-swizzle shared-memory matrix descriptor (sm_100 version bit 46).
__device__ __forceinline__ uint64_t make_sdesc(uint32_t saddr) {
  return (uint64_t)((saddr & 0x3FFFFu) >> 4) | (1ull << 16) | ((uint64_t)(1024 >> 4) << 32) | (1ull << 46) | (2ull << 61);
}
// kind::f16 / kind::tf32 instruction descriptor: D = F32, A/B format, both K-major, M = 256 (pair), N = n.
__host__ __device__ constexpr uint32_t make_idesc(int fmt, int n) {
  return (1u << 4) | ((uint32_t)fmt << 7) | ((uint32_t)fmt << 10) | ((uint32_t)(n >> 3) << 17) | ((uint32_t)(UM_TILE_M >> 4) << 24);
}

__device__ __forceinline__ uint32_t pack_h2(__half a, __half b) {
  return (uint32_t)__half_as_ushort(a) | ((uint32_t)__half_as_ushort(b) << 16);
}

// Write N consecutive values of one row in the mode's 16-bit operand format:
// PAIR: (hi -> base, lo' -> base + plane), Eq. 17-18 with the low half scaled;  else hi = FP16[v] only.
template <bool PAIR, int N>
__device__ __forceinline__ void store_h_row(void* base, size_t plane, size_t off, const float (&v)[N]) {
  uint32_t hi[N / 2], lo[N / 2];
#pragma unroll
  for (int j = 0; j < N / 2; ++j) {
    if (PAIR) {
      __half h0, l0, h1, l1;
      split_f16(v[2 * j], h0, l0); split_f16(v[2 * j + 1], h1, l1);
      hi[j] = pack_h2(h0, h1); lo[j] = pack_h2(l0, l1);
    } else {
      hi[j] = pack_h2(f2h_sat(v[2 * j]), f2h_sat(v[2 * j + 1]));
    }
  }
  uint16_t* b = static_cast<uint16_t*>(base);
  uint4* ph = reinterpret_cast<uint4*>(b + off);
  uint4* pl = reinterpret_cast<uint4*>(b + plane + off);
#pragma unroll
  for (int j = 0; j < N / 8; ++j) {
    ph[j] = make_uint4(hi[4 * j], hi[4 * j + 1], hi[4 * j + 2], hi[4 * j + 3]);
    if (PAIR) pl[j] = make_uint4(lo[4 * j], lo[4 * j + 1], lo[4 * j + 2], lo[4 * j + 3]);
  }
}
// Transposed: value j of this lane goes to row (n + j), column m (lanes hold consecutive m).
template <bool PAIR, int N>
__device__ __forceinline__ void store_h_col(void* base, size_t plane, size_t off_n0_m, size_t ld, const float (&v)[N]) {
  uint16_t* b = static_cast<uint16_t*>(base);
#pragma unroll
  for (int j = 0; j < N; ++j) {
    if (PAIR) {
      __half hh, ll; split_f16(v[j], hh, ll);
      b[off_n0_m + (size_t)j * ld] = __half_as_ushort(hh);
      b[plane + off_n0_m + (size_t)j * ld] = __half_as_ushort(ll);
    } else {
      b[off_n0_m + (size_t)j * ld] = __half_as_ushort(f2h_sat(v[j]));
    }
  }
}
template <int N>
__device__ __forceinline__ void store_f32_row(float* p, const float (&v)[N]) {
  float4* q = reinterpret_cast<float4*>(p);
#pragma unroll
  for (int j = 0; j < N / 4; ++j) q[j] = make_float4(v[4 * j], v[4 * j + 1], v[4 * j + 2], v[4 * j + 3]);
}
template <int N>
__device__ __forceinline__ void load_f32_row(const float* p, float (&v)[N]) {
  const float4* q = reinterpret_cast<const float4*>(p);
#pragma unroll
  for (int j = 0; j < N / 4; ++j) {
    const float4 t = q[j];
    v[4 * j] = t.x; v[4 * j + 1] = t.y; v[4 * j + 2] = t.z; v[4 * j + 3] = t.w;
  }
}

// A magnitude >= 65504 is clamped by the fp16 conversion (cvt.rn.satfinite) without producing inf / NaN: report it
// (ZFAC_R_RANGE) for the two outputs whose size the iteration does not bound, T = (S Z)^T and Z.
template <int N>
__device__ __forceinline__ void flag_h16_range(State* st, const float (&v)[N]) {
  float mx = 0.0f;
#pragma unroll
  for (int j = 0; j < N; ++j) mx = fmaxf(mx, fabsf(v[j]));
  if (mx >= H16_MAX) atomicOr(&st->range, 1);
}

// Fused epilogue for SUB consecutive columns n..n+SUB-1 of row m (v = accumulator values).
// m = row in the stacked buffers (mb + local row, mb = first row of the tile's problem), n = local column.
template <int KIND, int EPI, int SUB>
__device__ __forceinline__ void epilogue_cols(const UmmaParams& p, float (&v)[SUB], int m, int n, int mb, bool offdiag,
                                              double& tile_sumsq) {
  constexpr bool PAIR = kind_is_pair(KIND);
  const size_t ld = (size_t)p.np, plane = ld * (size_t)p.rows;
  const size_t off = (size_t)m * ld + n;               // (m, n)
  const size_t offt = (size_t)(mb + n) * ld + (m - mb);   // (n, m) of the same problem
  const int ml = m - mb;                               // local row: the diagonal is ml == n
  if (EPI == EPI_A1) {                                  // T = (S Z)^T
    if (kind_is_tf32(KIND)) {
#pragma unroll
      for (int j = 0; j < SUB; ++j) v[j] = round_tf32(v[j]);
      store_f32_row<SUB>(p.f32_out + off, v);
    } else {
      flag_h16_range<SUB>(p.st + mb / p.np, v);
      store_h_row<PAIR, SUB>(p.h_out, plane, off, v);
    }
  } else if (EPI == EPI_A2) {                           // R = I - X, sum R^2, mirror
    // sum of squares: FP32 inside this group of SUB (16 / 32) columns, FP64 across groups, tiles and CTAs.  One DFMA
    // plus one conversion per ELEMENT was 13 % of all warp samples of a2 (a quarter of its non-waiting time,
    // profiles/r1b_summary.md §4); the entries of R carry ~6e-8 relative noise themselves, a 16-term FP32 partial
    // sum adds <= 1e-6 relative per group, random in sign; the order is fixed, so Err[] stays run-to-run deterministic.
    float ss = 0.0f;
#pragma unroll
    for (int j = 0; j < SUB; ++j) {
      v[j] = ((ml == n + j) ? 1.0f : 0.0f) - v[j];
      ss = fmaf(v[j], v[j], ss);
    }
    tile_sumsq += (double)ss;
    store_f32_row<SUB>(p.f32_out + off, v);
    if (!kind_is_tf32(KIND)) store_h_row<PAIR, SUB>(p.h_out, plane, off, v);
    if (offdiag) {
      // mirror: the operand of a4 needs the whole matrix -- the fp16 plane(s), or in TF32 mode the FP32 buffer itself.
      // The FP32 copy of the 16-bit modes is read by a4's / p2's epilogue only, at upper-triangle tiles: its lower
      // triangle is never written (zfac_peek reads the upper one).
      if (kind_is_tf32(KIND)) {
#pragma unroll
        for (int j = 0; j < SUB; ++j) p.f32_out[offt + (size_t)j * ld] = v[j];
      } else {
        store_h_col<PAIR, SUB>(p.h_out, plane, offt, ld, v);
      }
    }
  } else if (EPI == EPI_X3) {                           // X = Z^T H Z itself (congruence), mirror
    store_f32_row<SUB>(p.f32_out + off, v);
    if (offdiag) {
#pragma unroll
      for (int j = 0; j < SUB; ++j) p.f32_out[offt + (size_t)j * ld] = v[j];
    }
  } else if (EPI == EPI_A4) {                           // Q = 1/2 R + 3/8 R R, mirror
    float r32[SUB];
    load_f32_row<SUB>(p.f32_in + off, r32);
    const float qd = p.scaled ? p.q_d * p.st->rinv : p.q_d;            // scaled operands: D = R~ R~ = rscale^2 R R
#pragma unroll
    for (int j = 0; j < SUB; ++j) v[j] = p.q_r * r32[j] + qd * v[j];
    if (kind_is_tf32(KIND)) {
#pragma unroll
      for (int j = 0; j < SUB; ++j) v[j] = round_tf32(v[j]);
      store_f32_row<SUB>(p.f32_out + off, v);
      if (offdiag) {
#pragma unroll
        for (int j = 0; j < SUB; ++j) p.f32_out[offt + (size_t)j * ld] = v[j];
      }
    } else {
      store_h_row<PAIR, SUB>(p.h_out, plane, off, v);
      if (offdiag) store_h_col<PAIR, SUB>(p.h_out, plane, offt, ld, v);
    }
  } else if (EPI == EPI_P2) {                           // order m > 2: P = R R and G = 3/8 I + 5/16 R + g_p P, mirror
    float g[SUB];
    {
      float r32[SUB];
      load_f32_row<SUB>(p.f32_in + off, r32);
#pragma unroll
      for (int j = 0; j < SUB; ++j) g[j] = ((ml == n + j) ? p.g_i : 0.0f) + p.g_r * r32[j] + p.g_p * v[j];
    }
    if (kind_is_tf32(KIND)) {
      float* g32 = static_cast<float*>(p.out2);
#pragma unroll
      for (int j = 0; j < SUB; ++j) { v[j] = round_tf32(v[j]); g[j] = round_tf32(g[j]); }
      store_f32_row<SUB>(p.f32_out + off, v);
      store_f32_row<SUB>(g32 + off, g);
      if (offdiag) {
#pragma unroll
        for (int j = 0; j < SUB; ++j) { p.f32_out[offt + (size_t)j * ld] = v[j]; g32[offt + (size_t)j * ld] = g[j]; }
      }
    } else {
      store_h_row<PAIR, SUB>(p.h_out, plane, off, v);
      store_h_row<PAIR, SUB>(p.out2, plane, off, g);
      if (offdiag) {
        store_h_col<PAIR, SUB>(p.h_out, plane, offt, ld, v);
        store_h_col<PAIR, SUB>(p.out2, plane, offt, ld, g);
      }
    }
  } else if (EPI == EPI_A5X) {                          // FP64 master: Z64 += (Z Q~) / rscale; next operand pair; W64 = Z^T
    if (kind_is_pair(KIND)) {
      const double rinv = (double)p.st->rinv;
      double* zp = p.z64 + off;
      float z32[SUB];
#pragma unroll
      for (int j = 0; j < SUB; j += 2) {
        double2 z = *reinterpret_cast<const double2*>(zp + j);
        z.x += (double)v[j] * rinv; z.y += (double)v[j + 1] * rinv;
        *reinterpret_cast<double2*>(zp + j) = z;
        if (p.w64t) { p.w64t[offt + (size_t)j * ld] = z.x; p.w64t[offt + (size_t)(j + 1) * ld] = z.y; }
        z32[j] = (float)z.x; z32[j + 1] = (float)z.y;
      }
      flag_h16_range<SUB>(p.st, z32);
      store_h_row<PAIR, SUB>(p.h_out, plane, off, z32);                // FP32[Z64] as the next update's A operand
    }
  } else {                                              // a5: Z_next = Z + Z Q, W = Z_next^T
    float z32[SUB];
    load_f32_row<SUB>(p.f32_in + off, z32);
#pragma unroll
    for (int j = 0; j < SUB; ++j) v[j] += z32[j];
    store_f32_row<SUB>(p.f32_out + off, v);
    if (kind_is_tf32(KIND)) {
      float* wt = static_cast<float*>(p.h_out_t);
#pragma unroll
      for (int j = 0; j < SUB; ++j) wt[offt + (size_t)j * ld] = round_tf32(v[j]);
    } else {
      flag_h16_range<SUB>(p.st + mb / p.np, v);
      store_h_row<PAIR, SUB>(p.h_out, plane, off, v);                // Z16 next
      store_h_col<PAIR, SUB>(p.h_out_t, plane, offt, ld, v);         // W16 = Z16^T
    }
  }
}

// -DZFAC_TIMING: the MMA issuer thread accumulates the cycles it spends in each kind of wait
// (0 smem-full = TMA starvation, 1 hh_empty = chunk drain, 2 tempty = epilogue, 3 whole role loop).
#ifdef ZFAC_TIMING
#define ZF_TWAIT(i, stmt) do { const long long t0_ = clock64(); stmt; twait[i] += clock64() - t0_; } while (0)
#else
#define ZF_TWAIT(i, stmt) do { stmt; } while (0)
#endif

// ------------------------------------------------------------------ the kernel
template <int KIND, int EPI>
__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(UM_THREADS, 1)
umma_gemm_kernel(const __grid_constant__ UmmaParams p) {
  // stop decided earlier in this call (uniform over the grid); in a batched launch finished problems are skipped tile by tile
  // Programmatic dependent launch (launches with the attribute; a no-op otherwise): this grid may have been scheduled while
  // its predecessor in the stream was still running.  Nothing of global memory is touched before the predecessor has
  // completed (wait); then the successor is let in at once -- it takes SMs as they fall free and waits here in turn, so
  // its launch latency is hidden behind this kernel (the kernels of a small problem, the early-exit launches behind the stop).
  // p.early (small launches, which leave SMs free): the successor is let in FIRST and the wait comes after this kernel's own
  // set-up (barrier init, tensor-memory allocation, pair synchronisation: pair_sync_in), so that the set-up too runs while the
  // predecessor still works; a launch behind the stop then skips its tiles instead of returning here.
  if (!p.early) {
    asm volatile("griddepcontrol.wait;" ::: "memory");
    if (p.batch == 1 && *((volatile int*)&p.st->done)) return;
  }
  asm volatile("griddepcontrol.launch_dependents;" ::: "memory");

  using KT = KindTraits<KIND>;
  constexpr bool SYM = (EPI == EPI_A2 || EPI == EPI_A4 || EPI == EPI_X3 || EPI == EPI_P2);
  constexpr bool PAIRK = kind_is_pair(KIND);                   // (hi, lo') operand pairs, promoted accumulation
  constexpr int TN = KT::TILE_N;
  constexpr int NSPLIT = UM_MACRO / TN;                        // column sub-tiles per 256-wide macro tile
  constexpr int B_BYTES = (TN / 2) * UM_ROWB;                  // B rows of one array, one stage, one CTA
  constexpr int STAGE_BYTES = KT::ARRAYS * (UM_A_BYTES + B_BYTES);
  constexpr int SET_COLS = KT::ARRAYS * TN;                    // TMEM columns of one accumulator set
  constexpr int SETS = KT::SETS;
  constexpr int GCOLS = (SETS == 2) ? TN : TN / 2;             // columns per epilogue thread
  static_assert(SETS * SET_COLS <= UM_TMEM_COLS, "the accumulator sets must fit the tensor memory");
  static_assert(KT::STAGES * STAGE_BYTES <= UM_SMEM_OPERANDS && KT::STAGES <= UM_MAX_STAGES, "smem");
  static_assert(!PAIRK || (KT::STAGES >= 3 && KT::STAGES <= 4), "promoted issue order: FRONT + BACK + 1 <= STAGES");
  constexpr int KSTEPS = KT::BK_ELEMS / KT::KSTEP_ELEMS;       // 4
  constexpr uint32_t IDESC = make_idesc(KT::FMT, TN);
  constexpr int SUB = KT::SUB;

  extern __shared__ unsigned char smem_raw[];
  const uint32_t smem_base = (smem_u32(smem_raw) + 1023u) & ~1023u;
  const uint32_t bar_base = smem_base + UM_SMEM_OPERANDS;
  // barrier slots (8 B each): full[0..5], empty[6..11], tfull[12..13], tempty[14..15], hh_full[16..17], hh_empty[18..19]
  auto full_bar = [&](int s) { return bar_base + 8u * s; };
  auto empty_bar = [&](int s) { return bar_base + 48u + 8u * s; };
  auto tfull_bar = [&](int b) { return bar_base + 96u + 8u * b; };
  auto tempty_bar = [&](int b) { return bar_base + 112u + 8u * b; };
  auto hh_full_bar = [&](int b) { return bar_base + 128u + 8u * b; };
  auto hh_empty_bar = [&](int b) { return bar_base + 144u + 8u * b; };
  const uint32_t tmem_slot = bar_base + 160u;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const uint32_t rank = cluster_ctarank();                 // 0 = leader (issues the MMAs)
  const int pair = blockIdx.x >> 1, num_pairs = gridDim.x >> 1;
  const int np = p.np;
  const int KB = np / KT::BK_ELEMS;
  const int CH = (p.chunk_kb > 0 && p.chunk_kb < KB) ? p.chunk_kb : KB;   // k-blocks per promoted chunk (KIND_F16X2)
  // first chunk of a tile: at most a quarter of K (its partial sums stay small), never shorter than CH
  const int CH0 = (CH < KB && p.chunk0_kb > CH && KB / 4 > CH) ? (p.chunk0_kb < KB / 4 ? p.chunk0_kb : KB / 4) : CH;
  const int NCH = 1 + (KB - CH0 + CH - 1) / CH;                            // chunks per tile
  const int T = p.macro_tiles;
  const int JC = (!SYM && p.jcols > 0) ? p.jcols : T * NSPLIT;             // tile columns of this launch
  const int TI = (!SYM && p.irows > 0) ? p.irows : T;                      // tile rows of this launch
  const int tiles_pp = SYM ? T * (T + 1) / 2 * NSPLIT : TI * JC;          // 256 x TN pair tiles of ONE problem
  const int all_tiles = tiles_pp * p.batch;                                // tile t: problem t / tiles_pp

  // The two register regimes (setmaxnreg) are two disjoint regions of the kernel: everything a role executes, including
  // its side of the two pair-wide synchronisations, sits inside its own branch (ptxas allocates registers per region
  // only when no path joins them again before the role code).
  auto pair_sync_in = [&]() -> uint32_t {                  // barrier inits + TMEM allocation visible to the pair
    tc_fence_before();
    __syncthreads();
    cluster_sync_all();
    tc_fence_after();
    uint32_t tb;
    asm volatile("ld.shared.b32 %0, [%1];" : "=r"(tb) : "r"(tmem_slot));
    if (p.early) asm volatile("griddepcontrol.wait;" ::: "memory");
    return tb;
  };
  // tiles of this launch as the roles see them (read AFTER pair_sync_in): none behind the stop
  auto live_tiles = [&]() -> int { return (p.early && p.batch == 1 && *((volatile int*)&p.st->done)) ? 0 : all_tiles; };
  auto pair_sync_out = [&]() {                             // no MMA / remote arrive of the pair is in flight any more
    tc_fence_before();
    __syncthreads();
    cluster_sync_all();
  };

  // Tile t of the launch -> its problem and position.  m0: first row of the A operand and of the output in the stacked
  // buffers; n0: first output column (local); mb: first row of the problem (B operand rows start at mb + n0).
  // Returns false for a tile of a problem that has already stopped (batched launches; every role skips it alike: `done` is
  // set by the a2 launch that evaluates the problem's last tile, i.e. never while a role still has a tile of it ahead).
  // hh: one pass for a second-order product (a4 / p2, KIND_F16X2), taken from the Err[n] that a2 of this iteration wrote
  // for this problem (a completed kernel: visible), so issuer and epilogues of both CTAs agree.  (n_iter < 0, loop body
  // of a zfac_graph: the update is taken from the last residual written, State::iters.)
  auto decode_local = [&](int t, int& m0, int& n0, bool& offdiag) {
    int I, J;
    if (SYM) {
      const int macro = t / NSPLIT, sub = t - macro * NSPLIT;
      tri_decode(macro, I, J);
      n0 = J * UM_MACRO + sub * TN;
      offdiag = (I != J);
    } else {
      band_decode(t, TI, JC, p.band * NSPLIT, I, J);
      I += p.ioff;
      J += p.joff;
      n0 = J * TN;
      offdiag = true;                                      // (unused by the full-output epilogues)
    }
    m0 = I * UM_TILE_M;
  };
  auto decode = [&](int t, int& m0, int& n0, int& mb, int& tl, bool& offdiag, bool& hh) -> bool {
    const int b = t / tiles_pp;
    tl = t - b * tiles_pp;
    if (p.batch > 1 && *((volatile int*)&p.st[b].done)) return false;
    decode_local(tl, m0, n0, offdiag);
    mb = b * np;
    m0 += mb;
    hh = false;
    if (PAIRK && p.hh_only)
      hh = __ldcg(p.stop.d_err + (size_t)b * p.stop.err_stride + (p.stop.n_iter >= 0 ? p.stop.n_iter : p.st[b].iters)) <= p.hh_err_max;
    return true;
  };

  if (warp < UM_EPI_WARP0) {
  reg_dealloc<UM_REGS_CONTROL>();
  if (threadIdx.x == 0) {
    for (int s = 0; s < KT::STAGES; ++s) { mbar_init(full_bar(s), 1); mbar_init(empty_bar(s), 1); }
    for (int b = 0; b < 2; ++b) {                  // arrivals: the warps of both CTAs that read the set
      mbar_init(tfull_bar(b), 1); mbar_init(tempty_bar(b), 2 * UM_EPI_WARPS / SETS);
      mbar_init(hh_full_bar(b), 1); mbar_init(hh_empty_bar(b), 2 * UM_EPI_WARPS / SETS);
    }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    asm volatile("prefetch.tensormap [%0];" ::"l"(reinterpret_cast<uint64_t>(&p.mapA)) : "memory");
    asm volatile("prefetch.tensormap [%0];" ::"l"(reinterpret_cast<uint64_t>(&p.mapB)) : "memory");
  }
  if (warp == 1) {
    asm volatile("tcgen05.alloc.cta_group::2.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(tmem_slot), "r"(UM_TMEM_COLS) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::2.sync.aligned;" ::: "memory");
  }
  const uint32_t tmem_base = pair_sync_in();
  const int num_tiles = live_tiles();
  if (warp == 0) {
    // ===================================================== TMA producer (both CTAs)
    if (lane == 0) {
      int stage = 0; uint32_t phase = 0;
      const int aoff = (int)rank * UM_ROWS, boff = (int)rank * (TN / 2);
      for (int t = pair; t < num_tiles; t += num_pairs) {
        int m0, n0, mb, tl; bool od, hh_only;
        if (!decode(t, m0, n0, mb, tl, od, hh_only)) continue;
        n0 += mb;                                              // B operand rows of this problem
        for (int kb = 0; kb < KB; ++kb) {
          mbar_wait(empty_bar(stage), phase ^ 1u);
          // one-pass tile of the pair kind (hh_only): the lo' planes are never read -- do not load them
          const int narr = hh_only ? 1 : KT::ARRAYS;
          if (rank == 0) mbar_expect_tx(full_bar(stage), 2u * (uint32_t)narr * (UM_A_BYTES + B_BYTES));   // both CTAs' boxes
          const uint32_t lead_full = mapa_u32(full_bar(stage), 0);
          const uint32_t sa = smem_base + stage * STAGE_BYTES;
          const uint32_t sb = sa + KT::ARRAYS * UM_A_BYTES;
          const int kc = kb * KT::BK_ELEMS;
#pragma unroll
          for (int a = 0; a < KT::ARRAYS; ++a) {
            if (a >= narr) break;
#pragma unroll
            for (int b = 0; b < UM_ROWS / UM_BOX_ROWS; ++b)
              tma_load_2d_pair(sa + a * UM_A_BYTES + b * UM_BOX_BYTES, &p.mapA, kc, a * p.rows + m0 + aoff + b * UM_BOX_ROWS, lead_full);
#pragma unroll
            for (int b = 0; b < TN / 2 / UM_BOX_ROWS; ++b)
              tma_load_2d_pair(sb + a * B_BYTES + b * UM_BOX_BYTES, &p.mapB, kc, a * p.rows + n0 + boff + b * UM_BOX_ROWS, lead_full);
          }
          if (++stage == KT::STAGES) { stage = 0; phase ^= 1u; }
        }
      }
    }
  } else if (warp == 1) {
    // ===================================================== MMA issuer (leader CTA, one lane)
    if (rank == 0 && lane == 0) {
      // tile li of this pair uses accumulator set li & 1 and is that set's (li >> 1)-th tile: the phase parities
      // of the per-set barriers follow from li alone
#ifdef ZFAC_TIMING
      long long twait[4] = {0, 0, 0, 0};
      const long long tstart = clock64();
#endif
      if (PAIRK) {
        // (h)(h) products go to D_hh, the 2^11-scaled cross products (h)(l') + (l')(h) to D_x.  D_hh is handed to
        // the epilogue warps every CH k-blocks (promoted accumulation).  Issue order of a chunk of
        // c k-blocks (H = 4 (h)(h) MMAs, C = 8 cross MMAs of one k-block; FRONT = BACK = 1 with 3 stages):
        //     C0 | wait(D_hh drained) | H0 | H1 C1 ... | H(c-1) | commit(D_hh full) | C(c-1)
        // so that the cross products of 2 k-blocks (16 MMAs, 2048 cycles) cover the drain of D_hh between chunks.
        // The FIRST chunk of a tile is CH0 >= CH k-blocks long: while it runs, the epilogue warps still store
        // the previous tile from registers (they released the tensor memory first), and its partial sums are
        // small, so the truncation of the FP32 accumulator costs the least there.
        constexpr int FRONT = (KT::STAGES >= 4) ? 2 : 1, BACK = FRONT;
        uint32_t it = 0;                                       // k-block sequence number = position in the smem ring
        int li = -1;                                           // tiles of this pair that are processed (skipped ones do not count)
        for (int t = pair; t < num_tiles; t += num_pairs) {
          int m0_, n0_, mb_, tl_; bool od_, hh_only;
          if (!decode(t, m0_, n0_, mb_, tl_, od_, hh_only)) continue;
          ++li;
          const int set = (SETS == 2) ? (li & 1) : 0;
          const uint32_t nuse = (SETS == 2) ? (uint32_t)(li >> 1) : (uint32_t)li;   // earlier tiles of this set
          const uint32_t d0 = tmem_base + set * SET_COLS, d1 = d0 + TN;
          ZF_TWAIT(2, mbar_wait(tempty_bar(set), (nuse & 1u) ^ 1u));
          tc_fence_after();
          uint32_t xacc = 0u;
          uint32_t hch = nuse * (uint32_t)NCH;                 // chunks committed into this set so far
          auto ring = [&](int j, uint32_t& st, uint32_t& ph) {
            const uint32_t x = it + (uint32_t)j;
            st = x % (uint32_t)KT::STAGES; ph = (x / (uint32_t)KT::STAGES) & 1u;
          };
          auto sdescs = [&](int j, uint64_t& a_hi, uint64_t& a_lo, uint64_t& b_hi, uint64_t& b_lo) {
            uint32_t st, ph; ring(j, st, ph);
            const uint32_t sa = smem_base + st * STAGE_BYTES;
            a_hi = make_sdesc(sa); a_lo = make_sdesc(sa + UM_A_BYTES);
            b_hi = make_sdesc(sa + 2 * UM_A_BYTES); b_lo = make_sdesc(sa + 2 * UM_A_BYTES + B_BYTES);
          };
          auto wait_full = [&](int j) {
            uint32_t st, ph; ring(j, st, ph);
            ZF_TWAIT(0, mbar_wait(full_bar(st), ph));
            tc_fence_after();
          };
          auto issue_cross = [&](int j) {
            if (hh_only) return;                               // second-order product (a4 / p2): (h)(h) pass only
            uint64_t a_hi, a_lo, b_hi, b_lo; sdescs(j, a_hi, a_lo, b_hi, b_lo);
#pragma unroll
            for (int k = 0; k < KSTEPS; ++k) {
              const uint64_t ko = (uint64_t)(k * 2);           // 32 bytes per k-step, in 16-byte units
              tc_mma_pair<KIND>(d1, a_hi + ko, b_lo + ko, IDESC, xacc);
              xacc = 1u;
              tc_mma_pair<KIND>(d1, a_lo + ko, b_hi + ko, IDESC, 1u);
            }
          };
          auto issue_hh = [&](int j, bool fresh) {
            uint64_t a_hi, a_lo, b_hi, b_lo; sdescs(j, a_hi, a_lo, b_hi, b_lo);
#pragma unroll
            for (int k = 0; k < KSTEPS; ++k)
              tc_mma_pair<KIND>(d0, a_hi + (uint64_t)(k * 2), b_hi + (uint64_t)(k * 2), IDESC, (fresh && k == 0) ? 0u : 1u);
          };
          auto release = [&](int j) {                          // frees the stage in both CTAs when its MMAs retire
            uint32_t st, ph; ring(j, st, ph);
            tc_commit_pair(empty_bar(st));
          };
          for (int kb0 = 0; kb0 < KB;) {
            const int want = (kb0 == 0) ? CH0 : CH;
            const int c = (KB - kb0 < want) ? (KB - kb0) : want;
            const int f = c < FRONT ? c : FRONT;
            const int b = (c - f) < BACK ? (c - f) : BACK;
            for (int j = 0; j < f; ++j) { wait_full(j); issue_cross(j); }
            ZF_TWAIT(1, mbar_wait(hh_empty_bar(set), (hch & 1u) ^ 1u));
            tc_fence_after();
            for (int j = 0; j < f; ++j) { issue_hh(j, j == 0); release(j); }
            for (int j = f; j < c - b; ++j) { wait_full(j); issue_hh(j, false); issue_cross(j); release(j); }
            for (int j = c - b; j < c; ++j) { wait_full(j); issue_hh(j, false); }
            tc_commit_pair(hh_full_bar(set)); ++hch;
            for (int j = c - b; j < c; ++j) { issue_cross(j); release(j); }
            it += (uint32_t)c;
            kb0 += c;
          }
          tc_commit_pair(tfull_bar(set));                      // D_x complete, both CTAs
        }
      } else {
        int stage = 0; uint32_t phase = 0;
        int li = -1;
        for (int t = pair; t < num_tiles; t += num_pairs) {
          int m0_, n0_, mb_, tl_; bool od_, hh_;
          if (!decode(t, m0_, n0_, mb_, tl_, od_, hh_)) continue;
          ++li;
          const int set = (SETS == 2) ? (li & 1) : 0;
          const uint32_t nuse = (SETS == 2) ? (uint32_t)(li >> 1) : (uint32_t)li;
          const uint32_t d0 = tmem_base + set * SET_COLS;
          ZF_TWAIT(2, mbar_wait(tempty_bar(set), (nuse & 1u) ^ 1u));
          tc_fence_after();
          for (int kb = 0; kb < KB; ++kb) {
            ZF_TWAIT(0, mbar_wait(full_bar(stage), phase));
            tc_fence_after();
            const uint32_t sa = smem_base + stage * STAGE_BYTES;
            const uint64_t ad = make_sdesc(sa), bd = make_sdesc(sa + UM_A_BYTES);
#pragma unroll
            for (int k = 0; k < KSTEPS; ++k)                   // 32 bytes per k-step, in 16-byte units
              tc_mma_pair<KIND>(d0, ad + (uint64_t)(k * 2), bd + (uint64_t)(k * 2), IDESC, (kb | k) ? 1u : 0u);
            tc_commit_pair(empty_bar(stage));                  // frees the smem stage in both CTAs when the MMAs retire
            if (++stage == KT::STAGES) { stage = 0; phase ^= 1u; }
          }
          tc_commit_pair(tfull_bar(set));                      // accumulator complete, both CTAs
        }
      }
#ifdef ZFAC_TIMING
      if (p.dbg) {
        twait[3] = clock64() - tstart;
        for (int i = 0; i < 4; ++i) atomicAdd(p.dbg + (size_t)(EPI * 148 + pair) * 8 + i, (unsigned long long)twait[i]);
      }
#endif
    }
  }
  pair_sync_out();
  if (warp == 1) {
    tc_fence_after();
    asm volatile("tcgen05.dealloc.cta_group::2.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "r"(UM_TMEM_COLS) : "memory");
  }
  } else {
    reg_alloc<UM_REGS_EPILOGUE>();
    const uint32_t tmem_base = pair_sync_in();
    const int num_tiles = live_tiles();
    // ===================================================== epilogue warps (4 .. 11), both CTAs
    // Group g = warps 4 + 4 g .. 7 + 4 g (one warp per TMEM lane quarter).  SETS == 2: group g owns accumulator
    // set g, i.e. the tiles with local index li = g (mod 2), all TN columns: its stores overlap the other set's
    // mainloop.  SETS == 1: both groups work on every tile, group g on columns [g TN/2, (g + 1) TN/2).
    const int q = warp & 3;                                    // TMEM lane quarter this warp may read
    const int g = (warp - UM_EPI_WARP0) >> 2;
    const int set = (SETS == 2) ? g : 0;
    const int col0 = (SETS == 2) ? 0 : g * GCOLS;              // first column of the tile handled by this thread
    const int row = (int)rank * UM_ROWS + q * 32 + lane;       // row of the pair tile held by this thread
    const uint32_t lead_hh_empty = mapa_u32(hh_empty_bar(set), 0), lead_tempty = mapa_u32(tempty_bar(set), 0);
    const uint32_t tbase = tmem_base + ((uint32_t)(q * 32) << 16) + set * SET_COLS + col0;
    int li = -1;
#ifdef ZFAC_TIMING
    long long twait[4] = {0, 0, 0, 0};     // 4 wait for MMA (hh_full / tfull), 5 TMEM -> registers, 6 global loads / stores
#endif
    for (int t = pair; t < num_tiles; t += num_pairs) {
      int m0, n0, mb, tl; bool offdiag, hh_only;
      if (!decode(t, m0, n0, mb, tl, offdiag, hh_only)) continue;
      ++li;
      if (SETS == 2 && (li & 1) != g) continue;
      const uint32_t tuse = (SETS == 2) ? (uint32_t)(li >> 1) : (uint32_t)li;   // tiles this thread has finished
      const int m = m0 + row;
      double tile_sumsq = 0.0, first_half_sumsq = 0.0;
      if (PAIRK) {
        uint32_t hcnt = tuse * (uint32_t)NCH;                  // chunks drained from this set so far
        float sum[GCOLS];
#pragma unroll
        for (int j = 0; j < GCOLS; ++j) sum[j] = 0.0f;
        for (int c = 0; c < NCH; ++c) {
          ZF_TWAIT(0, mbar_wait(hh_full_bar(set), hcnt & 1u));
          tc_fence_after();
          // DRAIN_W columns per tcgen05.ld; the chunk is handed back (arrive) as soon as its last columns are in registers,
          // BEFORE they are added: the drain is on the critical path of the next chunk's (h)(h) MMAs
          constexpr int DRAIN_W = ZFAC_DRAIN_W;
#pragma unroll
          for (int i = 0; i < GCOLS / DRAIN_W; ++i) {
            uint32_t r[DRAIN_W];
            tmem_ld(tbase + i * DRAIN_W, r);
            tmem_ld_wait();
            if (i == GCOLS / DRAIN_W - 1) {
              tc_fence_before();
              __syncwarp();
              mbar_arrive_cluster_lane0(lead_hh_empty, lane);
            }
#pragma unroll
            for (int j = 0; j < DRAIN_W; ++j) sum[i * DRAIN_W + j] += __uint_as_float(r[j]);
          }
          ++hcnt;
        }
        // D_hh + 2^-11 D_x into registers, then hand the tensor memory back BEFORE the global loads / stores:
        // the next tile's MMAs run while this tile is written out.
        ZF_TWAIT(0, mbar_wait(tfull_bar(set), tuse & 1u));
        tc_fence_after();
#ifdef ZFAC_TIMING
        const long long te0 = clock64();
#endif
        if (!hh_only) {
#pragma unroll
          for (int i = 0; i < GCOLS / 32; ++i) {
            uint32_t x[32];
            tmem_ld(tbase + TN + i * 32, x);
            tmem_ld_wait();
#pragma unroll
            for (int j = 0; j < 32; ++j) sum[i * 32 + j] += __uint_as_float(x[j]) * LO_UNSCALE;
          }
        }
        tc_fence_before();
        __syncwarp();
        mbar_arrive_cluster_lane0(lead_tempty, lane);
        // ptxas is free to sink a relaxed arrive below the (independent) global loads / stores that follow, which
        // would give the tensor memory back only after the tile is written; a CTA-scope fence pins it here.
        asm volatile("fence.acq_rel.cta;" ::: "memory");
#ifdef ZFAC_TIMING
        const long long te1 = clock64();
#endif
#pragma unroll
        for (int cc = 0; cc < GCOLS / SUB; ++cc) {
          float v[SUB];
#pragma unroll
          for (int j = 0; j < SUB; ++j) v[j] = sum[cc * SUB + j];
          epilogue_cols<KIND, EPI, SUB>(p, v, m, n0 + col0 + cc * SUB, mb, offdiag, tile_sumsq);
        }
#ifdef ZFAC_TIMING
        twait[1] += te1 - te0; twait[2] += clock64() - te1;
#endif
      } else {
        mbar_wait(tfull_bar(set), tuse & 1u);
        tc_fence_after();
#pragma unroll 1
        for (int cc = 0; cc < GCOLS / SUB; ++cc) {
          float v[SUB];
          {
            uint32_t r[SUB];
            tmem_ld(tbase + cc * SUB, r);
            tmem_ld_wait();
#pragma unroll
            for (int j = 0; j < SUB; ++j) v[j] = __uint_as_float(r[j]);
          }
          // a2 on a 256-column tile: one partial sum per 128-column half (as the 128-column kinds form them)
          if (EPI == EPI_A2 && GCOLS == 256 && cc == GCOLS / SUB / 2) { first_half_sumsq = tile_sumsq; tile_sumsq = 0.0; }
          epilogue_cols<KIND, EPI, SUB>(p, v, m, n0 + col0 + cc * SUB, mb, offdiag, tile_sumsq);
        }
        tc_fence_before();
        __syncwarp();
        mbar_arrive_cluster_lane0(lead_tempty, lane);            // frees the accumulator set
      }
      // step a3: this warp's share of the tile (slot: CTA of the pair x warp of the tile's epilogue group(s))
      if (EPI == EPI_A2) {
        // One sum per warp and 128-column half of a 256 x 256 macro tile, stored at (macro tile, CTA, column half, lane
        // quarter): 16 per macro tile whatever the kind's tile width and accumulator sets, formed from the same elements in
        // the same order -- Err[] does not depend on the tile width (ZFAC_OPT_NARROW_TILES).
        const int macro = kind_is_narrow(KIND) ? (tl >> 1) : tl;
        const int base = macro * 16 + (int)rank * 8 + q;
        if (GCOLS == 256) {                                    // one-pass kinds on 256-column tiles: this thread holds both halves
          stop_test_index_warp(p.stop, mb / np, base, offdiag ? 2.0 * first_half_sumsq : first_half_sumsq, lane);
          stop_test_index_warp(p.stop, mb / np, base + 4, offdiag ? 2.0 * tile_sumsq : tile_sumsq, lane);
        } else {
          const int half = kind_is_narrow(KIND) ? (tl & 1) : g;   // F16X2 on 256 columns: group g holds columns [128 g, 128 g + 128)
          stop_test_index_warp(p.stop, mb / np, base + half * 4, offdiag ? 2.0 * tile_sumsq : tile_sumsq, lane);
        }
      }
    }
#ifdef ZFAC_TIMING
    if (p.dbg && rank == 0 && warp == UM_EPI_WARP0 && lane == 0)
      for (int i = 0; i < 3; ++i) atomicAdd(p.dbg + (size_t)(EPI * 148 + pair) * 8 + 4 + i, (unsigned long long)twait[i]);
#endif
    pair_sync_out();
  }
}

// ------------------------------------------------------------------ host side
typedef CUresult (*PFN_encodeTiled)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                    const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                    CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

struct UmmaPlan {
  Layout L;
  char* ws = nullptr;
  int max_pairs = 0;  // CTA pairs that are co-resident on the device (74 on a B200)
  int mode = 0;
  const Options* opt = nullptr;   // the context's options (zfac_set_option): chunk lengths, band, one-pass a4, max_pairs
  int pairs() const { return (opt->max_pairs > 0 && opt->max_pairs < max_pairs) ? opt->max_pairs : max_pairs; }
  // tensor maps of every operand buffer (box 128 B x 64 rows, 128B swizzle)
  CUtensorMap mS, mW, mT, mR, mQ, mZ[2];
};

inline cudaError_t make_map(PFN_encodeTiled enc, CUtensorMap* m, void* base, CUtensorMapDataType dt, size_t elt,
                            uint64_t rows, uint64_t cols) {
  cuuint64_t gdim[2] = {cols, rows};
  cuuint64_t gstr[1] = {cols * elt};
  cuuint32_t box[2] = {(cuuint32_t)(UM_ROWB / elt), (cuuint32_t)UM_BOX_ROWS};
  cuuint32_t estr[2] = {1u, 1u};
  CUresult r = enc(m, dt, 2, base, gdim, gstr, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B,
                   CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  return r == CUDA_SUCCESS ? cudaSuccess : cudaErrorInvalidValue;
}

template <int KIND, int EPI>
inline cudaError_t prepare_kernel(int* max_pairs, int sm_count) {
  cudaError_t e = cudaFuncSetAttribute(umma_gemm_kernel<KIND, EPI>, cudaFuncAttributeMaxDynamicSharedMemorySize, UM_SMEM_BYTES);
  if (e != cudaSuccess) return e;
  cudaLaunchConfig_t cfg{};
  cfg.gridDim = dim3(2 * (sm_count / 2)); cfg.blockDim = dim3(UM_THREADS); cfg.dynamicSmemBytes = UM_SMEM_BYTES;
  int nc = 0;
  e = cudaOccupancyMaxActiveClusters(&nc, umma_gemm_kernel<KIND, EPI>, &cfg);
  if (e != cudaSuccess) return e;
  if (nc < 1) {
    cudaFuncAttributes fa;
    cudaFuncGetAttributes(&fa, umma_gemm_kernel<KIND, EPI>);
    fprintf(stderr, "zfac: kernel<%d,%d> does not fit an SM pair: regs=%d threads=%d static smem=%zu dyn smem=%d\n",
            KIND, EPI, fa.numRegs, UM_THREADS, fa.sharedSizeBytes, UM_SMEM_BYTES);
    return cudaErrorLaunchOutOfResources;
  }
  if (*max_pairs == 0 || nc < *max_pairs) *max_pairs = nc;
  return cudaSuccess;
}

template <int KIND>
inline cudaError_t prepare_kind(int* max_pairs, int sm_count) {
  cudaError_t e;
  if ((e = prepare_kernel<KIND, EPI_A1>(max_pairs, sm_count)) != cudaSuccess) return e;
  if ((e = prepare_kernel<KIND, EPI_A2>(max_pairs, sm_count)) != cudaSuccess) return e;
  if ((e = prepare_kernel<KIND, EPI_X3>(max_pairs, sm_count)) != cudaSuccess) return e;
  if ((e = prepare_kernel<KIND, EPI_A4>(max_pairs, sm_count)) != cudaSuccess) return e;
  if ((e = prepare_kernel<KIND, EPI_P2>(max_pairs, sm_count)) != cudaSuccess) return e;
  return prepare_kernel<KIND, EPI_A5>(max_pairs, sm_count);
}

inline cudaError_t umma_plan_create(UmmaPlan* pl, const Layout& L, char* ws, int sm_count, const Options* opt) {
  pl->L = L; pl->ws = ws; pl->mode = L.mode; pl->max_pairs = 0; pl->opt = opt;
  void* fn = nullptr;
  cudaDriverEntryPointQueryResult qres;
  cudaError_t e = cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres);
  if (e != cudaSuccess) return e;
  if (!fn || qres != cudaDriverEntryPointSuccess) return cudaErrorNotSupported;
  PFN_encodeTiled enc = reinterpret_cast<PFN_encodeTiled>(fn);
  const uint64_t np = (uint64_t)L.np;
  if (L.mode == ZFAC_MODE_SPLIT16 || L.mode == ZFAC_MODE_HH16) {
    const CUtensorMapDataType H = CU_TENSOR_MAP_DATA_TYPE_FLOAT16;
    const uint64_t rows = (L.mode == ZFAC_MODE_SPLIT16 ? 2 : 1) * (uint64_t)L.rows;
    if ((e = make_map(enc, &pl->mS, ws + L.off_S, H, 2, rows, np)) != cudaSuccess) return e;
    if ((e = make_map(enc, &pl->mW, ws + L.off_W, H, 2, rows, np)) != cudaSuccess) return e;
    if ((e = make_map(enc, &pl->mT, ws + L.off_T, H, 2, rows, np)) != cudaSuccess) return e;
    if ((e = make_map(enc, &pl->mR, ws + L.off_Rb, H, 2, rows, np)) != cudaSuccess) return e;
    if ((e = make_map(enc, &pl->mQ, ws + L.off_Qb, H, 2, rows, np)) != cudaSuccess) return e;
    if ((e = make_map(enc, &pl->mZ[0], ws + L.off_Zb[0], H, 2, rows, np)) != cudaSuccess) return e;
    if ((e = make_map(enc, &pl->mZ[1], ws + L.off_Zb[1], H, 2, rows, np)) != cudaSuccess) return e;
    e = (L.mode == ZFAC_MODE_SPLIT16) ? prepare_kind<KIND_F16X2>(&pl->max_pairs, sm_count) : prepare_kind<KIND_HH16>(&pl->max_pairs, sm_count);
    if (e != cudaSuccess) return e;
    e = (L.mode == ZFAC_MODE_SPLIT16) ? prepare_kind<KIND_F16X2N>(&pl->max_pairs, sm_count) : prepare_kind<KIND_HH16N>(&pl->max_pairs, sm_count);
    if (e != cudaSuccess) return e;
  } else {
    const CUtensorMapDataType F = CU_TENSOR_MAP_DATA_TYPE_FLOAT32;
    const uint64_t rows = (uint64_t)L.rows;
    if ((e = make_map(enc, &pl->mS, ws + L.off_S, F, 4, rows, np)) != cudaSuccess) return e;
    if ((e = make_map(enc, &pl->mW, ws + L.off_W, F, 4, rows, np)) != cudaSuccess) return e;
    if ((e = make_map(enc, &pl->mT, ws + L.off_T, F, 4, rows, np)) != cudaSuccess) return e;
    if ((e = make_map(enc, &pl->mR, ws + L.off_R, F, 4, rows, np)) != cudaSuccess) return e;
    if ((e = make_map(enc, &pl->mQ, ws + L.off_Q, F, 4, rows, np)) != cudaSuccess) return e;
    if ((e = make_map(enc, &pl->mZ[0], ws + L.off_Z[0], F, 4, rows, np)) != cudaSuccess) return e;
    if ((e = make_map(enc, &pl->mZ[1], ws + L.off_Z[1], F, 4, rows, np)) != cudaSuccess) return e;
    if ((e = prepare_kind<KIND_TF32>(&pl->max_pairs, sm_count)) != cudaSuccess) return e;
    if ((e = prepare_kind<KIND_TF32N>(&pl->max_pairs, sm_count)) != cudaSuccess) return e;
  }
  if (pl->max_pairs > sm_count / 2) pl->max_pairs = sm_count / 2;
  return cudaSuccess;
}

// The mode's kind on 256 x 128 tiles (KIND_F16X2N / HH16N / TF32N)?  ZFAC_OPT_NARROW_TILES: 0 never, 1 always, -1 (default) when the full GEMMs of
// the launch have at most 37 wide tiles (one problem of N <= 1536, or a few smaller ones): the narrow ones then still fit
// the 74 CTA pairs in one wave.  Larger launches have tiles enough (measured: no gain, a loss from N = 2048 on).
inline bool umma_narrow(const UmmaPlan& pl) {
  if (pl.opt->narrow_tiles >= 0) return pl.opt->narrow_tiles != 0;
  const long T = (long)(pl.L.np / UM_MACRO);
  return (long)pl.L.batch * T * T <= 37;
}

// pdl: launch with cudaLaunchAttributeProgrammaticStreamSerialization (see the head of the kernel)
template <int KIND, int EPI>
inline void umma_launch_one(int grid, cudaStream_t s, const UmmaParams& p, bool pdl) {
  if (!pdl) { umma_gemm_kernel<KIND, EPI><<<grid, UM_THREADS, UM_SMEM_BYTES, s>>>(p); return; }
  cudaLaunchConfig_t cfg{};
  cfg.gridDim = dim3((unsigned)grid); cfg.blockDim = dim3(UM_THREADS); cfg.dynamicSmemBytes = UM_SMEM_BYTES; cfg.stream = s;
  cudaLaunchAttribute at[1];
  at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  at[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = at; cfg.numAttrs = 1;
  cudaLaunchKernelEx(&cfg, umma_gemm_kernel<KIND, EPI>, p);
}
template <int KIND>
inline void umma_launch(int epi, int grid, cudaStream_t s, const UmmaParams& p, bool pdl = false) {
  switch (epi) {
    case EPI_A1: umma_launch_one<KIND, EPI_A1>(grid, s, p, pdl); break;
    case EPI_A2: umma_launch_one<KIND, EPI_A2>(grid, s, p, pdl); break;
    case EPI_X3: umma_launch_one<KIND, EPI_X3>(grid, s, p, pdl); break;
    case EPI_A4: umma_launch_one<KIND, EPI_A4>(grid, s, p, pdl); break;
    case EPI_P2: umma_launch_one<KIND, EPI_P2>(grid, s, p, pdl); break;
    case EPI_A5X:
      if (KIND == KIND_F16X2) umma_launch_one<KIND_F16X2, EPI_A5X>(grid, s, p, pdl);
      break;                                               // (FP64-master modes: wide tiles only)
    default:     umma_launch_one<KIND, EPI_A5>(grid, s, p, pdl); break;
  }
}
inline void umma_launch_mode(int mode, int epi, int grid, cudaStream_t s, const UmmaParams& p, bool narrow = false, bool pdl = false) {
  if (mode == ZFAC_MODE_SPLIT16) { if (narrow) umma_launch<KIND_F16X2N>(epi, grid, s, p, pdl); else umma_launch<KIND_F16X2>(epi, grid, s, p, pdl); }
  else if (mode == ZFAC_MODE_HH16) { if (narrow) umma_launch<KIND_HH16N>(epi, grid, s, p, pdl); else umma_launch<KIND_HH16>(epi, grid, s, p, pdl); }
  else { if (narrow) umma_launch<KIND_TF32N>(epi, grid, s, p, pdl); else umma_launch<KIND_TF32>(epi, grid, s, p, pdl); }
}

// The two halves of one iteration as the host enqueues them.  The only dependence on the iteration index n is (i) the
// index of the Err[] entry a2 writes and a4 reads -- `n_stop`, or -1 = "take it from State::iters on the device" -- and
// (ii) the parity of n, which selects the Z operand buffers.  zfac_refine loops over (residual, update); a zfac_graph
// puts update(0), residual, update(1), residual into the body of a WHILE node (fixed kernel parameters, hence the
// parity-unrolled body and the device-side index).
struct UmmaSeq {
  const UmmaPlan& pl;
  UmmaParams p{};
  int grid_full = 0, grid_sym = 0, order = 2, nl = 0;
  bool h16 = false;
  float* R32 = nullptr;

  UmmaSeq(const UmmaPlan& pl_, int max_iter, int stop, int order_, double* d_err, unsigned long long cond) : pl(pl_) {
    const Layout& L = pl.L;
    char* ws = pl.ws;
    const int T = (int)(L.np / UM_MACRO);
    narrow = umma_narrow(pl);
    // measured (10 updates, off / on / on with the early set-up): HH16 N = 512 / 1024 0.64 / 0.53 / 0.50 and 0.74 / 0.64 / 0.61 ms,
    // N = 2048 1.25 / 1.16 ms, a tie at N = 3072, TF32 alike; SPLIT16 N = 512 / 1024 0.93 / 0.92 / 0.88 and 1.19 / 1.19 / 1.15 ms,
    // +-1.5 % beyond; a launch behind the stop costs 1.4 .. 1.9 us instead of 2.7 .. 4.2 us, which decides for runs that stop well
    // before max_iter (SPLIT16 N = 2048 to its stop, max_iter = 40: 2.47 -> 2.2 ms)
    const bool small = (long)L.batch * T * T <= 37;
    // N = 4096 / 8192: the working kernels within the noise, calls that stop well before max_iter -1.3 % -> every single problem
    pdl = (cond == 0ull) && (pl.opt->pdl >= 0 ? pl.opt->pdl != 0 : (small || L.batch == 1));   // (batched, not small: -4 % measured)
    p.early = (pdl && pl.opt->pdl != 2 && small) ? 1 : 0;      // small launches: set-up ahead of the wait
    const int nsplit = narrow ? 2 : 1;                       // 256 / TILE_N of the kind that runs
    const int full_tiles = T * T * nsplit * L.batch, sym_tiles = T * (T + 1) / 2 * nsplit * L.batch;
    grid_full = 2 * (full_tiles < pl.pairs() ? full_tiles : pl.pairs());
    grid_sym = 2 * (sym_tiles < pl.pairs() ? sym_tiles : pl.pairs());
    order = order_;
    nsplit_ = nsplit;
    p.np = (int)L.np; p.batch = L.batch; p.rows = (int)L.rows; p.macro_tiles = T; p.band = pl.opt->band;
    p.st = reinterpret_cast<State*>(ws + L.off_state);
#ifdef ZFAC_TIMING
    p.dbg = reinterpret_cast<unsigned long long*>(ws + L.off_dbg);
#endif
    p.stop.st = p.st; p.stop.partials = reinterpret_cast<double*>(ws + L.off_partials);
    p.stop.num_partials = 0; p.stop.d_err = d_err; p.stop.max_iter = max_iter; p.stop.stop = stop;
    p.stop.order = order; p.stop.cond = cond;
    p.stop.tiles_pp = T * (T + 1) / 2 * nsplit; p.stop.err_stride = (long long)max_iter + 1;
    p.stop.slots_pt = 16 / nsplit;                           // a2: 16 partial sums per 256 x 256 macro tile (see the epilogue)
    const PolyCoef pc = poly_coef(order);
    p.q_r = (float)pc.q_r; p.q_d = (float)pc.q_d; p.g_i = (float)pc.g_i; p.g_r = (float)pc.g_r; p.g_p = (float)pc.g_p;
    R32 = reinterpret_cast<float*>(ws + L.off_R);
    h16 = (L.mode != ZFAC_MODE_TF32);
  }

  int nsplit_ = 1;
  bool narrow = false;
  bool pdl = false;            // programmatic dependent launch of the GEMM kernels (not inside a captured graph)

  // a1 restricted to the macro-tile columns [mc0, mc0 + mcn) of T, i.e. to the rows [256 mc0, 256 (mc0 + mcn)) of S
  // (mcn = 0: all of T).  Tiles do not overlap between bands, so a banded a1 is bit-identical to the full launch.
  void a1(int mc0, int mcn, cudaStream_t s) {
    const Layout& L = pl.L;
    char* ws = pl.ws;
    p.hh_only = 0;
    p.chunk_kb = pl.opt->chunk_kb; p.chunk0_kb = pl.opt->chunk0_kb;
    p.mapA = pl.mW; p.mapB = pl.mS; p.f32_in = nullptr; p.h_out_t = nullptr;
    if (h16) { p.f32_out = nullptr; p.h_out = ws + L.off_T; }
    else { p.f32_out = reinterpret_cast<float*>(ws + L.off_T); p.h_out = nullptr; }
    int grid = grid_full;
    if (mcn > 0) {
      p.joff = mc0 * nsplit_; p.jcols = mcn * nsplit_;
      const int tiles = p.macro_tiles * p.jcols;
      grid = 2 * (tiles < pl.pairs() ? tiles : pl.pairs());
    }
    umma_launch_mode(L.mode, EPI_A1, grid, s, p, narrow, pdl);
    p.joff = 0; p.jcols = 0;
    nl += 1;
  }

  // a1 + a2 (+ a3): residual number n_stop (-1: device-side index); skip_a1: a1 was already enqueued band by band
  void residual(int n_stop, int tagn, cudaStream_t s, Prof* prof, bool skip_a1 = false) {
    const Layout& L = pl.L;
    char* ws = pl.ws;
    // a1: T = W S^T            (promoted accumulation: T and X are O(1) quantities)
    if (prof) prof->mark(s, EPI_A1 + 16 * tagn);
    if (!skip_a1) a1(0, 0, s);
    p.hh_only = 0; p.f32_in = nullptr; p.h_out_t = nullptr;
    p.chunk_kb = pl.opt->chunk_kb; p.chunk0_kb = pl.opt->chunk0_kb;
    // a2: R = I - W T^T
    if (prof) prof->mark(s, EPI_A2 + 16 * tagn);
    p.mapA = pl.mW; p.mapB = pl.mT; p.f32_out = R32; p.stop.n_iter = n_stop;
    // a2 writes four outputs per element: its stores take twice as long, so a long first chunk (if one is set) doubles
    if (pl.opt->chunk0_kb > pl.opt->chunk_kb) p.chunk0_kb = 2 * pl.opt->chunk0_kb;
    p.h_out = h16 ? ws + L.off_Rb : nullptr;
    umma_launch_mode(L.mode, EPI_A2, grid_sym, s, p, narrow, pdl);
    nl += 1;
    if (p.stop.cond) graph_cond_kernel<<<1, 1, 0, s>>>(p.st, p.stop.cond);       // zfac_graph_*: loop condition
  }

  // (p2,) a4, a5: update number n with n & 1 = par, taken from residual n_stop (-1: device-side index)
  // hook + bands > 1: a5 runs in `bands` launches over whole macro-tile rows; after each, hook->after_a5_band is told
  // which rows of Z_next are final (disjoint whole tiles: bit-identical to the single launch)
  void update(int par, int n_stop, int tagn, cudaStream_t s, Prof* prof, const IterHook* hook = nullptr, int bands = 1) {
    const Layout& L = pl.L;
    char* ws = pl.ws;
    p.stop.n_iter = n_stop;
    // a4: Q = 1/2 R + 3/8 R R^T   (the product is a correction of size |R|^2: no promotion needed)
    if (pl.opt->promote_update) { p.chunk_kb = pl.opt->chunk_kb; p.chunk0_kb = pl.opt->chunk0_kb; }
    else { p.chunk_kb = 0; p.chunk0_kb = 0; }
    p.hh_only = (L.mode == ZFAC_MODE_SPLIT16 && pl.opt->hh_square) ? 1 : 0;      // p2 and a4 only; a5 below needs all passes
    p.hh_err_max = pl.opt->hh_square_err;
    if (order > 2) {
      // order m > 2 (zfac.h, zfac_set_order): P = R R^T -> T buffer (free between a2 and the next a1),
      // G = 3/8 I + 5/16 R (+ 35/128 P) -> the Z operand buffer a5 is about to overwrite; then Q = 1/2 R + P G^T
      if (prof) prof->mark(s, EPI_P2 + 16 * tagn);
      p.mapA = pl.mR; p.mapB = pl.mR; p.f32_in = R32;
      if (h16) { p.f32_out = nullptr; p.h_out = ws + L.off_T; p.out2 = ws + L.off_Zb[(par + 1) & 1]; }
      else { p.f32_out = reinterpret_cast<float*>(ws + L.off_T); p.h_out = nullptr; p.out2 = ws + L.off_Z[(par + 1) & 1]; }
      umma_launch_mode(L.mode, EPI_P2, grid_sym, s, p, narrow, pdl);
      nl += 1;
      p.out2 = nullptr;
    }
    if (prof) prof->mark(s, EPI_A4 + 16 * tagn);
    if (order > 2) { p.mapA = pl.mT; p.mapB = pl.mZ[(par + 1) & 1]; }
    else { p.mapA = pl.mR; p.mapB = pl.mR; }
    p.f32_in = R32;
    if (h16) { p.f32_out = nullptr; p.h_out = ws + L.off_Qb; }
    else { p.f32_out = reinterpret_cast<float*>(ws + L.off_Q); p.h_out = nullptr; }
    umma_launch_mode(L.mode, EPI_A4, grid_sym, s, p, narrow, pdl);
    // a5: Z_next = Z + Z Q^T ; W = Z_next^T   (first order in R: all three passes)
    p.hh_only = 0;
    if (prof) prof->mark(s, EPI_A5 + 16 * tagn);
    p.mapA = pl.mZ[par]; p.mapB = pl.mQ;
    if (h16) {
      float* Z32 = reinterpret_cast<float*>(ws + L.off_Z[0]);       // FP32 master copy, updated in place
      p.f32_in = Z32; p.f32_out = Z32; p.h_out = ws + L.off_Zb[(par + 1) & 1]; p.h_out_t = ws + L.off_W;
    } else {
      p.f32_in = reinterpret_cast<float*>(ws + L.off_Z[par]);
      p.f32_out = reinterpret_cast<float*>(ws + L.off_Z[(par + 1) & 1]); p.h_out = nullptr; p.h_out_t = ws + L.off_W;
    }
    if (hook && bands > 1 && hook->after_a5_band) {
      const int T = p.macro_tiles;
      for (int b = 0; b < bands; ++b) {
        const int i0 = (int)((long long)T * b / bands), i1 = (int)((long long)T * (b + 1) / bands);
        p.ioff = i0; p.irows = i1 - i0;
        const int tiles = p.irows * T * nsplit_;
        umma_launch_mode(L.mode, EPI_A5, 2 * (tiles < pl.pairs() ? tiles : pl.pairs()), s, p, narrow, pdl);
        hook->after_a5_band(hook->self, i0 * UM_MACRO, i1 * UM_MACRO, b == bands - 1, s);
      }
      p.ioff = 0; p.irows = 0;
      nl += 1 + bands;
      return;
    }
    umma_launch_mode(L.mode, EPI_A5, grid_full, s, p, narrow, pdl);
    nl += 2;
  }
};

// skip_last: Alg. 3 as printed ends after the update, without evaluating the residual of the result.
inline cudaError_t umma_refine(const UmmaPlan& pl, int max_iter, int stop, int order, double* d_err, cudaStream_t s, int* launches, Prof* prof,
                               const IterHook* hook = nullptr, bool skip_last = false) {
  UmmaSeq q(pl, max_iter, stop, order, d_err, 0ull);
  const bool banded = hook && hook->first_a1 && hook->first_a1(hook->self, &q, s);   // copy-in of S + a1, band by band
  for (int n = 0; n <= max_iter; ++n) {
    if (n == max_iter && skip_last) break;
    q.residual(n, n, s, prof, banded && n == 0);
    if (n == max_iter) break;
    const bool a5_banded = (n == 0 && hook && hook->a5_bands > 1 && hook->after_a5_band);
    q.update(n & 1, n, n, s, prof, hook, a5_banded ? hook->a5_bands : 1);
    if (hook && hook->after_a5 && !a5_banded) hook->after_a5(hook->self, n, s);
  }
  prof->mark(s, 0);
  *launches = q.nl;
  return cudaGetLastError();
}

// Congruence H_perp = Z^T H Z (Eq. 11) with H in the S buffer: T = W H^T, X = W T^T -> R32 buffer.
inline cudaError_t umma_congruence(const UmmaPlan& pl, cudaStream_t s, int* launches) {
  const Layout& L = pl.L;
  char* ws = pl.ws;
  const int T = (int)(L.np / UM_MACRO);
  const bool narrow = umma_narrow(pl);
  const int nsplit = narrow ? 2 : 1;
  const int full_tiles = T * T * nsplit, sym_tiles = T * (T + 1) / 2 * nsplit;
  const int grid_full = 2 * (full_tiles < pl.pairs() ? full_tiles : pl.pairs());
  const int grid_sym = 2 * (sym_tiles < pl.pairs() ? sym_tiles : pl.pairs());
  UmmaParams p{};
  p.np = (int)L.np; p.batch = 1; p.rows = (int)L.np; p.macro_tiles = T; p.band = pl.opt->band;
  p.chunk_kb = pl.opt->chunk_kb; p.chunk0_kb = pl.opt->chunk0_kb;
  p.st = reinterpret_cast<State*>(ws + L.off_state);
  const bool h16 = (L.mode != ZFAC_MODE_TF32);
  p.mapA = pl.mW; p.mapB = pl.mS;
  if (h16) p.h_out = ws + L.off_T; else p.f32_out = reinterpret_cast<float*>(ws + L.off_T);
  umma_launch_mode(L.mode, EPI_A1, grid_full, s, p, narrow);
  p.mapA = pl.mW; p.mapB = pl.mT; p.f32_out = reinterpret_cast<float*>(ws + L.off_R); p.h_out = nullptr;
  umma_launch_mode(L.mode, EPI_X3, grid_sym, s, p, narrow);
  *launches = 2;
  return cudaGetLastError();
}

}  // namespace zfac
