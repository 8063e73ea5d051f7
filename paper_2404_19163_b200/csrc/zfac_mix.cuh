// FP64-master modes: the enhanced-precision stage of Alg. 3 rebuilt for a chip whose FP64 tensor
// pipe is 40x slower than its FP16 pipe and 100x slower than its INT8 pipe.
//
// What must be accurate to the FP64 level in one refinement iteration is the RESIDUAL R = I - Z^T (S Z): X ~ I is formed
// from O(1) terms and the signal is what is left after the cancellation.  The UPDATE Z <- Z + Z (1/2 R + 3/8 R R) is a
// correction of relative size ||R||: evaluated in FP32-class arithmetic (the SPLIT16 kernels of zfac_umma.cuh on the FP32
// parts of Z and R) and ADDED to the FP64 master, its rounding leaves only ~2^-22 ||R|| in the next residual
// (pinned on the CPU side of the tests).  Two modes, same update, two residual engines:
//
//   ZFAC_MODE_F64_MIXED   residual by the DMMA kernels of zfac_f64_tma.cuh (a1, a2 on FP64 S, W = Z^T, T);
//   ZFAC_MODE_F64_I8      residual on the INT8 tensor cores (tcgen05.mma kind::i8, exact INT32 accumulation in tensor
//                         memory) by error-free slicing of the FP64 operands -- the Ozaki scheme (Ootomo, Ozaki, Yokota,
//                         "DGEMM on integer matrix multiplication unit", 2024) restated for tcgen05: see i8_gemm_kernel.
//
// Per iteration:  residual (engine) -> a3 (stop test, unchanged) -> r_split (R -> R~ = rscale R as FP32 and as the
// (hi, lo') fp16 operand pair; rscale = power of two from ||R||_F) -> a4 (umma, Q~ = 1/2 R~ + (3/8 / rscale) R~ R~) ->
// a5x (umma, Z64 += (Z Q~) / rscale, next operand pair of Z [, W64 = Z^T]) [-> w_slice (I8 engine: W = Z^T int8 slices)].
#pragma once
#include "zfac_umma.cuh"
#include "zfac_f64_tma.cuh"

namespace zfac {

constexpr int I8_MAX_SLICES = 8;          // 7 bits per slice: 56 bits relative to the row maximum
constexpr int I8_SCRATCH_CTAS = 192;      // partial-sum scratch: one 128 x 256 FP64 half tile per CTA

// ------------------------------------------------------------------ r_split: R -> (rscale R) as FP32 and as fp16 pair
// rscale = 2^k with 48 < rscale ||R||_F <= 96: every |R~_ij| <= 96 and every |Q~_ij| <= 48 + 36 ||R||_F stay inside the
// FP16 range, and entries down to 2^-36 * 96 of the norm keep their leading bits in the (hi, lo') pair.
__device__ __forceinline__ double pick_rscale(double err) {
  if (!(err > 0.0) || !isfinite(err)) return 1.0;
  int k = ilogb(96.0 / err);
  k = k < -60 ? -60 : (k > 100 ? 100 : k);
  return ldexp(1.0, k);
}
template <typename Tin>
__global__ void __launch_bounds__(256) r_split_kernel(const Tin* __restrict__ R, float* __restrict__ R32s, __half* __restrict__ Rb,
                                                      size_t np2, State* st, const double* d_err, int n_iter) {
  if (*((volatile int*)&st->done)) return;
  const double sc = pick_rscale(d_err[n_iter >= 0 ? n_iter : st->iters]);
  if (blockIdx.x == 0 && threadIdx.x == 0) { st->rscale = (float)sc; st->rinv = (float)(1.0 / sc); }
  // grid-stride over groups of 8 elements: the grid is a few CTAs per SM, so that the statically enqueued launches after
  // the stop return in microseconds (a grid of Np^2 / 2048 CTAs that all exit at once still took 80 us at N = 8192)
  for (size_t o = ((size_t)blockIdx.x * 256 + threadIdx.x) * 8; o < np2; o += (size_t)gridDim.x * 256 * 8) {
    float v[8];
#pragma unroll
    for (int j = 0; j < 8; ++j) v[j] = (float)((double)R[o + j] * sc);
    *reinterpret_cast<float4*>(R32s + o) = make_float4(v[0], v[1], v[2], v[3]);
    *reinterpret_cast<float4*>(R32s + o + 4) = make_float4(v[4], v[5], v[6], v[7]);
    uint32_t hi[4], lo[4];
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      __half h0, l0, h1, l1;
      split_f16(v[2 * j], h0, l0); split_f16(v[2 * j + 1], h1, l1);
      hi[j] = pack_h2(h0, h1); lo[j] = pack_h2(l0, l1);
    }
    *reinterpret_cast<uint4*>(Rb + o) = make_uint4(hi[0], hi[1], hi[2], hi[3]);
    *reinterpret_cast<uint4*>(Rb + np2 + o) = make_uint4(lo[0], lo[1], lo[2], lo[3]);
  }
}
// Grid of the O(N^2) helper kernels: enough CTAs to fill the device, few enough to exit at once.
inline unsigned small_grid(size_t work_items, unsigned cap = 148 * 8) { return (unsigned)(work_items < cap ? (work_items ? work_items : 1) : cap); }

// FP32[Z64] as the (hi, lo') operand pair of the first update (later ones are written by a5x's epilogue).
__global__ void __launch_bounds__(256) z_planes_kernel(const double* __restrict__ Z, __half* __restrict__ Zb, size_t np2, State* st) {
  const size_t o = ((size_t)blockIdx.x * 256 + threadIdx.x) * 8;
  if (o >= np2) return;
  float v[8];
#pragma unroll
  for (int j = 0; j < 8; ++j) v[j] = (float)Z[o + j];
  flag_h16_range<8>(st, v);
  uint32_t hi[4], lo[4];
#pragma unroll
  for (int j = 0; j < 4; ++j) {
    __half h0, l0, h1, l1;
    split_f16(v[2 * j], h0, l0); split_f16(v[2 * j + 1], h1, l1);
    hi[j] = pack_h2(h0, h1); lo[j] = pack_h2(l0, l1);
  }
  *reinterpret_cast<uint4*>(Zb + o) = make_uint4(hi[0], hi[1], hi[2], hi[3]);
  *reinterpret_cast<uint4*>(Zb + np2 + o) = make_uint4(lo[0], lo[1], lo[2], lo[3]);
}

// ------------------------------------------------------------------ error-free slicing (I8 engine)
// A row a[0..K) is written as  a_k = sum_{i < s} q_i[k] 2^(e - 6 - 7 i) + rest,  q_i int8,  |rest| <= 2^(e - 7 s):
// q_0 = rint(a 2^(6 - e)), then the remainder times 128, and so on -- every step is exact in FP64.  The exponent e is the
// smallest with |q_0| <= 127 for the row's largest entry (the first slice uses the whole int8 range: one bit more than
// |a| < 2^e would give); all later slices lie in [-64, 64].
// One exponent per row (K-major operand rows: the GEMM's A rows and B rows), so the products of slices are exact
// integers and the scales factor out of the dot product:  sum_k a_k b_k = 2^(eA + eB - 12) sum_{i, j} 2^(-7 (i + j)) <q_i, q_j>.
__device__ __forceinline__ int slice_exponent(double amax) {
  if (!(amax > 0.0) || !isfinite(amax)) return 0;
  const int e = ilogb(amax) + 1;                             // amax in [2^(e-1), 2^e): q_0 in [32, 64)
  return (ldexp(amax, 7 - e) < 127.5) ? e - 1 : e;           // e - 1: q_0 in [64, 127] still fits
}

// A non-finite operand cannot be sliced (and fmax drops NaN from the row maximum): it is recorded in State::range bit 1 and
// turns the Err of the residual that uses the slices into NaN, so that ZFAC_R_NONFINITE fires as in the other modes.
__device__ __forceinline__ void slice16(const double (&a)[16], int e, int slices, int8_t* out, size_t plane, size_t o, State* st) {
  double x[16];
  const double s0 = ldexp(1.0, 6 - e);
  bool bad = false;
#pragma unroll
  for (int j = 0; j < 16; ++j) { x[j] = a[j] * s0; bad |= !isfinite(a[j]); }
  if (bad) {
    atomicOr(&st->range, 2);
#pragma unroll
    for (int j = 0; j < 16; ++j) x[j] = 0.0;
  }
  for (int i = 0; i < slices; ++i) {
    uint32_t w[4] = {0u, 0u, 0u, 0u};
#pragma unroll
    for (int j = 0; j < 16; ++j) {
      const double q = rint(x[j]);
      x[j] = (x[j] - q) * 128.0;
      w[j >> 2] |= ((uint32_t)(uint8_t)(int8_t)(int)q) << (8 * (j & 3));
    }
    *reinterpret_cast<uint4*>(out + (size_t)i * plane + o) = make_uint4(w[0], w[1], w[2], w[3]);
  }
}

// Rows of a row-major matrix (n valid rows / columns of leading dimension ld, identity beyond: the padding of zfac_io.cuh).
// One CTA per row: pass 1 = row maximum, pass 2 = slices.  Used for S (from the caller's buffer) and T = (S Z)^T.
template <typename Tin>
__global__ void __launch_bounds__(256) slice_rows_kernel(const Tin* __restrict__ src, int64_t ld, int n, int np, int slices,
                                                         int8_t* __restrict__ out, int* __restrict__ exps, State* st,
                                                         int row0 = 0, int rows = 0 /* 0: all np rows */) {
  if (*((volatile int*)&st->done)) return;
  __shared__ double red[8];
  __shared__ int e_sh;
  const int t = threadIdx.x;
  const int r_end = rows > 0 ? row0 + rows : np;
  for (int r = row0 + blockIdx.x; r < r_end; r += gridDim.x) {
  double mx = 0.0;
  if (r < n) {
    for (int c = t; c < n; c += 256) mx = fmax(mx, fabs((double)src[(size_t)r * ld + c]));
  } else {
    mx = 1.0;                                                  // identity row of the padding
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) mx = fmax(mx, __shfl_xor_sync(0xffffffffu, mx, o));
  if ((t & 31) == 0) red[t >> 5] = mx;
  __syncthreads();
  if (t == 0) {
    double m = red[0];
    for (int w = 1; w < 8; ++w) m = fmax(m, red[w]);
    e_sh = slice_exponent(m);
    exps[r] = e_sh;
  }
  __syncthreads();
  const int e = e_sh;
  const size_t plane = (size_t)np * np;
  for (int c0 = t * 16; c0 < np; c0 += 256 * 16) {
    double a[16];
#pragma unroll
    for (int j = 0; j < 16; ++j) {
      const int c = c0 + j;
      a[j] = (r < n && c < n) ? (double)src[(size_t)r * ld + c] : ((r == c) ? 1.0 : 0.0);
    }
    slice16(a, e, slices, out, plane, (size_t)r * np + c0, st);
  }
  __syncthreads();                                             // red / e_sh are reused by the next row
  }
}

// W = Z^T: the rows of W are the COLUMNS of Z.  Column maxima first (one CTA per 32 columns) ...
__global__ void __launch_bounds__(256) colmax_kernel(const double* __restrict__ Z, int np, int* __restrict__ exps, const State* st) {
  if (*((volatile int*)&st->done)) return;
  __shared__ double red[8][33];
  const int c = blockIdx.x * 32 + (threadIdx.x & 31), rl = threadIdx.x >> 5;
  double mx = 0.0;
  for (int r = rl; r < np; r += 8) mx = fmax(mx, fabs(Z[(size_t)r * np + c]));
  red[rl][threadIdx.x & 31] = mx;
  __syncthreads();
  if (rl == 0) {
    for (int w = 1; w < 8; ++w) mx = fmax(mx, red[w][threadIdx.x & 31]);
    exps[c] = slice_exponent(mx);
  }
}
// ... then 64 x 64 tiles of Z through shared memory: thread (c, k-chunk) takes 16 consecutive rows of one column of the tile
// = 16 consecutive k of one row of W.
__global__ void __launch_bounds__(256) slice_transpose_kernel(const double* __restrict__ Z, int np, int slices, int8_t* __restrict__ out,
                                                              const int* __restrict__ exps, State* st) {
  if (*((volatile int*)&st->done)) return;
  __shared__ double tile[64][65];
  const int t = threadIdx.x, tn = np / 64;
  for (int tt = blockIdx.x; tt < tn * tn; tt += gridDim.x) {
  const int r0 = (tt / tn) * 64, c0 = (tt % tn) * 64;
#pragma unroll
  for (int i = 0; i < 16; ++i) {
    const int idx = t + 256 * i, lr = idx >> 6, lc = idx & 63;
    tile[lr][lc] = Z[(size_t)(r0 + lr) * np + c0 + lc];
  }
  __syncthreads();
  const int wc = t >> 2, kc = (t & 3) * 16;                  // W row c0 + wc, k = r0 + kc .. + 16
  double a[16];
#pragma unroll
  for (int j = 0; j < 16; ++j) a[j] = tile[kc + j][wc];
  slice16(a, exps[c0 + wc], slices, out, (size_t)np * np, (size_t)(c0 + wc) * np + r0 + kc, st);
  __syncthreads();
  }
}

// ------------------------------------------------------------------ the INT8 GEMM (Ozaki scheme on tcgen05)
// D[m][n] = sum_k A[m][k] B[n][k] in FP64-equivalent accuracy from int8 slices A_i, B_j (i < sa, j < sb):
//     D = 2^(eA[m] + eB[n] - 12) sum_{d < orders} 2^(-7 d) sum_{i + j = d} <A_i[m], B_j[n]>        (orders d >= `orders` dropped)
// Same CTA-pair structure as umma_gemm_kernel (256 x 256 pair tile, TMA 128B-swizzle boxes, 6 stages of one k-block =
// 128 int8 per row, tcgen05.mma.cta_group::2.kind::i8 with M = 256, N = 256, K = 32).  Every inner product of slices is
// accumulated EXACTLY in an INT32 accumulator in tensor memory (|q_0| <= 127, |q_i| <= 64: an order's <= 8 slice pairs
// sum to at most (2 * 2^13 + 6 * 2^12) K < 2^31 for K <= 2^15).  The two 256-column accumulators alternate between consecutive orders d: while order d - 1
// runs on the tensor core, the 8 epilogue warps convert order d to FP64, weight it and add it to the tile's running sum.
// That sum (128 x 256 doubles per CTA) exceeds the register file, so it lives in a per-CTA scratch slab that stays in L2
// (38 MB for 148 CTAs); orders run from the highest (smallest terms) to d = 0, whose drain applies the fused epilogue.
struct I8Params {
  CUtensorMap mapA, mapB;     // [slices * Np rows][Np cols] int8, box 128 B x 64 rows, 128B swizzle
  int np, macro_tiles;
  int sa, sb, orders;         // slices of A, of B; orders d = i + j kept: 0 .. orders - 1
  const int* expA;            // per row of A
  const int* expB;            // per row of B
  double* scratch;            // I8_SCRATCH_CTAS x 128 x 256 doubles
  State* st;
  StopArgs stop;              // a2
  double* out64;              // a1: T (FP64)
  float* out32;               // a2: R (FP32, both triangles)
  int band;
  int joff, jcols;            // a1: this launch covers the tile columns [joff, joff + jcols) of T only (jcols = 0: all), i.e. the
                              // rows [256 joff, ...) of S: zfac_refine_host runs a1 band by band while the row chunks of S arrive
};

__device__ __forceinline__ void tc_mma_pair_i8(uint32_t d_tmem, uint64_t adesc, uint64_t bdesc, uint32_t idesc, uint32_t accum) {
  asm volatile("{\n .reg .pred p;\n setp.ne.b32 p, %4, 0;\n tcgen05.mma.cta_group::2.kind::i8 [%0], %1, %2, %3, p;\n}"
               ::"r"(d_tmem), "l"(adesc), "l"(bdesc), "r"(idesc), "r"(accum) : "memory");
}
// kind::i8 instruction descriptor: D = S32, A / B = signed 8-bit, both K-major, M = 256 (pair), N = n
__host__ __device__ constexpr uint32_t make_idesc_i8(int n) {
  return (2u << 4) | (1u << 7) | (1u << 10) | ((uint32_t)(n >> 3) << 17) | ((uint32_t)(UM_TILE_M >> 4) << 24);
}

constexpr int I8_STAGES = 4;
constexpr int I8_STAGE_BYTES = 3 * UM_A_BYTES;      // A_i, B_(d-i), B_(d-1-i) rows of one CTA, one k-block: 48 KB

// tcgen05.commit of the pair's MMAs arriving on the barrier at offset `bar` in every CTA of `mask` (cluster ranks)
__device__ __forceinline__ void tc_commit_mask(uint32_t bar, uint32_t mask) {
  asm volatile("tcgen05.commit.cta_group::2.mbarrier::arrive::one.shared::cluster.multicast::cluster.b64 [%0], %1;"
               ::"r"(bar), "h"((uint16_t)mask) : "memory");
}
// TMA load by one CTA into the SAME shared-memory offset of every CTA of `mask`; each destination counts the bytes on the
// barrier at offset `bar` of ITS pair's leader (the address is this CTA's own with the peer bit, bit 24, cleared).
__device__ __forceinline__ void tma_load_2d_pair_mc(uint32_t dst, const CUtensorMap* map, int c0, int c1, uint32_t bar, uint32_t mask) {
  asm volatile(
      "cp.async.bulk.tensor.2d.cta_group::2.shared::cluster.global.mbarrier::complete_tx::bytes.multicast::cluster [%0], [%1, {%2, %3}], [%4], %5;"
      ::"r"(dst), "l"(reinterpret_cast<uint64_t>(map)), "r"(c0), "r"(c1), "r"(bar & 0xFEFFFFFFu), "h"((uint16_t)mask)
      : "memory");
}

// CP = CTA pairs per cluster.  CP = 1: every pair on its own.  CP = 2 (full outputs, an even number of tile rows): a cluster
// of two pairs works on the tiles (2 I', J) and (2 I' + 1, J); they use the same rows of B, so each B box is fetched from L2
// ONCE and delivered to both pairs by TMA multicast (pair 0's CTAs fetch the B slice of order d, pair 1's the one of order
// d - 1): 2/3 of a stage's bytes are shared, the L2 -> SM traffic falls by a third.  The two pairs then move in lockstep, a
// stage at a time: a stage is refilled when BOTH pairs have released it (every MMA leader commits to the empty barriers of all
// four CTAs).  Same arithmetic per tile: bit-identical results.
// TN = 128 (CP = 1): the same on 256 x 128 tiles -- twice as many tiles for problems whose 256 x 256 tiles leave CTA pairs idle
// (ZFAC_OPT_I8_NARROW); every element is the same exact integer sum, so T and R are bit-identical, and Err[] differs in its last
// bits only (the partial sums of step a3 are grouped by tile).
template <int EPI, int CP = 1, int TN = 256>
__global__ void __cluster_dims__(2 * CP, 1, 1) __launch_bounds__(UM_THREADS, 1)
i8_gemm_kernel(const __grid_constant__ I8Params p) {
  static_assert(CP == 1 || EPI == EPI_A1, "clusters of two pairs: full outputs only");
  static_assert(TN == 256 || (TN == 128 && CP == 1), "tile widths");
  if (*((volatile int*)&p.st->done)) return;
  constexpr bool SYM = (EPI == EPI_A2);
  constexpr int NS = 256 / TN;                                 // tiles per 256-column macro tile
  constexpr int GC = TN / 2;                                   // columns per epilogue thread (two groups of warps)
  constexpr uint32_t IDESC = make_idesc_i8(TN);

  extern __shared__ unsigned char smem_raw[];
  const uint32_t smem_base = (smem_u32(smem_raw) + 1023u) & ~1023u;
  const uint32_t bar_base = smem_base + UM_SMEM_OPERANDS;
  auto full_bar = [&](int s) { return bar_base + 8u * s; };
  auto empty_bar = [&](int s) { return bar_base + 48u + 8u * s; };
  auto tfull_bar = [&](int b) { return bar_base + 96u + 8u * b; };
  auto tempty_bar = [&](int b) { return bar_base + 112u + 8u * b; };
  const uint32_t tmem_slot = bar_base + 160u;
  __shared__ double red[32];
  __shared__ int last_flag;

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const uint32_t crank = cluster_ctarank();                  // 0 .. 2 CP - 1
  const uint32_t rank = crank & 1u;                          // within the pair: 0 = leader (issues the MMAs)
  const uint32_t lead = crank & ~1u;                         // cluster rank of this pair's leader
  const int pp = (int)(crank >> 1);                          // pair within the cluster
  // unit of work distribution: the cluster.  CP = 2: one "tile" of the loops below is a 512 x 256 super tile
  const int pair = (int)blockIdx.x / (2 * CP), num_pairs = (int)gridDim.x / (2 * CP);
  const int np = p.np;
  const int KB = np / 128;                                   // k-blocks of 128 int8
  const int T = p.macro_tiles;
  const int JC = (!SYM && p.jcols > 0) ? p.jcols * NS : T * NS;   // tile columns of this launch (p.joff, p.jcols: macro columns)
  const int num_tiles = SYM ? T * (T + 1) / 2 * NS : (T / CP) * JC;
  const int ORD = p.orders;

  if (threadIdx.x == 0) {
    for (int s = 0; s < I8_STAGES; ++s) { mbar_init(full_bar(s), 1); mbar_init(empty_bar(s), CP); }
    mbar_init(tfull_bar(0), 1); mbar_init(tempty_bar(0), 2 * UM_EPI_WARPS);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    asm volatile("prefetch.tensormap [%0];" ::"l"(reinterpret_cast<uint64_t>(&p.mapA)) : "memory");
    asm volatile("prefetch.tensormap [%0];" ::"l"(reinterpret_cast<uint64_t>(&p.mapB)) : "memory");
  }
  if (warp == 1) {
    asm volatile("tcgen05.alloc.cta_group::2.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(tmem_slot), "r"(UM_TMEM_COLS) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::2.sync.aligned;" ::: "memory");
  }
  tc_fence_before();
  __syncthreads();
  cluster_sync_all();
  tc_fence_after();
  uint32_t tmem_base;
  asm volatile("ld.shared.b32 %0, [%1];" : "=r"(tmem_base) : "r"(tmem_slot));

  auto decode = [&](int t, int& m0, int& n0, bool& offdiag) {
    int I, J;
    if (SYM) { const int macro = t / NS; tri_decode(macro, I, J); offdiag = (I != J); J = J * NS + (t - macro * NS); }
    else { band_decode(t, T / CP, JC, p.band * NS, I, J); I = I * CP + pp; J += p.joff * NS; offdiag = true; }
    m0 = I * UM_TILE_M; n0 = J * TN;
  };


  if (warp == 0) {
    // ===================================================== TMA producer (both CTAs)
    if (lane == 0) {
      int stage = 0; uint32_t phase = 0;
      const int aoff = (int)rank * UM_ROWS, boff = (int)rank * (TN / 2);
      for (int t = pair; t < num_tiles; t += num_pairs) {
        int m0, n0; bool od; decode(t, m0, n0, od);
        for (int d = ORD - 1; d >= 0; d -= 2)                // sweep over the orders (d, d - 1)
          for (int i = 0; i <= d; ++i) {
            const int j1 = d - i, j2 = d - 1 - i;             // B slices for order d and order d - 1
            const bool v1 = (i < p.sa && j1 < p.sb), v2 = (i < p.sa && j2 >= 0 && j2 < p.sb);
            if (!v1 && !v2) continue;
            for (int kb = 0; kb < KB; ++kb) {
              mbar_wait(empty_bar(stage), phase ^ 1u);
              if (rank == 0) mbar_expect_tx(full_bar(stage), 2u * ((uint32_t)UM_A_BYTES + (uint32_t)(GC * UM_ROWB) * ((v1 ? 1u : 0u) + (v2 ? 1u : 0u))));
              const uint32_t lead_full = mapa_u32(full_bar(stage), lead);
              const uint32_t sa = smem_base + stage * I8_STAGE_BYTES, sb1 = sa + UM_A_BYTES, sb2 = sb1 + UM_A_BYTES;
              const int kc = kb * 128;
              const uint32_t mc = (1u << rank) | (1u << (rank + 2u));   // CP = 2: the CTAs of both pairs that hold this half of B
#pragma unroll
              for (int b = 0; b < UM_ROWS / UM_BOX_ROWS; ++b) {
                tma_load_2d_pair(sa + b * UM_BOX_BYTES, &p.mapA, kc, i * np + m0 + aoff + b * UM_BOX_ROWS, lead_full);
                if (CP == 1) {
                  if (b < GC / UM_BOX_ROWS) {                  // TN / 2 rows of B per CTA: one box (TN = 128) or two
                    if (v1) tma_load_2d_pair(sb1 + b * UM_BOX_BYTES, &p.mapB, kc, j1 * np + n0 + boff + b * UM_BOX_ROWS, lead_full);
                    if (v2) tma_load_2d_pair(sb2 + b * UM_BOX_BYTES, &p.mapB, kc, j2 * np + n0 + boff + b * UM_BOX_ROWS, lead_full);
                  }
                } else if (pp == 0) {
                  if (v1) tma_load_2d_pair_mc(sb1 + b * UM_BOX_BYTES, &p.mapB, kc, j1 * np + n0 + boff + b * UM_BOX_ROWS, full_bar(stage), mc);
                } else {
                  if (v2) tma_load_2d_pair_mc(sb2 + b * UM_BOX_BYTES, &p.mapB, kc, j2 * np + n0 + boff + b * UM_BOX_ROWS, full_bar(stage), mc);
                }
              }
              if (++stage == I8_STAGES) { stage = 0; phase ^= 1u; }
            }
          }
      }
    }
  } else if (warp == 1) {
    // ===================================================== MMA issuer (leader CTA, one lane)
    if (rank == 0 && lane == 0) {
      int stage = 0; uint32_t phase = 0;
      uint32_t seq = 0;                                      // sweeps finished by this pair
      for (int t = pair; t < num_tiles; t += num_pairs) {
        for (int d = ORD - 1; d >= 0; d -= 2, ++seq) {
          const uint32_t dA = tmem_base, dB = tmem_base + TN;  // order d -> columns [0, 256), order d - 1 -> [256, 512)
          mbar_wait(tempty_bar(0), (seq & 1u) ^ 1u);          // both accumulators drained
          tc_fence_after();
          uint32_t acc1 = 0u, acc2 = 0u;
          for (int i = 0; i <= d; ++i) {
            const int j1 = d - i, j2 = d - 1 - i;
            const bool v1 = (i < p.sa && j1 < p.sb), v2 = (i < p.sa && j2 >= 0 && j2 < p.sb);
            if (!v1 && !v2) continue;
            for (int kb = 0; kb < KB; ++kb) {
              mbar_wait(full_bar(stage), phase);
              tc_fence_after();
              const uint32_t sa = smem_base + stage * I8_STAGE_BYTES;
              const uint64_t ad = make_sdesc(sa), b1 = make_sdesc(sa + UM_A_BYTES), b2 = make_sdesc(sa + 2 * UM_A_BYTES);
#pragma unroll
              for (int k = 0; k < 4; ++k) {                  // K = 32 int8 = 32 bytes per MMA, in 16-byte units
                if (v1) { tc_mma_pair_i8(dA, ad + (uint64_t)(k * 2), b1 + (uint64_t)(k * 2), IDESC, acc1); acc1 = 1u; }
                if (v2) { tc_mma_pair_i8(dB, ad + (uint64_t)(k * 2), b2 + (uint64_t)(k * 2), IDESC, acc2); acc2 = 1u; }
              }
              tc_commit_mask(empty_bar(stage), (1u << (2 * CP)) - 1u);      // every CTA of the cluster: its stage is free
              if (++stage == I8_STAGES) { stage = 0; phase ^= 1u; }
            }
          }
          tc_commit_mask(tfull_bar(0), 3u << lead);           // orders d and d - 1 complete in both CTAs of the pair
        }
      }
    }
  } else if (warp >= UM_EPI_WARP0) {
    // ===================================================== epilogue warps 4 .. 11: thread = (row, 128-column half)
    const int q = warp & 3, g = (warp - UM_EPI_WARP0) >> 2;
    const int rowl = q * 32 + lane;                            // row of this CTA's 128-row half tile
    const uint32_t lead_tempty = mapa_u32(tempty_bar(0), lead);
    double* slab = p.scratch + (size_t)blockIdx.x * (128 * 256);
    uint32_t seq = 0;
    for (int t = pair; t < num_tiles; t += num_pairs) {
      int m0, n0; bool offdiag; decode(t, m0, n0, offdiag);
      const int m = m0 + (int)rank * UM_ROWS + rowl;
      const int eA = p.expA[m];
      double tile_sumsq = 0.0;
      for (int d = ORD - 1; d >= 0; d -= 2, ++seq) {
        mbar_wait(tfull_bar(0), seq & 1u);
        tc_fence_after();
        const bool two = (d >= 1);                             // the sweep carries order d - 1 as well
        const bool first = (d == ORD - 1), last = (d <= 1);
        const double w1 = ldexp(1.0, -7 * d), w2 = ldexp(1.0, -7 * (d - 1));
        const uint32_t tbase = tmem_base + ((uint32_t)(q * 32) << 16) + g * GC;
#pragma unroll 1
        for (int c = 0; c < GC / 32; ++c) {
          uint32_t r1[32], r2[32];
          tmem_ld(tbase + c * 32, r1);
          if (two) tmem_ld(tbase + TN + c * 32, r2);
          tmem_ld_wait();
          if (c == GC / 32 - 1) {                              // accumulators read out: hand them back before the arithmetic
            tc_fence_before();
            __syncwarp();
            mbar_arrive_cluster_lane0(lead_tempty, lane);
            asm volatile("fence.acq_rel.cta;" ::: "memory");
          }
          const int col0 = g * GC + c * 32;
          double* sl = slab + (size_t)col0 * 128 + rowl;     // element (row, col) at (col * 128 + row): coalesced per column
          if (!last) {
#pragma unroll
            for (int j = 0; j < 32; ++j) {
              double v = (double)(int)r1[j] * w1 + (double)(int)r2[j] * w2;
              if (!first) v += sl[(size_t)j * 128];
              sl[(size_t)j * 128] = v;
            }
          } else {
            // last sweep: the sum is complete -> scale by the row / column exponents and apply the fused epilogue
            const size_t ld = (size_t)np;
            const int n = n0 + col0;
#pragma unroll
            for (int j = 0; j < 32; ++j) {
              double v = (double)(int)r1[j] * w1;
              if (two) v += (double)(int)r2[j] * w2;
              if (!first) v += sl[(size_t)j * 128];
              v = ldexp(v, eA + p.expB[n + j] - 12);
              if (EPI == EPI_A1) {
                p.out64[(size_t)m * ld + n + j] = v;
              } else {
                const float rr = (float)(((m == n + j) ? 1.0 : 0.0) - v);          // R = I - X
                tile_sumsq += (double)rr * (double)rr;
                p.out32[(size_t)m * ld + n + j] = rr;
                if (offdiag) p.out32[(size_t)(n + j) * ld + m] = rr;
              }
            }
          }
        }
      }
      if (EPI == EPI_A2) {
        // step a3, first half: one partial sum per tile, CTA of the pair, column half and lane quarter, stored by TILE index --
        // Err[] does not depend on which pair computed which tile (ZFAC_OPT_MAX_PAIRS, another SM count)
        const double ws_ = warp_sum(offdiag ? 2.0 * tile_sumsq : tile_sumsq);
        if (lane == 0) { p.stop.partials[(size_t)t * 16 + rank * 8 + g * 4 + q] = ws_; __threadfence(); }
      }
    }
  }

  // ------------------------------------------------------- teardown (+ step a3 for a2)
  tc_fence_before();
  __syncthreads();
  cluster_sync_all();
  if (warp == 1) {
    tc_fence_after();
    asm volatile("tcgen05.dealloc.cta_group::2.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "r"(UM_TMEM_COLS) : "memory");
  }
  if (EPI == EPI_A2) {
    // a non-finite operand was met while slicing: Err[n] is NaN (one slot of this CTA's first tile carries it)
    if (threadIdx.x == 0 && (*((volatile int*)&p.st->range) & 2)) p.stop.partials[(size_t)pair * 16 + rank * 8] = nan("");
    if (arrive_is_last(&p.st->arrive[0], gridDim.x, &last_flag)) stop_test_last_cta(p.stop, red);
  }
}

// ------------------------------------------------------------------ host side: plan + sequencer of the FP64-master modes
struct MixPlan {
  Layout L;
  char* ws = nullptr;
  int mode = 0;
  int max_pairs = 0;
  int max_quads = 0;                    // I8 engine: co-resident clusters of two pairs (i8_gemm_kernel<EPI_A1, 2>)
  const Options* opt = nullptr;
  F64Plan f64;                          // DMMA engine: S, W, T, R (FP64)
  CUtensorMap mR, mQ, mZ[2];            // fp16 pair planes of R~, Q~, FP32[Z] (update GEMMs)
  CUtensorMap mS8, mW8, mT8;            // I8 engine: int8 slices
  int pairs() const { return (opt->max_pairs > 0 && opt->max_pairs < max_pairs) ? opt->max_pairs : max_pairs; }
};

template <int EPI, int CP = 1, int TN = 256>
inline cudaError_t i8_prepare(int* max_pairs, int sm_count) {
  cudaError_t e = cudaFuncSetAttribute(i8_gemm_kernel<EPI, CP, TN>, cudaFuncAttributeMaxDynamicSharedMemorySize, UM_SMEM_BYTES);
  if (e != cudaSuccess) return e;
  cudaLaunchConfig_t cfg{};
  cfg.gridDim = dim3(2 * CP * (sm_count / (2 * CP))); cfg.blockDim = dim3(UM_THREADS); cfg.dynamicSmemBytes = UM_SMEM_BYTES;
  int nc = 0;
  e = cudaOccupancyMaxActiveClusters(&nc, i8_gemm_kernel<EPI, CP, TN>, &cfg);
  if (e != cudaSuccess) return e;
  if (nc < 1) return cudaErrorLaunchOutOfResources;
  if (*max_pairs == 0 || nc < *max_pairs) *max_pairs = nc;
  return cudaSuccess;
}

inline cudaError_t mix_plan_create(MixPlan* pl, const Layout& L, char* ws, int sm_count, const Options* opt) {
  pl->L = L; pl->ws = ws; pl->mode = L.mode; pl->opt = opt; pl->max_pairs = 0;
  void* fn = nullptr;
  cudaDriverEntryPointQueryResult qres;
  cudaError_t e = cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres);
  if (e != cudaSuccess) return e;
  if (!fn || qres != cudaDriverEntryPointSuccess) return cudaErrorNotSupported;
  PFN_encodeTiled enc = reinterpret_cast<PFN_encodeTiled>(fn);
  const uint64_t np = (uint64_t)L.np;
  const CUtensorMapDataType H = CU_TENSOR_MAP_DATA_TYPE_FLOAT16;
  if ((e = make_map(enc, &pl->mR, ws + L.off_Rb, H, 2, 2 * np, np)) != cudaSuccess) return e;
  if ((e = make_map(enc, &pl->mQ, ws + L.off_Qb, H, 2, 2 * np, np)) != cudaSuccess) return e;
  if ((e = make_map(enc, &pl->mZ[0], ws + L.off_Zb[0], H, 2, 2 * np, np)) != cudaSuccess) return e;
  if ((e = make_map(enc, &pl->mZ[1], ws + L.off_Zb[1], H, 2, 2 * np, np)) != cudaSuccess) return e;
  if ((e = prepare_kernel<KIND_F16X2, EPI_A4>(&pl->max_pairs, sm_count)) != cudaSuccess) return e;
  if ((e = prepare_kernel<KIND_F16X2, EPI_A5X>(&pl->max_pairs, sm_count)) != cudaSuccess) return e;
  if (L.mode == ZFAC_MODE_F64_MIXED) {
    if ((e = f64_plan_create(&pl->f64, L, ws)) != cudaSuccess) return e;
    if ((e = f64_tma_prepare<EPI_A1>()) != cudaSuccess) return e;
    if ((e = f64_tma_prepare<EPI_A2>()) != cudaSuccess) return e;
  } else {
    const CUtensorMapDataType B8 = CU_TENSOR_MAP_DATA_TYPE_UINT8;
    const uint64_t rows = (uint64_t)I8_MAX_SLICES * np;
    if ((e = make_map(enc, &pl->mS8, ws + L.off_S8, B8, 1, rows, np)) != cudaSuccess) return e;
    if ((e = make_map(enc, &pl->mW8, ws + L.off_W8, B8, 1, rows, np)) != cudaSuccess) return e;
    if ((e = make_map(enc, &pl->mT8, ws + L.off_T8, B8, 1, rows, np)) != cudaSuccess) return e;
    if ((e = i8_prepare<EPI_A1>(&pl->max_pairs, sm_count)) != cudaSuccess) return e;
    if ((e = i8_prepare<EPI_A2>(&pl->max_pairs, sm_count)) != cudaSuccess) return e;
    if ((e = i8_prepare<EPI_A1, 2>(&pl->max_quads, sm_count)) != cudaSuccess) { pl->max_quads = 0; (void)cudaGetLastError(); }
    if ((e = i8_prepare<EPI_A1, 1, 128>(&pl->max_pairs, sm_count)) != cudaSuccess) return e;
    if ((e = i8_prepare<EPI_A2, 1, 128>(&pl->max_pairs, sm_count)) != cudaSuccess) return e;
  }
  if (pl->max_pairs > sm_count / 2) pl->max_pairs = sm_count / 2;
  if (2 * pl->max_pairs > I8_SCRATCH_CTAS) pl->max_pairs = I8_SCRATCH_CTAS / 2;
  return cudaSuccess;
}

// The two halves of one iteration (same contract as UmmaSeq / F64Seq: n_stop = index of the Err entry, -1 = device-side).
struct MixSeq {
  const MixPlan& pl;
  int nl = 0;
  int grid_full = 0, grid_sym = 0;
  StopArgs stop{};
  State* st;
  double* d_err;
  float* R32s;
  size_t np2;

  MixSeq(const MixPlan& pl_, int max_iter, int stop_rule, double* d_err_, unsigned long long cond) : pl(pl_), d_err(d_err_) {
    const Layout& L = pl.L;
    char* ws = pl.ws;
    const int T = (int)(L.np / UM_MACRO);
    const int full_tiles = T * T, sym_tiles = T * (T + 1) / 2;
    grid_full = 2 * (full_tiles < pl.pairs() ? full_tiles : pl.pairs());
    grid_sym = 2 * (sym_tiles < pl.pairs() ? sym_tiles : pl.pairs());
    st = reinterpret_cast<State*>(ws + L.off_state);
    stop.st = st; stop.partials = reinterpret_cast<double*>(ws + L.off_partials);
    stop.d_err = d_err; stop.max_iter = max_iter; stop.stop = stop_rule; stop.order = 2; stop.cond = cond; stop.extra = pl.opt->extra_update;
    stop.nocheck = pl.opt->final_check ? 0 : 1; stop.floor = ldexp(1.0, -53) * sqrt((double)L.n);
    R32s = reinterpret_cast<float*>(ws + L.off_R32);
    np2 = (size_t)L.np * (size_t)L.np;
    // I8 engine on 256 x 128 tiles: -1 (default) up to 6 x 6 macro tiles (4 updates, wide -> narrow: N = 512 / 1024 / 1536
    // 1.56 / 2.16 / 2.83 -> 1.19 / 1.74 / 2.34 ms; N = 2048 / 3072 +5 / +15 %)
    i8_narrow = (L.mode == ZFAC_MODE_F64_I8) && (pl.opt->i8_narrow >= 0 ? pl.opt->i8_narrow != 0 : T <= 6);
  }
  bool i8_narrow = false;
  int i8_grid(int wide_tiles) const {
    const int tiles = wide_tiles * (i8_narrow ? 2 : 1);
    return 2 * (tiles < pl.pairs() ? tiles : pl.pairs());
  }

  void residual(int n_stop, int tagn, cudaStream_t s, Prof* prof, bool skip_a1 = false) {
    const Layout& L = pl.L;
    char* ws = pl.ws;
    stop.n_iter = n_stop;
    if (stop.nocheck && stop.stop == ZFAC_STOP_PAPER) { finish_kernel<<<1, 1, 0, s>>>(st, d_err); ++nl; }
    if (L.mode == ZFAC_MODE_F64_MIXED) {
      const int tiles = (int)(L.np / F64_BM);
      F64TParams P{};
      F64Params& q = P.q;
      q.ld = (int)L.np; q.K = (int)L.np; q.tiles = tiles; q.st = st; q.pc = poly_coef(2);
      q.stop = stop; q.stop.num_partials = tiles * (tiles + 1) / 2;
      P.mapA = pl.f64.mW; P.mapB = pl.f64.mS; q.out0 = reinterpret_cast<double*>(ws + L.off_T);
      if (prof) prof->mark(s, EPI_A1 + 16 * tagn);
      f64_tma_launch(EPI_A1, tiles * tiles, s, P);
      P.mapA = pl.f64.mW; P.mapB = pl.f64.mT; q.out0 = reinterpret_cast<double*>(ws + L.off_R);
      if (prof) prof->mark(s, EPI_A2 + 16 * tagn);
      f64_tma_launch(EPI_A2, tiles * (tiles + 1) / 2, s, P);
      nl += 2;
      if (stop.cond) graph_cond_kernel<<<1, 1, 0, s>>>(st, stop.cond);
    } else {
      I8Params p{};
      // rasterisation band of the full GEMM: half the width of the fp16 kernels' (their operand rows are twice as long in
      // bytes per slice pass here; measured 2 / 4 / 8 / 16 / 32 columns: 11.9 / 11.85 / 12.3 / 12.9 / 14.1 ms at N = 8192)
      p.np = (int)L.np; p.macro_tiles = (int)(L.np / UM_MACRO); p.band = pl.opt->band > 1 ? pl.opt->band / 2 : 1;
      p.sa = p.sb = p.orders = pl.opt->i8_slices;
      p.scratch = reinterpret_cast<double*>(ws + L.off_scratch);
      p.st = st; p.stop = stop;
      p.stop.num_partials = 16 * (i8_narrow ? 2 : 1) * p.macro_tiles * (p.macro_tiles + 1) / 2;           // a2: 16 per tile
      int* eS = reinterpret_cast<int*>(ws + L.off_exp);
      int* eW = eS + L.np; int* eT = eW + L.np;
      // a1: T = W S^T (FP64 out), then its rows sliced for a2
      p.mapA = pl.mW8; p.mapB = pl.mS8; p.expA = eW; p.expB = eS; p.out64 = reinterpret_cast<double*>(ws + L.off_T);
      if (prof) prof->mark(s, EPI_A1 + 16 * tagn);
      if (!skip_a1) {
      // clusters of two pairs (B slices shared by TMA multicast) when the option is on and the tile rows pair up
      int quads = pl.max_quads;
      if (pl.opt->max_pairs > 0 && pl.opt->max_pairs / 2 < quads) quads = pl.opt->max_pairs / 2;
      if (2 * quads * 2 > I8_SCRATCH_CTAS) quads = I8_SCRATCH_CTAS / 4;
      if (pl.opt->i8_cluster && !i8_narrow && quads > 0 && p.macro_tiles % 2 == 0) {
        const int super_tiles = (p.macro_tiles / 2) * p.macro_tiles;
        const int nq = super_tiles < quads ? super_tiles : quads;
        i8_gemm_kernel<EPI_A1, 2><<<4 * nq, UM_THREADS, UM_SMEM_BYTES, s>>>(p);
      } else if (i8_narrow)
      i8_gemm_kernel<EPI_A1, 1, 128><<<i8_grid(p.macro_tiles * p.macro_tiles), UM_THREADS, UM_SMEM_BYTES, s>>>(p);
      else
      i8_gemm_kernel<EPI_A1><<<grid_full, UM_THREADS, UM_SMEM_BYTES, s>>>(p);
      ++nl;
      }
      slice_rows_kernel<double><<<small_grid((size_t)L.np), 256, 0, s>>>(p.out64, L.np, (int)L.np, (int)L.np, p.orders,
                                                                 reinterpret_cast<int8_t*>(ws + L.off_T8), eT, st);
      // a2: R = I - W T^T (FP32 out, both triangles), sum R^2, stop test
      p.mapA = pl.mW8; p.mapB = pl.mT8; p.expA = eW; p.expB = eT; p.out64 = nullptr; p.out32 = reinterpret_cast<float*>(ws + L.off_R);
      if (prof) prof->mark(s, EPI_A2 + 16 * tagn);
      if (i8_narrow) i8_gemm_kernel<EPI_A2, 1, 128><<<i8_grid(p.macro_tiles * (p.macro_tiles + 1) / 2), UM_THREADS, UM_SMEM_BYTES, s>>>(p);
      else i8_gemm_kernel<EPI_A2><<<grid_sym, UM_THREADS, UM_SMEM_BYTES, s>>>(p);
      nl += 2;
      if (stop.cond) graph_cond_kernel<<<1, 1, 0, s>>>(st, stop.cond);
    }
  }

  void update(int par, int n_stop, int tagn, cudaStream_t s, Prof* prof, const IterHook* = nullptr, int = 1) {
    const Layout& L = pl.L;
    char* ws = pl.ws;
    const unsigned g8 = small_grid((np2 / 8 + 255) / 256);
    __half* Rb = reinterpret_cast<__half*>(ws + L.off_Rb);
    if (prof) prof->mark(s, EPI_A4 + 16 * tagn);
    if (L.mode == ZFAC_MODE_F64_MIXED)
      r_split_kernel<double><<<g8, 256, 0, s>>>(reinterpret_cast<const double*>(ws + L.off_R), R32s, Rb, np2, st, d_err, n_stop);
    else
      r_split_kernel<float><<<g8, 256, 0, s>>>(reinterpret_cast<const float*>(ws + L.off_R), R32s, Rb, np2, st, d_err, n_stop);
    UmmaParams p{};
    p.np = (int)L.np; p.batch = 1; p.rows = (int)L.np; p.macro_tiles = (int)(L.np / UM_MACRO); p.band = pl.opt->band; p.st = st;
    p.stop = stop; p.stop.n_iter = n_stop; p.stop.err_stride = 0;
    const PolyCoef pc = poly_coef(2);
    p.q_r = (float)pc.q_r; p.q_d = (float)pc.q_d; p.scaled = 1;
    // a4: Q~ = 1/2 R~ + (3/8 / rscale) R~ R~^T
    p.hh_only = pl.opt->hh_square ? 1 : 0; p.hh_err_max = pl.opt->hh_square_err;
    p.mapA = pl.mR; p.mapB = pl.mR; p.f32_in = R32s; p.h_out = ws + L.off_Qb;
    umma_launch<KIND_F16X2>(EPI_A4, grid_sym, s, p);
    // a5x: Z64 += (Z Q~^T) / rscale; operand pair of the new Z; DMMA engine: W64 = Z^T
    if (prof) prof->mark(s, EPI_A5 + 16 * tagn);
    p.hh_only = 0; p.f32_in = nullptr;
    p.mapA = pl.mZ[par]; p.mapB = pl.mQ;
    p.z64 = reinterpret_cast<double*>(ws + L.off_Z[0]); p.h_out = ws + L.off_Zb[(par + 1) & 1];
    p.w64t = (L.mode == ZFAC_MODE_F64_MIXED) ? reinterpret_cast<double*>(ws + L.off_W) : nullptr;
    umma_launch<KIND_F16X2>(EPI_A5X, grid_full, s, p);
    nl += 3;
    if (L.mode == ZFAC_MODE_F64_I8) { w_slices(s); }
  }

  // I8 engine, zfac_refine_host: the rows [256 mc0, 256 (mc0 + mcn)) of S (at d_S, element type float if in_f32) are sliced
  // and the tile columns [mc0, mc0 + mcn) of T = W S^T computed from them.  Tiles do not overlap between bands and every
  // element is formed as in the full launch: bit-identical to it.
  void a1_band(const void* d_S, int64_t lds, bool in_f32, int n, int mc0, int mcn, cudaStream_t s) {
    const Layout& L = pl.L;
    char* ws = pl.ws;
    int* eS = reinterpret_cast<int*>(ws + L.off_exp);
    int8_t* S8 = reinterpret_cast<int8_t*>(ws + L.off_S8);
    const int row0 = mc0 * UM_MACRO, rows = mcn * UM_MACRO;
    if (in_f32) slice_rows_kernel<float><<<small_grid((size_t)rows), 256, 0, s>>>(static_cast<const float*>(d_S), lds, n, (int)L.np, pl.opt->i8_slices, S8, eS, st, row0, rows);
    else slice_rows_kernel<double><<<small_grid((size_t)rows), 256, 0, s>>>(static_cast<const double*>(d_S), lds, n, (int)L.np, pl.opt->i8_slices, S8, eS, st, row0, rows);
    I8Params p{};
    p.np = (int)L.np; p.macro_tiles = (int)(L.np / UM_MACRO); p.band = pl.opt->band > 1 ? pl.opt->band / 2 : 1;
    p.sa = p.sb = p.orders = pl.opt->i8_slices;
    p.scratch = reinterpret_cast<double*>(ws + L.off_scratch);
    p.st = st; p.stop = stop;
    p.mapA = pl.mW8; p.mapB = pl.mS8; p.expA = eS + L.np; p.expB = eS; p.out64 = reinterpret_cast<double*>(ws + L.off_T);
    p.joff = mc0; p.jcols = mcn;
    const int tiles = p.macro_tiles * mcn;
    if (i8_narrow) i8_gemm_kernel<EPI_A1, 1, 128><<<i8_grid(tiles), UM_THREADS, UM_SMEM_BYTES, s>>>(p);
    else i8_gemm_kernel<EPI_A1><<<2 * (tiles < pl.pairs() ? tiles : pl.pairs()), UM_THREADS, UM_SMEM_BYTES, s>>>(p);
    nl += 2;
  }

  // I8 engine: W = Z^T as int8 slices (column maxima of Z, then transposed slicing)
  void w_slices(cudaStream_t s) {
    const Layout& L = pl.L;
    char* ws = pl.ws;
    int* eW = reinterpret_cast<int*>(ws + L.off_exp) + L.np;
    const double* Z = reinterpret_cast<const double*>(ws + L.off_Z[0]);
    colmax_kernel<<<(unsigned)(L.np / 32), 256, 0, s>>>(Z, (int)L.np, eW, st);
    slice_transpose_kernel<<<small_grid((size_t)(L.np / 64) * (size_t)(L.np / 64)), 256, 0, s>>>(Z, (int)L.np, pl.opt->i8_slices, reinterpret_cast<int8_t*>(ws + L.off_W8), eW, st);
    nl += 2;
  }
};

}  // namespace zfac
