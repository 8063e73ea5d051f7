// FP64 mode (the paper's `double` scheme, Table I) on the FP64 tensor pipe: shared definitions.
//
// tcgen05.mma has no f64 kind on sm_100a, so this mode uses warp-level mma.sync.m8n8k4.f64 (SASS: DMMA.8x8x4) with
// register accumulators; the kernel itself (TMA-fed shared-memory stages, per-stage mbarriers) is in zfac_f64_tma.cuh.
// All four GEMMs of an iteration are brought to the one form  D[m][n] = sum_k A[m][k] * B[n][k]  (both operands
// K-major, row-major storage) by keeping W = Z^T next to Z:
//   a1  T = (S Z)^T  : A = W, B = S         T[m][n] = sum_k Z[k][m] S[n][k]        (Eq. 22)
//   a2  X = Z^T (SZ) : A = W, B = T         X[m][n] = sum_k Z[k][m] (SZ)[k][n]      (Eq. 26)
//   a4  P = R R      : A = R, B = R         (R symmetric)                           (Eq. 30)
//   a5  Z Q          : A = Z, B = Q         (Q symmetric)                           (Eq. 13)
// Epilogues are fused: a2 forms R = I - X, mirrors the tile (X symmetric: only the upper triangle of tiles is
// computed) and reduces sum R^2; a4 forms Q = 1/2 R + 3/8 P and mirrors; a5 forms Z + ZQ and also stores its transpose W.
#pragma once
#include "zfac_common.cuh"

namespace zfac {

constexpr int F64_BM = 128, F64_BN = 128, F64_BK = 16;   // CTA tile; 8 warps x (64 x 32)
constexpr int F64_THREADS = 256;

enum { EPI_A1 = 1, EPI_A2 = 2, EPI_X3 = 3 /* X = Z^T H Z itself (congruence, Eq. 11) */, EPI_A4 = 4, EPI_A5 = 5,
       EPI_P2 = 6 /* order m > 2: P = R R and G = 3/8 I + 5/16 R (+ 35/128 P), both mirrored */,
       EPI_A5X = 7 /* FP64-master modes: Z64 += (Z Q~) / rscale, next FP32 operand pair of Z, optional W64 = Z^T */ };

// Polynomial coefficients of step a4 (Eq. 13 / 16 with order m; c_k = C(2k,k)/4^k, zfac.h):
//   m = 2:  Q = 1/2 R + 3/8 (R R)                                   one symmetric GEMM   (EPI_A4, q_d = 3/8)
//   m > 2:  P = R R,  G = 3/8 I + 5/16 R + g_p P                     (EPI_P2)
//           Q = 1/2 R + P G        (P and G commute: symmetric)      (EPI_A4, q_d = 1)
struct PolyCoef {
  double q_r;   // EPI_A4: weight of R            (1/2)
  double q_d;   // EPI_A4: weight of the product  (3/8 for m = 2, 1 for m > 2)
  double g_i;   // EPI_P2: weight of I in G       (3/8)
  double g_r;   // EPI_P2: weight of R in G       (5/16)
  double g_p;   // EPI_P2: weight of P in G       (35/128 for m = 4, 0 for m = 3)
};
inline PolyCoef poly_coef(int order) {
  PolyCoef c;
  c.q_r = 0.5; c.q_d = (order == 2) ? 0.375 : 1.0;
  c.g_i = 0.375; c.g_r = 0.3125; c.g_p = (order >= 4) ? 35.0 / 128.0 : 0.0;
  return c;
}

struct F64Params {
  int ld;               // = Np
  int K;                // = Np
  int tiles;            // Np / 128
  State* st;
  double* out0;         // a1: T   a2: R   a4: Q   a5: Z_next   p2: P
  double* out1;         // a5: W   p2: G
  const double* in0;    // a4: R   a5: Z_cur   p2: R
  PolyCoef pc;          // a4, p2
  StopArgs stop;        // a2 only
};

__device__ __forceinline__ void dmma8x8x4(double& d0, double& d1, double a, double b) {
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
               : "+d"(d0), "+d"(d1)
               : "d"(a), "d"(b));
}

}  // namespace zfac
