// FP64 mode (the paper's `double` scheme, Table I) on the FP64 tensor pipe.
//
// tcgen05.mma has no f64 kind on sm_100a, so this mode uses warp-level
// mma.sync.m8n8k4.f64 (SASS: DMMA.8x8x4) with register accumulators and a cp.async
// multi-stage shared-memory pipeline.  All four GEMMs of an iteration are brought to the one
// form  D[m][n] = sum_k A[m][k] * B[n][k]  (both operands K-major, row-major storage) by
// keeping W = Z^T next to Z:
//   a1  T = (S Z)^T  : A = W, B = S         T[m][n] = sum_k Z[k][m] S[n][k]        (Eq. 22)
//   a2  X = Z^T (SZ) : A = W, B = T         X[m][n] = sum_k Z[k][m] (SZ)[k][n]      (Eq. 26)
//   a4  P = R R      : A = R, B = R         (R symmetric)                           (Eq. 30)
//   a5  Z Q          : A = Z, B = Q         (Q symmetric)                           (Eq. 13)
// Epilogues are fused: a2 forms R = I - X, mirrors the tile (X symmetric: only the upper
// triangle of tiles is computed) and reduces sum R^2; a4 forms Q = 1/2 R + 3/8 P and mirrors;
// a5 forms Z + ZQ and also stores its transpose W.
#pragma once
#include "zfac_common.cuh"

namespace zfac {

constexpr int F64_BM = 128, F64_BN = 128, F64_BK = 16;
constexpr int F64_LDS = F64_BK + 4;          // padded row (doubles): conflict-free 64-bit fragment loads
constexpr int F64_STAGES = 4;
constexpr int F64_THREADS = 256;
constexpr int F64_STAGE_DOUBLES = (F64_BM + F64_BN) * F64_LDS;
constexpr int F64_SMEM_BYTES = F64_STAGES * F64_STAGE_DOUBLES * 8;

enum { EPI_A1 = 1, EPI_A2 = 2, EPI_X3 = 3 /* X = Z^T H Z itself (congruence, Eq. 11) */, EPI_A4 = 4, EPI_A5 = 5,
       EPI_P2 = 6 /* order m > 2: P = R R and G = 3/8 I + 5/16 R (+ 35/128 P), both mirrored */ };

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
  const double* A;      // [Np][ld]
  const double* B;      // [Np][ld]
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

__device__ __forceinline__ void cp_async16(void* smem, const void* gmem) {
  const uint32_t s = (uint32_t)__cvta_generic_to_shared(smem);
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" ::"r"(s), "l"(gmem));
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;\n" ::"n"(N)); }

__device__ __forceinline__ void dmma8x8x4(double& d0, double& d1, double a, double b) {
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
               : "+d"(d0), "+d"(d1)
               : "d"(a), "d"(b));
}

template <int EPI>
__global__ void __launch_bounds__(F64_THREADS, 1) f64_gemm_kernel(const F64Params p) {
  if (*((volatile int*)&p.st->done)) return;       // stop decided earlier in this call

  extern __shared__ __align__(16) unsigned char smem_raw[];
  double* smem = reinterpret_cast<double*>(smem_raw);
  __shared__ double red[32];
  __shared__ int last_flag;

  constexpr bool SYM = (EPI == EPI_A2 || EPI == EPI_A4 || EPI == EPI_X3 || EPI == EPI_P2);
  int tm, tn;
  if (SYM) tri_decode((int)blockIdx.x, tm, tn);
  else band_decode((int)blockIdx.x, p.tiles, p.tiles, 8, tm, tn);
  const int m0 = tm * F64_BM, n0 = tn * F64_BN;

  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int wm = warp >> 2, wn = warp & 3;         // 2 x 4 warps; warp tile 64 x 32
  const int g = lane >> 2, q = lane & 3;

  const double* gA = p.A + (size_t)m0 * p.ld;
  const double* gB = p.B + (size_t)n0 * p.ld;
  const int KT = p.K / F64_BK;

  auto load_stage = [&](int stage, int kt) {
    double* sA = smem + stage * F64_STAGE_DOUBLES;
    double* sB = sA + F64_BM * F64_LDS;
    const int k0 = kt * F64_BK;
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      const int c = tid + i * F64_THREADS;         // 0..1023
      const int row = c >> 3, ck = (c & 7) * 2;
      cp_async16(sA + row * F64_LDS + ck, gA + (size_t)row * p.ld + k0 + ck);
      cp_async16(sB + row * F64_LDS + ck, gB + (size_t)row * p.ld + k0 + ck);
    }
  };

  double acc[8][4][2];
#pragma unroll
  for (int i = 0; i < 8; ++i)
#pragma unroll
    for (int j = 0; j < 4; ++j) acc[i][j][0] = acc[i][j][1] = 0.0;

#pragma unroll
  for (int s = 0; s < F64_STAGES - 1; ++s) {
    if (s < KT) load_stage(s, s);
    cp_async_commit();
  }

  for (int kt = 0; kt < KT; ++kt) {
    cp_async_wait<F64_STAGES - 2>();
    __syncthreads();
    {
      const int nk = kt + F64_STAGES - 1;
      if (nk < KT) load_stage(nk % F64_STAGES, nk);
      cp_async_commit();
    }
    const double* sA = smem + (kt % F64_STAGES) * F64_STAGE_DOUBLES + (wm * 64 + g) * F64_LDS + q;
    const double* sB = smem + (kt % F64_STAGES) * F64_STAGE_DOUBLES + F64_BM * F64_LDS + (wn * 32 + g) * F64_LDS + q;
#pragma unroll
    for (int ks = 0; ks < F64_BK / 4; ++ks) {
      double a[8], b[4];
#pragma unroll
      for (int i = 0; i < 8; ++i) a[i] = sA[i * 8 * F64_LDS + ks * 4];
#pragma unroll
      for (int j = 0; j < 4; ++j) b[j] = sB[j * 8 * F64_LDS + ks * 4];
#pragma unroll
      for (int i = 0; i < 8; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) dmma8x8x4(acc[i][j][0], acc[i][j][1], a[i], b[j]);
    }
  }
  cp_async_wait<0>();

  // ---------------------------------------------------------------- fused epilogues
  // fragment (i, j): rows m = m0 + wm*64 + i*8 + g, cols n = n0 + wn*32 + j*8 + 2q + {0,1}
  const size_t ld = (size_t)p.ld;
  double sumsq = 0.0;
#pragma unroll
  for (int i = 0; i < 8; ++i) {
    const int m = m0 + wm * 64 + i * 8 + g;
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      const int n = n0 + wn * 32 + j * 8 + 2 * q;
      double v0 = acc[i][j][0], v1 = acc[i][j][1];
      if (EPI == EPI_A1) {
        *reinterpret_cast<double2*>(p.out0 + m * ld + n) = make_double2(v0, v1);
      } else if (EPI == EPI_A2) {
        v0 = (m == n ? 1.0 : 0.0) - v0;              // R = I - X
        v1 = (m == n + 1 ? 1.0 : 0.0) - v1;
        sumsq += v0 * v0 + v1 * v1;
        *reinterpret_cast<double2*>(p.out0 + m * ld + n) = make_double2(v0, v1);
        if (tm != tn) { p.out0[(size_t)n * ld + m] = v0; p.out0[(size_t)(n + 1) * ld + m] = v1; }
      } else if (EPI == EPI_X3) {
        *reinterpret_cast<double2*>(p.out0 + m * ld + n) = make_double2(v0, v1);
        if (tm != tn) { p.out0[(size_t)n * ld + m] = v0; p.out0[(size_t)(n + 1) * ld + m] = v1; }
      } else if (EPI == EPI_A4) {
        const double2 r = *reinterpret_cast<const double2*>(p.in0 + m * ld + n);
        v0 = p.pc.q_r * r.x + p.pc.q_d * v0;         // Q = 1/2 R + 3/8 R R   (m > 2: 1/2 R + P G)
        v1 = p.pc.q_r * r.y + p.pc.q_d * v1;
        *reinterpret_cast<double2*>(p.out0 + m * ld + n) = make_double2(v0, v1);
        if (tm != tn) { p.out0[(size_t)n * ld + m] = v0; p.out0[(size_t)(n + 1) * ld + m] = v1; }
      } else if (EPI == EPI_P2) {
        const double2 r = *reinterpret_cast<const double2*>(p.in0 + m * ld + n);
        const double g0 = (m == n ? p.pc.g_i : 0.0) + p.pc.g_r * r.x + p.pc.g_p * v0;      // G = 3/8 I + 5/16 R + g_p P
        const double g1 = (m == n + 1 ? p.pc.g_i : 0.0) + p.pc.g_r * r.y + p.pc.g_p * v1;
        *reinterpret_cast<double2*>(p.out0 + m * ld + n) = make_double2(v0, v1);            // P = R R
        *reinterpret_cast<double2*>(p.out1 + m * ld + n) = make_double2(g0, g1);
        if (tm != tn) {
          p.out0[(size_t)n * ld + m] = v0; p.out0[(size_t)(n + 1) * ld + m] = v1;
          p.out1[(size_t)n * ld + m] = g0; p.out1[(size_t)(n + 1) * ld + m] = g1;
        }
      } else {  // EPI_A5
        const double2 z = *reinterpret_cast<const double2*>(p.in0 + m * ld + n);
        v0 += z.x;                                   // Z_next = Z + Z Q
        v1 += z.y;
        *reinterpret_cast<double2*>(p.out0 + m * ld + n) = make_double2(v0, v1);
        p.out1[(size_t)n * ld + m] = v0;             // W = Z_next^T
        p.out1[(size_t)(n + 1) * ld + m] = v1;
      }
    }
  }

  if (EPI == EPI_A2) {
    if (tm != tn) sumsq *= 2.0;                      // the mirrored tile
    sumsq = warp_sum(sumsq);
    if (lane == 0) red[warp] = sumsq;
    __syncthreads();
    if (tid == 0) {
      double t = 0.0;
#pragma unroll
      for (int w = 0; w < F64_THREADS / 32; ++w) t += red[w];
      p.stop.partials[blockIdx.x] = t;
    }
    if (arrive_is_last(&p.st->arrive[0], gridDim.x, &last_flag)) stop_test_last_cta(p.stop, red);
  }
}

}  // namespace zfac
