// FP64 mode, main loop fed by TMA (replaces the cp.async + __syncthreads loop of f64_gemm_kernel).
//
// Same product form, tiling (128 x 128 x 16 CTA tile, 8 warps x (64 x 32), mma.sync.m8n8k4.f64 = DMMA.8x8x4,
// register accumulators) and the same fused epilogues as zfac_f64.cuh -- only the way the operand tiles reach
// shared memory and the way the warps synchronise change:
//   * each stage holds an A tile and a B tile of 128 rows x 16 doubles (= 128 bytes per row), written by TMA
//     (cp.async.bulk.tensor.2d, boxes of 64 rows) with the 128-byte swizzle: the 16-byte chunk c of row r lands at
//     chunk c ^ (r & 7).  The m8n8k4 fragment load (8 rows g x 4 k-values q per instruction) then touches, per
//     half-warp wavefront, the eight different chunks (2 ks + (q >> 1)) ^ g: conflict-free without padding;
//   * a full / empty mbarrier pair per stage instead of one __syncthreads per k-tile: a warp waits for DATA only,
//     never for the other warps, so the FP64 tensor pipe does not drain once per k-tile;
//   * the loads are issued by lane 0 of warp 0, F64T_DIST k-tiles ahead, into the stage that was consumed two k-tiles
//     ago (its wait on that stage's empty barrier is normally already satisfied).  No dedicated producer warp: a
//     ninth warp would put three warps on one SM sub-partition and cap every thread at 168 registers.
#pragma once
#include "zfac_f64.cuh"
#include "zfac_umma.cuh"   // smem_u32, mbar_*, make_map, PFN_encodeTiled

namespace zfac {

constexpr int F64T_STAGES = 6;
constexpr int F64T_DIST = F64T_STAGES - 2;                   // prefetch distance in k-tiles
constexpr int F64T_TILE_BYTES = F64_BM * F64_BK * 8;         // 16 KB: 128 rows x 128 bytes
constexpr int F64T_STAGE_BYTES = 2 * F64T_TILE_BYTES;        // A + B
constexpr int F64T_SMEM_BYTES = F64T_STAGES * F64T_STAGE_BYTES + 1024 /*align*/ + 128 /*barriers*/;
static_assert(F64_BK * 8 == 128, "one k-tile row is one 128-byte swizzle span");

struct F64TParams {
  CUtensorMap mapA, mapB;   // [Np rows][Np cols] FP64, box 16 x 64, 128B swizzle
  F64Params q;              // everything else (pointers for the epilogues, stop test)
};

__device__ __forceinline__ void tma_load_2d(uint32_t dst, const CUtensorMap* map, int c0, int c1, uint32_t bar) {
  asm volatile(
      "cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];"
      ::"r"(dst), "l"(reinterpret_cast<uint64_t>(map)), "r"(c0), "r"(c1), "r"(bar)
      : "memory");
}
__device__ __forceinline__ void mbar_arrive_cta(uint32_t bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ double lds_f64(uint32_t addr) {
  double v;
  asm volatile("ld.shared.f64 %0, [%1];" : "=d"(v) : "r"(addr));
  return v;
}

template <int EPI>
__global__ void __launch_bounds__(F64_THREADS, 1) f64_tma_gemm_kernel(const __grid_constant__ F64TParams P) {
  const F64Params& p = P.q;
  if (*((volatile int*)&p.st->done)) return;       // stop decided earlier in this call

  extern __shared__ unsigned char smem_raw[];
  const uint32_t smem_base = (smem_u32(smem_raw) + 1023u) & ~1023u;
  const uint32_t bar_base = smem_base + F64T_STAGES * F64T_STAGE_BYTES;
  auto full_bar = [&](int s) { return bar_base + 8u * s; };
  auto empty_bar = [&](int s) { return bar_base + 8u * (F64T_STAGES + s); };
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
  const int KT = p.K / F64_BK;

  if (tid == 0) {
    for (int s = 0; s < F64T_STAGES; ++s) { mbar_init(full_bar(s), 1); mbar_init(empty_bar(s), F64_THREADS / 32); }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    asm volatile("prefetch.tensormap [%0];" ::"l"(reinterpret_cast<uint64_t>(&P.mapA)) : "memory");
    asm volatile("prefetch.tensormap [%0];" ::"l"(reinterpret_cast<uint64_t>(&P.mapB)) : "memory");
  }
  __syncthreads();

  auto issue = [&](int kt) {                       // one thread: fill stage kt % STAGES with k-tile kt
    const int s = kt % F64T_STAGES;
    const uint32_t sa = smem_base + s * F64T_STAGE_BYTES, sb = sa + F64T_TILE_BYTES;
    mbar_expect_tx(full_bar(s), F64T_STAGE_BYTES);
    const int kc = kt * F64_BK;
#pragma unroll
    for (int b = 0; b < F64_BM / UM_BOX_ROWS; ++b) {
      tma_load_2d(sa + b * UM_BOX_BYTES, &P.mapA, kc, m0 + b * UM_BOX_ROWS, full_bar(s));
      tma_load_2d(sb + b * UM_BOX_BYTES, &P.mapB, kc, n0 + b * UM_BOX_ROWS, full_bar(s));
    }
  };
  if (tid == 0) {
    for (int kt = 0; kt < F64T_DIST && kt < KT; ++kt) issue(kt);
  }

  double acc[8][4][2];
#pragma unroll
  for (int i = 0; i < 8; ++i)
#pragma unroll
    for (int j = 0; j < 4; ++j) acc[i][j][0] = acc[i][j][1] = 0.0;

  // swizzled fragment addresses: row r = (multiple of 8) + g, so r & 7 = g; element k = 4 ks + q sits in the 16-byte
  // chunk (2 ks + (q >> 1)) ^ g of the row, at byte (q & 1) * 8 inside it
  const uint32_t a_row = (uint32_t)(wm * 64 + g) * 128u, b_row = (uint32_t)F64T_TILE_BYTES + (uint32_t)(wn * 32 + g) * 128u;
  const uint32_t sub = (uint32_t)(q & 1) * 8u, qh = (uint32_t)(q >> 1);

  for (int kt = 0; kt < KT; ++kt) {
    if (tid == 0) {
      const int nk = kt + F64T_DIST;
      if (nk < KT) {
        if (nk >= F64T_STAGES) mbar_wait(empty_bar(nk % F64T_STAGES), (uint32_t)((nk / F64T_STAGES - 1) & 1));
        issue(nk);
      }
    }
    __syncwarp();
    const int s = kt % F64T_STAGES;
    mbar_wait(full_bar(s), (uint32_t)((kt / F64T_STAGES) & 1));
    const uint32_t st = smem_base + s * F64T_STAGE_BYTES;
#pragma unroll
    for (int ks = 0; ks < F64_BK / 4; ++ks) {
      const uint32_t coff = ((((uint32_t)(2 * ks) + qh) ^ (uint32_t)g) << 4) + sub;
      double a[8], b[4];
#pragma unroll
      for (int i = 0; i < 8; ++i) a[i] = lds_f64(st + a_row + (uint32_t)i * 1024u + coff);
#pragma unroll
      for (int j = 0; j < 4; ++j) b[j] = lds_f64(st + b_row + (uint32_t)j * 1024u + coff);
#pragma unroll
      for (int i = 0; i < 8; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) dmma8x8x4(acc[i][j][0], acc[i][j][1], a[i], b[j]);
    }
    __syncwarp();
    if (lane == 0) mbar_arrive_cta(empty_bar(s));   // this warp is done with the stage
  }

  // ---------------------------------------------------------------- fused epilogues (as in f64_gemm_kernel)
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

// Tensor maps of the seven FP64 buffers of a ZFAC_MODE_F64 context.
struct F64Plan {
  CUtensorMap mS, mW, mT, mR, mQ, mZ[2];
};

inline cudaError_t f64_plan_create(F64Plan* pl, const Layout& L, char* ws) {
  void* fn = nullptr;
  cudaDriverEntryPointQueryResult qres;
  cudaError_t e = cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres);
  if (e != cudaSuccess) return e;
  if (!fn || qres != cudaDriverEntryPointSuccess) return cudaErrorNotSupported;
  PFN_encodeTiled enc = reinterpret_cast<PFN_encodeTiled>(fn);
  const uint64_t np = (uint64_t)L.np;
  const CUtensorMapDataType D = CU_TENSOR_MAP_DATA_TYPE_FLOAT64;
  if ((e = make_map(enc, &pl->mS, ws + L.off_S, D, 8, np, np)) != cudaSuccess) return e;
  if ((e = make_map(enc, &pl->mW, ws + L.off_W, D, 8, np, np)) != cudaSuccess) return e;
  if ((e = make_map(enc, &pl->mT, ws + L.off_T, D, 8, np, np)) != cudaSuccess) return e;
  if ((e = make_map(enc, &pl->mR, ws + L.off_R, D, 8, np, np)) != cudaSuccess) return e;
  if ((e = make_map(enc, &pl->mQ, ws + L.off_Q, D, 8, np, np)) != cudaSuccess) return e;
  if ((e = make_map(enc, &pl->mZ[0], ws + L.off_Z[0], D, 8, np, np)) != cudaSuccess) return e;
  if ((e = make_map(enc, &pl->mZ[1], ws + L.off_Z[1], D, 8, np, np)) != cudaSuccess) return e;
  return cudaSuccess;
}

template <int EPI>
inline cudaError_t f64_tma_prepare() {
  return cudaFuncSetAttribute(f64_tma_gemm_kernel<EPI>, cudaFuncAttributeMaxDynamicSharedMemorySize, F64T_SMEM_BYTES);
}

inline void f64_tma_launch(int epi, int grid, cudaStream_t s, const F64TParams& P) {
  switch (epi) {
    case EPI_A1: f64_tma_gemm_kernel<EPI_A1><<<grid, F64_THREADS, F64T_SMEM_BYTES, s>>>(P); break;
    case EPI_A2: f64_tma_gemm_kernel<EPI_A2><<<grid, F64_THREADS, F64T_SMEM_BYTES, s>>>(P); break;
    case EPI_X3: f64_tma_gemm_kernel<EPI_X3><<<grid, F64_THREADS, F64T_SMEM_BYTES, s>>>(P); break;
    case EPI_A4: f64_tma_gemm_kernel<EPI_A4><<<grid, F64_THREADS, F64T_SMEM_BYTES, s>>>(P); break;
    case EPI_P2: f64_tma_gemm_kernel<EPI_P2><<<grid, F64_THREADS, F64T_SMEM_BYTES, s>>>(P); break;
    default:     f64_tma_gemm_kernel<EPI_A5><<<grid, F64_THREADS, F64T_SMEM_BYTES, s>>>(P); break;
  }
}

}  // namespace zfac
