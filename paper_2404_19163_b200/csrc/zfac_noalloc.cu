// zfac_residual_norm_noalloc: Err = || I - Z^T (S Z) ||_F  (Alg. 2; Eq. 22-29) for a given S and Z,
// FP64, WITHOUT a context, a workspace or any allocation -- for callers that cannot call cudaMalloc (code under CUDA graph
// capture, tight serving loops, harnesses that forbid it).  It is the check a consumer makes on a Z it holds ("is this still
// an inverse factor of the S of this MD step, or must it be refined?").
//
// The library's regular path (zfac_refine, max_iter = 0) evaluates the same quantity with its steps a1 (T = S Z), a2
// (R = I - Z^T T, sum of squares per tile) and a3 (last CTA adds the partial sums) in a caller-provided workspace.  The
// kernels here are the variant of a2 + a3 whose scratch -- T, the per-CTA partial sums and the arrival counter -- lives in a
// file-scope device array of fixed size instead:
//
//     static __device__ __align__(256) g_scratch : ZFAC_NOALLOC_MAX_N^2 doubles (T) + 4096 doubles (partials) + 256 B
//     = 8 MiB + 32 KiB + 256 B, held by every GPU that loads libzfac.so until the process exits.
//
// Every call on a device shares that array.  Nothing in it has to survive between calls; the arrival counter, the one word
// that must start at zero, is cleared by a memset on the caller's stream at the head of every call.  Two calls that OVERLAP
// on the GPU (different streams, or concurrent host threads on different streams) race on the array: serialise them (same
// stream, or an event between them).  Calls on different devices do not interact (one array per device).
//
// Plain FP64 SIMT kernels (64 x 64 tiles, 4 x 4 per thread): at n <= 1024 the two products are 4.3 GFLOP, ~1 ms; this is
// a utility, not the hot path, which stays in zfac_umma.cuh / zfac_f64_tma.cuh / zfac_mix.cuh.
#include <cuda_runtime.h>

#include <cstdint>
#include <cstdio>
#include <mutex>

#include "../../include/zfac.h"

namespace {

constexpr int NA_MAX_N = ZFAC_NOALLOC_MAX_N;           // include/zfac.h: 1024
constexpr int NA_TILE = 64;                            // output tile of one CTA
constexpr int NA_KB = 16;                              // k-block
constexpr int NA_MAX_TILES = (NA_MAX_N / NA_TILE) * (NA_MAX_N / NA_TILE);      // 256 partial sums at most
constexpr size_t NA_T_DOUBLES = (size_t)NA_MAX_N * NA_MAX_N;
constexpr size_t NA_PART_DOUBLES = 4096;               // >= NA_MAX_TILES, keeps the counter 256-byte aligned
constexpr size_t NA_SCRATCH_DOUBLES = NA_T_DOUBLES + NA_PART_DOUBLES + 32;    // + 256 B: arrival counter
static_assert(NA_MAX_TILES <= (int)NA_PART_DOUBLES, "partials");

// The scratch.  In HOST code this name is a host-side stand-in, not a device address: the address handed to the kernels comes
// from cudaGetSymbolAddress (scratch_for_current_device below).
static __device__ __align__(256) double g_scratch[NA_SCRATCH_DOUBLES];

static thread_local char g_err[256] = "";

// C[i][j] = sum_k A(i,k) B(k,j) on a 64 x 64 tile; A(i,k) = TRANS_A ? a[k * lda + i] : a[i * lda + k]; B row-major.
// Rows / columns / k beyond n read as zero.  Thread (ty, tx) of 16 x 16 owns rows ty * 4 .. + 3, columns tx * 4 .. + 3.
template <bool TRANS_A>
__device__ __forceinline__ void tile_product(const double* __restrict__ a, int64_t lda, const double* __restrict__ b, int64_t ldb,
                                             int n, int i0, int j0, double (&acc)[4][4], double (*sA)[NA_TILE + 1],
                                             double (*sB)[NA_TILE + 1]) {
  const int t = threadIdx.x, tx = t & 15, ty = t >> 4;
#pragma unroll
  for (int r = 0; r < 4; ++r)
#pragma unroll
    for (int c = 0; c < 4; ++c) acc[r][c] = 0.0;
  for (int k0 = 0; k0 < n; k0 += NA_KB) {
    // stage A as sA[k][i] and B as sB[k][j]: 16 x 64 each, 4 elements per thread
#pragma unroll
    for (int e = 0; e < 4; ++e) {
      const int idx = t + 256 * e;                                  // 0 .. 1023
      if (TRANS_A) {
        const int k = idx >> 6, i = idx & 63;                       // consecutive threads: consecutive i (contiguous in memory)
        const int gk = k0 + k, gi = i0 + i;
        sA[k][i] = (gk < n && gi < n) ? a[(int64_t)gk * lda + gi] : 0.0;
      } else {
        const int i = idx >> 4, k = idx & 15;                       // consecutive threads: consecutive k (contiguous in memory)
        const int gk = k0 + k, gi = i0 + i;
        sA[k][i] = (gk < n && gi < n) ? a[(int64_t)gi * lda + gk] : 0.0;
      }
      const int kb = idx >> 6, j = idx & 63;
      const int gkb = k0 + kb, gj = j0 + j;
      sB[kb][j] = (gkb < n && gj < n) ? b[(int64_t)gkb * ldb + gj] : 0.0;
    }
    __syncthreads();
#pragma unroll
    for (int k = 0; k < NA_KB; ++k) {
      double av[4], bv[4];
#pragma unroll
      for (int r = 0; r < 4; ++r) av[r] = sA[k][ty * 4 + r];
#pragma unroll
      for (int c = 0; c < 4; ++c) bv[c] = sB[k][tx * 4 + c];
#pragma unroll
      for (int r = 0; r < 4; ++r)
#pragma unroll
        for (int c = 0; c < 4; ++c) acc[r][c] = fma(av[r], bv[c], acc[r][c]);
    }
    __syncthreads();
  }
}

// Step a1 of the variant: T = S Z into the scratch (row-major, leading dimension n).
__global__ void __launch_bounds__(256) noalloc_sz_kernel(const double* __restrict__ S, int64_t lds, const double* __restrict__ Z,
                                                         int64_t ldz, int n, double* __restrict__ T) {
  __shared__ double sA[NA_KB][NA_TILE + 1];
  __shared__ double sB[NA_KB][NA_TILE + 1];
  const int i0 = blockIdx.y * NA_TILE, j0 = blockIdx.x * NA_TILE;
  double acc[4][4];
  tile_product<false>(S, lds, Z, ldz, n, i0, j0, acc, sA, sB);
  const int tx = threadIdx.x & 15, ty = threadIdx.x >> 4;
#pragma unroll
  for (int r = 0; r < 4; ++r)
#pragma unroll
    for (int c = 0; c < 4; ++c) {
      const int i = i0 + ty * 4 + r, j = j0 + tx * 4 + c;
      if (i < n && j < n) T[(int64_t)i * n + j] = acc[r][c];
    }
}

// Steps a2 + a3 of the variant: X = Z^T T tile by tile, sum of (delta_ij - X_ij)^2 per CTA into partials[]; the CTA that
// arrives last adds the partials in index order with a fixed tree (the result does not depend on which CTA that is) and
// writes Err = sqrt(sum).  It leaves the counter at zero for the next call.
__global__ void __launch_bounds__(256) noalloc_residual_norm_kernel(const double* __restrict__ Z, int64_t ldz,
                                                                    const double* __restrict__ T, int n,
                                                                    double* __restrict__ partials, unsigned int* counter,
                                                                    double* __restrict__ d_err) {
  __shared__ double sA[NA_KB][NA_TILE + 1];
  __shared__ double sB[NA_KB][NA_TILE + 1];
  __shared__ double red[8];
  __shared__ int is_last;
  const int i0 = blockIdx.y * NA_TILE, j0 = blockIdx.x * NA_TILE;
  double acc[4][4];
  tile_product<true>(Z, ldz, T, (int64_t)n, n, i0, j0, acc, sA, sB);
  const int t = threadIdx.x, tx = t & 15, ty = t >> 4, lane = t & 31, warp = t >> 5;
  double ss = 0.0;
#pragma unroll
  for (int r = 0; r < 4; ++r)
#pragma unroll
    for (int c = 0; c < 4; ++c) {
      const int i = i0 + ty * 4 + r, j = j0 + tx * 4 + c;
      if (i < n && j < n) {
        const double rr = ((i == j) ? 1.0 : 0.0) - acc[r][c];
        ss = fma(rr, rr, ss);
      }
    }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) ss += __shfl_xor_sync(0xffffffffu, ss, o);
  if (lane == 0) red[warp] = ss;
  __syncthreads();
  const int nblocks = (int)(gridDim.x * gridDim.y), bid = (int)(blockIdx.y * gridDim.x + blockIdx.x);
  if (t == 0) {
    double tot = 0.0;
    for (int w = 0; w < 8; ++w) tot += red[w];
    partials[bid] = tot;
    __threadfence();
    const unsigned int prev = atomicAdd(counter, 1u);
    is_last = (prev == (unsigned int)(nblocks - 1)) ? 1 : 0;
  }
  __syncthreads();
  if (!is_last) return;
  __threadfence();
  double s = 0.0;
  for (int i = t; i < nblocks; i += 256) s += __ldcg(partials + i);
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
  if (lane == 0) red[warp] = s;
  __syncthreads();
  if (t == 0) {
    double tot = 0.0;
    for (int w = 0; w < 8; ++w) tot += red[w];
    *d_err = sqrt(tot);
    *counter = 0u;
  }
}

// Device address of g_scratch on the CURRENT device: looked up once per device, with that device current.
constexpr int NA_MAX_DEVICES = 64;
static std::mutex g_mu;
static double* g_addr[NA_MAX_DEVICES] = {nullptr};

static cudaError_t scratch_for_current_device(double** out) {
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  if (dev < 0 || dev >= NA_MAX_DEVICES) return cudaErrorInvalidDevice;
  std::lock_guard<std::mutex> lock(g_mu);
  if (!g_addr[dev]) {
    double* p = nullptr;
    e = cudaGetSymbolAddress((void**)&p, g_scratch);
    if (e != cudaSuccess) return e;
    if (!p) return cudaErrorInvalidSymbol;
    g_addr[dev] = p;
  }
  *out = g_addr[dev];
  return cudaSuccess;
}

}  // namespace

extern "C" {

const char* zfac_noalloc_last_error(void) { return g_err; }

zfac_status zfac_residual_norm_noalloc(const double* d_S, int64_t lds, const double* d_Z, int64_t ldz, int64_t n,
                                       double* d_err, void* stream_) {
  cudaStream_t stream = static_cast<cudaStream_t>(stream_);
  g_err[0] = '\0';
  if (!d_S || !d_Z || !d_err) {
    snprintf(g_err, sizeof(g_err), "zfac_residual_norm_noalloc: null pointer argument");
    return ZFAC_E_INVALID;
  }
  if (n < 1 || lds < n || ldz < n) {
    snprintf(g_err, sizeof(g_err), "zfac_residual_norm_noalloc: need n >= 1, lds >= n, ldz >= n (n = %lld, lds = %lld, ldz = %lld)",
             (long long)n, (long long)lds, (long long)ldz);
    return ZFAC_E_INVALID;
  }
  if (n > NA_MAX_N) {
    snprintf(g_err, sizeof(g_err),
             "zfac_residual_norm_noalloc: n = %lld exceeds ZFAC_NOALLOC_MAX_N = %d (the static scratch holds T = S Z for at most "
             "that order); use zfac_create / zfac_refine with a workspace for larger problems",
             (long long)n, NA_MAX_N);
    return ZFAC_E_INVALID;
  }
  double* scratch = nullptr;
  cudaError_t e = scratch_for_current_device(&scratch);
  if (e != cudaSuccess) {
    snprintf(g_err, sizeof(g_err), "zfac_residual_norm_noalloc: cudaGetSymbolAddress: %s", cudaGetErrorString(e));
    return ZFAC_E_CUDA;
  }
  double* T = scratch;
  double* partials = scratch + NA_T_DOUBLES;
  unsigned int* counter = reinterpret_cast<unsigned int*>(scratch + NA_T_DOUBLES + NA_PART_DOUBLES);
  // the one word that must start at zero (a memset node: no allocation, capturable)
  if ((e = cudaMemsetAsync(counter, 0, sizeof(unsigned int), stream)) != cudaSuccess) {
    snprintf(g_err, sizeof(g_err), "zfac_residual_norm_noalloc: cudaMemsetAsync: %s", cudaGetErrorString(e));
    return ZFAC_E_CUDA;
  }
  const int ni = (int)n, tiles = (ni + NA_TILE - 1) / NA_TILE;
  const dim3 grid((unsigned)tiles, (unsigned)tiles);
  noalloc_sz_kernel<<<grid, 256, 0, stream>>>(d_S, lds, d_Z, ldz, ni, T);
  noalloc_residual_norm_kernel<<<grid, 256, 0, stream>>>(d_Z, ldz, T, ni, partials, counter, d_err);
  if ((e = cudaGetLastError()) != cudaSuccess) {
    snprintf(g_err, sizeof(g_err), "zfac_residual_norm_noalloc: launch: %s", cudaGetErrorString(e));
    return ZFAC_E_CUDA;
  }
  return ZFAC_OK;
}

}  // extern "C"
