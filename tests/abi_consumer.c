/* A plain C99 consumer of libzfac.so: exercises the C ABI of include/zfac.h without Python.
 *
 *   gcc -std=c99 -Iinclude -I/usr/local/cuda/include tests/abi_consumer.c -o abi_consumer \
 *       -Lpaper_2404_19163_b200 -lzfac -L/usr/local/cuda/lib64 -lcudart -lm -Wl,-rpath,...
 *
 * Problem: S = tridiagonal-plus-decay SPD matrix of order N (diagonally dominant), Z0 = I / sqrt(bound on lambda_max)
 * (Gershgorin), so ||I - Z0^T S Z0||_2 < 1 (Eq. 14).  Runs Algorithm 2 (zfac_refine) in FP64 and in SPLIT16
 * with the paper's stop rule, and checks the invariant ||Z^T S Z - I||_F / sqrt(N) of the returned Z with plain loops
 * on the host.  Exit code 0 = all checks passed.  tests/test_abi_cpu.py compiles it (no GPU needed);
 * tests/test_parity_gpu.py runs it on the GPU. */
#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include <cuda_runtime_api.h>

#include "zfac.h"

#define N 200

static double invariant(const double* S, const double* Z) {
  /* ||Z^T (S Z) - I||_F / sqrt(N), triple loops */
  static double A[N * N];
  double ss = 0.0;
  for (int i = 0; i < N; ++i)
    for (int j = 0; j < N; ++j) {
      double a = 0.0;
      for (int k = 0; k < N; ++k) a += S[i * N + k] * Z[k * N + j];
      A[i * N + j] = a;
    }
  for (int i = 0; i < N; ++i)
    for (int j = 0; j < N; ++j) {
      double x = 0.0;
      for (int k = 0; k < N; ++k) x += Z[k * N + i] * A[k * N + j];
      x -= (i == j) ? 1.0 : 0.0;
      ss += x * x;
    }
  return sqrt(ss / N);
}

static int run_mode(zfac_mode mode, const double* S64, const double* Z064, double gate) {
  const size_t elt = (mode == ZFAC_MODE_F64) ? 8 : 4;
  const size_t bytes = zfac_workspace_bytes(N, mode);
  void *ws = NULL, *dS = NULL, *dZ0 = NULL, *dZ = NULL;
  int *dInts = NULL;
  double* dErr = NULL;
  enum { MAXIT = 30 };
  if (bytes == 0) { fprintf(stderr, "workspace_bytes = 0\n"); return 1; }
  if (cudaMalloc(&ws, bytes) || cudaMalloc(&dS, N * N * elt) || cudaMalloc(&dZ0, N * N * elt) || cudaMalloc(&dZ, N * N * elt) ||
      cudaMalloc((void**)&dInts, 2 * sizeof(int)) || cudaMalloc((void**)&dErr, (MAXIT + 1) * sizeof(double))) {
    fprintf(stderr, "cudaMalloc failed\n");
    return 1;
  }
  void* hS = malloc(N * N * elt);
  void* hZ = malloc(N * N * elt);
  for (int i = 0; i < N * N; ++i) {
    if (elt == 8) { ((double*)hS)[i] = S64[i]; ((double*)hZ)[i] = Z064[i]; }
    else { ((float*)hS)[i] = (float)S64[i]; ((float*)hZ)[i] = (float)Z064[i]; }
  }
  cudaMemcpy(dS, hS, N * N * elt, cudaMemcpyHostToDevice);
  cudaMemcpy(dZ0, hZ, N * N * elt, cudaMemcpyHostToDevice);

  zfac_ctx* ctx = NULL;
  zfac_status st = zfac_create(&ctx, N, mode, ws, bytes);
  if (st != ZFAC_OK) { fprintf(stderr, "zfac_create: %s %s\n", zfac_status_string(st), zfac_last_cuda_error()); return 1; }
  double v = -1.0;
  if (zfac_get_option(ctx, ZFAC_OPT_CHUNK_KB, &v) != ZFAC_OK || v != 1.0) { fprintf(stderr, "option default\n"); return 1; }
  if (zfac_set_option(ctx, (zfac_option)99, 1.0) != ZFAC_E_INVALID) { fprintf(stderr, "unknown option accepted\n"); return 1; }
  if (zfac_refine(ctx, dS, N - 1, dZ0, N, dZ, N, MAXIT, ZFAC_STOP_PAPER, dInts, dErr, dInts + 1, NULL) != ZFAC_E_INVALID) {
    fprintf(stderr, "ld < n accepted\n");
    return 1;
  }
  st = zfac_refine(ctx, dS, N, dZ0, N, dZ, N, MAXIT, ZFAC_STOP_PAPER, dInts, dErr, dInts + 1, NULL);
  if (st != ZFAC_OK) { fprintf(stderr, "zfac_refine: %s %s\n", zfac_status_string(st), zfac_last_cuda_error()); return 1; }
  if (cudaDeviceSynchronize() != cudaSuccess) { fprintf(stderr, "sync failed\n"); return 1; }
  int ints[2];
  double err[MAXIT + 1];
  cudaMemcpy(ints, dInts, sizeof(ints), cudaMemcpyDeviceToHost);
  cudaMemcpy(err, dErr, sizeof(err), cudaMemcpyDeviceToHost);
  cudaMemcpy(hZ, dZ, N * N * elt, cudaMemcpyDeviceToHost);
  static double Z64[N * N];
  for (int i = 0; i < N * N; ++i) Z64[i] = (elt == 8) ? ((double*)hZ)[i] : (double)((float*)hZ)[i];
  /* the FP32 modes work on the FP32-rounded S: evaluate the invariant against what the library was given */
  static double Sused[N * N];
  for (int i = 0; i < N * N; ++i) Sused[i] = (elt == 8) ? S64[i] : (double)(float)S64[i];
  const double inv = invariant(Sused, Z64);
  printf("mode %d: iters=%d flags=%d launches=%d Err[0]=%.3e Err[last]=%.3e  ||Z^T S Z - I||_F/sqrt(N)=%.3e (gate %.0e)\n",
         (int)mode, ints[0], ints[1], zfac_last_launch_count(ctx), err[0], err[ints[0]], inv, gate);
  int bad = 0;
  if (!(ints[1] & ZFAC_R_STOPPED) || ints[0] < 2 || ints[0] > MAXIT) bad = 1;     /* the paper's test fired        */
  if (!(inv <= gate)) bad = 1;                                                      /* Z is an inverse factor        */
  if (!(err[ints[0]] <= 10.0 * gate * sqrt((double)N) + 1e-12)) bad = 1;            /* the history says so too       */
  for (int k = 1; k < ints[0]; ++k) if (!(err[k] <= err[k - 1] * err[k - 1] * err[k - 1])) bad = 1;   /* Eq. 38 held before */
  zfac_destroy(ctx);
  cudaFree(ws); cudaFree(dS); cudaFree(dZ0); cudaFree(dZ); cudaFree(dInts); cudaFree(dErr);
  free(hS); free(hZ);
  return bad;
}

int main(void) {
  static double S[N * N], Z0[N * N];
  double bound = 0.0;
  for (int i = 0; i < N; ++i) {
    double rowsum = 0.0;
    for (int j = 0; j < N; ++j) {
      const int d = abs(i - j);
      S[i * N + j] = (d == 0) ? 1.0 : 0.45 * exp(-1.1 * (double)d) * (1.0 + 0.1 * sin((double)(i + j)));
      rowsum += fabs(S[i * N + j]);
    }
    if (rowsum > bound) bound = rowsum;
  }
  for (int i = 0; i < N; ++i)                      /* symmetrise exactly */
    for (int j = 0; j < i; ++j) S[i * N + j] = S[j * N + i];
  memset(Z0, 0, sizeof(Z0));
  for (int i = 0; i < N; ++i) Z0[i * N + i] = 1.0 / sqrt(bound);
  if (zfac_workspace_bytes(0, ZFAC_MODE_F64) != 0 || zfac_padded_n(N, ZFAC_MODE_SPLIT16) != 256) { fprintf(stderr, "size queries\n"); return 1; }
  int bad = run_mode(ZFAC_MODE_F64, S, Z0, 1e-12);
  bad |= run_mode(ZFAC_MODE_SPLIT16, S, Z0, 1e-5);
  printf(bad ? "abi_consumer: FAILED\n" : "abi_consumer: OK\n");
  return bad;
}
