/* ringx_c1.c -- a plain C program (no Python, no PyTorch in the process) that links libringx.so and libcudart and
 * runs BASELINE.json configs[0] (C1: fp32, B=1, H=1, N=1024, d=64, four KV chunks of 256) through the C ABI of
 * include/ringx.h, two ways:
 *   (1) ringx_attn_fwd with kv_chunk = 256                                   (Eq. 1 via the chunk loop)
 *   (2) four ringx_attn_chunk_fwd calls, one per key chunk, whose (loc_out, loc_lse) are folded left to right with
 *       three ringx_lse_merge calls                                           (Eq. 5 literally)
 * and compares both with expected values the fp64 oracle wrote to tests/golden/c1_expected.txt (written by
 * tests/golden/make_c1_golden.py, which calls only oracle/ and the seeded input generator).
 *
 *   ringx_c1 <inputs.bin> <expected.txt>
 * inputs.bin: q, k, v as raw little-endian float32 [1024*64] each, in this order (the seeded C1 tensors).
 * expected.txt: lines "lse <row> <value>" and "o <row> <col> <value>".  Exit status 0 = every value within 1e-5. */
#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include <cuda_runtime_api.h>

#include "ringx.h"

enum { N = 1024, D = 64, CHUNK = 256 };

static void die(const char* what, int code) {
  fprintf(stderr, "ringx_c1: %s (%d)\n", what, code);
  exit(2);
}
#define CUDA_OK(x) do { cudaError_t e_ = (x); if (e_ != cudaSuccess) die(cudaGetErrorString(e_), (int)e_); } while (0)
#define RINGX_CHECK(x) do { int s_ = (x); if (s_ != RINGX_OK) die(ringx_status_string(s_), s_); } while (0)

/* max |got - expected| over the entries listed in the expected file */
static double compare(const char* path, const float* o, const float* lse, int* n_checked) {
  FILE* f = fopen(path, "r");
  char tag[16];
  double worst = 0.0;
  int n = 0;
  if (!f) die("cannot open the expected-value file", 0);
  while (fscanf(f, "%15s", tag) == 1) {
    int row, col;
    double want, got;
    if (tag[0] == '#') {                       /* comment line */
      int c;
      while ((c = fgetc(f)) != '\n' && c != EOF) {}
      continue;
    }
    if (strcmp(tag, "lse") == 0) {
      if (fscanf(f, "%d %lf", &row, &want) != 2) die("bad lse line", n);
      got = lse[row];
    } else if (strcmp(tag, "o") == 0) {
      if (fscanf(f, "%d %d %lf", &row, &col, &want) != 3) die("bad o line", n);
      got = o[(size_t)row * D + col];
    } else {
      die("unknown tag in the expected-value file", n);
    }
    if (!(fabs(got - want) <= worst)) worst = fabs(got - want);   /* also catches NaN */
    ++n;
  }
  fclose(f);
  *n_checked = n;
  return worst;
}

int main(int argc, char** argv) {
  const size_t elems = (size_t)N * D, bytes = elems * sizeof(float);
  const float scale = 0.125f;                                     /* 1/sqrt(64) */
  float *h_in, *h_o, *h_lse;
  float *q, *k, *v, *o, *lse, *acc_o, *acc_lse, *part_o, *part_lse;
  void* ws = NULL;
  size_t ws_bytes;
  FILE* f;
  int c, n1 = 0, n2 = 0;
  double e1, e2;

  if (argc != 3) die("usage: ringx_c1 <inputs.bin> <expected.txt>", argc);
  h_in = (float*)malloc(3 * bytes);
  h_o = (float*)malloc(bytes);
  h_lse = (float*)malloc(N * sizeof(float));
  f = fopen(argv[1], "rb");
  if (!f || fread(h_in, 1, 3 * bytes, f) != 3 * bytes) die("cannot read q,k,v", 0);
  fclose(f);

  CUDA_OK(cudaSetDevice(0));
  CUDA_OK(cudaMalloc((void**)&q, bytes));
  CUDA_OK(cudaMalloc((void**)&k, bytes));
  CUDA_OK(cudaMalloc((void**)&v, bytes));
  CUDA_OK(cudaMalloc((void**)&o, bytes));
  CUDA_OK(cudaMalloc((void**)&lse, N * sizeof(float)));
  CUDA_OK(cudaMalloc((void**)&acc_o, bytes));
  CUDA_OK(cudaMalloc((void**)&acc_lse, N * sizeof(float)));
  CUDA_OK(cudaMalloc((void**)&part_o, bytes));
  CUDA_OK(cudaMalloc((void**)&part_lse, N * sizeof(float)));
  CUDA_OK(cudaMemcpy(q, h_in, bytes, cudaMemcpyHostToDevice));
  CUDA_OK(cudaMemcpy(k, h_in + elems, bytes, cudaMemcpyHostToDevice));
  CUDA_OK(cudaMemcpy(v, h_in + 2 * elems, bytes, cudaMemcpyHostToDevice));

  /* (1) the chunked forward as one call */
  ws_bytes = ringx_attn_fwd_workspace_bytes(1, 1, N, D, CHUNK, RINGX_F32);
  if (ws_bytes) CUDA_OK(cudaMalloc(&ws, ws_bytes));
  RINGX_CHECK(ringx_attn_fwd(q, k, v, o, lse, 1, 1, N, D, CHUNK, scale, RINGX_F32, ws, ws_bytes, NULL));
  CUDA_OK(cudaDeviceSynchronize());
  CUDA_OK(cudaMemcpy(h_o, o, bytes, cudaMemcpyDeviceToHost));
  CUDA_OK(cudaMemcpy(h_lse, lse, N * sizeof(float), cudaMemcpyDeviceToHost));
  e1 = compare(argv[2], h_o, h_lse, &n1);

  /* (2) Eq. 5 by hand: per-chunk partials, folded with ringx_lse_merge (in place on operand a) */
  for (c = 0; c < N / CHUNK; ++c) {
    const float* kc = k + (size_t)c * CHUNK * D;
    const float* vc = v + (size_t)c * CHUNK * D;
    if (c == 0) {
      RINGX_CHECK(ringx_attn_chunk_fwd(q, kc, vc, acc_o, acc_lse, 1, 1, N, CHUNK, D, scale, RINGX_F32, NULL));
    } else {
      RINGX_CHECK(ringx_attn_chunk_fwd(q, kc, vc, part_o, part_lse, 1, 1, N, CHUNK, D, scale, RINGX_F32, NULL));
      RINGX_CHECK(ringx_lse_merge(acc_o, acc_lse, part_o, part_lse, acc_o, acc_lse, N, D, RINGX_F32, RINGX_F32, NULL));
    }
  }
  CUDA_OK(cudaDeviceSynchronize());
  CUDA_OK(cudaMemcpy(h_o, acc_o, bytes, cudaMemcpyDeviceToHost));
  CUDA_OK(cudaMemcpy(h_lse, acc_lse, N * sizeof(float), cudaMemcpyDeviceToHost));
  e2 = compare(argv[2], h_o, h_lse, &n2);

  printf("ringx_c1: version %d; ringx_attn_fwd max|err| %.3e over %d values; chunk_fwd + lse_merge max|err| %.3e over %d values\n",
         ringx_version(), e1, n1, e2, n2);
  if (n1 < 1000 || n2 != n1) die("too few expected values", n1);
  if (!(e1 <= 1e-5) || !(e2 <= 1e-5)) die("mismatch against the fp64 oracle's values (tolerance 1e-5)", 1);
  printf("RINGX_C1_OK\n");
  return 0;
}
