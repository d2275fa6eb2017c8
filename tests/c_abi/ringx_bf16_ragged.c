/* ringx_bf16_ragged.c -- a plain C program (no Python, no PyTorch in the process) that links libringx.so and libcudart
 * and runs the bf16 forward AND backward of a ragged sequence through the C ABI of include/ringx.h:
 *   B = 1, H = 2, N = 333 (no multiple of the 128-row tile), d = 128, kv_chunk = 256 (two passes: 256 keys and 77 keys)
 *   ringx_attn_fwd  -> o, lse            (Eq. 1 via the chunk loop and the Eq. 5 fold)
 *   ringx_attn_bwd  -> dq, dk, dv        (derivative of Eq. 1; data flow of PAPER.md:143), default and deterministic mode
 * and compares with expected values the fp64 oracle wrote to tests/golden/bf16_ragged_expected.txt (written by
 * tests/golden/make_bf16_ragged_golden.py, which calls only oracle/ and the seeded input generator).  Every device
 * buffer is cudaMalloc'ed at exactly its size, so a store past the end of a head would be an out-of-bounds access.
 *
 *   ringx_bf16_ragged <inputs.bin> <expected.txt>
 * inputs.bin: q, k, v, dO as raw little-endian bf16 (uint16) [2*333*128] each, in this order.
 * expected.txt: lines "<tensor> <flat index> <value>", tensor in {o, lse, dq, dk, dv}.
 * Exit status 0 = o within 1e-2 * max|v| (and 1e-2 relative Frobenius over the listed entries), lse within 1e-3,
 * gradients within 2e-2 relative Frobenius over the listed entries (BASELINE.json's tolerances). */
#include <math.h>
#include <stdint.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include <cuda_runtime_api.h>

#include "ringx.h"

enum { BH = 2, N = 333, D = 128, CHUNK = 256, ELEMS = BH * N * D, ROWS = BH * N };

static void die(const char* what, int code) {
  fprintf(stderr, "ringx_bf16_ragged: %s (%d)\n", what, code);
  exit(2);
}
#define CUDA_OK(x) do { cudaError_t e_ = (x); if (e_ != cudaSuccess) die(cudaGetErrorString(e_), (int)e_); } while (0)
#define RINGX_CHECK(x) do { int s_ = (x); if (s_ != RINGX_OK) die(ringx_status_string(s_), s_); } while (0)

static double bf16_to_double(uint16_t h) {
  uint32_t u = (uint32_t)h << 16;
  float f;
  memcpy(&f, &u, sizeof(f));
  return (double)f;
}

struct Stat {
  double max_abs, err2, ref2;
  int n;
};

/* accumulates |got - want| statistics of one tensor over the entries listed for it in the expected file */
static void compare(const char* path, const char* tensor, const uint16_t* got_bf16, const float* got_f32, struct Stat* st) {
  FILE* f = fopen(path, "r");
  char tag[16];
  memset(st, 0, sizeof(*st));
  if (!f) die("cannot open the expected-value file", 0);
  while (fscanf(f, "%15s", tag) == 1) {
    long idx;
    double want, got, e;
    if (tag[0] == '#') {
      int c;
      while ((c = fgetc(f)) != '\n' && c != EOF) {}
      continue;
    }
    if (fscanf(f, "%ld %lf", &idx, &want) != 2) die("bad line in the expected-value file", st->n);
    if (strcmp(tag, tensor) != 0) continue;
    got = got_bf16 ? bf16_to_double(got_bf16[idx]) : (double)got_f32[idx];
    e = fabs(got - want);
    if (!(e <= st->max_abs)) st->max_abs = e;      /* also catches NaN */
    st->err2 += e * e;
    st->ref2 += want * want;
    st->n += 1;
  }
  fclose(f);
}

static double relf(const struct Stat* st) { return st->ref2 > 0.0 ? sqrt(st->err2 / st->ref2) : sqrt(st->err2); }

int main(int argc, char** argv) {
  const size_t tb = (size_t)ELEMS * sizeof(uint16_t);
  const float scale = 0.08838834764831845f;                       /* 1/sqrt(128) */
  uint16_t *h_in, *h_out, *h_dq_first;
  float* h_lse;
  void *q, *k, *v, *dO, *o, *dq, *dk, *dv, *ws_f = NULL, *ws_b = NULL;
  float* lse;
  size_t wf, wb;
  double vmax = 0.0;
  struct Stat so, sl, sq, sk, sv;
  FILE* f;
  int i, mode;

  if (argc != 3) die("usage: ringx_bf16_ragged <inputs.bin> <expected.txt>", argc);
  h_in = (uint16_t*)malloc(4 * tb);
  h_out = (uint16_t*)malloc(tb);
  h_dq_first = (uint16_t*)malloc(tb);
  h_lse = (float*)malloc(ROWS * sizeof(float));
  f = fopen(argv[1], "rb");
  if (!f || fread(h_in, 1, 4 * tb, f) != 4 * tb) die("cannot read q,k,v,dO", 0);
  fclose(f);
  for (i = 0; i < ELEMS; ++i) {
    const double a = fabs(bf16_to_double(h_in[2 * ELEMS + i]));
    if (a > vmax) vmax = a;
  }

  CUDA_OK(cudaSetDevice(0));
  CUDA_OK(cudaMalloc(&q, tb));
  CUDA_OK(cudaMalloc(&k, tb));
  CUDA_OK(cudaMalloc(&v, tb));
  CUDA_OK(cudaMalloc(&dO, tb));
  CUDA_OK(cudaMalloc(&o, tb));
  CUDA_OK(cudaMalloc(&dq, tb));
  CUDA_OK(cudaMalloc(&dk, tb));
  CUDA_OK(cudaMalloc(&dv, tb));
  CUDA_OK(cudaMalloc((void**)&lse, ROWS * sizeof(float)));
  CUDA_OK(cudaMemcpy(q, h_in, tb, cudaMemcpyHostToDevice));
  CUDA_OK(cudaMemcpy(k, h_in + ELEMS, tb, cudaMemcpyHostToDevice));
  CUDA_OK(cudaMemcpy(v, h_in + 2 * ELEMS, tb, cudaMemcpyHostToDevice));
  CUDA_OK(cudaMemcpy(dO, h_in + 3 * ELEMS, tb, cudaMemcpyHostToDevice));

  wf = ringx_attn_fwd_workspace_bytes(1, BH, N, D, CHUNK, RINGX_BF16);
  wb = ringx_attn_bwd_workspace_bytes(1, BH, N, D, CHUNK, RINGX_BF16);
  if (!wf || !wb) die("workspace query rejected the ragged shape", 0);
  CUDA_OK(cudaMalloc(&ws_f, wf));
  CUDA_OK(cudaMalloc(&ws_b, wb));

  RINGX_CHECK(ringx_attn_fwd(q, k, v, o, lse, 1, BH, N, D, CHUNK, scale, RINGX_BF16, ws_f, wf, NULL));
  CUDA_OK(cudaDeviceSynchronize());
  CUDA_OK(cudaMemcpy(h_out, o, tb, cudaMemcpyDeviceToHost));
  CUDA_OK(cudaMemcpy(h_lse, lse, ROWS * sizeof(float), cudaMemcpyDeviceToHost));
  compare(argv[2], "o", h_out, NULL, &so);
  compare(argv[2], "lse", NULL, h_lse, &sl);
  printf("ringx_bf16_ragged: version %d; o max|err| %.3e relF %.3e over %d values (max|v| %.2f); lse max|err| %.3e over %d\n",
         ringx_version(), so.max_abs, relf(&so), so.n, vmax, sl.max_abs, sl.n);
  if (so.n < 1000 || sl.n < 100) die("too few expected forward values", so.n);
  if (!(so.max_abs <= 1e-2 * vmax) || !(relf(&so) <= 1e-2) || !(sl.max_abs <= 1e-3)) die("forward mismatch against the oracle", 1);

  for (mode = 0; mode < 2; ++mode) {            /* default (fp32 reduce-adds), then bit-reproducible fixed point */
    int rep;
    RINGX_CHECK(ringx_set_deterministic(mode));
    for (rep = 0; rep < 1 + mode; ++rep) {
      RINGX_CHECK(ringx_attn_bwd(q, k, v, o, lse, dO, dq, dk, dv, 1, BH, N, D, CHUNK, scale, RINGX_BF16, ws_b, wb, NULL));
      CUDA_OK(cudaDeviceSynchronize());
      CUDA_OK(cudaMemcpy(h_out, dq, tb, cudaMemcpyDeviceToHost));
      if (mode == 1 && rep == 0) memcpy(h_dq_first, h_out, tb);
      if (mode == 1 && rep == 1 && memcmp(h_dq_first, h_out, tb) != 0) die("deterministic mode: dq differs between two runs", 1);
    }
    compare(argv[2], "dq", h_out, NULL, &sq);
    CUDA_OK(cudaMemcpy(h_out, dk, tb, cudaMemcpyDeviceToHost));
    compare(argv[2], "dk", h_out, NULL, &sk);
    CUDA_OK(cudaMemcpy(h_out, dv, tb, cudaMemcpyDeviceToHost));
    compare(argv[2], "dv", h_out, NULL, &sv);
    printf("ringx_bf16_ragged: %s backward: relF dq %.3e dk %.3e dv %.3e over %d / %d / %d values\n",
           mode ? "deterministic" : "default", relf(&sq), relf(&sk), relf(&sv), sq.n, sk.n, sv.n);
    if (sq.n < 1000 || sk.n < 1000 || sv.n < 1000) die("too few expected gradient values", sq.n);
    if (!(relf(&sq) <= 2e-2) || !(relf(&sk) <= 2e-2) || !(relf(&sv) <= 2e-2)) die("gradient mismatch against the oracle", 1);
  }
  RINGX_CHECK(ringx_set_deterministic(0));
  printf("RINGX_BF16_RAGGED_OK\n");
  return 0;
}
