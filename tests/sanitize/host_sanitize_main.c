/* Host-side sanitizer driver (ASan / UBSan build of the host logic and of the C oracle).
 *
 * Built by tests/test_host_sanitizers.py with  gcc -fsanitize=address,undefined -fno-sanitize-recover=all  together
 * with  paper_2606_01483_b200/csrc/chunk_plan.cu  (pure host C: murmur_chunk_plan, murmur_batch_plan) and
 * oracle/c/murmur_oracle.c (the plain-C oracle twin), and run on seeded inputs that include the edge cases: empty
 * input, capacity too small, over-long segments, a single position, ragged sizes.  Any out-of-bounds access, leak,
 * signed overflow or misaligned access aborts the program with a non-zero status; on success it prints "OK". */
#include <math.h>
#include <stdint.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include "murmur.h"

int murmur_oracle_attend(int n_layers, int n_q, int n_kv, int d, const uint16_t* k, const uint16_t* v, int64_t n_pos,
                         const int32_t* retained, int n_ret, const uint16_t* q, double scale, double* out, double* lse,
                         int n_threads);
int murmur_oracle_prefill(int n_layers, int n_q, int n_kv, int d, const uint16_t* k, const uint16_t* v, int64_t n_pos,
                          int pos_begin, int n_tok, const uint16_t* q, double scale, double* out, double* lse,
                          int n_threads);
int murmur_oracle_retained(int P, int S, int M, int t, int w_s, int delay, int k_s, int w_o, int k_o, int length,
                           int32_t* out, int cap);

static uint32_t rng_state = 12345u;
static uint32_t rnd(void) {
  rng_state = rng_state * 1664525u + 1013904223u;
  return rng_state >> 8;
}
static uint16_t rnd_bf16(void) { /* a finite bf16 in roughly [-2, 2] */
  float f = ((float)(rnd() % 4001) - 2000.0f) / 1000.0f;
  uint32_t u;
  memcpy(&u, &f, 4);
  return (uint16_t)(u >> 16);
}
#define CHECK(x)                                                   \
  do {                                                             \
    if (!(x)) {                                                    \
      fprintf(stderr, "%s:%d: check failed: %s\n", __FILE__, __LINE__, #x); \
      return 1;                                                    \
    }                                                              \
  } while (0)

static int run_plans(void) {
  for (int trial = 0; trial < 200; ++trial) {
    const int n = (int)(rnd() % 60);
    float* a = (float*)malloc(sizeof(float) * (size_t)(n ? n : 1));
    float* b = (float*)malloc(sizeof(float) * (size_t)(n ? n : 1));
    float t = 0.f;
    for (int i = 0; i < n; ++i) {
      t += (float)(rnd() % 2000) / 100.f;
      a[i] = t;
      t += 0.2f + (float)(rnd() % (trial % 3 == 0 ? 50000 : 9000)) / 100.f;
      b[i] = t;
    }
    int32_t n_chunks = -1;
    /* exact capacity: the array is allocated with exactly n entries so that one write too many is caught */
    int32_t* first = (int32_t*)malloc(sizeof(int32_t) * (size_t)(n ? n : 1));
    CHECK(murmur_chunk_plan(a, b, n, 300.f, first, n, &n_chunks) == MURMUR_OK);
    CHECK(n_chunks >= 0 && n_chunks <= n);
    if (n_chunks > 1) { /* capacity too small: the count is still reported, nothing is written past cap */
      int32_t n2 = -1;
      int32_t* small = (int32_t*)malloc(sizeof(int32_t) * (size_t)(n_chunks - 1));
      CHECK(murmur_chunk_plan(a, b, n, 300.f, small, n_chunks - 1, &n2) == MURMUR_ERR_INVALID_ARG && n2 == n_chunks);
      free(small);
    }
    murmur_batch_entry_t* e = (murmur_batch_entry_t*)malloc(sizeof(murmur_batch_entry_t) * (size_t)(n_chunks ? n_chunks : 1));
    int32_t n_batches = -1;
    const int bs = 1 + (int)(rnd() % 16);
    CHECK(murmur_batch_plan(a, b, n, first, n_chunks, bs, 7.5, 32768, 3600.0, 64, 0, 64, e, &n_batches) == MURMUR_OK);
    CHECK(n_batches == (n_chunks + bs - 1) / bs);
    for (int j = 0; j < n_chunks; ++j) CHECK(e[j].chunk == j && e[j].batch == j / bs && e[j].slot == j % bs && e[j].n_speech >= 0 && e[j].max_new >= 1);
    /* a rate that overflows int32 must be refused, not wrapped */
    if (n_chunks > 0) CHECK(murmur_batch_plan(a, b, n, first, n_chunks, bs, 1e12, 32768, 3600.0, 0, 0, 16, e, &n_batches) == MURMUR_ERR_INVALID_ARG);
    free(e); free(first); free(a); free(b);
  }
  int32_t nc = 7;
  CHECK(murmur_chunk_plan(NULL, NULL, 0, 300.f, NULL, 0, &nc) == MURMUR_OK && nc == 0);
  CHECK(murmur_chunk_plan(NULL, NULL, 3, 300.f, NULL, 0, &nc) == MURMUR_ERR_INVALID_ARG);
  CHECK(murmur_batch_plan(NULL, NULL, 0, NULL, 0, 16, 7.5, 32768, 3600.0, 0, 0, 64, NULL, &nc) == MURMUR_OK && nc == 0);
  return 0;
}

static int run_oracle(void) {
  const int shapes[4][5] = {/* L, n_q, n_kv, d, n_pos */ {2, 28, 4, 128, 37}, {1, 4, 2, 16, 1}, {3, 8, 8, 32, 65}, {1, 7, 1, 128, 130}};
  for (int sidx = 0; sidx < 4; ++sidx) {
    const int L = shapes[sidx][0], n_q = shapes[sidx][1], n_kv = shapes[sidx][2], d = shapes[sidx][3], n_pos = shapes[sidx][4];
    const size_t kv_n = (size_t)L * n_pos * n_kv * d;
    uint16_t* k = (uint16_t*)malloc(kv_n * 2);
    uint16_t* v = (uint16_t*)malloc(kv_n * 2);
    for (size_t i = 0; i < kv_n; ++i) { k[i] = rnd_bf16(); v[i] = rnd_bf16(); }
    /* decode: a ragged retained set that ends at the last position */
    int n_ret = 0;
    int32_t* ret = (int32_t*)malloc(sizeof(int32_t) * (size_t)n_pos);
    for (int x = 0; x < n_pos; ++x)
      if (x == n_pos - 1 || rnd() % 3) ret[n_ret++] = x;
    uint16_t* q = (uint16_t*)malloc((size_t)L * n_q * d * 2);
    for (size_t i = 0; i < (size_t)L * n_q * d; ++i) q[i] = rnd_bf16();
    double* out = (double*)malloc(sizeof(double) * (size_t)L * n_q * d);
    double* lse = (double*)malloc(sizeof(double) * (size_t)L * n_q);
    CHECK(murmur_oracle_attend(L, n_q, n_kv, d, k, v, n_pos, ret, n_ret, q, 0.1, out, lse, 2) >= 1);
    for (size_t i = 0; i < (size_t)L * n_q * d; ++i) CHECK(isfinite(out[i]));
    CHECK(murmur_oracle_attend(L, n_q, n_kv, d, k, v, n_pos, ret, 0, q, 0.1, out, lse, 1) == -1);
    free(out); free(lse); free(q);
    /* prefill: the last n_tok positions, and the whole range */
    for (int pass = 0; pass < 2; ++pass) {
      const int n_tok = pass ? n_pos : (n_pos + 1) / 2, pos_begin = n_pos - n_tok;
      uint16_t* qp = (uint16_t*)malloc((size_t)L * n_tok * n_q * d * 2);
      for (size_t i = 0; i < (size_t)L * n_tok * n_q * d; ++i) qp[i] = rnd_bf16();
      double* op = (double*)malloc(sizeof(double) * (size_t)L * n_tok * n_q * d);
      double* lp = (double*)malloc(sizeof(double) * (size_t)L * n_tok * n_q);
      CHECK(murmur_oracle_prefill(L, n_q, n_kv, d, k, v, n_pos, pos_begin, n_tok, qp, 0.1, op, lp, 2) >= 1);
      for (size_t i = 0; i < (size_t)L * n_tok * n_q * d; ++i) CHECK(isfinite(op[i]));
      CHECK(murmur_oracle_prefill(L, n_q, n_kv, d, k, v, n_pos, pos_begin + 1, n_tok, qp, 0.1, op, lp, 1) == -1);
      free(qp); free(op); free(lp);
    }
    free(ret); free(k); free(v);
  }
  /* retained sets: exact-capacity output buffers over a grid of small policies */
  for (int t = 0; t <= 20; ++t)
    for (int w = 0; w <= 6; w += 3) {
      const int P = 2, S = 9, M = 1, total = P + S + M + t;
      int32_t* out = (int32_t*)malloc(sizeof(int32_t) * (size_t)total);
      const int n = murmur_oracle_retained(P, S, M, t, w, 2, 1, w + 1, 1, total, out, total);
      CHECK(n >= 0 && n <= total);
      for (int i = 1; i < n; ++i) CHECK(out[i] > out[i - 1] && out[i] < total);
      free(out);
    }
  return 0;
}

int main(void) {
  if (run_plans()) return 1;
  if (run_oracle()) return 1;
  puts("OK");
  return 0;
}
