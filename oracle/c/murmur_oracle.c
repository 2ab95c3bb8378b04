/* Plain C twin of oracle/policy.py + oracle/attention.py, for the timed CPU baseline.
 *
 * TEST INFRASTRUCTURE - see oracle/__init__.py.  Shares no code with the CUDA path.
 * fp64 throughout, no intrinsics, no blocking or fusion beyond the definition; the only
 * parallelism is an OpenMP "parallel for" over independent (layer, query head) pairs.
 *
 * Retained-set rule: Alg. 1 on the output region, Eq. 2 / Alg. 2
 * on the speech region, system prompts always kept;
 * readings as in oracle/policy.py / DESIGN.md.
 * Attention: Eq. 1, max-subtracted softmax, o = sum alpha_i v_i.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

static double bf16_to_f64(uint16_t b) {
  uint32_t u = ((uint32_t)b) << 16;
  float f;
  memcpy(&f, &u, sizeof f);
  return (double)f;
}

static int64_t imin(int64_t a, int64_t b) { return a < b ? a : b; }
static int64_t imax(int64_t a, int64_t b) { return a > b ? a : b; }

/* A(t) restricted to positions < length, ascending.  Returns the count, or -1 if cap is
 * too small. */
int murmur_oracle_retained(int P, int S, int M, int t, int w_speech, int delay, int n_sink_speech,
                           int w_out, int n_sink_out, int length, int32_t* out, int cap) {
  int n = 0;
  int64_t l = imin(imax(0, (int64_t)t - delay), imax(0, (int64_t)S - w_speech));
  for (int x = 0; x < P + S + M + t && x < length; ++x) {
    int keep;
    if (x < P) {
      keep = 1; /* system prompt */
    } else if (x < P + S) {
      int64_t r = x - P;
      keep = (r < n_sink_speech) || (r >= l && r < l + (int64_t)w_speech);
    } else if (x < P + S + M) {
      keep = 1; /* second system prompt */
    } else {
      int64_t u = x - (P + S + M);
      keep = (u < n_sink_out) || (u >= (int64_t)t - w_out);
    }
    if (keep) {
      if (n >= cap) return -1;
      out[n++] = x;
    }
  }
  return n;
}

/* Eq. 1 over the retained set for one sequence, all layers and query heads.
 * k, v : [n_layers][n_pos][n_kv][d] bf16 bits, rows by absolute position
 * q    : [n_layers][n_q][d]         bf16 bits
 * out  : [n_layers][n_q][d]         fp64;   lse: [n_layers][n_q] fp64 or NULL
 * n_threads <= 0: OpenMP default.  Returns the number of threads used, or -1 on error. */
int murmur_oracle_attend(int n_layers, int n_q, int n_kv, int d, const uint16_t* k, const uint16_t* v,
                         int64_t n_pos, const int32_t* retained, int n_ret, const uint16_t* q,
                         double scale, double* out, double* lse, int n_threads) {
  if (n_ret <= 0 || n_q % n_kv != 0) return -1;
  const int G = n_q / n_kv;
  int used = 1;
#ifdef _OPENMP
  if (n_threads > 0) omp_set_num_threads(n_threads);
  used = omp_get_max_threads();
#else
  (void)n_threads;
#endif
  int failed = 0;
#pragma omp parallel for collapse(2) schedule(dynamic, 1)
  for (int layer = 0; layer < n_layers; ++layer) {
    for (int h = 0; h < n_q; ++h) {
      const int g = h / G;
      double* s = (double*)malloc((size_t)n_ret * sizeof(double));
      double* qf = (double*)malloc((size_t)d * sizeof(double));
      if (!s || !qf) {
        failed = 1;
        free(s);
        free(qf);
        continue;
      }
      const uint16_t* qrow = q + ((size_t)layer * n_q + h) * d;
      for (int c = 0; c < d; ++c) qf[c] = bf16_to_f64(qrow[c]);
      double m = -INFINITY;
      for (int i = 0; i < n_ret; ++i) { /* s_i = q . k_i / sqrt(d) */
        const uint16_t* krow = k + (((size_t)layer * n_pos + retained[i]) * n_kv + g) * d;
        double acc = 0.0;
        for (int c = 0; c < d; ++c) acc += qf[c] * bf16_to_f64(krow[c]);
        s[i] = acc * scale;
        if (s[i] > m) m = s[i];
      }
      double denom = 0.0;
      for (int i = 0; i < n_ret; ++i) { /* e_i = exp(s_i - m) */
        s[i] = exp(s[i] - m);
        denom += s[i];
      }
      double* o = out + ((size_t)layer * n_q + h) * d;
      for (int c = 0; c < d; ++c) o[c] = 0.0;
      for (int i = 0; i < n_ret; ++i) { /* o = sum alpha_i v_i */
        const uint16_t* vrow = v + (((size_t)layer * n_pos + retained[i]) * n_kv + g) * d;
        const double a = s[i] / denom;
        for (int c = 0; c < d; ++c) o[c] += a * bf16_to_f64(vrow[c]);
      }
      if (lse) lse[(size_t)layer * n_q + h] = m + log(denom);
      free(s);
      free(qf);
    }
  }
  return failed ? -1 : used;
}

/* Causal self-attention of prefill tokens, Eq. 1 of every query position over the cache positions
 * y <= x (the model is a decoder) - the plain-C twin of oracle/prefill.py::causal_attention, several
 * layers at once.  One query row at a time, written out: scores, maximum, exponentials, sum, weighted V sum; no
 * blocking, no running maximum.  OpenMP over (layer, query head) only.
 * k, v : [n_layers][n_pos][n_kv][d] bf16 bits by absolute position, n_pos >= pos_begin + n_tok
 * q    : [n_layers][n_tok][n_q][d]  bf16 bits, row i = position pos_begin + i
 * out  : [n_layers][n_tok][n_q][d]  fp64;   lse: [n_layers][n_tok][n_q] fp64 or NULL
 * Returns the number of threads used, or -1 on error. */
int murmur_oracle_prefill(int n_layers, int n_q, int n_kv, int d, const uint16_t* k, const uint16_t* v,
                          int64_t n_pos, int pos_begin, int n_tok, const uint16_t* q, double scale, double* out,
                          double* lse, int n_threads) {
  if (n_tok <= 0 || pos_begin < 0 || n_q % n_kv != 0 || (int64_t)pos_begin + n_tok > n_pos) return -1;
  const int G = n_q / n_kv;
  int used = 1;
#ifdef _OPENMP
  if (n_threads > 0) omp_set_num_threads(n_threads);
  used = omp_get_max_threads();
#else
  (void)n_threads;
#endif
  int failed = 0;
#pragma omp parallel for collapse(2) schedule(dynamic, 1)
  for (int layer = 0; layer < n_layers; ++layer) {
    for (int h = 0; h < n_q; ++h) {
      const int g = h / G;
      const int64_t n_max = (int64_t)pos_begin + n_tok;
      double* s = (double*)malloc((size_t)n_max * sizeof(double));
      double* kf = (double*)malloc((size_t)n_max * d * sizeof(double)); /* this head's K and V rows as fp64 */
      double* vf = (double*)malloc((size_t)n_max * d * sizeof(double));
      double* qf = (double*)malloc((size_t)d * sizeof(double));
      if (!s || !kf || !vf || !qf) {
        failed = 1;
        free(s); free(kf); free(vf); free(qf);
        continue;
      }
      for (int64_t y = 0; y < n_max; ++y) {
        const uint16_t* krow = k + (((size_t)layer * n_pos + y) * n_kv + g) * d;
        const uint16_t* vrow = v + (((size_t)layer * n_pos + y) * n_kv + g) * d;
        for (int c = 0; c < d; ++c) {
          kf[y * d + c] = bf16_to_f64(krow[c]);
          vf[y * d + c] = bf16_to_f64(vrow[c]);
        }
      }
      for (int i = 0; i < n_tok; ++i) {
        const int64_t x = (int64_t)pos_begin + i; /* attends y = 0 .. x */
        const uint16_t* qrow = q + (((size_t)layer * n_tok + i) * n_q + h) * d;
        for (int c = 0; c < d; ++c) qf[c] = bf16_to_f64(qrow[c]);
        double m = -INFINITY;
        for (int64_t y = 0; y <= x; ++y) { /* s_y = q . k_y * scale */
          double acc = 0.0;
          for (int c = 0; c < d; ++c) acc += qf[c] * kf[y * d + c];
          s[y] = acc * scale;
          if (s[y] > m) m = s[y];
        }
        double denom = 0.0;
        for (int64_t y = 0; y <= x; ++y) { /* e_y = exp(s_y - m) */
          s[y] = exp(s[y] - m);
          denom += s[y];
        }
        double* o = out + (((size_t)layer * n_tok + i) * n_q + h) * d;
        for (int c = 0; c < d; ++c) o[c] = 0.0;
        for (int64_t y = 0; y <= x; ++y) { /* o = sum alpha_y v_y */
          const double a = s[y] / denom;
          for (int c = 0; c < d; ++c) o[c] += a * vf[y * d + c];
        }
        if (lse) lse[((size_t)layer * n_tok + i) * n_q + h] = m + log(denom);
      }
      free(s); free(kf); free(vf); free(qf);
    }
  }
  return failed ? -1 : used;
}
