/*
 * saf3r_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Plain, slow, obviously-correct CPU restatement of the SAF3R hot path
 * (arxiv/paper_2607_03612): pool -> score -> select -> masked softmax attention,
 * plus a separately written dense attention and the NMSE of Eq. 1.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
 * legs may build, load or call this file.  It shares no code, header, table or helper
 * with the CUDA path under paper_2607_03612_b200/csrc and neither includes the other.
 *
 * Arithmetic convention: inputs are bf16 bit patterns decoded
 * exactly to fp32; every sum is accumulated in double; pooled vectors, scores and
 * outputs are stored as fp32.  No blocking, fusion or reordering beyond what the cited
 * passage states.  OpenMP is used only across independent rows (timing convenience).
 *
 * Citations are PAPER.md line numbers and DESIGN.md readings.
 *
 * Parity pins: every function below is pinned by tests/test_oracle_pins.py (P1..P20 of
 * DESIGN.md; P14-P16 pin orc_attn_tokens / orc_token_probe, P17 orc_union_lists, P18 orc_attn_broadcast_frame0,
 * P19 orc_token_topk_per_frame / orc_token_cosine_row / orc_attn_token_lists; P20 the kept set of the GLOBAL top-n and probe
 * rules of select_row, P4 the floor form of the fractional stride).  Unpinned *choices* (not arithmetic): POSITION_BAND radius and the
 * DOT-vs-COSINE default for correspondence heads -- "parity unpinned" for those choices.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

/* ---- head configuration (the oracle's own declaration; field order documented in DESIGN.md) ---- */
enum { ORC_HEAD_DENSE = 0, ORC_HEAD_UNIFORM_STRIDE = 1, ORC_HEAD_STATIC = 2,
       ORC_HEAD_QUERY_PROBE_TOPK = 3, ORC_HEAD_BLOCK_TOPK = 4 };
enum { ORC_STATIC_ANCHOR = 0, ORC_STATIC_FRAME_LOCAL = 1, ORC_STATIC_POSITION_BAND = 2 };
enum { ORC_SCOPE_GLOBAL = 0, ORC_SCOPE_PER_FRAME = 1 };
enum { ORC_SCORE_DOT = 0, ORC_SCORE_COSINE = 1 };

typedef struct {
  int32_t type;
  int32_t stride, offset;
  int32_t keep_blocks;
  int32_t static_mode, anchor_frame, band_radius;
  int32_t topk_scope, topk_per_frame;
  int32_t score_mode;
} orc_head_cfg;

/* bf16 -> fp32 is exact: the 16 bits are the top half of the fp32 pattern. */
static inline float bf16_to_f32(uint16_t b) {
  uint32_t u = ((uint32_t)b) << 16;
  float f;
  memcpy(&f, &u, 4);
  return f;
}

static inline int64_t ceil_div64(int64_t a, int64_t b) { return (a + b - 1) / b; }

int64_t orc_num_blocks(int64_t N, int64_t B) { return ceil_div64(N, B); }

/* ------------------------------------------------------------------------------------------------
 * O1  Pool.  PAPER.md:L126 ("block-level similarities averaged over multiple tokens"):
 *   X~_J = (1/c_J) * sum_{t in block J} x^_t,  x^ = x (DOT) or x/||x||_2 (COSINE; 0 if ||x|| < 1e-20).
 * c_J is the true token count of block J (the tail block is partial; reading A12).
 * x: one head, [N][D] bf16 bits.  pooled: [NB][D] fp32.
 * ---------------------------------------------------------------------------------------------- */
void orc_pool(const uint16_t *x, int64_t N, int32_t D, int32_t B, int32_t cosine, float *pooled) {
  int64_t NB = ceil_div64(N, B);
#pragma omp parallel for schedule(static)
  for (int64_t J = 0; J < NB; ++J) {
    int64_t t0 = J * B, t1 = t0 + B < N ? t0 + B : N;
    double *acc = (double *)calloc((size_t)D, sizeof(double));
    for (int64_t t = t0; t < t1; ++t) {
      double inv = 1.0;
      if (cosine) {
        double nn = 0.0;
        for (int d = 0; d < D; ++d) { double v = bf16_to_f32(x[t * D + d]); nn += v * v; }
        double nrm = sqrt(nn);
        inv = nrm < 1e-20 ? 0.0 : 1.0 / nrm;
      }
      for (int d = 0; d < D; ++d) acc[d] += (double)bf16_to_f32(x[t * D + d]) * inv;
    }
    double cnt = (double)(t1 - t0);
    for (int d = 0; d < D; ++d) pooled[J * D + d] = (float)(acc[d] / cnt);
    free(acc);
  }
}

/* O1  Mean query.  PAPER.md:L124: qbar = (1/N) sum_{i=1..N} q_i  (all N tokens, un-normalised; reading A4). */
void orc_mean_query(const uint16_t *q, int64_t N, int32_t D, float *qbar) {
  for (int d = 0; d < D; ++d) {
    double acc = 0.0;
    for (int64_t t = 0; t < N; ++t) acc += (double)bf16_to_f32(q[t * D + d]);
    qbar[d] = (float)(acc / (double)N);
  }
}

/* ------------------------------------------------------------------------------------------------
 * O2  Score.  One row: s[J] = (a . K~_J) * c, J = 0..NB-1.
 *   BLOCK_TOPK  : a = Q~_I, c = 1/sqrt(D) (DOT, the attention scale of PAPER.md:L124) or 1 (COSINE)
 *   QUERY_PROBE : a = qbar, c = 1/sqrt(D)  ("single probe vector qbar K^T / sqrt(D)")
 * ---------------------------------------------------------------------------------------------- */
void orc_score_row(const float *a, const float *kt, int64_t NB, int32_t D, double c, float *s) {
  for (int64_t J = 0; J < NB; ++J) {
    double acc = 0.0;
    for (int d = 0; d < D; ++d) acc += (double)a[d] * (double)kt[J * D + d];
    s[J] = (float)(acc * c);
  }
}

/* Top-n on the total order (score descending, then index ascending) over candidates
 * cand[0..m): marks keep[cand[i]] = 1 for the n winners.  Plain selection: repeat "take the best
 * remaining" n times (no sort, no heap), so the tie rule is visible on the page (reading A11). */
static void topn_mark(const float *s, const int32_t *cand, int64_t m, int64_t n, uint8_t *keep) {
  if (n > m) n = m;
  uint8_t *taken = (uint8_t *)calloc((size_t)(m > 0 ? m : 1), 1);
  for (int64_t r = 0; r < n; ++r) {
    int64_t best = -1;
    for (int64_t i = 0; i < m; ++i) {
      if (taken[i]) continue;
      if (best < 0 || s[cand[i]] > s[cand[best]]) best = i; /* strict '>' keeps the lower index on ties (cand ascending) */
    }
    taken[best] = 1;
    keep[cand[best]] = 1;
  }
  free(taken);
}

/* Faster equivalent of topn_mark for large rows (same total order): sort candidate indices by
 * (score desc, index asc) with qsort on a key array.  Used when m*n would be too slow; the two are
 * cross-checked against each other in tests (pin P10). */
typedef struct { float s; int32_t j; } orc_sj;
static int cmp_sj(const void *pa, const void *pb) {
  const orc_sj *a = (const orc_sj *)pa, *b = (const orc_sj *)pb;
  if (a->s > b->s) return -1;
  if (a->s < b->s) return 1;
  return a->j < b->j ? -1 : (a->j > b->j ? 1 : 0);
}
static void topn_mark_sorted(const float *s, const int32_t *cand, int64_t m, int64_t n, uint8_t *keep) {
  if (n > m) n = m;
  orc_sj *a = (orc_sj *)malloc(sizeof(orc_sj) * (size_t)(m > 0 ? m : 1));
  for (int64_t i = 0; i < m; ++i) { a[i].s = s[cand[i]]; a[i].j = cand[i]; }
  qsort(a, (size_t)m, sizeof(orc_sj), cmp_sj);
  for (int64_t r = 0; r < n; ++r) keep[a[r].j] = 1;
  free(a);
}

/* exported for pin P10: top-n of a row by either routine; writes the kept indices ascending; returns count */
int64_t orc_topn(const float *s, int64_t NB, int64_t n, int32_t use_sort, int32_t *out_idx) {
  int32_t *cand = (int32_t *)malloc(sizeof(int32_t) * (size_t)NB);
  uint8_t *keep = (uint8_t *)calloc((size_t)NB, 1);
  for (int64_t j = 0; j < NB; ++j) cand[j] = (int32_t)j;
  if (use_sort) topn_mark_sorted(s, cand, NB, n, keep); else topn_mark(s, cand, NB, n, keep);
  int64_t c = 0;
  for (int64_t j = 0; j < NB; ++j) if (keep[j]) out_idx[c++] = (int32_t)j;
  free(cand); free(keep);
  return c;
}

/* ------------------------------------------------------------------------------------------------
 * O3  Select: the keep-mask (over k-blocks) of q-block I for one head.  DESIGN.md table "O3".
 *   S frames, T tokens per frame, N = S*T, B block size, NB = ceil(N/B).
 *   blk(t) = floor(t/B); frame of token f(t) = floor(t/T); position p(t) = t mod T;
 *   frame of a block fr(J) = floor(J*B/T) (frame of its first token).
 * srow: the score row this q-block uses (probe row or its own row); may be NULL for content-free types.
 * ---------------------------------------------------------------------------------------------- */
static void select_row(const orc_head_cfg *cfg, int64_t S, int64_t T, int64_t B, int64_t I,
                       const float *srow, uint8_t *keep /* [NB], zeroed by caller */) {
  const int64_t N = S * T, NB = ceil_div64(N, B);
  switch (cfg->type) {
  case ORC_HEAD_DENSE: /* O_full */
    for (int64_t J = 0; J < NB; ++J) keep[J] = 1;
    break;
  case ORC_HEAD_UNIFORM_STRIDE: /* PAPER.md:L102 "selects key positions with a fixed stride" (reading A1: on k-blocks) */
    if (cfg->stride >= 1) {
      for (int64_t J = cfg->offset; J < NB; J += cfg->stride) keep[J] = 1;
    } else { /* fractional ratio: n blocks at floor(i*NB/n) */
      int64_t n = cfg->keep_blocks;
      for (int64_t i = 0; i < n; ++i) keep[(i * NB) / n] = 1;
    }
    break;
  case ORC_HEAD_STATIC:
    if (cfg->static_mode == ORC_STATIC_ANCHOR) { /* PAPER.md:L96 "all queries attend to a designated anchor frame" */
      int64_t a = cfg->anchor_frame;
      for (int64_t J = (a * T) / B; J <= ((a + 1) * T - 1) / B; ++J) keep[J] = 1;
    } else if (cfg->static_mode == ORC_STATIC_FRAME_LOCAL) { /* reading A5: each query's own frame(s) */
      int64_t t0 = I * B, t1 = t0 + B < N ? t0 + B : N;
      int64_t f0 = t0 / T, f1 = (t1 - 1) / T;
      for (int64_t J = (f0 * T) / B; J <= ((f1 + 1) * T - 1) / B; ++J) keep[J] = 1;
    } else { /* POSITION_BAND, reading A5/A6: same in-frame positions +- r in EVERY frame */
      int64_t r = cfg->band_radius;
      int64_t t0 = I * B, t1 = t0 + B < N ? t0 + B : N;
      int64_t f0 = t0 / T, f1 = (t1 - 1) / T;
      for (int64_t f = f0; f <= f1; ++f) {
        int64_t a = t0 > f * T ? t0 : f * T;                     /* tokens of I inside frame f: [a, b] */
        int64_t b = (t1 - 1) < ((f + 1) * T - 1) ? (t1 - 1) : ((f + 1) * T - 1);
        int64_t pa = a - f * T, pb = b - f * T;
        int64_t lo = pa - r > 0 ? pa - r : 0;
        int64_t hi = pb + r < T - 1 ? pb + r : T - 1;
        for (int64_t g = 0; g < S; ++g)
          for (int64_t J = (g * T + lo) / B; J <= (g * T + hi) / B; ++J) keep[J] = 1;
      }
    }
    break;
  case ORC_HEAD_QUERY_PROBE_TOPK: /* top-n of the probe row, same for every I */
  case ORC_HEAD_BLOCK_TOPK:
    if (cfg->type == ORC_HEAD_QUERY_PROBE_TOPK || cfg->topk_scope == ORC_SCOPE_GLOBAL) {
      int32_t *cand = (int32_t *)malloc(sizeof(int32_t) * (size_t)NB);
      for (int64_t j = 0; j < NB; ++j) cand[j] = (int32_t)j;
      topn_mark_sorted(srow, cand, NB, cfg->keep_blocks, keep);
      free(cand);
    } else { /* PER_FRAME: "Top-K most similar tokens from each frame", L126; reading A7 */
      int32_t *cand = (int32_t *)malloc(sizeof(int32_t) * (size_t)NB);
      for (int64_t g = 0; g < S; ++g) {
        int64_t m = 0;
        for (int64_t J = 0; J < NB; ++J) if ((J * B) / T == g) cand[m++] = (int32_t)J; /* C_g = {J : fr(J) = g} */
        topn_mark(srow, cand, m, cfg->topk_per_frame, keep);
      }
      free(cand);
    }
    break;
  default: break;
  }
}

/* Full per-head selection.  q,k: this head's [N][D] bf16.  Writes CSR lists for all NB q-blocks:
 * row_ptr[NB+1] (relative to this head, row_ptr[0] = 0) and col_idx (ascending).  Returns the number
 * of entries, or -(needed) if capacity is too small.  If scores_out != NULL and the head is a Top-K
 * type, also stores the score rows used: [NB][NB] for BLOCK_TOPK, [1][NB] for QUERY_PROBE. */
int64_t orc_select_head(const uint16_t *q, const uint16_t *k, int64_t S, int64_t T, int32_t D, int32_t B,
                        const orc_head_cfg *cfg, int64_t *row_ptr, int32_t *col_idx, int64_t capacity,
                        float *scores_out) {
  const int64_t N = S * T, NB = ceil_div64(N, B);
  float *qt = NULL, *kt = NULL, *qbar = NULL, *probe = NULL;
  const int topk = cfg->type == ORC_HEAD_QUERY_PROBE_TOPK || cfg->type == ORC_HEAD_BLOCK_TOPK;
  if (topk) {
    kt = (float *)malloc(sizeof(float) * (size_t)(NB * D));
    if (cfg->type == ORC_HEAD_BLOCK_TOPK) {
      int cosine = cfg->score_mode == ORC_SCORE_COSINE;
      qt = (float *)malloc(sizeof(float) * (size_t)(NB * D));
      orc_pool(q, N, D, B, cosine, qt);
      orc_pool(k, N, D, B, cosine, kt);
    } else {
      qbar = (float *)malloc(sizeof(float) * (size_t)D);
      probe = (float *)malloc(sizeof(float) * (size_t)NB);
      orc_mean_query(q, N, D, qbar);
      orc_pool(k, N, D, B, 0, kt);
      orc_score_row(qbar, kt, NB, D, 1.0 / sqrt((double)D), probe);
      if (scores_out) memcpy(scores_out, probe, sizeof(float) * (size_t)NB);
    }
  }
  uint8_t *keep_all = (uint8_t *)calloc((size_t)(NB * NB), 1);
  const double c = (cfg->type == ORC_HEAD_BLOCK_TOPK && cfg->score_mode == ORC_SCORE_COSINE) ? 1.0 : 1.0 / sqrt((double)D);
#pragma omp parallel for schedule(dynamic, 4)
  for (int64_t I = 0; I < NB; ++I) {
    const float *srow = probe;
    float *mine = NULL;
    if (cfg->type == ORC_HEAD_BLOCK_TOPK) {
      mine = scores_out ? scores_out + I * NB : (float *)malloc(sizeof(float) * (size_t)NB);
      orc_score_row(qt + I * D, kt, NB, D, c, mine);
      srow = mine;
    }
    select_row(cfg, S, T, B, I, srow, keep_all + I * NB);
    if (mine && !scores_out) free(mine);
  }
  int64_t cnt = 0;
  row_ptr[0] = 0;
  for (int64_t I = 0; I < NB; ++I) {
    for (int64_t J = 0; J < NB; ++J)
      if (keep_all[I * NB + J]) {
        if (cnt < capacity) col_idx[cnt] = (int32_t)J;
        ++cnt;
      }
    row_ptr[I + 1] = cnt;
  }
  free(keep_all); free(qt); free(kt); free(qbar); free(probe);
  return cnt <= capacity ? cnt : -cnt;
}

/* ------------------------------------------------------------------------------------------------
 * O4  Masked softmax attention for one head over CSR block lists.  PAPER.md:L106 (O_sparse), L124 (S = QK^T/sqrt(D)).
 *   For q token i in q-block I:  A(i) = {j < N : blk(j) in list(I)},  z_ij = (q_i . k_j)/sqrt(D),
 *   m_i = max z_ij,  l_i = sum exp(z_ij - m_i),  o_i = (1/l_i) sum exp(z_ij - m_i) v_j,  lse_i = m_i + ln l_i.
 *   A(i) empty  =>  o_i = 0, lse_i = -inf.
 * Only the q-blocks listed in qblocks[0..nq) are computed; out is [N][D] fp32 (rows of other blocks untouched),
 * lse is [N] fp32 (may be NULL).  Two passes over the keys, exactly as the formulas read.
 * ---------------------------------------------------------------------------------------------- */
void orc_attn_lists(const uint16_t *q, const uint16_t *k, const uint16_t *v, int64_t N, int32_t D, int32_t B,
                    const int64_t *row_ptr, const int32_t *col_idx, const int64_t *qblocks, int64_t nq,
                    float *out, float *lse) {
  const double scale = 1.0 / sqrt((double)D);
#pragma omp parallel for schedule(dynamic, 1)
  for (int64_t qi = 0; qi < nq; ++qi) {
    const int64_t I = qblocks[qi];
    const int64_t t0 = I * B, t1 = t0 + B < N ? t0 + B : N;
    double *acc = (double *)malloc(sizeof(double) * (size_t)D);
    for (int64_t i = t0; i < t1; ++i) {
      double m = -INFINITY;
      int64_t nkeys = 0;
      for (int64_t e = row_ptr[I]; e < row_ptr[I + 1]; ++e) {
        int64_t J = col_idx[e];
        int64_t j1 = (J + 1) * B < N ? (J + 1) * B : N;
        for (int64_t j = J * B; j < j1; ++j) {
          double z = 0.0;
          for (int d = 0; d < D; ++d) z += (double)bf16_to_f32(q[i * D + d]) * (double)bf16_to_f32(k[j * D + d]);
          z *= scale;
          if (z > m) m = z;
          ++nkeys;
        }
      }
      if (nkeys == 0) {
        for (int d = 0; d < D; ++d) out[i * D + d] = 0.0f;
        if (lse) lse[i] = -INFINITY;
        continue;
      }
      double l = 0.0;
      for (int d = 0; d < D; ++d) acc[d] = 0.0;
      for (int64_t e = row_ptr[I]; e < row_ptr[I + 1]; ++e) {
        int64_t J = col_idx[e];
        int64_t j1 = (J + 1) * B < N ? (J + 1) * B : N;
        for (int64_t j = J * B; j < j1; ++j) {
          double z = 0.0;
          for (int d = 0; d < D; ++d) z += (double)bf16_to_f32(q[i * D + d]) * (double)bf16_to_f32(k[j * D + d]);
          z *= scale;
          double w = exp(z - m);
          l += w;
          for (int d = 0; d < D; ++d) acc[d] += w * (double)bf16_to_f32(v[j * D + d]);
        }
      }
      for (int d = 0; d < D; ++d) out[i * D + d] = (float)(acc[d] / l);
      if (lse) lse[i] = (float)(m + log(l));
    }
    free(acc);
  }
}

/* O4 (dense), written separately so that pin P1 compares two code paths: O_full = softmax(QK^T/sqrt(D)) V over
 * all j < N.  Rows i in [i0, i1).  Materialises the row of logits, as the definition reads. */
void orc_attn_dense(const uint16_t *q, const uint16_t *k, const uint16_t *v, int64_t N, int32_t D,
                    int64_t i0, int64_t i1, float *out, float *lse) {
  const double inv_sqrt_d = 1.0 / sqrt((double)D);
#pragma omp parallel for schedule(dynamic, 8)
  for (int64_t i = i0; i < i1; ++i) {
    double *z = (double *)malloc(sizeof(double) * (size_t)N);
    double zmax = -INFINITY;
    for (int64_t j = 0; j < N; ++j) {
      double dot = 0.0;
      for (int d = 0; d < D; ++d) dot += (double)bf16_to_f32(q[i * D + d]) * (double)bf16_to_f32(k[j * D + d]);
      z[j] = dot * inv_sqrt_d;
      if (z[j] > zmax) zmax = z[j];
    }
    double denom = 0.0;
    for (int64_t j = 0; j < N; ++j) { z[j] = exp(z[j] - zmax); denom += z[j]; }
    for (int d = 0; d < D; ++d) {
      double o = 0.0;
      for (int64_t j = 0; j < N; ++j) o += z[j] * (double)bf16_to_f32(v[j * D + d]);
      out[i * D + d] = (float)(o / denom);
    }
    if (lse) lse[i] = (float)(zmax + log(denom));
    free(z);
  }
}

/* ---- token-granular variants: the paper's own, token-level definitions of two kernels ------------
 * O4-token: every query attends the SAME explicit key-token set idx[0..n) (ascending, unique).
 *   Uniform Sampling Kernel: "selects key positions with a fixed stride": idx = {o + i*s}.
 *   Query-Probe Top-K Kernel: "all queries attend only to these keys".
 * o_i = sum_{j in idx} softmax_j(q_i.k_j / sqrt(D)) v_j;  n == 0 -> o_i = 0, lse_i = -inf.  Rows [i0, i1). */
void orc_attn_tokens(const uint16_t *q, const uint16_t *k, const uint16_t *v, int64_t N, int32_t D, const int64_t *idx,
                     int64_t n, int64_t i0, int64_t i1, float *out, float *lse) {
  const double inv_sqrt_d = 1.0 / sqrt((double)D);
  (void)N;
#pragma omp parallel for schedule(dynamic, 8)
  for (int64_t i = i0; i < i1; ++i) {
    if (n == 0) {
      for (int d = 0; d < D; ++d) out[i * D + d] = 0.f;
      if (lse) lse[i] = -INFINITY;
      continue;
    }
    double *z = (double *)malloc(sizeof(double) * (size_t)n);
    double zmax = -INFINITY;
    for (int64_t t = 0; t < n; ++t) {
      const int64_t j = idx[t];
      double dot = 0.0;
      for (int d = 0; d < D; ++d) dot += (double)bf16_to_f32(q[i * D + d]) * (double)bf16_to_f32(k[j * D + d]);
      z[t] = dot * inv_sqrt_d;
      if (z[t] > zmax) zmax = z[t];
    }
    double denom = 0.0;
    for (int64_t t = 0; t < n; ++t) { z[t] = exp(z[t] - zmax); denom += z[t]; }
    for (int d = 0; d < D; ++d) {
      double o = 0.0;
      for (int64_t t = 0; t < n; ++t) o += z[t] * (double)bf16_to_f32(v[idx[t] * D + d]);
      out[i * D + d] = (float)(o / denom);
    }
    if (lse) lse[i] = (float)(zmax + log(denom));
    free(z);
  }
}

/* Token-level query probe: p[j] = qbar . k_j / sqrt(D) for every key token j, qbar = (1/N) sum_i q_i (double
 * accumulation, stored fp32 like every other score of this oracle). */
void orc_token_probe(const uint16_t *q, const uint16_t *k, int64_t N, int32_t D, float *p) {
  float *qbar = (float *)malloc(sizeof(float) * (size_t)D);
  orc_mean_query(q, N, D, qbar);
  const double inv_sqrt_d = 1.0 / sqrt((double)D);
#pragma omp parallel for schedule(static)
  for (int64_t j = 0; j < N; ++j) {
    double dot = 0.0;
    for (int d = 0; d < D; ++d) dot += (double)qbar[d] * (double)bf16_to_f32(k[j * D + d]);
    p[j] = (float)(dot * inv_sqrt_d);
  }
  free(qbar);
}

/* ---- DINO Top-K kernel, TOKEN-WISE (Tab. 6/7 L241-249) ------------------
 * "we pre-compute the cosine similarity between each patch token and all other patch tokens using the DINO features, and select
 * the Top-K most similar tokens from each frame as the keys and values for attention" (L100); "compute the global cosine similarity
 * between all patches, storing the indices of the per-frame Top-K matched patches ... token-wise ... exact token-level
 * similarities" (L126).  feat: per-sequence features [N][D] bf16 bits (the encoder's last-block output; shared by heads and layers).
 * For query token i and every frame g: cos_ij = (f_i . f_j) / (|f_i| |f_j|) for the T tokens j of frame g (0 if a norm < 1e-20),
 * double accumulation, stored fp32; keep the K best under (score desc, index asc); emit ascending.
 * DESIGN.md reading A19: every token of every frame is a candidate, the query's own frame and the query itself included
 * (cos = 1 ranks it first in its own frame); special tokens are ordinary tokens (reading A7).  Requires 1 <= K <= T.
 * idx_out: int32 [(i1 - i0)][S][K], global token indices.  Rows i in [i0, i1). */
void orc_token_topk_per_frame(const uint16_t *feat, int64_t S, int64_t T, int32_t D, int64_t K, int64_t i0, int64_t i1,
                              int32_t *idx_out) {
  const int64_t N = S * T;
  double *nrm = (double *)malloc(sizeof(double) * (size_t)N);
  for (int64_t t = 0; t < N; ++t) {
    double nn = 0.0;
    for (int d = 0; d < D; ++d) { double x = bf16_to_f32(feat[t * D + d]); nn += x * x; }
    nrm[t] = sqrt(nn);
  }
#pragma omp parallel for schedule(dynamic, 4)
  for (int64_t i = i0; i < i1; ++i) {
    float *cosr = (float *)malloc(sizeof(float) * (size_t)T);
    int32_t *cand = (int32_t *)malloc(sizeof(int32_t) * (size_t)T);
    uint8_t *keep = (uint8_t *)malloc((size_t)T);
    for (int64_t g = 0; g < S; ++g) {
      for (int64_t p = 0; p < T; ++p) {
        const int64_t j = g * T + p;
        double dot = 0.0;
        for (int d = 0; d < D; ++d) dot += (double)bf16_to_f32(feat[i * D + d]) * (double)bf16_to_f32(feat[j * D + d]);
        const double den = nrm[i] * nrm[j];
        cosr[p] = (nrm[i] < 1e-20 || nrm[j] < 1e-20) ? 0.0f : (float)(dot / den);
        cand[p] = (int32_t)p;
        keep[p] = 0;
      }
      topn_mark_sorted(cosr, cand, T, K, keep);
      int64_t c = 0;
      for (int64_t p = 0; p < T; ++p)
        if (keep[p]) idx_out[((i - i0) * S + g) * K + c++] = (int32_t)(g * T + p);
    }
    free(cosr); free(cand); free(keep);
  }
  free(nrm);
}

/* the cosine row of one query against ALL tokens (for the near-tie rule of the GPU-vs-oracle comparison and for pin P19) */
void orc_token_cosine_row(const uint16_t *feat, int64_t N, int32_t D, int64_t i, float *cos_out) {
  double ni = 0.0;
  for (int d = 0; d < D; ++d) { double x = bf16_to_f32(feat[i * D + d]); ni += x * x; }
  ni = sqrt(ni);
  for (int64_t j = 0; j < N; ++j) {
    double nj = 0.0, dot = 0.0;
    for (int d = 0; d < D; ++d) {
      double x = bf16_to_f32(feat[j * D + d]);
      nj += x * x;
      dot += (double)bf16_to_f32(feat[i * D + d]) * x;
    }
    nj = sqrt(nj);
    cos_out[j] = (ni < 1e-20 || nj < 1e-20) ? 0.0f : (float)(dot / (ni * nj));
  }
}

/* O4 with PER-QUERY key lists ("... as the keys and values for attention"): query i (rows [i0, i1)) attends the key
 * tokens idx[(i - i0) * L + 0 .. L); entries < 0 are padding and ignored.  o_i = sum_j softmax_j(q_i.k_j / sqrt(D)) v_j over its
 * list; an empty list gives o_i = 0, lse_i = -inf.  Two passes, as the formulas read. */
void orc_attn_token_lists(const uint16_t *q, const uint16_t *k, const uint16_t *v, int64_t N, int32_t D, const int32_t *idx, int64_t L,
                          int64_t i0, int64_t i1, float *out, float *lse) {
  const double scale = 1.0 / sqrt((double)D);
  (void)N;
#pragma omp parallel for schedule(dynamic, 8)
  for (int64_t i = i0; i < i1; ++i) {
    const int32_t *row = idx + (i - i0) * L;
    double m = -INFINITY;
    int64_t nk = 0;
    for (int64_t e = 0; e < L; ++e) {
      if (row[e] < 0) continue;
      const int64_t j = row[e];
      double z = 0.0;
      for (int d = 0; d < D; ++d) z += (double)bf16_to_f32(q[i * D + d]) * (double)bf16_to_f32(k[j * D + d]);
      z *= scale;
      if (z > m) m = z;
      ++nk;
    }
    if (nk == 0) {
      for (int d = 0; d < D; ++d) out[i * D + d] = 0.0f;
      if (lse) lse[i] = -INFINITY;
      continue;
    }
    double l = 0.0, acc[256];
    for (int d = 0; d < D; ++d) acc[d] = 0.0;
    for (int64_t e = 0; e < L; ++e) {
      if (row[e] < 0) continue;
      const int64_t j = row[e];
      double z = 0.0;
      for (int d = 0; d < D; ++d) z += (double)bf16_to_f32(q[i * D + d]) * (double)bf16_to_f32(k[j * D + d]);
      const double w = exp(z * scale - m);
      l += w;
      for (int d = 0; d < D; ++d) acc[d] += w * (double)bf16_to_f32(v[j * D + d]);
    }
    for (int d = 0; d < D; ++d) out[i * D + d] = (float)(acc[d] / l);
    if (lse) lse[i] = (float)(m + log(l));
  }
}

/* ---- Static kernel, "broadcasting the first frame's local attention map to other frames" ----
 * DESIGN.md reading A18: position heads are content-independent with a pattern "fixed across all image blocks", so
 * every T x T image block (f, g) of the N x N attention map carries frame 0's local logits z0[p][p'] = q_{0,p} . k_{0,p'} / sqrt(D).
 * Softmax over the whole row (all S*T keys) of that map gives the weight P0[p][p'] / S on key (g, p'), P0 = softmax_p'(z0), hence
 *     o_{f,p} = sum_g sum_p' (P0[p][p'] / S) v_{g,p'}          for every frame f,
 *     lse_{f,p} = ln( S * sum_p' exp(z0[p][p']) ).
 * Written as the double sum over (g, p') exactly as it reads (no pre-averaging of V).  out [N][D] fp32, lse [N] fp32 or NULL. */
void orc_attn_broadcast_frame0(const uint16_t *q, const uint16_t *k, const uint16_t *v, int64_t S, int64_t T, int32_t D, float *out,
                               float *lse) {
  const double inv_sqrt_d = 1.0 / sqrt((double)D);
#pragma omp parallel for schedule(dynamic, 8)
  for (int64_t p = 0; p < T; ++p) {
    double *w = (double *)malloc(sizeof(double) * (size_t)T);
    double zmax = -INFINITY;
    for (int64_t pp = 0; pp < T; ++pp) {
      double dot = 0.0;
      for (int d = 0; d < D; ++d) dot += (double)bf16_to_f32(q[p * D + d]) * (double)bf16_to_f32(k[pp * D + d]);
      w[pp] = dot * inv_sqrt_d;
      if (w[pp] > zmax) zmax = w[pp];
    }
    double denom = 0.0;
    for (int64_t pp = 0; pp < T; ++pp) { w[pp] = exp(w[pp] - zmax); denom += w[pp]; }
    for (int d = 0; d < D; ++d) {
      double o = 0.0;
      for (int64_t g = 0; g < S; ++g)
        for (int64_t pp = 0; pp < T; ++pp) o += (w[pp] / (denom * (double)S)) * (double)bf16_to_f32(v[(g * T + pp) * D + d]);
      for (int64_t f = 0; f < S; ++f) out[(f * T + p) * D + d] = (float)o;
    }
    if (lse)
      for (int64_t f = 0; f < S; ++f) lse[f * T + p] = (float)(zmax + log(denom * (double)S));
    free(w);
  }
}

/* ---- union of block lists ("combining Top-K with uniform striding") ----------------------
 * out(I) = a(I) U b(I) for every row I, by the definition of a set union: J is kept iff it is in a's row or in b's row.
 * Rows are emitted ascending.  Returns the number of entries, or -(needed) if capacity is too small. */
int64_t orc_union_lists(const int64_t *rp_a, const int32_t *col_a, const int64_t *rp_b, const int32_t *col_b, int64_t rows,
                        int64_t NB, int64_t *rp_o, int32_t *col_o, int64_t capacity) {
  uint8_t *keep = (uint8_t *)malloc((size_t)(NB > 0 ? NB : 1));
  int64_t cnt = 0;
  rp_o[0] = 0;
  for (int64_t I = 0; I < rows; ++I) {
    memset(keep, 0, (size_t)NB);
    for (int64_t e = rp_a[I]; e < rp_a[I + 1]; ++e) keep[col_a[e]] = 1;
    for (int64_t e = rp_b[I]; e < rp_b[I + 1]; ++e) keep[col_b[e]] = 1;
    for (int64_t J = 0; J < NB; ++J)
      if (keep[J]) {
        if (cnt < capacity) col_o[cnt] = (int32_t)J;
        ++cnt;
      }
    rp_o[I + 1] = cnt;
  }
  free(keep);
  return cnt <= capacity ? cnt : -cnt;
}

/* O5  NMSE, Eq. 1 (one sample): ||O_full - O_sparse||_2^2 / ||O_full||_2^2. */
double orc_nmse(const float *o_full, const float *o_sparse, int64_t count) {
  double num = 0.0, den = 0.0;
  for (int64_t i = 0; i < count; ++i) {
    double d = (double)o_full[i] - (double)o_sparse[i];
    num += d * d;
    den += (double)o_full[i] * (double)o_full[i];
  }
  return num / den;
}

int32_t orc_num_threads(void) {
#ifdef _OPENMP
  extern int omp_get_max_threads(void);
  return omp_get_max_threads();
#else
  return 1;
#endif
}
