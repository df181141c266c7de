/*
 * sp_oracle.c -- CPU fp64 ORACLE for oracle-guided sparse prefill of one causal GQA layer.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference legs may load it.  It shares no code, header,
 * table or helper with the CUDA path (paper_2606_07703_b200/csrc, include/sp.h) and never
 * receives a value the CUDA path produced.
 *
 * It is a plain, slow, literal transcription of the definitions in
 * /root/reference/PAPER.md (arxiv/paper_2606_07703), in fp64, with OpenMP over independent
 * support rows / queries only.  No blocking, fusion or reordering beyond what the paper's
 * equations state.  Inputs are the same bf16 bit patterns the GPU gets, widened exactly.
 *
 * Step names (O1..O7) are the ones used in SURVEY.md 8(c) and DESIGN.md:
 *   O1  logits            z[t,h,s] = scale*<q[t,h],k[s,g(h)]>, s<=t            PAPER.md:94  (Sec.3)
 *   O2  dense probs       A = softmax_{s'<=t}(z)
 *   O3  attention mass    P[t,s] = (1/Hq) sum_h A[t,h,s]                       PAPER.md:123 (Sec.4.1)
 *   O3' indexer           q_idx = W_q x, k_idx = W_k x (bf16 tensors),
 *                         z_idx[t,s] = idx_scale*<q_idx[t],k_idx[s]>           (Sec.6.3, Alg.2 step 2,4)
 *   O4  support-row score R_B(s) = max_{t in B, s<=t} score[t,s]               PAPER.md:154 (Sec.4.2), :299
 *   O5  top-k             first k of (score desc, index asc); ascending, -1 pad PAPER.md:127,145,156
 *   O6  sparse attention  softmax over S_eff = {s in S : s<=t}
 *   O7  dense attention   brute force, separately coded
 *
 * Readings of points where the paper is silent: 0-based positions, the
 * query's own position is a valid key (A1); ties go to the lower index (A2); fewer than k valid
 * keys -> keep all, pad with -1 (A3); indices emitted ascending (A4); g(h) = h / (Hq/Hkv) (A5);
 * head mean over all Hq heads (A6); block score = max over the block's valid per-query rows of the
 * final per-query score (A7); blocks aligned to the sequence start, last one ragged (A8); empty
 * effective support -> o = 0, lse = -inf (A9); the indexer projections are rounded ONCE to bf16
 * (round-to-nearest-even) from the fp64 sum, scores stay unrounded (A14); optional banded additive
 * logit term local_bias for 0 <= t-s < local_window wherever a causal logit is formed (A20);
 * varlen: everything is local to its sequence, emitted indices are packed positions (A24).
 *
 * Pins (tests/test_oracle_pins.py, -m "not gpu"): rows of P sum to 1, head-permutation invariance,
 * MHA-with-repeated-KV == GQA, kept-pair count k*L-k(k-1)/2 and the sparsities the paper prints
 * (PAPER.md:180,216,374), the hand-worked case tests/golden/handworked_L4.txt, Q=0 closed form,
 * k>=n sparse==dense, numpy stable argsort, torch SDPA, numpy brute force on tiny inputs, varlen
 * pack == separate sequences; the paged-cache routines (pure indexing) against numpy fancy indexing, scatter-then-
 * gather == identity, block-table permutation invariance and chunked+paged == full prefill, bit for bit.
 * Indexer *quality* / task gaps: parity unpinned and out of scope.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef struct orc_params {
  int32_t batch;             /* number of sequences in the pack                         */
  int32_t L;                 /* total packed tokens                                     */
  const int32_t *cu_seqlens; /* HOST ptr [batch+1]; NULL = one sequence of length L     */
  int32_t Hq, Hkv, d;        /* heads and head dim                                      */
  int32_t k;                 /* budget per support row                                  */
  int32_t b_sel;             /* selection block size (1 = per query)                    */
  int32_t hidden, d_idx;     /* indexer sizes                                           */
  double scale;              /* attention scale (1/sqrt(d))                             */
  double idx_scale;          /* indexer scale (1/sqrt(d_idx))                           */
  int32_t local_window;      /* 0 = off                                                 */
  double local_bias;         /* added to the scaled logit when 0 <= t-s < local_window  */
  int32_t flags;             /* ORC_F_* : the served scorer's ReLU / key LayerNorm / RoPE */
} orc_params;

/* The served scorer (Alg.2 steps 3-4): k_idx = LN(W_K x), RoPE on q and k_idx, ReLU on the scaled
 * similarity.  Readings where the paper is silent (A26-A28): LayerNorm over the d_idx channels of one
 * token, no affine, biased variance, eps = 1e-6; RoPE in the rotate-half pairing (i, i + d_idx/2) with
 * theta_i = pos * 10000^(-2i/d_idx), pos = position LOCAL to the sequence; ReLU applied to the final logit
 * (scaled similarity + the local term of A20).  The transforms run in fp64 on the fp64 projection sum and the
 * result is rounded ONCE to bf16 (A14). */
enum { ORC_F_RELU = 1, ORC_F_KEY_LN = 2, ORC_F_ROPE = 4 };

enum { ORC_MODE_ORACLE = 0, ORC_MODE_INDEXER = 1 };

/* ---------- exact bf16 <-> fp64 ---------- */

static inline double bf16_to_f64(uint16_t b) {
  uint32_t u = ((uint32_t)b) << 16;
  float f;
  memcpy(&f, &u, 4);
  return (double)f;
}

/* One round-to-nearest-even from fp64 to bf16 (8 significant bits), no intermediate fp32 rounding. */
static uint16_t f64_to_bf16_rne(double x) {
  if (x != x) return 0x7fc0;
  if (x == 0.0) return signbit(x) ? 0x8000 : 0x0000;
  int e;
  double m = frexp(fabs(x), &e);           /* |x| = m * 2^e, m in [0.5,1)            */
  double r;
  if (e - 1 < -126) {                      /* below the bf16 normal range: quantum 2^-133 */
    r = ldexp(nearbyint(ldexp(fabs(x), 133)), -133);
  } else {
    r = ldexp(nearbyint(ldexp(m, 8)), e - 8); /* nearbyint: ties-to-even in the default mode */
  }
  if (r >= ldexp(1.0, 128)) r = INFINITY;
  float f = (float)(signbit(x) ? -r : r);  /* exact: r has <= 8 significant bits      */
  uint32_t u;
  memcpy(&u, &f, 4);
  return (uint16_t)(u >> 16);
}

void orc_f64_to_bf16(const double *x, int64_t n, uint16_t *out) {
  for (int64_t i = 0; i < n; ++i) out[i] = f64_to_bf16_rne(x[i]);
}

/* ---------- sequences and support rows (A8, A24) ---------- */

static void seq_of_pos(const orc_params *p, int32_t pos, int32_t *start, int32_t *len) {
  if (!p->cu_seqlens) { *start = 0; *len = p->L; return; }
  for (int32_t i = 0; i < p->batch; ++i)
    if (pos >= p->cu_seqlens[i] && pos < p->cu_seqlens[i + 1]) {
      *start = p->cu_seqlens[i];
      *len = p->cu_seqlens[i + 1] - p->cu_seqlens[i];
      return;
    }
  *start = 0; *len = 0;
}

static int32_t seq_start_i(const orc_params *p, int32_t i) { return p->cu_seqlens ? p->cu_seqlens[i] : 0; }
static int32_t seq_len_i(const orc_params *p, int32_t i) {
  return p->cu_seqlens ? p->cu_seqlens[i + 1] - p->cu_seqlens[i] : p->L;
}
static int32_t rows_of_len(const orc_params *p, int32_t n) {
  return p->b_sel <= 1 ? n : (n + p->b_sel - 1) / p->b_sel;
}

int32_t orc_num_rows(const orc_params *p) {
  int32_t r = 0;
  for (int32_t i = 0; i < p->batch; ++i) r += rows_of_len(p, seq_len_i(p, i));
  return r;
}

/* Support row -> (sequence start, first local position, last local position). Returns 0 on success. */
int32_t orc_row_info(const orc_params *p, int32_t row, int32_t *seq_start, int32_t *t_first, int32_t *t_last) {
  int32_t r0 = 0;
  int32_t b = p->b_sel <= 1 ? 1 : p->b_sel;
  for (int32_t i = 0; i < p->batch; ++i) {
    int32_t n = seq_len_i(p, i), nr = rows_of_len(p, n);
    if (row < r0 + nr) {
      int32_t j = row - r0;
      *seq_start = seq_start_i(p, i);
      *t_first = j * b;
      *t_last = (j + 1) * b - 1 < n - 1 ? (j + 1) * b - 1 : n - 1;
      return 0;
    }
    r0 += nr;
  }
  return -1;
}

/* Packed query position -> its support row. */
int32_t orc_row_of_pos(const orc_params *p, int32_t pos) {
  int32_t r0 = 0;
  int32_t b = p->b_sel <= 1 ? 1 : p->b_sel;
  for (int32_t i = 0; i < p->batch; ++i) {
    int32_t s0 = seq_start_i(p, i), n = seq_len_i(p, i);
    if (pos >= s0 && pos < s0 + n) return r0 + (pos - s0) / b;
    r0 += rows_of_len(p, n);
  }
  return -1;
}

static inline int32_t g_of_h(const orc_params *p, int32_t h) { return h / (p->Hq / p->Hkv); } /* A5 */

static inline double local_term(const orc_params *p, int32_t t, int32_t s) {        /* A20 */
  return (p->local_window > 0 && t - s >= 0 && t - s < p->local_window) ? p->local_bias : 0.0;
}

/* ---------- O3': indexer projection, PAPER.md:270, :297 ---------- */

/* LayerNorm (key side only) then RoPE of one token's d channels, in place, fp64 (A27, A28). */
void orc_transform(double *y, int32_t d, int32_t pos_local, int32_t flags, int32_t is_key) {
  if (is_key && (flags & ORC_F_KEY_LN)) {
    double mean = 0.0, var = 0.0;
    for (int32_t c = 0; c < d; ++c) mean += y[c];
    mean /= d;
    for (int32_t c = 0; c < d; ++c) var += (y[c] - mean) * (y[c] - mean);
    var /= d;
    const double rstd = 1.0 / sqrt(var + 1e-6);
    for (int32_t c = 0; c < d; ++c) y[c] = (y[c] - mean) * rstd;
  }
  if (flags & ORC_F_ROPE) {
    const int32_t h = d / 2;
    for (int32_t i = 0; i < h; ++i) {
      const double theta = (double)pos_local * pow(10000.0, -2.0 * i / d);
      const double c = cos(theta), sn = sin(theta);
      const double a = y[i], b = y[i + h];
      y[i] = a * c - b * sn;
      y[i + h] = b * c + a * sn;
    }
  }
}

/* out[r,:] = bf16_rne( T( sum_j X[rows[r],j] * W[j,:] ) ), fp64 sum in index order j = 0..hidden-1; T = orc_transform
 * with p->flags (identity when flags == 0). */
void orc_project(const orc_params *p, const uint16_t *X, const uint16_t *W, int32_t is_key,
                 const int32_t *rows, int32_t nrows, uint16_t *out) {
  const int32_t hidden = p->hidden, d_idx = p->d_idx;
#pragma omp parallel
  {
    double *acc = (double *)malloc(sizeof(double) * (size_t)d_idx);
#pragma omp for schedule(dynamic, 16)
    for (int32_t r = 0; r < nrows; ++r) {
      const uint16_t *x = X + (size_t)rows[r] * hidden;
      for (int32_t c = 0; c < d_idx; ++c) acc[c] = 0.0;
      for (int32_t j = 0; j < hidden; ++j) {
        double xv = bf16_to_f64(x[j]);
        const uint16_t *w = W + (size_t)j * d_idx;
        for (int32_t c = 0; c < d_idx; ++c) acc[c] += xv * bf16_to_f64(w[c]);
      }
      if (p->flags & (ORC_F_KEY_LN | ORC_F_ROPE)) {
        int32_t s0, n;
        seq_of_pos(p, rows[r], &s0, &n);
        orc_transform(acc, d_idx, rows[r] - s0, p->flags, is_key);
      }
      for (int32_t c = 0; c < d_idx; ++c) out[(size_t)r * d_idx + c] = f64_to_bf16_rne(acc[c]);
    }
    free(acc);
  }
}

/* ---------- per-query score rows ---------- */

/* O3' scoring: z[s] = idx_scale*<q_idx[t],k_idx[s]> (+local term) for local s = 0..tl
 * (BASELINE.json configs 2-5 define the logits without LN/RoPE/ReLU: flags == 0; ORC_F_RELU clips at 0).
 * q_idx,k_idx are packed [L,d_idx], already transformed by orc_project. */
static void indexer_row(const orc_params *p, const uint16_t *q_idx, const uint16_t *k_idx,
                        int32_t s0, int32_t tl, double *z) {
  const uint16_t *q = q_idx + (size_t)(s0 + tl) * p->d_idx;
  for (int32_t s = 0; s <= tl; ++s) {
    const uint16_t *kk = k_idx + (size_t)(s0 + s) * p->d_idx;
    double acc = 0.0;
    for (int32_t c = 0; c < p->d_idx; ++c) acc += bf16_to_f64(q[c]) * bf16_to_f64(kk[c]);
    z[s] = p->idx_scale * acc + local_term(p, tl, s);
    if ((p->flags & ORC_F_RELU) && z[s] < 0.0) z[s] = 0.0; /* PAPER.md:274; A26 */
  }
}

/* O1-O3: P[s] = (1/Hq) sum_h softmax_{s'<=t}(z[t,h,.])[s]. tmp has tl+1 doubles. */
static void mass_row(const orc_params *p, const uint16_t *Q, const uint16_t *K,
                     int32_t s0, int32_t tl, double *P, double *tmp) {
  for (int32_t s = 0; s <= tl; ++s) P[s] = 0.0;
  for (int32_t h = 0; h < p->Hq; ++h) {
    const uint16_t *q = Q + ((size_t)(s0 + tl) * p->Hq + h) * p->d;
    int32_t g = g_of_h(p, h);
    double m = -INFINITY;
    for (int32_t s = 0; s <= tl; ++s) {                                   /* O1 */
      const uint16_t *kk = K + ((size_t)(s0 + s) * p->Hkv + g) * p->d;
      double acc = 0.0;
      for (int32_t c = 0; c < p->d; ++c) acc += bf16_to_f64(q[c]) * bf16_to_f64(kk[c]);
      tmp[s] = p->scale * acc + local_term(p, tl, s);
      if (tmp[s] > m) m = tmp[s];
    }
    double den = 0.0;                                                     /* O2 */
    for (int32_t s = 0; s <= tl; ++s) { tmp[s] = exp(tmp[s] - m); den += tmp[s]; }
    for (int32_t s = 0; s <= tl; ++s) P[s] += tmp[s] / den;
  }
  for (int32_t s = 0; s <= tl; ++s) P[s] /= (double)p->Hq;                /* O3 */
}

/* One per-query row of the score that top-k ranks (mass in oracle mode, indexer logit otherwise);
 * out has ld doubles, entries (tl, ld) are set to -inf. `pos` is a packed position. */
void orc_query_scores(const orc_params *p, int32_t mode, const uint16_t *A, const uint16_t *B,
                      const int32_t *pos, int32_t npos, double *out, int64_t ld) {
#pragma omp parallel
  {
    double *tmp = (double *)malloc(sizeof(double) * (size_t)(p->L + 1));
#pragma omp for schedule(dynamic, 1)
    for (int32_t i = 0; i < npos; ++i) {
      int32_t s0, n;
      seq_of_pos(p, pos[i], &s0, &n);
      int32_t tl = pos[i] - s0;
      double *o = out + (size_t)i * ld;
      if (mode == ORC_MODE_ORACLE) mass_row(p, A, B, s0, tl, o, tmp);
      else indexer_row(p, A, B, s0, tl, o);
      for (int64_t s = tl + 1; s < ld; ++s) o[s] = -INFINITY;
    }
    free(tmp);
  }
}

/* ---------- O4: support-row score, PAPER.md:154, :299 ----------
 * rows[] are support-row numbers. out[r, s] for local s in [0, n_valid[r]) ; -inf beyond.
 * b_sel == 1: the per-query row. b_sel > 1: max over the block's queries t with s <= t of the
 * per-query score (mass AFTER normalisation and head mean; indexer logit). */
void orc_support_scores(const orc_params *p, int32_t mode, const uint16_t *A, const uint16_t *B,
                        const int32_t *rows, int32_t nrows, double *out, int64_t ld, int32_t *n_valid) {
#pragma omp parallel
  {
    double *tmp = (double *)malloc(sizeof(double) * (size_t)(p->L + 1));
    double *row = (double *)malloc(sizeof(double) * (size_t)(p->L + 1));
#pragma omp for schedule(dynamic, 1)
    for (int32_t r = 0; r < nrows; ++r) {
      int32_t s0, t0, t1;
      double *o = out + (size_t)r * ld;
      if (orc_row_info(p, rows[r], &s0, &t0, &t1) != 0) { n_valid[r] = 0; continue; }
      n_valid[r] = t1 + 1;
      for (int64_t s = 0; s < ld; ++s) o[s] = -INFINITY;
      for (int32_t tl = t0; tl <= t1; ++tl) {
        if (mode == ORC_MODE_ORACLE) mass_row(p, A, B, s0, tl, row, tmp);
        else indexer_row(p, A, B, s0, tl, row);
        for (int32_t s = 0; s <= tl; ++s)
          if (row[s] > o[s]) o[s] = row[s];
      }
    }
    free(tmp);
    free(row);
  }
}

/* ---------- O5: top-k, PAPER.md:127, :145, :156 ---------- */

typedef struct { double v; int32_t i; } orc_pair;

static int cmp_desc_then_index(const void *a, const void *b) {
  const orc_pair *x = (const orc_pair *)a, *y = (const orc_pair *)b;
  if (x->v > y->v) return -1;
  if (x->v < y->v) return 1;
  return (x->i > y->i) - (x->i < y->i);
}
static int cmp_int(const void *a, const void *b) {
  int32_t x = *(const int32_t *)a, y = *(const int32_t *)b;
  return (x > y) - (x < y);
}

/* For each row: the first min(k,n) elements of the order (score descending, index ascending), emitted
 * ascending as PACKED positions (local + seq_start), padded with -1. scores rows hold local columns. */
void orc_topk(const double *scores, int64_t ld, const int32_t *n_valid, const int32_t *seq_start,
              int32_t nrows, int32_t k, int32_t *idx, int32_t *cnt) {
#pragma omp parallel for schedule(dynamic, 1)
  for (int32_t r = 0; r < nrows; ++r) {
    int32_t n = n_valid[r];
    int32_t *o = idx + (size_t)r * k;
    int32_t keep = n < k ? n : k;
    if (n <= k) {
      for (int32_t j = 0; j < n; ++j) o[j] = j;
    } else {
      orc_pair *pr = (orc_pair *)malloc(sizeof(orc_pair) * (size_t)n);
      for (int32_t j = 0; j < n; ++j) { pr[j].v = scores[(size_t)r * ld + j]; pr[j].i = j; }
      qsort(pr, (size_t)n, sizeof(orc_pair), cmp_desc_then_index);
      for (int32_t j = 0; j < k; ++j) o[j] = pr[j].i;
      qsort(o, (size_t)k, sizeof(int32_t), cmp_int);
      free(pr);
    }
    for (int32_t j = 0; j < keep; ++j) o[j] += seq_start ? seq_start[r] : 0;
    for (int32_t j = keep; j < k; ++j) o[j] = -1;
    if (cnt) cnt[r] = keep;
  }
}

/* ---------- O6: sparse attention on a support, PAPER.md:107, :156 ----------
 * pos[i]: packed query position; sup + i*k: the k support entries (packed positions, -1 = sentinel) of
 * that query's support row.  o: [npos, Hq, d] fp64, lse: [npos, Hq] (natural log of the softmax
 * denominator incl. the max), either may be NULL. */
void orc_sparse_attn(const orc_params *p, const uint16_t *Q, const uint16_t *K, const uint16_t *V,
                     const int32_t *pos, int32_t npos, const int32_t *sup, double *o, double *lse) {
#pragma omp parallel
  {
    double *z = (double *)malloc(sizeof(double) * (size_t)(p->k > 0 ? p->k : 1));
    int32_t *se = (int32_t *)malloc(sizeof(int32_t) * (size_t)(p->k > 0 ? p->k : 1));
#pragma omp for schedule(dynamic, 1)
    for (int32_t i = 0; i < npos; ++i) {
      int32_t s0, n;
      seq_of_pos(p, pos[i], &s0, &n);
      int32_t t = pos[i];
      int32_t ne = 0;                                  /* S_eff = { s in S : s0 <= s <= t } */
      for (int32_t j = 0; j < p->k; ++j) {
        int32_t s = sup[(size_t)i * p->k + j];
        if (s >= s0 && s <= t) se[ne++] = s;
      }
      for (int32_t h = 0; h < p->Hq; ++h) {
        const uint16_t *q = Q + ((size_t)t * p->Hq + h) * p->d;
        int32_t g = g_of_h(p, h);
        double *oo = o ? o + ((size_t)i * p->Hq + h) * p->d : NULL;
        double m = -INFINITY;
        for (int32_t j = 0; j < ne; ++j) {
          const uint16_t *kk = K + ((size_t)se[j] * p->Hkv + g) * p->d;
          double acc = 0.0;
          for (int32_t c = 0; c < p->d; ++c) acc += bf16_to_f64(q[c]) * bf16_to_f64(kk[c]);
          z[j] = p->scale * acc + local_term(p, t, se[j]);
          if (z[j] > m) m = z[j];
        }
        double den = 0.0;
        for (int32_t j = 0; j < ne; ++j) { z[j] = exp(z[j] - m); den += z[j]; }
        if (oo) {
          for (int32_t c = 0; c < p->d; ++c) oo[c] = 0.0;
          for (int32_t j = 0; j < ne; ++j) {
            const uint16_t *vv = V + ((size_t)se[j] * p->Hkv + g) * p->d;
            double w = z[j] / den;
            for (int32_t c = 0; c < p->d; ++c) oo[c] += w * bf16_to_f64(vv[c]);
          }
        }
        if (lse) lse[(size_t)i * p->Hq + h] = ne ? m + log(den) : -INFINITY;
      }
    }
    free(z);
    free(se);
  }
}

/* ---------- O7: dense causal GQA attention, brute force, PAPER.md:94 ---------- */
void orc_dense_attn(const orc_params *p, const uint16_t *Q, const uint16_t *K, const uint16_t *V,
                    const int32_t *pos, int32_t npos, double *o, double *lse) {
#pragma omp parallel
  {
    double *a = (double *)malloc(sizeof(double) * (size_t)(p->L + 1));
#pragma omp for schedule(dynamic, 1)
    for (int32_t i = 0; i < npos; ++i) {
      int32_t s0, n;
      seq_of_pos(p, pos[i], &s0, &n);
      int32_t t = pos[i];
      int32_t cnt = t - s0 + 1;
      for (int32_t h = 0; h < p->Hq; ++h) {
        const uint16_t *q = Q + ((size_t)t * p->Hq + h) * p->d;
        int32_t g = g_of_h(p, h);
        double m = -INFINITY;
        for (int32_t j = 0; j < cnt; ++j) {
          const uint16_t *kk = K + ((size_t)(s0 + j) * p->Hkv + g) * p->d;
          double acc = 0.0;
          for (int32_t c = 0; c < p->d; ++c) acc += bf16_to_f64(q[c]) * bf16_to_f64(kk[c]);
          a[j] = acc * p->scale + local_term(p, t, s0 + j);
          m = a[j] > m ? a[j] : m;
        }
        double den = 0.0;
        for (int32_t j = 0; j < cnt; ++j) { a[j] = exp(a[j] - m); den += a[j]; }
        if (o) {
          double *oo = o + ((size_t)i * p->Hq + h) * p->d;
          for (int32_t c = 0; c < p->d; ++c) {
            double acc = 0.0;
            for (int32_t j = 0; j < cnt; ++j)
              acc += (a[j] / den) * bf16_to_f64(V[((size_t)(s0 + j) * p->Hkv + g) * p->d + c]);
            oo[c] = acc;
          }
        }
        if (lse) lse[(size_t)i * p->Hq + h] = m + log(den);
      }
    }
    free(a);
  }
}

/* ---------------------------------------------------------------------------------------------------------
 * Paged KV cache (stage 4 of the five-stage serving path: "reconstruct K/V from the paged KV cache when
 * the chunked path requires contiguous tensors"; :331, :428 chunked prefill with max_num_batched_tokens 4K / 8K).
 * A cache tensor is [n_pages][page_size][row_elems] bf16; logical token t of the sequence lives in physical page
 * block_table[t / page_size] at slot t % page_size.  Both routines are pure indexing (no arithmetic), so anything
 * computed from the reconstructed tensors is bit-identical to the same computation on the original contiguous
 * tensors -- which is the pin (tests/test_oracle_pins.py::test_paged_*).
 * --------------------------------------------------------------------------------------------------------- */
/* contiguous[t - t_begin, :] = cache[block_table[t / page_size], t % page_size, :]  for t in [t_begin, t_end) */
void orc_paged_gather(const uint16_t *cache, const int32_t *block_table, int32_t page_size, int64_t row_elems,
                      int32_t t_begin, int32_t t_end, uint16_t *contiguous) {
  for (int32_t t = t_begin; t < t_end; ++t) {
    const int64_t page = block_table[t / page_size], slot = t % page_size;
    memcpy(contiguous + (int64_t)(t - t_begin) * row_elems, cache + (page * page_size + slot) * row_elems,
           (size_t)row_elems * sizeof(uint16_t));
  }
}
/* cache[block_table[t / page_size], t % page_size, :] = rows[t - t_begin, :]  for t in [t_begin, t_end): the write a
 * prefill chunk makes for its own tokens before it attends to the prefix */
void orc_paged_scatter(uint16_t *cache, const int32_t *block_table, int32_t page_size, int64_t row_elems,
                       int32_t t_begin, int32_t t_end, const uint16_t *rows) {
  for (int32_t t = t_begin; t < t_end; ++t) {
    const int64_t page = block_table[t / page_size], slot = t % page_size;
    memcpy(cache + (page * page_size + slot) * row_elems, rows + (int64_t)(t - t_begin) * row_elems,
           (size_t)row_elems * sizeof(uint16_t));
  }
}

int32_t orc_max_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}
