/*
 * stage_oracle.c — TEST INFRASTRUCTURE, not product.  A plain, slow, obviously-correct CPU statement of what one
 * ShuntServe pipeline stage computes (arxiv/paper_2606_18600).  Only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference legs may load it.  It shares no code with the CUDA path.
 *
 * What it follows.  The paper names the operations of a stage and costs them (Table 2: QKV
 * projection, attention prefill/decode, output projection, up-and-gate projection, down projection, logits) and
 * calls their math "the de-facto standard of transformer-based generative LLMs"; it evaluates on
 * Llama-3.1-70B and Qwen3-32B in BF16.  The result is therefore *defined* as the public pre-norm
 * Llama-3 / Qwen3 decoder layer stack evaluated over the logical (un-paged) KV sequence; paging, split-K, flash
 * tiling and fusion are implementation devices that must not change it.  This file is that definition written as
 * loops, in the order of DESIGN.md "Algorithm" (= SURVEY.md §8(c) steps 2.1-2.10), with the readings A1-A22
 * listed in DESIGN.md.  The migration claim it must satisfy exactly: prefilling prompt +
 * already-generated tokens reconstructs the same KV cache as incremental decode.
 *
 * Arithmetic contract.  Weights, stage input and KV pool are bf16 in memory, widened
 * exactly (bits << 16).  All arithmetic is in `real` = float (default build; north_star fixes "plain fp32") or
 * double (-DSO_F64 build, used to show the fp32 build's own error is small).  K and V are rounded to bf16
 * round-to-nearest-even when stored to the pool, always, and attention always reads K/V back from the pool,
 * including tokens appended by the same call.  rounding = 0 ("R0"): no other rounding.  rounding = 1 ("R1"):
 * additionally round to bf16 where a bf16 engine materialises a tensor (h after each RMSNorm, q after RoPE,
 * attention output, SwiGLU output); the residual stream stays `real`.
 *
 * Every output element is produced by one thread with a reduction order that depends only on the reduction
 * index — never on T, batch composition, thread count or call partitioning — so the invariants tested in
 * tests/test_oracle_pins.py (page permutation, migration, chunking, batch composition) hold bit for bit.
 *
 * Pins: tests/test_oracle_pins.py (P1-P13 of DESIGN.md).  Nothing here is "parity unpinned" except what
 * DESIGN.md lists under that name.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#ifdef SO_F64
typedef double real;
#define R_EXP exp
#define R_SQRT sqrt
#else
typedef float real;
#define R_EXP expf
#define R_SQRT sqrtf
#endif

typedef struct {
  int32_t hidden, n_q, n_kv, d, ffn, vocab;
  float eps, theta;
  int32_t qk_norm;   /* 1: per-head RMSNorm on q and k before RoPE (A11) */
  int32_t rounding;  /* 0 = R0, 1 = R1 */
} so_dims;

/* optional per-layer taps (any may be NULL); used by per-kernel parity tests */
typedef struct {
  real *h1;    /* [T,H]   after RMSNorm-1 (after R1 rounding if on) */
  real *q;     /* [T,Hq]  after QK-norm + RoPE (after R1 rounding if on) */
  real *attn;  /* [T,Hq]  attention output (after R1 rounding if on) */
  real *x1;    /* [T,H]   residual after the output projection */
  real *a;     /* [T,F]   SwiGLU output (after R1 rounding if on) */
} so_taps;

int so_real_bytes(void) { return (int)sizeof(real); }

/* ---- bf16 <-> real ------------------------------------------------------------------------------------- */
static inline float bf16_to_f32(uint16_t b) {
  uint32_t u = ((uint32_t)b) << 16;
  float f;
  memcpy(&f, &u, 4);
  return f;
}
/* round-to-nearest-even from fp32 bits; NaN stays NaN (quiet) */
static inline uint16_t f32_to_bf16_rne(float f) {
  uint32_t u;
  memcpy(&u, &f, 4);
  if ((u & 0x7fffffffu) > 0x7f800000u) return (uint16_t)((u >> 16) | 0x0040u);
  uint32_t lsb = (u >> 16) & 1u;
  u += 0x7fffu + lsb;
  return (uint16_t)(u >> 16);
}
/* real -> bf16: the value is first brought to fp32 (identity in the fp32 build), then RNE to bf16.  In the f64
 * build a double is rounded to fp32 first; the double rounding is part of that build's contract (it exists
 * only to bound the fp32 build's error). */
static inline uint16_t real_to_bf16(real v) { return f32_to_bf16_rne((float)v); }
static inline real round_bf16(real v) { return (real)bf16_to_f32(real_to_bf16(v)); }

uint16_t so_f32_to_bf16(float f) { return f32_to_bf16_rne(f); }
float so_bf16_to_f32(uint16_t b) { return bf16_to_f32(b); }

/* ---- S1/S8: RMSNorm.  out[t,:] = x[t,:] * (1/sqrt(mean_j x[t,j]^2 + eps)) * w[:]  (step 2.1 / 2.8) ------- */
void so_rmsnorm(const real *x, const uint16_t *w, real *out, int T, int n, float eps, int round_out) {
#pragma omp parallel for schedule(static)
  for (int t = 0; t < T; ++t) {
    const real *xr = x + (size_t)t * n;
    real ss = 0;
    for (int j = 0; j < n; ++j) ss += xr[j] * xr[j];
    real inv = (real)1 / R_SQRT(ss / (real)n + (real)eps);
    for (int j = 0; j < n; ++j) {
      real v = xr[j] * inv * (real)bf16_to_f32(w[j]);
      out[(size_t)t * n + j] = round_out ? round_bf16(v) : v;
    }
  }
}

/* ---- S2/S7/S9/S10/S11: projection.  out[t,n] = sum_k x[t,k] * W[n,k]   (Table 2 GEMM rows) ---------------
 * Row n of W is the weight vector of output feature n.  Parallel over n; W row widened once; 16 interleaved
 * partial sums indexed by k mod 16, combined in a fixed order.  The order depends on k only. */
#define SO_LANES 16
void so_matmul(const real *x, const uint16_t *W, real *out, int T, int N, int K, int ld_out) {
#pragma omp parallel
  {
    real *wrow = (real *)malloc(sizeof(real) * (size_t)K);
#pragma omp for schedule(static)
    for (int n = 0; n < N; ++n) {
      const uint16_t *wr = W + (size_t)n * K;
      for (int k = 0; k < K; ++k) wrow[k] = (real)bf16_to_f32(wr[k]);
      for (int t = 0; t < T; ++t) {
        const real *xr = x + (size_t)t * K;
        real acc[SO_LANES];
        for (int i = 0; i < SO_LANES; ++i) acc[i] = 0;
        int k = 0;
        for (; k + SO_LANES <= K; k += SO_LANES)
          for (int i = 0; i < SO_LANES; ++i) acc[i] += xr[k + i] * wrow[k + i];
        for (int i = 0; k + i < K; ++i) acc[i] += xr[k + i] * wrow[k + i];
        real s = 0;
        for (int i = 0; i < SO_LANES; ++i) s += acc[i];
        out[(size_t)t * ld_out + n] = s;
      }
    }
    free(wrow);
  }
}

/* ---- S3: per-head RMSNorm over d with a gain shared by all heads (Qwen3; A11) ---------------------------- */
void so_head_rmsnorm(real *u, const uint16_t *g, int T, int n_heads, int d, float eps) {
#pragma omp parallel for schedule(static)
  for (int t = 0; t < T; ++t)
    for (int h = 0; h < n_heads; ++h) {
      real *v = u + ((size_t)t * n_heads + h) * d;
      real ss = 0;
      for (int c = 0; c < d; ++c) ss += v[c] * v[c];
      real inv = (real)1 / R_SQRT(ss / (real)d + (real)eps);
      for (int c = 0; c < d; ++c) v[c] = v[c] * inv * (real)bf16_to_f32(g[c]);
    }
}

/* ---- S4: RoPE, rotate-half pairing (c, c+d/2), angle = pos * inv_freq[c] (A10).  cos/sin are computed in
 * double and stored as fp32 (the table a bf16 engine would hold); in the f64 build they stay double. -------- */
void so_rope(real *u, const int32_t *pos, int T, int n_heads, int d, float theta, const float *inv_freq) {
  int half = d / 2;
#pragma omp parallel for schedule(static)
  for (int t = 0; t < T; ++t) {
    for (int c = 0; c < half; ++c) {
      double f = inv_freq ? (double)inv_freq[c] : pow((double)theta, -2.0 * (double)c / (double)d);
      double ang = (double)pos[t] * f;
#ifdef SO_F64
      real cs = cos(ang), sn = sin(ang);
#else
      real cs = (float)cos(ang), sn = (float)sin(ang);
#endif
      for (int h = 0; h < n_heads; ++h) {
        real *v = u + ((size_t)t * n_heads + h) * d;
        real a = v[c], b = v[c + half];
        v[c] = a * cs - b * sn;
        v[c + half] = b * cs + a * sn;
      }
    }
  }
}

/* address of (page, head, slot) in one layer's K or V pool: [page][h_kv][16][d] */
static inline size_t pool_off(int page, int h, int slot, int n_kv, int d) {
  return (((size_t)page * n_kv + h) * 16 + (size_t)slot) * d;
}

/* ---- S5: KV append.  Kpool[bt[s][p>>4]][hk][p&15][:] = bf16_rne(k[t,hk,:]) (step 2.5) -------------------- */
void so_kv_append(const real *k, const real *v, uint16_t *kpool, uint16_t *vpool, int n_seqs,
                  const int32_t *cu_q, const int32_t *ctx_before, const int32_t *bt, int max_blocks, int n_kv,
                  int d) {
  for (int s = 0; s < n_seqs; ++s)
    for (int i = 0; i < cu_q[s + 1] - cu_q[s]; ++i) {
      int t = cu_q[s] + i, p = ctx_before[s] + i;
      int page = bt[(size_t)s * max_blocks + (p >> 4)], slot = p & 15;
      for (int h = 0; h < n_kv; ++h) {
        size_t o = pool_off(page, h, slot, n_kv, d);
        for (int c = 0; c < d; ++c) {
          kpool[o + c] = real_to_bf16(k[((size_t)t * n_kv + h) * d + c]);
          vpool[o + c] = real_to_bf16(v[((size_t)t * n_kv + h) * d + c]);
        }
      }
    }
}

/* ---- S6: attention (step 2.6).  Query at global position p attends keys j = 0..p read from the pool;
 * s_j = <q, K_j> / sqrt(d); m = max_j s_j; e_j = exp(s_j - m); l = sum_j e_j; o = (sum_j e_j V_j) / l,
 * j ascending, divide last.  q head hq uses kv head hq / G (A16).  Decode is the q_len = 1 case. ----------- */
void so_attention(const real *q, const uint16_t *kpool, const uint16_t *vpool, real *out, int n_seqs,
                  const int32_t *cu_q, const int32_t *ctx_before, const int32_t *bt, int max_blocks, int n_q,
                  int n_kv, int d, int round_out) {
  int G = n_q / n_kv;
  real scale = (real)1 / R_SQRT((real)d);
  int T = cu_q[n_seqs];
  /* token -> sequence map so the parallel loop is over (token, head) */
  int32_t *seq_of = (int32_t *)malloc(sizeof(int32_t) * (size_t)(T > 0 ? T : 1));
  for (int s = 0; s < n_seqs; ++s)
    for (int t = cu_q[s]; t < cu_q[s + 1]; ++t) seq_of[t] = s;
#pragma omp parallel
  {
    real *sc = NULL;
    size_t sc_cap = 0;
#pragma omp for schedule(dynamic, 4) collapse(2)
    for (int t = 0; t < T; ++t)
      for (int hq = 0; hq < n_q; ++hq) {
        int s = seq_of[t];
        int p = ctx_before[s] + (t - cu_q[s]);
        int hk = hq / G;
        const int32_t *row = bt + (size_t)s * max_blocks;
        const real *qv = q + ((size_t)t * n_q + hq) * d;
        if ((size_t)(p + 1) > sc_cap) {
          sc_cap = (size_t)(p + 1) * 2;
          sc = (real *)realloc(sc, sizeof(real) * sc_cap);
        }
        real m = -INFINITY;
        for (int j = 0; j <= p; ++j) {
          const uint16_t *kr = kpool + pool_off(row[j >> 4], hk, j & 15, n_kv, d);
          real dot = 0;
          for (int c = 0; c < d; ++c) dot += qv[c] * (real)bf16_to_f32(kr[c]);
          sc[j] = dot * scale;
          if (sc[j] > m) m = sc[j];
        }
        real l = 0;
        real *ov = out + ((size_t)t * n_q + hq) * d;
        for (int c = 0; c < d; ++c) ov[c] = 0;
        for (int j = 0; j <= p; ++j) {
          real e = R_EXP(sc[j] - m);
          l += e;
          const uint16_t *vr = vpool + pool_off(row[j >> 4], hk, j & 15, n_kv, d);
          for (int c = 0; c < d; ++c) ov[c] += e * (real)bf16_to_f32(vr[c]);
        }
        for (int c = 0; c < d; ++c) {
          real v = ov[c] / l;
          ov[c] = round_out ? round_bf16(v) : v;
        }
      }
    free(sc);
  }
  free(seq_of);
}

/* softmax weights of one (token, head) row, for the "rows sum to 1" pin: writes e_j / l into w[0..p] */
void so_attention_weights(const real *qv, const uint16_t *kpool, const int32_t *bt_row, int p, int hk, int n_kv,
                          int d, real *w) {
  real scale = (real)1 / R_SQRT((real)d);
  real m = -INFINITY;
  for (int j = 0; j <= p; ++j) {
    const uint16_t *kr = kpool + pool_off(bt_row[j >> 4], hk, j & 15, n_kv, d);
    real dot = 0;
    for (int c = 0; c < d; ++c) dot += qv[c] * (real)bf16_to_f32(kr[c]);
    w[j] = dot * scale;
    if (w[j] > m) m = w[j];
  }
  real l = 0;
  for (int j = 0; j <= p; ++j) {
    w[j] = R_EXP(w[j] - m);
    l += w[j];
  }
  for (int j = 0; j <= p; ++j) w[j] /= l;
}

/* ---- S9 elementwise: a = g / (1 + exp(-g)) * u (step 2.9) ------------------------------------------------ */
void so_swiglu(const real *g, const real *u, real *a, size_t n, int round_out) {
#pragma omp parallel for schedule(static)
  for (size_t i = 0; i < n; ++i) {
    real v = g[i] / ((real)1 + R_EXP(-g[i])) * u[i];
    a[i] = round_out ? round_bf16(v) : v;
  }
}

/* ---- one decoder layer over a packed varlen call (steps 2.1-2.10).  x [T,H] is the residual stream, updated
 * in place.  kpool/vpool are THIS layer's pools. ----------------------------------------------------------- */
int so_layer(const so_dims *dm, const uint16_t *ln1, const uint16_t *wq, const uint16_t *wk, const uint16_t *wv,
             const uint16_t *q_norm, const uint16_t *k_norm, const uint16_t *wo, const uint16_t *ln2,
             const uint16_t *w_gate, const uint16_t *w_up, const uint16_t *w_down, uint16_t *kpool,
             uint16_t *vpool, int n_seqs, const int32_t *cu_q, const int32_t *ctx_before, const int32_t *bt,
             int max_blocks, const float *inv_freq, real *x, const so_taps *taps) {
  const int H = dm->hidden, d = dm->d, Hq = dm->n_q * d, Hkv = dm->n_kv * d, F = dm->ffn;
  const int T = cu_q[n_seqs];
  const int r1 = dm->rounding;
  if (T <= 0) return 0;
  size_t big = (size_t)T * (size_t)(H > F ? H : F);
  real *h = (real *)malloc(sizeof(real) * big);
  real *q = (real *)malloc(sizeof(real) * (size_t)T * Hq);
  real *k = (real *)malloc(sizeof(real) * (size_t)T * Hkv);
  real *v = (real *)malloc(sizeof(real) * (size_t)T * Hkv);
  real *o = (real *)malloc(sizeof(real) * (size_t)T * Hq);
  real *g = (real *)malloc(sizeof(real) * (size_t)T * F);
  real *u = (real *)malloc(sizeof(real) * (size_t)T * F);
  real *y = (real *)malloc(sizeof(real) * (size_t)T * H);
  int32_t *pos = (int32_t *)malloc(sizeof(int32_t) * (size_t)T);
  if (!h || !q || !k || !v || !o || !g || !u || !y || !pos) return -1;
  for (int s = 0; s < n_seqs; ++s)
    for (int t = cu_q[s]; t < cu_q[s + 1]; ++t) pos[t] = ctx_before[s] + (t - cu_q[s]);

  so_rmsnorm(x, ln1, h, T, H, dm->eps, r1);                                   /* 2.1 */
  if (taps && taps->h1) memcpy(taps->h1, h, sizeof(real) * (size_t)T * H);
  so_matmul(h, wq, q, T, Hq, H, Hq);                                           /* 2.2 */
  so_matmul(h, wk, k, T, Hkv, H, Hkv);
  so_matmul(h, wv, v, T, Hkv, H, Hkv);
  if (dm->qk_norm) {                                                           /* 2.3 */
    so_head_rmsnorm(q, q_norm, T, dm->n_q, d, dm->eps);
    so_head_rmsnorm(k, k_norm, T, dm->n_kv, d, dm->eps);
  }
  so_rope(q, pos, T, dm->n_q, d, dm->theta, inv_freq);                         /* 2.4 */
  so_rope(k, pos, T, dm->n_kv, d, dm->theta, inv_freq);
  if (r1)
    for (size_t i = 0; i < (size_t)T * Hq; ++i) q[i] = round_bf16(q[i]);
  if (taps && taps->q) memcpy(taps->q, q, sizeof(real) * (size_t)T * Hq);
  so_kv_append(k, v, kpool, vpool, n_seqs, cu_q, ctx_before, bt, max_blocks, dm->n_kv, d); /* 2.5 */
  so_attention(q, kpool, vpool, o, n_seqs, cu_q, ctx_before, bt, max_blocks, dm->n_q, dm->n_kv, d, r1); /* 2.6 */
  if (taps && taps->attn) memcpy(taps->attn, o, sizeof(real) * (size_t)T * Hq);
  so_matmul(o, wo, y, T, H, Hq, H);                                            /* 2.7 */
  for (size_t i = 0; i < (size_t)T * H; ++i) x[i] = x[i] + y[i];
  if (taps && taps->x1) memcpy(taps->x1, x, sizeof(real) * (size_t)T * H);
  so_rmsnorm(x, ln2, h, T, H, dm->eps, r1);                                   /* 2.8 */
  so_matmul(h, w_gate, g, T, F, H, F);                                         /* 2.9 */
  so_matmul(h, w_up, u, T, F, H, F);
  so_swiglu(g, u, g, (size_t)T * F, r1);
  if (taps && taps->a) memcpy(taps->a, g, sizeof(real) * (size_t)T * F);
  so_matmul(g, w_down, y, T, H, F, H);                                         /* 2.10 */
  for (size_t i = 0; i < (size_t)T * H; ++i) x[i] = x[i] + y[i];

  free(h); free(q); free(k); free(v); free(o); free(g); free(u); free(y); free(pos);
  return 0;
}

/* ---- S0: embedding gather ------------------------------------------------------------------------------- */
void so_embed(const uint16_t *emb, const int32_t *ids, real *x, int T, int H) {
  for (int t = 0; t < T; ++t)
    for (int j = 0; j < H; ++j) x[(size_t)t * H + j] = (real)bf16_to_f32(emb[(size_t)ids[t] * H + j]);
}

/* ---- S11: logits of n_rows rows: z = rmsnorm(y; wf) * Wlm^T; argmax = lowest index among maxima; margin =
 * top1 - top2 (step 3; Table 2 "Logits Calculation") ------------------------------------- */
void so_logits(const so_dims *dm, const real *y, const uint16_t *final_norm, const uint16_t *lm_head, int n_rows,
               real *logits, int32_t *argmax, real *margin) {
  const int H = dm->hidden, V = dm->vocab;
  real *z = (real *)malloc(sizeof(real) * (size_t)n_rows * H);
  so_rmsnorm(y, final_norm, z, n_rows, H, dm->eps, dm->rounding);
  so_matmul(z, lm_head, logits, n_rows, V, H, V);
  for (int r = 0; r < n_rows; ++r) {
    const real *lr = logits + (size_t)r * V;
    int best = 0;
    for (int i = 1; i < V; ++i)
      if (lr[i] > lr[best]) best = i;
    real second = -INFINITY;
    for (int i = 0; i < V; ++i)
      if (i != best && lr[i] > second) second = lr[i];
    if (argmax) argmax[r] = best;
    if (margin) margin[r] = lr[best] - second;
  }
  free(z);
}
