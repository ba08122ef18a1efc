/*
 * dovetail_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * A plain, slow, fp64 CPU restatement of the Dovetail draft step
 * (arxiv 2412.18934), written from the paper. Only tests/, the smoke check in
 * __graft_entry__.py and bench.py's cpu_baseline / --impl reference legs may
 * call it. It shares no code with the CUDA path and includes none of its
 * headers; the layouts it reads (weights row-major [out,in], KV cache
 * [layer][kv_head][capacity][head_dim]) are those include/dovetail.h states.
 *
 * Every reduction is a plain sequential sum in double over the stored values
 * (bf16 / fp32 numbers widened exactly). The only rounding is where a value is
 * STORED in a 16-bit or 32-bit buffer: new K/V rows written to the cache
 * (round-to-nearest-even to the cache dtype), reading A12.
 * OpenMP is used over independent output elements only, so results do not
 * depend on the thread count.
 *
 * Steps follow SURVEY.md 8(c) O1-O9; citations are PAPER.md line numbers.
 * Parity pins: tests/test_oracle_*.py.
 * Unpinned: absolute logit values for real text (no trained weights exist
 * here) -- "parity unpinned" for that alone.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#define ORC_F32 0
#define ORC_BF16 1

typedef struct {
  int32_t hidden, n_q_heads, n_kv_heads, head_dim, n_layers, ffn, vocab;
  double rope_theta, rms_eps;
  int32_t dtype, dgf_proj, first_layer_input_norm, final_norm;
  int32_t fusion; /* 0: Dynamic Gating Fusion (the paper's); 1: concat + one Linear (the EAGLE-2 baseline, "w/o both") */
  int32_t wquant; /* 0: matrices stored in dtype; 1: int8, 2: fp8 e4m3, each with one fp32 scale per output row */
} orc_config_t;

typedef struct {
  const void *g_attn, *wq, *wk, *wv, *wo, *g_ffn, *wgate, *wup, *wdown;
  const float *sq, *sk, *sv, *so, *sgate, *sup, *sdown; /* wquant: per-row scales of the seven matrices */
} orc_layer_t;

typedef struct {
  const void *embed, *dgf_w1, *dgf_w2, *dgf_wg, *dgf_bg;
  const orc_layer_t* layers;
  const void* g_final;
  const void* lm_head;
  const float *dgf_s1, *dgf_s2, *dgf_sg, *lm_head_s; /* wquant: per-row scales */
} orc_weights_t;

/* ---- stored-value access ------------------------------------------------ */

/* Widen stored element i of a buffer of the given dtype to double (exact). */
static double ld(const void* p, size_t i, int dtype) {
  if (dtype == ORC_F32) return (double)((const float*)p)[i];
  uint32_t bits = (uint32_t)((const uint16_t*)p)[i] << 16; /* bf16 = top half of fp32 */
  float f;
  memcpy(&f, &bits, 4);
  return (double)f;
}

/* Round a double to bf16 (8 significant bits), nearest-even, directly (no
 * intermediate fp32 rounding). Range is that of normal floats; the draft's
 * activations are far from the limits. */
static uint16_t to_bf16(double x) {
  if (x == 0.0 || isnan(x) || isinf(x)) {
    float f = (float)x;
    uint32_t b;
    memcpy(&b, &f, 4);
    return (uint16_t)(b >> 16);
  }
  int e;
  double m = frexp(x, &e);          /* x = m * 2^e, 0.5 <= |m| < 1 */
  double q = nearbyint(m * 256.0);  /* 8 significant bits, ties to even */
  float f = (float)ldexp(q / 256.0, e); /* exact: q/256 has <= 9 bits */
  uint32_t b;
  memcpy(&b, &f, 4);
  return (uint16_t)(b >> 16);
}

/* exported for the rounding pin */
uint16_t orc_round_bf16(double x) { return to_bf16(x); }

static void st(void* p, size_t i, int dtype, double x) {
  if (dtype == ORC_F32) ((float*)p)[i] = (float)x;
  else ((uint16_t*)p)[i] = to_bf16(x);
}

/* ---- primitive steps (exported so the tests can pin each one) ----------- */

/* int8 weight-quantised draft (App. C.2: "it is advisable to apply int8 quantization to the drafting
 * model on the GPU"): a matrix is stored as int8 q[N,K] with one fp32 scale per output row; its value is the
 * dequantised W[n,k] = scale[n] * q[n,k] (exact in double), and everything else is the same fp64 arithmetic.
 * y[n] = sum_k (scale[n] * q[n,k]) x[k]. */
void orc_matvec_q8(const int8_t* Q, const float* scale, int N, int K, const double* x, double* y) {
#pragma omp parallel for schedule(static)
  for (int n = 0; n < N; ++n) {
    double s = 0.0, sc = (double)scale[n];
    size_t base = (size_t)n * (size_t)K;
    for (int k = 0; k < K; ++k) s += (sc * (double)Q[base + k]) * x[k];
    y[n] = s;
  }
}

/* The 8-bit float variant of the same scheme (reading A17b; SURVEY.md 8 f1 "int8 / fp8"): a matrix is stored as
 * fp8 e4m3 bytes with one fp32 scale per output row, W[n,k] = scale[n] * e4m3(q[n,k]).
 * e4m3 (the "fn" flavour: no infinities): 1 sign, 4 exponent (bias 7), 3 mantissa bits; exponent 0 is subnormal
 * (m / 8 * 2^-6); exponent 15 with mantissa 7 is NaN; the largest finite value is 1.75 * 2^8 = 448. */
double orc_e4m3_to_double(uint8_t b) {
  int s = b >> 7, e = (b >> 3) & 15, m = b & 7;
  double v;
  if (e == 15 && m == 7) return NAN;
  if (e == 0) v = ldexp((double)m / 8.0, -6);
  else v = ldexp(1.0 + (double)m / 8.0, e - 7);
  return s ? -v : v;
}

void orc_matvec_f8(const uint8_t* Q, const float* scale, int N, int K, const double* x, double* y) {
#pragma omp parallel for schedule(static)
  for (int n = 0; n < N; ++n) {
    double s = 0.0, sc = (double)scale[n];
    size_t base = (size_t)n * (size_t)K;
    for (int k = 0; k < K; ++k) s += (sc * orc_e4m3_to_double(Q[base + k])) * x[k];
    y[n] = s;
  }
}

/* A weight matrix of the model: stored in dtype, or (scale != NULL) 8-bit (wquant 1: int8, 2: e4m3) with per-row scales. */
static void mat(const void* W, const float* scale, int wquant, int dtype, int N, int K, const double* x, double* y);

/* y[n] = sum_k W[n,k] x[k], W row-major [N,K]. */
void orc_matvec(const void* W, int dtype, int N, int K, const double* x, double* y) {
#pragma omp parallel for schedule(static)
  for (int n = 0; n < N; ++n) {
    double s = 0.0;
    size_t base = (size_t)n * (size_t)K;
    for (int k = 0; k < K; ++k) s += ld(W, base + k, dtype) * x[k];
    y[n] = s;
  }
}

static void mat(const void* W, const float* scale, int wquant, int dtype, int N, int K, const double* x, double* y) {
  if (wquant == 1) orc_matvec_q8((const int8_t*)W, scale, N, K, x, y);
  else if (wquant == 2) orc_matvec_f8((const uint8_t*)W, scale, N, K, x, y);
  else orc_matvec(W, dtype, N, K, x, y);
}

/* RMSNorm: y = x / sqrt(mean(x^2) + eps) * g   (LLaMA block, reading A3). */
void orc_rmsnorm(const double* x, const void* g, int dtype, int d, double eps, double* y) {
  double ss = 0.0;
  for (int i = 0; i < d; ++i) ss += x[i] * x[i];
  double r = 1.0 / sqrt(ss / d + eps);
  for (int i = 0; i < d; ++i) y[i] = x[i] * r * ld(g, i, dtype);
}

/* Rotary embedding on one head vector, half-split pairing (i, i + dh/2):
 * angle_i = pos * theta^(-2i/dh)   (reading A3). In place. */
void orc_rope(double* v, int dh, int pos, double theta) {
  int half = dh / 2;
  for (int i = 0; i < half; ++i) {
    double ang = (double)pos * pow(theta, -2.0 * i / dh);
    double c = cos(ang), s = sin(ang);
    double a = v[i], b = v[i + half];
    v[i] = a * c - b * s;
    v[i + half] = b * c + a * s;
  }
}

static double sigmoid(double z) { return 1.0 / (1.0 + exp(-z)); }
static double silu(double z) { return z * sigmoid(z); }

/* O3 -- Dynamic Gating Fusion (Fig. 5 :98).
 * f: target hidden feature [d]; token: its id. x out [d].
 * h1 = W1 f, h2 = W2 e (identity when dgf_proj == 0), g = sigmoid(Wg [h1||h2] + bg),
 * x = g*h1 + (1-g)*h2  (readings A1, A2). */
void orc_dgf(const orc_config_t* c, const orc_weights_t* w, const double* f, int token, double* x) {
  int d = c->hidden, dt = c->dtype;
  double* e = (double*)malloc(sizeof(double) * d);
  double* h = (double*)malloc(sizeof(double) * 2 * d);
  double* z = (double*)malloc(sizeof(double) * d);
  for (int i = 0; i < d; ++i) e[i] = ld(w->embed, (size_t)token * d + i, dt);
  if (c->dgf_proj) {
    mat(w->dgf_w1, w->dgf_s1, c->wquant, dt, d, d, f, h);
    mat(w->dgf_w2, w->dgf_s2, c->wquant, dt, d, d, e, h + d);
  } else {
    for (int i = 0; i < d; ++i) { h[i] = f[i]; h[d + i] = e[i]; }
  }
  mat(w->dgf_wg, w->dgf_sg, c->wquant, dt, d, 2 * d, h, z);
  for (int i = 0; i < d; ++i) {
    double g = sigmoid(z[i] + ld(w->dgf_bg, i, dt));
    x[i] = g * h[i] + (1.0 - g) * h[d + i];
  }
  free(e); free(h); free(z);
}

/* The fusion DGF replaces ("simply concatenates the two and maps them to the hidden
 * state dimension through a single linear transformation"; Table 6 row "w/o both"):
 * x = Wfc [f || e] + bfc, Wfc [d, 2d] and bfc [d] in the dgf_wg / dgf_bg slots (reading A17: hidden
 * state first, as in DGF's [h1 || h2]; with bias, the 2d^2 + d count of SURVEY.md P1). */
void orc_fusion_linear(const orc_config_t* c, const orc_weights_t* w, const double* f, int token, double* x) {
  int d = c->hidden, dt = c->dtype;
  double* h = (double*)malloc(sizeof(double) * 2 * d);
  for (int i = 0; i < d; ++i) { h[i] = f[i]; h[d + i] = ld(w->embed, (size_t)token * d + i, dt); }
  mat(w->dgf_wg, w->dgf_sg, c->wquant, dt, d, 2 * d, h, x);
  for (int i = 0; i < d; ++i) x[i] += ld(w->dgf_bg, i, dt);
  free(h);
}

/* Attention of one row (O4): q [Hq*dh] already rotated; the row may attend the
 * cache slots listed in allowed[0..n_allowed). K (post-RoPE) and V are read
 * from the cache of this layer as stored. out [Hq*dh]. GQA: q-head h uses
 * kv-head h / (Hq/Hkv). */
void orc_attention_row(const orc_config_t* c, const void* kc, const void* vc, int capacity,
                       int layer, const double* q, const int* allowed, int n_allowed,
                       double* out) {
  int Hq = c->n_q_heads, Hkv = c->n_kv_heads, dh = c->head_dim, dt = c->dtype;
  int grp = Hq / Hkv;
  double scale = 1.0 / sqrt((double)dh);
#pragma omp parallel for schedule(static)
  for (int h = 0; h < Hq; ++h) {
    int kvh = h / grp;
    size_t hb = (((size_t)layer * Hkv + kvh) * (size_t)capacity) * dh;
    double* s = (double*)malloc(sizeof(double) * n_allowed);
    double mx = -INFINITY;
    for (int j = 0; j < n_allowed; ++j) {
      size_t rb = hb + (size_t)allowed[j] * dh;
      double a = 0.0;
      for (int t = 0; t < dh; ++t) a += q[h * dh + t] * ld(kc, rb + t, dt);
      s[j] = a * scale;
      if (s[j] > mx) mx = s[j];
    }
    double z = 0.0;
    for (int j = 0; j < n_allowed; ++j) { s[j] = exp(s[j] - mx); z += s[j]; }
    for (int t = 0; t < dh; ++t) {
      double a = 0.0;
      for (int j = 0; j < n_allowed; ++j)
        a += (s[j] / z) * ld(vc, hb + (size_t)allowed[j] * dh + t, dt);
      out[h * dh + t] = a;
    }
    free(s);
  }
}

/* log-softmax over the vocabulary: logp = logits - logsumexp(logits). */
void orc_log_softmax(const double* logits, int V, double* logp) {
  double mx = -INFINITY;
  for (int i = 0; i < V; ++i) if (logits[i] > mx) mx = logits[i];
  double z = 0.0;
  for (int i = 0; i < V; ++i) z += exp(logits[i] - mx);
  double lz = mx + log(z);
  for (int i = 0; i < V; ++i) logp[i] = logits[i] - lz;
}

/* Top-b of a length-n array by (value desc, index asc) (reading A7).
 * Plain repeated selection. idx out [b]. */
void orc_topk(const double* v, int n, int b, int* idx) {
  char* used = (char*)calloc((size_t)n, 1);
  for (int r = 0; r < b; ++r) {
    int best = -1;
    for (int i = 0; i < n; ++i) {
      if (used[i]) continue;
      if (best < 0 || v[i] > v[best]) best = i; /* strict >: lowest index wins ties */
    }
    idx[r] = best;
    used[best] = 1;
  }
  free(used);
}

/* ---- one forward of a set of rows (O3-O5) -------------------------------- */

typedef struct {
  int slot;           /* cache row this row's K/V is written to   */
  int pos;            /* rotary position                          */
  int n_allowed;      /* cache slots it may attend (incl. itself) */
  int* allowed;
} orc_row_t;

/* Runs rows through DGF and the decoder stack. feats [R][d] (double), tokens
 * [R]. Writes K/V rows into the cache, hhat [R][d] = output hidden state. */
static void forward_rows(const orc_config_t* c, const orc_weights_t* w, void* kc, void* vc,
                         int capacity, const orc_row_t* rows, int R, const double* feats,
                         const int* tokens, double* hhat) {
  int d = c->hidden, Hq = c->n_q_heads, Hkv = c->n_kv_heads, dh = c->head_dim, F = c->ffn;
  int dt = c->dtype;
  int dq = Hq * dh, dkv = Hkv * dh;
  double* x = (double*)malloc(sizeof(double) * (size_t)R * d);
  double* q = (double*)malloc(sizeof(double) * (size_t)R * dq);
  double* n = (double*)malloc(sizeof(double) * d);
  double* k = (double*)malloc(sizeof(double) * dkv);
  double* v = (double*)malloc(sizeof(double) * dkv);
  double* o = (double*)malloc(sizeof(double) * dq);
  double* t = (double*)malloc(sizeof(double) * d);
  double* ga = (double*)malloc(sizeof(double) * F);
  double* up = (double*)malloc(sizeof(double) * F);

  for (int r = 0; r < R; ++r) {
    if (c->fusion == 1) orc_fusion_linear(c, w, feats + (size_t)r * d, tokens[r], x + (size_t)r * d);
    else orc_dgf(c, w, feats + (size_t)r * d, tokens[r], x + (size_t)r * d);
  }

  for (int l = 0; l < c->n_layers; ++l) {
    const orc_layer_t* L = &w->layers[l];
    /* q, k, v of every row of this level first: a level-0 row attends the
     * earlier level-0 rows of the same forward (causal). */
    for (int r = 0; r < R; ++r) {
      double* xr = x + (size_t)r * d;
      if (l == 0 && !c->first_layer_input_norm) memcpy(n, xr, sizeof(double) * d);
      else orc_rmsnorm(xr, L->g_attn, dt, d, c->rms_eps, n);
      mat(L->wq, L->sq, c->wquant, dt, dq, d, n, q + (size_t)r * dq);
      mat(L->wk, L->sk, c->wquant, dt, dkv, d, n, k);
      mat(L->wv, L->sv, c->wquant, dt, dkv, d, n, v);
      for (int h = 0; h < Hq; ++h) orc_rope(q + (size_t)r * dq + h * dh, dh, rows[r].pos, c->rope_theta);
      for (int h = 0; h < Hkv; ++h) orc_rope(k + h * dh, dh, rows[r].pos, c->rope_theta);
      for (int h = 0; h < Hkv; ++h) {
        size_t rb = ((((size_t)l * Hkv + h) * (size_t)capacity) + rows[r].slot) * dh;
        for (int i = 0; i < dh; ++i) {
          st(kc, rb + i, dt, k[h * dh + i]); /* stored post-RoPE, rounded to cache dtype */
          st(vc, rb + i, dt, v[h * dh + i]);
        }
      }
    }
    for (int r = 0; r < R; ++r) {
      double* xr = x + (size_t)r * d;
      orc_attention_row(c, kc, vc, capacity, l, q + (size_t)r * dq, rows[r].allowed,
                        rows[r].n_allowed, o);
      mat(L->wo, L->so, c->wquant, dt, d, dq, o, t);
      for (int i = 0; i < d; ++i) xr[i] += t[i];
      orc_rmsnorm(xr, L->g_ffn, dt, d, c->rms_eps, n);
      mat(L->wgate, L->sgate, c->wquant, dt, F, d, n, ga);
      mat(L->wup, L->sup, c->wquant, dt, F, d, n, up);
      for (int i = 0; i < F; ++i) ga[i] = silu(ga[i]) * up[i];
      mat(L->wdown, L->sdown, c->wquant, dt, d, F, ga, t);
      for (int i = 0; i < d; ++i) xr[i] += t[i];
    }
  }
  memcpy(hhat, x, sizeof(double) * (size_t)R * d);
  free(x); free(q); free(n); free(k); free(v); free(o); free(t); free(ga); free(up);
}

/* O5: logits = Wlm * (optionally RMSNorm'd) hhat. */
void orc_lm_head(const orc_config_t* c, const orc_weights_t* w, const double* hhat, double* logits) {
  int d = c->hidden;
  if (c->final_norm) {
    double* n = (double*)malloc(sizeof(double) * d);
    orc_rmsnorm(hhat, w->g_final, c->dtype, d, c->rms_eps, n);
    mat(w->lm_head, w->lm_head_s, c->wquant, c->dtype, c->vocab, d, n, logits);
    free(n);
  } else {
    mat(w->lm_head, w->lm_head_s, c->wquant, c->dtype, c->vocab, d, hhat, logits);
  }
}

/* Exported single-forward entry for the pins: runs R rows whose attention sets
 * are given explicitly. allowed_flat holds the rows' lists back to back. */
void orc_forward(const orc_config_t* c, const orc_weights_t* w, void* kc, void* vc, int capacity,
                 int R, const int* slots, const int* pos, const int* n_allowed,
                 const int* allowed_flat, const double* feats, const int* tokens, double* hhat) {
  orc_row_t* rows = (orc_row_t*)malloc(sizeof(orc_row_t) * R);
  int off = 0;
  for (int r = 0; r < R; ++r) {
    rows[r].slot = slots[r];
    rows[r].pos = pos[r];
    rows[r].n_allowed = n_allowed[r];
    rows[r].allowed = (int*)(allowed_flat + off);
    off += n_allowed[r];
  }
  forward_rows(c, w, kc, vc, capacity, rows, R, feats, tokens, hhat);
  free(rows);
}

/* ---- tree bookkeeping (O6-O8), also exported on its own ------------------ */

typedef struct {
  int token, parent, depth; /* parent: pool index or -1 (child of the root); depth 1-based */
  double cum;               /* sum of natural-log probabilities root -> node (A9) */
  int row;                  /* step row that forwarded it, or -1                  */
} orc_node_t;

/* Order used everywhere a set of nodes is ranked: cum desc, pool index asc (A7). */
static int node_before(const orc_node_t* pool, int a, int b) {
  if (pool[a].cum != pool[b].cum) return pool[a].cum > pool[b].cum;
  return a < b;
}

/* top-n of ids[0..m) by node_before; result in rank order. Plain selection. */
static int select_top(const orc_node_t* pool, const int* ids, int m, int n, int* out) {
  if (n > m) n = m;
  char* used = (char*)calloc((size_t)(m > 0 ? m : 1), 1);
  for (int r = 0; r < n; ++r) {
    int best = -1;
    for (int i = 0; i < m; ++i) {
      if (used[i]) continue;
      if (best < 0 || node_before(pool, ids[i], ids[best])) best = i;
    }
    out[r] = ids[best];
    used[best] = 1;
  }
  free(used);
  return n;
}

/* O8: select top-min(gamma,P) of the pool, emit in pool order, remap parents. */
static int final_rerank(const orc_node_t* pool, int P, int gamma, int32_t* out_ids,
                        double* out_scores, int32_t* out_parents, int32_t* out_depths) {
  int* all = (int*)malloc(sizeof(int) * (P > 0 ? P : 1));
  int* sel = (int*)malloc(sizeof(int) * (P > 0 ? P : 1));
  int* newidx = (int*)malloc(sizeof(int) * (P > 0 ? P : 1));
  for (int i = 0; i < P; ++i) { all[i] = i; newidx[i] = -1; }
  int n = select_top(pool, all, P, gamma, sel);
  char* keep = (char*)calloc((size_t)(P > 0 ? P : 1), 1);
  for (int i = 0; i < n; ++i) keep[sel[i]] = 1;
  int o = 0;
  for (int i = 0; i < P; ++i) {
    if (!keep[i]) continue;
    newidx[i] = o;
    out_ids[o] = pool[i].token;
    out_scores[o] = pool[i].cum;
    out_parents[o] = pool[i].parent < 0 ? -1 : newidx[pool[i].parent];
    if (out_depths) out_depths[o] = pool[i].depth;
    ++o;
  }
  free(all); free(sel); free(newidx); free(keep);
  return o;
}

/* Bookkeeping alone, from given per-row top-b lists (used by the P6 / P10
 * pins and by dovetail_oracle_step itself through the same two helpers).
 * cand_tokens / cand_logp: [n_rows][max_b]; row 0 = the root's list, then the
 * forwarded rows of level 1, 2, ... in frontier order. */
int dovetail_oracle_tree_replay(int depth, const int32_t* branch, const int32_t* beam, int gamma,
                                const int32_t* cand_tokens, const double* cand_logp, int n_rows,
                                int max_b, int32_t* out_ids, double* out_scores,
                                int32_t* out_parents, int32_t* out_depths, int32_t* n_out,
                                int32_t* pool_token, int32_t* pool_parent, int32_t* pool_depth,
                                double* pool_cum, int32_t* pool_size) {
  int cap = 0, m = 1;
  for (int l = 0; l < depth; ++l) {
    if (l >= 1) { int n = m * branch[l - 1]; m = (beam[l] > 0 && beam[l] < n) ? beam[l] : n; }
    cap += m * branch[l];
  }
  orc_node_t* pool = (orc_node_t*)malloc(sizeof(orc_node_t) * (cap > 0 ? cap : 1));
  int P = 0, row = 0;
  /* O6: the root's top-branch[0] tokens are the level-1 candidates. */
  int lvl_begin = 0;
  for (int j = 0; j < branch[0]; ++j) {
    pool[P].token = cand_tokens[j]; pool[P].parent = -1; pool[P].depth = 1;
    pool[P].cum = cand_logp[j]; pool[P].row = -1; ++P;
  }
  row = 1;
  /* O7 */
  for (int l = 1; l < depth; ++l) {
    int n_l = P - lvl_begin;
    int* ids = (int*)malloc(sizeof(int) * n_l);
    int* fr = (int*)malloc(sizeof(int) * n_l);
    for (int i = 0; i < n_l; ++i) ids[i] = lvl_begin + i;
    int want = (beam[l] > 0 && beam[l] < n_l) ? beam[l] : n_l;
    int M = select_top(pool, ids, n_l, want, fr);
    lvl_begin = P;
    for (int i = 0; i < M; ++i) {
      if (row >= n_rows) { free(ids); free(fr); free(pool); return -1; }
      pool[fr[i]].row = row;
      for (int j = 0; j < branch[l]; ++j) {
        pool[P].token = cand_tokens[(size_t)row * max_b + j];
        pool[P].parent = fr[i];
        pool[P].depth = l + 1;
        pool[P].cum = pool[fr[i]].cum + cand_logp[(size_t)row * max_b + j];
        pool[P].row = -1;
        ++P;
      }
      ++row;
    }
    free(ids); free(fr);
  }
  *n_out = final_rerank(pool, P, gamma, out_ids, out_scores, out_parents, out_depths);
  for (int i = 0; i < P; ++i) {
    if (pool_token) pool_token[i] = pool[i].token;
    if (pool_parent) pool_parent[i] = pool[i].parent;
    if (pool_depth) pool_depth[i] = pool[i].depth;
    if (pool_cum) pool_cum[i] = pool[i].cum;
  }
  if (pool_size) *pool_size = P;
  free(pool);
  return 0;
}

/* ---- the step (O1-O8) ---------------------------------------------------- */

/* Returns 0, or -1 on a bad argument. Dumps (each nullable):
 *   row_logits [total_rows][V], row_hhat [total_rows][d]: per step row (level-0
 *   rows first, then tree rows in cache-slot order); level-0 logits are
 *   computed for the last row only. row_slot/row_pos [total_rows].
 *   pool_* : the whole candidate pool; pool_row = step row that forwarded the
 *   node or -1. */
int dovetail_oracle_step(const orc_config_t* c, const orc_weights_t* w, void* kc, void* vc,
                         int32_t capacity, int32_t committed_len, const float* feats,
                         const int32_t* tokens, int32_t n_new, int32_t depth,
                         const int32_t* branch, const int32_t* beam, int32_t gamma,
                         int32_t* out_ids, double* out_scores, int32_t* out_parents,
                         int32_t* out_depths, int32_t* n_out, int32_t* pool_token,
                         int32_t* pool_parent, int32_t* pool_depth, double* pool_cum,
                         int32_t* pool_row, int32_t* pool_size, double* row_logits,
                         double* row_hhat, int32_t* row_slot, int32_t* row_pos,
                         int32_t* total_rows) {
  int d = c->hidden, V = c->vocab;
  if (n_new < 1 || depth < 1) return -1;
  int L = committed_len, Lp = L + n_new;

  /* pool capacity and rows per level (shapes are fixed by the spec: V >= branch) */
  int cap = 0, m = 1, tree_rows = 0;
  for (int l = 0; l < depth; ++l) {
    if (l >= 1) {
      int n = m * branch[l - 1];
      m = (beam[l] > 0 && beam[l] < n) ? beam[l] : n;
      tree_rows += m;
    }
    if (branch[l] < 1 || branch[l] > V) return -1;
    cap += m * branch[l];
  }
  if (Lp + tree_rows > capacity) return -1;

  orc_node_t* pool = (orc_node_t*)malloc(sizeof(orc_node_t) * cap);
  int P = 0;
  int maxR = n_new;
  for (int l = 1, mm = 1; l < depth; ++l) {
    int n = mm * branch[l - 1];
    mm = (beam[l] > 0 && beam[l] < n) ? beam[l] : n;
    if (mm > maxR) maxR = mm;
  }
  double* hh_all = (double*)malloc(sizeof(double) * (size_t)(n_new + tree_rows) * d);
  double* logits = (double*)malloc(sizeof(double) * V);
  double* logp = (double*)malloc(sizeof(double) * V);
  double* fin = (double*)malloc(sizeof(double) * (size_t)maxR * d);
  int* tk = (int*)malloc(sizeof(int) * maxR);
  orc_row_t* rows = (orc_row_t*)malloc(sizeof(orc_row_t) * maxR);
  int* top = (int*)malloc(sizeof(int) * V);
  int step_row = 0;

  /* O2: level-0 rows, causal over the prefix and the earlier new rows
   * (hidden states "along with the corresponding tokens"). */
  for (int i = 0; i < n_new; ++i) {
    rows[i].slot = L + i;
    rows[i].pos = L + i;
    rows[i].n_allowed = L + i + 1;
    rows[i].allowed = (int*)malloc(sizeof(int) * (L + i + 1));
    for (int j = 0; j <= L + i; ++j) rows[i].allowed[j] = j;
    for (int t = 0; t < d; ++t) fin[(size_t)i * d + t] = (double)feats[(size_t)i * d + t];
    tk[i] = tokens[i];
    if (tokens[i] < 0 || tokens[i] >= V) return -1;
  }
  forward_rows(c, w, kc, vc, capacity, rows, n_new, fin, tk, hh_all);
  for (int i = 0; i < n_new; ++i) {
    if (row_slot) row_slot[step_row + i] = rows[i].slot;
    if (row_pos) row_pos[step_row + i] = rows[i].pos;
    free(rows[i].allowed);
  }
  if (row_logits) memset(row_logits, 0, sizeof(double) * (size_t)(n_new + tree_rows) * V);
  /* O5 + O6: the LAST level-0 row seeds the tree. */
  orc_lm_head(c, w, hh_all + (size_t)(n_new - 1) * d, logits);
  if (row_logits) memcpy(row_logits + (size_t)(n_new - 1) * V, logits, sizeof(double) * V);
  orc_log_softmax(logits, V, logp);
  orc_topk(logp, V, branch[0], top);
  for (int j = 0; j < branch[0]; ++j) {
    pool[P].token = top[j]; pool[P].parent = -1; pool[P].depth = 1;
    pool[P].cum = logp[top[j]]; pool[P].row = -1; ++P;
  }
  step_row = n_new;
  int root_row = n_new - 1;

  /* O7: each round forwards the top-beam nodes of the
   * current level by cumulative probability and expands each by its top-k. */
  int lvl_begin = 0, next_slot = Lp;
  for (int l = 1; l < depth; ++l) {
    int n_l = P - lvl_begin;
    int* ids = (int*)malloc(sizeof(int) * n_l);
    int* fr = (int*)malloc(sizeof(int) * n_l);
    for (int i = 0; i < n_l; ++i) ids[i] = lvl_begin + i;
    int want = (beam[l] > 0 && beam[l] < n_l) ? beam[l] : n_l;
    int M = select_top(pool, ids, n_l, want, fr);
    lvl_begin = P;
    for (int i = 0; i < M; ++i) {
      orc_node_t* nd = &pool[fr[i]];
      nd->row = step_row + i;
      rows[i].slot = next_slot + i;
      rows[i].pos = Lp + l - 1;
      /* prefix + ancestors (root -> parent order) + self */
      int na = 0;
      for (int a = nd->parent; a >= 0; a = pool[a].parent) ++na;
      rows[i].n_allowed = Lp + na + 1;
      rows[i].allowed = (int*)malloc(sizeof(int) * rows[i].n_allowed);
      for (int j = 0; j < Lp; ++j) rows[i].allowed[j] = j;
      int k = Lp + na;
      rows[i].allowed[k] = rows[i].slot;
      for (int a = nd->parent; a >= 0; a = pool[a].parent) {
        --k;
        rows[i].allowed[k] = (Lp) + (pool[a].row - n_new); /* ancestor's tree slot */
      }
      /* feature = output hidden state of the parent's row (A4) */
      int prow = nd->parent < 0 ? root_row : pool[nd->parent].row;
      memcpy(fin + (size_t)i * d, hh_all + (size_t)prow * d, sizeof(double) * d);
      tk[i] = nd->token;
    }
    forward_rows(c, w, kc, vc, capacity, rows, M, fin, tk, hh_all + (size_t)step_row * d);
    for (int i = 0; i < M; ++i) {
      if (row_slot) row_slot[step_row + i] = rows[i].slot;
      if (row_pos) row_pos[step_row + i] = rows[i].pos;
      free(rows[i].allowed);
      orc_lm_head(c, w, hh_all + (size_t)(step_row + i) * d, logits);
      if (row_logits) memcpy(row_logits + (size_t)(step_row + i) * V, logits, sizeof(double) * V);
      orc_log_softmax(logits, V, logp);
      orc_topk(logp, V, branch[l], top);
      for (int j = 0; j < branch[l]; ++j) {
        pool[P].token = top[j]; pool[P].parent = fr[i]; pool[P].depth = l + 1;
        pool[P].cum = pool[fr[i]].cum + logp[top[j]]; pool[P].row = -1; ++P;
      }
    }
    step_row += M;
    next_slot += M;
    free(ids); free(fr);
  }

  /* O8: rerank all nodes, keep the top-gamma. */
  *n_out = final_rerank(pool, P, gamma, out_ids, out_scores, out_parents, out_depths);

  for (int i = 0; i < P; ++i) {
    if (pool_token) pool_token[i] = pool[i].token;
    if (pool_parent) pool_parent[i] = pool[i].parent;
    if (pool_depth) pool_depth[i] = pool[i].depth;
    if (pool_cum) pool_cum[i] = pool[i].cum;
    if (pool_row) pool_row[i] = pool[i].row;
  }
  if (pool_size) *pool_size = P;
  if (row_hhat) memcpy(row_hhat, hh_all, sizeof(double) * (size_t)step_row * d);
  if (total_rows) *total_rows = step_row;
  free(pool); free(hh_all); free(logits); free(logp); free(fin); free(tk); free(rows); free(top);
  return 0;
}

/* O9 (reading A11). mode 0: nothing moves. mode 1: the K/V rows
 * of the accepted nodes that were forwarded (path_rows[i] >= 0 = tree-row
 * index, in path order; a leading run) move to cache rows Lp + i. Returns the
 * number of rows moved. Pure data movement on stored values. */
int dovetail_oracle_kv_commit(const orc_config_t* c, void* kc, void* vc, int32_t capacity,
                              int32_t Lp, const int32_t* path_tree_rows, int32_t n_acc,
                              int32_t mode) {
  if (mode == 0) return 0;
  int Hkv = c->n_kv_heads, dh = c->head_dim;
  size_t es = c->dtype == ORC_F32 ? 4 : 2;
  int moved = 0;
  for (int i = 0; i < n_acc; ++i) {
    if (path_tree_rows[i] < 0) break;
    int src = Lp + path_tree_rows[i], dst = Lp + i;
    for (int l = 0; l < c->n_layers; ++l)
      for (int h = 0; h < Hkv; ++h) {
        size_t hb = (((size_t)l * Hkv + h) * (size_t)capacity) * dh;
        memmove((char*)kc + (hb + (size_t)dst * dh) * es, (char*)kc + (hb + (size_t)src * dh) * es, dh * es);
        memmove((char*)vc + (hb + (size_t)dst * dh) * es, (char*)vc + (hb + (size_t)src * dh) * es, dh * es);
      }
    ++moved;
  }
  return moved;
}

/* ---- verification-side bookkeeping and acceptance ---------------------------
 * "These candidates are then sent to the target model ... for parallel verification. The target model
 * computes the logits of the candidate tokens in a single forward pass and applies a speculative sampling
 * algorithm to determine the accepted tokens. The accepted tokens are returned to the ... draft model."
 *
 * Verifier rows: row 0 is the root (the last verified token, whose successor distribution the target has
 * not computed yet), row i + 1 is candidate i of the draft step's output (pool order: parents precede
 * children, siblings in rank order). */

/* O10: what the verifier's single forward needs. mask [(n+1) x (n+1)] row-major, mask[r][c] = 1 iff row c is
 * row r itself or one of its ancestors (the root is everybody's ancestor); position_ids[r] = root_position +
 * depth(r) (root depth 0); paths [n_paths x (max_depth)] = the candidate indices root -> leaf of every leaf
 * (a candidate that is nobody's parent), leaves in candidate order, padded with -1. Returns n_paths. */
int dovetail_oracle_verify_plan(const int32_t* parents, const int32_t* depths, int32_t n, int32_t root_position,
                                int32_t max_depth, uint8_t* mask, int32_t* position_ids, int32_t* paths) {
  int R = n + 1;
  memset(mask, 0, (size_t)R * R);
  position_ids[0] = root_position;
  mask[0] = 1;
  for (int i = 0; i < n; ++i) {
    int r = i + 1;
    position_ids[r] = root_position + depths[i];
    mask[(size_t)r * R + 0] = 1;
    for (int a = i; a >= 0; a = parents[a]) mask[(size_t)r * R + a + 1] = 1;
  }
  int n_paths = 0;
  for (int i = 0; i < n; ++i) {
    int is_parent = 0;
    for (int j = 0; j < n; ++j) if (parents[j] == i) is_parent = 1;
    if (is_parent) continue;
    int32_t* row = paths + (size_t)n_paths * max_depth;
    for (int k = 0; k < max_depth; ++k) row[k] = -1;
    int len = 0;
    for (int a = i; a >= 0; a = parents[a]) ++len;
    int k = len - 1;
    for (int a = i; a >= 0; a = parents[a]) row[k--] = a;
    ++n_paths;
  }
  return n_paths;
}

/* O11: the acceptance rule. Walk down from the root; at the current node try its children in candidate order.
 *   mode 0 (greedy, T = 0): child i is accepted iff token_ids[i] == tgt_argmax[row of the current node].
 *   mode 1 (speculative sampling, T = 1; reading A18): the draft tree is a deterministic top-k expansion, so each
 *          child is a point-mass proposal. Child i with target probability p_cand[i] (of its token under the
 *          target's distribution at its parent) is accepted with probability p_cand[i] / rem, where rem = 1 - the
 *          target probability of the siblings already rejected at this node, i.e. iff uniforms[i] * rem <
 *          p_cand[i] (one fp32 multiply, one fp32 compare); on rejection rem -= p_cand[i] (fp32).
 * The first accepted child becomes the current node; when no child is accepted the walk stops. accepted_path
 * receives the candidate indices root -> last accepted node, *n_acc their count.
 * The bonus token (the target's own next token after the last accepted node): mode 0: tgt_argmax of that row;
 * mode 1: drawn from the target's distribution at that row, p_full[row][*], with the tokens of the children
 * rejected there removed: weights w(x) = (uint64)(p(x) * 2^32) (exact), W = sum of the kept weights,
 * r = (uint64)((double)uniforms[n] * (double)W), bonus = the smallest x (kept) whose running sum exceeds r
 * (integer arithmetic: any summation order gives the same token); -1 if W == 0. */
int dovetail_oracle_verify_accept(const int32_t* token_ids, const int32_t* parents, int32_t n, int32_t mode,
                                  const int32_t* tgt_argmax, const float* p_cand, const float* uniforms,
                                  const float* p_full, int32_t vocab, int32_t* accepted_path, int32_t* n_acc,
                                  int32_t* bonus_token) {
  int cur = -1, na = 0;
  int32_t* rej = (int32_t*)malloc(sizeof(int32_t) * (size_t)(n > 0 ? n : 1));
  int n_rej = 0;
  for (;;) {
    float rem = 1.0f;
    int found = -1;
    n_rej = 0;
    for (int i = 0; i < n && found < 0; ++i) {
      if (parents[i] != cur) continue;
      if (mode == 0) {
        if (token_ids[i] == tgt_argmax[cur + 1]) found = i;
      } else {
        float lhs = uniforms[i] * rem;
        if (lhs < p_cand[i]) found = i;
        else { rem = rem - p_cand[i]; rej[n_rej++] = token_ids[i]; }
      }
    }
    if (found < 0) break;
    accepted_path[na++] = found;
    cur = found;
  }
  *n_acc = na;
  if (mode == 0) {
    *bonus_token = tgt_argmax[cur + 1];
  } else {
    const float* p = p_full + (size_t)(cur + 1) * vocab;
    uint64_t W = 0;
    for (int x = 0; x < vocab; ++x) {
      int r = 0;
      for (int k = 0; k < n_rej; ++k) if (rej[k] == x) r = 1;
      if (!r) W += (uint64_t)(p[x] * 4294967296.0f);
    }
    int tok = -1;
    if (W > 0) {
      uint64_t r = (uint64_t)((double)uniforms[n] * (double)W), acc = 0;
      for (int x = 0; x < vocab && tok < 0; ++x) {
        int rj = 0;
        for (int k = 0; k < n_rej; ++k) if (rej[k] == x) rj = 1;
        if (rj) continue;
        acc += (uint64_t)(p[x] * 4294967296.0f);
        if (acc > r) tok = x;
      }
    }
    *bonus_token = tok;
  }
  free(rej);
  return 0;
}
