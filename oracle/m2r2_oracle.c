/* oracle/m2r2_oracle.c — TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, single-obvious-loop-nest CPU implementation of what the M2R2 hot path
 * computes (arxiv 2502.02040; /root/reference/PAPER.md), written from the paper and from
 * the readings listed in DESIGN.md §"Readings".  It shares no code with
 * paper_2502_02040_b200/ (the CUDA path) and neither imports the other.  Only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may call it.
 *
 * Arithmetic: values are fp32 (BASELINE.json north_star: "plain, slow fp32 CPU
 * implementation"); every reduction (dot product, mean of squares, softmax sum, weighted
 * value sum) accumulates in double and is rounded to fp32 once.  Storage contract (Q20):
 * weights and the KV cache hold the config's storage dtype (fp32 or bf16, RNE); the oracle
 * reads weights as stored and rounds K/V when storing them.
 *
 * Notation follows the paper: h = slow residual, p = accelerated residual, N layers,
 * gates E_1<...<E_J, head subset S, adapter rank r, draft length gamma.
 *
 * What pins this file (tests/test_oracle_pins.py, all `-m "not gpu"`): I1 accel-off ==
 * textbook pre-norm decoder built from torch CPU ops; I2 h independent of p; I3 zero
 * adapters + all heads => p == h; I4 gate reset; I5 brute-force h_{<t} (+) p_t attention;
 * I6 incremental == recompute; I7 lossless self-spec; I8 rollback; I9 spec(0)==decode;
 * I10 closed-form acceptance under the logit script; I12 RoPE relativity; I13 softmax /
 * top-k ties; I14 MoE n_e=1 == dense; I15 LRU vs brute force; I16 AoT targets {2i+2,2i+3};
 * I18 top-2 expert mixture, I19 MoE accelerated bottleneck, I20 un-scripted expert predictor,
 * I21 LM-head adapter (numpy brute force from the traces); I22 random speculation, I23
 * previous-layer-residual speculation (PAPER.md L242 strategies 3 and 4: draws / router restated,
 * counters vs the brute-force cache simulation); I24 top-k token-subset accelerated attention
 * (L158, L170: numpy brute force, k >= t == dense, invisible non-selected positions); I25 ARLA exit
 * scores (L105-117: numpy brute force, W_v = 0 and W_q = 0 special cases).
 * PARITY UNPINNED (the paper is silent ON THE CHOICE; the arithmetic of each choice is pinned above
 * — DESIGN.md): adapter parameterisation W x + B(A x) (Q3-Q5), accelerated MLP form (Q7), LM-head
 * adapter form (Q9), gate placement for plain decode (Q15), which p feeds the expert predictor
 * (Q16), router normalisation (Q19), RoPE pairing / eps (Q1), gain init (Q22), how many experts and
 * how far ahead the two comparison strategies speculate (Q24, Q25), the granularity of the top-k
 * token selection (Q21), ARLA's states, normalisation and output map (Q26).
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#define ORC_FP32 0
#define ORC_BF16 1
#define ORC_MAX_HEADS 128
#define ORC_MAX_GATES 16
#define ORC_MAX_LAYERS 128
#define ORC_MAX_TOPK 8

typedef struct {
  int32_t n_layers, d_model, n_heads, head_dim, d_ff, vocab;
  int32_t dtype, max_seq;
  float rms_eps, rope_theta;
  int32_t accel_enabled, n_accel_heads;
  int32_t accel_heads[ORC_MAX_HEADS];
  int32_t adapter_rank, n_gates;
  int32_t gates[ORC_MAX_GATES];
  int32_t accel_end_layer, lm_head_adapter;
  int32_t n_experts, top_k, d_ff_expert, cache_slots, accel_mlp_rank, renorm_topk;
  int32_t aot_lo[ORC_MAX_LAYERS], aot_hi[ORC_MAX_LAYERS];
  int32_t accel_topk_tokens; /* p attends only the top-k cached positions of the slow stream (0 = all) */
  int32_t arla_dim;          /* latent dimension d^s of the ARLA exit router (0 = none) */
} orc_config;

/* tensor ids for orc_set_tensor (same names as m2r2_synth.KIND_ID, own numbering) */
enum {
  T_EMBED = 0, T_GF, T_LM_HEAD, T_LM_A, T_LM_B,
  T_G1, T_G2, T_WQ, T_WK, T_WV, T_WO, T_WGATE, T_WUP, T_WDOWN,
  T_AQ, T_BQ, T_AK, T_BK, T_AV, T_BV, T_AO, T_BO, T_AG, T_BG, T_AU, T_BU, T_AD, T_BD,
  T_ROUTER, T_UG, T_UU, T_UD, T_EWG, T_EWU, T_EWD, T_ARLA, T_COUNT
};

typedef struct {
  const void* t[T_COUNT];
  const void** ewg; /* [n_experts] */
  const void** ewu;
  const void** ewd;
} orc_layer;

typedef struct {
  int64_t steps, drafted, accepted, emitted;
  int64_t expert_hits, expert_misses, prefetched, on_demand;
} orc_stats;

typedef struct orc {
  orc_config c;
  const void* g[T_COUNT]; /* global tensors */
  orc_layer* L;
  /* sequence state */
  float* K; /* [N][max_seq][d]  (position-major, heads contiguous inside d) */
  float* V;
  int32_t kv_len, pending, have_pending;
  /* scripts (borrowed copies) */
  int32_t *ls_full, *ls_draft, ls_first, ls_n;
  float ls_beta;
  int32_t *rs_actual, *rs_pred, rs_first, rs_n;
  float rs_beta;
  /* MoE logical cache model: lru[L][0] = most recent ... lru[L][C-1] = least recent */
  int32_t* lru;
  int32_t policy;
  orc_stats st;
  /* traces of the last decode_step (or last verify row) */
  float* trH;        /* [(N+1)][d]: h_0 .. h_N */
  float* slow_q;     /* [d]: rotated slow query of the last single-row slow_layer call */
  float topk_margin; /* smallest gap between the k-th and (k+1)-th slow score of any top-k selection of the last step */
  float* trP;        /* [(N+1)][d]: p_0 .. ; p_{i+1} is the value BEFORE a gate reset */
  float* logits;     /* [V] final-head logits, before script bias */
  float* exit_logits;/* [J][V] accelerated-stream exit logits at each gate, before bias */
  float exit_score[ORC_MAX_GATES]; /* ARLA exit scores of the last decode_step */
  float last_margin; /* top-2 margin of the last final argmax (after bias) */
  float last_draft_margin;
  float step_min_margin; /* introspection: smallest top-2 margin of any argmax (draft or verify) of the last spec_step / decode_step */
  int32_t* route_idx;  /* [N][top_k] routed experts of the last slow token */
  float* route_w;      /* [N][top_k] */
  int32_t* pred_idx;   /* [N][top_k] predicted experts per TARGET layer (-1: none) */
} orc;

/* ------------------------------------------------------------------ storage helpers */
static inline float bf16_to_f32(uint16_t b) {
  uint32_t u = (uint32_t)b << 16;
  float f;
  memcpy(&f, &u, 4);
  return f;
}
static inline float round_to_bf16(float f) {
  uint32_t u;
  memcpy(&u, &f, 4);
  if ((u & 0x7F800000u) != 0x7F800000u) u += 0x7FFFu + ((u >> 16) & 1u);
  u &= 0xFFFF0000u;
  memcpy(&f, &u, 4);
  return f;
}
static inline float round_store(const orc* o, float f) {
  return o->c.dtype == ORC_BF16 ? round_to_bf16(f) : f;
}
/* element i of a stored tensor, widened to fp32 (exact) */
static inline float wld(const orc* o, const void* W, size_t i) {
  return o->c.dtype == ORC_BF16 ? bf16_to_f32(((const uint16_t*)W)[i]) : ((const float*)W)[i];
}

/* dot(W[row, 0:K], x) with row stride ld, column offset col0 — double accumulation */
static double dot_row(const orc* o, const void* W, size_t row, size_t ld, size_t col0, size_t K,
                      const float* x) {
  double a0 = 0, a1 = 0, a2 = 0, a3 = 0;
  size_t k = 0;
  if (o->c.dtype == ORC_BF16) {
    const uint16_t* w = (const uint16_t*)W + row * ld + col0;
    for (; k + 4 <= K; k += 4) {
      a0 += (double)bf16_to_f32(w[k]) * x[k];
      a1 += (double)bf16_to_f32(w[k + 1]) * x[k + 1];
      a2 += (double)bf16_to_f32(w[k + 2]) * x[k + 2];
      a3 += (double)bf16_to_f32(w[k + 3]) * x[k + 3];
    }
    for (; k < K; ++k) a0 += (double)bf16_to_f32(w[k]) * x[k];
  } else {
    const float* w = (const float*)W + row * ld + col0;
    for (; k + 4 <= K; k += 4) {
      a0 += (double)w[k] * x[k];
      a1 += (double)w[k + 1] * x[k + 1];
      a2 += (double)w[k + 2] * x[k + 2];
      a3 += (double)w[k + 3] * x[k + 3];
    }
    for (; k < K; ++k) a0 += (double)w[k] * x[k];
  }
  return (a0 + a1) + (a2 + a3);
}

/* Y[t][n] = sum_k W[row0+n][k] X[t][k]   for t < m, n < n_out  (W row-major [.., K]) */
static void matmul_rows(const orc* o, const void* W, size_t row0, size_t n_out, size_t K,
                        const float* X, size_t ldx, int m, float* Y, size_t ldy) {
#pragma omp parallel for schedule(static)
  for (int64_t n = 0; n < (int64_t)n_out; ++n)
    for (int t = 0; t < m; ++t)
      Y[(size_t)t * ldy + n] = (float)dot_row(o, W, row0 + (size_t)n, K, 0, K, X + (size_t)t * ldx);
}

/* rms(x; g) = x * g / sqrt(mean(x^2) + eps)      (Q1; PAPER.md L60 says norms are applied) */
static void rmsnorm(const orc* o, const float* x, const void* g, float* y) {
  int d = o->c.d_model;
  double ss = 0;
  for (int j = 0; j < d; ++j) ss += (double)x[j] * x[j];
  double inv = 1.0 / sqrt(ss / d + (double)o->c.rms_eps);
  for (int j = 0; j < d; ++j) y[j] = (float)((double)x[j] * inv * (double)wld(o, g, j));
}

/* rope(v, t): rotate pairs (v[j], v[j + d_h/2]) by angle t * theta^(-2j/d_h)   (Q1) */
static void rope(const orc* o, float* v, int t) {
  int dh = o->c.head_dim, half = dh / 2;
  for (int j = 0; j < half; ++j) {
    double ang = (double)t * pow((double)o->c.rope_theta, -2.0 * j / dh);
    double cs = cos(ang), sn = sin(ang);
    double a = v[j], b = v[j + half];
    v[j] = (float)(a * cs - b * sn);
    v[j + half] = (float)(b * cs + a * sn);
  }
}

static inline float silu(float z) { return (float)((double)z / (1.0 + exp(-(double)z))); }

/* argmax, lowest index wins ties; also returns the top-2 margin */
static int argmax_margin(const float* v, int n, float* margin) {
  int best = 0;
  for (int i = 1; i < n; ++i)
    if (v[i] > v[best]) best = i;
  if (margin) {
    float second = -INFINITY;
    for (int i = 0; i < n; ++i)
      if (i != best && v[i] > second) second = v[i];
    *margin = v[best] - second;
  }
  return best;
}

/* y[n] += B[n, :] . (A x)   — rank-r parallel adapter, W x + B(A x)   (Q3) */
static void lora_add(const orc* o, const void* A, const void* B, int r, size_t K, size_t n_out,
                     const float* x, float* y) {
  float u[64];
  for (int j = 0; j < r; ++j) u[j] = (float)dot_row(o, A, (size_t)j, K, 0, K, x);
  for (size_t n = 0; n < n_out; ++n) y[n] += (float)dot_row(o, B, n, (size_t)r, 0, (size_t)r, u);
}

static int gate_index(const orc* o, int layer_out) { /* j with gates[j] == layer_out, else -1 */
  for (int j = 0; j < o->c.n_gates; ++j)
    if (o->c.gates[j] == layer_out) return j;
  return -1;
}

/* ------------------------------------------------------------------ MoE cache model */
static int lru_find(const orc* o, int L, int e) {
  for (int s = 0; s < o->c.cache_slots; ++s)
    if (o->lru[L * o->c.cache_slots + s] == e) return s;
  return -1;
}
static void lru_touch(orc* o, int L, int pos) { /* move entry at pos to front */
  int32_t* q = o->lru + L * o->c.cache_slots;
  int32_t e = q[pos];
  for (int s = pos; s > 0; --s) q[s] = q[s - 1];
  q[0] = e;
}
/* make `e` resident in cache[L]; never evict a member of keep[0..nk). returns 1 if loaded */
static int lru_insert(orc* o, int L, int e, const int32_t* keep, int nk) {
  int C = o->c.cache_slots;
  int32_t* q = o->lru + L * C;
  int pos = lru_find(o, L, e);
  if (pos >= 0) {
    lru_touch(o, L, pos);
    return 0;
  }
  /* victim = least-recent entry not in keep (empty slots, -1, go first) */
  int victim = -1;
  for (int s = C - 1; s >= 0 && victim < 0; --s)
    if (q[s] < 0) victim = s;
  for (int s = C - 1; s >= 0 && victim < 0; --s) {
    int kept = 0;
    for (int k = 0; k < nk; ++k)
      if (keep[k] == q[s]) kept = 1;
    if (!kept) victim = s;
  }
  if (victim < 0) victim = C - 1;
  q[victim] = e;
  lru_touch(o, L, victim);
  return 1;
}

/* policy 0: fixed residency (experts 0..C-1 stay; others are loaded on demand every time).
 * policy 1: LRU.  policy 2: LRU + ahead-of-time speculation from the accelerated residual.  policy 3: LRU + random
 * speculation.  policy 4: LRU + speculation from the previous layer's (slow) residual.  (the five strategies) */
static void moe_use_event(orc* o, int L, const int32_t* idx) {
  for (int k = 0; k < o->c.top_k; ++k) {
    if (o->policy == 0) {
      if (idx[k] < o->c.cache_slots) o->st.expert_hits++;
      else { o->st.expert_misses++; o->st.on_demand++; }
    } else {
      if (lru_find(o, L, idx[k]) >= 0) { o->st.expert_hits++; lru_insert(o, L, idx[k], idx, o->c.top_k); }
      else { o->st.expert_misses++; o->st.on_demand++; lru_insert(o, L, idx[k], idx, o->c.top_k); }
    }
  }
}
static void moe_predict_event(orc* o, int L, const int32_t* idx) {
  if (o->policy < 2) return;
  for (int k = 0; k < o->c.top_k; ++k)
    if (lru_insert(o, L, idx[k], idx, o->c.top_k)) o->st.prefetched++;
}
/* counter-based generator of the random-speculation policy (the CUDA side implements the same function) */
static uint64_t spec_mix(uint64_t counter) {
  uint64_t x = 0x5EC0DE5EEDull + 0x9E3779B97F4A7C15ull * (counter + 1);
  x = (x ^ (x >> 30)) * 0xBF58476D1CE4E5B9ull;
  x = (x ^ (x >> 27)) * 0x94D049BB133111EBull;
  return x ^ (x >> 31);
}
/* policy 3 (third strategy: "LRU ... adding speculative caching and randomly pre-loading experts"):
 * before layer Lt is reached, top_k distinct experts drawn uniformly are pre-loaded into its cache.  DESIGN.md Q24:
 * one layer ahead, top_k experts, draw d of (position t, layer Lt) = spec_mix((t * N + Lt) * 256 + d) mod n_experts,
 * duplicates skipped. */
static void random_speculation(orc* o, int Lt, int t) {
  const orc_config* c = &o->c;
  int32_t idx[ORC_MAX_TOPK];
  int n = 0;
  for (int dr = 0; n < c->top_k && dr < 256; ++dr) {
    int e = (int)(spec_mix(((uint64_t)t * (uint64_t)c->n_layers + (uint64_t)Lt) * 256u + (uint64_t)dr) % (uint64_t)c->n_experts);
    int dup = 0;
    for (int k = 0; k < n; ++k) dup |= idx[k] == e;
    if (!dup) idx[n++] = e;
  }
  for (int k = 0; k < c->top_k; ++k) o->pred_idx[Lt * c->top_k + k] = idx[k];
  moe_predict_event(o, Lt, idx);
}

/* router: softmax over all experts, top-k (lower index wins ties), renormalise (Q19) */
static void route(const orc* o, const void* Wr, const float* y, const int32_t* script_pair,
                  float beta, int32_t* idx, float* w) {
  int ne = o->c.n_experts, tk = o->c.top_k;
  float l[256] = {0};
  double pr[256];
  for (int e = 0; e < ne; ++e) l[e] = (float)dot_row(o, Wr, (size_t)e, o->c.d_model, 0, o->c.d_model, y);
  if (script_pair) { /* +beta on e1, +beta-8 on e2 (router script, DESIGN.md §Input recipe) */
    l[script_pair[0]] += beta;
    l[script_pair[1]] += beta - 8.0f;
  }
  float mx = l[0];
  for (int e = 1; e < ne; ++e) if (l[e] > mx) mx = l[e];
  double sum = 0;
  for (int e = 0; e < ne; ++e) { pr[e] = exp((double)(l[e] - mx)); sum += pr[e]; }
  for (int e = 0; e < ne; ++e) pr[e] /= sum;
  double wsum = 0;
  for (int k = 0; k < tk; ++k) {
    int best = -1;
    for (int e = 0; e < ne; ++e) {
      int taken = 0;
      for (int q = 0; q < k; ++q) if (idx[q] == e) taken = 1;
      if (taken) continue;
      if (best < 0 || l[e] > l[best]) best = e;
    }
    idx[k] = best;
    wsum += pr[best];
  }
  for (int k = 0; k < tk; ++k) w[k] = (float)(o->c.renorm_topk ? pr[idx[k]] / wsum : pr[idx[k]]);
}

/* ------------------------------------------------------------------ slow layer (Eq. 1) */
/* m tokens at positions t0..t0+m-1, residuals H[m][d] updated in place.
 * use_events: count MoE cache events (off during prefill). */
static void slow_layer(orc* o, int i, float* H, int m, int t0, int use_events) {
  const orc_config* c = &o->c;
  const orc_layer* L = &o->L[i];
  int d = c->d_model, nh = c->n_heads, dh = c->head_dim;
  float* X = (float*)malloc(sizeof(float) * (size_t)m * d);
  float* Q = (float*)malloc(sizeof(float) * (size_t)m * d);
  float* Kn = (float*)malloc(sizeof(float) * (size_t)m * d);
  float* Vn = (float*)malloc(sizeof(float) * (size_t)m * d);
  float* O = (float*)malloc(sizeof(float) * (size_t)m * d);
  float* Y = (float*)malloc(sizeof(float) * (size_t)m * d);
  /* 1. x = rms(h; g1); q,k,v = W x */
  for (int t = 0; t < m; ++t) rmsnorm(o, H + (size_t)t * d, L->t[T_G1], X + (size_t)t * d);
  matmul_rows(o, L->t[T_WQ], 0, d, d, X, d, m, Q, d);
  matmul_rows(o, L->t[T_WK], 0, d, d, X, d, m, Kn, d);
  matmul_rows(o, L->t[T_WV], 0, d, d, X, d, m, Vn, d);
  /* 2. rope(q), rope(k) per head at position t; store K[t], V[t] rounded to the cache dtype */
  float* Kc = o->K + (size_t)i * c->max_seq * d;
  float* Vc = o->V + (size_t)i * c->max_seq * d;
  for (int t = 0; t < m; ++t)
    for (int a = 0; a < nh; ++a) {
      rope(o, Q + (size_t)t * d + a * dh, t0 + t);
      rope(o, Kn + (size_t)t * d + a * dh, t0 + t);
    }
  for (int t = 0; t < m; ++t)
    for (int j = 0; j < d; ++j) {
      Kc[(size_t)(t0 + t) * d + j] = round_store(o, Kn[(size_t)t * d + j]);
      Vc[(size_t)(t0 + t) * d + j] = round_store(o, Vn[(size_t)t * d + j]);
    }
  /* 3. per head: s_u = q.K[u]/sqrt(d_h), u = 0..t; softmax; o = sum_u pi_u V[u] */
  double scale = 1.0 / sqrt((double)dh);
#pragma omp parallel for collapse(2) schedule(static)
  for (int t = 0; t < m; ++t)
    for (int a = 0; a < nh; ++a) {
      int T1 = t0 + t + 1;
      float* s = (float*)malloc(sizeof(float) * (size_t)T1);
      const float* q = Q + (size_t)t * d + a * dh;
      for (int u = 0; u < T1; ++u) {
        double acc = 0;
        const float* kk = Kc + (size_t)u * d + a * dh;
        for (int j = 0; j < dh; ++j) acc += (double)q[j] * kk[j];
        s[u] = (float)(acc * scale);
      }
      float mx = s[0];
      for (int u = 1; u < T1; ++u) if (s[u] > mx) mx = s[u];
      double* e = (double*)malloc(sizeof(double) * (size_t)T1);
      double sum = 0;
      for (int u = 0; u < T1; ++u) { e[u] = exp((double)(s[u] - mx)); sum += e[u]; }
      for (int j = 0; j < dh; ++j) {
        double acc = 0;
        for (int u = 0; u < T1; ++u) acc += e[u] * Vc[(size_t)u * d + a * dh + j];
        O[(size_t)t * d + a * dh + j] = (float)(acc / sum);
      }
      free(e);
      free(s);
    }
  /* 4. h' = h + W_o o */
  matmul_rows(o, L->t[T_WO], 0, d, d, O, d, m, Y, d);
  for (size_t j = 0; j < (size_t)m * d; ++j) H[j] += Y[j];
  /* 5. y = rms(h'; g2); h_{i+1} = h' + MLP(y) */
  for (int t = 0; t < m; ++t) rmsnorm(o, H + (size_t)t * d, L->t[T_G2], X + (size_t)t * d);
  if (c->n_experts == 0) {
    int F = c->d_ff;
    float* G = (float*)malloc(sizeof(float) * (size_t)m * F);
    float* U = (float*)malloc(sizeof(float) * (size_t)m * F);
    matmul_rows(o, L->t[T_WGATE], 0, F, d, X, d, m, G, F);
    matmul_rows(o, L->t[T_WUP], 0, F, d, X, d, m, U, F);
    for (size_t j = 0; j < (size_t)m * F; ++j) G[j] = silu(G[j]) * U[j];
    matmul_rows(o, L->t[T_WDOWN], 0, d, F, G, F, m, Y, d);
    for (size_t j = 0; j < (size_t)m * d; ++j) H[j] += Y[j];
    free(G);
    free(U);
  } else {
    int F = c->d_ff_expert, tk = c->top_k;
    float* G = (float*)malloc(sizeof(float) * F);
    float* U = (float*)malloc(sizeof(float) * F);
    float* Z = (float*)malloc(sizeof(float) * d);
    for (int t = 0; t < m; ++t) {
      int32_t idx[ORC_MAX_TOPK];
      float w[ORC_MAX_TOPK];
      const int32_t* sp = NULL;
      int pos = t0 + t;
      if (o->rs_actual && pos >= o->rs_first && pos < o->rs_first + o->rs_n)
        sp = o->rs_actual + ((size_t)(pos - o->rs_first) * c->n_layers + i) * 2;
      const float* y = X + (size_t)t * d;
      route(o, L->t[T_ROUTER], y, sp, o->rs_beta, idx, w);
      if (use_events) moe_use_event(o, i, idx);
      for (int k = 0; k < tk; ++k) { o->route_idx[i * tk + k] = idx[k]; o->route_w[i * tk + k] = w[k]; }
      /* m = sum_e w_e * W_d^e (silu(W_g^e y) * (W_u^e y)), e in selection order */
      float* Hh = H + (size_t)t * d;
      float* acc = (float*)calloc(d, sizeof(float));
      for (int k = 0; k < tk; ++k) {
        int e = idx[k];
        matmul_rows(o, L->ewg[e], 0, F, d, y, d, 1, G, F);
        matmul_rows(o, L->ewu[e], 0, F, d, y, d, 1, U, F);
        for (int j = 0; j < F; ++j) G[j] = silu(G[j]) * U[j];
        matmul_rows(o, L->ewd[e], 0, d, F, G, F, 1, Z, d);
        for (int j = 0; j < d; ++j) acc[j] += w[k] * Z[j];
      }
      for (int j = 0; j < d; ++j) Hh[j] += acc[j];
      free(acc);
    }
    free(G);
    free(U);
    free(Z);
  }
  if (m == 1 && o->slow_q) memcpy(o->slow_q, Q, sizeof(float) * d); /* rotated slow query of this token (top-k token selection of the accelerated stream) */
  free(X); free(Q); free(Kn); free(Vn); free(O); free(Y);
}

/* ------------------------------------------------------------------ accelerated layer (Eq. 2) */
/* One token at position t.  p updated in place.  Must be called AFTER slow_layer(i) of the
 * same token: it reads K_i[0..t-1], V_i[0..t-1] only (never position t — PAPER.md L76). */
static void accel_layer(orc* o, int i, float* p, int t) {
  const orc_config* c = &o->c;
  const orc_layer* L = &o->L[i];
  int d = c->d_model, dh = c->head_dim, ns = c->n_accel_heads, r = c->adapter_rank;
  int da = ns * dh;
  float* x = (float*)malloc(sizeof(float) * d);
  float* q = (float*)malloc(sizeof(float) * da);
  float* k = (float*)malloc(sizeof(float) * da);
  float* v = (float*)malloc(sizeof(float) * da);
  float* oh = (float*)malloc(sizeof(float) * da);
  float* y = (float*)malloc(sizeof(float) * d);
  /* 1. x^ = rms(p; g1)  (gain shared with the slow stream, Q8) */
  rmsnorm(o, p, L->t[T_G1], x);
  /* 2. q^ = W_q[S] x^ + B_q(A_q x^), likewise k^, v^; rope; NOT stored (no accel cache, L74) */
  for (int s = 0; s < ns; ++s) {
    size_t row0 = (size_t)c->accel_heads[s] * dh;
    matmul_rows(o, L->t[T_WQ], row0, dh, d, x, d, 1, q + s * dh, dh);
    matmul_rows(o, L->t[T_WK], row0, dh, d, x, d, 1, k + s * dh, dh);
    matmul_rows(o, L->t[T_WV], row0, dh, d, x, d, 1, v + s * dh, dh);
  }
  lora_add(o, L->t[T_AQ], L->t[T_BQ], r, d, da, x, q);
  lora_add(o, L->t[T_AK], L->t[T_BK], r, d, da, x, k);
  lora_add(o, L->t[T_AV], L->t[T_BV], r, d, da, x, v);
  for (int s = 0; s < ns; ++s) { rope(o, q + s * dh, t); rope(o, k + s * dh, t); }
  /* 3. MHA(p_t, h_{<t} (+) p_t, h_{<t} (+) p_t): t cached slow positions + own k^, v^ */
  const float* Kc = o->K + (size_t)i * c->max_seq * d;
  const float* Vc = o->V + (size_t)i * c->max_seq * d;
  double scale = 1.0 / sqrt((double)dh);
  float* sc = (float*)malloc(sizeof(float) * (size_t)(t + 1));
  double* ex = (double*)malloc(sizeof(double) * (size_t)(t + 1));
  const int topk = c->accel_topk_tokens;
  float* ssc = (float*)malloc(sizeof(float) * (size_t)(t + 1));   /* slow scores (selection) */
  char* keep = (char*)malloc((size_t)(t + 1));
  for (int s = 0; s < ns; ++s) {
    int a = c->accel_heads[s];
    /* Attention FLOPs optimisation (footnote 4 L170; Q21): per head, the accelerated stream
     * attends only the `topk` cached positions with the largest attention coefficients of the SLOW stream (same head,
     * same token; softmax is monotone, so: the largest scores q_h . K_h[u]; ties: lower position first) plus its own
     * k^_t, and assigns its own coefficients to them. */
    for (int u = 0; u <= t; ++u) keep[u] = 1;
    if (topk > 0 && t > topk) {
      for (int u = 0; u < t; ++u) {
        double acc = 0;
        for (int j = 0; j < dh; ++j) acc += (double)o->slow_q[a * dh + j] * Kc[(size_t)u * d + a * dh + j];
        ssc[u] = (float)(acc * scale);
        keep[u] = 0;
      }
      float last = 0.f;
      for (int r2 = 0; r2 < topk; ++r2) {
        int best = -1;
        for (int u = 0; u < t; ++u)
          if (!keep[u] && (best < 0 || ssc[u] > ssc[best])) best = u;
        keep[best] = 1;
        last = ssc[best];
      }
      float next = -INFINITY;
      for (int u = 0; u < t; ++u)
        if (!keep[u] && ssc[u] > next) next = ssc[u];
      if (last - next < o->topk_margin) o->topk_margin = last - next;
    }
    for (int u = 0; u < t; ++u) {
      double acc = 0;
      for (int j = 0; j < dh; ++j) acc += (double)q[s * dh + j] * Kc[(size_t)u * d + a * dh + j];
      sc[u] = (float)(acc * scale);
    }
    {
      double acc = 0;
      for (int j = 0; j < dh; ++j) acc += (double)q[s * dh + j] * k[s * dh + j];
      sc[t] = (float)(acc * scale);
    }
    float mx = sc[t];
    for (int u = 0; u < t; ++u) if (keep[u] && sc[u] > mx) mx = sc[u];
    double sum = 0;
    for (int u = 0; u <= t; ++u) { ex[u] = keep[u] ? exp((double)(sc[u] - mx)) : 0.0; sum += ex[u]; }
    for (int j = 0; j < dh; ++j) {
      double acc = 0;
      for (int u = 0; u < t; ++u) acc += ex[u] * Vc[(size_t)u * d + a * dh + j];
      acc += ex[t] * v[s * dh + j];
      oh[s * dh + j] = (float)(acc / sum);
    }
  }
  free(sc);
  free(ex);
  free(ssc);
  free(keep);
  /* 4. p' = p + W_o[:, S] o^ + B_o(A_o o^) */
  for (int n = 0; n < d; ++n) {
    double acc = 0;
    for (int s = 0; s < ns; ++s)
      acc += dot_row(o, L->t[T_WO], (size_t)n, d, (size_t)c->accel_heads[s] * dh, dh, oh + s * dh);
    y[n] = (float)acc;
  }
  lora_add(o, L->t[T_AO], L->t[T_BO], r, da, d, oh, y);
  for (int n = 0; n < d; ++n) p[n] += y[n];
  /* 5. y^ = rms(p'; g2); p_{i+1} = p' + M^(y^) */
  rmsnorm(o, p, L->t[T_G2], x);
  if (c->n_experts == 0) {
    /* dense: base SwiGLU + adapter deltas on gate, up, down (Q7) */
    int F = c->d_ff;
    float* G = (float*)malloc(sizeof(float) * F);
    float* U = (float*)malloc(sizeof(float) * F);
    matmul_rows(o, L->t[T_WGATE], 0, F, d, x, d, 1, G, F);
    matmul_rows(o, L->t[T_WUP], 0, F, d, x, d, 1, U, F);
    lora_add(o, L->t[T_AG], L->t[T_BG], r, d, F, x, G);
    lora_add(o, L->t[T_AU], L->t[T_BU], r, d, F, x, U);
    for (int j = 0; j < F; ++j) G[j] = silu(G[j]) * U[j];
    matmul_rows(o, L->t[T_WDOWN], 0, d, F, G, F, 1, y, d);
    lora_add(o, L->t[T_AD], L->t[T_BD], r, F, d, G, y);
    free(G);
    free(U);
  } else {
    /* MoE: fixed adapter-only bottleneck m^ = U_d (silu(U_g y^) * (U_u y^))  (L137; Q7) */
    int rm = c->accel_mlp_rank;
    float* G = (float*)malloc(sizeof(float) * rm);
    float* U = (float*)malloc(sizeof(float) * rm);
    matmul_rows(o, L->t[T_UG], 0, rm, d, x, d, 1, G, rm);
    matmul_rows(o, L->t[T_UU], 0, rm, d, x, d, 1, U, rm);
    for (int j = 0; j < rm; ++j) G[j] = silu(G[j]) * U[j];
    matmul_rows(o, L->t[T_UD], 0, d, rm, G, rm, 1, y, d);
    free(G);
    free(U);
  }
  for (int n = 0; n < d; ++n) p[n] += y[n];
  free(x); free(q); free(k); free(v); free(oh); free(y);
}

/* logits = W_lm rms(z; g_f)  [+ B_lm(A_lm rms(z))  for the accelerated exit head, Q9] */
static void head_logits(const orc* o, const float* z, int accel_head, float* logits) {
  int d = o->c.d_model, V = o->c.vocab;
  float* x = (float*)malloc(sizeof(float) * d);
  rmsnorm(o, z, o->g[T_GF], x);
  matmul_rows(o, o->g[T_LM_HEAD], 0, V, d, x, d, 1, logits, V);
  if (accel_head && o->c.lm_head_adapter)
    lora_add(o, o->g[T_LM_A], o->g[T_LM_B], o->c.adapter_rank, d, V, x, logits);
  free(x);
}

/* greedy token for the position `s` being predicted, with the script bias */
static int pick_token(const orc* o, const float* logits, int s, int draft, float* margin) {
  int V = o->c.vocab;
  const int32_t* tab = draft ? o->ls_draft : o->ls_full;
  if (tab && s >= o->ls_first && s < o->ls_first + o->ls_n) {
    float* tmp = (float*)malloc(sizeof(float) * V);
    memcpy(tmp, logits, sizeof(float) * V);
    tmp[tab[s - o->ls_first]] += o->ls_beta;
    int r = argmax_margin(tmp, V, margin);
    free(tmp);
    return r;
  }
  return argmax_margin(logits, V, margin);
}

/* expert predictor (A14): routers of the target layers applied to rms(p_{i+1}; g2_{L'}) */
static void predict_experts(orc* o, int src_layer, const float* p, int t) {
  const orc_config* c = &o->c;
  if (c->n_experts == 0) return;
  int d = c->d_model;
  float* y = (float*)malloc(sizeof(float) * d);
  for (int Lt = c->aot_lo[src_layer]; Lt < c->aot_hi[src_layer]; ++Lt) {
    int32_t idx[ORC_MAX_TOPK];
    float w[ORC_MAX_TOPK];
    const int32_t* sp = NULL;
    if (o->rs_pred && t >= o->rs_first && t < o->rs_first + o->rs_n)
      sp = o->rs_pred + ((size_t)(t - o->rs_first) * c->n_layers + Lt) * 2;
    rmsnorm(o, p, o->L[Lt].t[T_G2], y);
    route(o, o->L[Lt].t[T_ROUTER], y, sp, o->rs_beta, idx, w);
    for (int k = 0; k < c->top_k; ++k) o->pred_idx[Lt * c->top_k + k] = idx[k];
    if (o->policy == 2) moe_predict_event(o, Lt, idx);
  }
  free(y);
}

/* policy 4 (fourth strategy: "speculative loading based on residual states from the previous layer";
 * L244: started "only one layer before the current layer"): the router of layer Lt = i + 1 applied to the SLOW residual
 * entering that layer, rms(h_{i+1}; g2_{Lt}) (Q25). */
static void prev_layer_speculation(orc* o, int Lt, const float* h, int t) {
  const orc_config* c = &o->c;
  int d = c->d_model;
  float* y = (float*)malloc(sizeof(float) * d);
  int32_t idx[ORC_MAX_TOPK];
  float w[ORC_MAX_TOPK];
  const int32_t* sp = NULL;
  if (o->rs_pred && t >= o->rs_first && t < o->rs_first + o->rs_n)
    sp = o->rs_pred + ((size_t)(t - o->rs_first) * c->n_layers + Lt) * 2;
  rmsnorm(o, h, o->L[Lt].t[T_G2], y);
  route(o, o->L[Lt].t[T_ROUTER], y, sp, o->rs_beta, idx, w);
  for (int k = 0; k < c->top_k; ++k) o->pred_idx[Lt * c->top_k + k] = idx[k];
  moe_predict_event(o, Lt, idx);
  free(y);
}

/* One token through layers [0, n_run): slow stream always, accelerated stream if `accel`.
 * Writes slow K/V at position t.  exit_tokens[j] filled for gates passed (may be NULL).
 * On return h (and p) hold the residuals leaving layer n_run-1. */
static void dual_token(orc* o, int token, int t, int n_run, int accel, float* h, float* p,
                       int32_t* exit_tokens, int trace) {
  const orc_config* c = &o->c;
  int d = c->d_model;
  for (int j = 0; j < d; ++j) h[j] = wld(o, o->g[T_EMBED], (size_t)token * d + j);
  memcpy(p, h, sizeof(float) * d); /* p_0 <- h_0 */
  if (trace) {
    memcpy(o->trH, h, sizeof(float) * d);
    memcpy(o->trP, p, sizeof(float) * d);
    for (int k = 0; k < c->n_layers * c->top_k; ++k) o->pred_idx[k] = -1;
  }
  for (int i = 0; i < n_run; ++i) {
    int acc_on = accel && c->accel_enabled && i < c->accel_end_layer;
    slow_layer(o, i, h, 1, t, 1);
    if (c->n_experts && i + 1 < c->n_layers) {
      if (o->policy == 3) random_speculation(o, i + 1, t);
      if (o->policy == 4) prev_layer_speculation(o, i + 1, h, t);
    }
    if (acc_on) {
      accel_layer(o, i, p, t);
      if (c->n_experts && o->policy <= 2) predict_experts(o, i, p, t);   /* acts on the cache under policy 2 only */
    }
    if (trace) {
      memcpy(o->trH + (size_t)(i + 1) * d, h, sizeof(float) * d);
      memcpy(o->trP + (size_t)(i + 1) * d, acc_on ? p : h, sizeof(float) * d);
    }
    int gj = gate_index(o, i + 1);
    if (acc_on && gj >= 0) {
      /* exit prediction at the gate (Eq. 4), then p <- h (L82, L101) */
      float* el = o->exit_logits + (size_t)gj * c->vocab;
      head_logits(o, p, 1, el);
      float mg;
      int tok = pick_token(o, el, t + 1, 1, &mg);
      o->last_draft_margin = mg;
      if (exit_tokens) exit_tokens[gj] = tok;
      memcpy(p, h, sizeof(float) * d);
    }
  }
}

/* Accelerated Residual Latent Attention (Fig. 4a; Q26): the exit decision at gate E_j looks at
 * the accelerated residuals of the whole interval, z_i for i = E_{j-1} .. E_j (z at the interval's start = the slow residual p
 * was re-initialised from, L82; z_{E_j} = p before the reset).  The states are projected into a latent space of dimension d^s
 * (footnote 2: 64), Q^s = W_q z, K^s = W_k z, V^s = W_v z; the query of the state AT the gate attends the keys of all states
 * of the interval; the exit score is sigma(w_o . (softmax(q K^T / sqrt(d^s)) V) + b).  Mechanics only: the score is reported,
 * no layer is skipped (the paper does not say how skipped layers' K/V are filled, L248). */
static void arla_scores(orc* o) {
  const orc_config* c = &o->c;
  const int ds = c->arla_dim, d = c->d_model;
  if (ds <= 0 || !o->g[T_ARLA]) return;
  for (int j = 0; j < c->n_gates; ++j) {
    const int lo = j ? c->gates[j - 1] : 0, hi = c->gates[j], n = hi - lo + 1;
    const size_t r0 = (size_t)j * (3 * ds + 1);
    float* q = (float*)malloc(sizeof(float) * ds);
    float* K = (float*)malloc(sizeof(float) * (size_t)n * ds);
    float* V = (float*)malloc(sizeof(float) * (size_t)n * ds);
    for (int s = 0; s < n; ++s) {
      const int i = lo + s;
      const float* z = (s == 0) ? o->trH + (size_t)i * d : o->trP + (size_t)i * d;
      for (int e = 0; e < ds; ++e) {
        K[(size_t)s * ds + e] = (float)dot_row(o, o->g[T_ARLA], r0 + ds + e, (size_t)d, 0, (size_t)d, z);
        V[(size_t)s * ds + e] = (float)dot_row(o, o->g[T_ARLA], r0 + 2 * ds + e, (size_t)d, 0, (size_t)d, z);
        if (s == n - 1) q[e] = (float)dot_row(o, o->g[T_ARLA], r0 + e, (size_t)d, 0, (size_t)d, z);
      }
    }
    double sc[ORC_MAX_LAYERS + 1], mx = -INFINITY, sum = 0;
    for (int s = 0; s < n; ++s) {
      double acc = 0;
      for (int e = 0; e < ds; ++e) acc += (double)q[e] * K[(size_t)s * ds + e];
      sc[s] = acc / sqrt((double)ds);
      if (sc[s] > mx) mx = sc[s];
    }
    for (int s = 0; s < n; ++s) { sc[s] = exp(sc[s] - mx); sum += sc[s]; }
    double logit = wld(o, o->g[T_ARLA], (r0 + 3 * ds) * (size_t)d + ds); /* bias */
    for (int e = 0; e < ds; ++e) {
      double ce = 0;
      for (int s = 0; s < n; ++s) ce += sc[s] / sum * V[(size_t)s * ds + e];
      logit += (double)wld(o, o->g[T_ARLA], (r0 + 3 * ds) * (size_t)d + e) * (float)ce;
    }
    o->exit_score[j] = (float)(1.0 / (1.0 + exp(-logit)));
    free(q); free(K); free(V);
  }
}

/* ------------------------------------------------------------------ public API */
orc* orc_create(const orc_config* cfg) {
  orc* o = (orc*)calloc(1, sizeof(orc));
  o->c = *cfg;
  const orc_config* c = &o->c;
  int N = c->n_layers, d = c->d_model;
  o->L = (orc_layer*)calloc((size_t)N, sizeof(orc_layer));
  for (int i = 0; i < N; ++i)
    if (c->n_experts) {
      o->L[i].ewg = (const void**)calloc((size_t)c->n_experts, sizeof(void*));
      o->L[i].ewu = (const void**)calloc((size_t)c->n_experts, sizeof(void*));
      o->L[i].ewd = (const void**)calloc((size_t)c->n_experts, sizeof(void*));
    }
  o->K = (float*)calloc((size_t)N * c->max_seq * d, sizeof(float));
  o->V = (float*)calloc((size_t)N * c->max_seq * d, sizeof(float));
  o->trH = (float*)calloc((size_t)(N + 1) * d, sizeof(float));
  o->slow_q = (float*)calloc((size_t)d, sizeof(float));
  o->trP = (float*)calloc((size_t)(N + 1) * d, sizeof(float));
  o->logits = (float*)calloc((size_t)c->vocab, sizeof(float));
  o->exit_logits = (float*)calloc((size_t)(c->n_gates > 0 ? c->n_gates : 1) * c->vocab, sizeof(float));
  int tk = c->top_k > 0 ? c->top_k : 1;
  o->route_idx = (int32_t*)calloc((size_t)N * tk, sizeof(int32_t));
  o->route_w = (float*)calloc((size_t)N * tk, sizeof(float));
  o->pred_idx = (int32_t*)calloc((size_t)N * tk, sizeof(int32_t));
  if (c->n_experts) o->lru = (int32_t*)calloc((size_t)N * c->cache_slots, sizeof(int32_t));
  o->policy = 1;
  extern void orc_reset(orc*);
  orc_reset(o);
  return o;
}

void orc_reset(orc* o) {
  o->kv_len = 0;
  o->have_pending = 0;
  memset(&o->st, 0, sizeof(o->st));
  if (o->lru) /* initial residency: experts 0..C-1, expert 0 most recent */
    for (int L = 0; L < o->c.n_layers; ++L)
      for (int s = 0; s < o->c.cache_slots; ++s) o->lru[L * o->c.cache_slots + s] = s;
}

void orc_destroy(orc* o) {
  if (!o) return;
  for (int i = 0; i < o->c.n_layers; ++i) { free(o->L[i].ewg); free(o->L[i].ewu); free(o->L[i].ewd); }
  free(o->L); free(o->K); free(o->V); free(o->trH); free(o->slow_q); free(o->trP); free(o->logits);
  free(o->exit_logits); free(o->route_idx); free(o->route_w); free(o->pred_idx); free(o->lru);
  free(o->ls_full); free(o->ls_draft); free(o->rs_actual); free(o->rs_pred);
  free(o);
}

int orc_set_tensor(orc* o, int id, int layer, int expert, const void* ptr) {
  if (id < 0 || id >= T_COUNT) return -1;
  if (id <= T_LM_B || id == T_ARLA) { o->g[id] = ptr; return 0; }
  if (layer < 0 || layer >= o->c.n_layers) return -1;
  if (id >= T_EWG) {
    if (expert < 0 || expert >= o->c.n_experts) return -1;
    if (id == T_EWG) o->L[layer].ewg[expert] = ptr;
    if (id == T_EWU) o->L[layer].ewu[expert] = ptr;
    if (id == T_EWD) o->L[layer].ewd[expert] = ptr;
    return 0;
  }
  o->L[layer].t[id] = ptr;
  return 0;
}

static int32_t* dup_i32(const int32_t* src, size_t n) {
  int32_t* p = (int32_t*)malloc(sizeof(int32_t) * n);
  memcpy(p, src, sizeof(int32_t) * n);
  return p;
}

int orc_set_logit_script(orc* o, const int32_t* full_tok, const int32_t* draft_tok, int first_pos,
                         int n, float beta) {
  free(o->ls_full); free(o->ls_draft);
  o->ls_full = o->ls_draft = NULL;
  o->ls_n = 0;
  if (!full_tok || n <= 0) return 0;
  o->ls_full = dup_i32(full_tok, (size_t)n);
  o->ls_draft = dup_i32(draft_tok ? draft_tok : full_tok, (size_t)n);
  o->ls_first = first_pos; o->ls_n = n; o->ls_beta = beta;
  return 0;
}

int orc_set_router_script(orc* o, const int32_t* actual, const int32_t* pred, int first_pos, int n,
                          float beta) {
  free(o->rs_actual); free(o->rs_pred);
  o->rs_actual = o->rs_pred = NULL;
  o->rs_n = 0;
  if (!actual || n <= 0) return 0;
  size_t cnt = (size_t)n * o->c.n_layers * 2;
  o->rs_actual = dup_i32(actual, cnt);
  o->rs_pred = dup_i32(pred ? pred : actual, cnt);
  o->rs_first = first_pos; o->rs_n = n; o->rs_beta = beta;
  return 0;
}

int orc_set_policy(orc* o, int policy) {
  if (policy < 0 || policy > 4) return -1;
  o->policy = policy;
  return 0;
}

/* prefill: prompt through all layers, slow stream only, layer-major (identical per token to
 * token-by-token decoding: each token's arithmetic only reads K/V of positions <= its own). */
int orc_prefill(orc* o, const int32_t* tokens, int P, int32_t* first_token) {
  const orc_config* c = &o->c;
  if (P <= 0 || P > c->max_seq) return -1;
  int d = c->d_model;
  orc_reset(o);
  float* H = (float*)malloc(sizeof(float) * (size_t)P * d);
  for (int t = 0; t < P; ++t)
    for (int j = 0; j < d; ++j) H[(size_t)t * d + j] = wld(o, o->g[T_EMBED], (size_t)tokens[t] * d + j);
  for (int i = 0; i < c->n_layers; ++i) slow_layer(o, i, H, P, 0, 0);
  head_logits(o, H + (size_t)(P - 1) * d, 0, o->logits);
  int tok = pick_token(o, o->logits, P, 0, &o->last_margin);
  free(H);
  o->kv_len = P;
  o->pending = tok;
  o->have_pending = 1;
  if (first_token) *first_token = tok;
  return 0;
}

/* decode_step: both streams through all layers for the pending (or forced) token */
int orc_decode_step(orc* o, int force_token, int32_t* token_out, int32_t* exit_tokens) {
  o->topk_margin = INFINITY;
  const orc_config* c = &o->c;
  if (!o->have_pending && force_token < 0) return -2;
  if (o->kv_len + 1 > c->max_seq) return -3;
  int d = c->d_model;
  int tok_in = force_token >= 0 ? force_token : o->pending;
  float* h = (float*)malloc(sizeof(float) * d);
  float* p = (float*)malloc(sizeof(float) * d);
  int t = o->kv_len;
  dual_token(o, tok_in, t, c->n_layers, 1, h, p, exit_tokens, 1);
  arla_scores(o);
  head_logits(o, h, 0, o->logits);
  int tok = pick_token(o, o->logits, t + 1, 0, &o->last_margin);
  o->step_min_margin = o->last_margin;
  o->kv_len = t + 1;
  o->pending = tok;
  o->have_pending = 1;
  o->st.steps++;
  o->st.emitted++;
  if (token_out) *token_out = tok;
  free(h);
  free(p);
  return 0;
}

/* spec_step(gamma): draft gamma tokens from the accelerated stream at gate E = gates[0]
 * (§2.3.2), verify gamma+1 positions with the slow stream, accept the longest
 * matching prefix plus the verifier's own token, roll kv_len back (Q10-Q13). */
int orc_spec_step(orc* o, int gamma, int32_t* accepted, int32_t* n_accepted, int32_t* drafts_out) {
  o->topk_margin = INFINITY;
  const orc_config* c = &o->c;
  if (!o->have_pending) return -2;
  if (gamma < 0 || gamma > 16) return -1;
  if (gamma > 0 && (c->n_gates < 1 || !c->accel_enabled || c->accel_end_layer < c->gates[0])) return -1;
  int n = o->kv_len, d = c->d_model, m = gamma + 1;
  if (n + m > c->max_seq) return -3;
  int32_t drafts[17], tv[17];
  float* h = (float*)malloc(sizeof(float) * d);
  float* p = (float*)malloc(sizeof(float) * d);
  /* 1. draft: layers 0..E-1, both streams, feeding each draft back */
  int cur = o->pending;
  for (int j = 0; j < gamma; ++j) {
    int E = c->gates[0];
    int32_t ex[ORC_MAX_GATES];
    dual_token(o, cur, n + j, E, 1, h, p, ex, 0);
    if (j == 0 || o->last_draft_margin < o->step_min_margin) o->step_min_margin = o->last_draft_margin;
    drafts[j] = ex[0];
    cur = drafts[j];
  }
  /* 2. verify: [x_n, d_0..d_{gamma-1}] at positions n..n+gamma, slow stream, all layers */
  float* H = (float*)malloc(sizeof(float) * (size_t)m * d);
  for (int j = 0; j < m; ++j) {
    int tok = j == 0 ? o->pending : drafts[j - 1];
    for (int q = 0; q < d; ++q) H[(size_t)j * d + q] = wld(o, o->g[T_EMBED], (size_t)tok * d + q);
  }
  for (int i = 0; i < c->n_layers; ++i) slow_layer(o, i, H, m, n, 1);
  for (int j = 0; j < m; ++j) {
    head_logits(o, H + (size_t)j * d, 0, o->logits);
    tv[j] = pick_token(o, o->logits, n + j + 1, 0, &o->last_margin);
    if ((j == 0 && gamma == 0) || o->last_margin < o->step_min_margin) o->step_min_margin = o->last_margin;
  }
  /* 3. accept the longest matching prefix; 4. rollback = set kv_len */
  int a = 0;
  while (a < gamma && drafts[a] == tv[a]) ++a;
  for (int j = 0; j <= a; ++j) accepted[j] = tv[j];
  *n_accepted = a + 1;
  if (drafts_out) for (int j = 0; j < gamma; ++j) drafts_out[j] = drafts[j];
  o->kv_len = n + a + 1;
  o->pending = tv[a];
  o->st.steps++;
  o->st.drafted += gamma;
  o->st.accepted += a;
  o->st.emitted += a + 1;
  free(h); free(p); free(H);
  return 0;
}

/* ------------------------------------------------------------------ introspection */
int orc_kv_len(const orc* o) { return o->kv_len; }
int orc_pending(const orc* o) { return o->have_pending ? o->pending : -1; }
const float* orc_trace_h(const orc* o) { return o->trH; }
const float* orc_trace_p(const orc* o) { return o->trP; }
const float* orc_logits(const orc* o) { return o->logits; }
const float* orc_exit_logits(const orc* o, int gate) { return o->exit_logits + (size_t)gate * o->c.vocab; }
float orc_last_margin(const orc* o) { return o->last_margin; }
float orc_last_draft_margin(const orc* o) { return o->last_draft_margin; }
float orc_step_min_margin(const orc* o) { return o->step_min_margin; }
/* smallest gap between the k-th and (k+1)-th slow score over the top-k token selections of the last step (INFINITY: none) */
float orc_topk_margin(const orc* o) { return o->topk_margin; }
float orc_exit_score(const orc* o, int gate) { return (gate >= 0 && gate < o->c.n_gates) ? o->exit_score[gate] : -1.f; }
float* orc_kcache(orc* o, int layer) { return o->K + (size_t)layer * o->c.max_seq * o->c.d_model; }
float* orc_vcache(orc* o, int layer) { return o->V + (size_t)layer * o->c.max_seq * o->c.d_model; }
const int32_t* orc_route_idx(const orc* o) { return o->route_idx; }
const float* orc_route_w(const orc* o) { return o->route_w; }
const int32_t* orc_pred_idx(const orc* o) { return o->pred_idx; }
const int32_t* orc_lru(const orc* o) { return o->lru; }
void orc_get_stats(const orc* o, orc_stats* out) { *out = o->st; }

/* stand-alone pieces exposed so the pins can hit them directly */
void orc_rope(const orc* o, float* v, int t) { rope(o, v, t); }
void orc_rmsnorm(const orc* o, const float* x, const void* g, float* y) { rmsnorm(o, x, g, y); }
void orc_route(const orc* o, const void* Wr, const float* y, int32_t* idx, float* w) {
  route(o, Wr, y, NULL, 0.f, idx, w);
}
int orc_argmax(const float* v, int n) { return argmax_margin(v, n, NULL); }
void orc_accel_layer(orc* o, int i, float* p, int t) { accel_layer(o, i, p, t); }
void orc_slow_layer(orc* o, int i, float* h, int m, int t0) { slow_layer(o, i, h, m, t0, 0); }
int orc_lru_use(orc* o, int L, const int32_t* idx) { moe_use_event(o, L, idx); return 0; }
int orc_lru_predict(orc* o, int L, const int32_t* idx) { moe_predict_event(o, L, idx); return 0; }
