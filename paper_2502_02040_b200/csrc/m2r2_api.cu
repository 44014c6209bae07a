// m2r2_api.cu — host orchestration behind the C ABI of include/m2r2.h.
//
// Owns: the context, the HBM layout of weights / KV cache / scratch, the launch sequences of
// prefill, dual-stream decode, self-speculative decode (draft loop, k-token verify, accept +
// rollback on the device) and the MoE expert cache with ahead-of-time prefetch on a copy
// stream.  All arithmetic runs in the kernels of kernels_general.cu / kernels_fused.cu.
#include <math.h>
#include <stdarg.h>
#include <stdio.h>
#include <string.h>

#include <algorithm>
#include <map>
#include <vector>

#include "m2r2_internal.cuh"
#include "m2r2_fused.cuh"

// ------------------------------------------------------------------ small device kernels (control)
// Row set-up: everything a step needs (tokens, positions) is derived ON THE DEVICE from
// kv_len / pending / drafts, so steps can be enqueued back to back without host round trips.
enum { MODE_DUAL = 0, MODE_VERIFY = 1, MODE_PREFILL = 2 };

__global__ void setup_rows_kernel(int mode, int B, int m, int joff, int c0, int max_seq,
                                  const int* __restrict__ kv_len, const int* __restrict__ pending,
                                  const int* __restrict__ drafts, const int* __restrict__ force,
                                  const int* __restrict__ prompt, int* row_tok, int* row_seq,
                                  int* row_pos, int* row_limit, int* grp_rows) {
  int b = blockIdx.x;
  if (threadIdx.x != 0) return;
  for (int q = 0; q < M2R2_MAXQ; ++q) grp_rows[b * M2R2_MAXQ + q] = -1;
  if (mode == MODE_DUAL) {
    int tok = joff == 0 ? (force ? force[b] : pending[b]) : drafts[b * 8 + joff - 1];
    int pos = kv_len[b] + joff;
    row_tok[b] = tok; row_seq[b] = b; row_pos[b] = pos; row_limit[b] = pos + 1;
    row_tok[B + b] = tok; row_seq[B + b] = b; row_pos[B + b] = pos; row_limit[B + b] = pos;
    grp_rows[b * M2R2_MAXQ + 0] = b;
    grp_rows[b * M2R2_MAXQ + 1] = B + b;
  } else {
    for (int j = 0; j < m; ++j) {
      int r = b * m + j, pos, tok;
      if (mode == MODE_VERIFY) {
        pos = kv_len[b] + j;
        tok = j == 0 ? pending[b] : drafts[b * 8 + j - 1];
      } else {
        pos = c0 + j;
        tok = prompt[(size_t)b * max_seq + pos];
      }
      row_tok[r] = tok; row_seq[r] = b; row_pos[r] = pos; row_limit[r] = pos + 1;
      grp_rows[b * M2R2_MAXQ + j] = r;
    }
  }
}

// decode_step epilogue: kv_len += 1, pending = token
__global__ void advance_kernel(int B, int* kv_len, int* pending, const int* tok) {
  int b = threadIdx.x;
  if (b < B) { kv_len[b] += 1; pending[b] = tok[b]; }
}

// a12  accept + rollback: a = longest prefix with d_i == t_i; emit t_0..t_a; kv_len += a+1;
// pending = t_a.  Positions >= kv_len are dead and get overwritten (Q13).
__global__ void accept_kernel(int B, int k, const int* __restrict__ drafts, const int* __restrict__ vtok,
                              int* accepted, int* n_acc, int* kv_len, int* pending) {
  int b = threadIdx.x;
  if (b >= B) return;
  int a = 0;
  while (a < k && drafts[b * 8 + a] == vtok[b * 8 + a]) ++a;
  for (int j = 0; j <= a; ++j) accepted[b * 8 + j] = vtok[b * 8 + j];
  n_acc[b] = a + 1;
  kv_len[b] += a + 1;
  pending[b] = vtok[b * 8 + a];
}

__global__ void set_state_kernel(int B, int* kv_len, int* pending, int kv, const int* tok) {
  int b = threadIdx.x;
  if (b < B) { kv_len[b] = kv; if (tok) pending[b] = tok[b]; }
}

// ------------------------------------------------------------------ context
struct m2r2_ctx {
  m2r2_config c;
  m2r2_buffers b;
  cudaStream_t cs, cps, ods;   // compute, copy (prefetch), on-demand (internal, high priority)
  bool weights_loaded = false, have_pending = false, fused = true;
  int B = 0;                   // live sequences
  int R = 0;                   // max activation rows
  int kv_h[M2R2_MAX_BATCH];    // host mirror of kv_len
  size_t esz = 0;              // bytes per element
  // resident weights
  const void *embed = nullptr, *gf = nullptr, *lm_head = nullptr, *lm_A = nullptr, *lm_B = nullptr, *arla = nullptr;
  void* packed = nullptr;      // tile-major copy of the big matrices for the fused kernel
  std::vector<DevLayer> L;
  // MoE
  std::vector<std::vector<const void*>> eg, eu, ed;   // pinned host blobs [layer][expert]
  std::vector<std::vector<int>> lru;                  // [layer][slot order] expert ids, MRU first
  std::vector<std::vector<int>> slot_of;              // [layer][expert] -> slot or -1
  std::vector<std::vector<int>> slot_expert;          // [layer][slot] -> expert
  std::vector<cudaEvent_t> ev_layer_done, ev_copy_done;
  std::vector<char> copy_pending;
  cudaEvent_t ev_tmp = nullptr, ev_stage_free = nullptr;
  size_t expert_bytes = 0, eg_bytes = 0, ed_bytes = 0;
  int policy = M2R2_POLICY_LRU;
  int* h_pinned = nullptr;     // pinned host staging for small D2H reads
  // forced tokens are staged through a ring of pinned slots, each guarded by an event recorded behind its H2D
  // copy: decode_step(tokens_out == NULL) returns without synchronising, so the next call must not overwrite a
  // slot whose copy has not executed yet
  static constexpr int FORCE_SLOTS = 8;
  int* h_force = nullptr;      // [FORCE_SLOTS][M2R2_MAX_BATCH]
  cudaEvent_t ev_force[FORCE_SLOTS] = {};
  unsigned int force_ctr = 0;
  int sm_count = 148;
  // scripts
  int ls_first = 0, ls_n = 0; float ls_beta = 0.f; bool ls_on = false;
  int rs_first = 0, rs_n = 0; float rs_beta = 0.f; bool rs_on = false;
  // scratch
  int *d_kv_len, *d_pending, *d_row_tok, *d_row_seq, *d_row_pos, *d_row_limit, *d_grp_rows;
  int *d_drafts, *d_vtok, *d_accepted, *d_nacc, *d_exit_tok, *d_out_tok, *d_force, *d_prompt;
  int *d_qkv_bmap, *d_accel_cols, *d_accel_heads, *d_ls_full, *d_ls_draft, *d_rs_actual, *d_rs_pred;
  int *d_route_idx, *d_pred_idx, *d_moe_ridx;
  float *resid, *xn, *U, *qkv, *attn_o, *act, *part_o, *part_ml, *logits, *exit_logits, *trace;
  float *moe_tmp, *route_w, *pred_w, *moe_wtab, *moe_rw, *exit_score;
  int last_rows_per_seq = 1;
  // CUDA graphs of the verify pass (a11 + a12), keyed by what fixes its launch arguments
  std::map<unsigned long long, cudaGraphExec_t> vgraph;
  std::map<unsigned long long, int> vgraph_seen;      // eager runs so far; < 0: capture failed, stay eager
  std::map<unsigned long long, int> vgraph_launches;  // kernels inside the graph (for the launch counter)
  unsigned int ls_version = 0;
  float2* rope_tab;
  FusedState fs;
  uint32_t accel_mask[4];
  m2r2_stats st;
  // profiling: segment i = [pev[i], pev[i+1]) belongs to class pcls[i]
  bool prof = false;
  std::vector<cudaEvent_t> pev;
  std::vector<int> pcls;
  int pn = 0;
  m2r2_profile pr;
  char err[512];
};

static void prof_mark(m2r2_ctx* x, int cls) {
  if (!x->prof) return;
  if (x->pn > 0 && x->pcls[x->pn - 1] == cls) return;   // same class continues
  if (x->pn == (int)x->pev.size()) {
    cudaEvent_t e;
    if (cudaEventCreate(&e) != cudaSuccess) return;
    x->pev.push_back(e);
    x->pcls.push_back(-1);
  }
  cudaEventRecord(x->pev[x->pn], x->cs);
  x->pcls[x->pn] = cls;
  x->pn++;
}
static void prof_resolve(m2r2_ctx* x) {
  if (!x->prof || x->pn == 0) return;
  prof_mark(x, -1);
  cudaStreamSynchronize(x->cs);
  for (int i = 0; i + 1 < x->pn; ++i) {
    int c = x->pcls[i];
    float ms = 0.f;
    if (c >= 0 && c < M2R2_PROF_CLASSES && cudaEventElapsedTime(&ms, x->pev[i], x->pev[i + 1]) == cudaSuccess) {
      x->pr.ms[c] += ms;
      x->pr.segments[c]++;
    }
  }
  x->pr.steps++;
  x->pn = 0;
}

static int fail(m2r2_ctx* ctx, int code, const char* fmt, ...) {
  if (ctx) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(ctx->err, sizeof(ctx->err), fmt, ap);
    va_end(ap);
  }
  return code;
}
#define CU(ctx, call)                                                                          \
  do {                                                                                         \
    cudaError_t e_ = (call);                                                                   \
    if (e_ != cudaSuccess)                                                                     \
      return fail(ctx, M2R2_CUDA, "%s failed: %s (%s:%d)", #call, cudaGetErrorString(e_), __FILE__, __LINE__); \
  } while (0)

static int validate(const m2r2_config* c) {
  if (!c || c->struct_size != sizeof(m2r2_config)) return M2R2_INVALID_ARG;
  if (c->n_layers < 1 || c->n_layers > M2R2_MAX_LAYERS) return M2R2_INVALID_ARG;
  if (c->n_heads < 1 || c->n_heads > M2R2_MAX_HEADS) return M2R2_INVALID_ARG;
  if (c->d_model != c->n_heads * c->head_dim) return M2R2_INVALID_ARG;
  if (c->head_dim % 32 != 0 || c->head_dim > 128) return M2R2_INVALID_ARG;
  if (c->d_model % 8 || c->d_model > 12288) return M2R2_INVALID_ARG;
  if (c->dtype != M2R2_FP32 && c->dtype != M2R2_BF16) return M2R2_INVALID_ARG;
  if (c->max_batch < 1 || c->max_batch > M2R2_MAX_BATCH || c->max_seq < 1) return M2R2_INVALID_ARG;
  if (c->vocab < 2) return M2R2_INVALID_ARG;
  if (c->accel_topk_tokens < 0 || c->accel_topk_tokens > 4096) return M2R2_INVALID_ARG;
  if (c->arla_dim < 0 || c->arla_dim > 128) return M2R2_INVALID_ARG;
  if (c->arla_dim > 0 && ((size_t)2 * (c->n_layers + 1) * c->arla_dim + c->arla_dim + c->n_layers + 1) * 4 > (size_t)160 * 1024) return M2R2_INVALID_ARG;
  if (c->accel_topk_tokens > 0 && ((size_t)c->max_seq + 8 + 2 * (size_t)c->head_dim + 2 * (size_t)c->accel_topk_tokens + 1) * 4 > (size_t)200 * 1024) return M2R2_INVALID_ARG;
  if (c->n_gates < 0 || c->n_gates > M2R2_MAX_GATES) return M2R2_INVALID_ARG;
  for (int j = 0; j < c->n_gates; ++j) {
    if (c->gates[j] < 1 || c->gates[j] > c->n_layers) return M2R2_INVALID_ARG;
    if (j && c->gates[j] <= c->gates[j - 1]) return M2R2_INVALID_ARG;
  }
  if (c->accel_enabled) {
    if (c->n_accel_heads < 1 || c->n_accel_heads > c->n_heads) return M2R2_INVALID_ARG;
    for (int s = 0; s < c->n_accel_heads; ++s) {
      if (c->accel_heads[s] < 0 || c->accel_heads[s] >= c->n_heads) return M2R2_INVALID_ARG;
      if (s && c->accel_heads[s] <= c->accel_heads[s - 1]) return M2R2_INVALID_ARG;
    }
    if (c->adapter_rank < 1 || c->adapter_rank > 16) return M2R2_INVALID_ARG;
    if (c->accel_end_layer < 0 || c->accel_end_layer > c->n_layers) return M2R2_INVALID_ARG;
    // a gate above the last accelerated layer would never be evaluated (p is not live there): its exit token
    // slot would hold stale values that look like token ids
    for (int j = 0; j < c->n_gates; ++j)
      if (c->gates[j] > c->accel_end_layer) return M2R2_INVALID_ARG;
  }
  if (c->n_experts > 0) {
    if (c->n_experts > M2R2_MAX_EXPERTS || c->top_k < 1 || c->top_k > M2R2_MAX_TOPK ||
        c->top_k > c->n_experts) return M2R2_INVALID_ARG;
    if (c->d_ff_expert < 8 || c->d_ff_expert % 8) return M2R2_INVALID_ARG;
    if (c->cache_slots_per_layer < c->top_k || c->cache_slots_per_layer > c->n_experts) return M2R2_INVALID_ARG;
    if (c->accel_enabled && (c->accel_mlp_rank < 8 || c->accel_mlp_rank % 8)) return M2R2_INVALID_ARG;
    if (c->max_batch != 1) return M2R2_UNSUPPORTED;
    for (int i = 0; i < c->n_layers; ++i)
      if (c->aot_lo[i] < c->aot_hi[i] && (c->aot_lo[i] <= i || c->aot_hi[i] > c->n_layers)) return M2R2_INVALID_ARG;
  } else {
    if (c->d_ff < 8 || c->d_ff % 8) return M2R2_INVALID_ARG;
  }
  return M2R2_OK;
}

static bool layer_accel(const m2r2_config& c, int i) { return c.accel_enabled && i < c.accel_end_layer; }
static int fmax_act(const m2r2_config& c) {
  int f = c.d_ff;
  if (c.n_experts) f = std::max(c.d_ff_expert, c.accel_mlp_rank);
  return std::max(f, 8);
}

// HBM layout of the resident weights (same walk for sizing and for loading)
struct WeightWalk {
  Carver cv;
  size_t esz;
  explicit WeightWalk(void* base, size_t e) : cv(base), esz(e) {}
  void* take(size_t elems) { return cv.take<char>(elems * esz); }
};

static void walk_weights(const m2r2_config& c, WeightWalk& w, m2r2_ctx* ctx) {
  const size_t d = c.d_model, V = c.vocab, r = c.adapter_rank, F = c.d_ff;
  const size_t da = (size_t)c.n_accel_heads * c.head_dim;
  void* p;
  p = w.take(V * d); if (ctx) ctx->embed = p;
  p = w.take(d); if (ctx) ctx->gf = p;
  p = w.take(V * d); if (ctx) ctx->lm_head = p;
  if (c.lm_head_adapter && c.accel_enabled) {
    p = w.take(r * d); if (ctx) ctx->lm_A = p;
    p = w.take(V * r); if (ctx) ctx->lm_B = p;
  }
  if (c.arla_dim > 0 && c.accel_enabled && c.n_gates > 0) {
    p = w.take((size_t)c.n_gates * (3 * c.arla_dim + 1) * d); if (ctx) ctx->arla = p;
  }
  for (int i = 0; i < c.n_layers; ++i) {
    DevLayer L;
    memset(&L, 0, sizeof(L));
    L.g1 = w.take(d); L.g2 = w.take(d);
    L.wqkv = w.take(3 * d * d); L.wo = w.take(d * d);
    if (!c.n_experts) { L.wgate = w.take(F * d); L.wup = w.take(F * d); L.wdown = w.take(d * F); }
    else L.router = w.take((size_t)c.n_experts * d);
    if (layer_accel(c, i)) {
      L.Aqkv = w.take(3 * r * d); L.Bqkv = w.take(3 * da * r);
      L.Ao = w.take(r * da); L.Bo = w.take(d * r);
      if (!c.n_experts) {
        L.Agu = w.take(2 * r * d); L.Bg = w.take(F * r); L.Bu = w.take(F * r);
        L.Ad = w.take(r * F); L.Bd = w.take(d * r);
      } else {
        size_t rm = c.accel_mlp_rank;
        L.Ug = w.take(rm * d); L.Uu = w.take(rm * d); L.Ud = w.take(d * rm);
      }
    }
    if (ctx) ctx->L.push_back(L);
  }
  size_t fb = fused_weights_bytes(c);
  if (fb) {
    void* pk = w.cv.take<char>(fb);
    if (ctx) ctx->packed = pk;
  }
}

static void carve_scratch(const m2r2_config& c, Carver& cv, m2r2_ctx* x) {
  const size_t B = c.max_batch, R = B * 8, d = c.d_model, V = c.vocab, N = c.n_layers;
  const size_t G = std::max(1, c.n_gates), nh = c.n_heads, dh = c.head_dim, S = c.max_seq;
  const size_t da = (size_t)std::max(1, c.n_accel_heads) * dh, tk = std::max(1, c.top_k);
  m2r2_ctx* o = x;
#define TAKE(field, T, n) { T* p_ = cv.take<T>(n); if (o) o->field = p_; }
  TAKE(d_kv_len, int, B) TAKE(d_pending, int, B)
  TAKE(d_row_tok, int, R) TAKE(d_row_seq, int, R) TAKE(d_row_pos, int, R) TAKE(d_row_limit, int, R)
  TAKE(d_grp_rows, int, R * M2R2_MAXQ)
  TAKE(d_drafts, int, B * 8) TAKE(d_vtok, int, B * 8) TAKE(d_accepted, int, B * 8) TAKE(d_nacc, int, B)
  TAKE(d_exit_tok, int, B * G) TAKE(d_out_tok, int, B) TAKE(d_force, int, B)
  TAKE(d_prompt, int, B * S)
  TAKE(d_qkv_bmap, int, 3 * d) TAKE(d_accel_cols, int, da) TAKE(d_accel_heads, int, M2R2_MAX_HEADS)
  TAKE(d_ls_full, int, B * S) TAKE(d_ls_draft, int, B * S)
  TAKE(d_rs_actual, int, c.n_experts ? S * N * 2 : 1) TAKE(d_rs_pred, int, c.n_experts ? S * N * 2 : 1)
  TAKE(d_route_idx, int, N * tk) TAKE(d_pred_idx, int, N * tk) TAKE(exit_score, float, M2R2_MAX_BATCH * M2R2_MAX_GATES)
  TAKE(resid, float, R * d) TAKE(xn, float, R * d) TAKE(U, float, R * 64)
  TAKE(qkv, float, R * 3 * d) TAKE(attn_o, float, R * d) TAKE(act, float, R * (size_t)fmax_act(c))
  TAKE(part_o, float, R * nh * M2R2_MAX_SPLITS * dh) TAKE(part_ml, float, R * nh * M2R2_MAX_SPLITS * 2)
  TAKE(logits, float, R * V) TAKE(exit_logits, float, G * B * V)
  TAKE(trace, float, (N + 1) * 2 * B * d)
  TAKE(moe_tmp, float, R * d) TAKE(route_w, float, N * tk) TAKE(pred_w, float, N * tk)
  TAKE(moe_wtab, float, 8) TAKE(moe_rw, float, 8 * M2R2_MAX_TOPK) TAKE(d_moe_ridx, int, 8 * M2R2_MAX_TOPK)   // MoE prefill chunk tables
  TAKE(rope_tab, float2, S * (dh / 2))
#undef TAKE
  fused_carve(c, cv, o ? &o->fs : nullptr);
}

// m2r2_ctx has std::vector members; the sizing walk must not construct one on the stack with
// uninitialised pointers being read — carve_scratch only writes fields, so this is safe.

extern "C" int m2r2_query_sizes(const m2r2_config* cfg, m2r2_sizes* out) {
  int rc = validate(cfg);
  if (rc) return rc;
  if (!out) return M2R2_INVALID_ARG;
  const m2r2_config& c = *cfg;
  size_t esz = c.dtype == M2R2_FP32 ? 4 : 2;
  WeightWalk w(nullptr, esz);
  walk_weights(c, w, nullptr);
  out->weights_bytes = w.cv.size();
  out->kv_bytes = 2ull * c.n_layers * c.max_batch * c.n_heads * (size_t)c.max_seq * c.head_dim * esz + 512;
  Carver cv(nullptr);
  carve_scratch(c, cv, nullptr);
  out->scratch_bytes = cv.size();
  out->expert_cache_bytes = 0;
  out->expert_store_bytes = 0;
  if (c.n_experts) {
    size_t eb = 3ull * c.d_ff_expert * c.d_model * esz;
    eb = (eb + 255) & ~(size_t)255;
    out->expert_cache_bytes = ((size_t)c.n_layers * c.cache_slots_per_layer + c.top_k) * eb;
    out->expert_store_bytes = (size_t)c.n_layers * c.n_experts * 3ull * c.d_ff_expert * c.d_model * esz;
  }
  return M2R2_OK;
}

extern "C" int m2r2_create(const m2r2_config* cfg, const m2r2_buffers* bufs, void* compute_stream,
                           void* copy_stream, m2r2_ctx** out) {
  int rc = validate(cfg);
  if (rc) return rc;
  if (!bufs || !out || !bufs->weights || !bufs->kv || !bufs->scratch) return M2R2_INVALID_ARG;
  if (cfg->n_experts && !bufs->expert_cache) return M2R2_INVALID_ARG;
  int dev_count = 0;
  if (cudaGetDeviceCount(&dev_count) != cudaSuccess || dev_count < 1) return M2R2_CUDA;
  m2r2_ctx* x = new m2r2_ctx();
  x->c = *cfg;
  x->b = *bufs;
  x->cs = (cudaStream_t)compute_stream;
  x->cps = (cudaStream_t)copy_stream;
  x->err[0] = 0;
  memset(&x->st, 0, sizeof(x->st));
  memset(&x->pr, 0, sizeof(x->pr));
  memset(x->kv_h, 0, sizeof(x->kv_h));
  const m2r2_config& c = x->c;
  x->esz = c.dtype == M2R2_FP32 ? 4 : 2;
  x->R = c.max_batch * 8;
  WeightWalk w(bufs->weights, x->esz);
  walk_weights(c, w, x);
  rc = fused_create(c, &x->fs);   // before the carve: the fused scratch pointers land in fs.impl
  if (rc) { delete x; return rc; }
  x->fs.launch_counter = &x->st.kernel_launches;
  Carver cv(bufs->scratch);
  carve_scratch(c, cv, x);
  memset(x->accel_mask, 0, sizeof(x->accel_mask));
  if (c.accel_enabled)
    for (int s = 0; s < c.n_accel_heads; ++s) x->accel_mask[c.accel_heads[s] >> 5] |= 1u << (c.accel_heads[s] & 31);
#define CUX(call)                                                                     \
  do {                                                                                \
    cudaError_t e_ = (call);                                                          \
    if (e_ != cudaSuccess) {                                                          \
      fprintf(stderr, "m2r2_create: %s: %s\n", #call, cudaGetErrorString(e_));        \
      fused_destroy(&x->fs);                                                          \
      delete x;                                                                       \
      return M2R2_CUDA;                                                               \
    }                                                                                 \
  } while (0)
  // RoPE table in double precision on the host (Q1: full-precision sin/cos)
  {
    int half = c.head_dim / 2;
    std::vector<float2> tab((size_t)c.max_seq * half);
    for (int t = 0; t < c.max_seq; ++t)
      for (int j = 0; j < half; ++j) {
        double ang = (double)t * pow((double)c.rope_theta, -2.0 * j / c.head_dim);
        tab[(size_t)t * half + j] = make_float2((float)cos(ang), (float)sin(ang));
      }
    CUX(cudaMemcpyAsync(x->rope_tab, tab.data(), tab.size() * sizeof(float2), cudaMemcpyHostToDevice, x->cs));
    // adapter row maps
    int d = c.d_model, dh = c.head_dim, da = c.n_accel_heads * dh;
    std::vector<int> bmap(3 * (size_t)d, -1), cols(std::max(1, da), 0);
    std::vector<int> sidx(c.n_heads, -1);
    if (c.accel_enabled)
      for (int s = 0; s < c.n_accel_heads; ++s) sidx[c.accel_heads[s]] = s;
    for (int n = 0; n < 3 * d; ++n) {
      int which = n / d, a = (n % d) / dh, j = (n % d) % dh;
      if (sidx[a] >= 0) bmap[n] = which * da + sidx[a] * dh + j;
    }
    if (c.accel_enabled)
      for (int s = 0; s < c.n_accel_heads; ++s)
        for (int j = 0; j < dh; ++j) cols[s * dh + j] = c.accel_heads[s] * dh + j;
    CUX(cudaMemcpyAsync(x->d_qkv_bmap, bmap.data(), bmap.size() * sizeof(int), cudaMemcpyHostToDevice, x->cs));
    CUX(cudaMemcpyAsync(x->d_accel_cols, cols.data(), cols.size() * sizeof(int), cudaMemcpyHostToDevice, x->cs));
    if (c.accel_enabled && c.n_accel_heads > 0)
      CUX(cudaMemcpyAsync(x->d_accel_heads, c.accel_heads, sizeof(int) * c.n_accel_heads, cudaMemcpyHostToDevice, x->cs));
    CUX(cudaStreamSynchronize(x->cs));
  }
  CUX(cudaMallocHost((void**)&x->h_pinned, 4096 * sizeof(int)));
  CUX(cudaMallocHost((void**)&x->h_force, m2r2_ctx::FORCE_SLOTS * M2R2_MAX_BATCH * sizeof(int)));
  for (int i = 0; i < m2r2_ctx::FORCE_SLOTS; ++i) CUX(cudaEventCreateWithFlags(&x->ev_force[i], cudaEventDisableTiming));
  {
    int dev = 0;
    CUX(cudaGetDevice(&dev));
    CUX(cudaDeviceGetAttribute(&x->sm_count, cudaDevAttrMultiProcessorCount, dev));
  }
  CUX(cudaEventCreateWithFlags(&x->ev_tmp, cudaEventDisableTiming));
  CUX(cudaEventCreateWithFlags(&x->ev_stage_free, cudaEventDisableTiming));
  int lo = 0, hi = 0;
  cudaDeviceGetStreamPriorityRange(&lo, &hi);
  CUX(cudaStreamCreateWithPriority(&x->ods, cudaStreamNonBlocking, hi));
  if (c.n_experts) {
    size_t eb = 3ull * c.d_ff_expert * c.d_model * x->esz;
    x->eg_bytes = (size_t)c.d_ff_expert * c.d_model * x->esz;
    x->ed_bytes = x->eg_bytes;
    x->expert_bytes = (eb + 255) & ~(size_t)255;
    x->ev_layer_done.resize(c.n_layers);
    x->ev_copy_done.resize(c.n_layers);
    x->copy_pending.assign(c.n_layers, 0);
    for (int i = 0; i < c.n_layers; ++i) {
      CUX(cudaEventCreateWithFlags(&x->ev_layer_done[i], cudaEventDisableTiming));
      CUX(cudaEventCreateWithFlags(&x->ev_copy_done[i], cudaEventDisableTiming));
    }
  }
#undef CUX
  *out = x;
  return M2R2_OK;
}

extern "C" int m2r2_destroy(m2r2_ctx* x) {
  if (!x) return M2R2_INVALID_ARG;
  cudaStreamSynchronize(x->cs);
  for (auto& kv : x->vgraph) cudaGraphExecDestroy(kv.second);
  if (x->cps != x->cs) cudaStreamSynchronize(x->cps);
  if (x->ods) { cudaStreamSynchronize(x->ods); cudaStreamDestroy(x->ods); }
  for (auto e : x->ev_layer_done) cudaEventDestroy(e);
  for (auto e : x->ev_copy_done) cudaEventDestroy(e);
  if (x->ev_tmp) cudaEventDestroy(x->ev_tmp);
  if (x->ev_stage_free) cudaEventDestroy(x->ev_stage_free);
  if (x->h_pinned) cudaFreeHost(x->h_pinned);
  if (x->h_force) cudaFreeHost(x->h_force);
  for (auto e : x->ev_force) if (e) cudaEventDestroy(e);
  for (auto e : x->pev) cudaEventDestroy(e);
  fused_destroy(&x->fs);
  delete x;
  return M2R2_OK;
}

// ------------------------------------------------------------------ weights
static int up(m2r2_ctx* x, const void* dst, const void* src, size_t elems) {
  if (!src) return fail(x, M2R2_INVALID_ARG, "load_weights: a required tensor is NULL");
  CU(x, cudaMemcpyAsync((void*)dst, src, elems * x->esz, cudaMemcpyHostToDevice, x->cs));
  return 0;
}
static void* off(const void* base, size_t elems, size_t esz) { return (char*)base + elems * esz; }

static void* slot_ptr(m2r2_ctx* x, int layer, int slot) {
  return (char*)x->b.expert_cache + ((size_t)layer * x->c.cache_slots_per_layer + slot) * x->expert_bytes;
}
static void* stage_ptr(m2r2_ctx* x, int k) {
  return (char*)x->b.expert_cache + ((size_t)x->c.n_layers * x->c.cache_slots_per_layer + k) * x->expert_bytes;
}
// one expert = gate | up | down, three DMA copies into one slot
static int copy_expert(m2r2_ctx* x, int layer, int e, void* dst, cudaStream_t st) {
  char* p = (char*)dst;
  CU(x, cudaMemcpyAsync(p, x->eg[layer][e], x->eg_bytes, cudaMemcpyHostToDevice, st));
  CU(x, cudaMemcpyAsync(p + x->eg_bytes, x->eu[layer][e], x->eg_bytes, cudaMemcpyHostToDevice, st));
  CU(x, cudaMemcpyAsync(p + 2 * x->eg_bytes, x->ed[layer][e], x->ed_bytes, cudaMemcpyHostToDevice, st));
  x->st.h2d_bytes += (int64_t)(2 * x->eg_bytes + x->ed_bytes);
  return 0;
}

static int reset_expert_cache(m2r2_ctx* x) {
  const m2r2_config& c = x->c;
  if (!c.n_experts) return 0;
  int C = c.cache_slots_per_layer;
  x->lru.assign(c.n_layers, std::vector<int>());
  x->slot_of.assign(c.n_layers, std::vector<int>(c.n_experts, -1));
  x->slot_expert.assign(c.n_layers, std::vector<int>(C, -1));
  CU(x, cudaStreamSynchronize(x->cs));
  CU(x, cudaStreamSynchronize(x->cps));
  CU(x, cudaStreamSynchronize(x->ods));
  int64_t keep = x->st.h2d_bytes;
  for (int i = 0; i < c.n_layers; ++i) {
    for (int s = 0; s < C; ++s) {   // initial residency: experts 0..C-1, expert 0 most recent
      x->lru[i].push_back(s);
      x->slot_of[i][s] = s;
      x->slot_expert[i][s] = s;
      int rc = copy_expert(x, i, s, slot_ptr(x, i, s), x->cps);
      if (rc) return rc;
    }
    x->copy_pending[i] = 0;
  }
  CU(x, cudaStreamSynchronize(x->cps));
  x->st.h2d_bytes = keep;
  return 0;
}

extern "C" int m2r2_load_weights(m2r2_ctx* x, const m2r2_weight_table* t) {
  if (!x || !t || !t->layers) return M2R2_INVALID_ARG;
  const m2r2_config& c = x->c;
  const size_t d = c.d_model, V = c.vocab, r = c.adapter_rank, F = c.d_ff, e = x->esz;
  const size_t da = (size_t)c.n_accel_heads * c.head_dim;
  int rc;
#define UP(dst, src, n) if ((rc = up(x, dst, src, n))) return rc
  UP(x->embed, t->embed, V * d); UP(x->gf, t->gf, d); UP(x->lm_head, t->lm_head, V * d);
  if (x->lm_A) { UP(x->lm_A, t->lm_A, r * d); UP(x->lm_B, t->lm_B, V * r); }
  if (x->arla) {
    if (!t->arla) return fail(x, M2R2_INVALID_ARG, "arla_dim > 0 but the weight table has no ARLA router");
    UP(x->arla, t->arla, (size_t)c.n_gates * (3 * c.arla_dim + 1) * d);
  }
  if (c.n_experts) { x->eg.assign(c.n_layers, {}); x->eu.assign(c.n_layers, {}); x->ed.assign(c.n_layers, {}); }
  for (int i = 0; i < c.n_layers; ++i) {
    const m2r2_layer_weights& h = t->layers[i];
    const DevLayer& L = x->L[i];
    UP(L.g1, h.g1, d); UP(L.g2, h.g2, d);
    UP(L.wqkv, h.wq, d * d); UP(off(L.wqkv, d * d, e), h.wk, d * d); UP(off(L.wqkv, 2 * d * d, e), h.wv, d * d);
    UP(L.wo, h.wo, d * d);
    if (!c.n_experts) { UP(L.wgate, h.wgate, F * d); UP(L.wup, h.wup, F * d); UP(L.wdown, h.wdown, d * F); }
    else {
      UP(L.router, h.router, (size_t)c.n_experts * d);
      if (!h.expert_gate || !h.expert_up || !h.expert_down) return fail(x, M2R2_INVALID_ARG, "expert blobs missing");
      for (int q = 0; q < c.n_experts; ++q) {
        if (!h.expert_gate[q] || !h.expert_up[q] || !h.expert_down[q]) return fail(x, M2R2_INVALID_ARG, "expert blob NULL");
        x->eg[i].push_back(h.expert_gate[q]); x->eu[i].push_back(h.expert_up[q]); x->ed[i].push_back(h.expert_down[q]);
      }
    }
    if (layer_accel(c, i)) {
      UP(L.Aqkv, h.Aq, r * d); UP(off(L.Aqkv, r * d, e), h.Ak, r * d); UP(off(L.Aqkv, 2 * r * d, e), h.Av, r * d);
      UP(L.Bqkv, h.Bq, da * r); UP(off(L.Bqkv, da * r, e), h.Bk, da * r); UP(off(L.Bqkv, 2 * da * r, e), h.Bv, da * r);
      UP(L.Ao, h.Ao, r * da); UP(L.Bo, h.Bo, d * r);
      if (!c.n_experts) {
        UP(L.Agu, h.Ag, r * d); UP(off(L.Agu, r * d, e), h.Au, r * d);
        UP(L.Bg, h.Bg, F * r); UP(L.Bu, h.Bu, F * r); UP(L.Ad, h.Ad, r * F); UP(L.Bd, h.Bd, d * r);
      } else {
        size_t rm = c.accel_mlp_rank;
        UP(L.Ug, h.Ug, rm * d); UP(L.Uu, h.Uu, rm * d); UP(L.Ud, h.Ud, d * rm);
      }
    }
  }
#undef UP
  CU(x, cudaStreamSynchronize(x->cs));
  x->weights_loaded = true;
  rc = reset_expert_cache(x);
  if (rc) return rc;
  rc = fused_bind(x->c, &x->fs, x->cs, x->packed, x->embed, x->gf, x->lm_head, x->lm_A, x->lm_B, x->L.data(), x->b.kv,
                  x->rope_tab);
  if (rc) return fail(x, rc, "fused_bind failed: %s", cudaGetErrorString(cudaGetLastError()));
  return m2r2_reset(x);
}

extern "C" int m2r2_reset(m2r2_ctx* x) {
  if (!x) return M2R2_INVALID_ARG;
  CU(x, cudaMemsetAsync(x->d_kv_len, 0, sizeof(int) * x->c.max_batch, x->cs));
  CU(x, cudaMemsetAsync(x->d_pending, 0, sizeof(int) * x->c.max_batch, x->cs));
  CU(x, cudaStreamSynchronize(x->cs));
  memset(x->kv_h, 0, sizeof(x->kv_h));
  x->have_pending = false;
  x->B = 0;
  int64_t launches = x->st.kernel_launches;
  memset(&x->st, 0, sizeof(x->st));
  x->st.kernel_launches = launches;
  if (x->weights_loaded && x->c.n_experts) return reset_expert_cache(x);
  return M2R2_OK;
}

// counter-based generator of the random-speculation policy (the oracle implements the same function on its side)
static uint64_t spec_mix(uint64_t counter) {
  uint64_t v = 0x5EC0DE5EEDull + 0x9E3779B97F4A7C15ull * (counter + 1);
  v = (v ^ (v >> 30)) * 0xBF58476D1CE4E5B9ull;
  v = (v ^ (v >> 27)) * 0x94D049BB133111EBull;
  return v ^ (v >> 31);
}

// ------------------------------------------------------------------ MoE cache (host side, A15/A16)
static void lru_touch(std::vector<int>& q, int e) {
  auto it = std::find(q.begin(), q.end(), e);
  if (it != q.end()) q.erase(it);
  q.insert(q.begin(), e);
}
// make expert e resident in cache[layer] (never evicting `keep`); enqueue the H2D copy on `st`.
// returns 1 if a copy was enqueued, 0 if already resident, <0 on error.
static int cache_insert(m2r2_ctx* x, int layer, int e, const int* keep, int nk, cudaStream_t st) {
  if (x->slot_of[layer][e] >= 0) { lru_touch(x->lru[layer], e); return 0; }
  auto& q = x->lru[layer];
  int victim = -1;
  for (int s = (int)q.size() - 1; s >= 0 && victim < 0; --s) {
    bool kept = false;
    for (int k = 0; k < nk; ++k) kept |= (keep[k] == q[s]);
    if (!kept) victim = q[s];
  }
  if (victim < 0) victim = q.back();
  int slot = x->slot_of[layer][victim];
  // the slot may still be read by this layer's expert kernels of an earlier step
  if (cudaStreamWaitEvent(st, x->ev_layer_done[layer], 0) != cudaSuccess) return M2R2_CUDA;
  x->slot_of[layer][victim] = -1;
  q.erase(std::find(q.begin(), q.end(), victim));
  x->slot_of[layer][e] = slot;
  x->slot_expert[layer][slot] = e;
  q.insert(q.begin(), e);
  int rc = copy_expert(x, layer, e, slot_ptr(x, layer, slot), st);
  if (rc) return rc;
  return 1;
}

static int prefetch_pairs(m2r2_ctx* x, const int* pairs, int n) {
  // group by layer so that "never evict an expert predicted in the same event" holds
  int issued = 0;
  for (int i = 0; i < n;) {
    int layer = pairs[2 * i];
    int keep[M2R2_MAX_EXPERTS], nk = 0, j = i;
    while (j < n && pairs[2 * j] == layer && nk < M2R2_MAX_EXPERTS) keep[nk++] = pairs[2 * j++ + 1];
    bool any = false;
    for (int k = 0; k < nk; ++k) {
      int rc = cache_insert(x, layer, keep[k], keep, nk, x->cps);
      if (rc < 0) return rc;
      if (rc) { ++issued; any = true; x->st.expert_prefetched++; }
    }
    if (any) {
      if (cudaEventRecord(x->ev_copy_done[layer], x->cps) != cudaSuccess) return M2R2_CUDA;
      x->copy_pending[layer] = 1;
    }
    i = j;
  }
  return issued;
}

// ------------------------------------------------------------------ forward pass (per-operation kernels)
// mma: the tensor-core kernel of the k-token / dual-row attention (attn_mma_kernel: 2 CTAs of 4 warps per SM) takes the pass
static int n_splits_for(const m2r2_ctx* x, int groups, int max_len, bool mma = false) {
  const int items = x->c.n_heads * groups;
  int want = (4 * x->sm_count + items - 1) / items;
  // attn_mma_kernel: one wave of CTAs, rounded to the nearest count: at C4 (256 items, 296 slots) 1 / 2 / 3 / 4 / 8 splits
  // run a spec_step in 14.39 / 14.88 / 15.05 / 15.31 / 16.17 ms (every split pays its prologue, its partials and the merge)
  if (mma) want = std::max(1, (2 * x->sm_count + items / 2) / items);
  int cap = std::max(1, (max_len + 127) / 128);   // >= 128 positions per split: shorter items are all prologue and merge
  static const int force = xknob("M2R2_XSPLITS", 0);
  if (force > 0) return std::min(force, (int)M2R2_MAX_SPLITS);
  return std::max(1, std::min(std::min(want, cap), M2R2_MAX_SPLITS));
}

struct Pass {
  int mode;        // MODE_*
  int m;           // rows per sequence (verify / prefill)
  int joff;        // dual: draft offset
  int c0;          // prefill: first position of the chunk
  int n_layers;    // layers to run: [0, n_layers)
  bool accel;      // carry the accelerated stream
  bool trace;      // write h_i / p_i traces
  bool use_force;
  bool count_events;  // MoE: count cache events (off during prefill)
  bool draft;         // the gate at n_layers is the draft head: token -> drafts[joff]
};

static inline void count(m2r2_ctx* x, int n = 1) { x->st.kernel_launches += n; }

// exit / draft head on the accelerated rows: argmax(W_lm rms(p; g_f) + B_lm(A_lm .) + bias)
static int exit_head(m2r2_ctx* x, int B, int ns, float* logits_out, int* tok_out, int tok_stride) {
  const m2r2_config& c = x->c;
  const int d = c.d_model, V = c.vocab, r = c.adapter_rank;
  bool ad = x->lm_A != nullptr;
  prof_mark(x, M2R2_PROF_HEAD);
  // norm only the accelerated rows [ns, ns+B)
  launch_norm_lora(x->cs, c.dtype, x->resid + (size_t)ns * d, B, d, x->gf, c.rms_eps, x->xn + (size_t)ns * d,
                   ad ? x->lm_A : nullptr, 1, r, 0, x->U + (size_t)ns * 64, 64);
  GemvArgs g;
  memset(&g, 0, sizeof(g));
  g.W = x->lm_head; g.X = x->xn + (size_t)ns * d; g.ldx = d; g.n_rows = B; g.K = d; g.n_out = V;
  g.out = logits_out; g.ldo = V;
  if (ad) { g.Bm = x->lm_B; g.U = x->U + (size_t)ns * 64; g.ldu = 64; g.r = r; g.lora_row0 = 0; }
  // bf16 dense models with the fragment-major copy bound: the skinny tensor-core GEMM, adapter in its epilogue
  const bool mma_rows = B <= 64 && c.dtype == M2R2_BF16 && !c.n_experts && x->fused && fused_supported(c, &x->fs);
  if (!mma_rows || fused_gemv_rows(c, &x->fs, x->cs, 0, 4, g.X, d, B, logits_out, V, nullptr, nullptr, ad ? &g : nullptr))
    launch_gemv(x->cs, c.dtype, g, false);
  launch_argmax(x->cs, logits_out, V, B, V, x->d_row_seq + ns, x->d_row_pos + ns,
                x->ls_on ? x->d_ls_draft : nullptr, x->ls_first, x->ls_n, x->ls_beta, tok_out, tok_stride);
  count(x, 3);
  return 0;
}

static int moe_mlp(m2r2_ctx* x, const Pass& p, int i, int ns, int na);
static int moe_prefill(m2r2_ctx* x, int P);

static int run_pass(m2r2_ctx* x, const Pass& p) {
  const m2r2_config& c = x->c;
  const int B = x->B, d = c.d_model, dh = c.head_dim, nh = c.n_heads, r = c.adapter_rank;
  const int da = c.n_accel_heads * dh;
  const bool dual = p.mode == MODE_DUAL;
  const int ns = dual ? B : B * p.m;
  prof_mark(x, M2R2_PROF_OTHER);
  setup_rows_kernel<<<B, 32, 0, x->cs>>>(p.mode, B, p.m, p.joff, p.c0, c.max_seq, x->d_kv_len, x->d_pending,
                                         x->d_drafts, p.use_force ? x->d_force : nullptr, x->d_prompt,
                                         x->d_row_tok, x->d_row_seq, x->d_row_pos, x->d_row_limit, x->d_grp_rows);
  const bool any_accel = dual && p.accel && c.accel_enabled && c.accel_end_layer > 0;
  // slow-stream rows only, at most 8 of them, bf16 dense model with the fragment-major copy bound: the skinny
  // tensor-core GEMM (kernels_fused.cu) reads each weight once for all rows (a11)
  // (dual passes at batch >= 5 have 9..32 rows: the same kernel carries the accelerated rows' adapters)
  const bool mma_rows = ((!dual && ns <= 64) || (dual && 2 * B > 8 && 2 * B <= 64)) && c.dtype == M2R2_BF16 && !c.n_experts && x->fused && fused_supported(c, &x->fs);
  static const bool no_ring_fuse = xknob("M2R2_XNOFUSE", 0) != 0, no_merge_fuse = xknob("M2R2_XNOMERGEFUSE", 0) != 0;
  float* tr0 = p.trace ? x->trace : nullptr;
  launch_embed(x->cs, c.dtype, x->embed, x->d_row_tok, ns, d, x->resid, any_accel ? x->resid + (size_t)ns * d : nullptr,
               tr0, (tr0 && dual) ? tr0 + (size_t)B * d : nullptr);
  count(x, 2);
  int max_len = 0;
  for (int b = 0; b < B; ++b) max_len = std::max(max_len, x->kv_h[b]);
  max_len += (dual ? p.joff + 1 : (p.mode == MODE_VERIFY ? p.m : p.c0 + p.m));
  const int splits = n_splits_for(x, B, max_len, c.dtype == M2R2_BF16 && (dual ? 2 : p.m) >= 2 && (dh == 64 || dh == 96 || dh == 128));
  const float scale = 1.0f / sqrtf((float)dh);

  for (int i = 0; i < p.n_layers; ++i) {
    const DevLayer& L = x->L[i];
    const bool acc_on = any_accel && layer_accel(c, i);
    const int na = acc_on ? B : 0, rows = ns + na;
    char* Kc = (char*)x->b.kv + (size_t)i * c.max_batch * nh * c.max_seq * dh * x->esz;
    char* Vc = Kc + (size_t)c.n_layers * c.max_batch * nh * c.max_seq * dh * x->esz;
    // a2: RMSNorm + QKV (slow: all heads; accelerated: heads in S + adapters)
    prof_mark(x, M2R2_PROF_QKV);
    // <= 8 slow rows (the verify pass and prefill chunks at batch 1): the ring GEMM absorbs the layer's small kernels
    // (RMSNorm in its staging, RoPE + KV append in the QKV epilogue)
    const bool ring_fuse = mma_rows && !acc_on && rows <= 8 && !no_ring_fuse;
    int saved = 0;   // launches the fusion removed
    GemvArgs g;
    bool qkv_done = false;
    if (ring_fuse) {
      RowsFuse fz;
      fz.gain = L.g1; fz.eps = c.rms_eps; fz.row_seq = x->d_row_seq; fz.row_pos = x->d_row_pos; fz.rope_tab = x->rope_tab;
      fz.Kc = Kc; fz.Vc = Vc;
      qkv_done = fused_gemv_rows(c, &x->fs, x->cs, i, 0, x->resid, d, rows, x->qkv, 3 * d, nullptr, nullptr, nullptr, &fz) == 0;
      if (qkv_done) saved += 2;
    }
    if (!qkv_done) {
      // passes with more than 8 rows: the norm also leaves the rows as (hi, lo) words for the tensor-core GEMM
      int pk_ld = 0;
      uint2* pk = (mma_rows && rows > 8 && !no_ring_fuse) ? fused_xn_pack(&x->fs, &pk_ld) : nullptr;
      launch_norm_lora(x->cs, c.dtype, x->resid, rows, d, L.g1, c.rms_eps, x->xn, acc_on ? L.Aqkv : nullptr, 3, r, ns, x->U, 64, pk, pk_ld);
      memset(&g, 0, sizeof(g));
      g.W = L.wqkv; g.X = x->xn; g.ldx = d; g.n_rows = rows; g.K = d; g.n_out = 3 * d; g.out = x->qkv; g.ldo = 3 * d;
      if (acc_on) { g.Bm = L.Bqkv; g.bmap = x->d_qkv_bmap; g.U = x->U; g.ldu = 64; g.r = r; g.lora_row0 = ns; g.usel_div = d; }
      bool roped = false;
      if (mma_rows && rows > 8 && !no_ring_fuse) {
        // batched passes: RoPE + KV append in the tensor-core GEMM's epilogue
        RowsFuse fz;
        fz.row_seq = x->d_row_seq; fz.row_pos = x->d_row_pos; fz.rope_tab = x->rope_tab; fz.Kc = Kc; fz.Vc = Vc; fz.slow_rows = ns;
        fz.x_packed = pk != nullptr;
        roped = fused_gemv_rows(c, &x->fs, x->cs, i, 0, x->xn, d, rows, x->qkv, 3 * d, nullptr, nullptr, acc_on ? &g : nullptr, &fz) == 0;
        if (roped) saved += 1;
      }
      if (!roped) {
        if (!mma_rows || fused_gemv_rows(c, &x->fs, x->cs, i, 0, x->xn, d, rows, x->qkv, 3 * d, nullptr, nullptr, acc_on ? &g : nullptr)) launch_gemv(x->cs, c.dtype, g, false);
        // a3: RoPE + KV append
        prof_mark(x, M2R2_PROF_ROPE);
        launch_rope_append(x->cs, c.dtype, x->qkv, rows, ns, x->d_row_seq, x->d_row_pos, x->rope_tab, Kc, Vc, nh, dh, c.max_seq);
      }
    }
    // a4: split-K attention + merge
    prof_mark(x, M2R2_PROF_ATTN);
    AttnArgs a;
    memset(&a, 0, sizeof(a));
    a.qkv = x->qkv; a.Kc = Kc; a.Vc = Vc; a.row_seq = x->d_row_seq; a.row_limit = x->d_row_limit;
    a.grp_rows = x->d_grp_rows; a.part_o = x->part_o; a.part_ml = x->part_ml;
    a.n_heads = nh; a.dh = dh; a.d = d; a.max_seq = c.max_seq; a.n_splits = splits; a.slow_rows = acc_on ? ns : (1 << 30);
    memcpy(a.accel_head_mask, x->accel_mask, sizeof(a.accel_head_mask));
    a.scale = scale;
    // PAPER.md L158 / L170: with accel_topk_tokens the accelerated rows attend the slow stream's top-k positions in their own kernel
    const bool topk_accel = acc_on && c.accel_topk_tokens > 0;
    if ((!acc_on && dual) || topk_accel) {
      // groups still list the accelerated rows; hide them by marking every row as slow-limited
      a.slow_rows = ns;
      memset(a.accel_head_mask, 0, sizeof(a.accel_head_mask));
    }
    // slow rows only (verify, prefill) and one split: the tensor-core kernel writes the merged output itself
    if (!dual && splits == 1) a.direct_out = x->attn_o;
    const bool merged = launch_attn(x->cs, c.dtype, a, B, dual ? 2 : p.m);
    if (merged) saved += 1;
    MergeArgs mg;
    memset(&mg, 0, sizeof(mg));
    mg.qkv = x->qkv; mg.part_o = x->part_o; mg.part_ml = x->part_ml; mg.row_limit = x->d_row_limit; mg.out = x->attn_o;
    mg.n_heads = nh; mg.dh = dh; mg.d = d; mg.n_splits = splits; mg.slow_rows = ns;
    memcpy(mg.accel_head_mask, x->accel_mask, sizeof(mg.accel_head_mask));
    if (topk_accel) memset(mg.accel_head_mask, 0, sizeof(mg.accel_head_mask));   // accelerated rows: zero here, S heads written below
    mg.scale = scale;
    // (verify / prefill rows at batch 1: the O ring GEMM merges the splits while it stages its inputs)
    bool o_done = false;
    if (ring_fuse && !no_merge_fuse && !merged) {
      RowsFuse fz;
      fz.part_o = x->part_o; fz.part_ml = x->part_ml; fz.n_splits = splits;
      o_done = fused_gemv_rows(c, &x->fs, x->cs, i, 1, x->attn_o, d, rows, x->resid, d, x->resid, nullptr, nullptr, &fz) == 0;
      if (o_done) saved += 1;
    }
    if (!o_done && !merged) launch_merge(x->cs, mg, rows);
    if (topk_accel) {
      launch_accel_topk_attn(x->cs, c.dtype, x->qkv, Kc, Vc, x->d_row_limit, x->d_accel_heads, c.n_accel_heads, x->attn_o, B, nh, dh, d,
                             c.max_seq, c.accel_topk_tokens, scale);
      count(x);
    }
    count(x, 5 - saved);
    // a5: O-proj + residual
    prof_mark(x, M2R2_PROF_OPROJ);
    if (acc_on) { launch_lora_down(x->cs, c.dtype, x->attn_o, d, ns, na, da, x->d_accel_cols, L.Ao, r, x->U, 64); count(x); }
    if (!o_done) {
      memset(&g, 0, sizeof(g));
      g.W = L.wo; g.X = x->attn_o; g.ldx = d; g.n_rows = rows; g.K = d; g.n_out = d; g.out = x->resid; g.ldo = d; g.resid = x->resid;
      if (acc_on) { g.Bm = L.Bo; g.U = x->U; g.ldu = 64; g.r = r; g.lora_row0 = ns; }
      if (!mma_rows || fused_gemv_rows(c, &x->fs, x->cs, i, 1, x->attn_o, d, rows, x->resid, d, x->resid, nullptr, acc_on ? &g : nullptr)) launch_gemv(x->cs, c.dtype, g, false);
    }
    count(x);
    float* trl = p.trace ? x->trace + (size_t)(i + 1) * 2 * B * d : nullptr;
    if (!c.n_experts) {
      // a6: RMSNorm + gate/up + SwiGLU;  a7: down + residual (accelerated-residual update)
      prof_mark(x, M2R2_PROF_GATEUP);
      bool gu_done = false, act_packed = false;
      if (ring_fuse) {
        RowsFuse fz;
        fz.gain = L.g2; fz.eps = c.rms_eps;
        gu_done = fused_gemv_rows(c, &x->fs, x->cs, i, 2, x->resid, d, rows, x->act, c.d_ff, nullptr, nullptr, nullptr, &fz) == 0;
      }
      if (!gu_done) {
        int pk_ld = 0;
        uint2* pk = (mma_rows && rows > 8 && !no_ring_fuse) ? fused_xn_pack(&x->fs, &pk_ld) : nullptr;
        launch_norm_lora(x->cs, c.dtype, x->resid, rows, d, L.g2, c.rms_eps, x->xn, acc_on ? L.Agu : nullptr, 2, r, ns, x->U, 64, pk, pk_ld);
        memset(&g, 0, sizeof(g));
        g.W = L.wgate; g.W2 = L.wup; g.X = x->xn; g.ldx = d; g.n_rows = rows; g.K = d; g.n_out = c.d_ff; g.out = x->act; g.ldo = c.d_ff;
        if (acc_on) { g.Bm = L.Bg; g.Bm2 = L.Bu; g.U = x->U; g.ldu = 64; g.r = r; g.lora_row0 = ns; }
        if (pk) {
          // rows already packed by the norm; the epilogue leaves the activations packed for the down projection
          RowsFuse fz;
          fz.x_packed = true; fz.pack_out = true;
          act_packed = fused_gemv_rows(c, &x->fs, x->cs, i, 2, x->xn, d, rows, x->act, c.d_ff, nullptr, nullptr, acc_on ? &g : nullptr, &fz) == 0;
        }
        if (!act_packed && (!mma_rows || fused_gemv_rows(c, &x->fs, x->cs, i, 2, x->xn, d, rows, x->act, c.d_ff, nullptr, nullptr, acc_on ? &g : nullptr))) launch_gemv(x->cs, c.dtype, g, true);
      }
      prof_mark(x, M2R2_PROF_DOWN);
      if (acc_on) { launch_lora_down(x->cs, c.dtype, x->act, c.d_ff, ns, na, c.d_ff, nullptr, L.Ad, r, x->U, 64); count(x); }
      memset(&g, 0, sizeof(g));
      g.W = L.wdown; g.X = x->act; g.ldx = c.d_ff; g.n_rows = rows; g.K = c.d_ff; g.n_out = d; g.out = x->resid; g.ldo = d; g.resid = x->resid;
      g.trace = trl;
      if (acc_on) { g.Bm = L.Bd; g.U = x->U; g.ldu = 64; g.r = r; g.lora_row0 = ns; }
      bool down_done = false;
      if (act_packed) {
        RowsFuse fz;
        fz.x_packed = true;
        down_done = fused_gemv_rows(c, &x->fs, x->cs, i, 3, x->act, c.d_ff, rows, x->resid, d, x->resid, trl, acc_on ? &g : nullptr, &fz) == 0;
      }
      if (!down_done && (!mma_rows || fused_gemv_rows(c, &x->fs, x->cs, i, 3, x->act, c.d_ff, rows, x->resid, d, x->resid, trl, acc_on ? &g : nullptr))) launch_gemv(x->cs, c.dtype, g, false);
      count(x, gu_done ? 2 : 3);
    } else {
      int rc = moe_mlp(x, p, i, ns, na);
      if (rc) return rc;
      if (trl) { launch_copy_rows(x->cs, x->resid, trl, rows, d); count(x); }
    }
    prof_mark(x, M2R2_PROF_OTHER);
    if (trl && dual && !acc_on) { launch_copy_rows(x->cs, x->resid, trl + (size_t)B * d, B, d); count(x); }
    // gate: exit prediction on p (Eq. 4) then p <- h (L82, L101)
    if (acc_on) {
      int gj = -1;
      for (int j = 0; j < c.n_gates; ++j) if (c.gates[j] == i + 1) gj = j;
      if (gj >= 0) {
        if (p.draft && p.n_layers == i + 1)
          exit_head(x, B, ns, x->exit_logits + (size_t)gj * B * c.vocab, x->d_drafts + p.joff, 8);
        else if (c.exit_heads_enabled || p.n_layers == i + 1)
          exit_head(x, B, ns, x->exit_logits + (size_t)gj * B * c.vocab, x->d_exit_tok + gj, c.n_gates);
        launch_copy_rows(x->cs, x->resid, x->resid + (size_t)ns * d, B, d);
        count(x);
      }
    }
  }
  return 0;
}

// final head on the slow rows -> tokens (a9)
static int final_head(m2r2_ctx* x, int ns, int* tok_out, int tok_stride) {
  const m2r2_config& c = x->c;
  const int d = c.d_model, V = c.vocab;
  prof_mark(x, M2R2_PROF_HEAD);
  const bool mma_rows = ns <= 64 && c.dtype == M2R2_BF16 && !c.n_experts && x->fused && fused_supported(c, &x->fs);
  bool done = false;
  if (mma_rows && ns <= 8) {
    RowsFuse fz;   // RMSNorm inside the ring GEMM's staging
    fz.gain = x->gf; fz.eps = c.rms_eps;
    done = fused_gemv_rows(c, &x->fs, x->cs, 0, 4, x->resid, d, ns, x->logits, V, nullptr, nullptr, nullptr, &fz) == 0;
  }
  if (!done) {
    launch_norm_lora(x->cs, c.dtype, x->resid, ns, d, x->gf, c.rms_eps, x->xn, nullptr, 0, 0, 0, x->U, 64);
    GemvArgs g;
    memset(&g, 0, sizeof(g));
    g.W = x->lm_head; g.X = x->xn; g.ldx = d; g.n_rows = ns; g.K = d; g.n_out = V; g.out = x->logits; g.ldo = V;
    if (!mma_rows || fused_gemv_rows(c, &x->fs, x->cs, 0, 4, x->xn, d, ns, x->logits, V, nullptr, nullptr)) launch_gemv(x->cs, c.dtype, g, false);
    count(x);
  }
  launch_argmax(x->cs, x->logits, V, ns, V, x->d_row_seq, x->d_row_pos, x->ls_on ? x->d_ls_full : nullptr,
                x->ls_first, x->ls_n, x->ls_beta, tok_out, tok_stride);
  count(x, 2);
  return 0;
}

// ------------------------------------------------------------------ MoE layer (a13-a17)
static int expert_ffn(m2r2_ctx* x, const void* blob, int row, int n_rows, const float* scale, int scale_ld,
                      bool first, bool last) {
  const m2r2_config& c = x->c;
  const int d = c.d_model, F = c.d_ff_expert;
  const char* p = (const char*)blob;
  GemvArgs g;
  memset(&g, 0, sizeof(g));
  g.W = p; g.W2 = p + x->eg_bytes; g.X = x->xn + (size_t)row * d; g.ldx = d; g.n_rows = n_rows; g.K = d; g.n_out = F;
  g.out = x->act + (size_t)row * fmax_act(c); g.ldo = fmax_act(c);
  prof_mark(x, M2R2_PROF_GATEUP);
  launch_gemv(x->cs, c.dtype, g, true);
  prof_mark(x, M2R2_PROF_DOWN);
  memset(&g, 0, sizeof(g));
  g.W = p + 2 * x->eg_bytes; g.X = x->act + (size_t)row * fmax_act(c); g.ldx = fmax_act(c); g.n_rows = n_rows; g.K = F; g.n_out = d;
  g.ldo = d; g.scale = scale; g.scale_ld = scale_ld;
  float* tmp = x->moe_tmp + (size_t)row * d;
  float* res = x->resid + (size_t)row * d;
  if (!first) g.addin = tmp;
  if (last) { g.out = res; g.resid = res; } else g.out = tmp;
  launch_gemv(x->cs, c.dtype, g, false);
  count(x, 2);
  return 0;
}

static int moe_mlp(m2r2_ctx* x, const Pass& p, int i, int ns, int na) {
  const m2r2_config& c = x->c;
  const DevLayer& L = x->L[i];
  const int d = c.d_model, tk = c.top_k, rows = ns + na;
  if (ns != 1) return fail(x, M2R2_UNSUPPORTED, "MoE layers run one slow row per pass (prefill streams experts separately)");
  prof_mark(x, M2R2_PROF_OTHER);
  launch_norm_lora(x->cs, c.dtype, x->resid, rows, d, L.g2, c.rms_eps, x->xn, nullptr, 0, 0, 0, x->U, 64);
  count(x);
  // accelerated rows: fixed adapter MLP  m^ = U_d (silu(U_g y^) * (U_u y^))   (L137, Q7)
  if (na) {
    GemvArgs g;
    memset(&g, 0, sizeof(g));
    const int rm = c.accel_mlp_rank, fa = fmax_act(c);
    g.W = L.Ug; g.W2 = L.Uu; g.X = x->xn + (size_t)ns * d; g.ldx = d; g.n_rows = na; g.K = d; g.n_out = rm;
    g.out = x->act + (size_t)ns * fa; g.ldo = fa;
    launch_gemv(x->cs, c.dtype, g, true);
    memset(&g, 0, sizeof(g));
    g.W = L.Ud; g.X = x->act + (size_t)ns * fa; g.ldx = fa; g.n_rows = na; g.K = rm; g.n_out = d;
    g.out = x->resid + (size_t)ns * d; g.ldo = d; g.resid = x->resid + (size_t)ns * d;
    launch_gemv(x->cs, c.dtype, g, false);
    count(x, 2);
    // a14: expert predictor on p_{i+1} for this source layer's targets -> pinned host
    if (x->policy == M2R2_POLICY_LRU_AOT && c.aot_lo[i] < c.aot_hi[i] && p.count_events) {
      for (int Lt = c.aot_lo[i]; Lt < c.aot_hi[i]; ++Lt) {
        launch_route(x->cs, c.dtype, x->resid + (size_t)ns * d, d, 1, d, x->L[Lt].g2, c.rms_eps, 1, x->L[Lt].router,
                     c.n_experts, tk, c.renorm_topk, x->d_row_pos + ns, x->rs_on ? x->d_rs_pred : nullptr, x->rs_first,
                     x->rs_n, c.n_layers, Lt, x->rs_beta, x->d_pred_idx + Lt * tk, x->pred_w + Lt * tk);
        count(x);
      }
      int nt = c.aot_hi[i] - c.aot_lo[i];
      CU(x, cudaMemcpyAsync(x->h_pinned + 1024, x->d_pred_idx + c.aot_lo[i] * tk, sizeof(int) * nt * tk, cudaMemcpyDeviceToHost, x->cs));
      CU(x, cudaEventRecord(x->ev_tmp, x->cs));
      CU(x, cudaEventSynchronize(x->ev_tmp));
      std::vector<int> pairs;
      for (int t = 0; t < nt; ++t)
        for (int k = 0; k < tk; ++k) { pairs.push_back(c.aot_lo[i] + t); pairs.push_back(x->h_pinned[1024 + t * tk + k]); }
      int rc = prefetch_pairs(x, pairs.data(), (int)pairs.size() / 2);
      if (rc < 0) return fail(x, rc, "prefetch failed");
    }
  }
  // a13: router + top-k on the slow rows
  launch_route(x->cs, c.dtype, x->xn, d, ns, d, nullptr, 0.f, 0, L.router, c.n_experts, tk, c.renorm_topk, x->d_row_pos,
               x->rs_on ? x->d_rs_actual : nullptr, x->rs_first, x->rs_n, c.n_layers, i, x->rs_beta,
               x->d_route_idx + i * tk, x->route_w + i * tk);
  count(x);
  // the host has to learn the routed experts to manage the cache (App. B)
  CU(x, cudaMemcpyAsync(x->h_pinned, x->d_route_idx + i * tk, sizeof(int) * tk, cudaMemcpyDeviceToHost, x->cs));
  CU(x, cudaEventRecord(x->ev_tmp, x->cs));
  CU(x, cudaEventSynchronize(x->ev_tmp));
  int idx[M2R2_MAX_TOPK];
  for (int k = 0; k < tk; ++k) idx[k] = x->h_pinned[k];
  const void* blob[M2R2_MAX_TOPK];
  bool waited_copy = false;
  for (int k = 0; k < tk; ++k) {
    int e = idx[k];
    if (x->policy == M2R2_POLICY_FIXED) {
      if (e < c.cache_slots_per_layer) { x->st.expert_hits++; blob[k] = slot_ptr(x, i, e); }
      else {
        x->st.expert_misses++; x->st.expert_on_demand++;
        // staging slot k: wait until the previous layer's kernels stopped reading it
        CU(x, cudaStreamWaitEvent(x->ods, x->ev_stage_free, 0));
        int rc = copy_expert(x, i, e, stage_ptr(x, k), x->ods);
        if (rc) return rc;
        CU(x, cudaEventRecord(x->ev_tmp, x->ods));
        CU(x, cudaStreamWaitEvent(x->cs, x->ev_tmp, 0));
        blob[k] = stage_ptr(x, k);
      }
    } else {
      bool hit = x->slot_of[i][e] >= 0;
      if (hit) { x->st.expert_hits++; lru_touch(x->lru[i], e); }
      else {
        x->st.expert_misses++; x->st.expert_on_demand++;
        // prioritized on-demand load (L387): own high-priority stream, after any in-flight prefetch of this layer
        if (x->copy_pending[i]) CU(x, cudaStreamWaitEvent(x->ods, x->ev_copy_done[i], 0));
        int rc = cache_insert(x, i, e, idx, tk, x->ods);
        if (rc < 0) return fail(x, rc, "on-demand load failed");
        CU(x, cudaEventRecord(x->ev_tmp, x->ods));
        CU(x, cudaStreamWaitEvent(x->cs, x->ev_tmp, 0));
      }
      if (x->copy_pending[i] && !waited_copy) {   // prefetched experts may still be in flight
        CU(x, cudaStreamWaitEvent(x->cs, x->ev_copy_done[i], 0));
        waited_copy = true;
      }
      blob[k] = slot_ptr(x, i, x->slot_of[i][e]);
    }
  }
  x->copy_pending[i] = 0;
  // a16: grouped expert GEMV, y = sum_k w_k * Expert_k(x), selection order
  for (int k = 0; k < tk; ++k)
    expert_ffn(x, blob[k], 0, 1, x->route_w + i * tk + k, 0, k == 0, k == tk - 1);
  CU(x, cudaEventRecord(x->ev_layer_done[i], x->cs));
  if (x->policy == M2R2_POLICY_FIXED) CU(x, cudaEventRecord(x->ev_stage_free, x->cs));
  // the two comparison strategies of PAPER.md L242 that speculate ONE layer ahead (L244), through the same prefetch machinery
  if (p.count_events && i + 1 < c.n_layers && (x->policy == M2R2_POLICY_LRU_RANDOM || x->policy == M2R2_POLICY_LRU_PREV)) {
    const int Lt = i + 1;
    int pairs[2 * M2R2_MAX_TOPK];
    if (x->policy == M2R2_POLICY_LRU_RANDOM) {
      // top_k distinct experts, draw d of (position t, layer Lt) = spec_mix((t * N + Lt) * 256 + d) mod n_experts
      const uint64_t t = (uint64_t)x->kv_h[0] + (uint64_t)p.joff;
      int n = 0;
      for (int dr = 0; n < tk && dr < 256; ++dr) {
        const int e = (int)(spec_mix((t * (uint64_t)c.n_layers + (uint64_t)Lt) * 256u + (uint64_t)dr) % (uint64_t)c.n_experts);
        bool dup = false;
        for (int k = 0; k < n; ++k) dup |= pairs[2 * k + 1] == e;
        if (!dup) { pairs[2 * n] = Lt; pairs[2 * n + 1] = e; ++n; }
      }
      for (int k = 0; k < tk; ++k) x->h_pinned[2048 + k] = pairs[2 * k + 1];
      CU(x, cudaMemcpyAsync(x->d_pred_idx + Lt * tk, x->h_pinned + 2048, sizeof(int) * tk, cudaMemcpyHostToDevice, x->cs));
      CU(x, cudaEventRecord(x->ev_tmp, x->cs));
      CU(x, cudaEventSynchronize(x->ev_tmp));   // the pinned staging words are reused by the next layer
    } else {
      // the router of layer i + 1 on the slow residual h_{i+1} this layer just produced
      launch_route(x->cs, c.dtype, x->resid, d, 1, d, x->L[Lt].g2, c.rms_eps, 1, x->L[Lt].router, c.n_experts, tk, c.renorm_topk,
                   x->d_row_pos, x->rs_on ? x->d_rs_pred : nullptr, x->rs_first, x->rs_n, c.n_layers, Lt, x->rs_beta,
                   x->d_pred_idx + Lt * tk, x->pred_w + Lt * tk);
      count(x);
      CU(x, cudaMemcpyAsync(x->h_pinned + 1024, x->d_pred_idx + Lt * tk, sizeof(int) * tk, cudaMemcpyDeviceToHost, x->cs));
      CU(x, cudaEventRecord(x->ev_tmp, x->cs));
      CU(x, cudaEventSynchronize(x->ev_tmp));
      for (int k = 0; k < tk; ++k) { pairs[2 * k] = Lt; pairs[2 * k + 1] = x->h_pinned[1024 + k]; }
    }
    int rc = prefetch_pairs(x, pairs, tk);
    if (rc < 0) return fail(x, rc, "prefetch failed");
  }
  return 0;
}

// ------------------------------------------------------------------ ABI: prefill / decode / spec
static int check_ready(m2r2_ctx* x) {
  if (!x) return M2R2_INVALID_ARG;
  if (!x->weights_loaded) return fail(x, M2R2_BAD_STATE, "load_weights has not been called");
  // a fused launch whose device-side wait timed out left no sequence state behind; report it from whichever
  // call comes next (also when the caller never asked for tokens) and re-arm the kernel
  if (fused_abort_pending(&x->fs)) {
    int rc = fused_check(&x->fs, x->cs, x->err, sizeof(x->err));
    if (rc) return rc;
  }
  return 0;
}

static int64_t layer_bytes(const m2r2_ctx* x, int i, bool accel, int kv_positions) {
  const m2r2_config& c = x->c;
  int64_t d = c.d_model, F = c.d_ff, r = c.adapter_rank, e = (int64_t)x->esz;
  int64_t da = (int64_t)c.n_accel_heads * c.head_dim;
  int64_t w = 4 * d * d;
  if (!c.n_experts) w += 3 * d * F; else w += (int64_t)c.top_k * 3 * d * c.d_ff_expert + (int64_t)c.n_experts * d;
  if (accel && layer_accel(c, i)) {
    w += 3 * (r * d + da * r) + r * da + d * r;
    if (!c.n_experts) w += 2 * (r * d + F * r) + r * F + d * r; else w += 3 * (int64_t)c.accel_mlp_rank * d;
  }
  return (w + 2 * d * (int64_t)kv_positions) * e;
}

extern "C" int m2r2_prefill(m2r2_ctx* x, const int32_t* tokens, int32_t B, int32_t P, int32_t* first_tokens) {
  int rc = check_ready(x);
  if (rc) return rc;
  const m2r2_config& c = x->c;
  if (!tokens || B < 1 || B > c.max_batch || P < 1 || P > c.max_seq) return fail(x, M2R2_INVALID_ARG, "prefill: bad B/P");
  for (int64_t i = 0; i < (int64_t)B * P; ++i)
    if (tokens[i] < 0 || tokens[i] >= c.vocab) return fail(x, M2R2_INVALID_ARG, "prefill: token out of range");
  rc = m2r2_reset(x);
  if (rc) return rc;
  x->B = B;
  for (int b = 0; b < B; ++b)
    CU(x, cudaMemcpyAsync(x->d_prompt + (size_t)b * c.max_seq, tokens + (size_t)b * P, sizeof(int) * P, cudaMemcpyHostToDevice, x->cs));
  if (c.n_experts) {
    rc = moe_prefill(x, P);
    if (rc) return rc;
  } else {
    for (int c0 = 0; c0 < P; c0 += 8) {
      Pass p = {MODE_PREFILL, std::min(8, P - c0), 0, c0, c.n_layers, false, false, false, false, false};
      for (int b = 0; b < B; ++b) x->kv_h[b] = c0;
      rc = run_pass(x, p);
      if (rc) return rc;
      if (c0 + p.m >= P) {
        // first token = argmax at position P-1 (rows b*m + m-1)
        final_head(x, B * p.m, x->d_vtok, 1);
        // gather the last row of each sequence
        for (int b = 0; b < B; ++b)
          CU(x, cudaMemcpyAsync(x->d_out_tok + b, x->d_vtok + b * p.m + p.m - 1, sizeof(int), cudaMemcpyDeviceToDevice, x->cs));
      }
    }
  }
  set_state_kernel<<<1, 32, 0, x->cs>>>(B, x->d_kv_len, x->d_pending, P, x->d_out_tok);
  count(x);
  CU(x, cudaMemcpyAsync(x->h_pinned, x->d_out_tok, sizeof(int) * B, cudaMemcpyDeviceToHost, x->cs));
  CU(x, cudaStreamSynchronize(x->cs));
  CU(x, cudaGetLastError());
  for (int b = 0; b < B; ++b) { x->kv_h[b] = P; if (first_tokens) first_tokens[b] = x->h_pinned[b]; }
  x->last_rows_per_seq = P - ((P - 1) / 8) * 8;   // rows per sequence of the last prefill chunk (debug_read LOGITS)
  x->have_pending = true;
  return M2R2_OK;
}

extern "C" int m2r2_decode_step(m2r2_ctx* x, const int32_t* force_tokens, int32_t* tokens_out, int32_t* exit_tokens_out) {
  int rc = check_ready(x);
  if (rc) return rc;
  const m2r2_config& c = x->c;
  if (!x->have_pending) return fail(x, M2R2_BAD_STATE, "decode_step before prefill");
  const int B = x->B;
  for (int b = 0; b < B; ++b)
    if (x->kv_h[b] + 1 > c.max_seq) return fail(x, M2R2_CAPACITY, "kv cache full");
  if (force_tokens) {
    for (int b = 0; b < B; ++b)
      if (force_tokens[b] < 0 || force_tokens[b] >= c.vocab) return fail(x, M2R2_INVALID_ARG, "force token out of range");
    const unsigned int slot = x->force_ctr++ % m2r2_ctx::FORCE_SLOTS;
    int* hs = x->h_force + (size_t)slot * M2R2_MAX_BATCH;
    CU(x, cudaEventSynchronize(x->ev_force[slot]));   // the copy that last used this slot has executed
    memcpy(hs, force_tokens, sizeof(int) * B);
    CU(x, cudaMemcpyAsync(x->d_force, hs, sizeof(int) * B, cudaMemcpyHostToDevice, x->cs));
    CU(x, cudaEventRecord(x->ev_force[slot], x->cs));
  }
  int64_t bytes = 0;
  for (int i = 0; i < c.n_layers; ++i)
    for (int b = 0; b < B; ++b) bytes += (b == 0 ? layer_bytes(x, i, true, 0) : 0) + 2 * (int64_t)c.d_model * (x->kv_h[b] + 1 + 1) * x->esz;   // read T+1, append 1
  bytes += (int64_t)c.vocab * c.d_model * x->esz * (1 + (c.exit_heads_enabled ? c.n_gates : 0)) + (int64_t)c.d_model * x->esz * B;
  x->st.algorithmic_bytes_last = bytes;

  const bool use_fused = x->fused && fused_supported(c, &x->fs) && B == 1 && c.accel_topk_tokens == 0;   // the fused kernel keeps p's attention dense
  if (use_fused) {
    prof_mark(x, M2R2_PROF_FUSED_STEP);
    FusedRun fr = {c.n_layers, 0, force_tokens ? x->d_force : x->d_pending, 0, x->d_out_tok, 1, c.exit_heads_enabled, 1};
    rc = fused_run(c, &x->fs, x->cs, fr, x->d_kv_len, x->d_pending, x->kv_h[0], x->trace, x->logits, x->exit_logits,
                   x->d_exit_tok, x->ls_on ? x->d_ls_full : nullptr, x->ls_on ? x->d_ls_draft : nullptr, x->ls_first,
                   x->ls_n, x->ls_beta, &x->st.kernel_launches);
    if (rc) return fail(x, rc, "fused decode launch failed: %s", cudaGetErrorString(cudaGetLastError()));
  } else {
    Pass p = {MODE_DUAL, 1, 0, 0, c.n_layers, true, true, force_tokens != nullptr, true, false};
    rc = run_pass(x, p);
    if (rc) return rc;
    final_head(x, B, x->d_out_tok, 1);
    advance_kernel<<<1, 32, 0, x->cs>>>(B, x->d_kv_len, x->d_pending, x->d_out_tok);
    count(x);
  }
  if (x->arla) {
    // f-3 ARLA mechanics: exit score of every gate from the step's traced accelerated residuals
    launch_arla(x->cs, c.dtype, x->trace, x->arla, c.gates, c.n_gates, c.arla_dim, c.d_model, B, x->exit_score);
    count(x);
  }
  prof_resolve(x);
  for (int b = 0; b < B; ++b) x->kv_h[b] += 1;
  x->st.steps++;
  x->st.emitted += B;
  x->last_rows_per_seq = 1;
  if (tokens_out || exit_tokens_out) {
    CU(x, cudaMemcpyAsync(x->h_pinned, x->d_out_tok, sizeof(int) * B, cudaMemcpyDeviceToHost, x->cs));
    if (exit_tokens_out && c.n_gates)
      CU(x, cudaMemcpyAsync(x->h_pinned + 64, x->d_exit_tok, sizeof(int) * B * c.n_gates, cudaMemcpyDeviceToHost, x->cs));
    CU(x, cudaStreamSynchronize(x->cs));
    CU(x, cudaGetLastError());
    if (use_fused && (rc = fused_check(&x->fs, x->cs, x->err, sizeof(x->err)))) return rc;
    if (tokens_out) memcpy(tokens_out, x->h_pinned, sizeof(int) * B);
    if (exit_tokens_out && c.n_gates) memcpy(exit_tokens_out, x->h_pinned + 64, sizeof(int) * B * c.n_gates);
  }
  return M2R2_OK;
}

extern "C" int m2r2_spec_step(m2r2_ctx* x, int32_t k, int32_t* accepted, int32_t* n_accepted) {
  int rc = check_ready(x);
  if (rc) return rc;
  const m2r2_config& c = x->c;
  if (!x->have_pending) return fail(x, M2R2_BAD_STATE, "spec_step before prefill");
  if (k < 0 || k > M2R2_MAX_DRAFT || !accepted || !n_accepted) return fail(x, M2R2_INVALID_ARG, "spec_step: bad k/outputs");
  if (c.n_experts) return fail(x, M2R2_UNSUPPORTED, "spec_step on MoE models");
  if (k > 0 && (!c.accel_enabled || c.n_gates < 1 || c.accel_end_layer < c.gates[0]))
    return fail(x, M2R2_INVALID_ARG, "spec_step: config has no draft gate");
  const int B = x->B, E = c.n_gates ? c.gates[0] : 0;
  for (int b = 0; b < B; ++b)
    if (x->kv_h[b] + k + 1 > c.max_seq) return fail(x, M2R2_CAPACITY, "kv cache full");
  int64_t bytes = 0;
  // a10: draft loop — k dependent passes of layers 0..E-1 (both streams) + draft head
  const bool use_fused = x->fused && fused_supported(c, &x->fs) && B == 1 && c.accel_topk_tokens == 0;
  for (int j = 0; j < k; ++j) {
    if (use_fused) {
      prof_mark(x, M2R2_PROF_FUSED_STEP);
      FusedRun fr = {E, j, j == 0 ? x->d_pending : x->d_drafts + (j - 1), 1, x->d_drafts + j, 0, 0, 0};
      rc = fused_run(c, &x->fs, x->cs, fr, x->d_kv_len, x->d_pending, x->kv_h[0], x->trace, x->logits, x->exit_logits,
                     x->d_exit_tok, x->ls_on ? x->d_ls_full : nullptr, x->ls_on ? x->d_ls_draft : nullptr, x->ls_first,
                     x->ls_n, x->ls_beta, &x->st.kernel_launches);
      if (rc) return fail(x, rc, "fused draft launch failed: %s", cudaGetErrorString(cudaGetLastError()));
    } else {
      Pass p = {MODE_DUAL, 1, j, 0, E, true, false, false, true, true};
      rc = run_pass(x, p);
      if (rc) return rc;
    }
    for (int i = 0; i < E; ++i)
      for (int b = 0; b < B; ++b) bytes += (b == 0 ? layer_bytes(x, i, true, 0) : 0) + 2 * (int64_t)c.d_model * (x->kv_h[b] + j + 1 + 1) * x->esz;
    bytes += (int64_t)c.vocab * c.d_model * x->esz;
  }
  // a11: k+1-token verify pass, slow stream, all layers; a12: accept + rollback on the device.
  // The pass is ~290 dependent launches whose arguments depend only on (k, B, attention splits, script,
  // implementation): after one eager run it is captured into a CUDA graph and replayed (positions, kv_len,
  // drafts and tokens are read from device memory inside the kernels).
  {
    int max_len = 0;
    for (int b = 0; b < B; ++b) max_len = std::max(max_len, x->kv_h[b]);
    const int splits = n_splits_for(x, B, max_len + k + 1, c.dtype == M2R2_BF16 && (c.head_dim == 64 || c.head_dim == 96 || c.head_dim == 128));   // as run_pass will
    const unsigned long long key = ((unsigned long long)x->ls_version << 32) | ((unsigned long long)(x->ls_on ? 1 : 0) << 31) |
                                   ((unsigned long long)(x->fused ? 1 : 0) << 30) | ((unsigned long long)splits << 12) |
                                   ((unsigned long long)B << 4) | (unsigned long long)k;
    const bool can_graph = !x->prof;
    auto it = can_graph ? x->vgraph.find(key) : x->vgraph.end();
    if (it != x->vgraph.end()) {
      CU(x, cudaGraphLaunch(it->second, x->cs));
      x->st.kernel_launches += x->vgraph_launches[key];
    } else {
      int& seen = x->vgraph_seen[key];
      const bool capture = can_graph && seen >= 1;
      const int64_t l0 = x->st.kernel_launches;
      if (capture && cudaStreamBeginCapture(x->cs, cudaStreamCaptureModeRelaxed) != cudaSuccess) { cudaGetLastError(); seen = -1000000; }
      const bool capturing = capture && seen >= 1;
      Pass p = {MODE_VERIFY, k + 1, 0, 0, c.n_layers, false, false, false, true, false};
      rc = run_pass(x, p);
      if (!rc) {
        // tokens t_j: rows b*(k+1)+j -> d_vtok[b*8 + j]
        final_head(x, B * (k + 1), x->d_accepted, 1);   // temp: contiguous rows
        for (int b = 0; b < B; ++b)
          cudaMemcpyAsync(x->d_vtok + b * 8, x->d_accepted + b * (k + 1), sizeof(int) * (k + 1), cudaMemcpyDeviceToDevice, x->cs);
        prof_mark(x, M2R2_PROF_OTHER);
        accept_kernel<<<1, 32, 0, x->cs>>>(B, k, x->d_drafts, x->d_vtok, x->d_accepted, x->d_nacc, x->d_kv_len, x->d_pending);
        count(x);
      }
      if (capturing) {
        cudaGraph_t g = nullptr;
        cudaGraphExec_t ex = nullptr;
        cudaError_t e = cudaStreamEndCapture(x->cs, &g);
        if (e == cudaSuccess && !rc) e = cudaGraphInstantiate(&ex, g, 0);
        if (g) cudaGraphDestroy(g);
        if (rc) return rc;
        if (e != cudaSuccess || !ex) {
          cudaGetLastError();
          seen = -1000000;      // not capturable on this system: stay eager for this key
          return fail(x, M2R2_CUDA, "verify graph capture failed: %s", cudaGetErrorString(e));
        }
        x->vgraph[key] = ex;
        x->vgraph_launches[key] = (int)(x->st.kernel_launches - l0);
        CU(x, cudaGraphLaunch(ex, x->cs));   // the captured launches have not run yet
      } else if (rc) {
        return rc;
      }
      ++seen;
    }
    for (int i = 0; i < c.n_layers; ++i)
      for (int b = 0; b < B; ++b) bytes += (b == 0 ? layer_bytes(x, i, false, 0) : 0) + 2 * (int64_t)c.d_model * (x->kv_h[b] + k + 1 + k + 1) * x->esz;
    bytes += (int64_t)c.vocab * c.d_model * x->esz;
  }
  x->st.algorithmic_bytes_last = bytes;
  prof_resolve(x);
  CU(x, cudaMemcpyAsync(x->h_pinned, x->d_accepted, sizeof(int) * B * 8, cudaMemcpyDeviceToHost, x->cs));
  CU(x, cudaMemcpyAsync(x->h_pinned + 64, x->d_nacc, sizeof(int) * B, cudaMemcpyDeviceToHost, x->cs));
  CU(x, cudaStreamSynchronize(x->cs));
  CU(x, cudaGetLastError());
  if (use_fused && k > 0 && (rc = fused_check(&x->fs, x->cs, x->err, sizeof(x->err)))) return rc;
  for (int b = 0; b < B; ++b) {
    int n = x->h_pinned[64 + b];
    n_accepted[b] = n;
    for (int j = 0; j <= k; ++j) accepted[b * (k + 1) + j] = j < n ? x->h_pinned[b * 8 + j] : -1;
    x->kv_h[b] += n;
    x->st.accepted += n - 1;
    x->st.emitted += n;
  }
  x->st.drafted += (int64_t)k * B;
  x->last_rows_per_seq = k + 1;
  x->st.steps++;
  return M2R2_OK;
}

// ------------------------------------------------------------------ MoE prefill (chunked, experts streamed through the staging slot)
static int moe_prefill(m2r2_ctx* x, int P) {
  // Token-chunk-major like the dense prefill; per chunk and layer the routed experts of the
  // chunk's rows are streamed one by one through staging slot 0 and applied to all rows with
  // a per-row weight (0 for rows that did not select the expert).  Untimed supporting path:
  // it does not touch the cache model or its counters.
  const m2r2_config& c = x->c;
  const int d = c.d_model, tk = c.top_k, nh = c.n_heads, dh = c.head_dim;
  const float scale = 1.0f / sqrtf((float)dh);
  float* wtab = x->moe_wtab;                  // [8 rows] per-row weight of the current expert
  int* ridx = x->d_moe_ridx;                  // [8][tk] routed experts of the chunk's rows
  float* rw = x->moe_rw;                      // [8][tk] their weights
  for (int c0 = 0; c0 < P; c0 += 8) {
    const int m = std::min(8, P - c0);
    x->kv_h[0] = c0;
    setup_rows_kernel<<<1, 32, 0, x->cs>>>(MODE_PREFILL, 1, m, 0, c0, c.max_seq, x->d_kv_len, x->d_pending, x->d_drafts,
                                           nullptr, x->d_prompt, x->d_row_tok, x->d_row_seq, x->d_row_pos, x->d_row_limit, x->d_grp_rows);
    launch_embed(x->cs, c.dtype, x->embed, x->d_row_tok, m, d, x->resid, nullptr, nullptr, nullptr);
    count(x, 2);
    const int splits = n_splits_for(x, 1, c0 + m);
    for (int i = 0; i < c.n_layers; ++i) {
      const DevLayer& L = x->L[i];
      char* Kc = (char*)x->b.kv + (size_t)i * c.max_batch * nh * c.max_seq * dh * x->esz;
      char* Vc = Kc + (size_t)c.n_layers * c.max_batch * nh * c.max_seq * dh * x->esz;
      launch_norm_lora(x->cs, c.dtype, x->resid, m, d, L.g1, c.rms_eps, x->xn, nullptr, 0, 0, 0, x->U, 64);
      GemvArgs g;
      memset(&g, 0, sizeof(g));
      g.W = L.wqkv; g.X = x->xn; g.ldx = d; g.n_rows = m; g.K = d; g.n_out = 3 * d; g.out = x->qkv; g.ldo = 3 * d;
      launch_gemv(x->cs, c.dtype, g, false);
      launch_rope_append(x->cs, c.dtype, x->qkv, m, m, x->d_row_seq, x->d_row_pos, x->rope_tab, Kc, Vc, nh, dh, c.max_seq);
      AttnArgs a;
      memset(&a, 0, sizeof(a));
      a.qkv = x->qkv; a.Kc = Kc; a.Vc = Vc; a.row_seq = x->d_row_seq; a.row_limit = x->d_row_limit; a.grp_rows = x->d_grp_rows;
      a.part_o = x->part_o; a.part_ml = x->part_ml; a.n_heads = nh; a.dh = dh; a.d = d; a.max_seq = c.max_seq; a.n_splits = splits;
      a.slow_rows = 1 << 30; a.scale = scale;
      launch_attn(x->cs, c.dtype, a, 1, m);
      MergeArgs mg;
      memset(&mg, 0, sizeof(mg));
      mg.qkv = x->qkv; mg.part_o = x->part_o; mg.part_ml = x->part_ml; mg.row_limit = x->d_row_limit; mg.out = x->attn_o;
      mg.n_heads = nh; mg.dh = dh; mg.d = d; mg.n_splits = splits; mg.slow_rows = 1 << 30; mg.scale = scale;
      launch_merge(x->cs, mg, m);
      memset(&g, 0, sizeof(g));
      g.W = L.wo; g.X = x->attn_o; g.ldx = d; g.n_rows = m; g.K = d; g.n_out = d; g.out = x->resid; g.ldo = d; g.resid = x->resid;
      launch_gemv(x->cs, c.dtype, g, false);
      launch_norm_lora(x->cs, c.dtype, x->resid, m, d, L.g2, c.rms_eps, x->xn, nullptr, 0, 0, 0, x->U, 64);
      launch_route(x->cs, c.dtype, x->xn, d, m, d, nullptr, 0.f, 0, L.router, c.n_experts, tk, c.renorm_topk, x->d_row_pos,
                   x->rs_on ? x->d_rs_actual : nullptr, x->rs_first, x->rs_n, c.n_layers, i, x->rs_beta, ridx, rw);
      count(x, 9);
      CU(x, cudaMemcpyAsync(x->h_pinned, ridx, sizeof(int) * m * tk, cudaMemcpyDeviceToHost, x->cs));
      CU(x, cudaMemcpyAsync(x->h_pinned + 256, rw, sizeof(float) * m * tk, cudaMemcpyDeviceToHost, x->cs));
      CU(x, cudaStreamSynchronize(x->cs));
      std::vector<int> experts;
      for (int q = 0; q < m * tk; ++q)
        if (std::find(experts.begin(), experts.end(), x->h_pinned[q]) == experts.end()) experts.push_back(x->h_pinned[q]);
      const float* hw = (const float*)(x->h_pinned + 256);
      for (size_t q = 0; q < experts.size(); ++q) {
        int e = experts[q];
        float* wrow = (float*)(x->h_pinned + 512);
        for (int rr = 0; rr < 8; ++rr) {
          wrow[rr] = 0.f;
          if (rr < m) for (int k = 0; k < tk; ++k) if (x->h_pinned[rr * tk + k] == e) wrow[rr] = hw[rr * tk + k];
        }
        int rc = copy_expert(x, i, e, stage_ptr(x, 0), x->cs);   // same stream: ordered after the previous expert's kernels
        if (rc) return rc;
        CU(x, cudaMemcpyAsync(wtab, wrow, sizeof(float) * 8, cudaMemcpyHostToDevice, x->cs));
        expert_ffn(x, stage_ptr(x, 0), 0, m, wtab, 1, q == 0, q + 1 == experts.size());
        CU(x, cudaStreamSynchronize(x->cs));   // wrow / staging reuse
      }
    }
    if (c0 + m >= P) {
      final_head(x, m, x->d_vtok, 1);
      CU(x, cudaMemcpyAsync(x->d_out_tok, x->d_vtok + m - 1, sizeof(int), cudaMemcpyDeviceToDevice, x->cs));
    }
  }
  x->st.h2d_bytes = 0;
  return 0;
}

// ------------------------------------------------------------------ ABI: MoE prefetch / policy / scripts / stats / debug
extern "C" int m2r2_moe_prefetch(m2r2_ctx* x, int32_t src_layer, const int32_t* pairs, int32_t n) {
  int rc = check_ready(x);
  if (rc) return rc;
  const m2r2_config& c = x->c;
  if (!c.n_experts) return fail(x, M2R2_UNSUPPORTED, "moe_prefetch on a dense model");
  if (x->policy == M2R2_POLICY_FIXED) return fail(x, M2R2_BAD_STATE, "moe_prefetch under the fixed-residency policy");
  if (pairs) {
    if (n < 0) return fail(x, M2R2_INVALID_ARG, "moe_prefetch: n < 0");
    for (int i = 0; i < n; ++i)
      if (pairs[2 * i] < 0 || pairs[2 * i] >= c.n_layers || pairs[2 * i + 1] < 0 || pairs[2 * i + 1] >= c.n_experts)
        return fail(x, M2R2_INVALID_ARG, "moe_prefetch: pair out of range");
    return prefetch_pairs(x, pairs, n);
  }
  if (src_layer < 0 || src_layer >= c.n_layers || !layer_accel(c, src_layer)) return fail(x, M2R2_INVALID_ARG, "moe_prefetch: bad src_layer");
  if (c.aot_lo[src_layer] >= c.aot_hi[src_layer]) return 0;
  if (!x->have_pending || x->st.steps == 0) return fail(x, M2R2_BAD_STATE, "moe_prefetch: no accelerated residual held yet");
  // predict from the traced accelerated residual p_{src+1} of the last decode step
  const int d = c.d_model, tk = c.top_k, B = x->B;
  const float* p = x->trace + ((size_t)(src_layer + 1) * 2 * B + B) * d;
  int nt = c.aot_hi[src_layer] - c.aot_lo[src_layer];
  for (int Lt = c.aot_lo[src_layer]; Lt < c.aot_hi[src_layer]; ++Lt) {
    launch_route(x->cs, c.dtype, p, d, 1, d, x->L[Lt].g2, c.rms_eps, 1, x->L[Lt].router, c.n_experts, tk, c.renorm_topk,
                 x->d_row_pos + B, x->rs_on ? x->d_rs_pred : nullptr, x->rs_first, x->rs_n, c.n_layers, Lt, x->rs_beta,
                 x->d_pred_idx + Lt * tk, x->pred_w + Lt * tk);
    count(x);
  }
  CU(x, cudaMemcpyAsync(x->h_pinned + 1024, x->d_pred_idx + c.aot_lo[src_layer] * tk, sizeof(int) * nt * tk, cudaMemcpyDeviceToHost, x->cs));
  CU(x, cudaStreamSynchronize(x->cs));
  std::vector<int> pr;
  for (int t = 0; t < nt; ++t)
    for (int k = 0; k < tk; ++k) { pr.push_back(c.aot_lo[src_layer] + t); pr.push_back(x->h_pinned[1024 + t * tk + k]); }
  return prefetch_pairs(x, pr.data(), (int)pr.size() / 2);
}

extern "C" int m2r2_set_policy(m2r2_ctx* x, int32_t policy) {
  if (!x) return M2R2_INVALID_ARG;
  if (policy < 0 || policy > M2R2_POLICY_LRU_PREV) return fail(x, M2R2_INVALID_ARG, "bad policy");
  if (!x->c.n_experts) return fail(x, M2R2_UNSUPPORTED, "policy on a dense model");
  x->policy = policy;
  if (x->weights_loaded) return reset_expert_cache(x);
  return M2R2_OK;
}

extern "C" int m2r2_set_logit_script(m2r2_ctx* x, const int32_t* full_tok, const int32_t* draft_tok, int32_t first_pos,
                                     int32_t n, float beta) {
  if (!x) return M2R2_INVALID_ARG;
  x->ls_version++;
  // captured verify graphs are keyed by the script version: the old ones can never be launched again
  CU(x, cudaStreamSynchronize(x->cs));
  for (auto& kv : x->vgraph) cudaGraphExecDestroy(kv.second);
  x->vgraph.clear(); x->vgraph_seen.clear(); x->vgraph_launches.clear();
  if (!full_tok) { x->ls_on = false; return M2R2_OK; }
  const m2r2_config& c = x->c;
  if (n < 1 || n > c.max_seq || first_pos < 0) return fail(x, M2R2_INVALID_ARG, "logit script: bad n/first_pos");
  const int B = c.max_batch;
  for (int64_t i = 0; i < (int64_t)B * n; ++i) {
    if (full_tok[i] < 0 || full_tok[i] >= c.vocab) return fail(x, M2R2_INVALID_ARG, "logit script: token out of range");
    if (draft_tok && (draft_tok[i] < 0 || draft_tok[i] >= c.vocab)) return fail(x, M2R2_INVALID_ARG, "logit script: token out of range");
  }
  CU(x, cudaStreamSynchronize(x->cs));
  CU(x, cudaMemcpy(x->d_ls_full, full_tok, sizeof(int) * B * n, cudaMemcpyHostToDevice));
  CU(x, cudaMemcpy(x->d_ls_draft, draft_tok ? draft_tok : full_tok, sizeof(int) * B * n, cudaMemcpyHostToDevice));
  x->ls_first = first_pos; x->ls_n = n; x->ls_beta = beta; x->ls_on = true;
  return M2R2_OK;
}

extern "C" int m2r2_set_router_script(m2r2_ctx* x, const int32_t* actual, const int32_t* pred, int32_t first_pos, int32_t n,
                                      float beta) {
  if (!x) return M2R2_INVALID_ARG;
  if (!actual) { x->rs_on = false; return M2R2_OK; }
  const m2r2_config& c = x->c;
  if (!c.n_experts) return fail(x, M2R2_UNSUPPORTED, "router script on a dense model");
  if (n < 1 || n > c.max_seq || first_pos < 0) return fail(x, M2R2_INVALID_ARG, "router script: bad n/first_pos");
  size_t cnt = (size_t)n * c.n_layers * 2;
  for (size_t i = 0; i < cnt; ++i) {
    if (actual[i] < 0 || actual[i] >= c.n_experts) return fail(x, M2R2_INVALID_ARG, "router script: expert out of range");
    if (pred && (pred[i] < 0 || pred[i] >= c.n_experts)) return fail(x, M2R2_INVALID_ARG, "router script: expert out of range");
  }
  CU(x, cudaStreamSynchronize(x->cs));
  CU(x, cudaMemcpy(x->d_rs_actual, actual, sizeof(int) * cnt, cudaMemcpyHostToDevice));
  CU(x, cudaMemcpy(x->d_rs_pred, pred ? pred : actual, sizeof(int) * cnt, cudaMemcpyHostToDevice));
  x->rs_first = first_pos; x->rs_n = n; x->rs_beta = beta; x->rs_on = true;
  return M2R2_OK;
}

extern "C" int m2r2_get_stats(m2r2_ctx* x, m2r2_stats* out) {
  if (!x || !out) return M2R2_INVALID_ARG;
  if (fused_abort_pending(&x->fs)) {
    int rc = fused_check(&x->fs, x->cs, x->err, sizeof(x->err));
    if (rc) return rc;
  }
  *out = x->st;
  for (int b = 0; b < M2R2_MAX_BATCH; ++b) out->kv_len[b] = b < x->B ? x->kv_h[b] : 0;
  return M2R2_OK;
}

__global__ void kv_to_f32_kernel(const void* cache, int bf16, int n_heads, int dh, int max_seq, int t0, int T, float* out) {
  // out[t][head*dh + j] from cache[head][t0 + t][j]
  size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  size_t d = (size_t)n_heads * dh;
  if (i >= (size_t)T * d) return;
  int t = (int)(i / d), hd = (int)(i % d), head = hd / dh, j = hd % dh;
  size_t src = ((size_t)head * max_seq + t0 + t) * dh + j;
  out[i] = bf16 ? __bfloat162float(((const __nv_bfloat16*)cache)[src]) : ((const float*)cache)[src];
}
__global__ void i2f_kernel(const int* in, float* out, int n) {
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) out[i] = (float)in[i];
}

extern "C" int m2r2_debug_read(m2r2_ctx* x, int32_t what, int32_t layer, int32_t b, float* host_out, size_t n) {
  int rc = check_ready(x);
  if (rc) return rc;
  const m2r2_config& c = x->c;
  if (!host_out || n == 0) return fail(x, M2R2_INVALID_ARG, "debug_read: no output");
  const int B = std::max(1, x->B);
  if (b < 0 || b >= B) return fail(x, M2R2_INVALID_ARG, "debug_read: bad sequence");
  const size_t d = c.d_model, V = c.vocab, tk = std::max(1, c.top_k);
  const float* src = nullptr;
  size_t avail = 0;
  CU(x, cudaStreamSynchronize(x->cs));
  if (fused_abort_pending(&x->fs) && (rc = fused_check(&x->fs, x->cs, x->err, sizeof(x->err)))) return rc;
  switch (what) {
    case M2R2_DBG_H:
    case M2R2_DBG_P:
      if (layer < 0 || layer > c.n_layers) return fail(x, M2R2_INVALID_ARG, "debug_read: bad layer");
      src = x->trace + ((size_t)layer * 2 * B + (what == M2R2_DBG_P ? B : 0) + b) * d;
      avail = d;
      break;
    case M2R2_DBG_LOGITS:
      if (layer < 0 || layer >= 8) return fail(x, M2R2_INVALID_ARG, "debug_read: bad row");
      src = x->logits + ((size_t)b * (x->last_rows_per_seq) + layer) * V;
      avail = V;
      break;
    case M2R2_DBG_EXIT_LOGITS:
      if (layer < 0 || layer >= c.n_gates) return fail(x, M2R2_INVALID_ARG, "debug_read: bad gate");
      src = x->exit_logits + ((size_t)layer * B + b) * V;
      avail = V;
      break;
    case M2R2_DBG_K:
    case M2R2_DBG_V: {
      if (layer < 0 || layer >= c.n_layers) return fail(x, M2R2_INVALID_ARG, "debug_read: bad layer");
      size_t T = n / d;
      if (T < 1 || T > (size_t)c.max_seq) return fail(x, M2R2_INVALID_ARG, "debug_read: bad n");
      size_t per = (size_t)c.n_heads * c.max_seq * c.head_dim * x->esz;
      char* base = (char*)x->b.kv + ((size_t)layer * c.max_batch + b) * per;
      if (what == M2R2_DBG_V) base += (size_t)c.n_layers * c.max_batch * per;
      // converted through the attention-partials scratch (dead between steps, never read back) in chunks of
      // whole positions
      const size_t cap = (size_t)x->R * M2R2_MAX_SPLITS;   // part_o holds R * n_heads * splits * dh floats
      if (cap < 1) return fail(x, M2R2_UNSUPPORTED, "debug_read: scratch too small for one K/V row");
      for (size_t t0 = 0; t0 < T; t0 += cap) {
        const size_t nt = std::min(cap, T - t0);
        kv_to_f32_kernel<<<(unsigned)((nt * d + 255) / 256), 256, 0, x->cs>>>(base, c.dtype == M2R2_BF16, c.n_heads, c.head_dim, c.max_seq, (int)t0, (int)nt, x->part_o);
        CU(x, cudaMemcpyAsync(host_out + t0 * d, x->part_o, nt * d * sizeof(float), cudaMemcpyDeviceToHost, x->cs));
        CU(x, cudaStreamSynchronize(x->cs));
      }
      return M2R2_OK;
    }
    case M2R2_DBG_ROUTE_IDX:
    case M2R2_DBG_PRED_IDX: {
      size_t cnt = (size_t)c.n_layers * tk;
      if (n > cnt) return fail(x, M2R2_INVALID_ARG, "debug_read: n too large");
      float* tmp = x->moe_tmp;
      i2f_kernel<<<(unsigned)((cnt + 255) / 256), 256, 0, x->cs>>>(what == M2R2_DBG_ROUTE_IDX ? x->d_route_idx : x->d_pred_idx, tmp, (int)cnt);
      CU(x, cudaMemcpyAsync(host_out, tmp, n * sizeof(float), cudaMemcpyDeviceToHost, x->cs));
      CU(x, cudaStreamSynchronize(x->cs));
      return M2R2_OK;
    }
    case M2R2_DBG_EXIT_SCORE:
      if (!x->arla) return fail(x, M2R2_UNSUPPORTED, "debug_read: the config has no ARLA router");
      src = x->exit_score + (size_t)b * M2R2_MAX_GATES;
      avail = (size_t)c.n_gates;
      break;
    case M2R2_DBG_ROUTE_W:
      src = x->route_w;
      avail = (size_t)c.n_layers * tk;
      break;
    default:
      return fail(x, M2R2_INVALID_ARG, "debug_read: unknown tensor");
  }
  if (n > avail) return fail(x, M2R2_INVALID_ARG, "debug_read: n too large");
  CU(x, cudaMemcpy(host_out, src, n * sizeof(float), cudaMemcpyDeviceToHost));
  return M2R2_OK;
}

extern "C" int m2r2_set_fused(m2r2_ctx* x, int32_t enabled) {
  if (!x) return M2R2_INVALID_ARG;
  x->fused = enabled != 0;
  return M2R2_OK;
}

extern "C" int m2r2_set_profile(m2r2_ctx* x, int32_t enabled) {
  if (!x) return M2R2_INVALID_ARG;
  x->prof = enabled != 0;
  x->pn = 0;
  if (x->prof) memset(&x->pr, 0, sizeof(x->pr));
  return M2R2_OK;
}
extern "C" int m2r2_get_profile(m2r2_ctx* x, m2r2_profile* out) {
  if (!x || !out) return M2R2_INVALID_ARG;
  *out = x->pr;
  return M2R2_OK;
}

extern "C" const char* m2r2_last_error(const m2r2_ctx* x) { return x ? x->err : "null context"; }
extern "C" const char* m2r2_version(void) { return "m2r2-b200 0.1 (sm_100a)"; }
