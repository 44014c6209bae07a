/* m2r2.h — C ABI of the B200-native M2R2 decode hot path (arxiv 2502.02040).
 *
 * M2R2 = Mixture of Multi-Rate Residuals.  The library carries, through every decoder layer,
 * the ordinary slow residual stream h (Eq. 1) and the accelerated residual
 * stream p (Eq. 2): p runs through the frozen base weights plus rank-r parallel adapters
 * (L74), uses a subset S of the attention heads (§2.5), attends to the SLOW stream's KV
 * cache plus its own key/value, MHA(p_t, h_<t (+) p_t, h_<t (+) p_t) (L76), and is
 * re-initialised from h at every gate (L82, L101).  On top of that step the library provides
 * self-speculative decoding (§2.3.2) and MoE ahead-of-time expert loading
 * (§2.3.3; App. B).  Readings of everything the paper leaves open are listed
 * in DESIGN.md §"Readings".
 *
 * Conventions
 *  - Every call returns M2R2_OK (0) or a negative m2r2_status.  Argument errors leave the
 *    context untouched.  No exceptions or C++ types cross this boundary.
 *  - "host" / "device" is stated for every pointer.  Host output pointers are valid when the
 *    call returns (the call synchronises the compute stream before writing them).
 *  - The library never allocates caller-visible device memory: the caller allocates the
 *    buffers sized by m2r2_query_sizes (e.g. with torch) and keeps them alive until
 *    m2r2_destroy.  Streams are borrowed cudaStream_t handles.
 *  - One context, one caller thread.  Every step of the path runs in sm_100a CUDA kernels;
 *    there is no CPU fallback.
 *  - Matrices are row-major [out, in] in the storage dtype (fp32 or bf16 bit patterns).
 *    All inner dimensions (d_model, d_ff, d_ff_expert, n_accel_heads*head_dim) must be
 *    multiples of 8 elements; head_dim must be a multiple of 32 and <= 128.
 */
#ifndef M2R2_H_
#define M2R2_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define M2R2_MAX_HEADS 128
#define M2R2_MAX_GATES 16
#define M2R2_MAX_LAYERS 128
#define M2R2_MAX_BATCH 8
#define M2R2_MAX_DRAFT 7   /* spec_step k <= 7  =>  k+1 <= 8 verify rows per sequence */
#define M2R2_MAX_TOPK 8
#define M2R2_MAX_EXPERTS 64

typedef enum {
  M2R2_OK = 0,
  M2R2_INVALID_ARG = -1,
  M2R2_BAD_STATE = -2,   /* e.g. decode before prefill / before load_weights */
  M2R2_CAPACITY = -3,    /* kv_len + k + 1 > max_seq */
  M2R2_CUDA = -4,        /* a CUDA call failed; see m2r2_last_error */
  M2R2_UNSUPPORTED = -5
} m2r2_status;

enum { M2R2_FP32 = 0, M2R2_BF16 = 1 };

/* MoE expert-loading policy: the five strategies of PAPER.md L242.
 *   FIXED       experts 0..C-1 of a layer stay resident, every other expert is loaded on demand each time
 *   LRU         least-recently-used replacement, loads on demand only
 *   LRU_AOT     LRU + ahead-of-time speculation from the accelerated residual (L137-139, L244, App. B: the paper's)
 *   LRU_RANDOM  LRU + top_k uniformly drawn experts pre-loaded one layer ahead (seeded counter-based generator)
 *   LRU_PREV    LRU + speculation one layer ahead from the previous layer's slow residual: the router of layer i + 1
 *               applied to rms(h_{i+1}; g2_{i+1})                                                                        */
enum { M2R2_POLICY_FIXED = 0, M2R2_POLICY_LRU = 1, M2R2_POLICY_LRU_AOT = 2, M2R2_POLICY_LRU_RANDOM = 3, M2R2_POLICY_LRU_PREV = 4 };

typedef struct m2r2_config {
  uint32_t struct_size;          /* = sizeof(m2r2_config); versions the struct */
  int32_t n_layers, d_model, n_heads, head_dim, d_ff, vocab;   /* d_model == n_heads*head_dim */
  int32_t dtype;                 /* M2R2_FP32 | M2R2_BF16: storage of weights AND KV cache */
  int32_t max_batch, max_seq;
  float rms_eps, rope_theta;
  /* accelerated stream */
  int32_t accel_enabled;
  int32_t n_accel_heads;
  int32_t accel_heads[M2R2_MAX_HEADS];   /* sorted head subset S */
  int32_t adapter_rank;                  /* r (L74, L399) */
  int32_t n_gates;
  int32_t gates[M2R2_MAX_GATES];         /* E_1 < ... < E_J: p <- h after layer E_j - 1 (L82) */
  int32_t accel_end_layer;               /* p is carried through layers [0, accel_end_layer) */
  int32_t lm_head_adapter;               /* rank-r adapter on the exit/draft head (L162) */
  int32_t exit_heads_enabled;            /* decode_step evaluates the exit argmax at gates */
  /* MoE (0 experts = dense SwiGLU FFN) */
  int32_t n_experts, top_k, d_ff_expert;
  int32_t cache_slots_per_layer;         /* HBM expert cache capacity C per layer (L242) */
  int32_t accel_mlp_rank;                /* r_m: accelerated stream's fixed adapter MLP (L137) */
  int32_t renorm_topk;
  int32_t aot_lo[M2R2_MAX_LAYERS];       /* source layer i predicts experts of layers        */
  int32_t aot_hi[M2R2_MAX_LAYERS];       /* [aot_lo[i], aot_hi[i]); R=2 -> {2i+2, 2i+3} L137 */
  /* Attention FLOPs optimisation (footnote 4 L170: k = 64): per head, the accelerated stream attends only the
   * k cached positions with the largest attention coefficients of the slow stream (same head, same token; ties: lower
   * position), plus its own k^_t.  0 = every cached position.  With k > 0 a step runs the per-operation kernels. */
  int32_t accel_topk_tokens;
  /* Accelerated Residual Latent Attention (footnote 2: d^s = 64): latent dimension of the exit router that
   * scores each gate from the accelerated residuals of its whole interval.  0 = none.  Mechanics only: decode_step reports the
   * scores (m2r2_debug_read M2R2_DBG_EXIT_SCORE); no layer is skipped. */
  int32_t arla_dim;
} m2r2_config;

typedef struct m2r2_sizes {
  uint64_t weights_bytes;       /* device: resident (non-expert) weights, repacked */
  uint64_t kv_bytes;            /* device: K and V, [layer][batch][head][max_seq][head_dim] */
  uint64_t scratch_bytes;       /* device: activations, partials, traces, device state */
  uint64_t expert_cache_bytes;  /* device: n_layers*C + top_k staging slots (0 if dense) */
  uint64_t expert_store_bytes;  /* pinned host bytes the caller's expert blobs occupy (info) */
} m2r2_sizes;

typedef struct m2r2_buffers {   /* all DEVICE pointers, 256-byte aligned, caller-owned */
  void* weights;
  void* kv;
  void* scratch;
  void* expert_cache;           /* NULL if dense */
} m2r2_buffers;

/* One layer's HOST pointers (storage dtype).  NULL for tensors the config does not have. */
typedef struct m2r2_layer_weights {
  const void *g1, *g2;                        /* [d] RMSNorm gains */
  const void *wq, *wk, *wv, *wo;              /* [d, d] */
  const void *wgate, *wup, *wdown;            /* [F, d], [F, d], [d, F] (dense only) */
  const void *Aq, *Bq, *Ak, *Bk, *Av, *Bv;    /* A [r, d], B [n_accel_heads*head_dim, r] */
  const void *Ao, *Bo;                        /* [r, n_accel_heads*head_dim], [d, r] */
  const void *Ag, *Bg, *Au, *Bu, *Ad, *Bd;    /* [r,d],[F,r],[r,d],[F,r],[r,F],[d,r] (dense) */
  const void* router;                         /* [n_experts, d] (MoE) */
  const void *Ug, *Uu, *Ud;                   /* [r_m, d], [r_m, d], [d, r_m] (MoE accel MLP) */
  /* MoE expert blobs: arrays [n_experts] of pointers into PINNED host memory.  They stay
   * owned by the caller and are read by DMA for the whole context lifetime. */
  const void* const* expert_gate;             /* each [F_e, d] */
  const void* const* expert_up;               /* each [F_e, d] */
  const void* const* expert_down;             /* each [d, F_e] */
} m2r2_layer_weights;

typedef struct m2r2_weight_table {
  const void* embed;      /* host [V, d] */
  const void* gf;         /* host [d] final norm gain */
  const void* lm_head;    /* host [V, d] (untied) */
  const void* lm_A;       /* host [r, d]  or NULL */
  const void* lm_B;       /* host [V, r]  or NULL */
  const m2r2_layer_weights* layers;   /* host array [n_layers] */
  const void* arla;       /* host [n_gates * (3 d^s + 1), d] or NULL: per gate W_q^s, W_k^s, W_v^s [d^s, d], then one row = w_o[0..d^s), b */
} m2r2_weight_table;

typedef struct m2r2_stats {
  int32_t kv_len[M2R2_MAX_BATCH];
  int64_t steps, drafted, accepted, emitted;
  int64_t expert_hits, expert_misses, expert_prefetched, expert_on_demand;
  int64_t h2d_bytes;                 /* expert bytes copied host->device so far */
  int64_t algorithmic_bytes_last;    /* DESIGN.md byte model for the last step */
  int64_t kernel_launches;           /* kernels launched by this library so far */
} m2r2_stats;

/* Per-operation device timing (CUDA events on the compute stream, recorded between the kernel
 * groups of a step).  Classes follow SURVEY §8(a): a2 QKV (with its RMSNorm), a3 RoPE+append,
 * a4 attention (+ split merge), a5 O-proj, a6 gate/up+SwiGLU (with its RMSNorm), a7 down +
 * residual, a8/a9 heads (norm + LM head + argmax), everything else (embed, row set-up, gate
 * copies, router), and the persistent fused step when that implementation runs. */
#define M2R2_PROF_CLASSES 10
enum {
  M2R2_PROF_QKV = 0, M2R2_PROF_ROPE = 1, M2R2_PROF_ATTN = 2, M2R2_PROF_OPROJ = 3,
  M2R2_PROF_GATEUP = 4, M2R2_PROF_DOWN = 5, M2R2_PROF_HEAD = 6, M2R2_PROF_OTHER = 7,
  M2R2_PROF_FUSED_STEP = 8
};
typedef struct m2r2_profile {
  double ms[M2R2_PROF_CLASSES];        /* accumulated device time per class */
  int64_t segments[M2R2_PROF_CLASSES]; /* number of timed segments per class */
  int64_t steps;                       /* decode/spec steps accumulated */
} m2r2_profile;

typedef struct m2r2_ctx m2r2_ctx;

/* Bytes the caller must allocate for `cfg`.  host in / host out. */
int m2r2_query_sizes(const m2r2_config* cfg, m2r2_sizes* out);

/* Create a context that BORROWS `bufs` (device) and the two streams (cudaStream_t; 0 = legacy
 * default stream).  copy_stream carries the expert prefetch DMA (App. B). */
int m2r2_create(const m2r2_config* cfg, const m2r2_buffers* bufs, void* compute_stream,
                void* copy_stream, m2r2_ctx** out);
int m2r2_destroy(m2r2_ctx* ctx);

/* Copy (and repack) the resident weights host -> HBM.  The host copy of resident tensors is
 * not retained; expert blobs are retained by pointer (see m2r2_layer_weights). */
int m2r2_load_weights(m2r2_ctx* ctx, const m2r2_weight_table* host);

/* Reset sequence state, run the slow stream over the prompt (all sequences have length P),
 * fill the KV cache, kv_len[b] = P, pending token = greedy argmax at position P-1.
 * tokens: host [B][P].  first_tokens: host [B] or NULL. */
int m2r2_prefill(m2r2_ctx* ctx, const int32_t* tokens, int32_t B, int32_t P,
                 int32_t* first_tokens);

/* One dual-stream decode step: consume the pending (or forced) token at
 * position kv_len, carry h and p through the layers, append slow K/V, kv_len += 1, return the
 * slow stream's greedy next token (becomes pending) and optionally the accelerated stream's
 * exit argmax at every gate.  MoE models run routing / expert cache / AoT prefetch inside.
 * force_tokens: host [B] or NULL.  tokens_out: host [B] or NULL (NULL = do not synchronise;
 * the token stays on the device).  exit_tokens_out: host [B][n_gates] or NULL. */
int m2r2_decode_step(m2r2_ctx* ctx, const int32_t* force_tokens, int32_t* tokens_out,
                     int32_t* exit_tokens_out);

/* Self-speculative step (§2.3.2): draft k tokens from the accelerated stream at gate E_1
 * (layers 0..E_1-1, both streams), verify k+1 positions with the slow stream through all
 * layers, accept the longest matching prefix plus the verifier's next token, roll the KV
 * cache back by setting kv_len.  k = 0 is decode_step.  accepted: host [B][k+1];
 * n_accepted: host [B], each in 1..k+1. */
int m2r2_spec_step(m2r2_ctx* ctx, int32_t k, int32_t* accepted, int32_t* n_accepted);

/* MoE ahead-of-time loading (§2.3.3).  pairs == NULL: predict from the accelerated residual
 * leaving `src_layer` (held from the current/last step) for that layer's target range and
 * enqueue H2D copies + LRU updates on the copy stream.  pairs != NULL: host [n][2] =
 * (layer, expert) to prefetch exactly.  Returns the number of copies enqueued (>= 0) or a
 * negative status.  Never blocks the compute stream. */
int m2r2_moe_prefetch(m2r2_ctx* ctx, int32_t src_layer, const int32_t* pairs, int32_t n);

int m2r2_set_policy(m2r2_ctx* ctx, int32_t moe_policy);

/* Bench/test hooks: +beta on full_tok[s-first_pos] in the final-head logits
 * that predict position s, and on draft_tok[...] in the exit/draft-head logits.  Tables are
 * host [B][n]; NULL clears.  The bias is applied inside the argmax kernel. */
int m2r2_set_logit_script(m2r2_ctx* ctx, const int32_t* full_tok, const int32_t* draft_tok,
                          int32_t first_pos, int32_t n, float beta);
/* actual/pred: host [n][n_layers][2] expert pairs; +beta on the first, +beta-8 on the second
 * in the router (actual) / predictor (pred) logits of the token at position first_pos+i. */
int m2r2_set_router_script(m2r2_ctx* ctx, const int32_t* actual, const int32_t* pred,
                           int32_t first_pos, int32_t n, float beta);

int m2r2_get_stats(m2r2_ctx* ctx, m2r2_stats* out);

enum {
  M2R2_DBG_H = 0,          /* h_layer of the last decode_step, layer in [0, N]       -> [d] */
  M2R2_DBG_P = 1,          /* p_layer (value before a gate reset)                    -> [d] */
  M2R2_DBG_LOGITS = 2,     /* final-head logits; `layer` = verify row j for spec     -> [V] */
  M2R2_DBG_EXIT_LOGITS = 3,/* exit-head logits at gate index `layer`                 -> [V] */
  M2R2_DBG_K = 4,          /* K cache of `layer`, positions [0, n/d)         -> [n/d][d]    */
  M2R2_DBG_V = 5,
  M2R2_DBG_ROUTE_IDX = 6,  /* routed experts of the last step, all layers -> [N][top_k]     */
  M2R2_DBG_ROUTE_W = 7,
  M2R2_DBG_PRED_IDX = 8,   /* predicted experts per target layer (-1 none) -> [N][top_k]    */
  M2R2_DBG_EXIT_SCORE = 9  /* ARLA exit score of every gate, last decode_step      -> [J]    */
};
/* Copy n floats of an internal tensor of sequence b to host_out (integers as floats). */
int m2r2_debug_read(m2r2_ctx* ctx, int32_t what, int32_t layer, int32_t b, float* host_out,
                    size_t n);

/* Clear sequence state (kv_len = 0, no pending token, counters, expert cache residency). */
int m2r2_reset(m2r2_ctx* ctx);

/* Select the decode implementation: 1 (default) = persistent fused kernel where supported
 * (bf16 dense, batch 1), 0 = per-operation kernels.  Both are CUDA; results agree to fp32
 * rounding.  Exposed so tests can cross-check the two. */
int m2r2_set_fused(m2r2_ctx* ctx, int32_t enabled);

/* Profiling mode: enabled != 0 clears the accumulators and makes every following decode_step /
 * spec_step record events between its kernel groups and synchronise at its end (so it is NOT
 * the mode to measure whole-step throughput in).  m2r2_get_profile copies the accumulators. */
int m2r2_set_profile(m2r2_ctx* ctx, int32_t enabled);
int m2r2_get_profile(m2r2_ctx* ctx, m2r2_profile* out);

const char* m2r2_last_error(const m2r2_ctx* ctx);
const char* m2r2_version(void);

/* ---------------------------------------------------------------------------------------------
 * The final head with NO allocation (greedy decoding
 * takes the argmax of these logits):
 *     logits[row] = W_lm . rms(h[row]; g_f),   rms(x; g) = x * g / sqrt(mean(x^2) + rms_eps)
 * for callers that cannot call cudaMalloc (CUDA-graph capture, serving loops, harnesses that forbid
 * it).  It needs no context and no caller buffers beyond inputs and output: its one scratch tensor,
 * the normalised rows, lives in a file-scope device array of M2R2_NOALLOC_MAX_ROWS x
 * M2R2_NOALLOC_MAX_D floats (256 KB, held by every GPU that loads the library until exit).  The
 * call allocates nothing and launches the engine's own kernels, so the result equals the
 * per-operation path's final head bit for bit.
 *   h       device, fp32 [m][d] dense: the slow residual after the last layer (h_N)
 *   g_f     device, [d] in `dtype`: gain of the final RMSNorm
 *   w_lm    device, [vocab][d] row-major in `dtype`: LM head
 *   logits  device, fp32 [m][vocab], written
 *   dtype   M2R2_FP32 or M2R2_BF16 (storage type of g_f and w_lm; arithmetic is fp32)
 *   stream  cudaStream_t of the launches (NULL = default stream); asynchronous, nothing is owned
 * The current device is used.  The first call on a device resolves the array's device address
 * (cudaGetSymbolAddress): make that call outside stream capture.  All calls share the scratch
 * array and it keeps the last call's contents (nothing in it has to start at zero: rows [0, m) are
 * written before they are read); calls that OVERLAP on the GPU (two streams, two threads) race on
 * it: serialise them.
 * Errors: M2R2_CAPACITY if m > M2R2_NOALLOC_MAX_ROWS or d > M2R2_NOALLOC_MAX_D; M2R2_INVALID_ARG
 * for null pointers, d % 8 != 0, vocab < 1 or an unknown dtype; M2R2_CUDA for a CUDA error.
 * m2r2_noalloc_last_error() describes the calling thread's last failure ("" after success). */
#define M2R2_NOALLOC_MAX_ROWS 8
#define M2R2_NOALLOC_MAX_D 8192
int m2r2_final_head_noalloc(const float* h, const void* g_f, const void* w_lm, float* logits,
                            int32_t m, int32_t d, int32_t vocab, int32_t dtype, float rms_eps,
                            void* stream);
const char* m2r2_noalloc_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* M2R2_H_ */
