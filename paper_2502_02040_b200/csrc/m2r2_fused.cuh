// m2r2_fused.cuh — interface of the persistent fused decode kernel (kernels_fused.cu).
//
// One cooperative launch per decode step (or per draft pass): one CTA per SM, a producer
// thread streaming tile-major bf16 weight stages through a shared-memory ring with bulk
// async copies (cp.async.bulk + mbarrier), eight consumer warps doing the dual-row
// (slow h / accelerated p) dot products, grid barriers between the phases of a layer.
// DESIGN.md §"Fused decode kernel" has the layout and the phase list.
#pragma once
#include "m2r2_internal.cuh"

struct FusedImpl;
struct FusedState {
  bool supported = false;
  FusedImpl* impl = nullptr;
  int64_t* launch_counter = nullptr;   // fused_gemv_rows adds the launches beyond the one its caller counts
};

// what one launch runs
struct FusedRun {
  int n_layers;            // layers [0, n_layers)
  int joff;                // position = kv_len + joff (draft loop); 0 for decode_step
  const int* tok_in;       // device: token consumed by this pass
  int head_stream;         // 0: final head on h_N (decode_step); 1: draft head on p at the gate == n_layers
  int* tok_out;            // device: greedy token of the head
  int advance;             // kv_len += 1, pending = token (decode_step)
  int exit_heads;          // evaluate the exit argmax at every gate <= n_layers (decode_step)
  int trace;               // write h_i / p_i traces
};

// bytes of the tile-major weight region the fused path needs inside the weights buffer (0 if unsupported)
size_t fused_weights_bytes(const m2r2_config& c);
bool fused_config_ok(const m2r2_config& c);
void fused_carve(const m2r2_config& c, Carver& cv, FusedState* fs);
int fused_create(const m2r2_config& c, FusedState* fs);
void fused_destroy(FusedState* fs);
// repack the row-major resident weights (already in HBM) into the tile-major stage stream at `packed`
int fused_bind(const m2r2_config& c, FusedState* fs, cudaStream_t st, void* packed, const void* embed,
               const void* gf, const void* lm_head, const void* lm_A, const void* lm_B,
               const DevLayer* layers, void* kv, const float2* rope_tab);
bool fused_supported(const m2r2_config& c, const FusedState* fs);
int fused_run(const m2r2_config& c, FusedState* fs, cudaStream_t st, const FusedRun& run, int* d_kv_len,
              int* d_pending, int kv_len_host, float* trace, float* logits, float* exit_logits,
              int* d_exit_tok, const int* ls_full, const int* ls_draft, int ls_first, int ls_n,
              float ls_beta, int64_t* launches);
// 0 if the last launches completed normally; otherwise a description (device-side timeout)
int fused_check(FusedState* fs, cudaStream_t st, char* msg, size_t n);
// non-blocking variant: true once any launch has reported a timed-out wait (then call fused_check to re-arm)
bool fused_abort_pending(const FusedState* fs);
// a11: skinny GEMM of <= 8 slow-stream rows on the fragment-major weights (verify pass, prefill chunks).
// kind: 0 QKV (natural row order out), 1 O-proj (+resid), 2 gate/up + SwiGLU, 3 down (+resid, trace), 4 LM head.
// Returns M2R2_UNSUPPORTED when the fused weight copy is not bound or rows > 64.
// rows 9..64 (rows_mma_kernel) may carry the accelerated rows' parallel adapters: `lora` supplies Bm / Bm2 / bmap / U /
// ldu / r / lora_row0 / usel_div with the meaning they have in GemvArgs (nullptr: none).
// rows <= 8 without adapters (rows_ring_kernel, one CTA per SM streaming the matrix through a shared-memory ring) can also
// absorb the GEMM's neighbours in the layer, given in `fz`; with more rows (rows_mma_kernel) only RoPE + KV append; M2R2_UNSUPPORTED then means nothing was launched and the
// caller runs the separate kernels.
struct RowsFuse {
  const void* gain = nullptr;      // QKV, gate/up, LM head: X is the raw residual; RMSNorm(x; gain, eps) inside (a2, a6, a9)
  float eps = 0.f;
  const float* part_o = nullptr;   // O: X is ignored; the rows are merged from the attention partials of <= 8 splits (a4)
  const float* part_ml = nullptr;
  int n_splits = 0;
  const int* row_seq = nullptr;    // QKV: RoPE on q, k and the K/V cache append in the epilogue (a3)
  const int* row_pos = nullptr;
  const float2* rope_tab = nullptr;
  void* Kc = nullptr;
  void* Vc = nullptr;
  bool x_packed = false;           // > 8 rows: the rows are already in the fused state's (hi, lo) word buffer (QKV, gate/up: by
                                   // norm_lora_kernel through fused_xn_pack; down: by a gate/up call with pack_out): no pack_rows_kernel
  bool pack_out = false;           // gate/up, > 8 rows: also leave the activations as (hi, lo) words for the down call
  int slow_rows = 0;               // rows >= slow_rows (accelerated rows, > 8-row passes) are rotated but not cached; 0: all rows
};
int fused_gemv_rows(const m2r2_config& c, FusedState* fs, cudaStream_t st, int layer, int kind, const float* X, int ldx,
                    int rows, float* out, int ldo, const float* resid, float* trace, const GemvArgs* lora = nullptr,
                    const RowsFuse* fz = nullptr);
uint2* fused_xn_pack(const FusedState* fs, int* ld);
