// m2r2_fused.cuh — interface of the persistent fused decode kernel (kernels_fused.cu).
#pragma once
#include "m2r2_internal.cuh"

struct FusedState {
  bool supported = false;
  void* impl = nullptr;
};

void fused_carve(const m2r2_config& c, Carver& cv, FusedState* fs);
int fused_create(const m2r2_config& c, FusedState* fs);
void fused_destroy(FusedState* fs);
int fused_bind(const m2r2_config& c, FusedState* fs, const void* embed, const void* gf, const void* lm_head,
               const DevLayer* layers, size_t layer_stride);
bool fused_supported(const m2r2_config& c, const FusedState* fs);
int fused_decode_step(const m2r2_config& c, FusedState* fs, cudaStream_t st, int* d_kv_len, int* d_pending,
                      const int* d_force, int kv_len_host, void* kv, float* trace, float* logits,
                      float* exit_logits, int* d_out_tok, int* d_exit_tok, const int* ls_full,
                      const int* ls_draft, int ls_first, int ls_n, float ls_beta, int64_t* launches);
