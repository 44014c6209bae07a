// kernels_fused.cu — persistent fused dual-stream decode step (bf16, dense, batch 1).
// Placeholder until the fused kernel lands: reports "not supported" so decode_step uses the
// per-operation kernels.
#include "m2r2_fused.cuh"

void fused_carve(const m2r2_config&, Carver&, FusedState*) {}
int fused_create(const m2r2_config&, FusedState* fs) { fs->supported = false; return 0; }
void fused_destroy(FusedState*) {}
int fused_bind(const m2r2_config&, FusedState*, const void*, const void*, const void*, const DevLayer*, size_t) { return 0; }
bool fused_supported(const m2r2_config&, const FusedState* fs) { return fs->supported; }
int fused_decode_step(const m2r2_config&, FusedState*, cudaStream_t, int*, int*, const int*, int, void*, float*, float*,
                      float*, int*, int*, const int*, const int*, int, int, float, int64_t*) {
  return M2R2_UNSUPPORTED;
}
