// kernels_noalloc.cu — the final head (a9 of SURVEY §8(a): logits = W_lm rms(h_N; g_f), PAPER.md L182 greedy
// decoding reads its argmax) as ONE entry point that allocates nothing.
//
// Why: some callers cannot call cudaMalloc — code under CUDA-graph capture, tight serving loops, harnesses that forbid
// it.  The engine (m2r2_create) carves its scratch out of buffers the caller allocated; this entry point needs no
// buffers at all beyond the inputs and the output: the one scratch tensor of the op, the normalised rows
// xn = rms(h; g_f) that the head GEMV reads, lives in a file-scope device array of fixed size.
//
//   * The array costs M2R2_NOALLOC_MAX_ROWS x M2R2_NOALLOC_MAX_D x 4 B = 256 KB on every GPU that loads the library,
//     until the process exits.
//   * In host code the array's NAME is a host-side stand-in, not a device address; the device address is resolved once
//     per device with cudaGetSymbolAddress (device current), checked, cached, and passed to the kernels.
//   * Every call shares the array, which keeps the last call's contents.  Nothing in it has to start at zero: a call
//     writes rows [0, m) of xn before it reads them and reads nothing else.  Calls that overlap on the GPU (two streams,
//     two host threads) race on it: serialise them.
//   * No cudaMalloc / cudaFree / allocating library routine; the kernels are the engine's own (norm_lora_kernel,
//     gemv_kernel), so the result is bit-identical to the per-operation path's final head.
#include <cstdio>
#include <cstring>
#include <mutex>

#include "m2r2_internal.cuh"

namespace {

static __device__ __align__(256) float g_noalloc_xn[M2R2_NOALLOC_MAX_ROWS * M2R2_NOALLOC_MAX_D];

constexpr int MAX_DEVICES = 64;
std::mutex g_mu;
float* g_xn_ptr[MAX_DEVICES];   // device address of g_noalloc_xn per device ordinal (nullptr: not resolved yet)

thread_local char g_err[256] = "";

int fail(int code, const char* msg) {
  snprintf(g_err, sizeof(g_err), "%s", msg);
  return code;
}

// set-up, once per device, with that device current
int scratch_for_current_device(float** out) {
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) {
    snprintf(g_err, sizeof(g_err), "final_head_noalloc: cudaGetDevice: %s", cudaGetErrorString(e));
    return M2R2_CUDA;
  }
  if (dev < 0 || dev >= MAX_DEVICES) return fail(M2R2_UNSUPPORTED, "final_head_noalloc: device ordinal >= 64");
  std::lock_guard<std::mutex> lk(g_mu);
  if (!g_xn_ptr[dev]) {
    float* p = nullptr;
    e = cudaGetSymbolAddress((void**)&p, g_noalloc_xn);
    if (e != cudaSuccess || !p) {
      snprintf(g_err, sizeof(g_err), "final_head_noalloc: cudaGetSymbolAddress: %s", cudaGetErrorString(e));
      return M2R2_CUDA;
    }
    g_xn_ptr[dev] = p;
  }
  *out = g_xn_ptr[dev];
  return M2R2_OK;
}

}  // namespace

extern "C" int m2r2_final_head_noalloc(const float* h, const void* g_f, const void* w_lm, float* logits, int32_t m,
                                       int32_t d, int32_t vocab, int32_t dtype, float rms_eps, void* stream) {
  g_err[0] = 0;
  if (!h || !g_f || !w_lm || !logits) return fail(M2R2_INVALID_ARG, "final_head_noalloc: null pointer");
  if (dtype != M2R2_FP32 && dtype != M2R2_BF16) return fail(M2R2_INVALID_ARG, "final_head_noalloc: dtype must be M2R2_FP32 or M2R2_BF16");
  if (m < 1 || m > M2R2_NOALLOC_MAX_ROWS) {
    snprintf(g_err, sizeof(g_err), "final_head_noalloc: m = %d rows outside [1, %d] (M2R2_NOALLOC_MAX_ROWS: the static scratch holds no more)",
             (int)m, M2R2_NOALLOC_MAX_ROWS);
    return M2R2_CAPACITY;
  }
  if (d < 8 || d > M2R2_NOALLOC_MAX_D) {
    snprintf(g_err, sizeof(g_err), "final_head_noalloc: d = %d outside [8, %d] (M2R2_NOALLOC_MAX_D: the static scratch holds no more)",
             (int)d, M2R2_NOALLOC_MAX_D);
    return M2R2_CAPACITY;
  }
  if (d % 8) return fail(M2R2_INVALID_ARG, "final_head_noalloc: d must be a multiple of 8 (16-byte weight loads)");
  if (vocab < 1) return fail(M2R2_INVALID_ARG, "final_head_noalloc: vocab < 1");
  float* xn = nullptr;
  int rc = scratch_for_current_device(&xn);
  if (rc) return rc;
  cudaStream_t st = (cudaStream_t)stream;
  // xn[row] = rms(h[row]; g_f)   (Q1)   -> the static scratch
  launch_norm_lora(st, dtype, h, m, d, g_f, rms_eps, xn, nullptr, 0, 0, 0, nullptr, 0);
  // logits[row] = W_lm xn[row]
  GemvArgs g;
  memset(&g, 0, sizeof(g));
  g.W = w_lm; g.X = xn; g.ldx = d; g.n_rows = m; g.K = d; g.n_out = vocab; g.out = logits; g.ldo = vocab;
  launch_gemv(st, dtype, g, false);
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) {
    snprintf(g_err, sizeof(g_err), "final_head_noalloc: launch: %s", cudaGetErrorString(e));
    return M2R2_CUDA;
  }
  return M2R2_OK;
}

extern "C" const char* m2r2_noalloc_last_error(void) { return g_err; }
