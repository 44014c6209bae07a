// kernels_fused.cu — persistent fused dual-stream decode pass (bf16 storage, dense FFN, batch 1).
//
// One cooperative launch runs a whole pass (a1-a9 of SURVEY §8(a)): embed, then per layer
//   QKV   fused RMSNorm + QKV GEMV for h and p (+ adapters) with RoPE + KV append in the epilogue
//   ATTN  split-K flash-decode attention, slow query and accelerated query on the same K/V tiles
//   OPROJ O-projection + residual                        GATEUP RMSNorm + gate/up GEMV + SwiGLU
//   DOWN  down GEMV + residual = accelerated-residual update, gate reset p <- h
// and the LM head + greedy argmax (final head on h_N, or exit/draft head on p at a gate).
//
// Design (DESIGN.md §"Fused decode kernel"): one CTA per SM.  The big matrices are stored
// TILE-MAJOR: a stage = 64 output rows x 256 inputs of bf16 = 32 KB contiguous, stages ordered
// (row-block, k-chunk).  Weights never depend on activations, so ONE producer thread per CTA
// streams the CTA's statically known stage sequence of the WHOLE pass through a shared-memory
// ring with cp.async.bulk (UBLKCP) + mbarrier, running ahead across phase and grid barriers: HBM
// stays busy while the consumers wait for activations.  Eight consumer warps take 8 rows each of
// a stage, lanes stride K with 128-bit LDS, both activation rows (h, p) in registers per k-chunk.
// The stages of a phase are split evenly over the CTAs (a CTA's range may start/end inside a
// row-block): partial sums go to a fixed slot, the LAST contributor (atomic ticket) adds the slots
// in slot order and runs the phase epilogue, so results are deterministic.
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include <algorithm>
#include <vector>

#include "m2r2_fused.cuh"

namespace {

typedef __nv_bfloat16 bf16;
typedef unsigned long long u64;

constexpr int TILE_ROWS = 64;
constexpr int TILE_K = 256;
constexpr int STAGE_BYTES = TILE_ROWS * TILE_K * 2;   // 32 KB
constexpr int NSTAGE = 4;
constexpr int NCW = 8;                 // consumer warps
constexpr int NCT = NCW * 32;          // consumer threads
constexpr int NTHREADS = NCT + 32;     // + producer warp
constexpr int AREA_BYTES = 96 * 1024;  // activation rows (x) / attention K,V staging
constexpr int ATT_RED_FLOATS = 16 * 2 * (128 + 2);
constexpr int MISC_BYTES = 2560;
constexpr int SMEM_BYTES = NSTAGE * STAGE_BYTES + AREA_BYTES + MISC_BYTES;
constexpr int MAX_R = 16;              // adapter rank limit
constexpr long long SPIN_LIMIT = 4000000000ll;   // ~2 s of SM clocks before a wait gives up

enum { PH_QKV = 0, PH_OPROJ = 1, PH_GATEUP = 2, PH_DOWN = 3, PH_HEAD = 4, PH_EXIT = 5, N_PH = 6 };

struct FLayer {
  const uint4 *Wqkv, *Wo, *Wgu, *Wd;   // tile-major
  const bf16 *g1, *g2;
  const bf16 *Aqkv, *Bqkv, *Ao, *Bo, *Agu, *Bg, *Bu, *Ad, *Bd;
  bf16 *Kc, *Vc;                        // this layer's cache, sequence 0: [head][max_seq][dh]
  int accel;                            // layer carries p
  int gate;                             // 1 + gate index if layer+1 is a gate E_j, else 0
};

struct Ctl {
  unsigned int bar;        // grid-barrier arrivals (monotonic across launches)
  unsigned int abort_flag; // a wait timed out
  unsigned int abort_where;
  unsigned int pad;
  u64 amax[1 + M2R2_MAX_GATES];   // argmax keys: [0] head of the pass, [1+j] exit head of gate j
};

struct FParams {
  int n_layers_run, d, n_heads, dh, F, V, r, da, max_seq;
  int d_pad, F_pad;
  int rb_qkv, rb_o, rb_gu, rb_d, rb_v;
  float eps, scale;
  const FLayer* layers;
  const bf16 *embed, *gf, *lmA, *lmB;
  const uint4* Wlm;
  const int *sidx, *accel_cols;
  const float2* rope_tab;
  int *kv_len, *pending;
  const int* tok_in;
  int* tok_out;
  int* exit_tok;
  int n_gates, exit_heads, advance, head_stream, joff, do_trace, head_gate;
  float *resid, *attn_o, *act, *qbuf, *khat, *vhat, *pexit;
  float *part;
  int *cnt;
  float* apart;
  int* acnt;
  float *trace, *logits, *exit_logits;
  Ctl* ctl;
  unsigned int bar_base;
  const int *ls_full, *ls_draft;
  int ls_first, ls_n;
  float ls_beta;
  int ns;   // attention splits
  u64* tl;  // debug timeline (M2R2_FUSED_DEBUG builds), else nullptr
};

// ------------------------------------------------------------------ PTX helpers
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(u64* b, int count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(b)), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(u64* b, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(b)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(u64* b) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(b)) : "memory");
}
__device__ __forceinline__ bool mbar_try_wait(u64* b, uint32_t parity) {
  uint32_t ok;
  asm volatile(
      "{\n .reg .pred p;\n mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n selp.u32 %0, 1, 0, p;\n}\n"
      : "=r"(ok)
      : "r"(smem_u32(b)), "r"(parity)
      : "memory");
  return ok != 0;
}
// bulk async copy global -> shared, completion on an mbarrier (SASS: UBLKCP); weights are read
// once per pass: evict-first in L2
__device__ __forceinline__ void bulk_g2s(void* dst, const void* src, uint32_t bytes, u64* bar, u64 policy) {
  asm volatile(
      "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;"
      ::"r"(smem_u32(dst)), "l"(src), "r"(bytes), "r"(smem_u32(bar)), "l"(policy)
      : "memory");
}
__device__ __forceinline__ u64 policy_evict_first() {
  u64 p;
  asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(p));
  return p;
}
__device__ __forceinline__ u64 policy_evict_last() {
  u64 p;
  asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(p));
  return p;
}
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
__device__ __forceinline__ void bar_consumers() { asm volatile("bar.sync 1, %0;" ::"n"(NCT) : "memory"); }
__device__ __forceinline__ unsigned int ld_acquire(const unsigned int* p) {
  unsigned int v;
  asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
  return v;
}
__device__ __forceinline__ float ldcg(const float* p) { return __ldcg(p); }
__device__ __forceinline__ float4 ldcg4(const float* p) { return __ldcg((const float4*)p); }
__device__ __forceinline__ float bf(const bf16* p) { return __bfloat162float(*p); }
__device__ __forceinline__ float ldcg_bf16(const bf16* p) {   // written earlier in this launch by another SM: L2 only
  return __uint_as_float((unsigned int)__ldcg((const unsigned short*)p) << 16);
}
__device__ __forceinline__ float silu(float z) { return z / (1.f + __expf(-z)); }

__device__ __forceinline__ u64 amax_key(float v, int n) {
  unsigned int b = __float_as_uint(v);
  b = (b & 0x80000000u) ? ~b : (b | 0x80000000u);
  return ((u64)b << 32) | (u64)(0xFFFFFFFFu - (unsigned int)n);   // ties: lowest index wins
}

// stage range of virtual CTA v among G for a phase of S stages, and the owner of a stage
__device__ __forceinline__ int range_lo(int S, int v, int G) { return (int)(((long long)S * v) / G); }
__device__ __forceinline__ int stage_owner(int S, int s, int G) { return (int)((((long long)(s + 1)) * G + S - 1) / S) - 1; }
__device__ __forceinline__ int phase_rot(int layer, int ph, int G) { return (int)(((unsigned)(layer * 5 + ph) * 29u) % (unsigned)G); }

#ifdef M2R2_FUSED_DEBUG
constexpr int TL_MAX = 1024;
__device__ __forceinline__ u64 gtime() { u64 t; asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t)); return t; }
#define TL(ev) do { if (P.tl && threadIdx.x == 0 && tl_n < TL_MAX) { P.tl[(size_t)blockIdx.x * TL_MAX + tl_n] = (gtime() << 8) | (u64)(ev); ++tl_n; } } while (0)
#else
#define TL(ev) do { } while (0)
#endif

struct Smem {
  unsigned char* ring;
  float* area;
  float* tile_out;    // [64][2]
  float* u;           // [64] adapter down-projections of the current phase
  float* red;         // [64]
  u64* full;          // [NSTAGE]
  u64* empty;         // [NSTAGE]
  u64* abar;          // attention staging
  int* flag;          // [4]
};

__device__ __forceinline__ Smem carve_smem(unsigned char* base) {
  Smem s;
  s.ring = base;
  s.area = (float*)(base + NSTAGE * STAGE_BYTES);
  unsigned char* m = base + NSTAGE * STAGE_BYTES + AREA_BYTES;
  s.tile_out = (float*)m;            // 512 B
  s.u = (float*)(m + 512);           // 256 B
  s.red = (float*)(m + 768);         // 256 B
  s.full = (u64*)(m + 1024);
  s.empty = s.full + NSTAGE;
  s.abar = s.empty + NSTAGE;
  s.flag = (int*)(m + 1024 + 8 * (2 * NSTAGE + 1) + 8);
  return s;
}

__device__ __forceinline__ void set_abort(Ctl* ctl, unsigned int where) {
  if (atomicExch(&ctl->abort_flag, 1u) == 0u) ctl->abort_where = where;
}
__device__ __forceinline__ bool aborted(const Ctl* ctl) { return *(volatile const unsigned int*)&ctl->abort_flag != 0u; }

__device__ __forceinline__ void mbar_wait(u64* b, uint32_t parity, Ctl* ctl, unsigned int where) {
  if (mbar_try_wait(b, parity)) return;
  long long t0 = clock64();
  unsigned int n = 0;
  while (!mbar_try_wait(b, parity)) {
    if ((++n & 1023u) == 0u) {
      if (aborted(ctl)) return;
      if (clock64() - t0 > SPIN_LIMIT) { set_abort(ctl, where); return; }
    }
  }
}

// ------------------------------------------------------------------ grid barrier (all CTAs co-resident: cooperative launch)
__device__ __forceinline__ void grid_sync(const FParams& P, unsigned int& nbar, int G) {
  bar_consumers();
  if (threadIdx.x == 0) {
    __threadfence();
    atomicAdd(&P.ctl->bar, 1u);
    ++nbar;
    unsigned int target = P.bar_base + nbar * (unsigned int)G;
    long long t0 = clock64();
    unsigned int n = 0;
    while ((int)(ld_acquire(&P.ctl->bar) - target) < 0) {
      if ((++n & 255u) == 0u) {
        if (aborted(P.ctl)) break;
        if (clock64() - t0 > SPIN_LIMIT) { set_abort(P.ctl, 0x100u + nbar); break; }
      }
    }
    __threadfence();
  } else {
    ++nbar;
  }
  bar_consumers();
}

// ------------------------------------------------------------------ activation rows in shared memory
// x[stream][k] is stored as float4 planes so that a lane's 8 consecutive k are two conflict-free
// LDS.128: plane(half, stream)[g] = x[stream][8g + 4*half .. +4]
__device__ __forceinline__ float4* xplane(const Smem& sm, int half, int stream, int kpad8) {
  return (float4*)sm.area + (size_t)(half * 2 + stream) * kpad8;
}

// x <- rms(src; g) for both streams (stream 1 zero when the layer does not carry p)
__device__ void xload_norm(const FParams& P, const Smem& sm, const float* src0, const float* src1,
                           const bf16* g, int K, int kpad, bool have1) {
  const int tid = threadIdx.x, kpad8 = kpad / 8;
  float ss0 = 0.f, ss1 = 0.f;
  for (int i = tid; i < kpad / 4; i += NCT) {
    int k = i * 4;
    float4 a = make_float4(0.f, 0.f, 0.f, 0.f), b = a;
    if (k < K) {
      a = ldcg4(src0 + k);
      if (have1) b = ldcg4(src1 + k);
    }
    ss0 += a.x * a.x + a.y * a.y + a.z * a.z + a.w * a.w;
    ss1 += b.x * b.x + b.y * b.y + b.z * b.z + b.w * b.w;
    xplane(sm, i & 1, 0, kpad8)[i >> 1] = a;
    xplane(sm, i & 1, 1, kpad8)[i >> 1] = b;
  }
  ss0 = warp_sum(ss0);
  ss1 = warp_sum(ss1);
  if ((tid & 31) == 0) { sm.red[tid >> 5] = ss0; sm.red[8 + (tid >> 5)] = ss1; }
  bar_consumers();
  float t0 = 0.f, t1 = 0.f;
#pragma unroll
  for (int w = 0; w < NCW; ++w) { t0 += sm.red[w]; t1 += sm.red[8 + w]; }
  const float inv0 = rsqrtf(t0 / (float)K + P.eps), inv1 = rsqrtf(t1 / (float)K + P.eps);
  for (int i = tid; i < K / 4; i += NCT) {
    int k = i * 4;
    float g0 = bf(g + k), g1 = bf(g + k + 1), g2 = bf(g + k + 2), g3 = bf(g + k + 3);
    float4* pa = &xplane(sm, i & 1, 0, kpad8)[i >> 1];
    float4* pb = &xplane(sm, i & 1, 1, kpad8)[i >> 1];
    float4 a = *pa, b = *pb;
    a.x = a.x * inv0 * g0; a.y = a.y * inv0 * g1; a.z = a.z * inv0 * g2; a.w = a.w * inv0 * g3;
    b.x = b.x * inv1 * g0; b.y = b.y * inv1 * g1; b.z = b.z * inv1 * g2; b.w = b.w * inv1 * g3;
    *pa = a;
    *pb = b;
  }
  bar_consumers();
}

// x <- src (no norm)
__device__ void xload_plain(const Smem& sm, const float* src0, const float* src1, int K, int kpad, bool have1) {
  const int tid = threadIdx.x, kpad8 = kpad / 8;
  for (int i = tid; i < kpad / 4; i += NCT) {
    int k = i * 4;
    float4 a = make_float4(0.f, 0.f, 0.f, 0.f), b = a;
    if (k < K) {
      a = ldcg4(src0 + k);
      if (have1) b = ldcg4(src1 + k);
    }
    xplane(sm, i & 1, 0, kpad8)[i >> 1] = a;
    xplane(sm, i & 1, 1, kpad8)[i >> 1] = b;
  }
  bar_consumers();
}

// u[j] = A[j, :] . x^   (adapter down-projection of the accelerated row), rows j < n_rows.
// A is [n_rows][Kc] row-major; compact column c of A maps to x granule gmap[c/8 ...] when cols != nullptr.
__device__ void compute_u(const Smem& sm, const bf16* A, int n_rows, int Kc, const int* cols, int kpad8) {
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const float4* x0 = xplane(sm, 0, 1, kpad8);
  const float4* x1 = xplane(sm, 1, 1, kpad8);
  for (int j = warp; j < n_rows; j += NCW) {
    const bf16* a = A + (size_t)j * Kc;
    float acc = 0.f;
    for (int c = lane * 8; c < Kc; c += 256) {
      uint4 w = __ldg((const uint4*)(a + c));
      int g = (cols ? cols[c] : c) >> 3;
      float4 lo = x0[g], hi = x1[g];
      float f0, f1;
      bf16x2_to_f32(w.x, f0, f1); acc += f0 * lo.x + f1 * lo.y;
      bf16x2_to_f32(w.y, f0, f1); acc += f0 * lo.z + f1 * lo.w;
      bf16x2_to_f32(w.z, f0, f1); acc += f0 * hi.x + f1 * hi.y;
      bf16x2_to_f32(w.w, f0, f1); acc += f0 * hi.z + f1 * hi.w;
    }
    acc = warp_sum(acc);
    if (lane == 0) sm.u[j] = acc;
  }
  bar_consumers();
}

__device__ __forceinline__ float lora_dot(const bf16* Brow, const float* u, int r) {
  float s = 0.f;
  for (int q = 0; q < r; ++q) s += bf(Brow + q) * u[q];
  return s;
}

// ------------------------------------------------------------------ phase epilogues (one 64-row block, sums in sm.tile_out[row][stream])
struct PhaseCtx {
  int ph, layer, rb;
  const FLayer* L;
  int pos;          // position of the token of this pass
  bool accel;       // stream 1 live
};

__device__ void finalize_block(const FParams& P, const Smem& sm, const PhaseCtx& c) {
  const int tid = threadIdx.x;
  const float* T = sm.tile_out;
  const int d = P.d, dh = P.dh, half = dh >> 1, r = P.r;
  if (c.ph == PH_QKV) {
    // a3 fused: RoPE (pairs are adjacent packed rows) + KV append (slow) / k^,v^ kept in scratch (accel)
    if (tid < 64) {
      const int m = tid >> 1, s = tid & 1;
      const int r0 = c.rb * 64 + 2 * m;
      if (r0 < 3 * d && (s == 0 || c.accel)) {
        const int which = r0 / d, w = r0 % d, head = w / dh, i = w % dh;
        float v0 = T[(2 * m) * 2 + s], v1 = T[(2 * m + 1) * 2 + s];
        int e0, e1;   // element index inside the head of the two packed rows
        if (which < 2) { e0 = i >> 1; e1 = e0 + half; } else { e0 = i; e1 = i + 1; }
        bool live = true;
        if (s == 1) {
          const int si = P.sidx[head];
          live = si >= 0;
          if (live) {   // parallel adapters: + B (A x^)   (Q3)
            const bf16* B = c.L->Bqkv + ((size_t)which * P.da + (size_t)si * dh) * r;
            v0 += lora_dot(B + (size_t)e0 * r, sm.u + which * r, r);
            v1 += lora_dot(B + (size_t)e1 * r, sm.u + which * r, r);
          }
        }
        if (live) {
          if (which < 2) {
            float2 cs = P.rope_tab[(size_t)c.pos * half + e0];
            float a = v0 * cs.x - v1 * cs.y, b = v1 * cs.x + v0 * cs.y;
            v0 = a; v1 = b;
          }
          const int o0 = head * dh + e0, o1 = head * dh + e1;
          if (which == 0) {
            P.qbuf[s * d + o0] = v0; P.qbuf[s * d + o1] = v1;
          } else if (s == 0) {
            bf16* C = (which == 1 ? c.L->Kc : c.L->Vc) + ((size_t)head * P.max_seq + c.pos) * dh;
            C[e0] = __float2bfloat16_rn(v0);
            C[e1] = __float2bfloat16_rn(v1);
          } else {
            float* C = which == 1 ? P.khat : P.vhat;
            C[o0] = v0; C[o1] = v1;
          }
        }
      }
    }
  } else if (c.ph == PH_OPROJ) {
    if (tid < 128) {
      const int row = tid >> 1, s = tid & 1, n = c.rb * 64 + row;
      if (n < d && (s == 0 || c.accel)) {
        float v = T[row * 2 + s];
        if (s == 1) v += lora_dot(c.L->Bo + (size_t)n * r, sm.u, r);
        float* R = P.resid + s * d + n;
        *R = ldcg(R) + v;
      }
    }
  } else if (c.ph == PH_GATEUP) {
    // packed rows: warp-group of 8 = gate rows n..n+3 then up rows n..n+3
    if (tid < 64) {
      const int nl = tid >> 1, s = tid & 1, n = c.rb * 32 + nl;
      if (n < P.F && (s == 0 || c.accel)) {
        const int grow = (nl >> 2) * 8 + (nl & 3), urow = grow + 4;
        float g = T[grow * 2 + s], up = T[urow * 2 + s];
        if (s == 1) {
          g += lora_dot(c.L->Bg + (size_t)n * r, sm.u, r);
          up += lora_dot(c.L->Bu + (size_t)n * r, sm.u + r, r);
        }
        P.act[s * P.F_pad + n] = silu(g) * up;
      }
    }
  } else if (c.ph == PH_DOWN) {
    // accelerated-residual update (Eq. 2) and gate: p <- h (L82, L101)
    if (tid < 64) {
      const int n = c.rb * 64 + tid;
      if (n < d) {
        float h = ldcg(P.resid + n) + T[tid * 2];
        P.resid[n] = h;
        float p = h;
        if (c.accel) p = ldcg(P.resid + d + n) + T[tid * 2 + 1] + lora_dot(c.L->Bd + (size_t)n * r, sm.u, r);
        if (P.do_trace) {
          float* tr = P.trace + (size_t)(c.layer + 1) * 2 * d;
          tr[n] = h;
          tr[d + n] = p;
        }
        if (c.accel) {
          if (c.L->gate) {
            P.pexit[(size_t)(c.L->gate - 1) * d + n] = p;
            p = h;
          }
          P.resid[d + n] = p;
        }
      }
    }
  } else {
    // PH_HEAD (stream 0: final head on h_N) / PH_EXIT (stream 1: exit or draft head on p at a gate)
    const int s = c.ph == PH_HEAD ? P.head_stream : 1;
    const int gate = c.ph == PH_HEAD ? P.head_gate : c.layer;   // for PH_EXIT `layer` carries the gate index
    const bool is_final = (c.ph == PH_HEAD && P.head_stream == 0);
    if (tid < 64) {
      const int n = c.rb * 64 + tid;
      u64 key = 0ull;
      if (n < P.V) {
        float v = T[tid * 2 + s];
        if (s == 1 && P.lmB) v += lora_dot(P.lmB + (size_t)n * r, sm.u, r);
        float* lg = is_final ? P.logits : P.exit_logits + (size_t)gate * P.V;
        lg[n] = v;
        const int* script = is_final ? P.ls_full : P.ls_draft;
        if (script) {
          int q = c.pos + 1 - P.ls_first;   // logits of the token at pos predict pos+1
          if (q >= 0 && q < P.ls_n && script[q] == n) v += P.ls_beta;
        }
        key = amax_key(v, n);
      }
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) {
        u64 other = __shfl_xor_sync(0xffffffffu, key, o);
        key = other > key ? other : key;
      }
      if ((tid & 31) == 0 && key) atomicMax(&P.ctl->amax[c.ph == PH_HEAD ? 0 : 1 + gate], key);
    }
  }
}

// ------------------------------------------------------------------ one GEMV phase (consumer side)
struct GemvDesc {
  int n_rb, n_kc;     // row-blocks, k-chunks (stages = n_rb * n_kc)
  int kpad8;          // kpad / 8
};

__device__ __noinline__ void gemv_phase(const FParams& P, const Smem& sm, const GemvDesc& gd, const PhaseCtx& pc0, int G,
                                        unsigned int& stage_ctr, float* part, int* cnt, int& tl_n) {
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int S = gd.n_rb * gd.n_kc;
  const int rot = phase_rot(pc0.layer, pc0.ph, G);
  const int v = ((int)blockIdx.x + rot) % G;
  const int s0 = range_lo(S, v, G), s1 = range_lo(S, v + 1, G);
  float acc[8][2];
#pragma unroll
  for (int i = 0; i < 8; ++i) acc[i][0] = acc[i][1] = 0.f;
  const float4* xa0p = xplane(sm, 0, 0, gd.kpad8);
  const float4* xa1p = xplane(sm, 1, 0, gd.kpad8);
  const float4* xb0p = xplane(sm, 0, 1, gd.kpad8);
  const float4* xb1p = xplane(sm, 1, 1, gd.kpad8);
  for (int s = s0; s < s1; ++s) {
    const int rb = s / gd.n_kc, kc = s - rb * gd.n_kc;
    const unsigned int slot = stage_ctr % NSTAGE, use = stage_ctr / NSTAGE;
    ++stage_ctr;
    const int g = kc * 32 + lane;
    const float4 xa0 = xa0p[g], xa1 = xa1p[g], xb0 = xb0p[g], xb1 = xb1p[g];
    mbar_wait(&sm.full[slot], use & 1u, P.ctl, 0x200u + pc0.ph);
    const uint4* st = (const uint4*)(sm.ring + (size_t)slot * STAGE_BYTES) + (warp * 8) * 32 + lane;
#pragma unroll
    for (int i = 0; i < 8; ++i) {
      const uint4 w = st[i * 32];
      float f0, f1;
      bf16x2_to_f32(w.x, f0, f1);
      acc[i][0] += f0 * xa0.x; acc[i][1] += f0 * xb0.x; acc[i][0] += f1 * xa0.y; acc[i][1] += f1 * xb0.y;
      bf16x2_to_f32(w.y, f0, f1);
      acc[i][0] += f0 * xa0.z; acc[i][1] += f0 * xb0.z; acc[i][0] += f1 * xa0.w; acc[i][1] += f1 * xb0.w;
      bf16x2_to_f32(w.z, f0, f1);
      acc[i][0] += f0 * xa1.x; acc[i][1] += f0 * xb1.x; acc[i][0] += f1 * xa1.y; acc[i][1] += f1 * xb1.y;
      bf16x2_to_f32(w.w, f0, f1);
      acc[i][0] += f0 * xa1.z; acc[i][1] += f0 * xb1.z; acc[i][0] += f1 * xa1.w; acc[i][1] += f1 * xb1.w;
    }
    __syncwarp();
    if (lane == 0) mbar_arrive(&sm.empty[slot]);   // stage consumed by this warp
    TL(40);
    if (kc == gd.n_kc - 1 || s == s1 - 1) {
      // ---- end of this CTA's segment of row-block rb: reduce over lanes (16 values, butterfly)
      float v16[16];
#pragma unroll
      for (int i = 0; i < 8; ++i) { v16[2 * i] = acc[i][0]; v16[2 * i + 1] = acc[i][1]; acc[i][0] = acc[i][1] = 0.f; }
#pragma unroll
      for (int i = 0; i < 8; ++i) {
        bool up = lane & 16;
        float send = up ? v16[i] : v16[i + 8], keep = up ? v16[i + 8] : v16[i];
        v16[i] = keep + __shfl_xor_sync(0xffffffffu, send, 16);
      }
#pragma unroll
      for (int i = 0; i < 4; ++i) {
        bool up = lane & 8;
        float send = up ? v16[i] : v16[i + 4], keep = up ? v16[i + 4] : v16[i];
        v16[i] = keep + __shfl_xor_sync(0xffffffffu, send, 8);
      }
#pragma unroll
      for (int i = 0; i < 2; ++i) {
        bool up = lane & 4;
        float send = up ? v16[i] : v16[i + 2], keep = up ? v16[i + 2] : v16[i];
        v16[i] = keep + __shfl_xor_sync(0xffffffffu, send, 4);
      }
      {
        bool up = lane & 2;
        float send = up ? v16[0] : v16[1], keep = up ? v16[1] : v16[0];
        v16[0] = keep + __shfl_xor_sync(0xffffffffu, send, 2);
      }
      v16[0] += __shfl_xor_sync(0xffffffffu, v16[0], 1);
      const int idx = (lane >> 1) & 15;   // = row_in_warp*2 + stream
      if ((lane & 1) == 0) sm.tile_out[(warp * 8 + (idx >> 1)) * 2 + (idx & 1)] = v16[0];
      bar_consumers();
      // ---- contributors of this row-block
      // (S >= G: every CTA owns >= 1 stage, so the owners of a row-block are consecutive CTAs;
      //  S < G: every stage has its own CTA, so there is one contributor per k-chunk)
      const int vf = stage_owner(S, rb * gd.n_kc, G), vl = stage_owner(S, rb * gd.n_kc + gd.n_kc - 1, G);
      const int ncontrib = S >= G ? vl - vf + 1 : gd.n_kc;
      const int myslot = S >= G ? v - vf : kc;
      PhaseCtx pc = pc0;
      pc.rb = rb;
      if (ncontrib == 1) {
        finalize_block(P, sm, pc);
      } else {
        if (tid < 128) __stcg(part + ((size_t)(rb * gd.n_kc + myslot) * 128 + tid), sm.tile_out[tid]);
        __threadfence();
        bar_consumers();
        if (tid == 0) {
          int old = atomicAdd(&cnt[rb], 1);
          int last = old == ncontrib - 1;
          if (last) cnt[rb] = 0;
          sm.flag[0] = last;
        }
        bar_consumers();
        if (sm.flag[0]) {
          __threadfence();
          if (tid < 128) {
            float sum = 0.f;
            for (int sl = 0; sl < ncontrib; ++sl) sum += ldcg(part + ((size_t)(rb * gd.n_kc + sl) * 128 + tid));
            sm.tile_out[tid] = sum;
          }
          bar_consumers();
          finalize_block(P, sm, pc);
        }
      }
      bar_consumers();   // tile_out / flag reuse
    }
  }
}

// ------------------------------------------------------------------ attention phase (a4): split-K flash-decode, dual query
// Work item = (head, split).  K/V of positions [0, pos) come from the cache through a bulk copy into
// the activation area; the token's own key/value (slow: K[pos], V[pos] as stored = rounded; accel:
// k^, v^ from scratch) is added by the head's last contributor, which also merges
// the split partials in split order.
__device__ void attn_phase(const FParams& P, const Smem& sm, const FLayer* L, int pos, bool accel, int G,
                           unsigned int& attn_uses) {
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int dh = P.dh, d = P.d, lpp = dh >> 3, NS = P.ns;
  const int seg = lane >> 4, sl = lane & 15;
  const bool active = sl < lpp;
  const int CH = (AREA_BYTES - ATT_RED_FLOATS * 4) / (4 * dh);   // positions per staging round
  bf16* Ks = (bf16*)sm.area;
  bf16* Vs = Ks + (size_t)CH * dh;
  float* red = sm.area + (size_t)CH * dh;   // after K and V staging (2*CH*dh bf16 = CH*dh floats)
  const u64 pol = policy_evict_last();
  const int items = P.n_heads * NS;
  for (int w = blockIdx.x; w < items; w += G) {
    const int head = w / NS, sp = w - head * NS;
    const bool q1 = accel && P.sidx[head] >= 0;
    const int chunk = (pos + NS - 1) / NS;
    const int p0 = min(pos, sp * chunk), p1 = min(pos, p0 + chunk);
    float qa[8], qb[8];
#pragma unroll
    for (int e = 0; e < 8; ++e) { qa[e] = 0.f; qb[e] = 0.f; }
    if (active) {
#pragma unroll
      for (int e = 0; e < 8; ++e) {
        qa[e] = ldcg(P.qbuf + head * dh + sl * 8 + e) * P.scale;
        if (q1) qb[e] = ldcg(P.qbuf + d + head * dh + sl * 8 + e) * P.scale;
      }
    }
    float m0 = -INFINITY, l0 = 0.f, m1 = -INFINITY, l1 = 0.f, o0[8], o1[8];
#pragma unroll
    for (int e = 0; e < 8; ++e) { o0[e] = 0.f; o1[e] = 0.f; }
    for (int c0 = p0; c0 < p1; c0 += CH) {
      const int cn = min(CH, p1 - c0);
      if (tid == 0) {
        fence_proxy_async();
        const uint32_t bytes = (uint32_t)cn * dh * 2;
        mbar_expect_tx(sm.abar, 2 * bytes);
        bulk_g2s(Ks, L->Kc + ((size_t)head * P.max_seq + c0) * dh, bytes, sm.abar, pol);
        bulk_g2s(Vs, L->Vc + ((size_t)head * P.max_seq + c0) * dh, bytes, sm.abar, pol);
      }
      mbar_wait(sm.abar, attn_uses & 1u, P.ctl, 0x300u);
      ++attn_uses;
      for (int ub = warp * 2; ub < cn; ub += NCW * 2) {
        const int u = ub + seg;
        const bool valid = u < cn;
        float kf[8], vf[8];
#pragma unroll
        for (int e = 0; e < 8; ++e) { kf[e] = 0.f; vf[e] = 0.f; }
        if (valid && active) {
          uint4 kk = *(const uint4*)(Ks + (size_t)u * dh + sl * 8);
          uint4 vv = *(const uint4*)(Vs + (size_t)u * dh + sl * 8);
          bf16x2_to_f32(kk.x, kf[0], kf[1]); bf16x2_to_f32(kk.y, kf[2], kf[3]);
          bf16x2_to_f32(kk.z, kf[4], kf[5]); bf16x2_to_f32(kk.w, kf[6], kf[7]);
          bf16x2_to_f32(vv.x, vf[0], vf[1]); bf16x2_to_f32(vv.y, vf[2], vf[3]);
          bf16x2_to_f32(vv.z, vf[4], vf[5]); bf16x2_to_f32(vv.w, vf[6], vf[7]);
        }
        float sa = 0.f, sb = 0.f;
#pragma unroll
        for (int e = 0; e < 8; ++e) { sa += qa[e] * kf[e]; sb += qb[e] * kf[e]; }
#pragma unroll
        for (int o = 8; o > 0; o >>= 1) {
          sa += __shfl_xor_sync(0xffffffffu, sa, o);
          sb += __shfl_xor_sync(0xffffffffu, sb, o);
        }
        if (valid) {
          float mn = fmaxf(m0, sa), corr = __expf(m0 - mn), p = __expf(sa - mn);
          l0 = l0 * corr + p;
#pragma unroll
          for (int e = 0; e < 8; ++e) o0[e] = o0[e] * corr + p * vf[e];
          m0 = mn;
          if (q1) {
            mn = fmaxf(m1, sb); corr = __expf(m1 - mn); p = __expf(sb - mn);
            l1 = l1 * corr + p;
#pragma unroll
            for (int e = 0; e < 8; ++e) o1[e] = o1[e] * corr + p * vf[e];
            m1 = mn;
          }
        }
      }
      bar_consumers();   // staging buffers free for the next round / phase
    }
    // ---- merge the 16 lane segments of the CTA -> one partial per query
    {
      const int gseg = warp * 2 + seg;
      float* dst0 = red + ((size_t)gseg * 2 + 0) * (dh + 2);
      float* dst1 = red + ((size_t)gseg * 2 + 1) * (dh + 2);
      if (active) {
#pragma unroll
        for (int e = 0; e < 8; ++e) { dst0[sl * 8 + e] = o0[e]; dst1[sl * 8 + e] = o1[e]; }
      }
      if (sl == 0) { dst0[dh] = m0; dst0[dh + 1] = l0; dst1[dh] = m1; dst1[dh + 1] = l1; }
    }
    bar_consumers();
    for (int i = tid; i < 2 * dh; i += NCT) {
      const int q = i / dh, j = i - q * dh;
      float M = -INFINITY;
      for (int s = 0; s < 16; ++s) {
        const float* src = red + ((size_t)s * 2 + q) * (dh + 2);
        if (src[dh + 1] > 0.f) M = fmaxf(M, src[dh]);
      }
      float Lsum = 0.f, O = 0.f;
      for (int s = 0; s < 16; ++s) {
        const float* src = red + ((size_t)s * 2 + q) * (dh + 2);
        float ls = src[dh + 1];
        if (ls > 0.f) {
          float wgt = __expf(src[dh] - M);
          Lsum += ls * wgt;
          O += src[j] * wgt;
        }
      }
      float* pp = P.apart + ((size_t)(head * NS + sp) * 2 + q) * (dh + 2);
      __stcg(pp + j, O);
      if (j == 0) { __stcg(pp + dh, M); __stcg(pp + dh + 1, Lsum); }
    }
    __threadfence();
    bar_consumers();
    if (tid == 0) {
      int old = atomicAdd(&P.acnt[head], 1);
      int last = old == NS - 1;
      if (last) P.acnt[head] = 0;
      sm.flag[1] = last;
    }
    bar_consumers();
    if (sm.flag[1]) {
      __threadfence();
      // own-token scores: warp 0 -> slow query vs K[pos] (as stored), warp 1 -> accel query vs k^
      if (warp < 2) {
        float part = 0.f;
        if (warp == 0 || q1) {
          for (int j = lane; j < dh; j += 32) {
            float qv = ldcg(P.qbuf + warp * d + head * dh + j);
            float kv = warp == 0 ? ldcg_bf16(L->Kc + ((size_t)head * P.max_seq + pos) * dh + j) : ldcg(P.khat + head * dh + j);
            part += qv * kv;
          }
        }
        part = warp_sum(part);
        if (lane == 0) sm.red[16 + warp] = part * P.scale;
      }
      bar_consumers();
      for (int i = tid; i < 2 * dh; i += NCT) {
        const int q = i / dh, j = i - q * dh;
        if (q == 1 && !q1) continue;
        const float s_own = sm.red[16 + q];
        float M = s_own;
        for (int s = 0; s < NS; ++s) {
          const float* pp = P.apart + ((size_t)(head * NS + s) * 2 + q) * (dh + 2);
          if (ldcg(pp + dh + 1) > 0.f) M = fmaxf(M, ldcg(pp + dh));
        }
        float Lsum = 0.f, O = 0.f;
        for (int s = 0; s < NS; ++s) {
          const float* pp = P.apart + ((size_t)(head * NS + s) * 2 + q) * (dh + 2);
          float ls = ldcg(pp + dh + 1);
          if (ls > 0.f) {
            float wgt = __expf(ldcg(pp + dh) - M);
            Lsum += ls * wgt;
            O += ldcg(pp + j) * wgt;
          }
        }
        float wgt = __expf(s_own - M);
        float vown = q == 0 ? ldcg_bf16(L->Vc + ((size_t)head * P.max_seq + pos) * dh + j) : ldcg(P.vhat + head * dh + j);
        Lsum += wgt;
        O += wgt * vown;
        P.attn_o[q * d + head * dh + j] = O / Lsum;
      }
    }
    bar_consumers();
  }
}

// ------------------------------------------------------------------ producer: the CTA's weight-stage stream of the whole pass
__device__ __forceinline__ void produce_phase(const FParams& P, const Smem& sm, const uint4* W, int n_rb, int n_kc,
                                              int layer, int ph, int G, unsigned int& ctr, u64 pol) {
  const int S = n_rb * n_kc;
  const int v = ((int)blockIdx.x + phase_rot(layer, ph, G)) % G;
  const int s0 = range_lo(S, v, G), s1 = range_lo(S, v + 1, G);
  for (int s = s0; s < s1; ++s) {
    const unsigned int slot = ctr % NSTAGE, use = ctr / NSTAGE;
    ++ctr;
    mbar_wait(&sm.empty[slot], (use & 1u) ^ 1u, P.ctl, 0x400u + ph);
    mbar_expect_tx(&sm.full[slot], STAGE_BYTES);
    bulk_g2s(sm.ring + (size_t)slot * STAGE_BYTES, (const unsigned char*)W + (size_t)s * STAGE_BYTES, STAGE_BYTES,
             &sm.full[slot], pol);
  }
}

__global__ void __launch_bounds__(NTHREADS, 1) m2r2_fused_decode_kernel(const FParams P) {
  extern __shared__ __align__(1024) unsigned char smem_raw[];
  const Smem sm = carve_smem(smem_raw);
  const int tid = threadIdx.x, G = gridDim.x;
  if (tid == 0) {
    for (int i = 0; i < NSTAGE; ++i) { mbar_init(&sm.full[i], 1); mbar_init(&sm.empty[i], NCW); }
    mbar_init(sm.abar, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();
  const int n_kc_d = P.d_pad / TILE_K, n_kc_f = P.F_pad / TILE_K;
  const int head_layers = P.n_layers_run;

  if (tid >= NCT) {
    // ================= producer warp: one thread streams every weight stage of the pass
    if (tid == NCT) {
      const u64 pol = policy_evict_first();
      unsigned int ctr = 0;
      for (int i = 0; i < P.n_layers_run; ++i) {
        const FLayer* L = P.layers + i;
        produce_phase(P, sm, L->Wqkv, P.rb_qkv, n_kc_d, i, PH_QKV, G, ctr, pol);
        produce_phase(P, sm, L->Wo, P.rb_o, n_kc_d, i, PH_OPROJ, G, ctr, pol);
        produce_phase(P, sm, L->Wgu, P.rb_gu, n_kc_d, i, PH_GATEUP, G, ctr, pol);
        produce_phase(P, sm, L->Wd, P.rb_d, n_kc_f, i, PH_DOWN, G, ctr, pol);
        if (L->gate && L->accel && P.exit_heads && !(P.head_stream == 1 && i + 1 == head_layers))
          produce_phase(P, sm, P.Wlm, P.rb_v, n_kc_d, L->gate - 1, PH_EXIT, G, ctr, pol);
      }
      produce_phase(P, sm, P.Wlm, P.rb_v, n_kc_d, head_layers, PH_HEAD, G, ctr, pol);
    }
    return;
  }

  // ================= consumers
  unsigned int nbar = 0, stage_ctr = 0, attn_uses = 0;
  int tl_n = 0;
  (void)tl_n;
  const int d = P.d;
  const int pos = *(volatile int*)P.kv_len + P.joff;
  const int tok = *(volatile const int*)P.tok_in;
  // a1: embed + stream init, p_0 <- h_0 (L82)
  for (int k = blockIdx.x * NCT + tid; k < d; k += G * NCT) {
    float v = bf(P.embed + (size_t)tok * d + k);
    P.resid[k] = v;
    P.resid[d + k] = v;
    if (P.do_trace) { P.trace[k] = v; P.trace[d + k] = v; }
  }
  TL(1);
  grid_sync(P, nbar, G);
  TL(2);

  for (int i = 0; i < P.n_layers_run; ++i) {
    const FLayer* L = P.layers + i;
    const bool accel = L->accel != 0;
    PhaseCtx pc;
    pc.layer = i; pc.L = L; pc.pos = pos; pc.accel = accel; pc.rb = 0;
    GemvDesc gd;
    // ---- a2 (+a3): RMSNorm + QKV, RoPE + KV append
    xload_norm(P, sm, P.resid, P.resid + d, L->g1, d, P.d_pad, accel);
    if (accel) compute_u(sm, L->Aqkv, 3 * P.r, d, nullptr, P.d_pad / 8);
    TL(10);
    pc.ph = PH_QKV; gd.n_rb = P.rb_qkv; gd.n_kc = n_kc_d; gd.kpad8 = P.d_pad / 8;
    gemv_phase(P, sm, gd, pc, G, stage_ctr, P.part, P.cnt, tl_n);
    TL(11);
    grid_sync(P, nbar, G);
    TL(12);
    // ---- a4: attention
    attn_phase(P, sm, L, pos, accel, G, attn_uses);
    TL(13);
    grid_sync(P, nbar, G);
    TL(14);
    // ---- a5: O-proj + residual
    xload_plain(sm, P.attn_o, P.attn_o + d, d, P.d_pad, accel);
    if (accel) compute_u(sm, L->Ao, P.r, P.da, P.accel_cols, P.d_pad / 8);
    TL(15);
    pc.ph = PH_OPROJ; gd.n_rb = P.rb_o;
    gemv_phase(P, sm, gd, pc, G, stage_ctr, P.part, P.cnt, tl_n);
    TL(16);
    grid_sync(P, nbar, G);
    TL(17);
    // ---- a6: RMSNorm + gate/up + SwiGLU
    xload_norm(P, sm, P.resid, P.resid + d, L->g2, d, P.d_pad, accel);
    if (accel) compute_u(sm, L->Agu, 2 * P.r, d, nullptr, P.d_pad / 8);
    TL(18);
    pc.ph = PH_GATEUP; gd.n_rb = P.rb_gu;
    gemv_phase(P, sm, gd, pc, G, stage_ctr, P.part, P.cnt, tl_n);
    TL(19);
    grid_sync(P, nbar, G);
    TL(20);
    // ---- a7: down + residual, gate
    xload_plain(sm, P.act, P.act + P.F_pad, P.F, P.F_pad, accel);
    if (accel) compute_u(sm, L->Ad, P.r, P.F, nullptr, P.F_pad / 8);
    TL(21);
    pc.ph = PH_DOWN; gd.n_rb = P.rb_d; gd.n_kc = n_kc_f; gd.kpad8 = P.F_pad / 8;
    gemv_phase(P, sm, gd, pc, G, stage_ctr, P.part, P.cnt, tl_n);
    TL(22);
    grid_sync(P, nbar, G);
    TL(23);
    // ---- a8: exit head at a gate (Eq. 4), when asked
    if (L->gate && accel && P.exit_heads && !(P.head_stream == 1 && i + 1 == head_layers)) {
      const float* pe = P.pexit + (size_t)(L->gate - 1) * d;
      xload_norm(P, sm, pe, pe, P.gf, d, P.d_pad, true);
      if (P.lmA) compute_u(sm, P.lmA, P.r, d, nullptr, P.d_pad / 8);
      PhaseCtx pe_c = pc;
      pe_c.ph = PH_EXIT; pe_c.layer = L->gate - 1;
      gd.n_rb = P.rb_v; gd.n_kc = n_kc_d; gd.kpad8 = P.d_pad / 8;
      gemv_phase(P, sm, gd, pe_c, G, stage_ctr, P.part, P.cnt, tl_n);
      grid_sync(P, nbar, G);
    }
  }
  // ---- a9 / a8: head of the pass
  {
    PhaseCtx pc;
    pc.layer = head_layers; pc.L = nullptr; pc.pos = pos; pc.accel = true; pc.rb = 0; pc.ph = PH_HEAD;
    const float* src = P.head_stream == 0 ? P.resid : P.pexit + (size_t)P.head_gate * d;
    xload_norm(P, sm, src, src, P.gf, d, P.d_pad, true);
    if (P.head_stream == 1 && P.lmA) compute_u(sm, P.lmA, P.r, d, nullptr, P.d_pad / 8);
    GemvDesc gd;
    gd.n_rb = P.rb_v; gd.n_kc = n_kc_d; gd.kpad8 = P.d_pad / 8;
    TL(30);
    gemv_phase(P, sm, gd, pc, G, stage_ctr, P.part, P.cnt, tl_n);
    TL(31);
    grid_sync(P, nbar, G);
    TL(32);
  }
  if (blockIdx.x == 0 && tid == 0) {
    u64 key = *(volatile u64*)&P.ctl->amax[0];
    int t = (int)(0xFFFFFFFFu - (unsigned int)(key & 0xFFFFFFFFull));
    *P.tok_out = t;
    P.ctl->amax[0] = 0ull;
    for (int j = 0; j < P.n_gates; ++j) {
      u64 kj = *(volatile u64*)&P.ctl->amax[1 + j];
      if (kj) P.exit_tok[j] = (int)(0xFFFFFFFFu - (unsigned int)(kj & 0xFFFFFFFFull));
      P.ctl->amax[1 + j] = 0ull;
    }
    if (P.advance) { *P.kv_len = pos + 1; *P.pending = t; }
  }
}

// ------------------------------------------------------------------ repack: row-major [n_out, K] -> tile-major stages
// map 0: natural rows; 1: QKV (RoPE pairs (j, j+dh/2) of q and k made adjacent); 2: gate/up interleaved
// (8-row groups = gate n..n+3, up n..n+3).  Rows / columns beyond the matrix are zero.
__global__ void pack_kernel(uint4* __restrict__ dst, const bf16* __restrict__ src, const bf16* __restrict__ src2,
                            int map, int n_out, int K, int n_rb, int n_kc, int d, int dh) {
  const size_t total = (size_t)n_rb * n_kc * (STAGE_BYTES / 16);
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < total; i += (size_t)gridDim.x * blockDim.x) {
    const size_t stage = i / (STAGE_BYTES / 16);
    const int within = (int)(i % (STAGE_BYTES / 16));
    const int row = within / 32, c8 = within % 32;
    const int rb = (int)(stage / n_kc), kc = (int)(stage % n_kc);
    const int r = rb * 64 + row, k = kc * TILE_K + c8 * 8;
    const bf16* base = nullptr;
    if (map == 0) {
      if (r < n_out) base = src + (size_t)r * K;
    } else if (map == 1) {
      if (r < n_out) {
        int which = r / d, w = r % d, sr = r;
        if (which < 2) {
          int head = w / dh, e = w % dh;
          sr = which * d + head * dh + (e >> 1) + (e & 1) * (dh >> 1);
        }
        base = src + (size_t)sr * K;
      }
    } else {
      int n = (r >> 3) * 4 + (r & 3);
      if (n < n_out) base = ((r & 7) < 4 ? src : src2) + (size_t)n * K;
    }
    uint4 v = make_uint4(0u, 0u, 0u, 0u);
    if (base && k < K) v = *(const uint4*)(base + k);   // K % 8 == 0
    dst[i] = v;
  }
}

}  // namespace

// ==================================================================================== host side
struct FusedImpl {
  int G = 0;                  // CTAs = SMs
  FParams p;                  // template (per-launch fields filled in fused_run)
  FLayer* d_layers = nullptr; // in scratch
  Ctl* d_ctl = nullptr;
  int* d_sidx = nullptr;
  unsigned int bar_base = 0;
  Ctl* h_ctl = nullptr;       // pinned
  bool bound = false;
  u64* d_tl = nullptr;        // debug timeline (M2R2_FUSED_DEBUG builds)
  // scratch carve
  float *resid, *attn_o, *act, *qbuf, *khat, *vhat, *pexit, *part, *apart;
  int *cnt, *acnt, *accel_cols;
};

static int pad_to(int v, int m) { return (v + m - 1) / m * m; }

bool fused_config_ok(const m2r2_config& c) {
  if (c.dtype != M2R2_BF16 || c.n_experts != 0) return false;
  if (c.head_dim % 8 || c.head_dim > 128 || (c.head_dim & 1)) return false;
  if (c.d_model % 8 || c.d_ff % 8) return false;
  if (c.accel_enabled && c.adapter_rank > MAX_R) return false;
  int kmax = std::max(pad_to(c.d_model, TILE_K), pad_to(c.d_ff, TILE_K));
  if ((size_t)kmax * 2 * sizeof(float) > AREA_BYTES) return false;
  if ((AREA_BYTES - ATT_RED_FLOATS * 4) / (4 * c.head_dim) < 16) return false;
  return true;
}

struct PackedDims {
  int d_pad, F_pad, rb_qkv, rb_o, rb_gu, rb_d, rb_v;
  size_t st_qkv, st_o, st_gu, st_d, st_v;   // stages
};
static PackedDims packed_dims(const m2r2_config& c) {
  PackedDims q;
  q.d_pad = pad_to(c.d_model, TILE_K);
  q.F_pad = pad_to(c.d_ff, TILE_K);
  q.rb_qkv = pad_to(3 * c.d_model, TILE_ROWS) / TILE_ROWS;
  q.rb_o = pad_to(c.d_model, TILE_ROWS) / TILE_ROWS;
  q.rb_gu = pad_to(2 * pad_to(c.d_ff, 4), TILE_ROWS) / TILE_ROWS;
  q.rb_d = q.rb_o;
  q.rb_v = pad_to(c.vocab, TILE_ROWS) / TILE_ROWS;
  q.st_qkv = (size_t)q.rb_qkv * (q.d_pad / TILE_K);
  q.st_o = (size_t)q.rb_o * (q.d_pad / TILE_K);
  q.st_gu = (size_t)q.rb_gu * (q.d_pad / TILE_K);
  q.st_d = (size_t)q.rb_d * (q.F_pad / TILE_K);
  q.st_v = (size_t)q.rb_v * (q.d_pad / TILE_K);
  return q;
}

size_t fused_weights_bytes(const m2r2_config& c) {
  if (!fused_config_ok(c)) return 0;
  PackedDims q = packed_dims(c);
  return ((q.st_qkv + q.st_o + q.st_gu + q.st_d) * (size_t)c.n_layers + q.st_v) * STAGE_BYTES + 1024;
}

void fused_carve(const m2r2_config& c, Carver& cv, FusedState* fs) {
  if (!fused_config_ok(c)) return;
  PackedDims q = packed_dims(c);
  const size_t d = c.d_model, G = std::max(1, c.n_gates);
  int max_rb = std::max(std::max(q.rb_qkv, q.rb_gu), std::max(q.rb_v, q.rb_o));
  int max_kc = std::max(q.d_pad, q.F_pad) / TILE_K;
  FusedImpl* im = fs ? fs->impl : nullptr;
#define FTAKE(field, T, n) { T* p_ = cv.take<T>(n); if (im) im->field = p_; }
  FTAKE(d_layers, FLayer, c.n_layers)
  FTAKE(d_ctl, Ctl, 1)
  FTAKE(d_sidx, int, c.n_heads)
  FTAKE(accel_cols, int, std::max(8, c.n_accel_heads * c.head_dim))
  FTAKE(resid, float, 2 * d) FTAKE(attn_o, float, 2 * d) FTAKE(act, float, 2 * (size_t)q.F_pad)
  FTAKE(qbuf, float, 2 * d) FTAKE(khat, float, d) FTAKE(vhat, float, d) FTAKE(pexit, float, G * d)
  FTAKE(part, float, (size_t)max_rb * max_kc * 128)
  FTAKE(cnt, int, max_rb)
  FTAKE(apart, float, (size_t)c.n_heads * M2R2_MAX_SPLITS * 2 * (c.head_dim + 2))
  FTAKE(acnt, int, c.n_heads)
#undef FTAKE
}

int fused_create(const m2r2_config& c, FusedState* fs) {
  fs->supported = false;
  fs->impl = nullptr;
  if (!fused_config_ok(c)) return 0;
  int dev = 0, sms = 0, coop = 0, max_smem = 0;
  if (cudaGetDevice(&dev) != cudaSuccess) return M2R2_CUDA;
  cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, dev);
  cudaDeviceGetAttribute(&max_smem, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev);
  if (!coop || max_smem < SMEM_BYTES || sms < 1) return 0;   // per-operation kernels serve this device
  if (cudaFuncSetAttribute(m2r2_fused_decode_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM_BYTES) != cudaSuccess) {
    cudaGetLastError();
    return 0;
  }
  int occ = 0;
  if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, m2r2_fused_decode_kernel, NTHREADS, SMEM_BYTES) != cudaSuccess || occ < 1) {
    cudaGetLastError();
    return 0;
  }
  FusedImpl* im = new FusedImpl();
  im->G = sms;
  if (cudaMallocHost((void**)&im->h_ctl, sizeof(Ctl)) != cudaSuccess) { delete im; return M2R2_CUDA; }
  fs->impl = im;
  fs->supported = true;
  return 0;
}

void fused_destroy(FusedState* fs) {
  if (fs->impl) {
    if (fs->impl->h_ctl) cudaFreeHost(fs->impl->h_ctl);
    delete fs->impl;
  }
  fs->impl = nullptr;
  fs->supported = false;
}

bool fused_supported(const m2r2_config&, const FusedState* fs) { return fs->supported && fs->impl && fs->impl->bound; }

static int pack(cudaStream_t st, void* dst, const void* src, const void* src2, int map, int n_out, int K, int n_rb,
                int n_kc, int d, int dh) {
  pack_kernel<<<1184, 256, 0, st>>>((uint4*)dst, (const bf16*)src, (const bf16*)src2, map, n_out, K, n_rb, n_kc, d, dh);
  return cudaGetLastError() == cudaSuccess ? 0 : M2R2_CUDA;
}

int fused_bind(const m2r2_config& c, FusedState* fs, cudaStream_t st, void* packed, const void* embed,
               const void* gf, const void* lm_head, const void* lm_A, const void* lm_B, const DevLayer* layers,
               void* kv, const float2* rope_tab) {
  if (!fs->supported) return 0;
  FusedImpl* im = fs->impl;
  PackedDims q = packed_dims(c);
  const int d = c.d_model, dh = c.head_dim, F = c.d_ff;
  const int kc_d = q.d_pad / TILE_K, kc_f = q.F_pad / TILE_K;
  char* wp = (char*)packed;
  wp = (char*)(((uintptr_t)wp + 1023) & ~(uintptr_t)1023);
  std::vector<FLayer> hl(c.n_layers);
  const size_t per = (size_t)c.max_batch * c.n_heads * c.max_seq * dh;   // elements per layer of K (or V)
  for (int i = 0; i < c.n_layers; ++i) {
    const DevLayer& L = layers[i];
    FLayer& f = hl[i];
    memset(&f, 0, sizeof(f));
    f.Wqkv = (const uint4*)wp; wp += q.st_qkv * STAGE_BYTES;
    f.Wo = (const uint4*)wp; wp += q.st_o * STAGE_BYTES;
    f.Wgu = (const uint4*)wp; wp += q.st_gu * STAGE_BYTES;
    f.Wd = (const uint4*)wp; wp += q.st_d * STAGE_BYTES;
    if (pack(st, (void*)f.Wqkv, L.wqkv, nullptr, 1, 3 * d, d, q.rb_qkv, kc_d, d, dh)) return M2R2_CUDA;
    if (pack(st, (void*)f.Wo, L.wo, nullptr, 0, d, d, q.rb_o, kc_d, d, dh)) return M2R2_CUDA;
    if (pack(st, (void*)f.Wgu, L.wgate, L.wup, 2, F, d, q.rb_gu, kc_d, d, dh)) return M2R2_CUDA;
    if (pack(st, (void*)f.Wd, L.wdown, nullptr, 0, d, F, q.rb_d, kc_f, d, dh)) return M2R2_CUDA;
    f.g1 = (const bf16*)L.g1; f.g2 = (const bf16*)L.g2;
    f.Aqkv = (const bf16*)L.Aqkv; f.Bqkv = (const bf16*)L.Bqkv; f.Ao = (const bf16*)L.Ao; f.Bo = (const bf16*)L.Bo;
    f.Agu = (const bf16*)L.Agu; f.Bg = (const bf16*)L.Bg; f.Bu = (const bf16*)L.Bu; f.Ad = (const bf16*)L.Ad; f.Bd = (const bf16*)L.Bd;
    f.Kc = (bf16*)kv + (size_t)i * per;
    f.Vc = (bf16*)kv + (size_t)c.n_layers * per + (size_t)i * per;
    f.accel = (c.accel_enabled && i < c.accel_end_layer) ? 1 : 0;
    f.gate = 0;
    for (int j = 0; j < c.n_gates; ++j) if (c.gates[j] == i + 1) f.gate = j + 1;
  }
  const uint4* Wlm = (const uint4*)wp;
  if (pack(st, (void*)Wlm, lm_head, nullptr, 0, c.vocab, d, q.rb_v, kc_d, d, dh)) return M2R2_CUDA;
  if (cudaMemcpyAsync(im->d_layers, hl.data(), sizeof(FLayer) * c.n_layers, cudaMemcpyHostToDevice, st) != cudaSuccess) return M2R2_CUDA;
  std::vector<int> sidx(c.n_heads, -1), cols(std::max(8, c.n_accel_heads * dh), 0);
  if (c.accel_enabled)
    for (int s = 0; s < c.n_accel_heads; ++s) {
      sidx[c.accel_heads[s]] = s;
      for (int j = 0; j < dh; ++j) cols[s * dh + j] = c.accel_heads[s] * dh + j;
    }
  if (cudaMemcpyAsync(im->d_sidx, sidx.data(), sizeof(int) * c.n_heads, cudaMemcpyHostToDevice, st) != cudaSuccess) return M2R2_CUDA;
  if (cudaMemcpyAsync(im->accel_cols, cols.data(), sizeof(int) * cols.size(), cudaMemcpyHostToDevice, st) != cudaSuccess) return M2R2_CUDA;
  cudaMemsetAsync(im->d_ctl, 0, sizeof(Ctl), st);
  cudaMemsetAsync(im->attn_o, 0, sizeof(float) * 2 * d, st);
  cudaMemsetAsync(im->act, 0, sizeof(float) * 2 * q.F_pad, st);
  cudaMemsetAsync(im->cnt, 0, sizeof(int) * std::max(std::max(q.rb_qkv, q.rb_gu), std::max(q.rb_v, q.rb_o)), st);
  cudaMemsetAsync(im->acnt, 0, sizeof(int) * c.n_heads, st);
  cudaMemsetAsync(im->pexit, 0, sizeof(float) * std::max(1, c.n_gates) * d, st);
  if (cudaStreamSynchronize(st) != cudaSuccess) return M2R2_CUDA;   // hl / sidx / cols are stack-owned
  im->bar_base = 0;
  FParams& p = im->p;
  memset(&p, 0, sizeof(p));
  p.d = d; p.n_heads = c.n_heads; p.dh = dh; p.F = F; p.V = c.vocab; p.r = c.accel_enabled ? c.adapter_rank : 0;
  p.da = c.n_accel_heads * dh; p.max_seq = c.max_seq;
  p.d_pad = q.d_pad; p.F_pad = q.F_pad;
  p.rb_qkv = q.rb_qkv; p.rb_o = q.rb_o; p.rb_gu = q.rb_gu; p.rb_d = q.rb_d; p.rb_v = q.rb_v;
  p.eps = c.rms_eps; p.scale = 1.0f / sqrtf((float)dh);
  p.layers = im->d_layers;
  p.embed = (const bf16*)embed; p.gf = (const bf16*)gf; p.lmA = (const bf16*)lm_A; p.lmB = (const bf16*)lm_B;
  p.Wlm = Wlm;
  p.sidx = im->d_sidx; p.accel_cols = im->accel_cols; p.rope_tab = rope_tab;
  p.n_gates = c.n_gates;
  p.resid = im->resid; p.attn_o = im->attn_o; p.act = im->act; p.qbuf = im->qbuf; p.khat = im->khat; p.vhat = im->vhat;
  p.pexit = im->pexit; p.part = im->part; p.cnt = im->cnt; p.apart = im->apart; p.acnt = im->acnt;
  p.ctl = im->d_ctl;
  p.tl = nullptr;
#ifdef M2R2_FUSED_DEBUG
  if (getenv("M2R2_TL_OUT") && !im->d_tl) cudaMalloc((void**)&im->d_tl, sizeof(u64) * TL_MAX * im->G);
  p.tl = im->d_tl;
#endif
  im->bound = true;
  return 0;
}

int fused_run(const m2r2_config& c, FusedState* fs, cudaStream_t st, const FusedRun& run, int* d_kv_len,
              int* d_pending, int kv_len_host, float* trace, float* logits, float* exit_logits, int* d_exit_tok,
              const int* ls_full, const int* ls_draft, int ls_first, int ls_n, float ls_beta, int64_t* launches) {
  FusedImpl* im = fs->impl;
  FParams p = im->p;
  const int G = im->G;
  p.n_layers_run = run.n_layers;
  p.kv_len = d_kv_len; p.pending = d_pending; p.tok_in = run.tok_in; p.tok_out = run.tok_out; p.exit_tok = d_exit_tok;
  p.exit_heads = run.exit_heads; p.advance = run.advance; p.head_stream = run.head_stream; p.joff = run.joff;
  p.do_trace = run.trace;
  p.head_gate = 0;
  if (run.head_stream == 1) {
    int gj = -1;
    for (int j = 0; j < c.n_gates; ++j) if (c.gates[j] == run.n_layers) gj = j;
    if (gj < 0) return M2R2_INVALID_ARG;
    p.head_gate = gj;
  }
  p.trace = trace; p.logits = logits; p.exit_logits = exit_logits;
  p.ls_full = ls_full; p.ls_draft = ls_draft; p.ls_first = ls_first; p.ls_n = ls_n; p.ls_beta = ls_beta;
  // attention splits: one item per CTA where possible
  const int pos = kv_len_host + run.joff;
  int ns = std::max(1, G / c.n_heads);
  ns = std::min(ns, std::max(1, (pos + 31) / 32));
  ns = std::min(ns, (int)M2R2_MAX_SPLITS);
  p.ns = ns;
  // grid barriers of this launch (must match the kernel's sequence)
  unsigned int nbar = 1;
  for (int i = 0; i < run.n_layers; ++i) {
    nbar += 5;
    bool accel = c.accel_enabled && i < c.accel_end_layer;
    bool gate = false;
    for (int j = 0; j < c.n_gates; ++j) gate |= (c.gates[j] == i + 1);
    if (gate && accel && run.exit_heads && !(run.head_stream == 1 && i + 1 == run.n_layers)) nbar += 1;
  }
  nbar += 1;
  p.bar_base = im->bar_base;
  im->bar_base += nbar * (unsigned int)G;
  void* args[] = {(void*)&p};
  cudaError_t e = cudaLaunchCooperativeKernel((const void*)m2r2_fused_decode_kernel, dim3(G), dim3(NTHREADS), args,
                                              SMEM_BYTES, st);
  if (e != cudaSuccess) return M2R2_CUDA;
  if (launches) *launches += 1;
  return 0;
}

int fused_check(FusedState* fs, cudaStream_t st, char* msg, size_t n) {
  if (!fs->supported || !fs->impl || !fs->impl->bound) return 0;
  FusedImpl* im = fs->impl;
  if (cudaMemcpyAsync(im->h_ctl, im->d_ctl, sizeof(Ctl), cudaMemcpyDeviceToHost, st) != cudaSuccess) return M2R2_CUDA;
  if (cudaStreamSynchronize(st) != cudaSuccess) return M2R2_CUDA;
#ifdef M2R2_FUSED_DEBUG
  if (im->d_tl && getenv("M2R2_TL_OUT")) {   // dump the timeline of the last launch
    std::vector<u64> h((size_t)TL_MAX * im->G);
    cudaMemcpy(h.data(), im->d_tl, h.size() * sizeof(u64), cudaMemcpyDeviceToHost);
    FILE* f = fopen(getenv("M2R2_TL_OUT"), "wb");
    if (f) { int hdr[2] = {im->G, TL_MAX}; fwrite(hdr, sizeof(int), 2, f); fwrite(h.data(), sizeof(u64), h.size(), f); fclose(f); }
  }
#endif
  if (im->h_ctl->abort_flag) {
    snprintf(msg, n, "fused kernel wait timed out (site 0x%x)", im->h_ctl->abort_where);
    // re-arm: barrier counter and flags back to a clean state
    cudaMemsetAsync(im->d_ctl, 0, sizeof(Ctl), st);
    cudaStreamSynchronize(st);
    im->bar_base = 0;
    return M2R2_CUDA;
  }
  return 0;
}
