// kernels_fused.cu — persistent fused dual-stream decode pass, v2 (bf16 storage, dense FFN, batch 1).
//
// One cooperative launch runs a whole pass (a1-a9 of SURVEY §8(a)): embed, then per layer
//   QKV   fused RMSNorm + QKV GEMV for h and p (+ adapters) with RoPE + KV append in the epilogue
//   ATTN  split-K flash-decode attention, slow query and accelerated query on the same K/V loads
//   OPROJ O-projection (split-K, partial sums to fixed slots)
//   GATEUP residual + RMSNorm + gate/up GEMV + SwiGLU
//   DOWN  down GEMV (split-K slots); the accelerated-residual update and the gate reset p <- h
//          happen where the next phase loads the residual
// and the LM head + greedy argmax (final head on h_N, or exit/draft head on p at a gate).
//
// Design (DESIGN.md §"Fused decode kernel"): one CTA per SM, 8 consumer warps + 1 producer warp.
//  * Weights are stored FRAGMENT-MAJOR: a tile = 16 output rows x 16 inputs laid out so that lane
//    L's 16 bytes are its A fragment of mma.sync.m16n8k16; a stage = one row-tile x 1024 inputs =
//    64 tiles = 32 KB contiguous; stages ordered (row-tile, k-stage).
//  * Weights never depend on activations, so ONE producer thread per CTA streams the CTA's
//    statically known stage sequence of the WHOLE pass through a 4-stage shared-memory ring with
//    cp.async.bulk (UBLKCP) + mbarrier, and keeps an L2 prefetch window (cp.async.bulk.prefetch.L2)
//    running further ahead, across phase boundaries and grid barriers: HBM stays busy while the
//    consumers wait for activations.  The KV ranges a CTA will attend to are prefetched the same way.
//  * Consumers: one LDS.128 per lane = one A fragment; the B operand is the activation vector split
//    into bf16 hi + lo parts (columns h_hi, h_lo, p_hi, p_lo of the n=8 tile), so the product is
//    exact to ~2^-17 and accumulates in fp32 on the tensor pipe (HMMA) at ~2 instructions per 256
//    weights.  It is a GEMV, not a contraction: the tensor pipe is used as a wide FMA, the bound is HBM.
//  * Row-owned phases (QKV, GATEUP, heads): a CTA owns whole row-tiles, epilogue is local.
//    Split-K phases (OPROJ, DOWN): a CTA owns a contiguous stage range; partial sums of a row-tile go
//    to slot (contributor index); the NEXT phase's loader adds residual + slots in slot order
//    (deterministic, no tickets, no atomics on data).
//  * Adapter down-projections u = A x^ are computed distributed (each CTA one row
//    chunk) right after the loader, published with a release counter, and picked up at the first
//    epilogue of the phase.
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include <algorithm>
#include <vector>

#include "m2r2_fused.cuh"

namespace {

typedef __nv_bfloat16 bf16;
typedef unsigned long long u64;

constexpr int STAGE_K = 1024;                  // inputs per stage
constexpr int STAGE_TILES = STAGE_K / 16;      // 64 m16k16 tiles
constexpr int STAGE_BYTES = STAGE_TILES * 512; // 32 KB
constexpr int NSTAGE = 4;
constexpr int NCW = 8;                 // consumer warps
constexpr int NCT = NCW * 32;          // consumer threads
constexpr int NTHREADS = NCT + 32;     // + producer warp
constexpr int TPW = STAGE_TILES / NCW; // tiles per warp per stage (8)
constexpr int KMAX = 8192;             // largest padded inner dimension
constexpr int XCOL = KMAX + 8;         // bf16 elements per activation column (+8: LDS.128 bank spread)
constexpr int X_BYTES = 4 * XCOL * 2;  // h_hi, h_lo, p_hi, p_lo
constexpr int RED_FLOATS = 2 * NCW * 32;
constexpr int MISC_BYTES = RED_FLOATS * 4 + 4096;
constexpr int SMEM_BYTES = NSTAGE * STAGE_BYTES + X_BYTES + MISC_BYTES;
constexpr int MAX_R = 16;              // adapter rank limit
constexpr int MAX_NJ = 3 * MAX_R;
constexpr int UPART_Q = 64;            // max k-chunks per adapter row
constexpr int MAX_SLOTS = KMAX / STAGE_K;
constexpr int NORM_CH = 4;             // float4 chunks per thread in a norm loader (d <= 4096)
constexpr int PF_DEFAULT = 10;         // L2 prefetch window, stages ahead of the ring
constexpr long long SPIN_LIMIT = 4000000000ll;   // ~2 s of SM clocks before a wait gives up

enum { PH_QKV = 0, PH_OPROJ = 1, PH_GATEUP = 2, PH_DOWN = 3, PH_HEAD = 4, PH_EXIT = 5, N_PH = 6 };

struct FLayer {
  const uint4 *Wqkv, *Wo, *Wgu, *Wd;   // fragment-major
  const bf16 *g1, *g2;
  const bf16 *Aqkv, *Bqkv, *Ao, *Bo, *Agu, *Bg, *Bu, *Ad, *Bd;
  bf16 *Kc, *Vc;                        // this layer's cache, sequence 0: [head][max_seq][dh]
  int accel;                            // layer carries p
  int gate;                             // 1 + gate index if layer+1 is a gate E_j, else 0
  const unsigned char* ad_lo;           // the layer's adapter tensors are one contiguous HBM range
  unsigned int ad_bytes;
};

struct Ctl {
  unsigned int bar;        // grid-barrier arrivals (monotonic across launches)
  unsigned int abort_flag; // a wait timed out
  unsigned int abort_where;
  unsigned int ucnt;       // adapter-partial publications of this launch (reset at its end)
  u64 amax[1 + M2R2_MAX_GATES];   // argmax keys: [0] head of the pass, [1+j] exit head of gate j
};

struct FParams {
  int n_layers_run, d, n_heads, dh, F, V, r, da, max_seq;
  int d_pad, F_pad;
  int rt_qkv, rt_o, rt_gu, rt_d, rt_v;    // row-tiles per matrix
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
  float *RA, *RB;            // residual pair [2][d]: RA = (h', p') after attention; RB = (h_i, p_i) entering a layer
  float *oslots, *dslots;    // [MAX_SLOTS][2][d] split-K partial sums of OPROJ / DOWN
  float *act, *qbuf, *khat, *vhat, *pexit;
  float *apart;              // [head][split][2][dh+4]
  float *upart;              // [2][MAX_NJ][UPART_Q]
  float *trace, *logits, *exit_logits;
  Ctl* ctl;
  unsigned int bar_base;
  const int *ls_full, *ls_draft;
  int ls_first, ls_n;
  float ls_beta;
  int ns;        // attention splits
  int pos_host;  // kv_len + joff as the host knows it (producer-side KV prefetch only)
  int pf_ahead;  // L2 prefetch window in stages
  u64* tl;       // debug timeline (M2R2_FUSED_DEBUG builds), else nullptr
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
__device__ __forceinline__ void bulk_prefetch_l2(const void* src, uint32_t bytes) {
  asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(src), "r"(bytes) : "memory");
}
__device__ __forceinline__ u64 policy_evict_first() {
  u64 p;
  asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(p));
  return p;
}
__device__ __forceinline__ void bar_consumers() { asm volatile("bar.sync 1, %0;" ::"n"(NCT) : "memory"); }
__device__ __forceinline__ unsigned int ld_acquire(const unsigned int* p) {
  unsigned int v;
  asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
  return v;
}
__device__ __forceinline__ float ldcg(const float* p) { return __ldcg(p); }
__device__ __forceinline__ float4 ldcg4(const float* p) { return __ldcg((const float4*)p); }
__device__ __forceinline__ uint4 ldcg16(const void* p) { return __ldcg((const uint4*)p); }
__device__ __forceinline__ float bf(const bf16* p) { return __bfloat162float(*p); }
__device__ __forceinline__ float silu(float z) { return z / (1.f + __expf(-z)); }
__device__ __forceinline__ void mma_bf16(float c[4], const uint4& a, uint32_t b0, uint32_t b1) {
  asm volatile(
      "mma.sync.aligned.m16n8k16.row.col.f32.bf16.bf16.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
      : "+f"(c[0]), "+f"(c[1]), "+f"(c[2]), "+f"(c[3])
      : "r"(a.x), "r"(a.y), "r"(a.z), "r"(a.w), "r"(b0), "r"(b1));
}

__device__ __forceinline__ u64 amax_key(float v, int n) {
  unsigned int b = __float_as_uint(v);
  b = (b & 0x80000000u) ? ~b : (b | 0x80000000u);
  return ((u64)b << 32) | (u64)(0xFFFFFFFFu - (unsigned int)n);   // ties: lowest index wins
}

// ------------------------------------------------------------------ static work split
// A phase has S stages (row-tile-major).  Virtual CTA v of G owns units [U*v/G, U*(v+1)/G) where a
// unit is `gran` consecutive stages (gran = stages per row-tile for row-owned phases, 1 for split-K).
__device__ __forceinline__ int range_lo(int U, int v, int G) { return (int)(((long long)U * v) / G); }
__device__ __forceinline__ int unit_owner(int U, int u, int G) { return (int)((((long long)(u + 1)) * G + U - 1) / U) - 1; }
__device__ __forceinline__ int phase_rot(int layer, int ph, int G) { return (int)(((unsigned)(layer * 5 + ph) * 29u) % (unsigned)G); }

#ifdef M2R2_FUSED_DEBUG
constexpr int TL_MAX = 2048;
__device__ __forceinline__ u64 gtime() { u64 t; asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t)); return t; }
#define TL(ev) do { if (P.tl && threadIdx.x == 0 && tl_n < TL_MAX) { P.tl[(size_t)blockIdx.x * TL_MAX + tl_n] = (gtime() << 8) | (u64)(ev); ++tl_n; } } while (0)
#else
#define TL(ev) do { } while (0)
#endif

// ------------------------------------------------------------------ shared memory map (fixed offsets: every access stays in the shared window)
constexpr int OFF_X = NSTAGE * STAGE_BYTES;
constexpr int OFF_RED = OFF_X + X_BYTES;              // [2][NCW][32] floats
constexpr int OFF_TILE = OFF_RED + RED_FLOATS * 4;    // [16][2] floats
constexpr int OFF_U = OFF_TILE + 256;                 // [MAX_NJ] floats
constexpr int OFF_SRED = OFF_U + 256;                 // [64] floats
constexpr int OFF_BAR = OFF_SRED + 256;               // full[NSTAGE], empty[NSTAGE]
constexpr int OFF_UTMP = OFF_BAR + 256;               // [256] floats
static_assert(OFF_UTMP + 1024 <= SMEM_BYTES, "shared memory map");

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
__device__ __forceinline__ void grid_sync(Ctl* ctl, unsigned int bar_base, unsigned int& nbar, int G) {
  bar_consumers();
  ++nbar;
  if (threadIdx.x == 0) {
    __threadfence();
    atomicAdd(&ctl->bar, 1u);
    const unsigned int target = bar_base + nbar * (unsigned int)G;
    long long t0 = clock64();
    unsigned int n = 0;
    while ((int)(ld_acquire(&ctl->bar) - target) < 0) {
      if ((++n & 255u) == 0u) {
        if (aborted(ctl)) break;
        if (clock64() - t0 > SPIN_LIMIT) { set_abort(ctl, 0x100u + nbar); break; }
      }
    }
    __threadfence();
  }
  bar_consumers();
}

// ------------------------------------------------------------------ activation vectors in shared memory
// Four bf16 columns (h_hi, h_lo, p_hi, p_lo) of XCOL elements.  Within every group of 64 inputs the
// order is [t][tile i][half][2] so that lane (g, t) of a warp reads the B fragments (b0, b1) of four
// consecutive m16n8k16 tiles with two LDS.128:  pos(k) = 64*(k/64) + 16*t + 4*i + 2*half + (k&1),
// i = (k/16)%4, t = ((k%16)%8)/2, half = (k%16)/8.
__device__ __forceinline__ int xpos(int k) {
  const int o = k & 15;
  return (k & ~63) + (((o & 7) >> 1) << 4) + (((k >> 4) & 3) << 2) + ((o >> 3) << 1) + (o & 1);
}
__device__ __forceinline__ uint32_t pack_bf16(bf16 a, bf16 b) {
  return (uint32_t)__bfloat16_as_ushort(a) | ((uint32_t)__bfloat16_as_ushort(b) << 16);
}
// store x[k..k+3] (k % 4 == 0) as hi + lo parts into the column pair (hi, lo)
__device__ __forceinline__ void xstore4(bf16* hi, bf16* lo, int k, float4 v) {
  const int p = xpos(k);
  const bf16 h0 = __float2bfloat16_rn(v.x), h1 = __float2bfloat16_rn(v.y), h2 = __float2bfloat16_rn(v.z), h3 = __float2bfloat16_rn(v.w);
  const bf16 l0 = __float2bfloat16_rn(v.x - __bfloat162float(h0)), l1 = __float2bfloat16_rn(v.y - __bfloat162float(h1));
  const bf16 l2 = __float2bfloat16_rn(v.z - __bfloat162float(h2)), l3 = __float2bfloat16_rn(v.w - __bfloat162float(h3));
  *(uint32_t*)(hi + p) = pack_bf16(h0, h1);
  *(uint32_t*)(hi + p + 16) = pack_bf16(h2, h3);
  *(uint32_t*)(lo + p) = pack_bf16(l0, l1);
  *(uint32_t*)(lo + p + 16) = pack_bf16(l2, l3);
}
__device__ __forceinline__ float xval(const bf16* hi, const bf16* lo, int k) {
  const int p = xpos(k);
  return __bfloat162float(hi[p]) + __bfloat162float(lo[p]);
}
__device__ __forceinline__ float4 f4add(float4 a, float4 b) { return make_float4(a.x + b.x, a.y + b.y, a.z + b.z, a.w + b.w); }
__device__ __forceinline__ float f4ss(float4 a) { return a.x * a.x + a.y * a.y + a.z * a.z + a.w * a.w; }
__device__ __forceinline__ void st4(float* p, float4 v) { __stcg((float4*)p, v); }

// contributors of row-tile rt in a split-K phase of n_rt x nks stages
__device__ __forceinline__ int n_contrib(int n_rt, int nks, int rt, int G) {
  const int S = n_rt * nks;
  if (S < G) return nks;
  return unit_owner(S, rt * nks + nks - 1, G) - unit_owner(S, rt * nks, G) + 1;
}

enum { LN_QKV = 0, LN_GU = 1, LN_HEAD_H = 2, LN_HEAD_P = 3 };

// Residual loader of the norm phases.  Every CTA rebuilds the full residual pair
//   (h, p) = base + sum over split-K slots of the producing phase      (Eq. 1 / Eq. 2 residual adds)
// applies the gate  p <- h when the producing layer ends at a gate, writes its
// share of the pair back (wb), and leaves x = rms(.; g) of both streams in shared memory.
struct LoadSrc {
  const float* base;     // [2][d] or nullptr (then emb)
  const bf16* emb;       // embedding row
  const float* slots;    // or nullptr
  int n_rt, nks;         // geometry of the producing split-K phase
  bool p_live;           // the producing layer carried p
  int gate;              // 1 + gate index: emit pexit, then p <- h
};
__device__ __forceinline__ void loader_norm(const FParams& P, bf16* x, float* sred, int mode, const LoadSrc& src, float* wb,
                                            float* trace_dst, const bf16* g, int G) {
  const int tid = threadIdx.x, d = P.d;
  bar_consumers();   // x of the previous phase is dead in every warp
  float4 xh[NORM_CH], xp[NORM_CH];
  uint2 ge[NORM_CH];
  float ssh = 0.f, ssp = 0.f;
#pragma unroll
  for (int j = 0; j < NORM_CH; ++j) {
    const int ci = tid + j * NCT, k = ci * 4;
    xh[j] = make_float4(0.f, 0.f, 0.f, 0.f);
    xp[j] = xh[j];
    ge[j] = make_uint2(0u, 0u);
    if (k < d) {
      // every load of this chunk is independent of the others: one L2 round trip
      ge[j] = __ldg((const uint2*)(g + k));
      float4 hv, pv;
      if (src.base) {
        hv = ldcg4(src.base + k);
        pv = src.p_live ? ldcg4(src.base + d + k) : hv;
      } else {
        const uint2 e = __ldg((const uint2*)(src.emb + k));
        bf16x2_to_f32(e.x, hv.x, hv.y);
        bf16x2_to_f32(e.y, hv.z, hv.w);
        pv = hv;
      }
      if (src.slots) {
        const int nc = n_contrib(src.n_rt, src.nks, k >> 4, G);
        float4 sh[3], sp[3];
#pragma unroll
        for (int sl = 0; sl < 3; ++sl) {
          sh[sl] = make_float4(0.f, 0.f, 0.f, 0.f);
          sp[sl] = sh[sl];
          if (sl < nc) {
            sh[sl] = ldcg4(src.slots + (size_t)(sl * 2) * d + k);
            if (src.p_live) sp[sl] = ldcg4(src.slots + (size_t)(sl * 2 + 1) * d + k);
          }
        }
#pragma unroll
        for (int sl = 0; sl < 3; ++sl) {
          if (sl < nc) { hv = f4add(hv, sh[sl]); pv = f4add(pv, sp[sl]); }
        }
        for (int sl = 3; sl < nc; ++sl) {
          hv = f4add(hv, ldcg4(src.slots + (size_t)(sl * 2) * d + k));
          if (src.p_live) pv = f4add(pv, ldcg4(src.slots + (size_t)(sl * 2 + 1) * d + k));
        }
      }
      if (!src.p_live) pv = hv;
      const bool owner = (ci % G) == (int)blockIdx.x;
      const float4 pbefore = pv;
      if (src.gate) {
        if (owner) st4(P.pexit + (size_t)(src.gate - 1) * d + k, pv);
        pv = hv;
      }
      if (owner && trace_dst) { st4(trace_dst + k, hv); st4(trace_dst + d + k, pbefore); }
      if (owner && wb) { st4(wb + k, hv); st4(wb + d + k, pv); }
      if (mode == LN_HEAD_P) { xh[j] = pbefore; xp[j] = pbefore; }
      else if (mode == LN_HEAD_H) { xh[j] = hv; xp[j] = hv; }
      else { xh[j] = hv; xp[j] = pv; }
      ssh += f4ss(xh[j]);
      ssp += f4ss(xp[j]);
    }
  }
  ssh = warp_sum(ssh);
  ssp = warp_sum(ssp);
  if ((tid & 31) == 0) { sred[tid >> 5] = ssh; sred[NCW + (tid >> 5)] = ssp; }
  bar_consumers();
  float th = 0.f, tp = 0.f;
#pragma unroll
  for (int w = 0; w < NCW; ++w) { th += sred[w]; tp += sred[NCW + w]; }
  const float ih = rsqrtf(th / (float)d + P.eps), ip = rsqrtf(tp / (float)d + P.eps);
  bf16 *c0 = x, *c1 = x + XCOL, *c2 = x + 2 * XCOL, *c3 = x + 3 * XCOL;
#pragma unroll
  for (int j = 0; j < NORM_CH; ++j) {
    const int ci = tid + j * NCT, k = ci * 4;
    if (k < P.d_pad) {
      float4 a = xh[j], b = xp[j];
      if (k < d) {
        float g0, g1, g2, g3;
        bf16x2_to_f32(ge[j].x, g0, g1);
        bf16x2_to_f32(ge[j].y, g2, g3);
        a.x = a.x * ih * g0; a.y = a.y * ih * g1; a.z = a.z * ih * g2; a.w = a.w * ih * g3;
        b.x = b.x * ip * g0; b.y = b.y * ip * g1; b.z = b.z * ip * g2; b.w = b.w * ip * g3;
      }
      xstore4(c0, c1, k, a);
      xstore4(c2, c3, k, b);
    }
  }
  bar_consumers();
}

// x <- attention output of both queries: merge of the split partials (m, l, o) in split order (a4)
__device__ __forceinline__ void loader_attn(const FParams& P, bf16* x, bool accel) {
  const int tid = threadIdx.x, d = P.d, dh = P.dh, NS = P.ns;
  bar_consumers();
  bf16 *c0 = x, *c1 = x + XCOL, *c2 = x + 2 * XCOL, *c3 = x + 3 * XCOL;
  for (int idx = tid; idx < 2 * (P.d_pad >> 2); idx += NCT) {
    const int q = idx >= (P.d_pad >> 2), k = (idx - q * (P.d_pad >> 2)) * 4;
    float4 o = make_float4(0.f, 0.f, 0.f, 0.f);
    if (k < d) {
      const int head = k / dh, j = k - head * dh;
      if (q == 0 || (accel && P.sidx[head] >= 0)) {
        const float* pp = P.apart + ((size_t)(head * NS) * 2 + q) * (dh + 4);
        float M = -INFINITY;
        for (int s = 0; s < NS; ++s) {
          const float* ps = pp + (size_t)s * 2 * (dh + 4);
          if (ldcg(ps + dh + 1) > 0.f) M = fmaxf(M, ldcg(ps + dh));
        }
        float Lsum = 0.f;
        for (int s = 0; s < NS; ++s) {
          const float* ps = pp + (size_t)s * 2 * (dh + 4);
          const float ls = ldcg(ps + dh + 1);
          if (ls > 0.f) {
            const float wgt = __expf(ldcg(ps + dh) - M);
            const float4 v = ldcg4(ps + j);
            Lsum += ls * wgt;
            o.x += v.x * wgt; o.y += v.y * wgt; o.z += v.z * wgt; o.w += v.w * wgt;
          }
        }
        const float inv = 1.f / Lsum;
        o.x *= inv; o.y *= inv; o.z *= inv; o.w *= inv;
      }
    }
    if (q == 0) xstore4(c0, c1, k, o); else xstore4(c2, c3, k, o);
  }
  bar_consumers();
}

// x <- SwiGLU activations of both streams (a7 input)
__device__ __forceinline__ void loader_act(const FParams& P, bf16* x, bool accel) {
  const int tid = threadIdx.x;
  bar_consumers();
  bf16 *c0 = x, *c1 = x + XCOL, *c2 = x + 2 * XCOL, *c3 = x + 3 * XCOL;
  for (int idx = tid; idx < (P.F_pad >> 2); idx += NCT) {
    const int k = idx * 4;
    float4 a = make_float4(0.f, 0.f, 0.f, 0.f), b = a;
    if (k < P.F) {
      a = ldcg4(P.act + k);
      if (accel) b = ldcg4(P.act + P.F_pad + k);
    }
    xstore4(c0, c1, k, a);
    xstore4(c2, c3, k, b);
  }
  bar_consumers();
}

// Adapter down-projection u = A x^ of the accelerated row, distributed: CTA c computes
// row j = c / q over k-chunk c % q and publishes it; fetch_u() sums the q chunks of every row in order.
struct UState {
  unsigned int target;   // publications expected so far in this launch
  int buf;               // upart buffer of the current phase
  int nj, q;             // geometry of the current phase
  bool ready;            // warp 0: smem u holds the current phase's u
};
__device__ __forceinline__ void publish_u(const FParams& P, const bf16* x, UState& us, const bf16* A, int nj, int Kc,
                                          const int* cols, int G) {
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int q = min(min(G / nj, UPART_Q), 256 / nj);
  us.buf ^= 1;
  us.nj = nj;
  us.q = q;
  us.target += (unsigned int)(nj * q);
  us.ready = false;
  const int c = blockIdx.x;
  if (warp == 1 && c < nj * q) {
    const int j = c / q, ch = c - j * q;
    const int chunk = (((Kc + q - 1) / q) + 7) & ~7;
    const int k0 = ch * chunk, k1 = min(Kc, k0 + chunk);
    const bf16* a = A + (size_t)j * Kc;
    const bf16 *xh = x + 2 * XCOL, *xl = x + 3 * XCOL;
    float acc = 0.f;
    for (int k = k0 + lane * 8; k < k1; k += 256) {   // chunk and Kc are multiples of 8
      const uint4 w = __ldg((const uint4*)(a + k));
      float f[8];
      bf16x2_to_f32(w.x, f[0], f[1]); bf16x2_to_f32(w.y, f[2], f[3]);
      bf16x2_to_f32(w.z, f[4], f[5]); bf16x2_to_f32(w.w, f[6], f[7]);
#pragma unroll
      for (int e = 0; e < 8; ++e) acc += f[e] * xval(xh, xl, cols ? cols[k + e] : k + e);
    }
    acc = warp_sum(acc);
    if (lane == 0) {
      __stcg(P.upart + ((size_t)us.buf * MAX_NJ + j) * UPART_Q + ch, acc);
      __threadfence();
      atomicAdd(&P.ctl->ucnt, 1u);
    }
  }
}
// warp 0 only
__device__ __forceinline__ void fetch_u(const FParams& P, float* u, float* utmp, UState& us) {
  const int lane = threadIdx.x & 31;
  if (lane == 0) {
    long long t0 = clock64();
    unsigned int n = 0;
    while ((int)(ld_acquire(&P.ctl->ucnt) - us.target) < 0) {
      if ((++n & 255u) == 0u) {
        if (aborted(P.ctl)) break;
        if (clock64() - t0 > SPIN_LIMIT) { set_abort(P.ctl, 0x500u); break; }
      }
    }
    __threadfence();
  }
  __syncwarp();
  const int total = us.nj * us.q;   // <= 256
  float v[8];
#pragma unroll
  for (int i = 0; i < 8; ++i) {
    const int idx = lane + 32 * i;
    v[i] = 0.f;
    if (idx < total) v[i] = ldcg(P.upart + ((size_t)us.buf * MAX_NJ + idx / us.q) * UPART_Q + idx % us.q);
  }
#pragma unroll
  for (int i = 0; i < 8; ++i) {
    const int idx = lane + 32 * i;
    if (idx < total) utmp[idx] = v[i];
  }
  __syncwarp();
  for (int j = lane; j < us.nj; j += 32) {
    float s = 0.f;
    for (int ch = 0; ch < us.q; ++ch) s += utmp[j * us.q + ch];
    u[j] = s;
  }
  __syncwarp();
  us.ready = true;
}

__device__ __forceinline__ float lora_dot(const bf16* Brow, const float* u, int r) {
  float s = 0.f;
  if ((r & 7) == 0) {
    for (int q = 0; q < r; q += 8) {
      const uint4 w = __ldg((const uint4*)(Brow + q));
      float f[8];
      bf16x2_to_f32(w.x, f[0], f[1]); bf16x2_to_f32(w.y, f[2], f[3]);
      bf16x2_to_f32(w.z, f[4], f[5]); bf16x2_to_f32(w.w, f[6], f[7]);
#pragma unroll
      for (int e = 0; e < 8; ++e) s += f[e] * u[q + e];
    }
  } else {
    for (int q = 0; q < r; ++q) s += bf(Brow + q) * u[q];
  }
  return s;
}

// ------------------------------------------------------------------ phase epilogues (warp 0; one 16-row tile, sums in T[row][stream])
struct PhaseCtx {
  int ph, layer;
  const FLayer* L;
  int pos;          // position of the token of this pass
  bool accel;       // stream 1 live
};

__device__ __forceinline__ void epilogue_tile(const FParams& P, const float* T, const float* u, const PhaseCtx& c, int rt, int slot) {
  const int lane = threadIdx.x & 31;
  const int d = P.d, dh = P.dh, half = dh >> 1, r = P.r;
  if (c.ph == PH_QKV) {
    // a3 fused: RoPE (pairs are adjacent packed rows) + KV append (slow) / k^,v^ kept in scratch (accel)
    if (lane < 16) {
      const int m = lane >> 1, s = lane & 1;
      const int r0 = rt * 16 + 2 * m;
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
            v0 += lora_dot(B + (size_t)e0 * r, u + which * r, r);
            v1 += lora_dot(B + (size_t)e1 * r, u + which * r, r);
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
            __stcg(P.qbuf + s * d + o0, v0); __stcg(P.qbuf + s * d + o1, v1);
          } else if (s == 0) {
            bf16* C = (which == 1 ? c.L->Kc : c.L->Vc) + ((size_t)head * P.max_seq + c.pos) * dh;
            C[e0] = __float2bfloat16_rn(v0);
            C[e1] = __float2bfloat16_rn(v1);
          } else {
            float* C = which == 1 ? P.khat : P.vhat;
            __stcg(C + o0, v0); __stcg(C + o1, v1);
          }
        }
      }
    }
  } else if (c.ph == PH_OPROJ || c.ph == PH_DOWN) {
    // split-K partial of a row-tile -> slot; the contributor of slot 0 adds the adapter term once
    const int row = lane >> 1, s = lane & 1, n = rt * 16 + row;
    if (n < d && (s == 0 || c.accel)) {
      float v = T[lane];
      if (s == 1 && slot == 0) v += lora_dot((c.ph == PH_OPROJ ? c.L->Bo : c.L->Bd) + (size_t)n * r, u, r);
      float* S = c.ph == PH_OPROJ ? P.oslots : P.dslots;
      __stcg(S + (size_t)(slot * 2 + s) * d + n, v);
    }
  } else if (c.ph == PH_GATEUP) {
    // packed tile: gate rows n..n+7 then up rows n..n+7
    if (lane < 16) {
      const int nl = lane >> 1, s = lane & 1, n = rt * 8 + nl;
      if (n < P.F && (s == 0 || c.accel)) {
        float g = T[nl * 2 + s], up = T[(8 + nl) * 2 + s];
        if (s == 1) {
          g += lora_dot(c.L->Bg + (size_t)n * r, u, r);
          up += lora_dot(c.L->Bu + (size_t)n * r, u + r, r);
        }
        __stcg(P.act + s * P.F_pad + n, silu(g) * up);
      }
    }
  } else {
    // PH_HEAD (final head on h_N, or draft head on p) / PH_EXIT (exit head on p at a gate); the loader
    // put the head's input into both columns
    const bool on_p = (c.ph == PH_EXIT) || P.head_stream == 1;
    const int gate = c.ph == PH_HEAD ? P.head_gate : c.layer;   // for PH_EXIT `layer` carries the gate index
    const bool is_final = (c.ph == PH_HEAD && P.head_stream == 0);
    u64 key = 0ull;
    const int n = rt * 16 + lane;
    if (lane < 16 && n < P.V) {
      float v = T[lane * 2];
      if (on_p && P.lmB) v += lora_dot(P.lmB + (size_t)n * r, u, r);
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
    if (lane == 0 && key) atomicMax(&P.ctl->amax[c.ph == PH_HEAD ? 0 : 1 + gate], key);
  }
}

// ------------------------------------------------------------------ attention phase (a4): split-K flash-decode, dual query
// Work item = (head, split), one per CTA.  Keys/values of positions [p0, p1) < pos come from the cache
// (prefetched into L2 by the producer); both queries share every load.  The last split also takes the
// token's own key/value: slow = K[pos], V[pos] as stored (rounded), accelerated = k^, v^ from scratch
// (p_t attends h_<t (+) p_t).  Partials (m, l, o) go to P.apart; the O-proj loader merges.
__device__ __forceinline__ void attn_phase(const FParams& P, float* red, const FLayer* L, int pos, bool accel, int G) {
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int dh = P.dh, d = P.d, lpp = dh >> 3, NS = P.ns;
  const int seg = lane >> 4, sl = lane & 15;
  const bool active = sl < lpp;
  const int items = P.n_heads * NS;   // red: [2 NCW segments][2 queries][dh + 2]
  for (int w = blockIdx.x; w < items; w += G) {
    const int head = w / NS, sp = w - head * NS;
    const bool q1 = accel && P.sidx[head] >= 0;
    const int chunk = (pos + NS - 1) / NS;
    const int p0 = min(pos, sp * chunk), p1 = min(pos, p0 + chunk);
    float qa[8], qb[8];
#pragma unroll
    for (int e = 0; e < 8; ++e) { qa[e] = 0.f; qb[e] = 0.f; }
    if (active) {
      const float4 a0 = ldcg4(P.qbuf + head * dh + sl * 8), a1 = ldcg4(P.qbuf + head * dh + sl * 8 + 4);
      qa[0] = a0.x * P.scale; qa[1] = a0.y * P.scale; qa[2] = a0.z * P.scale; qa[3] = a0.w * P.scale;
      qa[4] = a1.x * P.scale; qa[5] = a1.y * P.scale; qa[6] = a1.z * P.scale; qa[7] = a1.w * P.scale;
      if (q1) {
        const float4 b0 = ldcg4(P.qbuf + d + head * dh + sl * 8), b1 = ldcg4(P.qbuf + d + head * dh + sl * 8 + 4);
        qb[0] = b0.x * P.scale; qb[1] = b0.y * P.scale; qb[2] = b0.z * P.scale; qb[3] = b0.w * P.scale;
        qb[4] = b1.x * P.scale; qb[5] = b1.y * P.scale; qb[6] = b1.z * P.scale; qb[7] = b1.w * P.scale;
      }
    }
    float m0 = -INFINITY, l0 = 0.f, m1 = -INFINITY, l1 = 0.f, o0[8], o1[8];
#pragma unroll
    for (int e = 0; e < 8; ++e) { o0[e] = 0.f; o1[e] = 0.f; }
    const bf16* Kb = L->Kc + (size_t)head * P.max_seq * dh + sl * 8;
    const bf16* Vb = L->Vc + (size_t)head * P.max_seq * dh + sl * 8;
    // positions of this warp: p0 + 2*warp + seg + 2*NCW*i; AIF iterations in flight
    constexpr int AIF = 4;
    for (int ub = p0 + warp * 2; ub < p1; ub += AIF * NCW * 2) {
      uint4 kk[AIF], vv[AIF];
      bool valid[AIF];
#pragma unroll
      for (int it = 0; it < AIF; ++it) {
        const int u = ub + it * NCW * 2 + seg;
        valid[it] = u < p1;
        kk[it] = make_uint4(0u, 0u, 0u, 0u);
        vv[it] = kk[it];
        if (valid[it] && active) {
          kk[it] = ldcg16(Kb + (size_t)u * dh);
          vv[it] = ldcg16(Vb + (size_t)u * dh);
        }
      }
#pragma unroll
      for (int it = 0; it < AIF; ++it) {
        float kf[8], vf[8];
        bf16x2_to_f32(kk[it].x, kf[0], kf[1]); bf16x2_to_f32(kk[it].y, kf[2], kf[3]);
        bf16x2_to_f32(kk[it].z, kf[4], kf[5]); bf16x2_to_f32(kk[it].w, kf[6], kf[7]);
        bf16x2_to_f32(vv[it].x, vf[0], vf[1]); bf16x2_to_f32(vv[it].y, vf[2], vf[3]);
        bf16x2_to_f32(vv[it].z, vf[4], vf[5]); bf16x2_to_f32(vv[it].w, vf[6], vf[7]);
        float sa = 0.f, sb = 0.f;
#pragma unroll
        for (int e = 0; e < 8; ++e) { sa += qa[e] * kf[e]; sb += qb[e] * kf[e]; }
#pragma unroll
        for (int o = 8; o > 0; o >>= 1) {
          sa += __shfl_xor_sync(0xffffffffu, sa, o);
          sb += __shfl_xor_sync(0xffffffffu, sb, o);
        }
        if (valid[it]) {
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
    }
    // ---- the token's own key/value (last split, warp 0, segment 0)
    if (sp == NS - 1 && warp == 0) {
      float kf[8], vf[8], k2[8], v2[8];
#pragma unroll
      for (int e = 0; e < 8; ++e) { kf[e] = vf[e] = k2[e] = v2[e] = 0.f; }
      if (seg == 0 && active) {
        const uint4 kk = ldcg16(Kb + (size_t)pos * dh), vv = ldcg16(Vb + (size_t)pos * dh);
        bf16x2_to_f32(kk.x, kf[0], kf[1]); bf16x2_to_f32(kk.y, kf[2], kf[3]);
        bf16x2_to_f32(kk.z, kf[4], kf[5]); bf16x2_to_f32(kk.w, kf[6], kf[7]);
        bf16x2_to_f32(vv.x, vf[0], vf[1]); bf16x2_to_f32(vv.y, vf[2], vf[3]);
        bf16x2_to_f32(vv.z, vf[4], vf[5]); bf16x2_to_f32(vv.w, vf[6], vf[7]);
        if (q1) {
          const float4 ka = ldcg4(P.khat + head * dh + sl * 8), kb = ldcg4(P.khat + head * dh + sl * 8 + 4);
          const float4 va = ldcg4(P.vhat + head * dh + sl * 8), vb = ldcg4(P.vhat + head * dh + sl * 8 + 4);
          k2[0] = ka.x; k2[1] = ka.y; k2[2] = ka.z; k2[3] = ka.w; k2[4] = kb.x; k2[5] = kb.y; k2[6] = kb.z; k2[7] = kb.w;
          v2[0] = va.x; v2[1] = va.y; v2[2] = va.z; v2[3] = va.w; v2[4] = vb.x; v2[5] = vb.y; v2[6] = vb.z; v2[7] = vb.w;
        }
      }
      float sa = 0.f, sb = 0.f;
#pragma unroll
      for (int e = 0; e < 8; ++e) { sa += qa[e] * kf[e]; sb += qb[e] * k2[e]; }
#pragma unroll
      for (int o = 8; o > 0; o >>= 1) {
        sa += __shfl_xor_sync(0xffffffffu, sa, o);
        sb += __shfl_xor_sync(0xffffffffu, sb, o);
      }
      if (seg == 0) {
        float mn = fmaxf(m0, sa), corr = __expf(m0 - mn), p = __expf(sa - mn);
        l0 = l0 * corr + p;
#pragma unroll
        for (int e = 0; e < 8; ++e) o0[e] = o0[e] * corr + p * vf[e];
        m0 = mn;
        if (q1) {
          mn = fmaxf(m1, sb); corr = __expf(m1 - mn); p = __expf(sb - mn);
          l1 = l1 * corr + p;
#pragma unroll
          for (int e = 0; e < 8; ++e) o1[e] = o1[e] * corr + p * v2[e];
          m1 = mn;
        }
      }
    }
    // ---- merge the lane segments of the CTA -> one partial per query
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
      for (int s = 0; s < 2 * NCW; ++s) {
        const float* src = red + ((size_t)s * 2 + q) * (dh + 2);
        if (src[dh + 1] > 0.f) M = fmaxf(M, src[dh]);
      }
      float Lsum = 0.f, O = 0.f;
      for (int s = 0; s < 2 * NCW; ++s) {
        const float* src = red + ((size_t)s * 2 + q) * (dh + 2);
        float ls = src[dh + 1];
        if (ls > 0.f) {
          float wgt = __expf(src[dh] - M);
          Lsum += ls * wgt;
          O += src[j] * wgt;
        }
      }
      float* pp = P.apart + ((size_t)(head * NS + sp) * 2 + q) * (dh + 4);
      __stcg(pp + j, O);
      if (j == 0) { __stcg(pp + dh, M); __stcg(pp + dh + 1, Lsum); }
    }
    bar_consumers();
  }
}

// ------------------------------------------------------------------ producer: the CTA's weight-stage stream of the whole pass
__device__ __forceinline__ bool exit_phase_after(const FParams& P, int layer) {
  const FLayer* L = P.layers + layer;
  return L->gate && L->accel && P.exit_heads && !(P.head_stream == 1 && layer + 1 == P.n_layers_run);
}

// Walks the CTA's stages of the pass in consumption order (must mirror the consumer loop).
struct Cursor {
  int layer, ph;     // ph = -1 before the first phase
  int s, s1;
  const unsigned char* W;
  bool new_layer;    // set when the walk enters a layer's QKV phase
};
__device__ __noinline__ bool cursor_advance(const FParams& P, Cursor& c, int G) {
  const int n = P.n_layers_run;
  if (c.ph == PH_HEAD) return false;
  bool next_layer = false;
  if (c.ph < 0) { c.layer = -1; next_layer = true; }
  else if (c.ph == PH_QKV) c.ph = PH_OPROJ;
  else if (c.ph == PH_OPROJ) c.ph = PH_GATEUP;
  else if (c.ph == PH_GATEUP) c.ph = PH_DOWN;
  else if (c.ph == PH_DOWN) { if (exit_phase_after(P, c.layer)) c.ph = PH_EXIT; else next_layer = true; }
  else next_layer = true;   // PH_EXIT
  if (next_layer) {
    ++c.layer;
    c.ph = c.layer < n ? PH_QKV : PH_HEAD;
    c.new_layer = c.ph == PH_QKV;
  }
  const int nks_d = P.d_pad / STAGE_K, nks_f = P.F_pad / STAGE_K;
  int n_rt, nks, gran, rot_layer = c.layer;
  const FLayer* L = P.layers + (c.layer < n ? c.layer : 0);
  switch (c.ph) {
    case PH_QKV:    c.W = (const unsigned char*)L->Wqkv; n_rt = P.rt_qkv; nks = nks_d; gran = nks; break;
    case PH_OPROJ:  c.W = (const unsigned char*)L->Wo;   n_rt = P.rt_o;   nks = nks_d; gran = 1;   break;
    case PH_GATEUP: c.W = (const unsigned char*)L->Wgu;  n_rt = P.rt_gu;  nks = nks_d; gran = nks; break;
    case PH_DOWN:   c.W = (const unsigned char*)L->Wd;   n_rt = P.rt_d;   nks = nks_f; gran = 1;   break;
    case PH_EXIT:   c.W = (const unsigned char*)P.Wlm;   n_rt = P.rt_v;   nks = nks_d; gran = nks; rot_layer = L->gate - 1; break;
    default:        c.W = (const unsigned char*)P.Wlm;   n_rt = P.rt_v;   nks = nks_d; gran = nks; rot_layer = n; break;
  }
  const int U = n_rt * nks / gran;
  const int v = ((int)blockIdx.x + phase_rot(rot_layer, c.ph, G)) % G;
  c.s = range_lo(U, v, G) * gran;
  c.s1 = range_lo(U, v + 1, G) * gran;
  return true;
}
__device__ __forceinline__ bool cursor_get(const FParams& P, Cursor& c, int G, const unsigned char*& addr) {
  while (c.s >= c.s1) {
    if (!cursor_advance(P, c, G)) return false;
  }
  addr = c.W + (size_t)c.s * STAGE_BYTES;
  ++c.s;
  return true;
}

// L2 prefetch of the K/V positions this CTA will attend to in `layer`
__device__ __noinline__ void prefetch_kv(const FParams& P, int layer, int G) {
  const int NS = P.ns, pos = P.pos_host, dh = P.dh;
  const FLayer* L = P.layers + layer;
  for (int w = blockIdx.x; w < P.n_heads * NS; w += G) {
    const int head = w / NS, sp = w - head * NS;
    const int chunk = (pos + NS - 1) / NS;
    const int p0 = min(pos, sp * chunk), p1 = min(pos, p0 + chunk);
    size_t bytes = (size_t)(p1 - p0) * dh * 2;
    const unsigned char* kp = (const unsigned char*)(L->Kc + ((size_t)head * P.max_seq + p0) * dh);
    const unsigned char* vp = (const unsigned char*)(L->Vc + ((size_t)head * P.max_seq + p0) * dh);
    for (size_t o = 0; o < bytes; o += 16384) {
      const uint32_t n = (uint32_t)min((size_t)16384, bytes - o);
      bulk_prefetch_l2(kp + o, n);
      bulk_prefetch_l2(vp + o, n);
    }
  }
}

// L2 prefetch of what the consumers will read with plain loads on their critical path: the layer's
// norm gains and adapter tensors (each CTA one slice: together the whole range), the RoPE row.
__device__ __forceinline__ void prefetch_slice(const void* base, size_t bytes, int G) {
  const size_t per = (((bytes + G - 1) / G) + 15) & ~(size_t)15;
  const size_t o = (size_t)blockIdx.x * per;
  if (o < bytes) bulk_prefetch_l2((const unsigned char*)base + o, (uint32_t)min(per, ((bytes - o) + 15) & ~(size_t)15));
}
__device__ __noinline__ void prefetch_params(const FParams& P, int layer, int G) {
  const FLayer* L = P.layers + layer;
  if ((int)blockIdx.x == layer % G) {
    bulk_prefetch_l2(L->g1, (uint32_t)((P.d * 2 + 15) & ~15));
    bulk_prefetch_l2(L->g2, (uint32_t)((P.d * 2 + 15) & ~15));
    if (layer == 0) {
      bulk_prefetch_l2(P.rope_tab + (size_t)P.pos_host * (P.dh >> 1), (uint32_t)(((P.dh >> 1) * 8 + 15) & ~15));
      bulk_prefetch_l2(P.gf, (uint32_t)((P.d * 2 + 15) & ~15));
    }
  }
  if (L->accel && L->ad_bytes) prefetch_slice(L->ad_lo, L->ad_bytes, G);
  if (layer == 0 && P.lmA && (P.head_stream == 1 || P.exit_heads)) {
    prefetch_slice(P.lmA, (size_t)P.r * P.d * 2, G);
    prefetch_slice(P.lmB, (size_t)P.V * P.r * 2, G);
  }
}

constexpr int PH_ATTN = N_PH;   // consumer-only phase (no weights)

__global__ void __launch_bounds__(NTHREADS, 1) m2r2_fused_decode_kernel(const __grid_constant__ FParams P) {
  extern __shared__ __align__(1024) unsigned char smem_raw[];
  unsigned char* const ring = smem_raw;
  bf16* const x = (bf16*)(smem_raw + OFF_X);
  float* const red = (float*)(smem_raw + OFF_RED);
  float* const tile_out = (float*)(smem_raw + OFF_TILE);
  float* const u_s = (float*)(smem_raw + OFF_U);
  float* const sred = (float*)(smem_raw + OFF_SRED);
  u64* const full = (u64*)(smem_raw + OFF_BAR);
  u64* const empty = full + NSTAGE;
  float* const utmp = (float*)(smem_raw + OFF_UTMP);
  const int tid = threadIdx.x, G = gridDim.x;
  if (tid == 0) {
    for (int i = 0; i < NSTAGE; ++i) { mbar_init(&full[i], 1); mbar_init(&empty[i], NCW); }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();
  const int nks_d = P.d_pad / STAGE_K, nks_f = P.F_pad / STAGE_K;
  const int n_run = P.n_layers_run;

  if (tid >= NCT) {
    // ================= producer warp: one thread streams every weight stage of the pass
    if (tid == NCT) {
      const u64 pol = policy_evict_first();
      Cursor ld, pf;
      ld.layer = 0; ld.ph = -1; ld.s = ld.s1 = 0; ld.W = nullptr; ld.new_layer = false;
      pf = ld;
      bool pf_live = P.pf_ahead > 0;
      const unsigned char* a;
      for (int i = 0; i < P.pf_ahead && pf_live; ++i) {
        pf_live = cursor_get(P, pf, G, a);
        if (pf_live) bulk_prefetch_l2(a, STAGE_BYTES);
        if (pf.new_layer) { pf.new_layer = false; prefetch_kv(P, pf.layer, G); prefetch_params(P, pf.layer, G); }
      }
      unsigned int ctr = 0;
      while (cursor_get(P, ld, G, a)) {
        if (pf_live) {
          const unsigned char* b;
          pf_live = cursor_get(P, pf, G, b);
          if (pf_live) bulk_prefetch_l2(b, STAGE_BYTES);
          if (pf.new_layer) { pf.new_layer = false; prefetch_kv(P, pf.layer, G); prefetch_params(P, pf.layer, G); }
        } else if (P.pf_ahead <= 0 && ld.new_layer) {
          ld.new_layer = false;
          prefetch_kv(P, ld.layer, G);
          prefetch_params(P, ld.layer, G);
        }
        const unsigned int slot = ctr % NSTAGE, use = ctr / NSTAGE;
        ++ctr;
        mbar_wait(&empty[slot], (use & 1u) ^ 1u, P.ctl, 0x400u + ld.ph);
        mbar_expect_tx(&full[slot], STAGE_BYTES);
        bulk_g2s(ring + (size_t)slot * STAGE_BYTES, a, STAGE_BYTES, &full[slot], pol);
      }
    }
    return;
  }

  // ================= consumers: one loop over the phases of the pass (every routine has one call site)
  const int lane = tid & 31, warp = tid >> 5, g = lane >> 2, t = lane & 3;
  unsigned int nbar = 0, stage_ctr = 0, flushes = 0;
  int tl_n = 0;
  (void)tl_n;
  UState us;
  us.target = 0; us.buf = 0; us.nj = 0; us.q = 1; us.ready = false;
  const int d = P.d;
  const int pos = *(volatile int*)P.kv_len + P.joff;
  const int tok = *(volatile const int*)P.tok_in;
  TL(1);

  int layer = 0, ph = n_run > 0 ? PH_QKV : PH_HEAD;
  for (;;) {
    const FLayer* L = P.layers + (layer < n_run ? layer : (n_run > 0 ? n_run - 1 : 0));
    const bool accel = ph == PH_HEAD || ph == PH_EXIT ? true : L->accel != 0;
    if (ph == PH_ATTN) {
      // ---- a4: attention
      attn_phase(P, (float*)x, L, pos, accel, G);
      TL(13);
      grid_sync(P.ctl, P.bar_base, nbar, G);
      TL(14);
      ph = PH_OPROJ;
      continue;
    }
    // ---- geometry of the phase
    PhaseCtx pc;
    pc.ph = ph; pc.layer = layer; pc.L = L; pc.pos = pos; pc.accel = accel;
    int n_rt, nks = nks_d, nj = 0, Kc = d;
    bool split = false, need_u = accel && P.r > 0;
    const bf16* A = nullptr;
    const int* cols = nullptr;
    if (ph == PH_QKV) { n_rt = P.rt_qkv; A = L->Aqkv; nj = 3 * P.r; }
    else if (ph == PH_OPROJ) { n_rt = P.rt_o; split = true; A = L->Ao; nj = P.r; Kc = P.da; cols = P.accel_cols; }
    else if (ph == PH_GATEUP) { n_rt = P.rt_gu; A = L->Agu; nj = 2 * P.r; }
    else if (ph == PH_DOWN) { n_rt = P.rt_d; nks = nks_f; split = true; A = L->Ad; nj = P.r; Kc = P.F; }
    else {
      n_rt = P.rt_v; A = P.lmA; nj = P.r;
      need_u = P.lmA != nullptr && (ph == PH_EXIT || P.head_stream == 1);
      pc.layer = ph == PH_EXIT ? L->gate - 1 : n_run;
    }
    // ---- loader: the phase's input vector(s) -> shared memory
    if (ph == PH_OPROJ) {
      loader_attn(P, x, accel);
    } else if (ph == PH_DOWN) {
      loader_act(P, x, accel);
    } else {
      LoadSrc src;
      int mode;
      float *wb = nullptr, *tr = nullptr;
      const bf16* gn;
      src.emb = nullptr; src.gate = 0;
      if (ph == PH_GATEUP) {
        // a5-tail: h' = h + O-proj sums
        src.base = P.RB; src.slots = P.oslots; src.n_rt = P.rt_o; src.nks = nks_d; src.p_live = accel;
        mode = LN_GU; wb = P.RA; gn = L->g2;
      } else if ((ph == PH_QKV && layer == 0) || (ph == PH_HEAD && n_run == 0)) {
        // a1: embedding, p_0 <- h_0 (L82)
        src.base = nullptr; src.emb = P.embed + (size_t)tok * d; src.slots = nullptr; src.n_rt = 0; src.nks = 1; src.p_live = false;
        mode = ph == PH_QKV ? LN_QKV : (P.head_stream == 0 ? LN_HEAD_H : LN_HEAD_P);
        wb = ph == PH_QKV ? P.RB : nullptr;
        gn = ph == PH_QKV ? L->g1 : P.gf;
        tr = P.do_trace ? P.trace : nullptr;
      } else {
        // a7-tail: residual + down sums of the layer below (accelerated-residual update, Eq. 2), gate
        const FLayer* Lp = ph == PH_QKV ? L - 1 : L;
        src.base = P.RA; src.slots = P.dslots; src.n_rt = P.rt_d; src.nks = nks_f; src.p_live = Lp->accel != 0;
        if (ph == PH_QKV) {
          src.gate = Lp->accel ? Lp->gate : 0;
          mode = LN_QKV; wb = P.RB; gn = L->g1;
          tr = P.do_trace ? P.trace + (size_t)layer * 2 * d : nullptr;
        } else if (ph == PH_EXIT) {
          mode = LN_HEAD_P; gn = P.gf;
        } else {
          mode = P.head_stream == 0 ? LN_HEAD_H : LN_HEAD_P; gn = P.gf;
          tr = P.do_trace ? P.trace + (size_t)n_run * 2 * d : nullptr;
        }
      }
      loader_norm(P, x, sred, mode, src, wb, tr, gn, G);
    }
    if (need_u) publish_u(P, x, us, A, nj, Kc, cols, G);
    TL(10 + ph);
    // ---- GEMV over this CTA's stages.  Stage (rt, ks): 64 tiles of row-tile rt, inputs [1024 ks, +1024).
    // Warp w multiplies tiles 8w..8w+7: 8 LDS.128 (A fragments) + 4 LDS.128 (B fragments) + 8 HMMA.
    {
      const int S = n_rt * nks, gran = split ? 1 : nks, U = S / gran;
      const int v = ((int)blockIdx.x + phase_rot(pc.layer, ph, G)) % G;
      const int s0 = range_lo(U, v, G) * gran, s1 = range_lo(U, v + 1, G) * gran;
      float ca[4] = {0.f, 0.f, 0.f, 0.f}, cb[4] = {0.f, 0.f, 0.f, 0.f};
      const bf16* xcol = x + (size_t)(g & 3) * XCOL + t * 16 + warp * 128;
      int rt = s0 / nks, ks = s0 - rt * nks;
      for (int s = s0; s < s1; ++s) {
        const unsigned int slot = stage_ctr % NSTAGE, use = stage_ctr / NSTAGE;
        ++stage_ctr;
        uint4 b0 = make_uint4(0u, 0u, 0u, 0u), b1 = b0, b2 = b0, b3 = b0;
        if (g < 4) {
          const uint4* xb = (const uint4*)(xcol + (size_t)ks * STAGE_K);
          b0 = xb[0]; b1 = xb[1]; b2 = xb[8]; b3 = xb[9];
        }
        mbar_wait(&full[slot], use & 1u, P.ctl, 0x200u + ph);
        const uint4* st = (const uint4*)(ring + (size_t)slot * STAGE_BYTES) + (warp * TPW) * 32 + lane;
        const uint4 a0 = st[0], a1 = st[32], a2 = st[64], a3 = st[96];
        const uint4 a4 = st[128], a5 = st[160], a6 = st[192], a7 = st[224];
        mma_bf16(ca, a0, b0.x, b0.y);
        mma_bf16(cb, a1, b0.z, b0.w);
        mma_bf16(ca, a2, b1.x, b1.y);
        mma_bf16(cb, a3, b1.z, b1.w);
        mma_bf16(ca, a4, b2.x, b2.y);
        mma_bf16(cb, a5, b2.z, b2.w);
        mma_bf16(ca, a6, b3.x, b3.y);
        mma_bf16(cb, a7, b3.z, b3.w);
        __syncwarp();
        if (lane == 0) mbar_arrive(&empty[slot]);   // stage consumed by this warp
        if (ks == nks - 1 || s == s1 - 1) {
          // ---- end of this CTA's segment of row-tile rt: columns 0,1 = h (hi, lo parts), 2,3 = p
          float* rw = red + (size_t)(flushes & 1u) * NCW * 32 + warp * 32;
          if (t < 2) {
            rw[g * 2 + t] = (ca[0] + ca[1]) + (cb[0] + cb[1]);
            rw[(g + 8) * 2 + t] = (ca[2] + ca[3]) + (cb[2] + cb[3]);
          }
#pragma unroll
          for (int i = 0; i < 4; ++i) ca[i] = cb[i] = 0.f;
          bar_consumers();
          if (warp == 0) {
            const float* rb = red + (size_t)(flushes & 1u) * NCW * 32 + lane;
            float sum = 0.f;
#pragma unroll
            for (int w = 0; w < NCW; ++w) sum += rb[w * 32];
            tile_out[lane] = sum;
            __syncwarp();
            if (need_u && !us.ready) fetch_u(P, u_s, utmp, us);
            int sl = 0;
            if (split) sl = S >= G ? v - unit_owner(S, rt * nks, G) : ks;
            epilogue_tile(P, tile_out, u_s, pc, rt, sl);
            __syncwarp();
          }
          ++flushes;
          TL(40);
        }
        if (++ks == nks) { ks = 0; ++rt; }
      }
    }
    TL(20 + ph);
    if (ph == PH_HEAD) {
      grid_sync(P.ctl, P.bar_base, nbar, G);
      break;
    }
    if (ph != PH_EXIT) grid_sync(P.ctl, P.bar_base, nbar, G);   // nothing after an exit head depends on it
    TL(30 + ph);
    // ---- next phase
    if (ph == PH_QKV) ph = PH_ATTN;
    else if (ph == PH_OPROJ) ph = PH_GATEUP;
    else if (ph == PH_GATEUP) ph = PH_DOWN;
    else if (ph == PH_DOWN && exit_phase_after(P, layer)) ph = PH_EXIT;
    else { ++layer; ph = layer < n_run ? PH_QKV : PH_HEAD; }
  }
  TL(50);
  if (blockIdx.x == 0 && tid == 0) {
    u64 key = *(volatile u64*)&P.ctl->amax[0];
    int tk = (int)(0xFFFFFFFFu - (unsigned int)(key & 0xFFFFFFFFull));
    *P.tok_out = tk;
    P.ctl->amax[0] = 0ull;
    for (int j = 0; j < P.n_gates; ++j) {
      u64 kj = *(volatile u64*)&P.ctl->amax[1 + j];
      if (kj) P.exit_tok[j] = (int)(0xFFFFFFFFu - (unsigned int)(kj & 0xFFFFFFFFull));
      P.ctl->amax[1 + j] = 0ull;
    }
    P.ctl->ucnt = 0u;
    if (P.advance) { *P.kv_len = pos + 1; *P.pending = tk; }
  }
}

// ------------------------------------------------------------------ repack: row-major [n_out, K] -> fragment-major stages
// map 0: natural rows; 1: QKV (RoPE pairs (j, j+dh/2) of q and k made adjacent); 2: gate/up interleaved
// (16-row tile = gate n..n+7, up n..n+7).  Rows / columns beyond the matrix are zero.
__device__ __forceinline__ const bf16* pack_src_row(const bf16* src, const bf16* src2, int map, int r, int n_out, int K, int d, int dh) {
  if (map == 0) return r < n_out ? src + (size_t)r * K : nullptr;
  if (map == 1) {
    if (r >= n_out) return nullptr;
    int which = r / d, w = r % d, sr = r;
    if (which < 2) {
      int head = w / dh, e = w % dh;
      sr = which * d + head * dh + (e >> 1) + (e & 1) * (dh >> 1);
    }
    return src + (size_t)sr * K;
  }
  const int n = (r >> 4) * 8 + (r & 7);
  if (n >= n_out) return nullptr;
  return ((r & 15) < 8 ? src : src2) + (size_t)n * K;
}
__global__ void pack_kernel(uint4* __restrict__ dst, const bf16* __restrict__ src, const bf16* __restrict__ src2,
                            int map, int n_out, int K, int n_rt, int nks, int d, int dh) {
  const size_t total = (size_t)n_rt * nks * (STAGE_BYTES / 16);
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < total; i += (size_t)gridDim.x * blockDim.x) {
    const size_t stage = i / (STAGE_BYTES / 16);
    const int within = (int)(i % (STAGE_BYTES / 16));
    const int tile = within >> 5, lane = within & 31, g = lane >> 2, t = lane & 3;
    const int rt = (int)(stage / nks), ks = (int)(stage % nks);
    const int k = ks * STAGE_K + tile * 16 + 2 * t;
    const bf16* r0 = pack_src_row(src, src2, map, rt * 16 + g, n_out, K, d, dh);
    const bf16* r1 = pack_src_row(src, src2, map, rt * 16 + g + 8, n_out, K, d, dh);
    uint4 v = make_uint4(0u, 0u, 0u, 0u);   // K % 8 == 0: a pair never straddles the end
    if (r0 && k < K) v.x = *(const uint32_t*)(r0 + k);
    if (r1 && k < K) v.y = *(const uint32_t*)(r1 + k);
    if (r0 && k + 8 < K) v.z = *(const uint32_t*)(r0 + k + 8);
    if (r1 && k + 8 < K) v.w = *(const uint32_t*)(r1 + k + 8);
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
  float *RA, *RB, *oslots, *dslots, *act, *qbuf, *khat, *vhat, *pexit, *apart, *upart;
  int* accel_cols;
};

static int pad_to(int v, int m) { return (v + m - 1) / m * m; }

bool fused_config_ok(const m2r2_config& c) {
  if (c.dtype != M2R2_BF16 || c.n_experts != 0) return false;
  if (c.head_dim % 8 || c.head_dim > 128) return false;
  if (c.d_model % 16 || c.d_ff % 8) return false;
  if (c.accel_enabled && (c.adapter_rank > MAX_R || c.adapter_rank < 1)) return false;
  if (pad_to(c.d_model, STAGE_K) > NORM_CH * NCT * 4 || pad_to(c.d_ff, STAGE_K) > KMAX) return false;
  if ((size_t)2 * NCW * 2 * (c.head_dim + 2) * sizeof(float) > (size_t)X_BYTES) return false;
  return true;
}

struct PackedDims {
  int d_pad, F_pad, rt_qkv, rt_o, rt_gu, rt_d, rt_v;
  size_t st_qkv, st_o, st_gu, st_d, st_v;   // stages
};
static PackedDims packed_dims(const m2r2_config& c) {
  PackedDims q;
  q.d_pad = pad_to(c.d_model, STAGE_K);
  q.F_pad = pad_to(c.d_ff, STAGE_K);
  q.rt_qkv = pad_to(3 * c.d_model, 16) / 16;
  q.rt_o = pad_to(c.d_model, 16) / 16;
  q.rt_gu = pad_to(c.d_ff, 8) / 8;
  q.rt_d = q.rt_o;
  q.rt_v = pad_to(c.vocab, 16) / 16;
  q.st_qkv = (size_t)q.rt_qkv * (q.d_pad / STAGE_K);
  q.st_o = (size_t)q.rt_o * (q.d_pad / STAGE_K);
  q.st_gu = (size_t)q.rt_gu * (q.d_pad / STAGE_K);
  q.st_d = (size_t)q.rt_d * (q.F_pad / STAGE_K);
  q.st_v = (size_t)q.rt_v * (q.d_pad / STAGE_K);
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
  const size_t d = c.d_model, NG = std::max(1, c.n_gates);
  FusedImpl* im = fs ? fs->impl : nullptr;
#define FTAKE(field, T, n) { T* p_ = cv.take<T>(n); if (im) im->field = p_; }
  FTAKE(d_layers, FLayer, c.n_layers)
  FTAKE(d_ctl, Ctl, 1)
  FTAKE(d_sidx, int, c.n_heads)
  FTAKE(accel_cols, int, std::max(8, c.n_accel_heads * c.head_dim))
  FTAKE(RA, float, 2 * d) FTAKE(RB, float, 2 * d)
  FTAKE(oslots, float, (size_t)MAX_SLOTS * 2 * d) FTAKE(dslots, float, (size_t)MAX_SLOTS * 2 * d)
  FTAKE(act, float, 2 * (size_t)q.F_pad)
  FTAKE(qbuf, float, 2 * d) FTAKE(khat, float, d) FTAKE(vhat, float, d) FTAKE(pexit, float, NG * d)
  FTAKE(apart, float, (size_t)c.n_heads * M2R2_MAX_SPLITS * 2 * (c.head_dim + 4))
  FTAKE(upart, float, (size_t)2 * MAX_NJ * UPART_Q)
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
  if (!coop || max_smem < SMEM_BYTES || sms < 2 * MAX_NJ) return 0;   // per-operation kernels serve this device
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

static int pack(cudaStream_t st, void* dst, const void* src, const void* src2, int map, int n_out, int K, int n_rt,
                int nks, int d, int dh) {
  pack_kernel<<<1184, 256, 0, st>>>((uint4*)dst, (const bf16*)src, (const bf16*)src2, map, n_out, K, n_rt, nks, d, dh);
  return cudaGetLastError() == cudaSuccess ? 0 : M2R2_CUDA;
}

int fused_bind(const m2r2_config& c, FusedState* fs, cudaStream_t st, void* packed, const void* embed,
               const void* gf, const void* lm_head, const void* lm_A, const void* lm_B, const DevLayer* layers,
               void* kv, const float2* rope_tab) {
  if (!fs->supported) return 0;
  FusedImpl* im = fs->impl;
  PackedDims q = packed_dims(c);
  const int d = c.d_model, dh = c.head_dim, F = c.d_ff;
  const int ks_d = q.d_pad / STAGE_K, ks_f = q.F_pad / STAGE_K;
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
    if (pack(st, (void*)f.Wqkv, L.wqkv, nullptr, 1, 3 * d, d, q.rt_qkv, ks_d, d, dh)) return M2R2_CUDA;
    if (pack(st, (void*)f.Wo, L.wo, nullptr, 0, d, d, q.rt_o, ks_d, d, dh)) return M2R2_CUDA;
    if (pack(st, (void*)f.Wgu, L.wgate, L.wup, 2, F, d, q.rt_gu, ks_d, d, dh)) return M2R2_CUDA;
    if (pack(st, (void*)f.Wd, L.wdown, nullptr, 0, d, F, q.rt_d, ks_f, d, dh)) return M2R2_CUDA;
    f.g1 = (const bf16*)L.g1; f.g2 = (const bf16*)L.g2;
    f.Aqkv = (const bf16*)L.Aqkv; f.Bqkv = (const bf16*)L.Bqkv; f.Ao = (const bf16*)L.Ao; f.Bo = (const bf16*)L.Bo;
    f.Agu = (const bf16*)L.Agu; f.Bg = (const bf16*)L.Bg; f.Bu = (const bf16*)L.Bu; f.Ad = (const bf16*)L.Ad; f.Bd = (const bf16*)L.Bd;
    f.Kc = (bf16*)kv + (size_t)i * per;
    f.Vc = (bf16*)kv + (size_t)c.n_layers * per + (size_t)i * per;
    f.accel = (c.accel_enabled && i < c.accel_end_layer) ? 1 : 0;
    if (f.accel && L.Aqkv && L.Bd) {   // Aqkv .. Bd are carved back to back (m2r2_api.cu walk_weights)
      f.ad_lo = (const unsigned char*)L.Aqkv;
      f.ad_bytes = (unsigned int)(((const unsigned char*)L.Bd + (size_t)d * c.adapter_rank * 2) - f.ad_lo);
    }
    f.gate = 0;
    for (int j = 0; j < c.n_gates; ++j) if (c.gates[j] == i + 1) f.gate = j + 1;
  }
  const uint4* Wlm = (const uint4*)wp;
  if (pack(st, (void*)Wlm, lm_head, nullptr, 0, c.vocab, d, q.rt_v, ks_d, d, dh)) return M2R2_CUDA;
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
  cudaMemsetAsync(im->act, 0, sizeof(float) * 2 * q.F_pad, st);
  cudaMemsetAsync(im->pexit, 0, sizeof(float) * std::max(1, c.n_gates) * d, st);
  if (cudaStreamSynchronize(st) != cudaSuccess) return M2R2_CUDA;   // hl / sidx / cols are stack-owned
  im->bar_base = 0;
  FParams& p = im->p;
  memset(&p, 0, sizeof(p));
  p.d = d; p.n_heads = c.n_heads; p.dh = dh; p.F = F; p.V = c.vocab; p.r = c.accel_enabled ? c.adapter_rank : 0;
  p.da = c.n_accel_heads * dh; p.max_seq = c.max_seq;
  p.d_pad = q.d_pad; p.F_pad = q.F_pad;
  p.rt_qkv = q.rt_qkv; p.rt_o = q.rt_o; p.rt_gu = q.rt_gu; p.rt_d = q.rt_d; p.rt_v = q.rt_v;
  p.eps = c.rms_eps; p.scale = 1.0f / sqrtf((float)dh);
  p.layers = im->d_layers;
  p.embed = (const bf16*)embed; p.gf = (const bf16*)gf; p.lmA = (const bf16*)lm_A; p.lmB = (const bf16*)lm_B;
  p.Wlm = Wlm;
  p.sidx = im->d_sidx; p.accel_cols = im->accel_cols; p.rope_tab = rope_tab;
  p.n_gates = c.n_gates;
  p.RA = im->RA; p.RB = im->RB; p.oslots = im->oslots; p.dslots = im->dslots;
  p.act = im->act; p.qbuf = im->qbuf; p.khat = im->khat; p.vhat = im->vhat;
  p.pexit = im->pexit; p.apart = im->apart; p.upart = im->upart;
  p.ctl = im->d_ctl;
  p.pf_ahead = getenv("M2R2_PF") ? atoi(getenv("M2R2_PF")) : PF_DEFAULT;
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
  p.pos_host = pos;
  // grid barriers of this launch (must match the kernel's sequence): 5 per layer + the final one
  const unsigned int nbar = 5u * (unsigned int)run.n_layers + 1u;
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
