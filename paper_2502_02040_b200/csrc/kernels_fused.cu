// kernels_fused.cu — persistent fused dual-stream decode pass, v3 (bf16 storage, dense FFN, batch 1).
//
// One cooperative launch runs a whole pass (a1-a9 of SURVEY §8(a)): embed, then per layer
//   QKV    fused RMSNorm + QKV GEMV for h and p (+ adapters) with RoPE + KV append in the epilogue
//   ATTN   split-K flash-decode attention, slow query and accelerated query on the same K/V loads
//   OPROJ  O-projection, split-K: partial sums are added into the residual pair R = (h, p)
//   GATEUP RMSNorm + gate/up GEMV + SwiGLU
//   DOWN   down GEMV, split-K into R: the accelerated-residual update (Eq. 2); the gate reset p <- h
//           happens where the next phase loads the residual
// and the LM head + greedy argmax (final head on h_N, or exit/draft head on p at a gate).
//
// Design: one CTA per SM = 8 consumer warps + producer, auxiliary and L2-prefetch warps.
//  * Weights are stored FRAGMENT-MAJOR: a tile = 16 output rows x 16 inputs laid out so that lane
//    L's 16 bytes are its A fragment of mma.sync.m16n8k16; a stage = 64 tiles = 32 KB contiguous.
//      row-owned matrices (QKV, gate/up, LM head): stage = one row-tile x 1024 inputs, ordered
//        (row-tile, k-stage); a CTA owns whole row-tiles, its 8 warps split the 1024 inputs.
//      split-K matrices (O, down): stage = 8 row-tiles x 128 inputs, ordered (row-tile group, k-chunk);
//        a CTA owns a contiguous stage range, warp w owns row-tile w of the stage and accumulates in
//        registers across the k-chunks of a group, then adds its 16x2 partial sums into R with
//        red.global.add.f32.  A CTA therefore needs only its own <= ~12 k-chunks of the input vector.
//  * Weights never depend on activations, so ONE producer thread per CTA streams the CTA's statically
//    known stage sequence of the WHOLE pass through a 4-stage shared-memory ring with cp.async.bulk
//    (UBLKCP) + mbarrier: HBM stays busy while the consumers sit in a barrier or a loader.
//  * Consumers: one LDS.128 per lane = one A fragment; the B operand is the activation vector split
//    into bf16 hi + lo parts (columns h_hi, h_lo, p_hi, p_lo of the n=8 tile), so products are exact
//    to ~2^-17 and accumulate in fp32 on the tensor pipe.  It is a GEMV: the bound is HBM.
//  * What every CTA must read of the other CTAs' results is kept minimal, because those replicated
//    L2 reads (148 x the vector) share the L2->SM path with the weight stream: row-owned phases read
//    the 24 KB residual pair, split-K phases read only their slice of the attention output / SwiGLU
//    activations.
//  * Epilogues of row-owned phases are deferred: partial sums of up to 8 finished row-tiles wait in
//    shared memory and are finished by all 8 warps at once.
//  * The auxiliary warp computes the adapter down-projections u = A x^ distributed
//    over the CTAs (one row chunk each, published as (value, epoch) 8-byte entries), gathers them and hands u
//    to the consumers' epilogue (QKV, GATEUP, heads); in the split-K phases (OPROJ, DOWN) it combines the
//    r-vectors the producing phase left behind and adds B u into R.p itself.
//  * The code a layer executes is kept small (rolled loops, staged loads): the instruction cache holds 32 KB.
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include <algorithm>
#include <vector>

#include "m2r2_fused.cuh"

namespace {

typedef __nv_bfloat16 bf16;
typedef unsigned long long u64;

constexpr int STAGE_K = 1024;                  // inputs per row-owned stage
constexpr int STAGE_TILES = 64;                // m16k16 tiles per stage
constexpr int STAGE_BYTES = STAGE_TILES * 512; // 32 KB
constexpr int SK_K = 128;                      // inputs per split-K stage
constexpr int SK_RT = 8;                       // row-tiles per split-K stage
constexpr int NSTAGE = 4;
constexpr int NCW = 8;                 // consumer warps
constexpr int NCT = NCW * 32;          // consumer threads
constexpr int NTHREADS = NCT + 96;     // + producer warp + auxiliary warp + L2 prefetch warp
constexpr int TPW = STAGE_TILES / NCW; // tiles per warp per stage (8)
constexpr int XMAX = 4096;             // inputs held in shared memory (d_pad limit; 32 split-K chunks)
constexpr int XSLOTS = XMAX / SK_K;
constexpr int XCOL = XMAX + 8;         // bf16 elements per activation column (+8: LDS.128 bank spread)
constexpr int X_BYTES = 4 * XCOL * 2;  // h_hi, h_lo, p_hi, p_lo
constexpr int KMAX = 16384;            // largest inner dimension of a split-K matrix
constexpr int FB = 8;                  // finished row-tiles whose epilogue is deferred (one per warp)
constexpr int RED_FLOATS = FB * NCW * 32;
constexpr int MAX_R = 8;               // adapter rank limit (PAPER.md L399 uses 8); larger ranks take the per-operation kernels
constexpr int MAX_NJ = 3 * MAX_R;
constexpr int UPART_Q = 64;            // max k-chunks per adapter row
// exchanged adapter scratch: strides of the flagged partials (8 bytes each) and of the r-vectors.  One 128-byte
// line per item (strides 16 / 32) takes the serialisation of 148 CTAs polling one line away and is 1.5 % faster
// with exit heads on, but 3 % slower on the C2 bench workload (no exit heads) in the same GPU session: dense.
constexpr int UPART_N = 256;           // flagged partials of one phase (n_j * q <= 256)
#ifdef M2R2_PAD_SCRATCH                // test builds only: the layout under which the ring race of DESIGN.md 6.3 fired
constexpr int UPART_STRIDE = 16;       // in 8-byte entries: one 128-byte line per partial
constexpr int RV_STRIDE = 32;          // in floats: one 128-byte line per r-vector
#else
constexpr int UPART_STRIDE = 1;        // in 8-byte entries
constexpr int RV_STRIDE = MAX_R;       // in floats
#endif
static_assert(RV_STRIDE >= MAX_R, "r-vector stride");
constexpr int PF_DEFAULT = 6;           // L2 prefetch window of the prefetch warp, in stages (M2R2_PF overrides; 0 = off)
constexpr int MERGE_NS = 4;            // attention splits combined from registers by the auxiliary warp; more take a looped path
constexpr long long SPIN_LIMIT = 4000000000ll;   // ~2 s of SM clocks before a wait gives up

enum { PH_QKV = 0, PH_OPROJ = 1, PH_GATEUP = 2, PH_DOWN = 3, PH_HEAD = 4, PH_EXIT = 5, N_PH = 6 };

struct FLayer {
  const uint4 *Wqkv, *Wo, *Wgu, *Wd;   // fragment-major
  const bf16 *g1, *g2;
  const bf16 *Aqkv, *Bqkv, *Ao, *Bo, *Agu, *Bg, *Bu, *Ad, *Bd;
  const bf16 *AdT, *AoT;                // A_d transposed [F][r], A_o transposed [da][r] (fused copies)
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
  unsigned int* host_abort;   // host-mapped word written on abort (nullptr: none)
  u64 amax[1 + M2R2_MAX_GATES];   // argmax keys: [0] head of the pass, [1+j] exit head of gate j
};

struct FParams {
  int n_layers_run, d, n_heads, dh, F, V, r, da, max_seq;
  int d_pad, F_pad;                       // d padded to 1024 (row-owned K), F padded to 128 (split-K K)
  int rt_qkv, rt_gu, rt_v;                // row-tiles of the row-owned matrices
  int ng_d;                               // row-tile groups (128 rows) of the split-K matrices (n_out = d)
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
  float* R;                  // residual pair [2][d]: h then p; split-K phases add into it
  float *act, *qbuf, *khat, *vhat;
  float *apart;              // [head][split][2][dh+4]
  u64 *upart;                // [UPART_N] entries UPART_STRIDE apart (epoch << 32 | fp32 bits)
  float *apu;                // [head][split][RV_STRIDE]: A_o applied to the unnormalised accelerated attention partial
  float *udpart;             // [CTA][RV_STRIDE]: A_d applied to the CTA's own accelerated SwiGLU activations
  int nah;                   // accelerated heads
  float *trace, *logits, *exit_logits;
  Ctl* ctl;
  unsigned int bar_base;
  const int *ls_full, *ls_draft;
  int ls_first, ls_n;
  float ls_beta;
  int ns;        // attention splits
  int pos_host;  // kv_len + joff as the host knows it (producer-side KV prefetch only)
  int pf_ahead;  // L2 prefetch window in stages beyond the producer's cursor (0 = prefetch warp idle)
  unsigned int zero;   // 0 at run time, unknown to the compiler (release_stage)
  u64* tl;       // debug timeline (M2R2_FUSED_DEBUG builds), else nullptr
};

// ------------------------------------------------------------------ shared memory map (fixed offsets)
constexpr int OFF_X = NSTAGE * STAGE_BYTES;
constexpr int OFF_RED = OFF_X + X_BYTES;              // [FB][NCW][32] floats
constexpr int KV_EXTRA = 32 * 1024;                   // with the x columns and the parked sums: the attention K/V staging area
constexpr int OFF_TILE = OFF_RED + RED_FLOATS * 4 + KV_EXTRA;   // [NCW][32] floats
constexpr int OFF_U = OFF_TILE + NCW * 32 * 4;        // [MAX_NJ] floats (64 reserved)
constexpr int OFF_SRED = OFF_U + 256;                 // [64] floats
constexpr int OFF_BAR = OFF_SRED + 256;               // full[NSTAGE], empty[NSTAGE]
constexpr int OFF_UTMP = OFF_BAR + 256;               // [256] floats
constexpr int OFF_FRT = OFF_UTMP + 1024;              // [FB] ints: row-tile of each deferred flush
constexpr int OFF_UD = OFF_FRT + 64;                  // [NCW][MAX_R] floats: per-warp A_d partials of the GATEUP phase
constexpr int OFF_SIDX = OFF_UD + NCW * MAX_R * 4;    // [M2R2_MAX_HEADS] ints: head -> index in S or -1
constexpr int MAXL_S = 64;                            // layers whose descriptors are cached in shared memory
constexpr int OFF_LAYERS = OFF_SIDX + M2R2_MAX_HEADS * 4;   // [MAXL_S] FLayer
constexpr int OFF_GEO = OFF_LAYERS + MAXL_S * (int)sizeof(FLayer);   // [N_PH] int4 {s0, s1, nkc, split}: this CTA's stage range per phase type
constexpr int OFF_PCTR = OFF_GEO + 8 * 16;            // stages the producer has issued into the ring (read by the prefetch warp)
constexpr int OFF_TLN = OFF_PCTR + 16;                // debug timeline cursor
constexpr int SMEM_BYTES = OFF_TLN + 64;
static_assert(SMEM_BYTES <= 227 * 1024, "shared memory budget");
extern __shared__ __align__(1024) unsigned char smem_raw[];
__device__ __forceinline__ int sidx_of(int head) { return ((const int*)(smem_raw + OFF_SIDX))[head]; }
// layer descriptors live in shared memory: every phase of every role reads them, and a global copy would
// cost an L2 round trip after each grid barrier (its fence drops L1)
__device__ __forceinline__ const FLayer* lay(int i) { return (const FLayer*)(smem_raw + OFF_LAYERS) + i; }

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
// A consumer warp hands a ring stage back to the producer.  The arrive must not become visible before the
// warp's fragment loads of that stage have RETURNED: ptxas schedules a plain mbarrier.arrive right behind the
// issue of the last LDS (it has no register dependence on the loads), the producer refills the slot as soon as
// the eighth warp has arrived, and a refill served from L2 was observed to overwrite fragments that were still
// being read (sporadic errors of ~1e-2 in one warp's 16 rows).  The barrier's address is
// therefore made to depend, through a run-time zero, on the accumulators the stage's fragments feed.
__device__ __forceinline__ void release_stage(u64* b, unsigned int zero, float dep) {
#ifdef M2R2_PLAIN_ARRIVE               // test builds only: the unguarded arrive, to show that the stress test catches the race
  const uint32_t a = smem_u32(b);
  (void)zero; (void)dep;
#else
  const uint32_t a = smem_u32(b) + (__float_as_uint(dep) & zero);
#endif
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(a) : "memory");
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
__device__ __forceinline__ void bulk_g2s_plain(void* dst, const void* src, uint32_t bytes, u64* bar) {
  asm volatile(
      "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
      ::"r"(smem_u32(dst)), "l"(src), "r"(bytes), "r"(smem_u32(bar))
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
// named barriers: 1 = the consumer warps; 2 = "phase input ready" (consumers arrive, auxiliary warp
// waits); 3 = "auxiliary work of the phase done" (auxiliary warp arrives, consumers wait)
__device__ __forceinline__ void bar_consumers() { asm volatile("bar.sync 1, %0;" ::"n"(NCT) : "memory"); }
__device__ __forceinline__ void bar_arrive(int id) { asm volatile("bar.arrive %0, %1;" ::"r"(id), "n"(NCT + 32) : "memory"); }
__device__ __forceinline__ void bar_wait(int id) { asm volatile("bar.sync %0, %1;" ::"r"(id), "n"(NCT + 32) : "memory"); }
__device__ __forceinline__ unsigned int ld_acquire(const unsigned int* p) {
  unsigned int v;
  asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
  return v;
}
__device__ __forceinline__ void red_add(float* p, float v) {
  asm volatile("red.global.add.f32 [%0], %1;" ::"l"(p), "f"(v) : "memory");
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
// A phase has S stages.  Virtual CTA v of G owns units [U*v/G, U*(v+1)/G) where a unit is `gran`
// consecutive stages (gran = stages per row-tile for row-owned phases, 1 for split-K).
__device__ __forceinline__ int range_lo(int U, int v, int G) { return (int)(((unsigned)U * (unsigned)v) / (unsigned)G); }   // U * G < 2^32

#ifdef M2R2_FUSED_DEBUG
constexpr int TL_MAX = 4096;
__device__ __forceinline__ u64 gtime() { u64 t; asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t)); return t; }
#define TL(ev) do { int* tlp_ = (int*)(smem_raw + OFF_TLN); if (P.tl && threadIdx.x == 0 && *tlp_ < TL_MAX) { P.tl[(size_t)blockIdx.x * TL_MAX + *tlp_] = (gtime() << 8) | (u64)(ev); ++*tlp_; } } while (0)
#else
#define TL(ev) do { } while (0)
#endif

__device__ __forceinline__ void set_abort(Ctl* ctl, unsigned int where) {
  if (atomicExch(&ctl->abort_flag, 1u) == 0u) {
    ctl->abort_where = where;
    if (ctl->host_abort) { *(volatile unsigned int*)ctl->host_abort = 0x80000000u | where; __threadfence_system(); }
  }
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
__device__ __noinline__ void grid_sync(Ctl* ctl, unsigned int bar_base, unsigned int& nbar, int G) {
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
__device__ __forceinline__ uint32_t bf2_u32(__nv_bfloat162 v) { return *(uint32_t*)&v; }
// store x[k..k+3] (k % 4 == 0) as hi + lo parts into the column pair (hi, lo); packed conversions
__device__ __forceinline__ void xstore4(bf16* hi, bf16* lo, int k, float4 v) {
  const int p = xpos(k);
  const __nv_bfloat162 h01 = __floats2bfloat162_rn(v.x, v.y), h23 = __floats2bfloat162_rn(v.z, v.w);
  const float2 f01 = __bfloat1622float2(h01), f23 = __bfloat1622float2(h23);
  const __nv_bfloat162 l01 = __floats2bfloat162_rn(v.x - f01.x, v.y - f01.y), l23 = __floats2bfloat162_rn(v.z - f23.x, v.w - f23.y);
  *(uint32_t*)(hi + p) = bf2_u32(h01);
  *(uint32_t*)(hi + p + 16) = bf2_u32(h23);
  *(uint32_t*)(lo + p) = bf2_u32(l01);
  *(uint32_t*)(lo + p + 16) = bf2_u32(l23);
}
__device__ __forceinline__ float xval(const bf16* hi, const bf16* lo, int k) {
  const int p = xpos(k);
  return __bfloat162float(hi[p]) + __bfloat162float(lo[p]);
}
__device__ __forceinline__ float f4ss(float4 a) { return a.x * a.x + a.y * a.y + a.z * a.z + a.w * a.w; }
__device__ __forceinline__ void st4(float* p, float4 v) { __stcg((float4*)p, v); }

enum { LN_QKV = 0, LN_GU = 1, LN_HEAD_H = 2, LN_HEAD_P = 3 };

// Residual loader of the row-owned phases.  Every CTA reads the residual pair (h, p) from R (or the
// embedding row at the start of the pass: p_0 <- h_0), applies the gate p <- h
// (L82, L101) when the producing layer ends at a gate, and leaves x = rms(.; g) of both streams in
// shared memory.  The chunk's owner CTA writes back what changed (embedding, gate) and the trace.
struct LoadSrc {
  const bf16* emb;       // embedding row, or nullptr (then R)
  bool p_live;           // the producing layer carried p
  int gate;              // 1 + gate index: p <- h
};
// Staging area of the loaders: raw fp32 / bf16 inputs land here with 16-byte cp.async (LDGSTS through L2,
// every copy of a thread in flight at once, no registers), then rolled loops convert them into the x columns.
// Rolled loops keep the code small: the instruction cache holds 32 KB and a layer's code runs once per layer.
constexpr int STG_BYTES = RED_FLOATS * 4 + KV_EXTRA;   // 40 KB: the parked sums + the K/V extension are dead here
__device__ __forceinline__ void cp_async16(void* dst, const void* src) {
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(smem_u32(dst)), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_all;" ::: "memory"); }

__device__ __noinline__ void loader_norm(const FParams& P, bf16* x, float* sred, int mode, const LoadSrc& src,
                                         float* trace_dst, const bf16* g, int G) {
  const int tid = threadIdx.x, d = P.d, nq = d >> 2;
  float* sh = (float*)(smem_raw + OFF_RED);      // h  [d_pad] fp32
  float* sp = sh + P.d_pad;                      // p  [d_pad] fp32
  bf16* sg = (bf16*)(sp + P.d_pad);              // gains [d_pad] bf16 (40 KB in all at d_pad = 4096)
  bf16* se = x;                                  // embedding row [d] bf16: the x columns are dead until pass 2
  bar_consumers();   // x and the staging area of the previous phase are dead in every warp
  if (src.emb) {
    for (int c = tid; c < (d >> 3); c += NCT) { cp_async16(sg + 8 * c, g + 8 * c); cp_async16(se + 8 * c, src.emb + 8 * c); }
  } else {
    for (int c = tid; c < nq; c += NCT) {
      cp_async16(sh + 4 * c, P.R + 4 * c);
      if (src.p_live) cp_async16(sp + 4 * c, P.R + d + 4 * c);
    }
    for (int c = tid; c < (d >> 3); c += NCT) cp_async16(sg + 8 * c, g + 8 * c);
  }
  cp_async_wait_all();
  bar_consumers();
  TL(64);
  // ---- pass 1: gate, write-back by the chunk's owner CTA, sums of squares of the phase's two inputs
  float ssh = 0.f, ssp = 0.f;
#pragma unroll 1
  for (int c = tid; c < nq; c += NCT) {
    const int k = 4 * c;
    float4 hv, pv;
    if (src.emb) {
      const uint2 e = *(const uint2*)(se + k);
      bf16x2_to_f32(e.x, hv.x, hv.y);
      bf16x2_to_f32(e.y, hv.z, hv.w);
    } else {
      hv = *(const float4*)(sh + k);
    }
    pv = src.p_live ? *(const float4*)(sp + k) : hv;
    const float4 pbefore = pv;
    if (src.gate) pv = hv;
    if ((c % G) == (int)blockIdx.x) {
      if (trace_dst) { st4(trace_dst + k, hv); st4(trace_dst + d + k, pbefore); }
      if (src.emb) st4(P.R + k, hv);
      if (src.emb || src.gate || !src.p_live) st4(P.R + d + k, pv);
    }
    const float4 a = mode == LN_HEAD_P ? pbefore : hv;
    const float4 b = mode == LN_HEAD_P ? pbefore : (mode == LN_HEAD_H ? hv : pv);
    if (src.emb || mode != LN_QKV || src.gate || !src.p_live) { *(float4*)(sh + k) = a; *(float4*)(sp + k) = b; }   // what pass 2 reads
    ssh += f4ss(a);
    ssp += f4ss(b);
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
  // ---- pass 2: x = rms(.; g) as bf16 hi + lo columns; zero padding up to d_pad
#pragma unroll 1
  for (int c = tid; c < (P.d_pad >> 2); c += NCT) {
    const int k = 4 * c;
    float4 a = make_float4(0.f, 0.f, 0.f, 0.f), b = a;
    if (k < d) {
      a = *(const float4*)(sh + k);
      b = *(const float4*)(sp + k);
      const uint2 ge = *(const uint2*)(sg + k);
      float g0, g1, g2, g3;
      bf16x2_to_f32(ge.x, g0, g1);
      bf16x2_to_f32(ge.y, g2, g3);
      a.x = a.x * ih * g0; a.y = a.y * ih * g1; a.z = a.z * ih * g2; a.w = a.w * ih * g3;
      b.x = b.x * ip * g0; b.y = b.y * ip * g1; b.z = b.z * ip * g2; b.w = b.w * ip * g3;
    }
    xstore4(c0, c1, k, a);
    xstore4(c2, c3, k, b);
  }
  bar_consumers();
}

// Input slice of a split-K phase: the CTA's stages [s0, s1) of a matrix with nkc k-chunks per row-tile
// group touch chunks kc0, kc0+1, ... (mod nkc), cnt of them; chunk kc lives in x slot kc % XSLOTS.
//   OPROJ: merged attention output of both queries (the accelerated stream has columns of S only): the
//          split partials (m, l, o) of the heads the chunks touch are staged, then merged in split order
//   DOWN:  SwiGLU activations of both streams
__device__ __noinline__ float4 merge_global(const FParams& P, int q, int k) {   // partials do not fit the staging area
  const int dh = P.dh, NS = P.ns, head = k / dh, j = k - head * dh;
  const float* pp = P.apart + ((size_t)(head * NS) * 2 + q) * (dh + 4);
  float M = -INFINITY, Lsum = 0.f;
  float4 o = make_float4(0.f, 0.f, 0.f, 0.f);
  for (int s = 0; s < NS; ++s) {
    const float* ps = pp + (size_t)s * 2 * (dh + 4);
    if (ldcg(ps + dh + 1) > 0.f) M = fmaxf(M, ldcg(ps + dh));
  }
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
  return o;
}
__device__ __noinline__ void loader_slice(const FParams& P, bf16* x, int ph, bool accel, int kc0, int cnt, int nkc) {
  const int tid = threadIdx.x;
  float* stg = (float*)(smem_raw + OFF_RED);
  bf16 *c0 = x, *c1 = x + XCOL, *c2 = x + 2 * XCOL, *c3 = x + 3 * XCOL;
  const int items = cnt * 64;   // (chunk, stream, float4)
  bar_consumers();
  if (ph == PH_DOWN) {
#pragma unroll 1
    for (int it = tid; it < items; it += NCT) {
      const int i = it >> 6, rem = it & 63, q = rem >> 5, c4 = rem & 31;
      int kc = kc0 + i;
      if (kc >= nkc) kc -= nkc;
      const int k = kc * SK_K + c4 * 4;
      if (k < P.F && (q == 0 || accel)) cp_async16(stg + 4 * it, P.act + (size_t)q * P.F_pad + k);
      else *(float4*)(stg + 4 * it) = make_float4(0.f, 0.f, 0.f, 0.f);
    }
    cp_async_wait_all();
    bar_consumers();
#pragma unroll 1
    for (int it = tid; it < items; it += NCT) {
      const int i = it >> 6, rem = it & 63, q = rem >> 5, c4 = rem & 31;
      int kc = kc0 + i;
      if (kc >= nkc) kc -= nkc;
      const int xs = (kc % XSLOTS) * SK_K + c4 * 4;
      const float4 v = *(const float4*)(stg + 4 * it);
      if (q == 0) xstore4(c0, c1, xs, v); else xstore4(c2, c3, xs, v);
    }
  } else {
    // heads touched by the two runs of chunks: [kc0, kcA) and, after the wrap, [0, kcB)
    const int dh = P.dh, NS = P.ns, rec = NS * 2 * (dh + 4);   // floats of one head's partials
    const int kcA = min(kc0 + cnt, nkc), kcB = kc0 + cnt - kcA;
    const int hA0 = (kc0 * SK_K) / dh, hA1 = min(P.n_heads - 1, (kcA * SK_K - 1) / dh);
    const int nA = hA1 - hA0 + 1, nB = kcB > 0 ? min(P.n_heads - 1, (kcB * SK_K - 1) / dh) + 1 : 0;
    const bool staged = (size_t)(nA + nB) * rec * 4 <= (size_t)STG_BYTES;
    if (staged) {
      const float* srcA = P.apart + (size_t)hA0 * rec;
#pragma unroll 1
      for (int i = tid; i < ((nA * rec) >> 2); i += NCT) cp_async16(stg + 4 * i, srcA + 4 * i);
#pragma unroll 1
      for (int i = tid; i < ((nB * rec) >> 2); i += NCT) cp_async16(stg + nA * rec + 4 * i, P.apart + 4 * i);
      cp_async_wait_all();
      bar_consumers();
    }
#pragma unroll 1
    for (int it = tid; it < items; it += NCT) {
      const int i = it >> 6, rem = it & 63, q = rem >> 5, c4 = rem & 31;
      int kc = kc0 + i;
      const bool wrapped = kc >= nkc;
      if (wrapped) kc -= nkc;
      const int k = kc * SK_K + c4 * 4;
      const int xs = (kc % XSLOTS) * SK_K + c4 * 4;
      float4 o = make_float4(0.f, 0.f, 0.f, 0.f);
      if (k < P.d && (q == 0 || (accel && sidx_of(k / dh) >= 0))) {
        if (staged) {
          const int head = k / dh, j = k - head * dh;
          const float* pp = stg + (size_t)(wrapped ? nA + head : head - hA0) * rec + q * (dh + 4);
          float M = -INFINITY, Lsum = 0.f;
#pragma unroll 1
          for (int sp = 0; sp < NS; ++sp) {
            const float* ps = pp + sp * 2 * (dh + 4);
            if (ps[dh + 1] > 0.f) M = fmaxf(M, ps[dh]);
          }
#pragma unroll 1
          for (int sp = 0; sp < NS; ++sp) {
            const float* ps = pp + sp * 2 * (dh + 4);
            const float ls = ps[dh + 1];
            if (ls > 0.f) {
              const float wgt = __expf(ps[dh] - M);
              const float4 v = *(const float4*)(ps + j);
              Lsum += ls * wgt;
              o.x += v.x * wgt; o.y += v.y * wgt; o.z += v.z * wgt; o.w += v.w * wgt;
            }
          }
          const float inv = 1.f / Lsum;
          o.x *= inv; o.y *= inv; o.z *= inv; o.w *= inv;
        } else {
          o = merge_global(P, q, k);
        }
      }
      if (q == 0) xstore4(c0, c1, xs, o); else xstore4(c2, c3, xs, o);
    }
  }
  bar_consumers();
}

// ------------------------------------------------------------------ auxiliary warp: adapter down-projections
// u = A x^ of the accelerated row in the row-owned phases, distributed: CTA c computes row
// j = c / q over k-chunk c % q and publishes (value, epoch) as ONE 8-byte store; every CTA's fetch_u() polls
// the nj * q entries until they carry the phase's epoch, then sums the q chunks of every row in chunk order
// (deterministic).  No counter, no fence: two L2 round trips from "x ready" to "u ready".
struct UState {
  unsigned int epoch;    // epoch of the current phase (unique per launch and phase, never 0)
  int nj, q;             // geometry of the current phase
};
constexpr int AW = 2;    // A-row chunks (256 inputs each) loaded before the phase's input is ready
struct APre {
  uint4 w[AW];
};
__device__ __forceinline__ void u_geometry(UState& us, int nj, int G) {
  us.nj = nj;
  us.q = min(min(G / nj, UPART_Q), UPART_N / nj);
}
__device__ __forceinline__ void publish_prefetch(const UState& us, APre& ap, const bf16* A, int Kc) {
  const int lane = threadIdx.x & 31, c = blockIdx.x;
#pragma unroll
  for (int i = 0; i < AW; ++i) ap.w[i] = make_uint4(0u, 0u, 0u, 0u);
  if (c < us.nj * us.q) {
    const int j = c / us.q, ch = c - j * us.q;
    const int chunk = (((Kc + us.q - 1) / us.q) + 7) & ~7;
    const int k0 = ch * chunk, k1 = min(Kc, k0 + chunk);
    const bf16* a = A + (size_t)j * Kc;
#pragma unroll
    for (int i = 0; i < AW; ++i) {
      const int k = k0 + lane * 8 + i * 256;
      if (k < k1) ap.w[i] = __ldg((const uint4*)(a + k));
    }
  }
}
__device__ __forceinline__ void publish_u(const FParams& P, const bf16* x, const UState& us, const APre& ap, const bf16* A, int Kc) {
  const int lane = threadIdx.x & 31, c = blockIdx.x;
  if (c < us.nj * us.q) {
    const int j = c / us.q, ch = c - j * us.q;
    const int chunk = (((Kc + us.q - 1) / us.q) + 7) & ~7;
    const int k0 = ch * chunk, k1 = min(Kc, k0 + chunk);
    const bf16* a = A + (size_t)j * Kc;
    const bf16 *xh = x + 2 * XCOL, *xl = x + 3 * XCOL;
    float acc = 0.f;
    int it = 0;
    for (int k = k0 + lane * 8; k < k1; k += 256, ++it) {   // chunk and Kc are multiples of 8
      uint4 w;
      if (it == 0) w = ap.w[0];
      else if (it == 1) w = ap.w[1];
      else w = __ldg((const uint4*)(a + k));
      float f[8];
      bf16x2_to_f32(w.x, f[0], f[1]); bf16x2_to_f32(w.y, f[2], f[3]);
      bf16x2_to_f32(w.z, f[4], f[5]); bf16x2_to_f32(w.w, f[6], f[7]);
#pragma unroll
      for (int e = 0; e < 8; ++e) acc += f[e] * xval(xh, xl, k + e);
    }
    acc = warp_sum(acc);
    if (lane == 0) {
      const u64 v = ((u64)us.epoch << 32) | (u64)__float_as_uint(acc);
      asm volatile("st.global.cg.u64 [%0], %1;" ::"l"(P.upart + (size_t)c * UPART_STRIDE), "l"(v) : "memory");   // entry index = j * q + ch = c
    }
  }
}
__device__ __forceinline__ void fetch_u(const FParams& P, float* u, float* utmp, const UState& us) {
  const int lane = threadIdx.x & 31;
  const int total = us.nj * us.q;   // <= 256
  float v[8];
  long long t0 = clock64();
  unsigned int n = 0;
  for (;;) {
    bool ok = true;
#pragma unroll
    for (int i = 0; i < 8; ++i) {
      const int idx = lane + 32 * i;
      v[i] = 0.f;
      if (idx < total) {
        u64 e;
        asm volatile("ld.relaxed.gpu.global.u64 %0, [%1];" : "=l"(e) : "l"(P.upart + (size_t)idx * UPART_STRIDE) : "memory");
        ok = ok && (unsigned int)(e >> 32) == us.epoch;
        v[i] = __uint_as_float((unsigned int)e);
      }
    }
    if (__all_sync(0xffffffffu, ok)) break;
    if ((++n & 255u) == 0u) {
      if (aborted(P.ctl)) break;
      if (clock64() - t0 > SPIN_LIMIT) { set_abort(P.ctl, 0x500u); break; }
    }
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
// a row of r <= 8 adapter weights loaded ahead of its use: one 16-byte load when r == 8
struct RVec {
  uint4 a;
  const bf16* p;
};
__device__ __forceinline__ RVec rv_load(const bf16* p, int r) {
  RVec v;
  v.p = p;
  v.a = make_uint4(0u, 0u, 0u, 0u);
  if (r == 8) v.a = __ldg((const uint4*)p);
  return v;
}
__device__ __forceinline__ void rv_unpack(const RVec& v, int r, float (&f)[MAX_R]) {
  if (r == 8) {
    bf16x2_to_f32(v.a.x, f[0], f[1]); bf16x2_to_f32(v.a.y, f[2], f[3]);
    bf16x2_to_f32(v.a.z, f[4], f[5]); bf16x2_to_f32(v.a.w, f[6], f[7]);
  } else {
#pragma unroll
    for (int j = 0; j < MAX_R; ++j) f[j] = j < r ? bf(v.p + j) : 0.f;
  }
}
__device__ __forceinline__ float rv_dot(const RVec& v, const float* u, int r) {
  float f[MAX_R], s = 0.f;
  rv_unpack(v, r, f);
#pragma unroll
  for (int j = 0; j < MAX_R; ++j) if (j < r) s += f[j] * u[j];
  return s;
}
// split-K phases: u of the adapter from partials the PRODUCING phase left behind (one L2 round trip, no
// publish / fetch): OPROJ  u = A_o o^ from the attention items' r-vectors and (m, l); DOWN  u = A_d a^ as
// the sum of the CTAs' r-vectors in CTA order.
__device__ __noinline__ float combine_slow(const FParams& P, int head, float (&part)[MAX_R]) {
  const int NS = P.ns, dh = P.dh, r = P.r;
  float M = -INFINITY, Lsum = 0.f;
  for (int s = 0; s < NS; ++s) {
    const float2 ml = __ldcg((const float2*)(P.apart + ((size_t)(head * NS + s) * 2 + 1) * (dh + 4) + dh));
    if (ml.y > 0.f) M = fmaxf(M, ml.x);
  }
  for (int s = 0; s < NS; ++s) {
    const float2 ml = __ldcg((const float2*)(P.apart + ((size_t)(head * NS + s) * 2 + 1) * (dh + 4) + dh));
    if (ml.y > 0.f) {
      const float wgt = __expf(ml.x - M);
      Lsum += ml.y * wgt;
      const float* q = P.apu + (size_t)(head * NS + s) * RV_STRIDE;
#pragma unroll
      for (int i = 0; i < MAX_R; ++i) if (i < r) part[i] += ldcg(q + i) * wgt;
    }
  }
  return Lsum;
}
__device__ __forceinline__ void combine_u(const FParams& P, float* u, int ph, int G) {
  const int lane = threadIdx.x & 31, r = P.r;
  float acc[MAX_R];
#pragma unroll
  for (int i = 0; i < MAX_R; ++i) acc[i] = 0.f;
  if (ph == PH_OPROJ) {
    const int NS = P.ns, dh = P.dh;
    for (int si = lane; si < P.nah; si += 32) {
      const int head = P.accel_cols[si * dh] / dh;
      float Lsum = 0.f, part[MAX_R];
#pragma unroll
      for (int i = 0; i < MAX_R; ++i) part[i] = 0.f;
      if (NS <= MERGE_NS) {
        // every load first (one L2 round trip), then the merge
        float2 ml[MERGE_NS];
        float4 pu[MERGE_NS][MAX_R / 4];
#pragma unroll
        for (int s = 0; s < MERGE_NS; ++s) {
          ml[s] = make_float2(0.f, 0.f);
#pragma unroll
          for (int c = 0; c < MAX_R / 4; ++c) pu[s][c] = make_float4(0.f, 0.f, 0.f, 0.f);
          if (s < NS) {
            ml[s] = __ldcg((const float2*)(P.apart + ((size_t)(head * NS + s) * 2 + 1) * (dh + 4) + dh));
            const float* q = P.apu + (size_t)(head * NS + s) * RV_STRIDE;
#pragma unroll
            for (int c = 0; c < MAX_R / 4; ++c) if (c * 4 < r) pu[s][c] = ldcg4(q + c * 4);
          }
        }
        float M = -INFINITY;
#pragma unroll
        for (int s = 0; s < MERGE_NS; ++s) if (s < NS && ml[s].y > 0.f) M = fmaxf(M, ml[s].x);
#pragma unroll
        for (int s = 0; s < MERGE_NS; ++s) {
          if (s < NS && ml[s].y > 0.f) {
            const float wgt = __expf(ml[s].x - M);
            Lsum += ml[s].y * wgt;
#pragma unroll
            for (int c = 0; c < MAX_R / 4; ++c) {
              part[c * 4 + 0] += pu[s][c].x * wgt; part[c * 4 + 1] += pu[s][c].y * wgt;
              part[c * 4 + 2] += pu[s][c].z * wgt; part[c * 4 + 3] += pu[s][c].w * wgt;
            }
          }
        }
      } else {
        Lsum = combine_slow(P, head, part);
      }
      const float inv = 1.f / Lsum;
#pragma unroll
      for (int i = 0; i < MAX_R; ++i) acc[i] += part[i] * inv;
    }
  } else {
    for (int c = lane; c < G; c += 32) {
      const float* pu = P.udpart + (size_t)c * RV_STRIDE;
#pragma unroll
      for (int i = 0; i < MAX_R; ++i) if (i < r) acc[i] += ldcg(pu + i);
    }
  }
#pragma unroll
  for (int i = 0; i < MAX_R; ++i) {
    if (i < r) {
      const float v = warp_sum(acc[i]);
      if (lane == 0) u[i] = v;
    }
  }
  __syncwarp();
}
// split-K phases: R.p[n] += B[n] . u for this CTA's share of the rows (the adapter up-projection)
struct BPre {
  RVec row;
  int n;
};
__device__ __forceinline__ void apply_prefetch(const FParams& P, BPre& bp, const bf16* B, int G) {
  const int lane = threadIdx.x & 31, d = P.d, r = P.r;
  const int per = (d + G - 1) / G, n0 = (int)blockIdx.x * per, n1 = min(d, n0 + per);
  bp.n = n0 + lane < n1 ? n0 + lane : -1;
  bp.row = rv_load(B + (size_t)(bp.n >= 0 ? bp.n : 0) * r, r);
}
__device__ __forceinline__ void apply_Bu(const FParams& P, const BPre& bp, const bf16* B, const float* u, int G) {
  const int lane = threadIdx.x & 31, d = P.d, r = P.r;
  const int per = (d + G - 1) / G, n0 = (int)blockIdx.x * per, n1 = min(d, n0 + per);
  if (bp.n >= 0) red_add(P.R + d + bp.n, rv_dot(bp.row, u, r));
  for (int n = n0 + lane + 32; n < n1; n += 32) red_add(P.R + d + n, lora_dot(B + (size_t)n * r, u, r));
}

// ------------------------------------------------------------------ row-owned phase epilogues (one warp per finished 16-row tile, sums in T[row][stream])
struct PhaseCtx {
  int ph, layer;
  const FLayer* L;
  int pos;          // position of the token of this pass
  bool accel;       // stream 1 live
};

__device__ __forceinline__ void epilogue_tile(const FParams& P, const float* T, const float* u, const PhaseCtx& c, int rt,
                                              float (&udacc)[MAX_R]) {
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
        const int si = sidx_of(head);
        const bool live = s == 0 || si >= 0;
        if (live) {
          // every global load of the lane first: adapter rows, RoPE pair
          const bool lora = s == 1 && r > 0;
          RVec b0, b1;
          float2 cs = make_float2(1.f, 0.f);
          if (lora) {
            const bf16* B = c.L->Bqkv + ((size_t)which * P.da + (size_t)si * dh) * r;
            b0 = rv_load(B + (size_t)e0 * r, r);
            b1 = rv_load(B + (size_t)e1 * r, r);
          }
          if (which < 2) cs = P.rope_tab[(size_t)c.pos * half + e0];
          if (lora) {   // parallel adapters: + B (A x^)   (Q3)
            v0 += rv_dot(b0, u + which * r, r);
            v1 += rv_dot(b1, u + which * r, r);
          }
          if (which < 2) {
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
  } else if (c.ph == PH_GATEUP) {
    // packed tile: gate rows n..n+7 then up rows n..n+7
    float a_p = 0.f;
    RVec at;
    bool have_p = false;
    if (lane < 16) {
      const int nl = lane >> 1, s = lane & 1, n = rt * 8 + nl;
      if (n < P.F && (s == 0 || c.accel)) {
        float g = T[nl * 2 + s], up = T[(8 + nl) * 2 + s];
        if (s == 1 && r > 0) {
          // every global load of the lane first: B_g, B_u rows and the A_d column
          const RVec bg = rv_load(c.L->Bg + (size_t)n * r, r), bu = rv_load(c.L->Bu + (size_t)n * r, r);
          at = rv_load(c.L->AdT + (size_t)n * r, r);
          have_p = true;
          g += rv_dot(bg, u, r);
          up += rv_dot(bu, u + r, r);
        }
        const float a = silu(g) * up;
        __stcg(P.act + s * P.F_pad + n, a);
        if (s == 1) a_p = a;
      }
    }
    if (c.accel && r > 0) {
      // A_d a^ over the tile's 8 activations: the down-projection adapter's u, accumulated per warp and
      // summed over the CTAs after the barrier (the auxiliary warp of the DOWN phase)
      float cj[MAX_R];
#pragma unroll
      for (int j = 0; j < MAX_R; ++j) cj[j] = 0.f;
      if (have_p) {
        rv_unpack(at, r, cj);
#pragma unroll
        for (int j = 0; j < MAX_R; ++j) cj[j] *= a_p;
      }
#pragma unroll
      for (int j = 0; j < MAX_R; ++j) {
        if (j < r) {
          cj[j] += __shfl_xor_sync(0xffffffffu, cj[j], 2);
          cj[j] += __shfl_xor_sync(0xffffffffu, cj[j], 4);
          cj[j] += __shfl_xor_sync(0xffffffffu, cj[j], 8);
          udacc[j] += cj[j];   // meaningful in lane 1
        }
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
// Work item = (head, split), one per CTA.  The item's keys and values of positions [p0, p1) < pos are two
// contiguous ranges of the cache ([head][position][dh]): one thread stages them into shared memory with two
// bulk copies per round (prefetched into L2 by the producer), then every half-warp walks its positions in a
// rolled loop; both queries share every K/V read.  The last split also takes the token's own key/value:
// slow = K[pos], V[pos] as stored (rounded), accelerated = k^, v^ from scratch (p_t attends
// h_<t (+) p_t).  Partials (m, l, o) go to P.apart; the O-proj loader merges them.
constexpr int KV_BYTES = X_BYTES + RED_FLOATS * 4 + KV_EXTRA;   // staging area: the x columns and the parked sums are dead here
__device__ __noinline__ void attn_phase(const FParams& P, unsigned char* kvbuf, float* osm, float* wsm, u64* abar, unsigned int& aphase,
                                        const FLayer* L, int pos, bool accel, int G) {
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int dh = P.dh, d = P.d, lpp = dh >> 3, NS = P.ns;
  const int seg = lane >> 4, sl = lane & 15, hw = warp * 2 + seg;
  const bool active = sl < lpp;
  const int items = P.n_heads * NS;
  const int cap = KV_BYTES / (4 * dh);   // positions per round (K and V rows of dh bf16 each)
  float* red = (float*)kvbuf;                    // after the rounds: [2 NCW segments][2 queries][dh + 2]
  for (int w = blockIdx.x; w < items; w += G) {
    const int head = w / NS, sp = w - head * NS;
    const bool q1 = accel && sidx_of(head) >= 0;
    const int chunk = (pos + NS - 1) / NS;
    const int p0 = min(pos, sp * chunk), p1 = min(pos, p0 + chunk);
    const bf16* Kg = L->Kc + (size_t)head * P.max_seq * dh;
    const bf16* Vg = L->Vc + (size_t)head * P.max_seq * dh;
    bf16* ks = (bf16*)kvbuf;
    bf16* vs = ks + (size_t)cap * dh;
    if (tid == 0 && p1 > p0) {   // first round in flight before the queries are even loaded
      const int n = min(cap, p1 - p0);
      asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
      mbar_expect_tx(abar, (uint32_t)(2 * n * dh * 2));
      bulk_g2s_plain(ks, Kg + (size_t)p0 * dh, (uint32_t)(n * dh * 2), abar);
      bulk_g2s_plain(vs, Vg + (size_t)p0 * dh, (uint32_t)(n * dh * 2), abar);
    }
    // the token's own key/value and the queries: every load issued before anything is used
    const bool own = sp == NS - 1 && warp == 0;   // this warp adds the token's own key/value (segment 0)
    uint4 ko = make_uint4(0u, 0u, 0u, 0u), vo = ko;
    float4 kh0 = make_float4(0.f, 0.f, 0.f, 0.f), kh1 = kh0, vh0 = kh0, vh1 = kh0;
    if (own && seg == 0 && active) {
      ko = ldcg16(Kg + (size_t)pos * dh + sl * 8);
      vo = ldcg16(Vg + (size_t)pos * dh + sl * 8);
      if (q1) {
        kh0 = ldcg4(P.khat + head * dh + sl * 8); kh1 = ldcg4(P.khat + head * dh + sl * 8 + 4);
        vh0 = ldcg4(P.vhat + head * dh + sl * 8); vh1 = ldcg4(P.vhat + head * dh + sl * 8 + 4);
      }
    }
    float qa[8], qb[8];
#pragma unroll
    for (int e = 0; e < 8; ++e) { qa[e] = 0.f; qb[e] = 0.f; }
    if (active) {
      const float4 a0 = ldcg4(P.qbuf + head * dh + sl * 8), a1 = ldcg4(P.qbuf + head * dh + sl * 8 + 4);
      float4 b0 = make_float4(0.f, 0.f, 0.f, 0.f), b1 = b0;
      if (q1) { b0 = ldcg4(P.qbuf + d + head * dh + sl * 8); b1 = ldcg4(P.qbuf + d + head * dh + sl * 8 + 4); }
      qa[0] = a0.x * P.scale; qa[1] = a0.y * P.scale; qa[2] = a0.z * P.scale; qa[3] = a0.w * P.scale;
      qa[4] = a1.x * P.scale; qa[5] = a1.y * P.scale; qa[6] = a1.z * P.scale; qa[7] = a1.w * P.scale;
      qb[0] = b0.x * P.scale; qb[1] = b0.y * P.scale; qb[2] = b0.z * P.scale; qb[3] = b0.w * P.scale;
      qb[4] = b1.x * P.scale; qb[5] = b1.y * P.scale; qb[6] = b1.z * P.scale; qb[7] = b1.w * P.scale;
    }
    float m0 = -INFINITY, l0 = 0.f, m1 = -INFINITY, l1 = 0.f, o0[8], o1[8];
#pragma unroll
    for (int e = 0; e < 8; ++e) { o0[e] = 0.f; o1[e] = 0.f; }
    for (int r0 = p0; r0 < p1; r0 += cap) {
      const int n = min(cap, p1 - r0);
      if (r0 > p0) {
        bar_consumers();   // the previous round's rows are consumed
        if (tid == 0) {
          asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
          mbar_expect_tx(abar, (uint32_t)(2 * n * dh * 2));
          bulk_g2s_plain(ks, Kg + (size_t)r0 * dh, (uint32_t)(n * dh * 2), abar);
          bulk_g2s_plain(vs, Vg + (size_t)r0 * dh, (uint32_t)(n * dh * 2), abar);
        }
      }
      TL(73);
      mbar_wait(abar, aphase & 1u, P.ctl, 0x300u);
      ++aphase;
      TL(74);
#pragma unroll 1
      for (int ub = warp * 2; ub < n; ub += 2 * NCW) {   // warp-uniform trip count (full-mask shuffles below)
        const int u = ub + seg;
        const bool valid = u < n;
        uint4 kk = make_uint4(0u, 0u, 0u, 0u), vv = kk;
        if (active && valid) {
          kk = *(const uint4*)(ks + (size_t)u * dh + sl * 8);
          vv = *(const uint4*)(vs + (size_t)u * dh + sl * 8);
        }
        float kf[8], vf[8];
        bf16x2_to_f32(kk.x, kf[0], kf[1]); bf16x2_to_f32(kk.y, kf[2], kf[3]);
        bf16x2_to_f32(kk.z, kf[4], kf[5]); bf16x2_to_f32(kk.w, kf[6], kf[7]);
        bf16x2_to_f32(vv.x, vf[0], vf[1]); bf16x2_to_f32(vv.y, vf[2], vf[3]);
        bf16x2_to_f32(vv.z, vf[4], vf[5]); bf16x2_to_f32(vv.w, vf[6], vf[7]);
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
    }
    TL(70);
    // ---- the token's own key/value (last split, warp 0, segment 0)
    if (own) {
      float kf[8], vf[8], k2[8], v2[8];
      bf16x2_to_f32(ko.x, kf[0], kf[1]); bf16x2_to_f32(ko.y, kf[2], kf[3]);
      bf16x2_to_f32(ko.z, kf[4], kf[5]); bf16x2_to_f32(ko.w, kf[6], kf[7]);
      bf16x2_to_f32(vo.x, vf[0], vf[1]); bf16x2_to_f32(vo.y, vf[2], vf[3]);
      bf16x2_to_f32(vo.z, vf[4], vf[5]); bf16x2_to_f32(vo.w, vf[6], vf[7]);
      k2[0] = kh0.x; k2[1] = kh0.y; k2[2] = kh0.z; k2[3] = kh0.w; k2[4] = kh1.x; k2[5] = kh1.y; k2[6] = kh1.z; k2[7] = kh1.w;
      v2[0] = vh0.x; v2[1] = vh0.y; v2[2] = vh0.z; v2[3] = vh0.w; v2[4] = vh1.x; v2[5] = vh1.y; v2[6] = vh1.z; v2[7] = vh1.w;
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
    TL(71);
    // ---- merge the lane segments of the CTA -> one partial per query
    bar_consumers();   // every half-warp is done with the staged rows: the area becomes the merge scratch
    {
      float* dst0 = red + ((size_t)hw * 2 + 0) * (dh + 2);
      float* dst1 = red + ((size_t)hw * 2 + 1) * (dh + 2);
      if (active) {
#pragma unroll
        for (int e = 0; e < 8; ++e) { dst0[sl * 8 + e] = o0[e]; dst1[sl * 8 + e] = o1[e]; }
      }
      if (sl == 0) { dst0[dh] = m0; dst0[dh + 1] = l0; dst1[dh] = m1; dst1[dh + 1] = l1; }
    }
    bar_consumers();
    if (warp == 0) {
      // weights of the 16 half-warp partials of each query: lane = (segment, query)
      const int s_ = lane >> 1, q_ = lane & 1;
      const float* src = red + ((size_t)s_ * 2 + q_) * (dh + 2);
      const float ms = src[dh], ls = src[dh + 1];
      float M = ls > 0.f ? ms : -INFINITY;
#pragma unroll
      for (int o = 2; o < 32; o <<= 1) M = fmaxf(M, __shfl_xor_sync(0xffffffffu, M, o));
      const float wgt = ls > 0.f ? __expf(ms - M) : 0.f;
      float Lsum = ls * wgt;
#pragma unroll
      for (int o = 2; o < 32; o <<= 1) Lsum += __shfl_xor_sync(0xffffffffu, Lsum, o);
      wsm[lane] = wgt;
      if (s_ == 0) { wsm[32 + q_] = M; wsm[34 + q_] = Lsum; }
    }
    bar_consumers();
    for (int i = tid; i < 2 * dh; i += NCT) {
      const int q = i / dh, j = i - q * dh;
      float O = 0.f;
#pragma unroll
      for (int s = 0; s < 2 * NCW; ++s) O += red[((size_t)s * 2 + q) * (dh + 2) + j] * wsm[s * 2 + q];
      float* pp = P.apart + ((size_t)(head * NS + sp) * 2 + q) * (dh + 4);
      __stcg(pp + j, O);
      if (j == 0) { __stcg(pp + dh, wsm[32 + q]); __stcg(pp + dh + 1, wsm[34 + q]); }
      if (q == 1) osm[j] = O;
    }
    bar_consumers();
    TL(72);
    if (q1 && P.r > 0 && warp == 0) {
      // O-projection adapter: A_o restricted to this head, applied to the unnormalised partial (linear in the
      // partials, so the auxiliary warp of the OPROJ phase only combines the splits' r-vectors)
      const bf16* At = L->AoT + (size_t)sidx_of(head) * dh * P.r;   // [column of the head][r]
      constexpr int JC = 4;   // dh <= 128
      RVec av[JC];
#pragma unroll
      for (int c = 0; c < JC; ++c) {
        const int j = lane + 32 * c;
        av[c] = rv_load(At + (size_t)(j < dh ? j : 0) * P.r, P.r);
      }
      float acc[MAX_R];
#pragma unroll
      for (int i = 0; i < MAX_R; ++i) acc[i] = 0.f;
#pragma unroll
      for (int c = 0; c < JC; ++c) {
        const int j = lane + 32 * c;
        if (j < dh) {
          float f[MAX_R];
          rv_unpack(av[c], P.r, f);
          const float o = osm[j];
#pragma unroll
          for (int i = 0; i < MAX_R; ++i) acc[i] += f[i] * o;
        }
      }
#pragma unroll
      for (int i = 0; i < MAX_R; ++i) {
        if (i < P.r) {
          const float v = warp_sum(acc[i]);
          if (lane == 0) __stcg(P.apu + (size_t)(head * NS + sp) * RV_STRIDE + i, v);
        }
      }
    }
  }
}

// ------------------------------------------------------------------ the phase sequence of a pass (shared by producer, consumers, auxiliary warp)
__device__ __forceinline__ bool exit_phase_after(const FParams& P, int layer) {
  const FLayer* L = lay(layer);
  return L->gate && L->accel && P.exit_heads && !(P.head_stream == 1 && layer + 1 == P.n_layers_run);
}
// geometry of a weight phase: stages S = U * gran; the CTA's stage range [s0, s1)
struct PhaseGeo {
  const unsigned char* W;
  int nkc;                   // k-chunks per row-tile group (split-K) / k-stages per row-tile (row-owned)
  bool split;
  int s0, s1;
};
// The CTA's stage range of every phase TYPE is the same in every layer: computed once per launch into
// shared memory (thread p < N_PH) so that a phase's set-up is four shared loads, not a page of integer code.
__device__ __forceinline__ void geo_init(const FParams& P, int ph, int G) {
  const int nks_d = P.d_pad / STAGE_K;
  int n_units, gran, nkc, split = 0;
  switch (ph) {
    case PH_QKV:    n_units = P.rt_qkv; gran = nks_d; nkc = nks_d; break;
    case PH_OPROJ:  nkc = (P.d + SK_K - 1) / SK_K; n_units = P.ng_d * nkc; gran = 1; split = 1; break;
    case PH_GATEUP: n_units = P.rt_gu; gran = nks_d; nkc = nks_d; break;
    case PH_DOWN:   nkc = P.F_pad / SK_K; n_units = P.ng_d * nkc; gran = 1; split = 1; break;
    default:        n_units = P.rt_v; gran = nks_d; nkc = nks_d; break;   // PH_HEAD, PH_EXIT
  }
  // rotate the owner of the short ranges between phase types
  const int v = ((int)blockIdx.x + ph * 29) % G;
  int4 e;
  e.x = range_lo(n_units, v, G) * gran;
  e.y = range_lo(n_units, v + 1, G) * gran;
  e.z = nkc;
  e.w = split;
  ((int4*)(smem_raw + OFF_GEO))[ph] = e;
}
__device__ __forceinline__ void phase_geo(const FParams& P, int layer, int ph, int G, PhaseGeo& g) {
  const int n = P.n_layers_run;
  const FLayer* L = lay(layer < n ? layer : 0);
  const int4 e = ((const int4*)(smem_raw + OFF_GEO))[ph];
  g.s0 = e.x; g.s1 = e.y; g.nkc = e.z; g.split = e.w != 0;
  g.W = (const unsigned char*)(ph == PH_QKV ? L->Wqkv : ph == PH_OPROJ ? L->Wo : ph == PH_GATEUP ? L->Wgu : ph == PH_DOWN ? L->Wd : P.Wlm);
}
// next weight phase after (layer, ph); ph = -1 before the first.  false at the end of the pass.
__device__ __forceinline__ bool next_weight_phase(const FParams& P, int& layer, int& ph) {
  const int n = P.n_layers_run;
  if (ph == PH_HEAD) return false;
  bool next_layer = false;
  if (ph < 0) { layer = -1; next_layer = true; }
  else if (ph == PH_QKV) ph = PH_OPROJ;
  else if (ph == PH_OPROJ) ph = PH_GATEUP;
  else if (ph == PH_GATEUP) ph = PH_DOWN;
  else if (ph == PH_DOWN) { if (exit_phase_after(P, layer)) ph = PH_EXIT; else next_layer = true; }
  else next_layer = true;   // PH_EXIT
  if (next_layer) {
    ++layer;
    ph = layer < n ? PH_QKV : PH_HEAD;
  }
  return true;
}

// producer cursor: walks the CTA's stages of the pass in consumption order
struct Cursor {
  int layer, ph;
  int s, s1;
  const unsigned char* W;
  bool new_layer;
};
__device__ __noinline__ bool cursor_advance(const FParams& P, Cursor& c, int G) {
  if (!next_weight_phase(P, c.layer, c.ph)) return false;
  c.new_layer = c.ph == PH_QKV;
  PhaseGeo g;
  phase_geo(P, c.layer, c.ph, G, g);
  c.W = g.W;
  c.s = g.s0;
  c.s1 = g.s1;
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
  const FLayer* L = lay(layer);
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
__device__ __forceinline__ void prefetch_slice(const void* base, unsigned int bytes, int G) {
  const unsigned int per = (((bytes + (unsigned)G - 1u) / (unsigned)G) + 15u) & ~15u;
  const unsigned int o = blockIdx.x * per;
  if (o < bytes) bulk_prefetch_l2((const unsigned char*)base + o, min(per, ((bytes - o) + 15u) & ~15u));
}
__device__ __noinline__ void prefetch_params(const FParams& P, int layer, int G) {
  const FLayer* L = lay(layer);
  if ((int)blockIdx.x == layer % G) {
    bulk_prefetch_l2(L->g1, (uint32_t)((P.d * 2 + 15) & ~15));
    bulk_prefetch_l2(L->g2, (uint32_t)((P.d * 2 + 15) & ~15));
    if (layer == 0) {
      bulk_prefetch_l2(P.rope_tab + (size_t)P.pos_host * (P.dh >> 1), (uint32_t)(((P.dh >> 1) * 8 + 15) & ~15));
      bulk_prefetch_l2(P.gf, (uint32_t)((P.d * 2 + 15) & ~15));
    }
  }
  if (L->accel && L->ad_bytes) prefetch_slice(L->ad_lo, L->ad_bytes, G);
  if (L->accel && L->AdT) { prefetch_slice(L->AdT, (unsigned)(P.F * P.r * 2), G); prefetch_slice(L->AoT, (unsigned)(P.da * P.r * 2), G); }
  if (layer == 0 && P.lmA && (P.head_stream == 1 || P.exit_heads)) {
    prefetch_slice(P.lmA, (unsigned)(P.r * P.d * 2), G);
    prefetch_slice(P.lmB, (unsigned)(P.V * P.r * 2), G);
  }
}

// auxiliary work of a weight phase: which adapter, if any
struct AuxGeo {
  const bf16 *A, *B;
  int nj, Kc;
  bool apply;       // split-K phase: the auxiliary warp adds B u into R.p itself
};
__device__ __forceinline__ bool aux_geo(const FParams& P, int layer, int ph, AuxGeo& a) {
  const int n = P.n_layers_run;
  const FLayer* L = lay(layer < n ? layer : (n > 0 ? n - 1 : 0));
  a.B = nullptr; a.apply = false; a.Kc = P.d;
  if (ph == PH_HEAD || ph == PH_EXIT) {
    a.A = P.lmA; a.nj = P.r;
    return P.lmA != nullptr && P.r > 0 && (ph == PH_EXIT || P.head_stream == 1);
  }
  if (!L->accel || P.r <= 0) return false;
  if (ph == PH_QKV) { a.A = L->Aqkv; a.nj = 3 * P.r; }
  else if (ph == PH_OPROJ) { a.A = L->Ao; a.B = L->Bo; a.nj = P.r; a.Kc = P.da; a.apply = true; }
  else if (ph == PH_GATEUP) { a.A = L->Agu; a.nj = 2 * P.r; }
  else { a.A = L->Ad; a.B = L->Bd; a.nj = P.r; a.Kc = P.F; a.apply = true; }
  return true;
}

__global__ void __launch_bounds__(NTHREADS, 1) m2r2_fused_decode_kernel(const __grid_constant__ FParams P) {
  unsigned char* const ring = smem_raw;
  bf16* const x = (bf16*)(smem_raw + OFF_X);
  float* const red = (float*)(smem_raw + OFF_RED);
  float* const tile_out = (float*)(smem_raw + OFF_TILE);
  float* const u_s = (float*)(smem_raw + OFF_U);
  float* const sred = (float*)(smem_raw + OFF_SRED);
  u64* const full = (u64*)(smem_raw + OFF_BAR);
  u64* const empty = full + NSTAGE;
  u64* const abar = full + 2 * NSTAGE;   // attention K/V staging
  float* const utmp = (float*)(smem_raw + OFF_UTMP);
  int* const frt = (int*)(smem_raw + OFF_FRT);
  const int tid = threadIdx.x, G = gridDim.x;
  if (tid == 0) {
    for (int i = 0; i < NSTAGE; ++i) { mbar_init(&full[i], 1); mbar_init(&empty[i], NCW); }
    mbar_init(abar, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    *(int*)(smem_raw + OFF_TLN) = 0;
    *(unsigned int*)(smem_raw + OFF_PCTR) = 0u;
  }
  if (tid < N_PH) geo_init(P, tid, G);
  for (int i = tid; i < P.n_heads; i += NTHREADS) ((int*)(smem_raw + OFF_SIDX))[i] = P.sidx[i];
  {
    const int words = P.n_layers_run * (int)(sizeof(FLayer) / 4);
    const uint32_t* src = (const uint32_t*)P.layers;
    uint32_t* dst = (uint32_t*)(smem_raw + OFF_LAYERS);
    for (int i = tid; i < words; i += NTHREADS) dst[i] = __ldg(src + i);
  }
  __syncthreads();
  const int n_run = P.n_layers_run;

  if (tid >= NCT + 64) {
    // ================= L2 prefetch warp: walks the CTA's stage sequence a window ahead of the producer and touches
    // every 128-byte line with prefetch.global.L2 (requests without return data through the LSU, not the bulk
    // copy unit), so HBM keeps streaming into L2 while the ring is full and the consumers sit in a gap
    const int W = P.pf_ahead, lane = tid & 31;
    if (W <= 0) return;
    volatile unsigned int* pctr = (volatile unsigned int*)(smem_raw + OFF_PCTR);
    Cursor pf;
    pf.layer = 0; pf.ph = -1; pf.s = pf.s1 = 0; pf.W = nullptr; pf.new_layer = false;
    const unsigned char* a;
    unsigned int n = 0;
    while (cursor_get(P, pf, G, a)) {
      unsigned int spins = 0;
      while ((int)(n - *pctr) >= W) {
        __nanosleep(100);
        if ((++spins & 1023u) == 0u && aborted(P.ctl)) break;
      }
      if ((int)(n - *pctr) >= 0) {   // still ahead of the producer: worth fetching
#pragma unroll
        for (int i = 0; i < STAGE_BYTES / 128 / 32; ++i)
          asm volatile("prefetch.global.L2 [%0];" ::"l"(a + (size_t)(lane + 32 * i) * 128));
      }
      ++n;
    }
    return;
  }
  if (tid >= NCT + 32) {
    // ================= auxiliary warp: adapter down-projections (u = A x^) of every phase that has one
    UState us;
    us.epoch = P.bar_base; us.nj = 0; us.q = 1;
    int layer = 0, ph = -1;
    while (next_weight_phase(P, layer, ph)) {
      AuxGeo a;
      if (!aux_geo(P, layer, ph, a)) continue;
      ++us.epoch;
      if (a.apply) {
        BPre bp;
        apply_prefetch(P, bp, a.B, G);   // B never depends on activations
        bar_wait(2);   // the grid barrier before this phase has passed: the producing phase's partials are visible
        combine_u(P, u_s, ph, G);
        apply_Bu(P, bp, a.B, u_s, G);
        __threadfence();
      } else {
        APre ap;
        u_geometry(us, a.nj, G);
        publish_prefetch(us, ap, a.A, a.Kc);   // A never depends on activations
        bar_wait(2);   // x^ of the phase is in shared memory
        publish_u(P, x, us, ap, a.A, a.Kc);
        fetch_u(P, u_s, utmp, us);
      }
      __threadfence_block();
      bar_arrive(3);
    }
    return;
  }
  if (tid >= NCT) {
    // ================= producer warp: one thread streams every weight stage of the pass
    if (tid == NCT) {
      const u64 pol = policy_evict_first();
      Cursor ld;
      ld.layer = 0; ld.ph = -1; ld.s = ld.s1 = 0; ld.W = nullptr; ld.new_layer = false;
      const unsigned char* a;
      unsigned int ctr = 0;
      while (cursor_get(P, ld, G, a)) {
        if (ld.new_layer) {
          ld.new_layer = false;
          prefetch_kv(P, ld.layer, G);
          prefetch_params(P, ld.layer, G);
        }
        const unsigned int slot = ctr % NSTAGE, use = ctr / NSTAGE;
        ++ctr;
        *(volatile unsigned int*)(smem_raw + OFF_PCTR) = ctr;
        mbar_wait(&empty[slot], (use & 1u) ^ 1u, P.ctl, 0x400u + ld.ph);
        mbar_expect_tx(&full[slot], STAGE_BYTES);
        bulk_g2s(ring + (size_t)slot * STAGE_BYTES, a, STAGE_BYTES, &full[slot], pol);
      }
    }
    return;
  }

  // ================= consumers: one loop over the phases of the pass
  const int lane = tid & 31, warp = tid >> 5, g = lane >> 2, t = lane & 3;
  unsigned int nbar = 0, stage_ctr = 0, aphase = 0;
  const int d = P.d;
  const int pos = *(volatile int*)P.kv_len + P.joff;
  const int tok = *(volatile const int*)P.tok_in;
  TL(1);

  int layer = 0, ph = -1;
  while (next_weight_phase(P, layer, ph)) {
    const FLayer* L = lay(layer < n_run ? layer : (n_run > 0 ? n_run - 1 : 0));
    const bool accel = ph == PH_HEAD || ph == PH_EXIT ? true : L->accel != 0;
    if (ph == PH_OPROJ) {
      // ---- a4: attention (its own phase between QKV and OPROJ; no weights)
      attn_phase(P, (unsigned char*)x, utmp, sred, abar, aphase, L, pos, accel, G);
      TL(13);
      grid_sync(P.ctl, P.bar_base, nbar, G);
      TL(14);
    }
    PhaseGeo pg;
    phase_geo(P, layer, ph, G, pg);
    PhaseCtx pc;
    pc.ph = ph; pc.layer = layer; pc.L = L; pc.pos = pos; pc.accel = accel;
    if (ph == PH_EXIT) pc.layer = L->gate - 1;
    if (ph == PH_HEAD) pc.layer = n_run;
    AuxGeo ag;
    const bool need_aux = aux_geo(P, layer, ph, ag);
    float udacc[MAX_R];
#pragma unroll
    for (int j = 0; j < MAX_R; ++j) udacc[j] = 0.f;
    // ---- loader: the phase's input vector(s) -> shared memory
    if (pg.split) {
      if (need_aux) bar_arrive(2);   // the auxiliary warp reads global partials only: it may start now
      const int len = pg.s1 - pg.s0;
      if (len > 0) loader_slice(P, x, ph, accel, pg.s0 % pg.nkc, min(len, pg.nkc), pg.nkc);
    } else {
      LoadSrc src;
      int mode;
      float* tr = nullptr;
      const bf16* gn;
      src.emb = nullptr; src.gate = 0; src.p_live = true;
      if (ph == PH_GATEUP) {
        src.p_live = accel;
        mode = LN_GU; gn = L->g2;
      } else if ((ph == PH_QKV && layer == 0) || (ph == PH_HEAD && n_run == 0)) {
        // a1: embedding, p_0 <- h_0 (L82)
        src.emb = P.embed + (size_t)tok * d; src.p_live = false;
        mode = ph == PH_QKV ? LN_QKV : (P.head_stream == 0 ? LN_HEAD_H : LN_HEAD_P);
        gn = ph == PH_QKV ? L->g1 : P.gf;
        tr = P.do_trace ? P.trace : nullptr;
      } else {
        // a7-tail: R already holds the accelerated-residual update of the layer below (Eq. 2); gate
        const FLayer* Lp = ph == PH_QKV ? L - 1 : L;
        src.p_live = Lp->accel != 0;
        if (ph == PH_QKV) {
          src.gate = Lp->accel ? Lp->gate : 0;
          mode = LN_QKV; gn = L->g1;
          tr = P.do_trace ? P.trace + (size_t)layer * 2 * d : nullptr;
        } else if (ph == PH_EXIT) {
          mode = LN_HEAD_P; gn = P.gf;
        } else {
          mode = P.head_stream == 0 ? LN_HEAD_H : LN_HEAD_P; gn = P.gf;
          tr = P.do_trace ? P.trace + (size_t)n_run * 2 * d : nullptr;
        }
      }
      loader_norm(P, x, sred, mode, src, tr, gn, G);
    }
    if (need_aux && !pg.split) { __threadfence_block(); bar_arrive(2); }
    TL(10 + ph);
    if (pg.split) {
      // ---- split-K GEMV: stage (grp, kc) = row-tiles 8 grp .. 8 grp + 7 x inputs [128 kc, +128); warp w owns
      // row-tile w, accumulates over the k-chunks of a group, then adds its 16 x 2 sums into R.
      float ca[4] = {0.f, 0.f, 0.f, 0.f}, cb[4] = {0.f, 0.f, 0.f, 0.f};
      int grp = pg.s0 / pg.nkc, kc = pg.s0 - grp * pg.nkc;
      for (int s = pg.s0; s < pg.s1; ++s) {
        const unsigned int slot = stage_ctr % NSTAGE, use = stage_ctr / NSTAGE;
        ++stage_ctr;
        uint4 b0 = make_uint4(0u, 0u, 0u, 0u), b1 = b0, b2 = b0, b3 = b0;
        if (g < 4) {
          const uint4* xb = (const uint4*)(x + (size_t)g * XCOL + t * 16 + (kc % XSLOTS) * SK_K);
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
        if (lane == 0) release_stage(&empty[slot], P.zero, ca[0] + cb[0]);   // stage consumed by this warp
        if (kc == pg.nkc - 1 || s == pg.s1 - 1) {
          // columns 0,1 = h (hi, lo parts), 2,3 = p: lanes t = 0 / 1 hold the h / p sums of rows g, g + 8
          if (t < 2 && (t == 0 || accel)) {
            const int r0 = (grp * SK_RT + warp) * 16 + g;
            if (r0 < d) red_add(P.R + (size_t)t * d + r0, (ca[0] + ca[1]) + (cb[0] + cb[1]));
            if (r0 + 8 < d) red_add(P.R + (size_t)t * d + r0 + 8, (ca[2] + ca[3]) + (cb[2] + cb[3]));
          }
#pragma unroll
          for (int i = 0; i < 4; ++i) ca[i] = cb[i] = 0.f;
        }
        if (++kc == pg.nkc) { kc = 0; ++grp; }
      }
      TL(43);
      if (need_aux) bar_wait(3);   // the auxiliary warp's adds of B u are issued and fenced
    } else {
      // ---- row-owned GEMV: stage (rt, ks) = 64 tiles of row-tile rt, inputs [1024 ks, +1024).  Warp w
      // multiplies tiles 8w..8w+7.  A finished row-tile leaves 8 x 32 partial sums in shared memory; every
      // FB finished row-tiles (and at the end) the 8 warps finish one row-tile each.
      const int nks = pg.nkc;
      float ca[4] = {0.f, 0.f, 0.f, 0.f}, cb[4] = {0.f, 0.f, 0.f, 0.f};
      const bf16* xcol = x + (size_t)(g & 3) * XCOL + t * 16 + warp * 128;
      int rt = pg.s0 / nks, ks = 0, pending_tiles = 0;
      bool u_ready = !need_aux;
      for (int s = pg.s0; s < pg.s1; ++s) {
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
        if (lane == 0) release_stage(&empty[slot], P.zero, ca[0] + cb[0]);   // stage consumed by this warp
        if (++ks == nks) {
          // ---- row-tile rt finished in this warp's k range: park the partial sums
          float* rw = red + ((size_t)pending_tiles * NCW + warp) * 32;
          if (t < 2) {
            rw[g * 2 + t] = (ca[0] + ca[1]) + (cb[0] + cb[1]);
            rw[(g + 8) * 2 + t] = (ca[2] + ca[3]) + (cb[2] + cb[3]);
          }
          if (tid == 0) frt[pending_tiles] = rt;
#pragma unroll
          for (int i = 0; i < 4; ++i) ca[i] = cb[i] = 0.f;
          ks = 0; ++rt; ++pending_tiles;
        }
        if (pending_tiles == FB || (s == pg.s1 - 1 && pending_tiles > 0)) {
          TL(41);
          if (!u_ready) { bar_wait(3); u_ready = true; }   // u of this phase is in shared memory
          bar_consumers();
          TL(42);
          if (warp < pending_tiles) {
            const float* rb = red + ((size_t)warp * NCW) * 32 + lane;
            float sum = 0.f;
#pragma unroll
            for (int w = 0; w < NCW; ++w) sum += rb[w * 32];
            float* T = tile_out + warp * 32;
            T[lane] = sum;
            __syncwarp();
            epilogue_tile(P, T, u_s, pc, frt[warp], udacc);
          }
          TL(44);
          pending_tiles = 0;
          if (s != pg.s1 - 1) bar_consumers();   // the parked sums are consumed before the next row-tile parks
          TL(40);
        }
      }
      if (!u_ready) bar_wait(3);   // a CTA without stages in this phase still completes the handshake
      if (ph == PH_GATEUP && accel && P.r > 0) {
        // this CTA's share of u = A_d a^ (every CTA writes, also one without row-tiles: the sum runs over all)
        float* ud_s = (float*)(smem_raw + OFF_UD);
        if (lane == 1) {
#pragma unroll
          for (int j = 0; j < MAX_R; ++j) ud_s[warp * MAX_R + j] = udacc[j];
        }
        bar_consumers();
        if (warp == 0 && lane < P.r) {
          float sum = 0.f;
#pragma unroll
          for (int w = 0; w < NCW; ++w) sum += ud_s[w * MAX_R + lane];
          __stcg(P.udpart + (size_t)blockIdx.x * RV_STRIDE + lane, sum);
        }
      }
    }
    TL(20 + ph);
    grid_sync(P.ctl, P.bar_base, nbar, G);
    TL(30 + ph);
  }
  TL(50);
  // A timed-out wait leaves the pass unsynchronised: nothing it computed may become sequence state.
  // The host sees the abort through ctl->host_abort at its next call and re-arms the control block.
  if (blockIdx.x == 0 && tid == 0 && !aborted(P.ctl)) {
    u64 key = *(volatile u64*)&P.ctl->amax[0];
    int tk = (int)(0xFFFFFFFFu - (unsigned int)(key & 0xFFFFFFFFull));
    *P.tok_out = tk;
    P.ctl->amax[0] = 0ull;
    for (int j = 0; j < P.n_gates; ++j) {
      u64 kj = *(volatile u64*)&P.ctl->amax[1 + j];
      if (kj) P.exit_tok[j] = (int)(0xFFFFFFFFu - (unsigned int)(kj & 0xFFFFFFFFull));
      P.ctl->amax[1 + j] = 0ull;
    }
    if (P.advance) { *P.kv_len = pos + 1; *P.pending = tk; }
  }
}

// ------------------------------------------------------------------ repack: row-major [n_out, K] -> fragment-major stages
// map 0: natural rows; 1: QKV (RoPE pairs (j, j+dh/2) of q and k made adjacent); 2: gate/up interleaved
// (16-row tile = gate n..n+7, up n..n+7): row-owned stages (row-tile, k-stage) of 1 x 1024.
// map 3: split-K stages (row-tile group, k-chunk) of 8 row-tiles x 128 inputs, natural rows.
// Rows / columns beyond the matrix are zero.
__device__ __forceinline__ const bf16* pack_src_row(const bf16* src, const bf16* src2, int map, int r, int n_out, int K, int d, int dh) {
  if (map == 0 || map == 3) return r < n_out ? src + (size_t)r * K : nullptr;
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
__global__ void transpose_kernel(bf16* __restrict__ dst, const bf16* __restrict__ src, int rows, int cols) {
  // src [rows][cols] -> dst [cols][rows]
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < (size_t)rows * cols; i += (size_t)gridDim.x * blockDim.x) {
    const int c = (int)(i / rows), r = (int)(i % rows);
    dst[i] = src[(size_t)r * cols + c];
  }
}
__global__ void pack_kernel(uint4* __restrict__ dst, const bf16* __restrict__ src, const bf16* __restrict__ src2,
                            int map, int n_out, int K, int n_units, int nks, int d, int dh) {
  const size_t total = (size_t)n_units * nks * (STAGE_BYTES / 16);
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < total; i += (size_t)gridDim.x * blockDim.x) {
    const size_t stage = i / (STAGE_BYTES / 16);
    const int within = (int)(i % (STAGE_BYTES / 16));
    const int tile = within >> 5, lane = within & 31, g = lane >> 2, t = lane & 3;
    const int un = (int)(stage / nks), ks = (int)(stage % nks);
    int rt, k;
    if (map == 3) { rt = un * SK_RT + (tile >> 3); k = ks * SK_K + (tile & 7) * 16 + 2 * t; }
    else { rt = un; k = ks * STAGE_K + tile * 16 + 2 * t; }
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

// ------------------------------------------------------------------ skinny GEMM on the fragment-major weights (a11, a18, batched a10)
// The k-token verify pass, prefill chunks and batched draft passes multiply each weight matrix with 1..64 activation
// rows.  Same fragment-major tiles as the fused kernel, weights as the M operand and the rows as N of mma.sync.m16n8k16:
// one LDG.128 per lane per tile straight into the A fragment, the rows' bf16 hi + lo parts as two B operands (fp32-class
// products, as in the fused kernel), fp32 accumulation on the tensor pipe.  HBM-bound: 2 m flop per byte.
enum { VK_QKV = 0, VK_OPROJ = 1, VK_GATEUP = 2, VK_DOWN = 3, VK_HEAD = 4 };
struct VArgs {
  const uint4* W;
  const float* X;        // [rows][ldx] fp32
  float* out;            // [rows][ldo]
  const float* resid;    // O / DOWN: out = resid + W x
  float* trace;          // DOWN: second copy of out, or nullptr
  int ldx, ldo, rows, K, n_out, nkt, nstage_k, split, d, dh;
  int ksplit;            // O / DOWN: CTAs per row tile along K; > 1 adds into out (= resid, in place) atomically
  int n_rt;              // row tiles of the matrix (rows_mma_kernel)
  // parallel adapters of the accelerated rows (rows_mma_kernel): rows >= lora_row0 get + B[bmap(n)] . U[row][usel * r ..)
  const bf16 *Bm, *Bm2;  // Bm2: the up projection's B (gate/up)
  const int* bmap;       // nullable -> identity; -1 = no adapter row for this output
  const float* U;
  int ldu, r, lora_row0, usel_div;
  const uint2* Xp;       // rows > 8: the rows as (bf16 hi pair, bf16 lo pair) words [NG * 8][Kp / 2], zero padded (pack_rows_kernel)
  int Kp;
  uint2* out_pk;         // gate/up, nullable: the activations also as (hi, lo) words [row][out_pk_ld] (down's packed input)
  int out_pk_ld;
  float* part;           // QKV / gate-up with ksplit > 1: partial sums [n_rt][NG][4][32], zero between launches
  // neighbours absorbed by rows_ring_kernel (RowsFuse)
  const bf16* gain;      // row-owned: X is the raw residual; RMSNorm(x; gain, eps) applied inside
  float eps;
  int n_heads;
  const float *part_o, *part_ml;   // O: X = the merge of the attention partials [rows][n_heads][n_splits] (<= 8 splits)
  int n_splits;
  const int *row_seq, *row_pos;    // QKV: RoPE on q, k and the K/V cache append in the epilogue
  const float2* rope_tab;
  bf16 *Kc, *Vc;
  int max_seq;
  int slow_rows;         // rows_mma_kernel with rope_tab: rows < slow_rows append k, v to the cache
  int tile_in_head;      // d % 16 == 0 && dh % 16 == 0 (QKV epilogue: index arithmetic once per tile)
};
__device__ __forceinline__ uint32_t pack_hi_lo(float a, float b, uint32_t& lo) {
  const __nv_bfloat162 h = __floats2bfloat162_rn(a, b);
  const float2 f = __bfloat1622float2(h);
  const __nv_bfloat162 l = __floats2bfloat162_rn(a - f.x, b - f.y);
  lo = bf2_u32(l);
  return bf2_u32(h);
}
// rows > 8: every CTA of the GEMM needs all rows of its k-chunks, and converting them to bf16 hi + lo in each CTA costs
// more instructions than the MMAs: convert ONCE, the GEMM's staging is then a plain 16-byte copy
__global__ void __launch_bounds__(256) pack_rows_kernel(const float* __restrict__ X, int ldx, int rows, int K, int rows_pad,
                                                        int Kp, uint2* __restrict__ Xp) {
  pdl_launch_dependents();
  pdl_wait();
  const int nq = Kp >> 2;
  for (int i = blockIdx.x * 256 + threadIdx.x; i < rows_pad * nq; i += gridDim.x * 256) {
    const int row = i / nq, q = i - row * nq, k = 4 * q;
    float4 v = make_float4(0.f, 0.f, 0.f, 0.f);
    if (row < rows && k < K) v = __ldcg((const float4*)(X + (size_t)row * ldx + k));
    uint4 w;
    w.x = pack_hi_lo(v.x, v.y, w.y);
    w.z = pack_hi_lo(v.z, v.w, w.w);
    *(uint4*)(Xp + (size_t)row * (Kp >> 1) + 2 * q) = w;
  }
}
// the epilogue of one 16-row weight tile, given the complete (or, for O / down under split-K, the CTA's partial) sums in
// the accumulator layout of mma.sync: c[gi][0], c[gi][1] = weight row g x activation rows 8 gi + 2t, + 1; c[gi][2],
// c[gi][3] = weight row g + 8.  first_k: this CTA adds the once-only terms (the accelerated rows' adapters).
template <int KIND, int NG>
__device__ __forceinline__ void rows_epilogue(const VArgs& a, int rt, float (&c)[NG][4], int lane, bool first_k, int n0 = 0) {
  const int g = lane >> 2, t = lane & 3;
  if (KIND == VK_QKV && a.tile_in_head) {
    // d % 16 == 0 and dh % 16 == 0: the tile's 16 packed rows lie in one head of q, k or v.  Packed rows 2i, 2i + 1 of a
    // q / k head are the elements i, i + dh / 2: the RoPE pair, the partner in lane ^ 4.  With rope_tab the epilogue also
    // rotates q, k (after the adapter term) and appends the slow rows' k, v to the cache (a3,
    // rope_append_kernel's arithmetic); accelerated rows keep k^, v^ in `out` only.
    const int base = rt * 16, which = base / a.d, w_ = base - which * a.d, head = w_ / a.dh, e0 = w_ - head * a.dh;
    const int half = a.dh >> 1;
#pragma unroll
    for (int gi = 0; gi < NG; ++gi) {
#pragma unroll
      for (int s = 0; s < 2; ++s) {
        const int n = n0 + gi * 8 + 2 * t + s;
        const bool live = n < a.rows;
        const bool lora = a.Bm != nullptr && live && n >= a.lora_row0 && first_k;
        int pos = 0;
        size_t cbase = 0;
        if (a.rope_tab && live) {
          pos = a.row_pos[n];
          cbase = (((size_t)a.row_seq[n] * a.n_heads + head) * a.max_seq + pos) * a.dh;
        }
#pragma unroll
        for (int hh = 0; hh < 2; ++hh) {
          const int e = e0 + g + 8 * hh, ne = which < 2 ? (e >> 1) + (e & 1) * half : e;
          const int nat = which * a.d + head * a.dh + ne;
          const bool inb = base + g + 8 * hh < a.n_out;
          float v = c[gi][2 * hh + s];
          if (lora && inb) {
            const int bn = a.bmap ? a.bmap[nat] : nat;
            if (bn >= 0) {
              const float* u = a.U + (size_t)n * a.ldu + (a.usel_div ? which : 0) * a.r;   // usel_div == d for QKV
              for (int q = 0; q < a.r; ++q) v += bf(a.Bm + (size_t)bn * a.r + q) * u[q];
            }
          }
          const float pv = __shfl_xor_sync(0xffffffffu, v, 4);
          if (!live || !inb) continue;
          if (a.rope_tab && which < 2) {
            const float2 cs = a.rope_tab[(size_t)pos * half + (e >> 1)];
            v = (e & 1) ? v * cs.x + pv * cs.y : v * cs.x - pv * cs.y;
          }
          a.out[(size_t)n * a.ldo + nat] = v;
          if (a.rope_tab && n < a.slow_rows) {
            if (which == 1) a.Kc[cbase + ne] = __float2bfloat16_rn(v);
            if (which == 2) a.Vc[cbase + e] = __float2bfloat16_rn(v);
          }
        }
      }
    }
    return;
  }
  // c[gi][0], c[gi][1] = weight row g x activation rows 8 gi + 2t, + 1; c[gi][2], c[gi][3] = weight row g + 8
#pragma unroll
  for (int gi = 0; gi < NG; ++gi) {
#pragma unroll
    for (int s = 0; s < 2; ++s) {
      const int n = n0 + gi * 8 + 2 * t + s;
      if (KIND == VK_GATEUP) {
        const int o = rt * 8 + g;
        const bool live = n < a.rows && o < a.n_out;
        float v0 = c[gi][s], v1 = c[gi][2 + s];
        if (live && a.Bm != nullptr && n >= a.lora_row0 && first_k) {   // + B (A x^) on accelerated rows
          const float* urow = a.U + (size_t)n * a.ldu;
          for (int q = 0; q < a.r; ++q) {
            v0 += bf(a.Bm + (size_t)o * a.r + q) * urow[q];
            v1 += bf(a.Bm2 + (size_t)o * a.r + q) * urow[a.r + q];
          }
        }
        const float act = live ? silu(v0) * v1 : 0.f;
        if (live) a.out[(size_t)n * a.ldo + o] = act;
        if (a.out_pk) {   // outputs o, o + 1 sit in lanes g, g + 1 (lane ^ 4): the even one writes the pair
          const float nb = __shfl_xor_sync(0xffffffffu, act, 4);
          if (!(g & 1) && n < a.rows && o < a.n_out) {
            const __nv_bfloat162 h = __floats2bfloat162_rn(act, nb);
            const float2 f = __bfloat1622float2(h);
            const __nv_bfloat162 l = __floats2bfloat162_rn(act - f.x, nb - f.y);
            a.out_pk[(size_t)n * a.out_pk_ld + (o >> 1)] = make_uint2(bf2_u32(h), bf2_u32(l));
          }
        }
        continue;
      }
      if (n >= a.rows) continue;
      float v0 = c[gi][s], v1 = c[gi][2 + s];
      const bool lora = a.Bm != nullptr && n >= a.lora_row0 && first_k;   // + B (A x^) on accelerated rows
      const float* urow = a.U + (size_t)n * a.ldu;
#pragma unroll
      for (int hh = 0; hh < 2; ++hh) {
        const int pr = rt * 16 + g + 8 * hh;
        float v = hh ? v1 : v0;
        if (pr >= a.n_out) continue;
        int nat = pr;
        if (KIND == VK_QKV) {
          const int which = pr / a.d, w_ = pr % a.d, head = w_ / a.dh, e = w_ % a.dh;
          nat = which < 2 ? which * a.d + head * a.dh + (e >> 1) + (e & 1) * (a.dh >> 1) : pr;
        }
        if (lora) {
          const int bn = a.bmap ? a.bmap[nat] : nat;
          if (bn >= 0) {
            const float* u = urow + (a.usel_div ? nat / a.usel_div : 0) * a.r;
            for (int q = 0; q < a.r; ++q) v += bf(a.Bm + (size_t)bn * a.r + q) * u[q];
          }
        }
        if (KIND == VK_QKV || KIND == VK_HEAD) {
          a.out[(size_t)n * a.ldo + nat] = v;
        } else if (a.ksplit > 1) {
          atomicAdd(a.out + (size_t)n * a.ldo + pr, v);   // out == resid (in place)
        } else {
          const float o = a.resid[(size_t)n * a.ldo + pr] + v;
          a.out[(size_t)n * a.ldo + pr] = o;
          if (a.trace) a.trace[(size_t)n * a.ldo + pr] = o;
        }
      }
    }
  }
}
// second stage of a row-owned matrix that was split along K: one warp per (row tile, group of 8 activation rows) reads the
// summed partials (and leaves zeros behind for the next launch) and runs the epilogue.  (One warp per tile for all groups
// left 4 warps per SM with a chain of dependent loads each: 13 us for the 40-row QKV.)
template <int KIND, int NG>
__global__ void __launch_bounds__(128) rows_epilogue_kernel(const VArgs a) {
  pdl_launch_dependents();
  pdl_wait();
  const int lane = threadIdx.x & 31, rt = blockIdx.x * 4 + (threadIdx.x >> 5), gi = blockIdx.y;
  if (rt >= a.n_rt) return;
  float c[1][4];
  float* src = a.part + ((size_t)rt * NG + gi) * 4 * 32 + lane;
#pragma unroll
  for (int e = 0; e < 4; ++e) {
    c[0][e] = __ldcg(src + e * 32);
    src[e * 32] = 0.f;
  }
  rows_epilogue<KIND, 1>(a, rt, c, lane, true, gi * 8);
}
// A CTA = 4 warps = 4 consecutive 16-row tiles over a K range; the activation rows of a 256-input chunk are staged
// ONCE per CTA in shared memory as bf16 hi + lo parts and shared by the four row tiles, so every weight is read from HBM
// once for all rows and the replicated activation traffic from L2 stays near the weight traffic; each warp keeps the
// chunk's 16 weight tiles (8 KB) in flight while the rows are staged.  NG groups of 8 rows = NG n8 MMA tiles (x2: hi, lo)
// per weight tile.  Epilogues: QKV undoes the RoPE row permutation of the packed matrix, gate/up applies SwiGLU on the
// lane's (gate, up) pair, O / down add the residual (split along K: atomic adds onto the in-place residual), LM head
// writes logits; accelerated rows add their parallel adapter term B u.
constexpr int RM_KC = 256;               // inputs per staged chunk (16 k16 tiles)
#ifndef M2R2_RM_NW
#define M2R2_RM_NW 8
#endif
constexpr int RM_NW = M2R2_RM_NW;        // warps = row tiles of a CTA with > 8 rows: they share one staged chunk of the rows
// SW (NG == 1): the CTA's four warps split the inputs of ONE row tile (a super-chunk of 4 x 256 inputs is staged, warp w
// takes its w-th quarter) and their sums meet in shared memory: four times the CTAs for matrices with few row tiles.
template <int KIND, int NG, bool SW>
__global__ void __launch_bounds__(SW ? 128 : RM_NW * 32) rows_mma_kernel(const VArgs a) {
  constexpr int NQ = SW ? 4 : 1;                   // 256-input chunks staged per iteration
  constexpr int LD = NQ * RM_KC + 8;               // bf16 elements per staged row (+8: bank spread)
  extern __shared__ __align__(16) unsigned char rm_smem[];
  bf16* xh = (bf16*)rm_smem;                       // [NG * 8][LD] hi parts
  bf16* xl = xh + (size_t)NG * 8 * LD;             // lo parts
  constexpr bool PK = !SW;                         // the rows arrive converted (a.Xp): staged by copy as (hi, lo) words
  constexpr int LD2 = RM_KC / 2 + 4;               // words per staged row; = 4 mod 16: a half-warp's LDS.64 hit 16 bank pairs
  uint2* xs = (uint2*)rm_smem;                     // [NG * 8][LD2]
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, g = lane >> 2, t = lane & 3;
  const int rt = SW ? blockIdx.x : blockIdx.x * RM_NW + warp;
  const bool mine = rt < a.n_rt;
  float c[NG][4];
#pragma unroll
  for (int i = 0; i < NG; ++i)
#pragma unroll
    for (int e = 0; e < 4; ++e) c[i][e] = 0.f;
  const int nch = (a.nkt + 16 * NQ - 1) / (16 * NQ);   // (super-)chunks of the whole K
  const int ch_lo = (int)(((long long)nch * blockIdx.y) / a.ksplit), ch_hi = (int)(((long long)nch * (blockIdx.y + 1)) / a.ksplit);
  const int wq = SW ? warp : 0;                    // the warp's quarter of the staged inputs
  pdl_launch_dependents();                         // the next kernel of the chain may begin to launch
  for (int ch = ch_lo; ch < ch_hi; ++ch) {
    const int kbase = ch * NQ * RM_KC;
    // the warp's 16 weight tiles of this iteration: 16 LDG.128 per lane in flight while the activations are staged
    // (requesting the next iteration's tiles before the MMAs as well costs 60 registers and an SM's third CTA: slower)
    uint4 w[16];
#pragma unroll
    for (int u = 0; u < 16; ++u) {
      const int kt = (ch * NQ + wq) * 16 + u;
      w[u] = make_uint4(0u, 0u, 0u, 0u);
      if (mine && kt < a.nkt) {
        const size_t tile = a.split ? ((size_t)((rt >> 3) * a.nstage_k + (kt >> 3)) * 64 + (rt & 7) * 8 + (kt & 7))
                                    : ((size_t)(rt * a.nstage_k + (kt >> 6)) * 64 + (kt & 63));
        w[u] = ldg_stream(a.W + tile * 32 + lane);
      }
    }
    // weights never depend on the previous kernel: under programmatic dependent launch the first iteration's tiles are
    // already in flight while the producer of the activation rows finishes
    if (ch == ch_lo) pdl_wait();
    __syncthreads();   // the previous iteration's staged rows are consumed
    if (PK) {
      for (int i = tid; i < NG * 8 * (RM_KC / 4); i += RM_NW * 32) {
        const int row = i >> 6, q = i & 63;   // RM_KC / 4 == 64 copies of 16 bytes per row
        cp_async16(xs + (size_t)row * LD2 + 2 * q, a.Xp + (size_t)row * (a.Kp >> 1) + (kbase >> 1) + 2 * q);
      }
      cp_async_wait_all();
    } else
    for (int i = tid; i < NG * 8 * (NQ * RM_KC / 4); i += 128) {
      const int row = i / (NQ * RM_KC / 4), q = i - row * (NQ * RM_KC / 4), k = kbase + 4 * q;
      float4 v = make_float4(0.f, 0.f, 0.f, 0.f);
      if (row < a.rows && k < a.K) v = __ldg((const float4*)(a.X + (size_t)row * a.ldx + k));   // K % 4 == 0
      uint32_t l0, l1;
      const uint32_t h0 = pack_hi_lo(v.x, v.y, l0), h1 = pack_hi_lo(v.z, v.w, l1);
      *(uint2*)(xh + (size_t)row * LD + 4 * q) = make_uint2(h0, h1);
      *(uint2*)(xl + (size_t)row * LD + 4 * q) = make_uint2(l0, l1);
    }
    __syncthreads();
    if (PK) {
#pragma unroll
      for (int u = 0; u < 16; ++u) {
#pragma unroll
        for (int gi = 0; gi < NG; ++gi) {
          const uint2* bp = xs + (size_t)(gi * 8 + g) * LD2 + u * 8 + t;   // inputs 16u + 2t (+1) and + 8: (hi, lo)
          const uint2 b0 = bp[0], b1 = bp[4];
          mma_bf16(c[gi], w[u], b0.x, b1.x);
          mma_bf16(c[gi], w[u], b0.y, b1.y);
        }
      }
    } else
#pragma unroll
    for (int u = 0; u < 16; ++u) {
#pragma unroll
      for (int gi = 0; gi < NG; ++gi) {
        const bf16* ph = xh + (size_t)(gi * 8 + g) * LD + wq * RM_KC + u * 16 + 2 * t;
        const bf16* pl = xl + (size_t)(gi * 8 + g) * LD + wq * RM_KC + u * 16 + 2 * t;
        mma_bf16(c[gi], w[u], *(const uint32_t*)ph, *(const uint32_t*)(ph + 8));
        mma_bf16(c[gi], w[u], *(const uint32_t*)pl, *(const uint32_t*)(pl + 8));
      }
    }
  }
  if (ch_lo >= ch_hi) pdl_wait();                  // (a CTA without chunks still orders its epilogue behind the predecessor)
  if (SW) {
    // the four warps' partial sums of the row tile -> warp 0
    __syncthreads();
    float* red = (float*)rm_smem;                  // [3][NG * 4][32]
    if (warp > 0) {
#pragma unroll
      for (int gi = 0; gi < NG; ++gi)
#pragma unroll
        for (int e = 0; e < 4; ++e) red[((warp - 1) * NG * 4 + gi * 4 + e) * 32 + lane] = c[gi][e];
    }
    __syncthreads();
    if (warp > 0) return;
#pragma unroll
    for (int ww = 0; ww < 3; ++ww)
#pragma unroll
      for (int gi = 0; gi < NG; ++gi)
#pragma unroll
        for (int e = 0; e < 4; ++e) c[gi][e] += red[(ww * NG * 4 + gi * 4 + e) * 32 + lane];
  }
  if (!mine) return;
  if ((KIND == VK_QKV || KIND == VK_GATEUP) && a.ksplit > 1) {
    // row-owned matrix split along K (many rows): the partial sums meet in a[part] in the accumulator layout;
    // rows_epilogue_kernel finishes the tile
    float* dst = a.part + (size_t)rt * NG * 4 * 32 + lane;
#pragma unroll
    for (int gi = 0; gi < NG; ++gi)
#pragma unroll
      for (int e = 0; e < 4; ++e) atomicAdd(dst + (gi * 4 + e) * 32, c[gi][e]);
    return;
  }
  rows_epilogue<KIND, NG>(a, rt, c, lane, blockIdx.y == 0);
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
  unsigned int* h_abort = nullptr;   // host-mapped: set by the kernel when a wait times out
  unsigned int* d_abort = nullptr;   // its device address
  bool bound = false;
  u64* d_tl = nullptr;        // debug timeline (M2R2_FUSED_DEBUG builds)
  std::vector<FLayer> h_layers;   // host copy of the layer descriptors (packed weight pointers)
  const uint4* h_Wlm = nullptr;
  std::vector<int> gate_of;   // per layer: 1 + gate index, or 0
  std::vector<int> accel_of;
  // scratch carve
  float *R, *act, *qbuf, *khat, *vhat, *apart, *apu, *udpart;
  u64* upart;
  int* accel_cols;
  uint2 *xn_pack, *act_pack;  // the same, written by their producers: norm_lora_kernel (QKV / gate-up input), the gate/up epilogue (down input)
  int xn_pack_ld = 0, act_pack_ld = 0;   // words per row; the columns beyond d / d_ff stay zero from fused_bind
  uint2* xpack;               // rows_mma_kernel with > 8 rows: the rows as (hi, lo) words (pack_rows_kernel)
  size_t xpack_n = 0;
  float* rows_part;           // rows_mma_kernel: partial sums of a row-owned matrix split along K (zero between launches)
  size_t rows_part_n = 0;
};

static int pad_to(int v, int m) { return (v + m - 1) / m * m; }

constexpr int RM_KC_HOST = 256;   // = RM_KC (rows_mma_kernel's staged chunk)
struct PackedDims {
  int d_pad, F_pad, rt_qkv, rt_gu, rt_v, ng_d, nkc_o, nkc_d;
  size_t st_qkv, st_o, st_gu, st_d, st_v;   // stages
};
static PackedDims packed_dims(const m2r2_config& c) {
  PackedDims q;
  q.d_pad = pad_to(c.d_model, STAGE_K);
  q.F_pad = pad_to(c.d_ff, SK_K);
  q.rt_qkv = pad_to(3 * c.d_model, 16) / 16;
  q.rt_gu = pad_to(c.d_ff, 8) / 8;
  q.rt_v = pad_to(c.vocab, 16) / 16;
  q.ng_d = pad_to(c.d_model, 16 * SK_RT) / (16 * SK_RT);
  q.nkc_o = pad_to(c.d_model, SK_K) / SK_K;
  q.nkc_d = q.F_pad / SK_K;
  q.st_qkv = (size_t)q.rt_qkv * (q.d_pad / STAGE_K);
  q.st_o = (size_t)q.ng_d * q.nkc_o;
  q.st_gu = (size_t)q.rt_gu * (q.d_pad / STAGE_K);
  q.st_d = (size_t)q.ng_d * q.nkc_d;
  q.st_v = (size_t)q.rt_v * (q.d_pad / STAGE_K);
  return q;
}

bool fused_config_ok(const m2r2_config& c) {
  if (c.dtype != M2R2_BF16 || c.n_experts != 0 || c.n_layers > MAXL_S) return false;
  if (c.head_dim % 8 || c.head_dim > 128) return false;
  if (c.d_model % 16 || c.d_ff % 8) return false;
  if (c.accel_enabled && (c.adapter_rank > MAX_R || c.adapter_rank < 1)) return false;
  if (pad_to(c.d_model, STAGE_K) > XMAX || c.d_ff > KMAX) return false;
  if ((size_t)2 * NCW * 2 * (c.head_dim + 2) * sizeof(float) > (size_t)KV_BYTES) return false;
  // a CTA's split-K stage range of the down matrix must fit the x slots (worst case: 100 CTAs)
  PackedDims q = packed_dims(c);
  if (q.nkc_d > XSLOTS && (q.st_d + 99) / 100 + 1 > (size_t)XSLOTS) return false;
  return true;
}

size_t fused_weights_bytes(const m2r2_config& c) {
  if (!fused_config_ok(c)) return 0;
  PackedDims q = packed_dims(c);
  const size_t adt = c.accel_enabled ? (((size_t)c.d_ff * c.adapter_rank * 2 + 255) & ~(size_t)255) + (((size_t)c.n_accel_heads * c.head_dim * c.adapter_rank * 2 + 255) & ~(size_t)255) : 0;
  return ((q.st_qkv + q.st_o + q.st_gu + q.st_d) * (size_t)c.n_layers + q.st_v) * STAGE_BYTES + adt * c.n_layers + 1024;
}

void fused_carve(const m2r2_config& c, Carver& cv, FusedState* fs) {
  if (!fused_config_ok(c)) return;
  PackedDims q = packed_dims(c);
  const size_t d = c.d_model;
  FusedImpl* im = fs ? fs->impl : nullptr;
#define FTAKE(field, T, n) { T* p_ = cv.take<T>(n); if (im) im->field = p_; }
  FTAKE(d_layers, FLayer, c.n_layers)
  FTAKE(d_ctl, Ctl, 1)
  FTAKE(d_sidx, int, c.n_heads)
  FTAKE(accel_cols, int, std::max(8, c.n_accel_heads * c.head_dim))
  FTAKE(R, float, 2 * d)
  FTAKE(act, float, 2 * (size_t)q.F_pad)
  FTAKE(qbuf, float, 2 * d) FTAKE(khat, float, d) FTAKE(vhat, float, d)
  FTAKE(apart, float, (size_t)c.n_heads * M2R2_MAX_SPLITS * 2 * (c.head_dim + 4))
  FTAKE(upart, u64, (size_t)UPART_N * UPART_STRIDE)
  FTAKE(apu, float, (size_t)c.n_heads * M2R2_MAX_SPLITS * RV_STRIDE)
  FTAKE(udpart, float, (size_t)1024 * RV_STRIDE)
  {
    const size_t n = (size_t)std::max(q.rt_qkv, q.rt_gu) * 8 * 4 * 32;   // [row tiles][NG <= 8][4][32]
    FTAKE(rows_part, float, n)
    if (im) im->rows_part_n = n;
    const size_t np = (size_t)64 * ((size_t)std::max(q.d_pad, q.F_pad) + 256) / 2;   // 64 rows x K (padded to 256) / 2 words
    FTAKE(xpack, uint2, np)
    if (im) im->xpack_n = np;
    const int ldx_ = q.d_pad / 2, lda_ = (pad_to(q.F_pad, RM_KC_HOST)) / 2;
    FTAKE(xn_pack, uint2, (size_t)64 * ldx_)
    FTAKE(act_pack, uint2, (size_t)64 * lda_)
    if (im) { im->xn_pack_ld = ldx_; im->act_pack_ld = lda_; }
  }
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
  if (!coop || max_smem < SMEM_BYTES || sms < 100) return 0;   // per-operation kernels serve this device
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
  if (cudaHostAlloc((void**)&im->h_abort, 64, cudaHostAllocMapped) != cudaSuccess ||
      cudaHostGetDevicePointer((void**)&im->d_abort, im->h_abort, 0) != cudaSuccess) {
    cudaGetLastError();
    if (im->h_abort) cudaFreeHost(im->h_abort);
    cudaFreeHost(im->h_ctl);
    delete im;
    return M2R2_CUDA;
  }
  *im->h_abort = 0u;
  fs->impl = im;
  fs->supported = true;
  return 0;
}

void fused_destroy(FusedState* fs) {
  if (fs->impl) {
    if (fs->impl->h_ctl) cudaFreeHost(fs->impl->h_ctl);
    if (fs->impl->h_abort) cudaFreeHost(fs->impl->h_abort);
    delete fs->impl;
  }
  fs->impl = nullptr;
  fs->supported = false;
}

bool fused_supported(const m2r2_config&, const FusedState* fs) { return fs->supported && fs->impl && fs->impl->bound; }

static int pack(cudaStream_t st, void* dst, const void* src, const void* src2, int map, int n_out, int K, int n_units,
                int nks, int d, int dh) {
  pack_kernel<<<1184, 256, 0, st>>>((uint4*)dst, (const bf16*)src, (const bf16*)src2, map, n_out, K, n_units, nks, d, dh);
  return cudaGetLastError() == cudaSuccess ? 0 : M2R2_CUDA;
}

int fused_bind(const m2r2_config& c, FusedState* fs, cudaStream_t st, void* packed, const void* embed,
               const void* gf, const void* lm_head, const void* lm_A, const void* lm_B, const DevLayer* layers,
               void* kv, const float2* rope_tab) {
  if (!fs->supported) return 0;
  FusedImpl* im = fs->impl;
  PackedDims q = packed_dims(c);
  const int d = c.d_model, dh = c.head_dim, F = c.d_ff;
  const int ks_d = q.d_pad / STAGE_K;
  char* wp = (char*)packed;
  wp = (char*)(((uintptr_t)wp + 1023) & ~(uintptr_t)1023);
  std::vector<FLayer> hl(c.n_layers);
  im->gate_of.assign(c.n_layers, 0);
  im->accel_of.assign(c.n_layers, 0);
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
    if (pack(st, (void*)f.Wo, L.wo, nullptr, 3, d, d, q.ng_d, q.nkc_o, d, dh)) return M2R2_CUDA;
    if (pack(st, (void*)f.Wgu, L.wgate, L.wup, 2, F, d, q.rt_gu, ks_d, d, dh)) return M2R2_CUDA;
    if (pack(st, (void*)f.Wd, L.wdown, nullptr, 3, d, F, q.ng_d, q.nkc_d, d, dh)) return M2R2_CUDA;
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
    im->gate_of[i] = f.gate;
    im->accel_of[i] = f.accel;
  }
  const uint4* Wlm = (const uint4*)wp;
  if (pack(st, (void*)Wlm, lm_head, nullptr, 0, c.vocab, d, q.rt_v, ks_d, d, dh)) return M2R2_CUDA;
  wp += q.st_v * STAGE_BYTES;
  if (c.accel_enabled) {
    const size_t adt = ((size_t)F * c.adapter_rank * 2 + 255) & ~(size_t)255;
    for (int i = 0; i < c.n_layers; ++i) {
      if (!hl[i].accel || !layers[i].Ad) continue;
      transpose_kernel<<<64, 256, 0, st>>>((bf16*)wp, (const bf16*)layers[i].Ad, c.adapter_rank, F);
      hl[i].AdT = (const bf16*)wp;
      wp += adt;
      transpose_kernel<<<16, 256, 0, st>>>((bf16*)wp, (const bf16*)layers[i].Ao, c.adapter_rank, c.n_accel_heads * dh);
      hl[i].AoT = (const bf16*)wp;
      wp += ((size_t)c.n_accel_heads * dh * c.adapter_rank * 2 + 255) & ~(size_t)255;
    }
    if (cudaGetLastError() != cudaSuccess) return M2R2_CUDA;
  }
  if (cudaMemcpyAsync(im->d_layers, hl.data(), sizeof(FLayer) * c.n_layers, cudaMemcpyHostToDevice, st) != cudaSuccess) return M2R2_CUDA;
  im->h_layers = hl;
  im->h_Wlm = Wlm;
  std::vector<int> sidx(c.n_heads, -1), cols(std::max(8, c.n_accel_heads * dh), 0);
  if (c.accel_enabled)
    for (int s = 0; s < c.n_accel_heads; ++s) {
      sidx[c.accel_heads[s]] = s;
      for (int j = 0; j < dh; ++j) cols[s * dh + j] = c.accel_heads[s] * dh + j;
    }
  if (cudaMemcpyAsync(im->d_sidx, sidx.data(), sizeof(int) * c.n_heads, cudaMemcpyHostToDevice, st) != cudaSuccess) return M2R2_CUDA;
  if (cudaMemcpyAsync(im->accel_cols, cols.data(), sizeof(int) * cols.size(), cudaMemcpyHostToDevice, st) != cudaSuccess) return M2R2_CUDA;
  {
    Ctl z;
    memset(&z, 0, sizeof(z));
    z.host_abort = im->d_abort;
    *im->h_ctl = z;
    cudaMemcpyAsync(im->d_ctl, im->h_ctl, sizeof(Ctl), cudaMemcpyHostToDevice, st);
  }
  cudaMemsetAsync(im->act, 0, sizeof(float) * 2 * q.F_pad, st);
  cudaMemsetAsync(im->R, 0, sizeof(float) * 2 * d, st);
  cudaMemsetAsync(im->udpart, 0, sizeof(float) * 1024 * RV_STRIDE, st);
  cudaMemsetAsync(im->rows_part, 0, sizeof(float) * im->rows_part_n, st);
  cudaMemsetAsync(im->xn_pack, 0, sizeof(uint2) * 64 * im->xn_pack_ld, st);
  cudaMemsetAsync(im->act_pack, 0, sizeof(uint2) * 64 * im->act_pack_ld, st);
  cudaMemsetAsync(im->upart, 0, sizeof(u64) * UPART_N * UPART_STRIDE, st);
  if (cudaStreamSynchronize(st) != cudaSuccess) return M2R2_CUDA;   // hl / sidx / cols are stack-owned
  im->bar_base = 0;
  FParams& p = im->p;
  memset(&p, 0, sizeof(p));
  p.d = d; p.n_heads = c.n_heads; p.dh = dh; p.F = F; p.V = c.vocab; p.r = c.accel_enabled ? c.adapter_rank : 0;
  p.da = c.n_accel_heads * dh; p.max_seq = c.max_seq;
  p.d_pad = q.d_pad; p.F_pad = q.F_pad;
  p.rt_qkv = q.rt_qkv; p.rt_gu = q.rt_gu; p.rt_v = q.rt_v; p.ng_d = q.ng_d;
  p.eps = c.rms_eps; p.scale = 1.0f / sqrtf((float)dh);
  p.layers = im->d_layers;
  p.embed = (const bf16*)embed; p.gf = (const bf16*)gf; p.lmA = (const bf16*)lm_A; p.lmB = (const bf16*)lm_B;
  p.Wlm = Wlm;
  p.sidx = im->d_sidx; p.accel_cols = im->accel_cols; p.rope_tab = rope_tab;
  p.n_gates = c.n_gates;
  p.R = im->R;
  p.act = im->act; p.qbuf = im->qbuf; p.khat = im->khat; p.vhat = im->vhat;
  p.apart = im->apart; p.upart = im->upart; p.apu = im->apu; p.udpart = im->udpart;
  p.nah = c.accel_enabled ? c.n_accel_heads : 0;
  p.ctl = im->d_ctl;
  p.pf_ahead = PF_DEFAULT;
  p.tl = nullptr;
#ifdef M2R2_FUSED_DEBUG
  if (getenv("M2R2_PF")) p.pf_ahead = atoi(getenv("M2R2_PF"));   // debug builds only: sweep the L2 prefetch window
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
  // grid barriers of this launch (must match the kernel's sequence): per layer 4 weight phases + attention,
  // one per exit head, one for the final head
  unsigned int nbar = 5u * (unsigned int)run.n_layers + 1u;
  for (int i = 0; i < run.n_layers; ++i)
    if (im->gate_of[i] && im->accel_of[i] && run.exit_heads && !(run.head_stream == 1 && i + 1 == run.n_layers)) ++nbar;
  p.bar_base = im->bar_base;
  void* args[] = {(void*)&p};
  cudaError_t e = cudaLaunchCooperativeKernel((const void*)m2r2_fused_decode_kernel, dim3(G), dim3(NTHREADS), args,
                                              SMEM_BYTES, st);
  if (e != cudaSuccess) return M2R2_CUDA;
  im->bar_base += nbar * (unsigned int)G;   // only a launch that was enqueued moves the barrier target
  if (launches) *launches += 1;
  return 0;
}

// non-blocking: has any launch so far reported a timed-out wait?  (host-mapped flag, no stream synchronisation)
bool fused_abort_pending(const FusedState* fs) {
  return fs->supported && fs->impl && fs->impl->bound && fs->impl->h_abort && *(volatile unsigned int*)fs->impl->h_abort != 0u;
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
    {
      Ctl z;
      memset(&z, 0, sizeof(z));
      z.host_abort = im->d_abort;
      *im->h_ctl = z;
      cudaMemcpyAsync(im->d_ctl, im->h_ctl, sizeof(Ctl), cudaMemcpyHostToDevice, st);
    }
    *im->h_abort = 0u;
    cudaMemsetAsync(im->upart, 0, sizeof(u64) * UPART_N * UPART_STRIDE, st);
    cudaStreamSynchronize(st);
    im->bar_base = 0;
    return M2R2_CUDA;
  }
  return 0;
}

// a11 on the fragment-major weights: out = f(W x) for rows <= 8 slow-stream rows (kinds: VK_*).  Returns
// M2R2_UNSUPPORTED when the fused copy is not bound (the caller then uses the row-major kernels).
// ------------------------------------------------------------------ <= 8 rows: the same GEMM as a persistent ring kernel
// For the k-token verify pass and prefill chunks at batch 1 the matrices are streamed exactly as the fused decode kernel
// streams them: one CTA per SM owns a contiguous range of the matrix's 32 KB stages, a producer thread moves them through a
// shared-memory ring with cp.async.bulk + mbarriers, eight consumer warps multiply.  Under programmatic dependent launch
// the producer starts BEFORE the previous kernel of the chain has finished (weights do not depend on it), so the ring is
// full when the activation rows arrive; the rows (<= 8) are staged once per CTA as (bf16 hi pair, bf16 lo pair) words, so
// that one LDS.64 yields a B fragment register of both MMAs.
//   row-owned matrices (QKV, gate/up, LM head): stage = one 16-row tile x 1024 inputs; the warps split the inputs and add
//     their partial sums of a finished row tile into one of RR_NB shared-memory accumulators; the warp that arrives last
//     runs the epilogue (no CTA barrier in the stream);
//   split-K matrices (O, down): stage = 8 row tiles x 128 inputs; warp w owns row tile w, accumulates over the k-chunks of
//     a group inside the CTA's range and adds onto the in-place residual atomically.
// The kernel can absorb its neighbours in the layer (RowsFuse): RMSNorm of the rows while they are staged (the sums of
// squares are collected on the way, 1 / rms multiplies the finished sums: W (g (.) x / rms) = (W (g (.) x)) / rms), and
// RoPE + the K/V cache append in the QKV epilogue.
// thread-block cluster of two CTAs: the pair stages the activation rows of a row-owned matrix together (each loads half of
// the columns from L2 and writes the converted words into both CTAs' shared memory)
__device__ __forceinline__ uint32_t cluster_ctarank() { uint32_t r; asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r)); return r; }
__device__ __forceinline__ uint32_t mapa_peer(const void* local, uint32_t rank) {
  uint32_t r;
  asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(smem_u32(local)), "r"(rank));
  return r;
}
__device__ __forceinline__ void st_cluster_v4(uint32_t raddr, uint4 v) {
  asm volatile("st.shared::cluster.v4.b32 [%0], {%1, %2, %3, %4};" ::"r"(raddr), "r"(v.x), "r"(v.y), "r"(v.z), "r"(v.w) : "memory");
}
__device__ __forceinline__ void st_cluster_f32(uint32_t raddr, float v) {
  asm volatile("st.shared::cluster.f32 [%0], %1;" ::"r"(raddr), "f"(v) : "memory");
}
__device__ __forceinline__ void mbar_arrive_cluster(uint32_t raddr) {   // releases the thread's earlier (remote) stores
  asm volatile("mbarrier.arrive.release.cluster.shared::cluster.b64 _, [%0];" ::"r"(raddr) : "memory");
}
__device__ __forceinline__ bool mbar_try_wait_cluster(u64* b, uint32_t parity) {
  uint32_t ok;
  asm volatile("{ .reg .pred p; mbarrier.try_wait.parity.acquire.cluster.shared::cta.b64 p, [%1], %2; selp.u32 %0, 1, 0, p; }"
               : "=r"(ok) : "r"(smem_u32(b)), "r"(parity) : "memory");
  return ok != 0;
}
__device__ __forceinline__ void cluster_sync_all() {
  asm volatile("barrier.cluster.arrive.release.aligned;\n\tbarrier.cluster.wait.acquire.aligned;" ::: "memory");
}
constexpr int RR_THREADS = NCT + 32;
constexpr int RR_NB = 8;   // row-tile accumulators: a warp runs at most nst (<= 6) stages = 6 / nks row tiles ahead of the slowest one;
                           // matrices with nks >= 2 stages per row tile use 4 of them
template <int KIND>
__global__ void __launch_bounds__(RR_THREADS, 1) rows_ring_kernel(const VArgs a, int nst, int ld2, int xs_chunks, int csize, int nb, unsigned int zero) {
  extern __shared__ __align__(1024) unsigned char rr_smem[];
  unsigned char* const ring = rr_smem;
  uint2* const xp = (uint2*)(rr_smem + (size_t)nst * STAGE_BYTES);    // [rows][ld2]: inputs 2p, 2p + 1 as (hi, lo)
  float* const acc = (float*)(xp + (size_t)a.rows * ld2);             // [nb][4][32]
  u64* const full = (u64*)(acc + nb * 4 * 32);
  u64* const empty = full + 8;
  float* const ssq = (float*)(empty + 8);                             // [2 ranks][8] sums of squares of the rows (fused RMSNorm)
  unsigned int* const cnt = (unsigned int*)(ssq + 2 * 8);             // [RR_NB] warps that have added their part
  u64* const xdone = (u64*)(cnt + RR_NB);                             // the cluster peer's half of the rows has arrived (NCT arrivals)
  float2* const rope_s = (float2*)(xdone + 1);                        // [rows][dh / 2] RoPE (cos, sin) of the rows' positions (QKV)
  int* const seq_s = (int*)(rope_s + a.rows * (a.dh >> 1));           // [8] row -> sequence, [8] row -> position (QKV)
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, g = lane >> 2, t = lane & 3;
  const int G = gridDim.x, v = blockIdx.x;
  constexpr bool split = KIND == VK_OPROJ || KIND == VK_DOWN;   // (= a.split)
  const int nks = a.nstage_k;
  int s0, s1;
  if (!split) { s0 = range_lo(a.n_rt, v, G) * nks; s1 = range_lo(a.n_rt, v + 1, G) * nks; }
  else { const int S = (a.n_rt / SK_RT) * nks; s0 = range_lo(S, v, G); s1 = range_lo(S, v + 1, G); }
  if (tid == 0) {
    for (int i = 0; i < nst; ++i) { mbar_init(&full[i], 1); mbar_init(&empty[i], NCW); }
    mbar_init(xdone, NCT);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  if (tid < 2 * 8) ssq[tid] = 0.f;
  const bool pair = csize == 2 && !split;        // the two CTAs of the cluster stage the rows together
  const uint32_t rank = csize == 2 ? cluster_ctarank() : 0u;
  if (csize == 2) cluster_sync_all(); else __syncthreads();   // barriers and ssq are initialised in both CTAs
  pdl_launch_dependents();
  if (tid >= NCT) {
    if (tid == NCT) {   // producer: every stage of the CTA's range, independent of the previous kernel
      // (requesting further stages into L2 while the consumers stage the rows was measured: the rows' loads slow down
      // by more than the stream gains, 4.80 -> 4.91 ms per C3 spec_step)
      const u64 pol = policy_evict_first();
      for (int s = s0, i = 0; s < s1; ++s, ++i) {
        const int slot = i % nst, use = i / nst;
        while (!mbar_try_wait(&empty[slot], (use & 1u) ^ 1u)) { }
        mbar_expect_tx(&full[slot], STAGE_BYTES);
        bulk_g2s(ring + (size_t)slot * STAGE_BYTES, a.W + (size_t)s * (STAGE_BYTES / 16), STAGE_BYTES, &full[slot], pol);
      }
    }
    return;
  }
  // ---- consumers
  for (int i = tid; i < nb * 4 * 32; i += NCT) acc[i] = 0.f;
  if (tid < RR_NB) cnt[tid] = 0u;
  pdl_wait();
  if (KIND == VK_QKV && a.rope_tab) {
    const int half = a.dh >> 1;
    for (int i = tid; i < a.rows * half; i += NCT) {
      const int n = i / half, j = i - n * half;
      rope_s[n * half + j] = a.rope_tab[(size_t)a.row_pos[n] * half + j];
    }
    if (tid < a.rows) { seq_s[tid] = a.row_seq[tid]; seq_s[8 + tid] = a.row_pos[tid]; }
  }
  // (kept compact on purpose: this loop form measured faster than a version with all eight rows unrolled per thread;
  // after the wait a CTA needs ~1.3 us for the loads to land, ~1.6 us to convert and store, ~0.7 us for the exchange)
  if (!split) {
    // all inputs of every row, in units of eight inputs (one 32-byte sector of fp32): this CTA loads the units u = rank
    // (mod cluster size), converts them and writes the words into its own and the peer's shared memory (all CTAs read
    // the same rows at the same moment: a pair halves that L2 traffic)
    const int nu = nks * (STAGE_K / 8);            // units per row
    const int step = pair ? 2 : 1, nu_mine = nu / step, items = a.rows * nu_mine;   // nu_mine % 32 == 0: a warp's items share the row
    const uint32_t peer_xp = pair ? mapa_peer(xp, rank ^ 1u) : 0u;
#pragma unroll 1
    for (int i0 = tid; i0 < items; i0 += 4 * NCT) {
      float4 xa[4], xb[4];
      uint4 gr[4];
#pragma unroll
      for (int u = 0; u < 4; ++u) {
        const int i = i0 + u * NCT;
        xa[u] = xb[u] = make_float4(0.f, 0.f, 0.f, 0.f);
        gr[u] = make_uint4(0x3f803f80u, 0x3f803f80u, 0x3f803f80u, 0x3f803f80u);   // bf16 ones
        if (i < items) {
          const int row = i / nu_mine, k = 8 * ((i - row * nu_mine) * step + (pair ? (int)rank : 0));
          if (k < a.K) {
            const float4* src = (const float4*)(a.X + (size_t)row * a.ldx + k);
            xa[u] = __ldg(src);
            xb[u] = __ldg(src + 1);
            if (a.gain) gr[u] = __ldg((const uint4*)(a.gain + k));
          }
        }
      }
#pragma unroll
      for (int u = 0; u < 4; ++u) {
        const int i = i0 + u * NCT;
        if (i < items) {
          const int row = i / nu_mine, k = 8 * ((i - row * nu_mine) * step + (pair ? (int)rank : 0));
          const float4 x0 = xa[u], x1 = xb[u];
          const float2 g0 = __bfloat1622float2(*(const __nv_bfloat162*)&gr[u].x), g1 = __bfloat1622float2(*(const __nv_bfloat162*)&gr[u].y);
          const float2 g2 = __bfloat1622float2(*(const __nv_bfloat162*)&gr[u].z), g3 = __bfloat1622float2(*(const __nv_bfloat162*)&gr[u].w);
          uint4 w0, w1;
          w0.x = pack_hi_lo(x0.x * g0.x, x0.y * g0.y, w0.y); w0.z = pack_hi_lo(x0.z * g1.x, x0.w * g1.y, w0.w);
          w1.x = pack_hi_lo(x1.x * g2.x, x1.y * g2.y, w1.y); w1.z = pack_hi_lo(x1.z * g3.x, x1.w * g3.y, w1.w);
          const size_t off = (size_t)row * ld2 + (k >> 1);
          *(uint4*)(xp + off) = w0;
          *(uint4*)(xp + off + 2) = w1;
          if (pair) {
            st_cluster_v4(peer_xp + (uint32_t)(off * sizeof(uint2)), w0);
            st_cluster_v4(peer_xp + (uint32_t)((off + 2) * sizeof(uint2)), w1);
          }
          if (a.gain) {
            const float sq = warp_sum(x0.x * x0.x + x0.y * x0.y + x0.z * x0.z + x0.w * x0.w + x1.x * x1.x + x1.y * x1.y + x1.z * x1.z + x1.w * x1.w);
            if (lane == 0) atomicAdd(&ssq[rank * 8 + row], sq);
          }
        }
      }
    }
    if (pair) {
      if (a.gain) {
        bar_consumers();   // this CTA's sums of squares are complete
        if (tid < 8) st_cluster_f32(mapa_peer(ssq, rank ^ 1u) + (uint32_t)((rank * 8 + tid) * sizeof(float)), ssq[rank * 8 + tid]);
      }
      mbar_arrive_cluster(mapa_peer(xdone, rank ^ 1u));
    }
  } else if (KIND == VK_OPROJ && a.part_o != nullptr && s1 > s0) {
    // O with the split merge absorbed (a4): the inputs of the CTA's k-chunks are merged from the attention partials of
    // their heads, merge_kernel's arithmetic (slow rows); the loads of all splits of an item are in flight together
    const int kc0 = s0 % nks, cnt_c = min(s1 - s0, nks), items = a.rows * cnt_c * (SK_K / 4);
    const int ns = a.n_splits;
#pragma unroll 1
    for (int i = tid; i < items; i += NCT) {
      const int q = i & 31, j = i >> 5, row = j / cnt_c, ci = j - row * cnt_c;
      int kc = kc0 + ci;
      if (kc >= nks) kc -= nks;
      const int k = kc * SK_K + 4 * q;
      float4 x4 = make_float4(0.f, 0.f, 0.f, 0.f);
      if (k < a.K) {
        const int head = k / a.dh, e = k - head * a.dh;   // dh % 4 == 0: the four inputs share the head
        const size_t pbase = ((size_t)row * a.n_heads + head) * ns;
        float2 ml[8];
        float4 o[8];
#pragma unroll
        for (int sp = 0; sp < 8; ++sp) {
          ml[sp] = make_float2(0.f, 0.f);
          o[sp] = make_float4(0.f, 0.f, 0.f, 0.f);
          if (sp < ns) {
            ml[sp] = __ldcg((const float2*)a.part_ml + pbase + sp);
            o[sp] = __ldcg((const float4*)(a.part_o + (pbase + sp) * a.dh + e));
          }
        }
        float M = -INFINITY, L = 0.f;
#pragma unroll
        for (int sp = 0; sp < 8; ++sp)
          if (ml[sp].y > 0.f) M = fmaxf(M, ml[sp].x);
#pragma unroll
        for (int sp = 0; sp < 8; ++sp) {
          if (ml[sp].y > 0.f) {
            const float w = __expf(ml[sp].x - M);
            L += ml[sp].y * w;
            x4.x += o[sp].x * w; x4.y += o[sp].y * w; x4.z += o[sp].z * w; x4.w += o[sp].w * w;
          }
        }
        x4.x /= L; x4.y /= L; x4.z /= L; x4.w /= L;
      }
      uint4 w;
      w.x = pack_hi_lo(x4.x, x4.y, w.y); w.z = pack_hi_lo(x4.z, x4.w, w.w);
      *(uint4*)(xp + (size_t)row * ld2 + (((kc % xs_chunks) * SK_K + 4 * q) >> 1)) = w;
    }
  } else if (s1 > s0) {
    // the k-chunks of the CTA's range (slots by chunk index modulo xs_chunks), four loads in flight per thread
    const int kc0 = s0 % nks, cnt_c = min(s1 - s0, nks), items = a.rows * cnt_c * (SK_K / 4);   // SK_K / 4 == 32
#pragma unroll 1
    for (int i0 = tid; i0 < items; i0 += 4 * NCT) {
      float4 xr[4];
      int xo[4];
#pragma unroll
      for (int u = 0; u < 4; ++u) {
        const int i = i0 + u * NCT;
        xr[u] = make_float4(0.f, 0.f, 0.f, 0.f);
        xo[u] = -1;
        if (i < items) {
          const int q = i & 31, j = i >> 5, row = j / cnt_c, ci = j - row * cnt_c;
          int kc = kc0 + ci;
          if (kc >= nks) kc -= nks;
          const int k = kc * SK_K + 4 * q;
          if (k < a.K) xr[u] = __ldg((const float4*)(a.X + (size_t)row * a.ldx + k));
          xo[u] = row * ld2 + (((kc % xs_chunks) * SK_K + 4 * q) >> 1);
        }
      }
#pragma unroll
      for (int u = 0; u < 4; ++u) {
        if (xo[u] >= 0) {
          uint4 w;
          w.x = pack_hi_lo(xr[u].x, xr[u].y, w.y); w.z = pack_hi_lo(xr[u].z, xr[u].w, w.w);
          *(uint4*)(xp + xo[u]) = w;
        }
      }
    }
  }
  bar_consumers();
  if (pair) while (!mbar_try_wait_cluster(xdone, 0u)) { }

  // (lanes of the MMA's columns >= a.rows read row a.rows - 1: those columns of the result are never stored)
  const uint2* bp = xp + (size_t)min(g, a.rows - 1) * ld2 + t;
  float c[4] = {0.f, 0.f, 0.f, 0.f}, cl[4] = {0.f, 0.f, 0.f, 0.f};
  float rs[2] = {1.f, 1.f};   // 1 / rms of activation rows 2t, 2t + 1
  if (!split && a.gain) {
#pragma unroll
    for (int sx = 0; sx < 2; ++sx) {
      const float tot = ssq[2 * t + sx] + ssq[8 + 2 * t + sx];
      rs[sx] = rsqrtf(tot / (float)a.K + a.eps);
    }
  }
  for (int s = s0, i = 0; s < s1; ++s, ++i) {
    const int slot = i % nst, use = i / nst;
    while (!mbar_try_wait(&full[slot], use & 1u)) { }
    const uint4* A = (const uint4*)(ring + (size_t)slot * STAGE_BYTES) + (warp * TPW) * 32 + lane;
    int p0;   // first input pair of the warp's eight tiles, in staged coordinates
    if (!split) p0 = ((s % nks) * STAGE_K + warp * (TPW * 16)) >> 1;
    else p0 = (((s % nks) % xs_chunks) * SK_K) >> 1;
    uint32_t dep = 0u;
#pragma unroll
    for (int u = 0; u < TPW; ++u) {
      const uint4 w = A[u * 32];
      const uint2 b0 = bp[p0 + u * 8], b1 = bp[p0 + u * 8 + 4];   // inputs 16u + 2t (+1) and + 8: (hi, lo)
      mma_bf16(c, w, b0.x, b1.x);
      mma_bf16(cl, w, b0.y, b1.y);   // the lo parts' products: a second, independent accumulation chain
      dep ^= w.x;
    }
    __syncwarp();
    if (lane == 0) release_stage(&empty[slot], zero, __uint_as_float(dep));
    if (!split) {
      if ((s % nks) != nks - 1) continue;
      // the row tile is finished in this warp's k range: add the partial sums into the tile's accumulator; the warp that
      // arrives last holds the complete sums and finishes the tile
      const int rt = s / nks, b = (i / nks) % nb;
      float* ab = acc + b * 4 * 32;
#pragma unroll
      for (int e = 0; e < 4; ++e) { atomicAdd(ab + e * 32 + lane, c[e] + cl[e]); c[e] = 0.f; cl[e] = 0.f; }
      __syncwarp();
      unsigned int old = 0u;
      if (lane == 0) { __threadfence_block(); old = atomicAdd(&cnt[b], 1u); }
      old = __shfl_sync(0xffffffffu, old, 0);
      if (old != NCW - 1) continue;
      __threadfence_block();
      float r4[4];
#pragma unroll
      for (int e = 0; e < 4; ++e) { r4[e] = ab[e * 32 + lane] * rs[e & 1]; ab[e * 32 + lane] = 0.f; }
      if (lane == 0) cnt[b] = 0u;
      // r4[0], r4[1] = weight row g x activation rows 2t, 2t + 1; r4[2], r4[3] = weight row g + 8
      if (KIND == VK_QKV) {
        // the tile's 16 packed rows lie in one head of q, k or v (d % 16 == 0, dh % 16 == 0): packed row 2i / 2i + 1 of a
        // q or k head = elements i / i + dh / 2 (the RoPE pair, the partner sits in lane ^ 4); v rows are in natural order
        const int base = rt * 16, which = base / a.d, w_ = base - which * a.d, head = w_ / a.dh, e0 = w_ - head * a.dh;
        const int half = a.dh >> 1;
        const bool rope = a.rope_tab != nullptr;
#pragma unroll
        for (int sx = 0; sx < 2; ++sx) {
          const int n = 2 * t + sx;
          const bool live = n < a.rows;
          float* orow = a.out + (size_t)n * a.ldo + which * a.d + head * a.dh;
          size_t cbase = 0;
          if (rope && live) cbase = (((size_t)seq_s[n] * a.n_heads + head) * a.max_seq + seq_s[8 + n]) * a.dh;
#pragma unroll
          for (int hh = 0; hh < 2; ++hh) {
            const float val = r4[2 * hh + sx];
            const float pv = __shfl_xor_sync(0xffffffffu, val, 4);
            const int e = e0 + g + 8 * hh;
            if (!live || base + g + 8 * hh >= a.n_out) continue;
            if (which < 2) {
              const int j = e >> 1, ne = j + (e & 1) * half;
              float o = val;
              if (rope) {   // a3, rope_append_kernel's arithmetic
                const float2 cs = rope_s[n * half + j];
                o = (e & 1) ? val * cs.x + pv * cs.y : val * cs.x - pv * cs.y;
                if (which == 1) a.Kc[cbase + ne] = __float2bfloat16_rn(o);
              }
              orow[ne] = o;
            } else {
              orow[e] = val;
              if (rope) a.Vc[cbase + e] = __float2bfloat16_rn(val);
            }
          }
        }
        continue;
      }
#pragma unroll
      for (int sx = 0; sx < 2; ++sx) {
        const int n = 2 * t + sx;
        if (n >= a.rows) continue;
        const float v0 = r4[sx], v1 = r4[2 + sx];
        if (KIND == VK_GATEUP) {
          const int o = rt * 8 + g;
          if (o < a.n_out) a.out[(size_t)n * a.ldo + o] = silu(v0) * v1;
          continue;
        }
#pragma unroll
        for (int hh = 0; hh < 2; ++hh) {
          const int pr = rt * 16 + g + 8 * hh;
          if (pr < a.n_out) a.out[(size_t)n * a.ldo + pr] = hh ? v1 : v0;
        }
      }
    } else {
      const int kc = s % nks;
      if (kc == nks - 1 || s == s1 - 1) {
        // split-K: this CTA's part of the sums of row tile (group, warp) onto the in-place residual
        const int rt = (s / nks) * SK_RT + warp;
#pragma unroll
        for (int sx = 0; sx < 2; ++sx) {
          const int n = 2 * t + sx;
          if (n >= a.rows) continue;
#pragma unroll
          for (int hh = 0; hh < 2; ++hh) {
            const int pr = rt * 16 + g + 8 * hh;
            if (pr < a.n_out) atomicAdd(a.out + (size_t)n * a.ldo + pr, c[2 * hh + sx] + cl[2 * hh + sx]);
          }
        }
#pragma unroll
        for (int e = 0; e < 4; ++e) { c[e] = 0.f; cl[e] = 0.f; }
      }
    }
  }
}
template <int KIND>
static int launch_rows_ring(const VArgs& a, int G, int smem_max, unsigned int zero, cudaStream_t st) {
  const int nks = a.nstage_k;
  int kx, xs_chunks = 1;   // staged inputs per row
  if (!a.split) {
    kx = nks * STAGE_K;
  } else {
    const int S = (a.n_rt / SK_RT) * nks, maxL = (S + G - 1) / G + 1;
    xs_chunks = std::min(nks, (maxL + 7) / 8 * 8);
    kx = xs_chunks * SK_K;
  }
  const int ld2 = kx / 2 + 4;   // (hi, lo) words per staged row; = 4 mod 16: the LDS.64 of a half-warp hit 16 distinct bank pairs
  const int nb = (!a.split && nks < 2) ? RR_NB : 4;
  const size_t xbytes = (size_t)a.rows * ld2 * sizeof(uint2);
  const size_t fixed = xbytes + (size_t)nb * 4 * 32 * sizeof(float) + 512 + (KIND == VK_QKV ? (size_t)a.rows * (a.dh / 2) * sizeof(float2) + 64 : 0);
  if ((size_t)smem_max < fixed + 2 * (size_t)STAGE_BYTES) return M2R2_UNSUPPORTED;
  // ring depth: what fits, no more than a CTA's stages, at most 6 (split-K) / 4 (row-owned: a fifth stage fits at d = 3072
  // with 5 rows and measured 0.6 % slower per C3 spec_step — more copies in flight while the rows are staged slow the
  // rows' loads down, as the L2 prefetch did)
  const int max_stages = a.split ? ((a.n_rt / SK_RT) * nks + G - 1) / G : (a.n_rt + G - 1) / G * nks;
  static const int xcap_r = xknob("M2R2_XCAPR", 4), xcap_s = xknob("M2R2_XCAPS", 6);
  const size_t cap = a.split ? xcap_s : xcap_r;
  const int nst = std::max(2, std::min((int)std::min<size_t>(cap, ((size_t)smem_max - fixed) / STAGE_BYTES), max_stages));
  const size_t sh = (size_t)nst * STAGE_BYTES + fixed;
  static bool attr_set = false;
  if (!attr_set) {
    cudaFuncSetAttribute(rows_ring_kernel<KIND>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_max);
    attr_set = true;
  }
  static const bool no_cluster = xknob("M2R2_XNOCLUSTER", 0) != 0;
  const int csize = (G % 2 == 0 && !no_cluster) ? 2 : 1;
  cudaLaunchConfig_t cfg = cudaLaunchConfig_t();
  cfg.gridDim = dim3(G); cfg.blockDim = dim3(RR_THREADS); cfg.dynamicSmemBytes = sh; cfg.stream = st;
  cudaLaunchAttribute at[2];
  at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  at[0].val.programmaticStreamSerializationAllowed = 1;
  at[1].id = cudaLaunchAttributeClusterDimension;
  at[1].val.clusterDim.x = csize; at[1].val.clusterDim.y = 1; at[1].val.clusterDim.z = 1;
  cfg.attrs = at; cfg.numAttrs = 2;
  return cudaLaunchKernelEx(&cfg, rows_ring_kernel<KIND>, a, nst, ld2, xs_chunks, csize, nb, zero) == cudaSuccess ? 0 : M2R2_CUDA;
}

template <int KIND, int NG, bool SW>
static void launch_rows_mma_t(const VArgs& a, dim3 grid, cudaStream_t st) {
  const size_t sh = (size_t)2 * NG * 8 * ((SW ? 4 : 1) * RM_KC + 8) * sizeof(bf16);
  static bool attr_set = false;
  if (!attr_set) {
    cudaFuncSetAttribute(rows_mma_kernel<KIND, NG, SW>, cudaFuncAttributeMaxDynamicSharedMemorySize, 96 * 1024);
    attr_set = true;
  }
  // programmatic dependent launch: the kernel starts while its predecessor in the stream drains and prefetches its first
  // weight tiles; it reads activations only behind pdl_wait()
  cudaLaunchConfig_t cfg;
  memset(&cfg, 0, sizeof(cfg));
  cfg.gridDim = grid; cfg.blockDim = dim3(SW ? 128 : RM_NW * 32); cfg.dynamicSmemBytes = sh; cfg.stream = st;
  cudaLaunchAttribute at[1];
  at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  at[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = at; cfg.numAttrs = 1;
  cudaLaunchKernelEx(&cfg, rows_mma_kernel<KIND, NG, SW>, a);
}
template <int KIND, int NG>
static void launch_rows_epilogue_t(const VArgs& a, cudaStream_t st) {
  launch_pdl(rows_epilogue_kernel<KIND, NG>, dim3((a.n_rt + 3) / 4, NG), dim3(128), 0, st, a);
}
template <int KIND>
static void launch_rows_epilogue(const VArgs& a, int ng, cudaStream_t st) {
  switch (ng) {
    case 2: launch_rows_epilogue_t<KIND, 2>(a, st); break;
    case 3: launch_rows_epilogue_t<KIND, 3>(a, st); break;
    case 4: launch_rows_epilogue_t<KIND, 4>(a, st); break;
    case 5: launch_rows_epilogue_t<KIND, 5>(a, st); break;
    case 6: launch_rows_epilogue_t<KIND, 6>(a, st); break;
    case 7: launch_rows_epilogue_t<KIND, 7>(a, st); break;
    default: launch_rows_epilogue_t<KIND, 8>(a, st); break;
  }
}
template <int KIND>
static void launch_rows_mma(const VArgs& a, dim3 grid, int ng, cudaStream_t st) {
  switch (ng) {
    case 1: launch_rows_mma_t<KIND, 1, true>(a, grid, st); break;
    case 2: launch_rows_mma_t<KIND, 2, false>(a, grid, st); break;
    case 3: launch_rows_mma_t<KIND, 3, false>(a, grid, st); break;
    case 4: launch_rows_mma_t<KIND, 4, false>(a, grid, st); break;
    case 5: launch_rows_mma_t<KIND, 5, false>(a, grid, st); break;
    case 6: launch_rows_mma_t<KIND, 6, false>(a, grid, st); break;
    case 7: launch_rows_mma_t<KIND, 7, false>(a, grid, st); break;
    default: launch_rows_mma_t<KIND, 8, false>(a, grid, st); break;
  }
}

int fused_gemv_rows(const m2r2_config& c, FusedState* fs, cudaStream_t st, int layer, int kind, const float* X, int ldx,
                    int rows, float* out, int ldo, const float* resid, float* trace, const GemvArgs* lora, const RowsFuse* fz) {
  if (!fs->supported || !fs->impl || !fs->impl->bound || rows < 1 || rows > 64 || (c.d_model % 4) || (c.d_ff % 4)) return M2R2_UNSUPPORTED;
  FusedImpl* im = fs->impl;
  PackedDims q = packed_dims(c);
  VArgs a;
  memset(&a, 0, sizeof(a));
  a.X = X; a.ldx = ldx; a.rows = rows; a.out = out; a.ldo = ldo; a.resid = resid; a.trace = trace;
  a.d = c.d_model; a.dh = c.head_dim;
  int n_rt = 0;
  a.ksplit = 1;
  const FLayer* L = kind == VK_HEAD ? nullptr : &im->h_layers[layer];
  switch (kind) {
    case VK_QKV:    a.W = L->Wqkv; a.K = c.d_model; a.n_out = 3 * c.d_model; a.nkt = q.d_pad / 16; a.nstage_k = q.d_pad / STAGE_K; a.split = 0; n_rt = q.rt_qkv; break;
    case VK_OPROJ:  a.W = L->Wo;   a.K = c.d_model; a.n_out = c.d_model; a.nkt = q.nkc_o * 8; a.nstage_k = q.nkc_o; a.split = 1; n_rt = q.ng_d * SK_RT; break;
    case VK_GATEUP: a.W = L->Wgu;  a.K = c.d_model; a.n_out = c.d_ff; a.nkt = q.d_pad / 16; a.nstage_k = q.d_pad / STAGE_K; a.split = 0; n_rt = q.rt_gu; break;
    case VK_DOWN:   a.W = L->Wd;   a.K = c.d_ff; a.n_out = c.d_model; a.nkt = q.nkc_d * 8; a.nstage_k = q.nkc_d; a.split = 1; n_rt = q.ng_d * SK_RT; break;
    default:        a.W = im->h_Wlm; a.K = c.d_model; a.n_out = c.vocab; a.nkt = q.d_pad / 16; a.nstage_k = q.d_pad / STAGE_K; a.split = 0; n_rt = q.rt_v; break;
  }
  a.n_rt = n_rt;
  if (lora && lora->Bm) {
    a.Bm = (const bf16*)lora->Bm; a.Bm2 = (const bf16*)lora->Bm2; a.bmap = lora->bmap; a.U = lora->U;
    a.ldu = lora->ldu; a.r = lora->r; a.lora_row0 = lora->lora_row0; a.usel_div = lora->usel_div;
  }
  static const bool no_ring = xknob("M2R2_XNORING", 0) != 0;
  const bool ring = rows <= 8 && !(lora && lora->Bm) && !no_ring && ((kind != VK_OPROJ && kind != VK_DOWN) || (resid == out && !trace)) &&
                    (kind != VK_QKV || (c.d_model % 16 == 0 && c.head_dim % 16 == 0));
  a.tile_in_head = (c.d_model % 16 == 0 && c.head_dim % 16 == 0) ? 1 : 0;
  a.slow_rows = rows;
  if (fz) {
    // the caller left the GEMM's neighbours to the kernel: the ring kernel honours all of them, rows_mma_kernel (> 8 rows)
    // RoPE + KV append in the QKV epilogue
    // (x_packed / pack_out concern rows_mma_kernel only and never make a call unsupported)
    const bool rope_ok = !fz->rope_tab || (kind == VK_QKV && a.tile_in_head && c.dtype == M2R2_BF16);
    const bool mma_ok = !fz->gain && !fz->part_o && rope_ok && rows > 8;
    if ((!ring && !mma_ok) || (c.head_dim % 4)) return M2R2_UNSUPPORTED;
    if (fz->rope_tab) a.slow_rows = fz->slow_rows > 0 ? fz->slow_rows : rows;
    a.gain = (const bf16*)fz->gain; a.eps = fz->eps;
    a.n_heads = c.n_heads;
    a.part_o = fz->part_o; a.part_ml = fz->part_ml; a.n_splits = fz->n_splits;
    if (a.part_o && (kind != VK_OPROJ || a.n_splits < 1 || a.n_splits > 8)) return M2R2_UNSUPPORTED;
    a.row_seq = fz->row_seq; a.row_pos = fz->row_pos; a.rope_tab = fz->rope_tab; a.Kc = (bf16*)fz->Kc; a.Vc = (bf16*)fz->Vc;
    a.max_seq = c.max_seq;
  }
  if (ring) {
    // batch-1 verify pass / prefill chunks: the persistent ring kernel (one CTA per SM)
    static int smem_max = 0;
    if (!smem_max) {
      int dev = 0;
      cudaGetDevice(&dev);
      cudaDeviceGetAttribute(&smem_max, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev);
    }
    int rc;
    switch (kind) {
      case VK_QKV:    rc = launch_rows_ring<VK_QKV>(a, im->G, smem_max, 0u, st); break;
      case VK_OPROJ:  rc = launch_rows_ring<VK_OPROJ>(a, im->G, smem_max, 0u, st); break;
      case VK_GATEUP: rc = launch_rows_ring<VK_GATEUP>(a, im->G, smem_max, 0u, st); break;
      case VK_DOWN:   rc = launch_rows_ring<VK_DOWN>(a, im->G, smem_max, 0u, st); break;
      default:        rc = launch_rows_ring<VK_HEAD>(a, im->G, smem_max, 0u, st); break;
    }
    if (rc != M2R2_UNSUPPORTED || fz) return rc;
  }
  {
    // 4 row tiles per CTA; O / down split along K (atomic adds onto the in-place residual) so that every SM streams
    const int ng = (rows + 7) / 8;
    const bool sw = ng <= 1;                       // one row tile per CTA, the warps split K (rows_mma_kernel SW); with more
                                                   // rows the replicated activation reads would exceed the weight stream
    const int gx = sw ? n_rt : (n_rt + RM_NW - 1) / RM_NW, nch = sw ? (a.nkt + 63) / 64 : (a.nkt + 15) / 16;
    static const int slots_per_sm = xknob("M2R2_XSLOTS", 512 / (RM_NW * 32));   // rows_mma_kernel: <= 128 registers per thread, 512 threads per SM
    if ((kind == VK_OPROJ || kind == VK_DOWN) && resid == out && !trace) {
      const int want = sw ? (4 * im->G + gx - 1) / gx : std::max(1, (slots_per_sm * im->G) / gx);   // one wave of CTAs
      a.ksplit = std::max(1, std::min(want, nch));
    }
    if (!sw && fz && fz->pack_out && kind == VK_GATEUP) { a.out_pk = im->act_pack; a.out_pk_ld = im->act_pack_ld; }
    const uint2* given = nullptr;   // the rows already as (hi, lo) words, left by their producer
    int given_ld = 0;
    if (!sw && fz && fz->x_packed) {
      if (kind == VK_QKV || kind == VK_GATEUP) { given = im->xn_pack; given_ld = im->xn_pack_ld; }
      else if (kind == VK_DOWN) { given = im->act_pack; given_ld = im->act_pack_ld; }
      if (given && 2 * given_ld < nch * RM_KC) given = nullptr;
    }
    if (given) {
      a.Xp = given; a.Kp = 2 * given_ld;
    } else if (!sw) {
      // > 8 rows: convert the rows once (pack_rows_kernel); the GEMM stages them by copy
      const int rows_pad = ng * 8, Kp = nch * RM_KC;
      if ((size_t)rows_pad * (Kp / 2) > im->xpack_n) return M2R2_UNSUPPORTED;
      const int items = rows_pad * (Kp / 4);
      launch_pdl(pack_rows_kernel, dim3(std::min((items + 255) / 256, 8 * im->G)), dim3(256), 0, st, a.X, a.ldx, a.rows, a.K, rows_pad, Kp, im->xpack);
      a.Xp = im->xpack; a.Kp = Kp;
      if (fs->launch_counter) ++*fs->launch_counter;
    }
    // QKV / gate-up with 9..64 rows: a CTA of 4 row tiles walks all of K with 8 KB per warp in flight, and there are only
    // n_rt / 4 = 144..256 CTAs: latency-bound at a fraction of the HBM rate.  Split along K as well; the partial sums meet
    // in rows_part (fp32 atomics, accumulator layout) and rows_epilogue_kernel finishes the tiles.
    static const bool no_two_stage = xknob("M2R2_XNOTWOSTAGE", 0) != 0;
    if ((kind == VK_QKV || kind == VK_GATEUP) && ng >= 2 && !no_two_stage && (size_t)n_rt * ng * 128 <= im->rows_part_n) {
      const int want = sw ? (4 * im->G + gx - 1) / gx : std::max(1, (slots_per_sm * im->G) / gx);   // one wave of CTAs
      a.ksplit = std::max(1, std::min(want, nch));
      if (a.ksplit > 1) a.part = im->rows_part;
    }
    const dim3 grid(gx, a.ksplit);
    if (a.part) {
      if (kind == VK_QKV) { launch_rows_mma<VK_QKV>(a, grid, ng, st); launch_rows_epilogue<VK_QKV>(a, ng, st); }
      else { launch_rows_mma<VK_GATEUP>(a, grid, ng, st); launch_rows_epilogue<VK_GATEUP>(a, ng, st); }
      if (fs->launch_counter) ++*fs->launch_counter;
      return cudaGetLastError() == cudaSuccess ? 0 : M2R2_CUDA;
    }
    switch (kind) {
      case VK_QKV:    launch_rows_mma<VK_QKV>(a, grid, ng, st); break;
      case VK_OPROJ:  launch_rows_mma<VK_OPROJ>(a, grid, ng, st); break;
      case VK_GATEUP: launch_rows_mma<VK_GATEUP>(a, grid, ng, st); break;
      case VK_DOWN:   launch_rows_mma<VK_DOWN>(a, grid, ng, st); break;
      default:        launch_rows_mma<VK_HEAD>(a, grid, ng, st); break;
    }
  }
  return cudaGetLastError() == cudaSuccess ? 0 : M2R2_CUDA;
}

// the (hi, lo) word buffers that producers outside this file fill for rows_mma_kernel (nullptr if the fused copy is not bound)
uint2* fused_xn_pack(const FusedState* fs, int* ld) {
  if (!fs || !fs->supported || !fs->impl || !fs->impl->bound) return nullptr;
  *ld = fs->impl->xn_pack_ld;
  return fs->impl->xn_pack;
}
