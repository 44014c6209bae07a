// kernels_general.cu — per-operation sm_100a kernels of the M2R2 path.
//
// These kernels serve every shape the ABI accepts (fp32 and bf16 storage, any number of
// activation rows: dual-stream decode, k-token verify, batched decode, chunked prefill, MoE).
// The batch-1 bf16 dense decode step has a faster persistent implementation in
// kernels_fused.cu; both compute the same operations.
//
// Row convention: activations are [rows][*] fp32.  Rows [0, slow_rows) belong to the slow
// stream h, rows [slow_rows, rows) to the accelerated stream p (Eq. 1 / Eq. 2).
#include "m2r2_internal.cuh"

// =====================================================================================
// a1  embed + stream init:  h_0 = Emb[token],  p_0 <- h_0
// =====================================================================================
template <typename WT>
__global__ void embed_kernel(const WT* __restrict__ emb, const int* __restrict__ tok, int d,
                             float* out, float* out2, float* trace, float* trace2) {
  int r = blockIdx.x;
  const WT* src = emb + (size_t)tok[r] * d;
  for (int j = threadIdx.x; j < d; j += blockDim.x) {
    float v = to_f32(src[j]);
    out[(size_t)r * d + j] = v;
    if (out2) out2[(size_t)r * d + j] = v;
    if (trace) trace[(size_t)r * d + j] = v;
    if (trace2) trace2[(size_t)r * d + j] = v;
  }
}

void launch_embed(cudaStream_t st, int dtype, const void* emb, const int* tok, int rows, int d,
                  float* out, float* out2, float* trace, float* trace2) {
  if (dtype == M2R2_FP32)
    embed_kernel<float><<<rows, 256, 0, st>>>((const float*)emb, tok, d, out, out2, trace, trace2);
  else
    embed_kernel<__nv_bfloat16><<<rows, 256, 0, st>>>((const __nv_bfloat16*)emb, tok, d, out, out2, trace, trace2);
}

// =====================================================================================
// RMSNorm (+ adapter down-projection u = A x^ for accelerated rows)
//   rms(x; g) = x * g / sqrt(mean(x^2) + eps)                       (Q1)
//   u[row][a*r + j] = A_a[j, :] . x^       a < nA packed adapters   (Q3)
// =====================================================================================
// (a, b) -> bf16 pair of the values and bf16 pair of what the first rounding lost: the two B operands of the GEMMs
__device__ __forceinline__ uint2 hi_lo_words(float a, float b) {
  const __nv_bfloat162 h = __floats2bfloat162_rn(a, b);
  const float2 f = __bfloat1622float2(h);
  const __nv_bfloat162 l = __floats2bfloat162_rn(a - f.x, b - f.y);
  return make_uint2(*(const uint32_t*)&h, *(const uint32_t*)&l);
}
// xn_pk (nullable): the normalised row also as (hi, lo) words [row][pk_ld], what rows_mma_kernel stages by copy for
// passes with more than 8 rows (the columns beyond d stay as the caller zeroed them)
template <typename WT>
__global__ void __launch_bounds__(256) norm_lora_kernel(const float* __restrict__ X, int d,
                                                        const WT* __restrict__ g, float eps,
                                                        float* __restrict__ xn, const WT* __restrict__ A,
                                                        int nA, int r, int lora_row0,
                                                        float* __restrict__ U, int ldu,
                                                        uint2* __restrict__ xn_pk, int pk_ld) {
  extern __shared__ float sx[];
  __shared__ float red[8];
  pdl_launch_dependents();   // the GEMM that consumes xn may begin to launch and prefetch its weights
  pdl_wait();
  int row = blockIdx.x, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  // blockIdx.y: part 0 writes xn; part p computes the adapter rows [8 p, 8 p + 8) of an accelerated row (every part
  // recomputes the norm: d elements, cheaper than a warp walking three adapter rows in turn)
  const int part = blockIdx.y;
  if (part > 0 && (A == nullptr || row < lora_row0)) return;
  const float* x = X + (size_t)row * d;
  float ss = 0.f;
  for (int j = tid; j < d; j += 256) {
    float v = x[j];
    sx[j] = v;
    ss += v * v;
  }
  ss = warp_sum(ss);
  if (lane == 0) red[warp] = ss;
  __syncthreads();
  float tot = 0.f;
#pragma unroll
  for (int w = 0; w < 8; ++w) tot += red[w];
  float inv = rsqrtf(tot / (float)d + eps);
  for (int p = tid; p < (d >> 1); p += 256) {   // d is even: pairs of elements
    const int j = 2 * p;
    const float v0 = sx[j] * inv * to_f32(g[j]), v1 = sx[j + 1] * inv * to_f32(g[j + 1]);
    sx[j] = v0;
    sx[j + 1] = v1;
    if (part == 0) {
      *(float2*)(xn + (size_t)row * d + j) = make_float2(v0, v1);
      if (xn_pk) xn_pk[(size_t)row * pk_ld + p] = hi_lo_words(v0, v1);
    }
  }
  if (A == nullptr || row < lora_row0) return;
  __syncthreads();
  for (int t = part * 8 + warp; t < nA * r; t += 8 * gridDim.y) {
    const WT* a = A + (size_t)t * d;
    float acc = 0.f;
    for (int k = lane * 8; k < d; k += 256) {
      float w[8];
      load8(a + k, w);
#pragma unroll
      for (int e = 0; e < 8; ++e) acc += w[e] * sx[k + e];
    }
    acc = warp_sum(acc);
    if (lane == 0) U[(size_t)row * ldu + t] = acc;
  }
}

void launch_norm_lora(cudaStream_t st, int dtype, const float* X, int rows, int d, const void* g,
                      float eps, float* xn, const void* A, int nA, int r, int lora_row0, float* U,
                      int ldu, uint2* xn_pk, int pk_ld) {
  size_t sh = (size_t)d * sizeof(float);
  const dim3 grid(rows, A ? std::max(1, (nA * r + 7) / 8) : 1);
  if (dtype == M2R2_FP32)
    launch_pdl(norm_lora_kernel<float>, grid, dim3(256), sh, st, X, d, (const float*)g, eps, xn, (const float*)A, nA, r, lora_row0, U, ldu, xn_pk, pk_ld);
  else
    launch_pdl(norm_lora_kernel<__nv_bfloat16>, grid, dim3(256), sh, st, X, d, (const __nv_bfloat16*)g, eps, xn, (const __nv_bfloat16*)A, nA, r, lora_row0, U, ldu, xn_pk, pk_ld);
}

// u[row][j] = A[j, :] . x[row][xmap(:)]   (no norm; A_o on the compact o^, A_d on the activations)
// One CTA per (row, j): with a CTA per row and a warp per j the d_ff-long dot products of A_d took 14 us on 8 CTAs.
template <typename WT>
__global__ void __launch_bounds__(256) lora_down_kernel(const float* __restrict__ X, int ldx, int row0, int K,
                                                        const int* __restrict__ xmap,
                                                        const WT* __restrict__ A, int r,
                                                        float* __restrict__ U, int ldu) {
  pdl_launch_dependents();
  pdl_wait();
  __shared__ float red[8];
  const int row = row0 + blockIdx.x, j = blockIdx.y, lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const float* x = X + (size_t)row * ldx;
  const WT* a = A + (size_t)j * K;
  float acc = 0.f;
  for (int k = threadIdx.x * 8; k < K; k += 2048) {
    float w[8];
    load8(a + k, w);
#pragma unroll
    for (int e = 0; e < 8; ++e) acc += w[e] * x[xmap ? xmap[k + e] : (k + e)];
  }
  acc = warp_sum(acc);
  if (lane == 0) red[warp] = acc;
  __syncthreads();
  if (threadIdx.x == 0) {
    float tot = 0.f;
#pragma unroll
    for (int w = 0; w < 8; ++w) tot += red[w];
    U[(size_t)row * ldu + j] = tot;
  }
}

void launch_lora_down(cudaStream_t st, int dtype, const float* X, int ldx, int row0, int rows, int K,
                      const int* xmap, const void* A, int r, float* U, int ldu) {
  if (rows <= 0 || r <= 0) return;
  if (dtype == M2R2_FP32)
    launch_pdl(lora_down_kernel<float>, dim3(rows, r), dim3(256), 0, st, X, ldx, row0, K, xmap, (const float*)A, r, U, ldu);
  else
    launch_pdl(lora_down_kernel<__nv_bfloat16>, dim3(rows, r), dim3(256), 0, st, X, ldx, row0, K, xmap, (const __nv_bfloat16*)A, r, U, ldu);
}

// =====================================================================================
// a2/a5/a6/a7/a8/a9/a16  weight-streaming GEMV / skinny GEMM on CUDA cores.
//   out[row][n] = resid + (addin + scale * (W[n,:] . x[row]))  (+ B[bmap(n),:] . u[row])
// One warp owns NW output rows for RT activation rows; lanes stride K with 128-bit loads;
// the RT activation rows live in shared memory in K-chunks of KC.
// swiglu variant: act[row][n] = silu(Wg[n].x + lora_g) * (Wu[n].x + lora_u)    (a6)
// =====================================================================================
constexpr int GEMV_KC = 1024;
constexpr int GEMV_NW = 2;

template <typename WT, int RT, bool SWIGLU>
__global__ void __launch_bounds__(256) gemv_kernel(GemvArgs a) {
  __shared__ __align__(16) float xs[RT][GEMV_KC];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int row0 = blockIdx.y * RT;
  const int n0 = (blockIdx.x * 8 + warp) * GEMV_NW;
  constexpr int NM = SWIGLU ? 2 : 1;   // matrices per output
  float acc[NM][GEMV_NW][RT];
#pragma unroll
  for (int m = 0; m < NM; ++m)
#pragma unroll
    for (int j = 0; j < GEMV_NW; ++j)
#pragma unroll
      for (int r = 0; r < RT; ++r) acc[m][j][r] = 0.f;

  const WT* W = (const WT*)a.W;
  const WT* W2 = (const WT*)a.W2;
  for (int kc0 = 0; kc0 < a.K; kc0 += GEMV_KC) {
    const int kl = min(GEMV_KC, a.K - kc0);
    __syncthreads();
    for (int i = tid; i < RT * (GEMV_KC / 4); i += 256) {
      int r = i / (GEMV_KC / 4), k4 = (i % (GEMV_KC / 4)) * 4;
      float4 v = make_float4(0.f, 0.f, 0.f, 0.f);
      if (row0 + r < a.n_rows && k4 < kl) v = *(const float4*)(a.X + (size_t)(row0 + r) * a.ldx + kc0 + k4);
      *(float4*)&xs[r][k4] = v;
    }
    __syncthreads();
    for (int k = lane * 8; k < kl; k += 256) {
      float xv[RT][8];
#pragma unroll
      for (int r = 0; r < RT; ++r) {
        float4 x0 = *(const float4*)&xs[r][k], x1 = *(const float4*)&xs[r][k + 4];
        xv[r][0] = x0.x; xv[r][1] = x0.y; xv[r][2] = x0.z; xv[r][3] = x0.w;
        xv[r][4] = x1.x; xv[r][5] = x1.y; xv[r][6] = x1.z; xv[r][7] = x1.w;
      }
#pragma unroll
      for (int j = 0; j < GEMV_NW; ++j) {
        if (n0 + j < a.n_out) {
          float w[8];
          load8(W + (size_t)(n0 + j) * a.K + kc0 + k, w);
#pragma unroll
          for (int r = 0; r < RT; ++r)
#pragma unroll
            for (int e = 0; e < 8; ++e) acc[0][j][r] += w[e] * xv[r][e];
          if (SWIGLU) {
            load8(W2 + (size_t)(n0 + j) * a.K + kc0 + k, w);
#pragma unroll
            for (int r = 0; r < RT; ++r)
#pragma unroll
              for (int e = 0; e < 8; ++e) acc[NM - 1][j][r] += w[e] * xv[r][e];
          }
        }
      }
    }
  }
  // reduce over lanes; lane (j*RT + r) finishes output (n0+j, row0+r)
#pragma unroll
  for (int m = 0; m < NM; ++m)
#pragma unroll
    for (int j = 0; j < GEMV_NW; ++j)
#pragma unroll
      for (int r = 0; r < RT; ++r) acc[m][j][r] = warp_sum(acc[m][j][r]);
  float v0 = 0.f, v1 = 0.f;
#pragma unroll
  for (int j = 0; j < GEMV_NW; ++j)
#pragma unroll
    for (int r = 0; r < RT; ++r)
      if (lane == j * RT + r) {
        v0 = acc[0][j][r];
        v1 = acc[NM - 1][j][r];
      }
  if (lane >= GEMV_NW * RT) return;
  const int n = n0 + lane / RT, row = row0 + lane % RT;
  if (n >= a.n_out || row >= a.n_rows) return;
  // parallel adapter term for accelerated rows
  if (a.Bm != nullptr && row >= a.lora_row0) {
    int bn = a.bmap ? a.bmap[n] : n;
    if (bn >= 0) {
      int usel = a.usel_div ? n / a.usel_div : 0;
      const float* u = a.U + (size_t)row * a.ldu + usel * a.r;
      const WT* b = (const WT*)a.Bm + (size_t)bn * a.r;
      float s = 0.f;
      for (int q = 0; q < a.r; ++q) s += to_f32(b[q]) * u[q];
      v0 += s;
      if (SWIGLU) {
        const float* u2 = a.U + (size_t)row * a.ldu + a.r;
        const WT* b2 = (const WT*)a.Bm2 + (size_t)bn * a.r;
        float s2 = 0.f;
        for (int q = 0; q < a.r; ++q) s2 += to_f32(b2[q]) * u2[q];
        v1 += s2;
      }
    }
  }
  float res;
  if (SWIGLU) {
    res = (v0 / (1.f + __expf(-v0))) * v1;
  } else {
    res = v0;
    if (a.scale) res *= a.scale[(size_t)row * a.scale_ld];
    if (a.addin) res += a.addin[(size_t)row * a.ldo + n];
    if (a.resid) res += a.resid[(size_t)row * a.ldo + n];
  }
  a.out[(size_t)row * a.ldo + n] = res;
  if (a.trace) a.trace[(size_t)row * a.ldo + n] = res;
}

template <typename WT, bool SWIGLU>
static void launch_gemv_t(cudaStream_t st, const GemvArgs& a) {
  int rt = a.n_rows <= 1 ? 1 : a.n_rows <= 2 ? 2 : a.n_rows <= 4 ? 4 : 8;
  dim3 grid((a.n_out + 8 * GEMV_NW - 1) / (8 * GEMV_NW), (a.n_rows + rt - 1) / rt);
  switch (rt) {
    case 1: gemv_kernel<WT, 1, SWIGLU><<<grid, 256, 0, st>>>(a); break;
    case 2: gemv_kernel<WT, 2, SWIGLU><<<grid, 256, 0, st>>>(a); break;
    case 4: gemv_kernel<WT, 4, SWIGLU><<<grid, 256, 0, st>>>(a); break;
    default: gemv_kernel<WT, 8, SWIGLU><<<grid, 256, 0, st>>>(a); break;
  }
}

void launch_gemv(cudaStream_t st, int dtype, const GemvArgs& a, bool swiglu) {
  if (a.n_rows <= 0 || a.n_out <= 0) return;
  if (dtype == M2R2_FP32) {
    if (swiglu) launch_gemv_t<float, true>(st, a); else launch_gemv_t<float, false>(st, a);
  } else {
    if (swiglu) launch_gemv_t<__nv_bfloat16, true>(st, a); else launch_gemv_t<__nv_bfloat16, false>(st, a);
  }
}

// =====================================================================================
// a3  RoPE + KV append.  rope(v, t): pairs (j, j + dh/2), angle t * theta^(-2j/dh) from a host
// double-precision table.  Slow rows store K/V (rounded to the cache dtype) at
// [seq][head][pos][dh]; accelerated rows keep k^, v^ in scratch (never cached).
// =====================================================================================
template <typename KT>
__global__ void rope_append_kernel(float* __restrict__ qkv, int slow_rows, const int* __restrict__ row_seq,
                                   const int* __restrict__ row_pos, const float2* __restrict__ rope_tab,
                                   KT* __restrict__ Kc, KT* __restrict__ Vc, int n_heads, int dh,
                                   int max_seq) {
  pdl_launch_dependents();
  pdl_wait();
  int row = blockIdx.x, head = blockIdx.y, half = dh / 2, d = n_heads * dh;
  int pos = row_pos[row], seq = row_seq[row];
  float* q = qkv + (size_t)row * 3 * d + head * dh;
  float* k = q + d;
  float* v = k + d;
  size_t cbase = (((size_t)seq * n_heads + head) * max_seq + pos) * dh;
  for (int j = threadIdx.x; j < half; j += blockDim.x) {
    float2 cs = rope_tab[(size_t)pos * half + j];
    float a = q[j], b = q[j + half];
    q[j] = a * cs.x - b * cs.y;
    q[j + half] = b * cs.x + a * cs.y;
    a = k[j]; b = k[j + half];
    float k0 = a * cs.x - b * cs.y, k1 = b * cs.x + a * cs.y;
    if (row < slow_rows) {
      Kc[cbase + j] = from_f32<KT>(k0);
      Kc[cbase + j + half] = from_f32<KT>(k1);
      Vc[cbase + j] = from_f32<KT>(v[j]);
      Vc[cbase + j + half] = from_f32<KT>(v[j + half]);
    } else {
      k[j] = k0;
      k[j + half] = k1;
    }
  }
}

void launch_rope_append(cudaStream_t st, int dtype, float* qkv, int rows, int slow_rows, const int* row_seq,
                        const int* row_pos, const float2* rope_tab, void* Kc, void* Vc, int n_heads,
                        int dh, int max_seq) {
  dim3 grid(rows, n_heads);
  if (dtype == M2R2_FP32)
    launch_pdl(rope_append_kernel<float>, grid, dim3(64), 0, st, qkv, slow_rows, row_seq, row_pos, rope_tab, (float*)Kc, (float*)Vc, n_heads, dh, max_seq);
  else
    launch_pdl(rope_append_kernel<__nv_bfloat16>, grid, dim3(64), 0, st, qkv, slow_rows, row_seq, row_pos, rope_tab, (__nv_bfloat16*)Kc, (__nv_bfloat16*)Vc, n_heads, dh, max_seq);
}

// =====================================================================================
// a4 / a11  split-K flash-decode attention, up to M2R2_MAXQ query rows of one sequence sharing
// every K/V tile (slow + accelerated row of a decode step, or the k+1 rows of a verify pass).
// Query row q sees cache positions [0, limit_q).  Online softmax per lane segment, merged
// through shared memory; one (m, l, o) partial per (row, head, split).
// Lane layout: a position's K row (dh elements) is covered by LPP lanes with 16-byte loads;
// SEG = next power of two >= LPP lanes form a segment; a warp handles 32/SEG positions at once.
// =====================================================================================
template <typename KT> struct KVec;
template <> struct KVec<__nv_bfloat16> {
  static constexpr int EPL = 8;
  typedef uint4 Raw;
  static __device__ __forceinline__ Raw zero() { return make_uint4(0u, 0u, 0u, 0u); }
  static __device__ __forceinline__ void unpack(const Raw& u, float out[8]) {
    bf16x2_to_f32(u.x, out[0], out[1]); bf16x2_to_f32(u.y, out[2], out[3]);
    bf16x2_to_f32(u.z, out[4], out[5]); bf16x2_to_f32(u.w, out[6], out[7]);
  }
};
template <> struct KVec<float> {
  static constexpr int EPL = 4;
  typedef float4 Raw;
  static __device__ __forceinline__ Raw zero() { return make_float4(0.f, 0.f, 0.f, 0.f); }
  static __device__ __forceinline__ void unpack(const Raw& u, float out[8]) {
    out[0] = u.x; out[1] = u.y; out[2] = u.z; out[3] = u.w;
    out[4] = out[5] = out[6] = out[7] = 0.f;
  }
};

template <typename KT>
__device__ __forceinline__ void load_kv(const KT* p, float out[8]);
template <>
__device__ __forceinline__ void load_kv<__nv_bfloat16>(const __nv_bfloat16* p, float out[8]) {
  uint4 u = *(const uint4*)p;
  bf16x2_to_f32(u.x, out[0], out[1]);
  bf16x2_to_f32(u.y, out[2], out[3]);
  bf16x2_to_f32(u.z, out[4], out[5]);
  bf16x2_to_f32(u.w, out[6], out[7]);
}
template <>
__device__ __forceinline__ void load_kv<float>(const float* p, float out[8]) {
  float4 u = *(const float4*)p;
  out[0] = u.x; out[1] = u.y; out[2] = u.z; out[3] = u.w;
  out[4] = out[5] = out[6] = out[7] = 0.f;
}

// NQ = query rows compiled in (the group's live rows are packed from slot 0); UN positions per segment are
// loaded before any is used, so a warp keeps 2 * UN 16-byte loads per lane in flight (the K/V stream is the bound).
template <typename KT, int SEG, int NQ>
__global__ void __launch_bounds__(128, NQ <= 5 ? 4 : 3) attn_kernel(AttnArgs a) {
  constexpr int EPL = KVec<KT>::EPL;
  constexpr int NSEG = 4 * (32 / SEG);           // segments per CTA
  constexpr int UN = 4;
  extern __shared__ float sm[];
  const int head = blockIdx.x, grp = blockIdx.y, split = blockIdx.z;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int dh = a.dh, lpp = dh / EPL;
  float* qs = sm;                                // [NQ][dh], pre-scaled
  float* red = sm + NQ * dh;                     // [NSEG][NQ][dh + 2]
  __shared__ int s_row[M2R2_MAXQ], s_lim[M2R2_MAXQ];
  __shared__ int s_seq, s_maxlim;
  const bool accel_head = (a.accel_head_mask[head >> 5] >> (head & 31)) & 1u;
  if (tid < M2R2_MAXQ) {
    int r = a.grp_rows[grp * M2R2_MAXQ + tid];
    if (r >= a.slow_rows && !accel_head) r = -1;  // accelerated rows only use heads in S
    s_row[tid] = r;
    s_lim[tid] = r >= 0 ? a.row_limit[r] : 0;
  }
  __syncthreads();
  if (tid == 0) {
    int mx = 0, sq = 0;
    for (int q = 0; q < NQ; ++q)
      if (s_row[q] >= 0) { mx = max(mx, s_lim[q]); sq = a.row_seq[s_row[q]]; }
    s_maxlim = mx;
    s_seq = sq;
  }
  for (int i = tid; i < NQ * dh; i += 128) {
    int q = i / dh, j = i % dh, r = s_row[q];
    qs[i] = r >= 0 ? a.qkv[(size_t)r * 3 * a.d + head * dh + j] * a.scale : 0.f;
  }
  __syncthreads();
  const int maxlim = s_maxlim;
  const int chunk = (maxlim + a.n_splits - 1) / a.n_splits;
  const int u0 = split * chunk, u1 = min(maxlim, u0 + chunk);
  const KT* Kb = (const KT*)a.Kc + ((size_t)s_seq * a.n_heads + head) * a.max_seq * dh;
  const KT* Vb = (const KT*)a.Vc + ((size_t)s_seq * a.n_heads + head) * a.max_seq * dh;

  const int seg = lane / SEG, sl = lane % SEG;   // segment in warp, lane in segment
  const bool active = sl < lpp;
  float m[NQ], l[NQ], o[NQ][EPL];
  int lim[NQ];
#pragma unroll
  for (int q = 0; q < NQ; ++q) {
    m[q] = -INFINITY; l[q] = 0.f; lim[q] = s_lim[q];
#pragma unroll
    for (int e = 0; e < EPL; ++e) o[q][e] = 0.f;
  }
  // the lane's slice of every query stays in shared memory (broadcast reads): registers hold the running
  // outputs and the raw K/V loads in flight, so that several CTAs fit an SM
  const float* ql = qs + (active ? sl * EPL : 0);
  constexpr int PPW = 32 / SEG;
  typedef typename KVec<KT>::Raw Raw;
  for (int ub = u0 + warp * PPW; ub < u1; ub += 4 * PPW * UN) {
    Raw kraw[UN], vraw[UN];
#pragma unroll
    for (int i = 0; i < UN; ++i) {
      const int u = ub + i * 4 * PPW + seg;
      kraw[i] = KVec<KT>::zero(); vraw[i] = kraw[i];
      if (u < u1 && active) {
        kraw[i] = *(const Raw*)(Kb + (size_t)u * dh + sl * EPL);
        vraw[i] = *(const Raw*)(Vb + (size_t)u * dh + sl * EPL);
      }
    }
#pragma unroll
    for (int i = 0; i < UN; ++i) {
      const int u = ub + i * 4 * PPW + seg;
      const bool valid = u < u1;
      float kv[8], vv[8];
      KVec<KT>::unpack(kraw[i], kv);
      KVec<KT>::unpack(vraw[i], vv);
#pragma unroll
      for (int q = 0; q < NQ; ++q) {
        float s = 0.f;
#pragma unroll
        for (int e = 0; e < EPL; e += 4) {
          const float4 qv = *(const float4*)(ql + q * dh + e);
          s += qv.x * kv[e] + qv.y * kv[e + 1] + qv.z * kv[e + 2] + qv.w * kv[e + 3];
        }
        if (!active) s = 0.f;
#pragma unroll
        for (int off = SEG / 2; off > 0; off >>= 1) s += __shfl_xor_sync(0xffffffffu, s, off);
        if (valid && u < lim[q]) {
          float mn = fmaxf(m[q], s);
          float corr = __expf(m[q] - mn), p = __expf(s - mn);
          l[q] = l[q] * corr + p;
#pragma unroll
          for (int e = 0; e < EPL; ++e) o[q][e] = o[q][e] * corr + p * vv[e];
          m[q] = mn;
        }
      }
    }
  }
  // merge the NSEG running states through shared memory
  const int gseg = warp * PPW + seg;
#pragma unroll
  for (int q = 0; q < NQ; ++q) {
    float* dst = red + ((size_t)gseg * NQ + q) * (dh + 2);
    if (active) {
#pragma unroll
      for (int e = 0; e < EPL; ++e) dst[sl * EPL + e] = o[q][e];
    }
    if (sl == 0) { dst[dh] = m[q]; dst[dh + 1] = l[q]; }
  }
  __syncthreads();
  for (int i = tid; i < NQ * dh; i += 128) {
    int q = i / dh, j = i % dh, r = s_row[q];
    if (r < 0) continue;
    float M = -INFINITY;
    for (int s = 0; s < NSEG; ++s) M = fmaxf(M, red[((size_t)s * NQ + q) * (dh + 2) + dh]);
    float L = 0.f, O = 0.f;
    for (int s = 0; s < NSEG; ++s) {
      const float* src = red + ((size_t)s * NQ + q) * (dh + 2);
      float ls = src[dh + 1];
      if (ls > 0.f) {
        float w = __expf(src[dh] - M);
        L += ls * w;
        O += src[j] * w;
      }
    }
    size_t pidx = ((size_t)r * a.n_heads + head) * a.n_splits + split;
    a.part_o[pidx * dh + j] = O;
    if (j == 0) { a.part_ml[pidx * 2] = M; a.part_ml[pidx * 2 + 1] = L; }
  }
}

// ------------------------------------------------------------------ a11: k-token verification attention on the tensor pipe
// Three to eight query rows of a sequence (the rows of a verify pass or a prefill chunk) against the bf16 K/V cache:
// the scores of 16 positions are one m16n8k16 contraction over d_h per 8 positions (A = the queries, rows 0..7 of the
// tile; B = K rows straight from the cache: each lane's 16-byte loads are its B fragments because the SAME permutation
// of d_h is applied to the queries), P V is a second contraction over the 16 positions (A = the probabilities from the
// score accumulators, B = V through ldmatrix.trans from a staged tile).  Queries and probabilities enter as bf16 hi + lo
// parts (two MMAs, fp32 accumulation): products exact to ~2^-17, as everywhere else on this path.  A warp owns the
// positions u0 + 16 (warp + 4 i); the four warps' online-softmax states meet in shared memory and leave one (m, l, o)
// partial per (row, head, split), exactly what attn_kernel leaves (merge_kernel is shared).
__device__ __forceinline__ void mma_a02(float c[4], uint32_t a0, uint32_t a2, uint32_t b0, uint32_t b1) {
  asm volatile(
      "mma.sync.aligned.m16n8k16.row.col.f32.bf16.bf16.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
      : "+f"(c[0]), "+f"(c[1]), "+f"(c[2]), "+f"(c[3])
      : "r"(a0), "r"(0u), "r"(a2), "r"(0u), "r"(b0), "r"(b1));
}
__device__ __forceinline__ uint32_t pack_bf16_hi_lo(float a, float b, uint32_t& lo) {
  const __nv_bfloat162 h = __floats2bfloat162_rn(a, b);
  const float2 f = __bfloat1622float2(h);
  const __nv_bfloat162 l = __floats2bfloat162_rn(a - f.x, b - f.y);
  lo = *(const uint32_t*)&l;
  return *(const uint32_t*)&h;
}
template <int DH>
__global__ void __launch_bounds__(128) attn_mma_kernel(AttnArgs a) {
  pdl_launch_dependents();
  pdl_wait();
  constexpr int NCC = DH / 32;        // 16-byte chunks of a K row per lane
  constexpr int NKS = DH / 16;        // k-steps of Q K^T
  constexpr int NB = DH / 8;          // n8 column blocks of the output
  constexpr int VLD = DH + 8;         // staged V row stride in elements (+16 bytes: conflict-free ldmatrix)
  extern __shared__ __align__(16) unsigned char am_smem[];
  const int head = blockIdx.x, grp = blockIdx.y, split = blockIdx.z;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, g = lane >> 2, t = lane & 3;
  __nv_bfloat16* vt = (__nv_bfloat16*)am_smem + (size_t)warp * 16 * VLD;   // the warp's staged V tiles [2 buffers][4 warps][16][VLD]
  float* red = (float*)(am_smem + 2 * 4 * 16 * VLD * 2);                  // [4 warps][8 rows][DH + 2]
  __shared__ int s_row[M2R2_MAXQ], s_lim[M2R2_MAXQ];
  __shared__ int s_seq, s_maxlim;
  const bool accel_head = (a.accel_head_mask[head >> 5] >> (head & 31)) & 1u;
  if (tid < M2R2_MAXQ) {
    int r = a.grp_rows[grp * M2R2_MAXQ + tid];
    if (r >= a.slow_rows && !accel_head) r = -1;
    s_row[tid] = r;
    s_lim[tid] = r >= 0 ? a.row_limit[r] : 0;
  }
  __syncthreads();
  if (tid == 0) {
    int mx = 0, sq = 0;
    for (int q = 0; q < M2R2_MAXQ; ++q)
      if (s_row[q] >= 0) { mx = max(mx, s_lim[q]); sq = a.row_seq[s_row[q]]; }
    s_maxlim = mx;
    s_seq = sq;
  }
  __syncthreads();
  const int maxlim = s_maxlim;
  const int chunk = (maxlim + a.n_splits - 1) / a.n_splits;
  const int u0 = split * chunk, u1 = min(maxlim, u0 + chunk);
  const __nv_bfloat16* Kb = (const __nv_bfloat16*)a.Kc + ((size_t)s_seq * a.n_heads + head) * a.max_seq * DH;
  const __nv_bfloat16* Vb = (const __nv_bfloat16*)a.Vc + ((size_t)s_seq * a.n_heads + head) * a.max_seq * DH;
  // the lane's query row g: A fragments (a0, a2) of every k-step, hi and lo parts.  k-step j, slots (2t, 2t+1 | 2t+8,
  // 2t+9) <-> elements 8 (t + 4 (j / 2)) + 4 (j % 2) + {0, 1 | 2, 3} of d_h: the K chunks a lane loads are its B fragments
  const int qrow = s_row[g], lim = s_lim[g];
  uint32_t qh[NKS][2], ql[NKS][2];
#pragma unroll
  for (int j = 0; j < NKS; ++j) {
    float4 v = make_float4(0.f, 0.f, 0.f, 0.f);
    if (qrow >= 0) v = *(const float4*)(a.qkv + (size_t)qrow * 3 * a.d + head * DH + 8 * (t + 4 * (j >> 1)) + 4 * (j & 1));
    qh[j][0] = pack_bf16_hi_lo(v.x * a.scale, v.y * a.scale, ql[j][0]);
    qh[j][1] = pack_bf16_hi_lo(v.z * a.scale, v.w * a.scale, ql[j][1]);
  }
  float m = -INFINITY, l = 0.f, o[NB][4];
#pragma unroll
  for (int nb = 0; nb < NB; ++nb)
#pragma unroll
    for (int e = 0; e < 4; ++e) o[nb][e] = 0.f;
  // software pipeline: the NEXT tile's V rows (cp.async into the other buffer) and K chunks (registers) are requested
  // before this tile is computed
  auto stage_v = [&](int p0, int buf) {   // rows past the split are zero: they meet probability 0, which must not meet a NaN
    __nv_bfloat16* vb = vt + (size_t)buf * 4 * 16 * VLD;
#pragma unroll
    for (int i = lane; i < 16 * (DH / 8); i += 32) {
      const int r = i / (DH / 8), c8 = i - r * (DH / 8);
      __nv_bfloat16* dst = vb + r * VLD + 8 * c8;
      if (p0 + r < u1) asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"((uint32_t)__cvta_generic_to_shared(dst)), "l"(Vb + (size_t)(p0 + r) * DH + 8 * c8) : "memory");
      else *(uint4*)dst = make_uint4(0u, 0u, 0u, 0u);
    }
    asm volatile("cp.async.commit_group;" ::: "memory");
  };
  auto load_k = [&](int p0, uint4 (&kr)[2][NCC]) {   // lane (g, t) loads chunks t, t + 4, .. of row p0 + 8 b + g
#pragma unroll
    for (int b = 0; b < 2; ++b)
#pragma unroll
      for (int cc = 0; cc < NCC; ++cc) {
        kr[b][cc] = make_uint4(0u, 0u, 0u, 0u);
        if (p0 + 8 * b + g < u1) kr[b][cc] = *(const uint4*)(Kb + (size_t)(p0 + 8 * b + g) * DH + 8 * (t + 4 * cc));
      }
  };
  uint4 kr[2][NCC], kn[2][NCC];
  int buf = 0;
  if (u0 + 16 * warp < u1) { stage_v(u0 + 16 * warp, 0); load_k(u0 + 16 * warp, kn); }
  for (int p0 = u0 + 16 * warp; p0 < u1; p0 += 64, buf ^= 1) {
#pragma unroll
    for (int b = 0; b < 2; ++b)
#pragma unroll
      for (int cc = 0; cc < NCC; ++cc) kr[b][cc] = kn[b][cc];
    const bool more = p0 + 64 < u1;
    __syncwarp();   // the other buffer's ldmatrix reads (previous tile) are done in every lane
    if (more) { stage_v(p0 + 64, buf ^ 1); load_k(p0 + 64, kn); }
    // ---- scores: s[b][0], s[b][1] = query g x positions p0 + 8 b + 2 t, + 1
    float s[2][4];
#pragma unroll
    for (int b = 0; b < 2; ++b) {
      s[b][0] = s[b][1] = s[b][2] = s[b][3] = 0.f;
#pragma unroll
      for (int j = 0; j < NKS; ++j) {
        const uint32_t b0 = (j & 1) ? kr[b][j >> 1].z : kr[b][j >> 1].x, b1 = (j & 1) ? kr[b][j >> 1].w : kr[b][j >> 1].y;
        mma_a02(s[b], qh[j][0], qh[j][1], b0, b1);
        mma_a02(s[b], ql[j][0], ql[j][1], b0, b1);
      }
    }
    // ---- online softmax of row g (its four lanes hold four positions each)
    float mt = -INFINITY;
#pragma unroll
    for (int b = 0; b < 2; ++b)
#pragma unroll
      for (int e = 0; e < 2; ++e) {
        const int u = p0 + 8 * b + 2 * t + e;
        if (!(u < u1 && u < lim)) s[b][e] = -INFINITY;
        mt = fmaxf(mt, s[b][e]);
      }
    mt = fmaxf(mt, __shfl_xor_sync(0xffffffffu, mt, 1));
    mt = fmaxf(mt, __shfl_xor_sync(0xffffffffu, mt, 2));
    const float mn = fmaxf(m, mt);
    const float corr = mn == -INFINITY ? 1.f : __expf(m - mn);
    float p[2][2];
#pragma unroll
    for (int b = 0; b < 2; ++b)
#pragma unroll
      for (int e = 0; e < 2; ++e) p[b][e] = s[b][e] == -INFINITY ? 0.f : __expf(s[b][e] - mn);
    l = l * corr + (p[0][0] + p[0][1]) + (p[1][0] + p[1][1]);
    m = mn;
#pragma unroll
    for (int nb = 0; nb < NB; ++nb) { o[nb][0] *= corr; o[nb][1] *= corr; }
    uint32_t pl0, pl1;
    const uint32_t ph0 = pack_bf16_hi_lo(p[0][0], p[0][1], pl0), ph1 = pack_bf16_hi_lo(p[1][0], p[1][1], pl1);
    // ---- o += P V: B fragments of V through ldmatrix.trans (rows 0-7 | 8-15 of the tile, 8 columns)
    if (more) asm volatile("cp.async.wait_group 1;" ::: "memory"); else asm volatile("cp.async.wait_group 0;" ::: "memory");
    __syncwarp();
    const uint32_t vaddr = (uint32_t)__cvta_generic_to_shared(vt + (size_t)buf * 4 * 16 * VLD + (lane & 15) * VLD);
#pragma unroll
    for (int nb = 0; nb < NB; ++nb) {
      uint32_t b0, b1;
      asm volatile("ldmatrix.sync.aligned.m8n8.x2.trans.shared.b16 {%0, %1}, [%2];" : "=r"(b0), "=r"(b1) : "r"(vaddr + nb * 16));
      mma_a02(o[nb], ph0, ph1, b0, b1);
      mma_a02(o[nb], pl0, pl1, b0, b1);
    }
  }
  // ---- the four warps' states -> one partial per query row
  l += __shfl_xor_sync(0xffffffffu, l, 1);
  l += __shfl_xor_sync(0xffffffffu, l, 2);
  __syncthreads();   // every warp is done with its staged tile (red does not alias it, but s_row / s_lim stay live)
  {
    float* dst = red + ((size_t)warp * 8 + g) * (DH + 2);
#pragma unroll
    for (int nb = 0; nb < NB; ++nb) { dst[8 * nb + 2 * t] = o[nb][0]; dst[8 * nb + 2 * t + 1] = o[nb][1]; }
    if (t == 0) { dst[DH] = m; dst[DH + 1] = l; }
  }
  __syncthreads();
  for (int i = tid; i < 8 * DH; i += 128) {
    const int q = i / DH, j = i % DH, r = s_row[q];
    if (r < 0) continue;
    float M = -INFINITY;
    for (int w = 0; w < 4; ++w) M = fmaxf(M, red[((size_t)w * 8 + q) * (DH + 2) + DH]);
    float L = 0.f, O = 0.f;
    for (int w = 0; w < 4; ++w) {
      const float* src = red + ((size_t)w * 8 + q) * (DH + 2);
      const float ls = src[DH + 1];
      if (ls > 0.f) {
        const float wgt = __expf(src[DH] - M);
        L += ls * wgt;
        O += src[j] * wgt;
      }
    }
    if (a.direct_out) {   // one split, slow rows only: this IS the merged output (merge_kernel's O / L)
      a.direct_out[(size_t)r * a.d + head * DH + j] = O / L;
      continue;
    }
    const size_t pidx = ((size_t)r * a.n_heads + head) * a.n_splits + split;
    a.part_o[pidx * DH + j] = O;
    if (j == 0) { a.part_ml[pidx * 2] = M; a.part_ml[pidx * 2 + 1] = L; }
  }
}
template <int DH>
static void launch_attn_mma(cudaStream_t st, const AttnArgs& a, dim3 grid) {
  const size_t sh = (size_t)2 * 4 * 16 * (DH + 8) * 2 + (size_t)4 * 8 * (DH + 2) * sizeof(float);
  static bool attr_set = false;
  if (!attr_set) {
    cudaFuncSetAttribute(attn_mma_kernel<DH>, cudaFuncAttributeMaxDynamicSharedMemorySize, 64 * 1024);
    attr_set = true;
  }
  launch_pdl(attn_mma_kernel<DH>, grid, dim3(128), sh, st, a);
}

template <typename KT, int SEG>
static void launch_attn_nq(cudaStream_t st, const AttnArgs& a, dim3 grid, int nq) {
  const int nseg = 4 * (32 / SEG);
#define ATTN_CASE(NQ)                                                                          \
  {                                                                                            \
    static bool attr_set = false;                                                              \
    if (!attr_set) {                                                                           \
      cudaFuncSetAttribute(attn_kernel<KT, SEG, NQ>, cudaFuncAttributeMaxDynamicSharedMemorySize, 160 * 1024); \
      attr_set = true;                                                                         \
    }                                                                                          \
    size_t sh = ((size_t)NQ * a.dh + (size_t)nseg * NQ * (a.dh + 2)) * sizeof(float);          \
    attn_kernel<KT, SEG, NQ><<<grid, 128, sh, st>>>(a);                                        \
  }
  if (nq <= 2) ATTN_CASE(2) else if (nq <= 4) ATTN_CASE(4) else if (nq <= 5) ATTN_CASE(5) else if (nq <= 6) ATTN_CASE(6) else ATTN_CASE(8)
#undef ATTN_CASE
}

// rows_per_group: live query rows of a group (<= M2R2_MAXQ), packed from slot 0 of grp_rows
bool launch_attn(cudaStream_t st, int dtype, const AttnArgs& a_in, int n_groups, int rows_per_group) {
  AttnArgs a = a_in;
  dim3 grid(a.n_heads, n_groups, a.n_splits);
  const bool direct = a.direct_out != nullptr && a.n_splits == 1 && dtype != M2R2_FP32 && rows_per_group >= 2 &&
                      (a.dh == 64 || a.dh == 96 || a.dh == 128);
  if (!direct) a.direct_out = nullptr;
  if (dtype != M2R2_FP32 && rows_per_group >= 2) {   // k-token verification attention: tensor pipe (bf16 cache)
    if (a.dh == 64) { launch_attn_mma<64>(st, a, grid); return direct; }
    if (a.dh == 96) { launch_attn_mma<96>(st, a, grid); return direct; }
    if (a.dh == 128) { launch_attn_mma<128>(st, a, grid); return direct; }
  }
  int epl = dtype == M2R2_FP32 ? 4 : 8;
  int lpp = a.dh / epl;
  int seg = lpp <= 4 ? 4 : lpp <= 8 ? 8 : lpp <= 16 ? 16 : 32;
  if (dtype == M2R2_FP32) {
    if (seg == 4) launch_attn_nq<float, 4>(st, a, grid, rows_per_group);
    else if (seg == 8) launch_attn_nq<float, 8>(st, a, grid, rows_per_group);
    else if (seg == 16) launch_attn_nq<float, 16>(st, a, grid, rows_per_group);
    else launch_attn_nq<float, 32>(st, a, grid, rows_per_group);
  } else {
    if (seg == 4) launch_attn_nq<__nv_bfloat16, 4>(st, a, grid, rows_per_group);
    else if (seg == 8) launch_attn_nq<__nv_bfloat16, 8>(st, a, grid, rows_per_group);
    else if (seg == 16) launch_attn_nq<__nv_bfloat16, 16>(st, a, grid, rows_per_group);
    else launch_attn_nq<__nv_bfloat16, 32>(st, a, grid, rows_per_group);
  }
  return false;
}

// ------------------------------------------------------------------ accelerated attention over the slow stream's top-k positions
// PAPER.md L158, footnote 4 L170 (k = 64), Q21.  One CTA per (accelerated head, sequence):
//   1. the SLOW query's scores q_h . K_h[u] / sqrt(d_h) over the cached positions u < t,
//   2. the k largest (ties: lower position) by k rounds of a block-wide arg-max,
//   3. the accelerated query's own softmax over those positions plus its own k^_t, v^_t (L76), written to attn_o.
// A correctness path: on this hardware the dense accelerated query rides on the slow query's K/V tiles for free, so the
// fused kernel keeps it dense and a model with accel_topk_tokens > 0 runs the per-operation kernels.
struct TopkAttnArgs {
  const float* qkv;      // [rows][3d], rotated; slow row b, accelerated row B + b
  const void *Kc, *Vc;   // this layer's cache [B][n_heads][max_seq][dh]
  const int* row_limit;  // [rows]: cached positions visible to the accelerated row = t
  const int* accel_heads;// [n_accel] head ids (device)
  float* out;            // attn_o [rows][d]
  int B, n_heads, dh, d, max_seq, topk;
  float scale;
};
template <typename KT>
__global__ void __launch_bounds__(256) accel_topk_attn_kernel(TopkAttnArgs a) {
  extern __shared__ float tk_sm[];
  const int head = a.accel_heads[blockIdx.x], b = blockIdx.y, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int dh = a.dh, t = a.row_limit[a.B + b], k = a.topk;
  float* sc = tk_sm;                       // [max(t, 1)] slow scores
  float* qs = sc + ((t + 3) & ~3) + 4;     // [dh] slow query, [dh] accelerated query
  float* qa = qs + dh;
  float* p = qa + dh;                      // [k + 1] accelerated scores / probabilities
  int* sel = (int*)(p + k + 1);            // [k] selected positions
  __shared__ float rv[8];
  __shared__ int ri[8];
  __shared__ float s_bc[2];
  const KT* Kb = (const KT*)a.Kc + ((size_t)b * a.n_heads + head) * a.max_seq * dh;
  const KT* Vb = (const KT*)a.Vc + ((size_t)b * a.n_heads + head) * a.max_seq * dh;
  const float* qrow = a.qkv + (size_t)b * 3 * a.d + head * dh;
  const float* arow = a.qkv + (size_t)(a.B + b) * 3 * a.d + head * dh;
  for (int j = tid; j < dh; j += 256) { qs[j] = qrow[j]; qa[j] = arow[j]; }
  __syncthreads();
  const int nsel = min(t, k);
  if (t > k) {
    for (int u = tid; u < t; u += 256) {
      float acc = 0.f;
      for (int j = 0; j < dh; ++j) acc += qs[j] * to_f32(Kb[(size_t)u * dh + j]);
      sc[u] = acc * a.scale;
    }
    __syncthreads();
    for (int r = 0; r < k; ++r) {
      float bv = -INFINITY;
      int bi = 0x7fffffff;
      for (int u = tid; u < t; u += 256) {
        const float v = sc[u];
        if (v > bv || (v == bv && u < bi)) { bv = v; bi = u; }
      }
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) {
        const float ov = __shfl_xor_sync(0xffffffffu, bv, o);
        const int oi = __shfl_xor_sync(0xffffffffu, bi, o);
        if (ov > bv || (ov == bv && oi < bi)) { bv = ov; bi = oi; }
      }
      if (lane == 0) { rv[warp] = bv; ri[warp] = bi; }
      __syncthreads();
      if (tid == 0) {
        for (int w = 1; w < 8; ++w)
          if (rv[w] > rv[0] || (rv[w] == rv[0] && ri[w] < ri[0])) { rv[0] = rv[w]; ri[0] = ri[w]; }
        sel[r] = ri[0];
        sc[ri[0]] = -INFINITY;   // taken (scores are finite: -inf never competes)
      }
      __syncthreads();
    }
  } else {
    for (int u = tid; u < t; u += 256) sel[u] = u;
    __syncthreads();
  }
  // accelerated scores on the selected positions and on the token's own key
  for (int i = tid; i <= nsel; i += 256) {
    float acc = 0.f;
    if (i < nsel) { for (int j = 0; j < dh; ++j) acc += qa[j] * to_f32(Kb[(size_t)sel[i] * dh + j]); }
    else { for (int j = 0; j < dh; ++j) acc += qa[j] * arow[a.d + j]; }
    p[i] = acc * a.scale;
  }
  __syncthreads();
  if (tid == 0) {
    float mx = p[0];
    for (int i = 1; i <= nsel; ++i) mx = fmaxf(mx, p[i]);
    float sum = 0.f;
    for (int i = 0; i <= nsel; ++i) { p[i] = __expf(p[i] - mx); sum += p[i]; }
    s_bc[0] = 1.f / sum;
  }
  __syncthreads();
  for (int j = tid; j < dh; j += 256) {
    float acc = 0.f;
    for (int i = 0; i < nsel; ++i) acc += p[i] * to_f32(Vb[(size_t)sel[i] * dh + j]);
    acc += p[nsel] * arow[2 * a.d + j];
    a.out[(size_t)(a.B + b) * a.d + head * dh + j] = acc * s_bc[0];
  }
}
void launch_accel_topk_attn(cudaStream_t st, int dtype, const float* qkv, const void* Kc, const void* Vc, const int* row_limit,
                            const int* accel_heads, int n_accel, float* out, int B, int n_heads, int dh, int d, int max_seq,
                            int topk, float scale) {
  TopkAttnArgs a;
  a.qkv = qkv; a.Kc = Kc; a.Vc = Vc; a.row_limit = row_limit; a.accel_heads = accel_heads; a.out = out;
  a.B = B; a.n_heads = n_heads; a.dh = dh; a.d = d; a.max_seq = max_seq; a.topk = topk; a.scale = scale;
  const size_t sh = ((size_t)((max_seq + 3) & ~3) + 4 + 2 * dh + topk + 1 + topk) * sizeof(float);
  dim3 grid(n_accel, B);
  if (dtype == M2R2_FP32) {
    static bool set = false;
    if (!set) { cudaFuncSetAttribute(accel_topk_attn_kernel<float>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024); set = true; }
    accel_topk_attn_kernel<float><<<grid, 256, sh, st>>>(a);
  } else {
    static bool set = false;
    if (!set) { cudaFuncSetAttribute(accel_topk_attn_kernel<__nv_bfloat16>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024); set = true; }
    accel_topk_attn_kernel<__nv_bfloat16><<<grid, 256, sh, st>>>(a);
  }
}

// merge of the split partials; accelerated rows add their own (k^_t, v^_t) as one more key:
//   MHA(p_t, h_<t (+) p_t, h_<t (+) p_t)
__global__ void merge_kernel(MergeArgs a) {
  pdl_launch_dependents();
  pdl_wait();
  const int row = blockIdx.x, head = blockIdx.y, j = threadIdx.x, dh = a.dh;
  const bool is_accel = row >= a.slow_rows;
  const bool accel_head = (a.accel_head_mask[head >> 5] >> (head & 31)) & 1u;
  float* out = a.out + (size_t)row * a.d + head * dh;
  if (is_accel && !accel_head) {
    if (j < dh) out[j] = 0.f;
    return;
  }
  __shared__ float red[4];
  float M = -INFINITY;
  size_t pbase = ((size_t)row * a.n_heads + head) * a.n_splits;
  for (int s = 0; s < a.n_splits; ++s)
    if (a.part_ml[(pbase + s) * 2 + 1] > 0.f) M = fmaxf(M, a.part_ml[(pbase + s) * 2]);
  float s_own = 0.f;
  if (is_accel) {
    const float* q = a.qkv + (size_t)row * 3 * a.d + head * dh;
    float part = j < dh ? q[j] * q[a.d + j] : 0.f;
    part = warp_sum(part);
    if ((j & 31) == 0) red[j >> 5] = part;
    __syncthreads();
    float tot = 0.f;
    for (int w = 0; w < (dh + 31) / 32; ++w) tot += red[w];
    s_own = tot * a.scale;
    M = fmaxf(M, s_own);
  }
  if (j >= dh) return;
  float L = 0.f, O = 0.f;
  for (int s = 0; s < a.n_splits; ++s) {
    float ls = a.part_ml[(pbase + s) * 2 + 1];
    if (ls > 0.f) {
      float w = __expf(a.part_ml[(pbase + s) * 2] - M);
      L += ls * w;
      O += a.part_o[(pbase + s) * dh + j] * w;
    }
  }
  if (is_accel) {
    float w = __expf(s_own - M);
    L += w;
    O += w * a.qkv[(size_t)row * 3 * a.d + 2 * a.d + head * dh + j];
  }
  out[j] = O / L;
}

void launch_merge(cudaStream_t st, const MergeArgs& a, int rows) {
  dim3 grid(rows, a.n_heads);
  launch_pdl(merge_kernel, grid, dim3(128), 0, st, a);
}

// =====================================================================================
// f-3  Accelerated Residual Latent Attention (Fig. 4a; Q26): one CTA per (gate, sequence).
// States of the interval [E_{j-1}, E_j]: the residual p was re-initialised from at its start (h), then p_i, the last
// one before the gate reset -- all in the step's trace.  K^s, V^s of every state and Q^s of the last one are d^s dot
// products of length d each (a warp per dot product), then a softmax over <= N + 1 states and the sigmoid score.
// =====================================================================================
struct ArlaArgs {
  const float* trace;    // [layer][2][B][d]
  const void* W;         // [n_gates][3 ds + 1][d]
  float* score;          // [B][M2R2_MAX_GATES]
  int gates[M2R2_MAX_GATES];
  int n_gates, ds, d, B;
};
template <typename WT>
__global__ void __launch_bounds__(256) arla_kernel(ArlaArgs a) {
  extern __shared__ float ar_sm[];   // K [n][ds], V [n][ds], q [ds], sc [n]
  const int j = blockIdx.x, b = blockIdx.y, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int lo = j ? a.gates[j - 1] : 0, hi = a.gates[j], n = hi - lo + 1, ds = a.ds, d = a.d;
  float* K = ar_sm;
  float* V = K + (size_t)n * ds;
  float* q = V + (size_t)n * ds;
  float* sc = q + ds;
  const WT* W = (const WT*)a.W + (size_t)j * (3 * ds + 1) * d;
  // dot products: item = (state s, which in {K, V, Q-of-last-state}, e)
  const int items = (2 * n + 1) * ds;
  for (int it = warp; it < items; it += 8) {
    int s, which, e;
    if (it < 2 * n * ds) { s = it / (2 * ds); which = (it / ds) & 1; e = it % ds; } else { s = n - 1; which = 2; e = it - 2 * n * ds; }
    const float* z = a.trace + (((size_t)(lo + s) * 2 + (s == 0 ? 0 : 1)) * a.B + b) * d;
    const WT* w = W + (size_t)((which == 2 ? 0 : (which == 0 ? ds : 2 * ds)) + e) * d;
    float acc = 0.f;
    for (int k = lane; k < d; k += 32) acc += to_f32(w[k]) * z[k];
    acc = warp_sum(acc);
    if (lane == 0) { if (which == 0) K[(size_t)s * ds + e] = acc; else if (which == 1) V[(size_t)s * ds + e] = acc; else q[e] = acc; }
  }
  __syncthreads();
  if (tid < n) {
    float acc = 0.f;
    for (int e = 0; e < ds; ++e) acc += q[e] * K[(size_t)tid * ds + e];
    sc[tid] = acc * rsqrtf((float)ds);
  }
  __syncthreads();
  if (tid == 0) {
    float mx = sc[0];
    for (int s = 1; s < n; ++s) mx = fmaxf(mx, sc[s]);
    float sum = 0.f;
    for (int s = 0; s < n; ++s) { sc[s] = expf(sc[s] - mx); sum += sc[s]; }
    const WT* wo = W + (size_t)(3 * ds) * d;
    float logit = to_f32(wo[ds]);
    for (int e = 0; e < ds; ++e) {
      float ce = 0.f;
      for (int s = 0; s < n; ++s) ce += sc[s] / sum * V[(size_t)s * ds + e];
      logit += to_f32(wo[e]) * ce;
    }
    a.score[(size_t)b * M2R2_MAX_GATES + j] = 1.f / (1.f + expf(-logit));
  }
}
void launch_arla(cudaStream_t st, int dtype, const float* trace, const void* W, const int* gates, int n_gates, int ds, int d, int B,
                 float* score_out) {
  if (n_gates <= 0 || ds <= 0) return;
  ArlaArgs a;
  a.trace = trace; a.W = W; a.score = score_out; a.n_gates = n_gates; a.ds = ds; a.d = d; a.B = B;
  int nmax = 1;
  for (int j = 0; j < n_gates; ++j) { a.gates[j] = gates[j]; nmax = max(nmax, gates[j] - (j ? gates[j - 1] : 0) + 1); }
  const size_t sh = ((size_t)2 * nmax * ds + ds + nmax) * sizeof(float);
  dim3 grid(n_gates, B);
  static bool set = false;
  if (!set) {
    cudaFuncSetAttribute(arla_kernel<float>, cudaFuncAttributeMaxDynamicSharedMemorySize, 160 * 1024);
    cudaFuncSetAttribute(arla_kernel<__nv_bfloat16>, cudaFuncAttributeMaxDynamicSharedMemorySize, 160 * 1024);
    set = true;
  }
  if (dtype == M2R2_FP32) arla_kernel<float><<<grid, 256, sh, st>>>(a);
  else arla_kernel<__nv_bfloat16><<<grid, 256, sh, st>>>(a);
}

// =====================================================================================
// a8/a9  greedy argmax with the logit-script bias hook; lowest index wins ties.
// =====================================================================================
__global__ void __launch_bounds__(1024) argmax_kernel(const float* __restrict__ logits, int ldl, int V,
                                                      const int* __restrict__ row_seq,
                                                      const int* __restrict__ row_pos,
                                                      const int* __restrict__ script, int script_first,
                                                      int script_n, float beta, int* __restrict__ out,
                                                      int out_stride) {
  int row = blockIdx.x;
  const float* lg = logits + (size_t)row * ldl;
  int bidx = -1;
  if (script) {
    int s = row_pos[row] + 1 - script_first;   // logits of the token at pos predict pos+1
    if (s >= 0 && s < script_n) bidx = script[(size_t)row_seq[row] * script_n + s];
  }
  float bv = -INFINITY;
  int bi = 0x7fffffff;
  for (int i = threadIdx.x; i < V; i += 1024) {
    float v = lg[i] + (i == bidx ? beta : 0.f);
    if (v > bv || (v == bv && i < bi)) { bv = v; bi = i; }
  }
#pragma unroll
  for (int off = 16; off > 0; off >>= 1) {
    float ov = __shfl_xor_sync(0xffffffffu, bv, off);
    int oi = __shfl_xor_sync(0xffffffffu, bi, off);
    if (ov > bv || (ov == bv && oi < bi)) { bv = ov; bi = oi; }
  }
  __shared__ float sv[32];
  __shared__ int si[32];
  int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  if (lane == 0) { sv[warp] = bv; si[warp] = bi; }
  __syncthreads();
  if (warp == 0) {
    bv = sv[lane]; bi = si[lane];
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) {
      float ov = __shfl_xor_sync(0xffffffffu, bv, off);
      int oi = __shfl_xor_sync(0xffffffffu, bi, off);
      if (ov > bv || (ov == bv && oi < bi)) { bv = ov; bi = oi; }
    }
    if (lane == 0) out[(size_t)row * out_stride] = bi;
  }
}

void launch_argmax(cudaStream_t st, const float* logits, int ldl, int rows, int V, const int* row_seq,
                   const int* row_pos, const int* script, int script_first, int script_n, float beta,
                   int* out, int out_stride) {
  if (rows <= 0) return;
  argmax_kernel<<<rows, 1024, 0, st>>>(logits, ldl, V, row_seq, row_pos, script, script_first, script_n, beta, out, out_stride);
}

__global__ void copy_rows_kernel(const float* __restrict__ src, float* __restrict__ dst, size_t n) {
  size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) dst[i] = src[i];
}
void launch_copy_rows(cudaStream_t st, const float* src, float* dst, int rows, int d) {
  size_t n = (size_t)rows * d;
  if (n == 0) return;
  copy_rows_kernel<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(src, dst, n);
}

// =====================================================================================
// a13/a14  router / expert predictor: logits = W_r . rms(x; g) (+ script), softmax over all
// experts, top-k (lower index wins ties), renormalise over the selected (Q19).
// One block per row.
// =====================================================================================
template <typename WT>
__global__ void __launch_bounds__(256) route_kernel(const float* __restrict__ X, int ldx, int d,
                                                    const WT* __restrict__ g, float eps, int do_norm,
                                                    const WT* __restrict__ Wr, int n_experts, int top_k,
                                                    int renorm, const int* __restrict__ row_pos,
                                                    const int* __restrict__ script, int script_first,
                                                    int script_n, int n_layers, int layer, float beta,
                                                    int* __restrict__ idx_out, float* __restrict__ w_out) {
  extern __shared__ float sx[];
  __shared__ float red[8];
  __shared__ float lg[M2R2_MAX_EXPERTS];
  int row = blockIdx.x, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const float* x = X + (size_t)row * ldx;
  float ss = 0.f;
  for (int j = tid; j < d; j += 256) { float v = x[j]; sx[j] = v; ss += v * v; }
  ss = warp_sum(ss);
  if (lane == 0) red[warp] = ss;
  __syncthreads();
  if (do_norm) {
    float tot = 0.f;
    for (int w = 0; w < 8; ++w) tot += red[w];
    float inv = rsqrtf(tot / (float)d + eps);
    for (int j = tid; j < d; j += 256) sx[j] = sx[j] * inv * to_f32(g[j]);
    __syncthreads();
  }
  for (int e = warp; e < n_experts; e += 8) {
    const WT* w = Wr + (size_t)e * d;
    float acc = 0.f;
    for (int k = lane * 8; k < d; k += 256) {
      float wv[8];
      load8(w + k, wv);
#pragma unroll
      for (int q = 0; q < 8; ++q) acc += wv[q] * sx[k + q];
    }
    acc = warp_sum(acc);
    if (lane == 0) lg[e] = acc;
  }
  __syncthreads();
  if (tid == 0) {
    if (script) {
      int s = row_pos[row] - script_first;
      if (s >= 0 && s < script_n) {
        const int* pr = script + ((size_t)s * n_layers + layer) * 2;
        lg[pr[0]] += beta;
        lg[pr[1]] += beta - 8.0f;
      }
    }
    float mx = lg[0];
    for (int e = 1; e < n_experts; ++e) mx = fmaxf(mx, lg[e]);
    float sum = 0.f;
    for (int e = 0; e < n_experts; ++e) sum += expf(lg[e] - mx);
    int sel[M2R2_MAX_TOPK];
    float wsum = 0.f;
    for (int k = 0; k < top_k; ++k) {
      int best = -1;
      for (int e = 0; e < n_experts; ++e) {
        bool taken = false;
        for (int q = 0; q < k; ++q) taken |= (sel[q] == e);
        if (taken) continue;
        if (best < 0 || lg[e] > lg[best]) best = e;
      }
      sel[k] = best;
      wsum += expf(lg[best] - mx) / sum;
    }
    for (int k = 0; k < top_k; ++k) {
      float p = expf(lg[sel[k]] - mx) / sum;
      idx_out[(size_t)row * top_k + k] = sel[k];
      w_out[(size_t)row * top_k + k] = renorm ? p / wsum : p;
    }
  }
}

void launch_route(cudaStream_t st, int dtype, const float* X, int ldx, int rows, int d, const void* g,
                  float eps, int do_norm, const void* Wr, int n_experts, int top_k, int renorm,
                  const int* row_pos, const int* script, int script_first, int script_n, int n_layers,
                  int layer, float beta, int* idx_out, float* w_out) {
  if (rows <= 0) return;
  size_t sh = (size_t)d * sizeof(float);
  if (dtype == M2R2_FP32)
    route_kernel<float><<<rows, 256, sh, st>>>(X, ldx, d, (const float*)g, eps, do_norm, (const float*)Wr, n_experts, top_k, renorm, row_pos, script, script_first, script_n, n_layers, layer, beta, idx_out, w_out);
  else
    route_kernel<__nv_bfloat16><<<rows, 256, sh, st>>>(X, ldx, d, (const __nv_bfloat16*)g, eps, do_norm, (const __nv_bfloat16*)Wr, n_experts, top_k, renorm, row_pos, script, script_first, script_n, n_layers, layer, beta, idx_out, w_out);
}
