/* m2r2_synth/synth.c — seeded synthetic INPUT generators (weights, prompts, scripts).
 *
 * This module serves both the CPU oracle (oracle/) and the CUDA path
 * (paper_2502_02040_b200/): it produces the bytes both are fed.  It holds NONE of
 * the method's arithmetic (no norm, attention, MLP, routing, LRU ...): only a
 * counter-based PRNG, a Gaussian transform, storage rounding of the generated
 * inputs, and the two "scripts" that BASELINE.json config 3/5 ask for
 * ("acceptance forced to 50% / 90% by seeded logit biasing", "seeded random
 * [router] logits"), which are plain integer tables.
 *
 * Recipe (SURVEY.md §8(d) "Synthetic inputs"):
 *   z      = splitmix64(seed ^ (tensor_id << 40) ^ element_index)
 *   u1,u2  = two 24-bit uniforms from z;  n = sqrt(-2 ln u1) * cos(2 pi u2)
 *   weight = offset + scale * n, rounded RNE to the storage dtype.
 * Stateless per element, so any slice can be generated in parallel.
 */
#include <stdint.h>
#include <stddef.h>
#include <math.h>
#include <string.h>

static inline uint64_t splitmix64(uint64_t x) {
  x += 0x9E3779B97F4A7C15ull;
  x = (x ^ (x >> 30)) * 0xBF58476D1CE4E5B9ull;
  x = (x ^ (x >> 27)) * 0x94D049BB133111EBull;
  return x ^ (x >> 31);
}

static inline uint64_t elem_key(uint64_t seed, uint64_t tensor_id, uint64_t i) {
  return splitmix64(seed ^ (tensor_id << 40) ^ i);
}

static inline float gauss_from_key(uint64_t z) {
  /* u1 in (0,1], u2 in [0,1) */
  double u1 = ((double)((z >> 40) & 0xFFFFFFull) + 1.0) / 16777216.0;
  double u2 = (double)((z >> 16) & 0xFFFFFFull) / 16777216.0;
  return (float)(sqrt(-2.0 * log(u1)) * cos(6.283185307179586476925 * u2));
}

static inline uint16_t f32_to_bf16_rne(float f) {
  uint32_t u;
  memcpy(&u, &f, 4);
  if ((u & 0x7F800000u) == 0x7F800000u) return (uint16_t)(u >> 16); /* inf/nan: truncate */
  u += 0x7FFFu + ((u >> 16) & 1u);
  return (uint16_t)(u >> 16);
}

/* out[i] = offset + scale * normal(seed, tensor_id, first + i), fp32 storage */
void synth_normal_f32(uint64_t seed, uint64_t tensor_id, uint64_t first, uint64_t n, float scale,
                      float offset, float* out) {
#pragma omp parallel for schedule(static)
  for (int64_t i = 0; i < (int64_t)n; ++i)
    out[i] = offset + scale * gauss_from_key(elem_key(seed, tensor_id, first + (uint64_t)i));
}

/* same values, rounded RNE to bf16 storage (raw uint16 bit patterns) */
void synth_normal_bf16(uint64_t seed, uint64_t tensor_id, uint64_t first, uint64_t n, float scale,
                       float offset, uint16_t* out) {
#pragma omp parallel for schedule(static)
  for (int64_t i = 0; i < (int64_t)n; ++i)
    out[i] = f32_to_bf16_rne(offset + scale * gauss_from_key(elem_key(seed, tensor_id, first + (uint64_t)i)));
}

/* i.i.d. uniform tokens on [0, vocab) */
void synth_tokens(uint64_t seed, uint64_t stream, uint64_t n, int32_t vocab, int32_t* out) {
  for (uint64_t i = 0; i < n; ++i)
    out[i] = (int32_t)(elem_key(seed, stream, i) % (uint64_t)vocab);
}

/* Logit script: for every scripted position s (index i = s - first_pos):
 *   full_tok[i]  = f_s uniform token;
 *   draft_tok[i] = f_s with probability alpha, else a different token.
 * The method adds +beta at these indices inside its argmax; nothing of that is done here. */
void synth_logit_script(uint64_t seed, uint64_t stream, uint64_t n, int32_t vocab, double alpha,
                        int32_t* full_tok, int32_t* draft_tok) {
  for (uint64_t i = 0; i < n; ++i) {
    uint64_t a = elem_key(seed, stream * 4 + 0, i);
    uint64_t b = elem_key(seed, stream * 4 + 1, i);
    uint64_t c = elem_key(seed, stream * 4 + 2, i);
    int32_t f = (int32_t)(a % (uint64_t)vocab);
    double u = (double)(b >> 11) / 9007199254740992.0;
    int32_t g = f;
    if (!(u < alpha)) g = (int32_t)(((uint64_t)f + 1 + (c % (uint64_t)(vocab - 1))) % (uint64_t)vocab);
    full_tok[i] = f;
    draft_tok[i] = g;
  }
}

static void fresh_pair(uint64_t key, int32_t n_experts, int32_t* e1, int32_t* e2) {
  int32_t a = (int32_t)(key % (uint64_t)n_experts);
  int32_t b = (int32_t)((key >> 32) % (uint64_t)(n_experts - 1));
  if (b >= a) b += 1;
  *e1 = a;
  *e2 = b;
}

/* Router script: tables [n_steps][n_layers][2].
 *   actual pair  = previous step's pair with probability rho, else a fresh distinct pair;
 *   predicted    = actual with probability pi, else a fresh distinct pair. */
void synth_router_script(uint64_t seed, uint64_t stream, int32_t n_steps, int32_t n_layers,
                         int32_t n_experts, double rho, double pi, int32_t* actual,
                         int32_t* predicted) {
  for (int32_t t = 0; t < n_steps; ++t)
    for (int32_t l = 0; l < n_layers; ++l) {
      uint64_t idx = (uint64_t)t * (uint64_t)n_layers + (uint64_t)l;
      uint64_t k0 = elem_key(seed, stream * 8 + 0, idx);
      uint64_t k1 = elem_key(seed, stream * 8 + 1, idx);
      uint64_t k2 = elem_key(seed, stream * 8 + 2, idx);
      uint64_t k3 = elem_key(seed, stream * 8 + 3, idx);
      int32_t* a = actual + idx * 2;
      int32_t* p = predicted + idx * 2;
      double u = (double)(k0 >> 11) / 9007199254740992.0;
      if (t > 0 && u < rho) {
        a[0] = actual[(idx - (uint64_t)n_layers) * 2 + 0];
        a[1] = actual[(idx - (uint64_t)n_layers) * 2 + 1];
      } else {
        fresh_pair(k1, n_experts, &a[0], &a[1]);
      }
      double v = (double)(k2 >> 11) / 9007199254740992.0;
      if (v < pi) {
        p[0] = a[0];
        p[1] = a[1];
      } else {
        fresh_pair(k3, n_experts, &p[0], &p[1]);
      }
    }
}
