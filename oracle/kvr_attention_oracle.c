/*
 * kvr_attention_oracle.c -- ORACLE.  TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Rotate-on-read (first alternative: "fusing the rotate into a consumer (rotate-on-read in
 * the attention K load ...) so K is never materialised twice"; reading R25).  A decode-step query attends
 * the cached keys and values of precompiled skills WHERE THEY LIE, at the positions they were compiled at; the
 * re-rotation "from their source positions to the target positions" is applied as the keys are read
 * instead of being written back first.  "Values are position-free"; the pass stays O(L)
 * and "works unchanged under FlashAttention / paged attention ... GQA/MQA".
 *
 * The result has a plain definition, which is what this file writes out, in fp64, in the order of the definition:
 *
 *   for query head g (kv head h = g / (q_heads / kv_heads), GQA), segment s, token t < len_s:
 *     K'_{s,t} = R(Delta_s) k_{s,t}      the RoPE re-rotation of kvr_oracle.c: per rotary pair i,
 *                                        phi = (double)Delta_s * inv_freq[i], (a,b) -> (a cos - b sin, b cos + a sin);
 *                                        dims outside the rotary window unchanged; NOT rounded to any storage format
 *     x_{s,t}  = scale * sum_d q_g[d] * K'_{s,t}[d]
 *   m   = max x ;  Z = sum exp(x - m) ;  lse_g = m + ln Z                      (natural logarithm)
 *   o_g = sum_{s,t} exp(x_{s,t} - lse_g) * v_{s,t}                             (softmax-weighted mean of the values)
 *
 * q is the query as the model produced it (already RoPE'd at its own position), k and v are bf16 bit patterns exactly
 * as cached, decoded exactly.  (o_g, lse_g) is the usual partial-attention pair: the caller merges it with the
 * attention over the rest of the context.  The product computes the same scores as (R(-Delta_s) q_g) . k_{s,t};
 * this file deliberately does NOT: it rotates every key, as the definition says.
 *
 * Shares nothing with the CUDA library.  Pins: tests/test_oracle_attention.py (-m "not gpu"): torch's fp64
 * scaled_dot_product_attention over keys re-rotated by an independent complex-exponential RoPE in numpy; the pi/2
 * closed form (Delta = 1 turns (a, b) into (-b, a): scores computed from the permuted integers by hand); the textbook
 * case (keys compiled at 0..L-1 and read at new_start + t equal ordinary RoPE attention at the true positions);
 * q = 0 (uniform weights: o = mean of V, lse = ln n); merge of two single-segment results; GQA head mapping by brute
 * force; strides.  Nothing here is "parity unpinned".
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#define KVRO_OK 0
#define KVRO_ERR_INVALID_ARG (-1)
#define KVRO_PAIR_NEOX_HALF 0
#define KVRO_PAIR_GPTJ_INTERLEAVED 1

static double bf16_value(uint16_t bits) {
  uint32_t w = (uint32_t)bits << 16;
  float f;
  memcpy(&f, &w, sizeof f);
  return (double)f; /* exact */
}

/*
 * One request, one layer.  All pointers are HOST pointers; strides are in ELEMENTS.
 *   q         bf16 bits [q_heads][head_dim]
 *   k_src[s], v_src[s]  bf16 bits of segment s AT THE LAYER ATTENDED: element (h, t, d) at h*stride_head[s] + t*stride_token[s] + d
 *   delta[s]  new_start - old_start of segment s
 *   o         fp64 [q_heads][head_dim],  lse fp64 [q_heads]
 * n_threads > 1 divides the query-head loop among OpenMP threads (disjoint outputs), for timing only.
 */
int kvr_oracle_rotate_on_read_attention(
    const uint16_t* q, int q_heads, int kv_heads, int head_dim, int rotary_dim, int rotary_offset, int pairing,
    const double* inv_freq, double scale,
    int n_segs, const uint16_t* const* k_src, const uint16_t* const* v_src,
    const int64_t* stride_head, const int64_t* stride_token, const int32_t* len, const int32_t* delta,
    double* o, double* lse, int n_threads) {
  if (!q || !inv_freq || !k_src || !v_src || !stride_head || !stride_token || !len || !delta || !o || !lse)
    return KVRO_ERR_INVALID_ARG;
  if (q_heads < 1 || kv_heads < 1 || q_heads % kv_heads || head_dim < 2 || n_segs < 1) return KVRO_ERR_INVALID_ARG;
  if (rotary_dim < 2 || (rotary_dim & 1) || rotary_offset < 0 || rotary_offset + rotary_dim > head_dim) return KVRO_ERR_INVALID_ARG;
  if (pairing != KVRO_PAIR_NEOX_HALF && pairing != KVRO_PAIR_GPTJ_INTERLEAVED) return KVRO_ERR_INVALID_ARG;
  int64_t total = 0;
  for (int s = 0; s < n_segs; ++s) {
    if (len[s] < 1 || !k_src[s] || !v_src[s]) return KVRO_ERR_INVALID_ARG;
    total += len[s];
  }
  const int group = q_heads / kv_heads;
  int fail = 0;
#pragma omp parallel for schedule(static) num_threads(n_threads > 1 ? n_threads : 1)
  for (int g = 0; g < q_heads; ++g) {
    const int h = g / group;
    double* x = (double*)malloc((size_t)total * sizeof(double));   /* every score of this head */
    double* kp = (double*)malloc((size_t)head_dim * sizeof(double));
    if (!x || !kp) {
#pragma omp atomic write
      fail = 1;
      free(x); free(kp); continue;
    }
    /* scores: rotate the key, then the dot product */
    int64_t n = 0;
    for (int s = 0; s < n_segs; ++s)
      for (int t = 0; t < len[s]; ++t) {
        const uint16_t* kr = k_src[s] + (int64_t)h * stride_head[s] + (int64_t)t * stride_token[s];
        for (int d = 0; d < head_dim; ++d) kp[d] = bf16_value(kr[d]);
        for (int i = 0; i < rotary_dim / 2; ++i) {
          int ia, ib;
          if (pairing == KVRO_PAIR_NEOX_HALF) { ia = rotary_offset + i; ib = rotary_offset + i + rotary_dim / 2; }
          else { ia = rotary_offset + 2 * i; ib = rotary_offset + 2 * i + 1; }
          const double phi = (double)delta[s] * inv_freq[i];
          const double c = cos(phi), sn = sin(phi);
          const double a = bf16_value(kr[ia]), b = bf16_value(kr[ib]);
          kp[ia] = a * c - b * sn;
          kp[ib] = b * c + a * sn;
        }
        double dot = 0.0;
        for (int d = 0; d < head_dim; ++d) dot += bf16_value(q[(int64_t)g * head_dim + d]) * kp[d];
        x[n++] = scale * dot;
      }
    /* softmax over every token of every segment */
    double m = x[0];
    for (int64_t j = 1; j < total; ++j) if (x[j] > m) m = x[j];
    double Z = 0.0;
    for (int64_t j = 0; j < total; ++j) Z += exp(x[j] - m);
    lse[g] = m + log(Z);
    for (int d = 0; d < head_dim; ++d) o[(int64_t)g * head_dim + d] = 0.0;
    n = 0;
    for (int s = 0; s < n_segs; ++s)
      for (int t = 0; t < len[s]; ++t) {
        const uint16_t* vr = v_src[s] + (int64_t)h * stride_head[s] + (int64_t)t * stride_token[s];
        const double w = exp(x[n++] - lse[g]);
        for (int d = 0; d < head_dim; ++d) o[(int64_t)g * head_dim + d] += w * bf16_value(vr[d]);
      }
    free(x); free(kp);
  }
  return fail ? KVRO_ERR_INVALID_ARG : KVRO_OK;
}

/* Bytes a rotate-on-read attention call must read (K and V of one layer, once): 2 * kv_heads * head_dim * 2 per token. */
uint64_t kvr_oracle_attention_bytes_read(int kv_heads, int head_dim, int64_t tokens) {
  return (uint64_t)2 * (uint64_t)kv_heads * (uint64_t)head_dim * 2u * (uint64_t)tokens;
}
