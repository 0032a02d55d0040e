/*
 * kvr_oracle.c -- ORACLE.  TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * A plain, slow, obviously-correct CPU statement (fp64) of what the hot path
 * of arxiv/paper_2606_17107 computes: RoPE repositioning of a precompiled
 * skill's cached keys plus the splice of its keys and values into a paged
 * destination KV cache.  Only tests/, __graft_entry__.smoke() and the
 * cpu_baseline / --impl reference legs of bench.py may build, load or call
 * anything in this directory.  It shares no code, header, table or helper
 * with the CUDA library (paper_2606_17107_b200/csrc, include/kvr.h); it even
 * uses a different calling convention (flat scalar arguments, one segment per
 * call) so that nothing can be shared by accident.
 *
 * What is computed, and where the paper says so (PAPER.md = /root/reference/PAPER.md
 * at build time; line numbers refer to that file):
 *
 *   PAPER.md:131 (sec. 5, "From mechanism to prediction"): "because the
 *     attention library caches post-RoPE keys, we re-rotate the chunk's keys
 *     from their source positions to the target positions (values are
 *     position-free) before concatenating".
 *   PAPER.md:393 (App. B): "The skill is prefilled once in isolation
 *     (positions 0..L-1), its keys re-rotated to the target offset, and
 *     spliced after the system prompt".
 *   PAPER.md:143 (sec. 5): the pass is O(L) ("a re-rotation pass").
 *   PAPER.md:54, :280 ([28] RoFormer): the rotation is the RoPE rotation.
 *
 * The method reaches exactly (up to rounding) a result that has a plain
 * definition: rotations compose additively, so rotating a key that was
 * RoPE'd at position p by the angle Delta*inv_freq[i] per rotary pair i gives
 * the key RoPE'd at p+Delta.  The oracle is that definition written out
 * (DESIGN.md "Readings" R1..R14 list every point the paper leaves open):
 *
 *   for layer l, kv head h, token t of the segment, rotary pair i < R/2:
 *     Delta_t = new_start - old_start            (or pos_map[t] - (old_start + t))
 *     phi     = (double)Delta_t * inv_freq[i]    one fp64 multiply
 *     (ia,ib) = (i, i + R/2)  NeoX-half   |  (2i, 2i+1)  GPT-J interleaved
 *     a' = a cos(phi) - b sin(phi) ;  b' = b cos(phi) + a sin(phi)      in fp64
 *     elements [R, D) pass through;  V is copied byte for byte
 *     the result is rounded ONCE to the cache dtype (bf16 RNE, or e4m3fn RNE
 *     with saturation after division by the destination scale)
 *     slot: j = dst_token_start + t ; blk = block_table[dst_seq][j / bs] ;
 *           off = j % bs ;  element offset = l*S_l + blk*S_b + off*S_t + h*S_h
 *   Delta_t == 0 (and, in fp8, equal scales) is a byte copy of the K row.
 *   Every destination byte not addressed keeps its prior value.
 *
 * Pins (tests/test_oracle_*.py, all -m "not gpu"): RoPE identity in fp64 and
 * through bf16, Delta=0, Delta then -Delta, norm preservation, the closed
 * form inv_freq = pi/2 (Delta = 1, 2, 4), exhaustive codec checks against
 * ml_dtypes, brute-force slot enumeration with a sentinel-filled pool, and a
 * cross-check of the direct-RoPE helper against the transformers library.
 * kvr_oracle_reposition_inplace (reading R20) is pinned by
 * tests/test_oracle_inplace.py: the pi/2 closed form through brute-force slot
 * enumeration, Delta = 0 leaves every byte, untouched slots and pass-through dims
 * keep their bytes, Delta then -Delta, and the RoPE identity through the pool.
 * kvr_oracle_reposition_splice_ex / _inplace_ex (reading R23, the MLA [latent | k_pe] row) are
 * pinned by tests/test_oracle_adapters.py: the pi/2 closed form at the window's offset pair indices, a numpy RoPE of
 * the k_pe sub-vector with exact-rational rounding, latent bytes equal, the RoPE identity through bf16,
 * exact-rational fp8 requantisation of the latent under a scale change, in-place == splice.
 * Nothing in this file is "parity unpinned".
 *
 * Build: gcc -O2 -std=c11 -fopenmp -shared -fPIC (oracle/build.py).  No
 * -ffast-math, no -mfma-contraction tricks: -ffp-contract=off is passed so
 * that every product below is rounded as written.
 */
#include <math.h>
#include <stdint.h>
#include <string.h>

#define KVRO_OK 0
#define KVRO_ERR_INVALID_ARG (-1)
#define KVRO_ERR_OUT_OF_RANGE (-4)

#define KVRO_BF16 0
#define KVRO_FP8_E4M3 1
#define KVRO_PAIR_NEOX_HALF 0
#define KVRO_PAIR_GPTJ_INTERLEAVED 1
/* Reading R24 (NEXT-4, "splice fused with the suffix-prefill KV write"; "TTFT is a
 * re-rotation pass plus the suffix"): a segment whose keys are NOT yet position-encoded -- freshly projected suffix
 * keys -- is a segment all of whose tokens sit at position old_start (0 for plain pre-RoPE keys, since RoPE at 0 is
 * the identity); token t is rotated to its target position new_start + t (or pos_map[t]):
 * Delta_t = target_t - old_start.  Everything else (pairing, rounding, slots, V) is unchanged. */
#define KVRO_SEG_PRE_ROPE 1

/* ------------------------------------------------------------------ codecs */

/* bf16 = the upper 16 bits of an IEEE binary32 (1 sign, 8 exponent, 7 fraction). */
double kvr_oracle_bf16_decode(uint16_t bits) {
  uint32_t w = (uint32_t)bits << 16;
  float f;
  memcpy(&f, &w, sizeof f);
  return (double)f; /* exact */
}

/* One round-to-nearest-even from fp64 to bf16; subnormals kept (no flush). */
uint16_t kvr_oracle_bf16_encode(double x) {
  uint16_t sign = signbit(x) ? 0x8000u : 0u;
  if (isnan(x)) return (uint16_t)(sign | 0x7FC0u);
  double ax = fabs(x);
  if (ax == 0.0) return sign;
  if (isinf(ax)) return (uint16_t)(sign | 0x7F80u);
  int e;
  (void)frexp(ax, &e);        /* ax = m * 2^e, m in [0.5, 1): leading bit has weight 2^(e-1) */
  int lead = e - 1;
  if (lead < -126) lead = -126; /* below the smallest normal the spacing stays 2^-133 */
  double quantum = ldexp(1.0, lead - 7); /* spacing of bf16 numbers in this binade */
  double r = nearbyint(ax / quantum);    /* exact scaling; ties to even (default FE mode) */
  double v = r * quantum;                /* exactly representable in bf16, or 2^128 */
  if (v >= ldexp(1.0, 128)) return (uint16_t)(sign | 0x7F80u); /* RNE overflow -> inf */
  float f = (float)v;                    /* exact */
  uint32_t w;
  memcpy(&w, &f, sizeof w);
  return (uint16_t)(sign | (uint16_t)(w >> 16));
}

/* e4m3fn: 1 sign, 4 exponent (bias 7), 3 fraction; no infinities; S.1111.111 = NaN;
 * subnormals m * 2^-9; largest finite 1.75 * 2^8 = 448. */
double kvr_oracle_e4m3_decode(uint8_t bits) {
  int s = bits >> 7, e = (bits >> 3) & 0xF, m = bits & 7;
  double v;
  if (e == 15 && m == 7) return s ? -NAN : NAN;
  if (e == 0) v = ldexp((double)m, -9);
  else v = ldexp(1.0 + (double)m / 8.0, e - 7);
  return s ? -v : v;
}

/* Saturating RNE encode: clamp to +-448 first, then round once (reading R7). */
uint8_t kvr_oracle_e4m3_encode_sat(double x) {
  uint8_t sign = signbit(x) ? 0x80u : 0u;
  if (isnan(x)) return (uint8_t)(sign | 0x7Fu);
  double ax = fabs(x);
  if (ax > 448.0) ax = 448.0; /* also maps +-inf to +-448 */
  if (ax == 0.0) return sign;
  int e;
  (void)frexp(ax, &e);
  int lead = e - 1;
  if (lead < -6) lead = -6;              /* subnormal spacing 2^-9 */
  double quantum = ldexp(1.0, lead - 3);
  double r = nearbyint(ax / quantum);    /* ties to even */
  double v = r * quantum;                /* <= 448 because 448 is representable */
  if (v == 0.0) return sign;
  if (v < ldexp(1.0, -6)) {              /* subnormal: v = m * 2^-9, m in 1..7 */
    int m = (int)(v / ldexp(1.0, -9));
    return (uint8_t)(sign | (uint8_t)m);
  }
  (void)frexp(v, &e);
  lead = e - 1;                          /* v = (1 + m/8) * 2^lead */
  int m = (int)((v / ldexp(1.0, lead) - 1.0) * 8.0);
  return (uint8_t)(sign | (uint8_t)(((lead + 7) << 3) | m));
}

/* --------------------------------------------------------------- rotation */

/* Index pair of rotary pair i (reading R1; BASELINE.json north_star (1)). */
static void pair_indices(int pairing, int rotary_dim, int i, int* ia, int* ib) {
  if (pairing == KVRO_PAIR_NEOX_HALF) { *ia = i; *ib = i + rotary_dim / 2; }
  else { *ia = 2 * i; *ib = 2 * i + 1; }
}

/*
 * Pure fp64 rotation of n rows of head_dim doubles, row r by delta[r] positions.
 * This is the arithmetic core, exposed so that the tests can pin it without any
 * storage-format rounding (RoPE identity, norm preservation, closed forms).
 * Applied to a pre-RoPE key with delta = p it IS RoPE at position p
 * (RoFormer [28]): rot(rot(k, p), d) = rot(k, p + d).
 */
int kvr_oracle_rotate_f64(const double* x, double* out, int64_t n, int head_dim,
                          int rotary_dim, int pairing, const double* inv_freq,
                          const int64_t* delta) {
  if (!x || !out || !inv_freq || !delta) return KVRO_ERR_INVALID_ARG;
  if (rotary_dim < 2 || (rotary_dim & 1) || rotary_dim > head_dim) return KVRO_ERR_INVALID_ARG;
  if (pairing != KVRO_PAIR_NEOX_HALF && pairing != KVRO_PAIR_GPTJ_INTERLEAVED) return KVRO_ERR_INVALID_ARG;
  for (int64_t r = 0; r < n; ++r) {
    const double* xr = x + r * head_dim;
    double* yr = out + r * head_dim;
    for (int d = 0; d < head_dim; ++d) yr[d] = xr[d]; /* pass-through dims [R, D) */
    for (int i = 0; i < rotary_dim / 2; ++i) {
      int ia, ib;
      pair_indices(pairing, rotary_dim, i, &ia, &ib);
      double phi = (double)delta[r] * inv_freq[i];
      double c = cos(phi), s = sin(phi);
      double a = xr[ia], b = xr[ib];
      yr[ia] = a * c - b * s;
      yr[ib] = b * c + a * s;
    }
  }
  return KVRO_OK;
}

/* ----------------------------------------------------- reposition + splice */

/*
 * One segment.  All pointers are HOST pointers.  Strides are in ELEMENTS.
 * Layers [layer_begin, layer_end) are processed (the others are left alone), so
 * that a test can check a slice of a large configuration; k_scale_* are indexed
 * [layer * kv_heads + head] with the absolute layer index.
 * n_threads == 1 is the canonical single-thread oracle; > 1 runs the very same
 * loop nest with the (layer, head) loops divided among OpenMP threads (they
 * write disjoint addresses), used only to time the CPU baseline.
 *
 * Returns KVRO_ERR_OUT_OF_RANGE (and writes nothing at all) if any block-table
 * entry the segment touches is < 0 or >= num_blocks (reading R12).
 */
static int splice_core(
    /* model */
    int layers, int kv_heads, int head_dim, int rotary_dim, int rotary_offset, int pairing, int dtype,
    const double* inv_freq,
    /* destination paged pool */
    void* k_cache, void* v_cache,
    int64_t stride_layer, int64_t stride_block, int64_t stride_token, int64_t stride_head,
    int num_blocks, int block_size,
    const int32_t* block_table, int num_seqs, int max_blocks_per_seq,
    const float* k_scale_dst,
    /* the segment */
    const void* k_src, const void* v_src,
    int64_t src_stride_layer, int64_t src_stride_head, int64_t src_stride_token,
    int len, int old_start, int new_start, int dst_seq, int dst_token_start,
    const int32_t* pos_map, const float* k_scale_src, int seg_flags,
    /* control */
    int layer_begin, int layer_end, int n_threads) {
  if (!inv_freq || !k_cache || !block_table || !k_src) return KVRO_ERR_INVALID_ARG;
  if ((v_cache == NULL) != (v_src == NULL)) return KVRO_ERR_INVALID_ARG; /* K-only (reading R23): both absent */
  if (layers <= 0 || kv_heads <= 0 || head_dim <= 0) return KVRO_ERR_INVALID_ARG;
  if (rotary_dim < 2 || (rotary_dim & 1) || rotary_offset < 0 || rotary_offset + rotary_dim > head_dim)
    return KVRO_ERR_INVALID_ARG;
  if (pairing != KVRO_PAIR_NEOX_HALF && pairing != KVRO_PAIR_GPTJ_INTERLEAVED) return KVRO_ERR_INVALID_ARG;
  if (dtype != KVRO_BF16 && dtype != KVRO_FP8_E4M3) return KVRO_ERR_INVALID_ARG;
  if (dtype == KVRO_FP8_E4M3 && !k_scale_dst) return KVRO_ERR_INVALID_ARG;
  if (block_size <= 0 || num_blocks <= 0 || num_seqs <= 0 || max_blocks_per_seq <= 0) return KVRO_ERR_INVALID_ARG;
  if (len <= 0 || dst_seq < 0 || dst_seq >= num_seqs || dst_token_start < 0) return KVRO_ERR_INVALID_ARG;
  if ((int64_t)dst_token_start + len > (int64_t)max_blocks_per_seq * block_size) return KVRO_ERR_INVALID_ARG;
  if (layer_begin < 0 || layer_end > layers || layer_begin > layer_end) return KVRO_ERR_INVALID_ARG;
  if (n_threads < 1 || (seg_flags & ~KVRO_SEG_PRE_ROPE)) return KVRO_ERR_INVALID_ARG;

  const int esz = (dtype == KVRO_BF16) ? 2 : 1;
  const int32_t* table_row = block_table + (int64_t)dst_seq * max_blocks_per_seq;
  if (!k_scale_src) k_scale_src = k_scale_dst; /* NULL = same scales (reading R8) */

  /* Refuse, before writing anything, a segment that touches an unallocated block. */
  for (int t = 0; t < len; ++t) {
    int64_t j = (int64_t)dst_token_start + t;
    int32_t blk = table_row[j / block_size];
    if (blk < 0 || blk >= num_blocks) return KVRO_ERR_OUT_OF_RANGE;
  }

#pragma omp parallel for collapse(2) schedule(static) num_threads(n_threads) if (n_threads > 1)
  for (int l = layer_begin; l < layer_end; ++l) {
    for (int h = 0; h < kv_heads; ++h) {
      const double s_src = (dtype == KVRO_FP8_E4M3) ? (double)k_scale_src[l * kv_heads + h] : 1.0;
      const double s_dst = (dtype == KVRO_FP8_E4M3) ? (double)k_scale_dst[l * kv_heads + h] : 1.0;
      for (int t = 0; t < len; ++t) {
        /* step 1: the position shift of this token */
        int64_t delta = pos_map ? (int64_t)pos_map[t] - ((int64_t)old_start + t)
                                : (int64_t)new_start - (int64_t)old_start;
        if (seg_flags & KVRO_SEG_PRE_ROPE) /* reading R24: every source token sits at old_start, token t goes to target_t */
          delta = (pos_map ? (int64_t)pos_map[t] : (int64_t)new_start + t) - (int64_t)old_start;
        /* step 7: the slot */
        int64_t j = (int64_t)dst_token_start + t;
        int64_t blk = table_row[j / block_size];
        int64_t off = j % block_size;
        int64_t dst_e = (int64_t)l * stride_layer + blk * stride_block + off * stride_token +
                        (int64_t)h * stride_head;
        int64_t src_e = (int64_t)l * src_stride_layer + (int64_t)h * src_stride_head +
                        (int64_t)t * src_stride_token;
        const uint8_t* ks = (const uint8_t*)k_src + src_e * esz;
        uint8_t* kd = (uint8_t*)k_cache + dst_e * esz;

        /* V: position-free, copied unchanged; absent for a latent cache (R23) */
        if (v_src)
          memcpy((uint8_t*)v_cache + dst_e * esz, (const uint8_t*)v_src + src_e * esz, (size_t)head_dim * esz);

        /* K: start from a byte copy -- this is the whole answer for the pass-through
         * dims (outside the rotary window) and for Delta == 0 with equal scales (readings R13, R8) */
        memcpy(kd, ks, (size_t)head_dim * esz);
        if (dtype == KVRO_BF16) {
          if (delta == 0) continue;
          for (int i = 0; i < rotary_dim / 2; ++i) {
            int ia, ib;
            pair_indices(pairing, rotary_dim, i, &ia, &ib);
            ia += rotary_offset; ib += rotary_offset; /* the rotary window starts at rotary_offset (R23) */
            double phi = (double)delta * inv_freq[i];
            double c = cos(phi), s = sin(phi);
            uint16_t ua, ub;
            memcpy(&ua, ks + 2 * ia, 2);
            memcpy(&ub, ks + 2 * ib, 2);
            double a = kvr_oracle_bf16_decode(ua), b = kvr_oracle_bf16_decode(ub);
            uint16_t ra = kvr_oracle_bf16_encode(a * c - b * s);
            uint16_t rb = kvr_oracle_bf16_encode(b * c + a * s);
            memcpy(kd + 2 * ia, &ra, 2);
            memcpy(kd + 2 * ib, &rb, 2);
          }
        } else {
          if (delta == 0 && s_src == s_dst) continue;
          for (int i = 0; i < rotary_dim / 2; ++i) {
            int ia, ib;
            pair_indices(pairing, rotary_dim, i, &ia, &ib);
            ia += rotary_offset; ib += rotary_offset; /* the rotary window starts at rotary_offset (R23) */
            double phi = (double)delta * inv_freq[i];
            double c = (delta == 0) ? 1.0 : cos(phi), s = (delta == 0) ? 0.0 : sin(phi);
            double a = kvr_oracle_e4m3_decode(ks[ia]) * s_src;
            double b = kvr_oracle_e4m3_decode(ks[ib]) * s_src;
            kd[ia] = kvr_oracle_e4m3_encode_sat((a * c - b * s) / s_dst);
            kd[ib] = kvr_oracle_e4m3_encode_sat((b * c + a * s) / s_dst);
          }
          if (s_src != s_dst) /* pass-through dims are re-expressed in the new scale */
            for (int d = 0; d < head_dim; ++d)
              if (d < rotary_offset || d >= rotary_offset + rotary_dim)
                kd[d] = kvr_oracle_e4m3_encode_sat(kvr_oracle_e4m3_decode(ks[d]) * s_src / s_dst);
        }
      }
    }
  }
  return KVRO_OK;
}


/* The hot path as BASELINE.json states it: rotary dims [0, R), K and V both present. */
int kvr_oracle_reposition_splice(
    int layers, int kv_heads, int head_dim, int rotary_dim, int pairing, int dtype, const double* inv_freq,
    void* k_cache, void* v_cache,
    int64_t stride_layer, int64_t stride_block, int64_t stride_token, int64_t stride_head,
    int num_blocks, int block_size, const int32_t* block_table, int num_seqs, int max_blocks_per_seq,
    const float* k_scale_dst,
    const void* k_src, const void* v_src,
    int64_t src_stride_layer, int64_t src_stride_head, int64_t src_stride_token,
    int len, int old_start, int new_start, int dst_seq, int dst_token_start,
    const int32_t* pos_map, const float* k_scale_src,
    int layer_begin, int layer_end, int n_threads) {
  if (!v_cache || !v_src) return KVRO_ERR_INVALID_ARG;
  return splice_core(layers, kv_heads, head_dim, rotary_dim, 0, pairing, dtype, inv_freq, k_cache, v_cache,
                     stride_layer, stride_block, stride_token, stride_head, num_blocks, block_size, block_table,
                     num_seqs, max_blocks_per_seq, k_scale_dst, k_src, v_src, src_stride_layer, src_stride_head,
                     src_stride_token, len, old_start, new_start, dst_seq, dst_token_start, pos_map, k_scale_src,
                     0, layer_begin, layer_end, n_threads);
}

/*
 * NEXT-3 representation adapter (reading R23).  PAPER.md:215 (sec. 8): "MLA (DeepSeek-V2/Coder-V2) caches a
 * position-free latent plus a small decoupled-RoPE sub-vector; our decoupled k_pe reposition re-rotates only that
 * sub-vector"; PAPER.md:514 (Fig. 22a): "repositioning re-rotates only k_pe and copies the latent as-is".
 * A cached row is [latent c_t | k_pe]: the rotary pairs live in dims [rotary_offset, rotary_offset + rotary_dim)
 * and every other dim is copied unchanged; such a cache has no separate V tensor (v_cache == v_src == NULL).
 * Same definition otherwise; rotary_offset = 0 with V present is kvr_oracle_reposition_splice.
 */
int kvr_oracle_reposition_splice_ex(
    int layers, int kv_heads, int head_dim, int rotary_dim, int rotary_offset, int pairing, int dtype,
    const double* inv_freq,
    void* k_cache, void* v_cache,
    int64_t stride_layer, int64_t stride_block, int64_t stride_token, int64_t stride_head,
    int num_blocks, int block_size, const int32_t* block_table, int num_seqs, int max_blocks_per_seq,
    const float* k_scale_dst,
    const void* k_src, const void* v_src,
    int64_t src_stride_layer, int64_t src_stride_head, int64_t src_stride_token,
    int len, int old_start, int new_start, int dst_seq, int dst_token_start,
    const int32_t* pos_map, const float* k_scale_src, int seg_flags,
    int layer_begin, int layer_end, int n_threads) {
  return splice_core(layers, kv_heads, head_dim, rotary_dim, rotary_offset, pairing, dtype, inv_freq, k_cache,
                     v_cache, stride_layer, stride_block, stride_token, stride_head, num_blocks, block_size,
                     block_table, num_seqs, max_blocks_per_seq, k_scale_dst, k_src, v_src, src_stride_layer,
                     src_stride_head, src_stride_token, len, old_start, new_start, dst_seq, dst_token_start,
                     pos_map, k_scale_src, seg_flags, layer_begin, layer_end, n_threads);
}

/* ------------------------------------------------- in-place reposition (NEXT-1) */

/*
 * Re-rotation of a chunk that is ALREADY RESIDENT in the paged pool (reading R20).
 *   PAPER.md:528 (App. H): "the user-memory chunk is precompiled once in isolation and
 *     RoPE-repositioned to float just before the query each turn (an O(L_mem) re-rotation,
 *     no re-prefill)";  PAPER.md:167 (sec. 7): the chunk is re-floated every turn.
 * The chunk occupies logical tokens [token_start, token_start + len) of block-table row `seq`.
 * Every K row of it is decoded, rotated by Delta_t exactly as in the splice (same readings R1,
 * R6, R7, R13), rounded once, and written back to the slot it came from.  V is position-free
 * and is not touched: there is no V argument.  fp8: the pool's scale is both the
 * source and the destination scale.  Delta_t == 0 leaves the row's bytes alone.
 * Returns KVRO_ERR_OUT_OF_RANGE, writing nothing, if a touched block-table entry is invalid.
 */
static int inplace_core(
    int layers, int kv_heads, int head_dim, int rotary_dim, int rotary_offset, int pairing, int dtype,
    const double* inv_freq,
    void* k_cache,
    int64_t stride_layer, int64_t stride_block, int64_t stride_token, int64_t stride_head,
    int num_blocks, int block_size,
    const int32_t* block_table, int num_seqs, int max_blocks_per_seq,
    const float* k_scale,
    int seq, int token_start, int len, int old_start, int new_start, const int32_t* pos_map,
    int layer_begin, int layer_end, int n_threads) {
  if (!inv_freq || !k_cache || !block_table) return KVRO_ERR_INVALID_ARG;
  if (layers <= 0 || kv_heads <= 0 || head_dim <= 0) return KVRO_ERR_INVALID_ARG;
  if (rotary_dim < 2 || (rotary_dim & 1) || rotary_offset < 0 || rotary_offset + rotary_dim > head_dim)
    return KVRO_ERR_INVALID_ARG;
  if (pairing != KVRO_PAIR_NEOX_HALF && pairing != KVRO_PAIR_GPTJ_INTERLEAVED) return KVRO_ERR_INVALID_ARG;
  if (dtype != KVRO_BF16 && dtype != KVRO_FP8_E4M3) return KVRO_ERR_INVALID_ARG;
  if (dtype == KVRO_FP8_E4M3 && !k_scale) return KVRO_ERR_INVALID_ARG;
  if (block_size <= 0 || num_blocks <= 0 || num_seqs <= 0 || max_blocks_per_seq <= 0) return KVRO_ERR_INVALID_ARG;
  if (len <= 0 || seq < 0 || seq >= num_seqs || token_start < 0) return KVRO_ERR_INVALID_ARG;
  if ((int64_t)token_start + len > (int64_t)max_blocks_per_seq * block_size) return KVRO_ERR_INVALID_ARG;
  if (layer_begin < 0 || layer_end > layers || layer_begin > layer_end) return KVRO_ERR_INVALID_ARG;
  if (n_threads < 1) return KVRO_ERR_INVALID_ARG;

  const int esz = (dtype == KVRO_BF16) ? 2 : 1;
  const int32_t* table_row = block_table + (int64_t)seq * max_blocks_per_seq;
  for (int t = 0; t < len; ++t) {
    int32_t blk = table_row[((int64_t)token_start + t) / block_size];
    if (blk < 0 || blk >= num_blocks) return KVRO_ERR_OUT_OF_RANGE;
  }

#pragma omp parallel for collapse(2) schedule(static) num_threads(n_threads) if (n_threads > 1)
  for (int l = layer_begin; l < layer_end; ++l) {
    for (int h = 0; h < kv_heads; ++h) {
      const double sc = (dtype == KVRO_FP8_E4M3) ? (double)k_scale[l * kv_heads + h] : 1.0;
      for (int t = 0; t < len; ++t) {
        int64_t delta = pos_map ? (int64_t)pos_map[t] - ((int64_t)old_start + t)
                                : (int64_t)new_start - (int64_t)old_start;
        if (delta == 0) continue;                       /* reading R13: bytes stay as they are */
        int64_t j = (int64_t)token_start + t;
        int64_t blk = table_row[j / block_size];
        int64_t off = j % block_size;
        uint8_t* row = (uint8_t*)k_cache + ((int64_t)l * stride_layer + blk * stride_block +
                                            off * stride_token + (int64_t)h * stride_head) * esz;
        for (int i = 0; i < rotary_dim / 2; ++i) {
          int ia, ib;
          pair_indices(pairing, rotary_dim, i, &ia, &ib);
          ia += rotary_offset; ib += rotary_offset;
          double phi = (double)delta * inv_freq[i];
          double c = cos(phi), s = sin(phi);
          if (dtype == KVRO_BF16) {
            uint16_t ua, ub;
            memcpy(&ua, row + 2 * ia, 2);
            memcpy(&ub, row + 2 * ib, 2);
            double a = kvr_oracle_bf16_decode(ua), b = kvr_oracle_bf16_decode(ub);
            uint16_t ra = kvr_oracle_bf16_encode(a * c - b * s);
            uint16_t rb = kvr_oracle_bf16_encode(b * c + a * s);
            memcpy(row + 2 * ia, &ra, 2);
            memcpy(row + 2 * ib, &rb, 2);
          } else {
            double a = kvr_oracle_e4m3_decode(row[ia]) * sc;
            double b = kvr_oracle_e4m3_decode(row[ib]) * sc;
            row[ia] = kvr_oracle_e4m3_encode_sat((a * c - b * s) / sc);
            row[ib] = kvr_oracle_e4m3_encode_sat((b * c + a * s) / sc);
          }
        }
      }
    }
  }
  return KVRO_OK;
}

int kvr_oracle_reposition_inplace(
    int layers, int kv_heads, int head_dim, int rotary_dim, int pairing, int dtype, const double* inv_freq,
    void* k_cache, int64_t stride_layer, int64_t stride_block, int64_t stride_token, int64_t stride_head,
    int num_blocks, int block_size, const int32_t* block_table, int num_seqs, int max_blocks_per_seq,
    const float* k_scale,
    int seq, int token_start, int len, int old_start, int new_start, const int32_t* pos_map,
    int layer_begin, int layer_end, int n_threads) {
  return inplace_core(layers, kv_heads, head_dim, rotary_dim, 0, pairing, dtype, inv_freq, k_cache, stride_layer,
                      stride_block, stride_token, stride_head, num_blocks, block_size, block_table, num_seqs,
                      max_blocks_per_seq, k_scale, seq, token_start, len, old_start, new_start, pos_map,
                      layer_begin, layer_end, n_threads);
}

/* In-place re-float of a resident [latent | k_pe] chunk: only the rotary window moves (R23). */
int kvr_oracle_reposition_inplace_ex(
    int layers, int kv_heads, int head_dim, int rotary_dim, int rotary_offset, int pairing, int dtype,
    const double* inv_freq,
    void* k_cache, int64_t stride_layer, int64_t stride_block, int64_t stride_token, int64_t stride_head,
    int num_blocks, int block_size, const int32_t* block_table, int num_seqs, int max_blocks_per_seq,
    const float* k_scale,
    int seq, int token_start, int len, int old_start, int new_start, const int32_t* pos_map,
    int layer_begin, int layer_end, int n_threads) {
  return inplace_core(layers, kv_heads, head_dim, rotary_dim, rotary_offset, pairing, dtype, inv_freq, k_cache,
                      stride_layer, stride_block, stride_token, stride_head, num_blocks, block_size, block_table,
                      num_seqs, max_blocks_per_seq, k_scale, seq, token_start, len, old_start, new_start, pos_map,
                      layer_begin, layer_end, n_threads);
}

/* Algorithmic bytes of one segment: read K, read V, write K, write V. */
uint64_t kvr_oracle_bytes_moved(int layers, int kv_heads, int head_dim, int dtype, int64_t tokens) {
  uint64_t esz = (dtype == KVRO_BF16) ? 2u : 1u;
  return 4u * (uint64_t)layers * (uint64_t)kv_heads * (uint64_t)head_dim * esz * (uint64_t)tokens;
}
