// kvr_common.cuh -- device-side structures and arithmetic shared by the kvr CUDA kernels.
// Product code (sm_100a).  Shares nothing with oracle/.
//
// Operation: include/kvr.h.  Arithmetic contract:
//   * the angle phi = (double)Delta * inv_freq[i] and sincos(phi) are evaluated in fp64 once per
//     (segment | token, pair) and kept as fp32 hi + lo parts;
//   * bf16: the rotation is a COMPENSATED fp32 evaluation (error-free product residual + the lo
//     parts), so the result is the fp64 result to ~2^-45 relative before the single bf16 rounding;
//     this is what keeps every element within 2 bf16 ulps even under cancellation;
//   * fp8: dequantise (x = q * s_src), plain fp32 rotate with FMAs, requantise with
//     cvt.rn.satfinite.e4m3x2.f32 after multiplying by 1/s_dst;
//   * Delta == 0 rows are byte copies (bf16 always; fp8 when the scales agree).
#pragma once
#include <cuda_bf16.h>
#include <cuda_fp16.h>
#include <cuda_fp8.h>
#include <cuda.h>            // CUtensorMap (type only; the encoder is fetched through cudaGetDriverEntryPoint)
#include <cuda_runtime.h>
#include <stdint.h>

namespace kvr {

struct SegDev {
  const uint8_t* k_src;
  const uint8_t* v_src;
  const int32_t* pos_map;      // nullptr in segment mode
  const float* k_scale_src;    // never nullptr in fp8 mode (host substitutes the dst scales)
  int64_t sl, sh, st;          // source strides, ELEMENTS
  int64_t unit_begin;          // first scheduled unit of this segment
  int32_t len, old_start, delta;
  int32_t dst_seq, dst_token_start;
  int32_t first_q;             // dst_token_start / cg
  int32_t n_chunks;            // chunks of <= cg tokens, aligned to cg in destination token space
  int32_t index;               // position in the caller's array (for the status word)
  int32_t pre_rope;            // KVR_SEG_PRE_ROPE: every source token sits at old_start (kvr.h)
  int32_t src_stable;          // KVR_SEG_SRC_STABLE: nothing earlier on the stream writes the sources (early loads)
  int32_t pad_;
};

constexpr int kInlineSegs = 8;    // calls with <= this many segments carry their descriptors in the kernel parameters

// TRANSPOSING loads (ring kernel, dense token-major pools): one TMA tensor map per source tensor, dims ordered
// (dim, head, token, layer) -- the head stride is larger than the token stride, which the encoder accepts -- so that a box
// of {head_dim, heads, ct tokens, 1} lands in shared memory as [token][head][dim], i.e. in the pool's own order.
struct TmapPair { CUtensorMap k, v; };
struct TmapInline { TmapPair m[kInlineSegs]; };

struct CallParams {
  // model
  int32_t layers, heads, head_dim, rotary_dim, pairing, dtype;
  const double* inv_freq;      // DEVICE, rotary_dim/2
  int32_t rotary_offset;       // first rotary dim of a row (kvr.h: MLA k_pe window); 0 for ordinary K caches
  int32_t pad0_;
  // destination
  uint8_t* k_cache;
  uint8_t* v_cache;
  int64_t d_sl, d_sb, d_st, d_sh;   // ELEMENTS
  const int32_t* block_table;
  const float* k_scale_dst;
  int32_t num_blocks, block_size, num_seqs, max_blocks;
  // work decomposition
  const SegDev* segs;
  int32_t n_segs;
  int32_t cg;                  // chunk granularity in tokens; cg divides block_size
  int32_t lpu;                 // layers per unit
  int32_t n_lgroups;           // ceil(layers / lpu)
  int64_t total_units;
  int32_t* status;             // DEVICE int32[4]: {flag, segment, token, -}
  int32_t any_pos_map;
  int32_t scales_differ;       // fp8: some segment has its own source scales
  // dynamic unit scheduler (ring kernel): sched[0] = next unit to hand out, sched[1] = CTAs that have finished;
  // both are zero between launches (the last CTA to finish resets them)
  unsigned long long* sched;
  int32_t grab;                // units handed out per atomic
  int32_t hsplit;              // ring kernel: a (chunk, layer group) is split into hsplit units over its head groups
  int32_t tile_min_bytes;      // ring kernel: a tile takes the fewest heads whose K run reaches this many bytes
  int32_t gather;              // ring kernel: gather mode (dense token-major pool; a tile = all heads of a few tokens)
  int32_t no_v;                // V is neither read nor written (in-place calls; K-only [latent | k_pe] caches)
  int32_t inplace;             // kvr_reposition_inplace: K rows are read from the pool slot they are written back to; no V
  int32_t tmajor;              // ring kernel: transposing tensor loads, tiles of ALL heads x ct tokens (see TmapPair)
  int32_t ct;                  // tmajor: tokens per tile (divides cg)
  const TmapPair* tmaps;       // tmajor, > kInlineSegs segments: DEVICE array [n_segs]
  SegDev inline_segs[kInlineSegs];
};

__device__ __forceinline__ const SegDev* seg_array(const CallParams& P) {
  return (P.n_segs <= kInlineSegs) ? P.inline_segs : P.segs;
}

__device__ __forceinline__ int find_segment(const SegDev* __restrict__ segs, int n, int64_t unit) {
  int lo = 0, hi = n - 1;      // last segment with unit_begin <= unit
  while (lo < hi) {
    int mid = (lo + hi + 1) >> 1;
    if (segs[mid].unit_begin <= unit) lo = mid; else hi = mid - 1;
  }
  return lo;
}

struct Chunk { int32_t t0, n_tok, blk_index, off; };  // tokens [t0, t0+n_tok) of the segment; table column; offset in block

__device__ __forceinline__ Chunk chunk_of(const SegDev& s, int32_t c, int32_t cg, int32_t block_size) {
  int64_t q = (int64_t)s.first_q + c;
  int64_t lo = q * cg, hi = lo + cg;
  int64_t a = s.dst_token_start, b = (int64_t)s.dst_token_start + s.len;
  if (lo < a) lo = a;
  if (hi > b) hi = b;
  Chunk ch;
  ch.t0 = (int32_t)(lo - a);
  ch.n_tok = (int32_t)(hi - lo);
  ch.blk_index = (int32_t)(lo / block_size);
  ch.off = (int32_t)(lo % block_size);
  return ch;
}

// Position shift of token i of a segment (kvr.h): new position minus old position.
__device__ __forceinline__ long long token_delta(const SegDev& s, int i) {
  if (s.pre_rope) return (s.pos_map ? (long long)s.pos_map[i] : (long long)s.old_start + s.delta + i) - (long long)s.old_start;
  return s.pos_map ? (long long)s.pos_map[i] - ((long long)s.old_start + i) : (long long)s.delta;
}

__device__ __forceinline__ void report_bad_block(int32_t* status, int32_t seg_index, int32_t token) {
  if (atomicCAS(&status[0], 0, 1) == 0) { status[1] = seg_index; status[2] = token; }
}

// ---- angle -> (cos_hi, cos_lo, sin_hi, sin_lo) ------------------------------------------------
__device__ __forceinline__ float4 angle_entry(int64_t delta, double inv_freq) {
  double phi = (double)delta * inv_freq;     // one fp64 multiply, as the definition states
  double s, c;
  sincos(phi, &s, &c);
  float ch = (float)c, sh = (float)s;
  float cl = (float)(c - (double)ch), sl = (float)(s - (double)sh);
  return make_float4(ch, cl, sh, sl);
}

__device__ __forceinline__ float4 angle_entry_cs(double c, double s) {
  float ch = (float)c, sh = (float)s;
  return make_float4(ch, (float)(c - (double)ch), sh, (float)(s - (double)sh));
}

// ---- compensated rotation (bf16 path) ---------------------------------------------------------
// ra = a*c - b*s ; rb = b*c + a*s with c = t.x + t.y, s = t.z + t.w.
__device__ __forceinline__ void rotate_comp(float a, float b, float4 t, float& ra, float& rb) {
  float p = __fmul_rn(b, t.z);
  float e = __fmaf_rn(b, t.z, -p);                       // b*s_hi = p + e exactly
  float hi = __fmaf_rn(a, t.x, -p);
  float corr = __fmaf_rn(a, t.y, -__fmaf_rn(b, t.w, e));
  ra = __fadd_rn(hi, corr);
  float p2 = __fmul_rn(a, t.z);
  float e2 = __fmaf_rn(a, t.z, -p2);
  float hi2 = __fmaf_rn(b, t.x, p2);
  float corr2 = __fmaf_rn(b, t.y, __fmaf_rn(a, t.w, e2));
  rb = __fadd_rn(hi2, corr2);
}

// ---- plain fp32 rotation (fp8 path) -------------------------------------------------------------
__device__ __forceinline__ void rotate_plain(float a, float b, float c, float s, float& ra, float& rb) {
  ra = __fmaf_rn(a, c, -__fmul_rn(b, s));
  rb = __fmaf_rn(b, c, __fmul_rn(a, s));
}

__device__ __forceinline__ float bf16_bits_to_f32(uint32_t bits16) { return __uint_as_float(bits16 << 16); }
__device__ __forceinline__ uint32_t f32_to_bf16_bits(float x) {
  return (uint32_t)__bfloat16_as_ushort(__float2bfloat16_rn(x));
}
__device__ __forceinline__ uint32_t pack_bf16x2(float lo, float hi) {
  __nv_bfloat162 v = __floats2bfloat162_rn(lo, hi);
  return *reinterpret_cast<uint32_t*>(&v);
}
__device__ __forceinline__ float e4m3_to_f32(uint32_t q) {
  __half_raw h = __nv_cvt_fp8_to_halfraw((__nv_fp8_storage_t)q, __NV_E4M3);
  return __half2float(*reinterpret_cast<__half*>(&h));
}
__device__ __forceinline__ uint32_t f32_to_e4m3_sat(float x) {
  return (uint32_t)__nv_cvt_float_to_fp8(x, __NV_SATFINITE, __NV_E4M3);
}
// two e4m3 in the low 16 bits -> two floats
__device__ __forceinline__ float2 e4m3x2_to_f32x2(uint32_t q2) {
  __half2_raw h = __nv_cvt_fp8x2_to_halfraw2((__nv_fp8x2_storage_t)q2, __NV_E4M3);
  return __half22float2(*reinterpret_cast<__half2*>(&h));
}
__device__ __forceinline__ uint32_t f32x2_to_e4m3x2_sat(float lo, float hi) {
  return (uint32_t)__nv_cvt_float2_to_fp8x2(make_float2(lo, hi), __NV_SATFINITE, __NV_E4M3);
}

// launch entry points implemented in the .cu files
cudaError_t launch_generic(const CallParams& P, int sm_count, cudaStream_t stream, int* grid, int* block, int* smem);

// the same kernel with 16-byte accesses, for shapes whose rotary window splits into whole vectors (kvr_generic_vec.cu)
bool generic_vec_supported(const CallParams& P);
cudaError_t launch_generic_vec(const CallParams& P, int sm_count, cudaStream_t stream, int* grid, int* block, int* smem);

// in-place re-float of a rotary window inside a longer row (kvr_window.cu)
bool window_inplace_supported(const CallParams& P);
cudaError_t launch_window_inplace(const CallParams& P, int sm_count, cudaStream_t stream, int* grid, int* block, int* smem);

struct RingConfig {
  int ctas_per_sm, consumer_warps, stages, v_bulk_store, max_ctas, grab, pdl, warps_per_stage, lanes_over_heads;
  const TmapInline* tmaps_inline;   // HOST pointer: tensor maps of a call with <= kInlineSegs segments (tmajor mode)
};
int ring_heads_per_tile(const CallParams& P);   // heads one tile of the ring kernel covers (needs P.cg)
bool ring_window_mode(const CallParams& P);      // rows outside the power-of-two slot layout (e.g. MLA [latent | k_pe])
bool ring_supported(const CallParams& P, const SegDev* host_segs, const RingConfig& cfg, int sm_count, const char** why);
cudaError_t launch_ring(const CallParams& P, const RingConfig& cfg, int sm_count, cudaStream_t stream,
                        int* grid, int* block, int* smem);

}  // namespace kvr
