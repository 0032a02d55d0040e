// kvr_generic.cu -- the GENERIC reposition+splice kernel: any head_dim / rotary_dim / strides the
// API accepts, both pairings, both dtypes, per-segment Delta or per-token position map.
// It is the fallback for shapes the TMA-ring kernel (kvr_ring.cu) does not take and an independent
// on-device cross-check of it.  One CTA per (segment, chunk of <= cg destination tokens, layer group):
//   1. angle table for the chunk's tokens: fp64 sincos -> fp32 hi/lo in shared memory (step a1)
//   2. block-table lookup for the chunk (step a4)
//   3. K rotary pairs, scalar element loads (a2, a3, a5); K pass-through dims; V 16-byte copies (a6)
// Steps refer to SURVEY.md 8(a) / DESIGN.md "Path".  With P.inplace (kvr_reposition_inplace, R20) the K row
// is read from the pool slot it is written back to, and pass-through dims and V are left alone.
// P.rotary_offset / P.no_v: the MLA adapter of kvr.h (rotary window inside the row; no V tensor).
#include "kvr_common.cuh"

namespace kvr {

template <int DTYPE>
__global__ void __launch_bounds__(256) kvr_generic_kernel(const __grid_constant__ CallParams P) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  float4* tab = reinterpret_cast<float4*>(smem_raw);                 // [cg][R/2]
  int32_t* is_copy = reinterpret_cast<int32_t*>(tab + (size_t)P.cg * (P.rotary_dim / 2));  // [cg]
  constexpr int E = (DTYPE == 0) ? 2 : 1;
  const int half = P.rotary_dim / 2;
  const int D = P.head_dim, R = P.rotary_dim;

  for (int64_t unit = blockIdx.x; unit < P.total_units; unit += gridDim.x) {
    const SegDev* segs = seg_array(P);
    const int si = find_segment(segs, P.n_segs, unit);
    const SegDev s = segs[si];
    const int64_t local = unit - s.unit_begin;
    const int lg = (int)(local / s.n_chunks);
    const int c = (int)(local % s.n_chunks);
    const Chunk ch = chunk_of(s, c, P.cg, P.block_size);
    const int l0 = lg * P.lpu, l1 = min(P.layers, l0 + P.lpu);

    __syncthreads();  // previous unit's table no longer in use
    // per-token shifts (position map, pre-RoPE keys): one table row per token; a constant shift: one row for all
    const bool per_token = s.pos_map != nullptr || s.pre_rope != 0;
    const int tab_rows = per_token ? ch.n_tok : 1;
    for (int idx = threadIdx.x; idx < tab_rows * half; idx += blockDim.x) {
      int t = idx / half, i = idx % half;
      int64_t delta = token_delta(s, ch.t0 + t);
      tab[t * half + i] = angle_entry(delta, P.inv_freq[i]);
    }
    for (int t = threadIdx.x; t < ch.n_tok; t += blockDim.x) is_copy[t] = (token_delta(s, ch.t0 + t) == 0);
    const int32_t blk = P.block_table[(int64_t)s.dst_seq * P.max_blocks + ch.blk_index];
    __syncthreads();
    if (blk < 0 || blk >= P.num_blocks) {
      if (threadIdx.x == 0) report_bad_block(P.status, s.index, ch.t0);
      continue;
    }
    const int64_t dst_base = (int64_t)blk * P.d_sb + (int64_t)ch.off * P.d_st;   // + l*d_sl + h*d_sh + t*d_st
    const int rows = (l1 - l0) * P.heads * ch.n_tok;

    // ---- K rotary pairs ----
    for (int64_t idx = threadIdx.x; idx < (int64_t)rows * half; idx += blockDim.x) {
      int i = (int)(idx % half);
      int row = (int)(idx / half);
      int t = row % ch.n_tok;
      int h = (row / ch.n_tok) % P.heads;
      int l = l0 + row / (ch.n_tok * P.heads);
      int ia = P.rotary_offset + ((P.pairing == 0) ? i : 2 * i);          // the rotary window starts at rotary_offset
      int ib = P.rotary_offset + ((P.pairing == 0) ? i + half : 2 * i + 1);
      uint8_t* dst = P.k_cache + ((int64_t)l * P.d_sl + (int64_t)h * P.d_sh + (int64_t)t * P.d_st + dst_base) * E;
      const uint8_t* src = P.inplace ? dst      // each pair is read and written by this one thread: aliasing-safe
                                     : s.k_src + ((int64_t)l * s.sl + (int64_t)h * s.sh + (int64_t)(ch.t0 + t) * s.st) * E;
      float4 cs = tab[(per_token ? t : 0) * half + i];
      if (DTYPE == 0) {
        uint16_t ua = reinterpret_cast<const uint16_t*>(src)[ia], ub = reinterpret_cast<const uint16_t*>(src)[ib];
        if (!is_copy[t]) {
          float ra, rb;
          rotate_comp(bf16_bits_to_f32(ua), bf16_bits_to_f32(ub), cs, ra, rb);
          ua = (uint16_t)f32_to_bf16_bits(ra);
          ub = (uint16_t)f32_to_bf16_bits(rb);
        }
        reinterpret_cast<uint16_t*>(dst)[ia] = ua;
        reinterpret_cast<uint16_t*>(dst)[ib] = ub;
      } else {
        uint8_t qa = src[ia], qb = src[ib];
        float s_src = s.k_scale_src[l * P.heads + h], s_dst = P.k_scale_dst[l * P.heads + h];
        if (s_src == s_dst) {
          // equal scales cancel exactly ((q s c - q' s s') / s = q c - q' s'): the codes are rotated as they are,
          // the same formulation as the ring kernel (kvr.h)
          if (!is_copy[t]) {
            float ra, rb;
            rotate_plain(e4m3_to_f32(qa), e4m3_to_f32(qb), cs.x, cs.z, ra, rb);
            qa = (uint8_t)f32_to_e4m3_sat(ra);
            qb = (uint8_t)f32_to_e4m3_sat(rb);
          }
        } else {
          float c_ = is_copy[t] ? 1.0f : cs.x, s_ = is_copy[t] ? 0.0f : cs.z;
          float ra, rb, inv = __frcp_rn(s_dst);
          rotate_plain(__fmul_rn(e4m3_to_f32(qa), s_src), __fmul_rn(e4m3_to_f32(qb), s_src), c_, s_, ra, rb);
          qa = (uint8_t)f32_to_e4m3_sat(__fmul_rn(ra, inv));
          qb = (uint8_t)f32_to_e4m3_sat(__fmul_rn(rb, inv));
        }
        dst[ia] = qa;
        dst[ib] = qb;
      }
    }
    if (P.inplace) continue;   // pass-through dims and V already hold their bytes
    // ---- K pass-through dims: [0, rotary_offset) and [rotary_offset + R, D) ----
    const int pass = D - R;
    for (int64_t idx = threadIdx.x; idx < (int64_t)rows * pass; idx += blockDim.x) {
      int d = (int)(idx % pass);
      if (d >= P.rotary_offset) d += R;
      int row = (int)(idx / pass);
      int t = row % ch.n_tok;
      int h = (row / ch.n_tok) % P.heads;
      int l = l0 + row / (ch.n_tok * P.heads);
      const uint8_t* src = s.k_src + ((int64_t)l * s.sl + (int64_t)h * s.sh + (int64_t)(ch.t0 + t) * s.st) * E;
      uint8_t* dst = P.k_cache + ((int64_t)l * P.d_sl + (int64_t)h * P.d_sh + (int64_t)t * P.d_st + dst_base) * E;
      if (DTYPE == 0) {
        reinterpret_cast<uint16_t*>(dst)[d] = reinterpret_cast<const uint16_t*>(src)[d];
      } else {
        uint8_t q = src[d];
        float s_src = s.k_scale_src[l * P.heads + h], s_dst = P.k_scale_dst[l * P.heads + h];
        if (s_src != s_dst) q = (uint8_t)f32_to_e4m3_sat(__fmul_rn(__fmul_rn(e4m3_to_f32(q), s_src), __frcp_rn(s_dst)));
        dst[d] = q;
      }
    }
    if (P.no_v) continue;      // K-only call: a [latent | k_pe] cache has no V tensor
    // ---- V: unchanged bytes, 16 B at a time (rows are 16-byte multiples and 16-byte aligned) ----
    const int vecs = D * E / 16;
    for (int64_t idx = threadIdx.x; idx < (int64_t)rows * vecs; idx += blockDim.x) {
      int v = (int)(idx % vecs);
      int row = (int)(idx / vecs);
      int t = row % ch.n_tok;
      int h = (row / ch.n_tok) % P.heads;
      int l = l0 + row / (ch.n_tok * P.heads);
      const uint4* src = reinterpret_cast<const uint4*>(
          s.v_src + ((int64_t)l * s.sl + (int64_t)h * s.sh + (int64_t)(ch.t0 + t) * s.st) * E);
      uint4* dst = reinterpret_cast<uint4*>(
          P.v_cache + ((int64_t)l * P.d_sl + (int64_t)h * P.d_sh + (int64_t)t * P.d_st + dst_base) * E);
      dst[v] = src[v];
    }
  }
}

cudaError_t launch_generic(const CallParams& P, int sm_count, cudaStream_t stream, int* grid, int* block, int* smem) {
  size_t sm = (size_t)P.cg * (P.rotary_dim / 2) * sizeof(float4) + (size_t)P.cg * sizeof(int32_t);
  int64_t g = P.total_units < (int64_t)sm_count * 32 ? P.total_units : (int64_t)sm_count * 32;
  if (g < 1) g = 1;
  *grid = (int)g; *block = 256; *smem = (int)sm;
  if (P.dtype == 0) kvr_generic_kernel<0><<<(unsigned)g, 256, sm, stream>>>(P);
  else kvr_generic_kernel<1><<<(unsigned)g, 256, sm, stream>>>(P);
  return cudaGetLastError();
}

}  // namespace kvr
