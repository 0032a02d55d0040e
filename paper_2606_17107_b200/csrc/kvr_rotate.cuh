// kvr_rotate.cuh -- word-level rotation of 16-byte vectors of cached keys (bf16: compensated fp32; fp8-e4m3: plain fp32
// on the codes, or dequantise / rotate / requantise under a scale change), shared by the ring kernel and the window
// in-place kernel.  Product code (sm_100a); shares nothing with oracle/.
#pragma once
#include "kvr_common.cuh"

namespace kvr {

// ------------------------------------------------------------------------------- word-level math
template <int DTYPE, int PAIRING> struct Geo;
template <> struct Geo<0, 0> { static constexpr int EPV = 8, PPV = 8, NT = 8; };    // bf16 NeoX : table regs = 8 pairs
template <> struct Geo<0, 1> { static constexpr int EPV = 8, PPV = 4, NT = 8; };    // bf16 GPT-J: 4 + 4
template <> struct Geo<1, 0> { static constexpr int EPV = 16, PPV = 16, NT = 16; }; // fp8 NeoX
template <> struct Geo<1, 1> { static constexpr int EPV = 16, PPV = 8, NT = 16; };  // fp8 GPT-J: 8 + 8

// bf16, NeoX: A = 8 "a" elements, B = the 8 partner "b" elements; T[j] belongs to element j.
__device__ __forceinline__ void rot_bf16_neox(uint4& A, uint4& B, const float4* T) {
  uint32_t* a = reinterpret_cast<uint32_t*>(&A);
  uint32_t* b = reinterpret_cast<uint32_t*>(&B);
#pragma unroll
  for (int w = 0; w < 4; ++w) {
    float ra0, rb0, ra1, rb1;
    rotate_comp(__uint_as_float(a[w] << 16), __uint_as_float(b[w] << 16), T[2 * w], ra0, rb0);
    rotate_comp(__uint_as_float(a[w] & 0xFFFF0000u), __uint_as_float(b[w] & 0xFFFF0000u), T[2 * w + 1], ra1, rb1);
    a[w] = pack_bf16x2(ra0, ra1);
    b[w] = pack_bf16x2(rb0, rb1);
  }
}
// bf16, GPT-J: each 32-bit word is one pair (lo = a, hi = b); T[w] belongs to word w.
__device__ __forceinline__ void rot_bf16_gptj(uint4& A, const float4* T) {
  uint32_t* a = reinterpret_cast<uint32_t*>(&A);
#pragma unroll
  for (int w = 0; w < 4; ++w) {
    float ra, rb;
    rotate_comp(__uint_as_float(a[w] << 16), __uint_as_float(a[w] & 0xFFFF0000u), T[w], ra, rb);
    a[w] = pack_bf16x2(ra, rb);
  }
}
// fp8, NeoX: A = 16 "a" codes, B = 16 "b" codes; T[j] = (cos, sin) of element j.
// SCALE = false: source and destination scales are the same number, so dequantise/requantise cancel exactly
// ((q s c - q' s s') / s = q c - q' s'): the codes are rotated as they are, which is both cheaper and closer to fp64.
template <bool SCALE>
__device__ __forceinline__ void rot_fp8_neox(uint4& A, uint4& B, const float2* T, float s_src, float inv_dst, bool rot) {
  uint32_t* a = reinterpret_cast<uint32_t*>(&A);
  uint32_t* b = reinterpret_cast<uint32_t*>(&B);
#pragma unroll
  for (int w = 0; w < 4; ++w) {
    float2 a01 = e4m3x2_to_f32x2(a[w] & 0xFFFFu), a23 = e4m3x2_to_f32x2(a[w] >> 16);
    float2 b01 = e4m3x2_to_f32x2(b[w] & 0xFFFFu), b23 = e4m3x2_to_f32x2(b[w] >> 16);
    float av[4] = {a01.x, a01.y, a23.x, a23.y}, bv[4] = {b01.x, b01.y, b23.x, b23.y};
    float ra[4], rb[4];
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      float2 cs = rot ? T[4 * w + j] : make_float2(1.0f, 0.0f);
      if (SCALE) {
        rotate_plain(__fmul_rn(av[j], s_src), __fmul_rn(bv[j], s_src), cs.x, cs.y, ra[j], rb[j]);
        ra[j] = __fmul_rn(ra[j], inv_dst);
        rb[j] = __fmul_rn(rb[j], inv_dst);
      } else {
        rotate_plain(av[j], bv[j], cs.x, cs.y, ra[j], rb[j]);
      }
    }
    a[w] = f32x2_to_e4m3x2_sat(ra[0], ra[1]) | (f32x2_to_e4m3x2_sat(ra[2], ra[3]) << 16);
    b[w] = f32x2_to_e4m3x2_sat(rb[0], rb[1]) | (f32x2_to_e4m3x2_sat(rb[2], rb[3]) << 16);
  }
}
// fp8, GPT-J: word w = codes (a, b, a, b) of pairs 2w, 2w+1.
template <bool SCALE>
__device__ __forceinline__ void rot_fp8_gptj(uint4& A, const float2* T, float s_src, float inv_dst, bool rot) {
  uint32_t* a = reinterpret_cast<uint32_t*>(&A);
#pragma unroll
  for (int w = 0; w < 4; ++w) {
    float2 p0 = e4m3x2_to_f32x2(a[w] & 0xFFFFu), p1 = e4m3x2_to_f32x2(a[w] >> 16);
    float2 c0 = rot ? T[2 * w] : make_float2(1.0f, 0.0f), c1 = rot ? T[2 * w + 1] : make_float2(1.0f, 0.0f);
    float ra0, rb0, ra1, rb1;
    if (SCALE) {
      rotate_plain(__fmul_rn(p0.x, s_src), __fmul_rn(p0.y, s_src), c0.x, c0.y, ra0, rb0);
      rotate_plain(__fmul_rn(p1.x, s_src), __fmul_rn(p1.y, s_src), c1.x, c1.y, ra1, rb1);
      a[w] = f32x2_to_e4m3x2_sat(__fmul_rn(ra0, inv_dst), __fmul_rn(rb0, inv_dst)) |
             (f32x2_to_e4m3x2_sat(__fmul_rn(ra1, inv_dst), __fmul_rn(rb1, inv_dst)) << 16);
    } else {
      rotate_plain(p0.x, p0.y, c0.x, c0.y, ra0, rb0);
      rotate_plain(p1.x, p1.y, c1.x, c1.y, ra1, rb1);
      a[w] = f32x2_to_e4m3x2_sat(ra0, rb0) | (f32x2_to_e4m3x2_sat(ra1, rb1) << 16);
    }
  }
}
// fp8 pass-through vector under a scale change: requantise every code
__device__ __forceinline__ void requant_fp8(uint4& A, float s_src, float inv_dst) {
  uint32_t* a = reinterpret_cast<uint32_t*>(&A);
#pragma unroll
  for (int w = 0; w < 4; ++w) {
    float2 p0 = e4m3x2_to_f32x2(a[w] & 0xFFFFu), p1 = e4m3x2_to_f32x2(a[w] >> 16);
    a[w] = f32x2_to_e4m3x2_sat(__fmul_rn(__fmul_rn(p0.x, s_src), inv_dst), __fmul_rn(__fmul_rn(p0.y, s_src), inv_dst)) |
           (f32x2_to_e4m3x2_sat(__fmul_rn(__fmul_rn(p1.x, s_src), inv_dst), __fmul_rn(__fmul_rn(p1.y, s_src), inv_dst)) << 16);
  }
}

}  // namespace kvr
