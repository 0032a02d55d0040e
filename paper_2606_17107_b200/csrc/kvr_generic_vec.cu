// kvr_generic_vec.cu -- the generic reposition+splice kernel with 16-byte accesses.
// Same work decomposition, same table and the same per-element arithmetic as kvr_generic.cu (so the two agree bit for
// bit), for the shapes the TMA-ring kernel declines (rotary widths that are not 32 * 2^k bytes, odd strides, very long
// rows): there the scalar kernel ran at a quarter of the copy bandwidth because every thread moved 2-4 bytes per access.
// Here a thread moves one 16-byte vector of a row per access (two for a NeoX pair-vector), several per iteration with
// all loads issued before the first store.  Needs rotary_dim * esz % 32 == 0 (NeoX: both halves are whole vectors) or
// % 16 == 0 (GPT-J: pairs never straddle a vector); other shapes stay on the scalar kernel.  Auto dispatch takes this
// kernel; tuning.path = 1 still forces the scalar one, which remains the on-device cross-check (kvr.h: path 5).
#include "kvr_common.cuh"

namespace kvr {
namespace {

__device__ __forceinline__ uint4 ld16(const uint8_t* p) { return *reinterpret_cast<const uint4*>(p); }
__device__ __forceinline__ void st16(uint8_t* p, const uint4& v) { *reinterpret_cast<uint4*>(p) = v; }

struct RowScale { float s_src, s_dst, inv_dst; bool equal; };

// One rotary pair, exactly as kvr_generic.cu evaluates it (codes in the low bits of ua / ub).
template <int DTYPE>
__device__ __forceinline__ void rot_pair(uint32_t& ua, uint32_t& ub, const float4& cs, bool copy, const RowScale& sc) {
  if (DTYPE == 0) {
    if (copy) return;
    float ra, rb;
    rotate_comp(bf16_bits_to_f32(ua), bf16_bits_to_f32(ub), cs, ra, rb);
    ua = f32_to_bf16_bits(ra);
    ub = f32_to_bf16_bits(rb);
  } else if (sc.equal) {
    if (copy) return;
    float ra, rb;
    rotate_plain(e4m3_to_f32(ua), e4m3_to_f32(ub), cs.x, cs.z, ra, rb);
    ua = f32_to_e4m3_sat(ra);
    ub = f32_to_e4m3_sat(rb);
  } else {
    const float c_ = copy ? 1.0f : cs.x, s_ = copy ? 0.0f : cs.z;
    float ra, rb;
    rotate_plain(__fmul_rn(e4m3_to_f32(ua), sc.s_src), __fmul_rn(e4m3_to_f32(ub), sc.s_src), c_, s_, ra, rb);
    ua = f32_to_e4m3_sat(__fmul_rn(ra, sc.inv_dst));
    ub = f32_to_e4m3_sat(__fmul_rn(rb, sc.inv_dst));
  }
}

// NeoX: A holds elements [i0, i0 + VE) of the first half, B the same of the second half; pair j is (A[j], B[j]).
template <int DTYPE>
__device__ __forceinline__ void rot_vec_neox(uint4& A, uint4& B, const float4* __restrict__ tab_row, int i0, bool copy,
                                             const RowScale& sc) {
  uint32_t a[4] = {A.x, A.y, A.z, A.w}, b[4] = {B.x, B.y, B.z, B.w};
  constexpr int PW = (DTYPE == 0) ? 2 : 4, BITS = (DTYPE == 0) ? 16 : 8;     // elements per 32-bit word
  constexpr uint32_t MASK = (DTYPE == 0) ? 0xFFFFu : 0xFFu;
#pragma unroll
  for (int k = 0; k < 4; ++k) {
    uint32_t wa = 0, wb = 0;
#pragma unroll
    for (int m = 0; m < PW; ++m) {
      uint32_t ua = (a[k] >> (BITS * m)) & MASK, ub = (b[k] >> (BITS * m)) & MASK;
      rot_pair<DTYPE>(ua, ub, tab_row[i0 + k * PW + m], copy, sc);
      wa |= (ua & MASK) << (BITS * m);
      wb |= (ub & MASK) << (BITS * m);
    }
    a[k] = wa; b[k] = wb;
  }
  A = make_uint4(a[0], a[1], a[2], a[3]);
  B = make_uint4(b[0], b[1], b[2], b[3]);
}

// GPT-J: A holds pairs [i0, i0 + VE/2) as adjacent elements (2j, 2j + 1).
template <int DTYPE>
__device__ __forceinline__ void rot_vec_gptj(uint4& A, const float4* __restrict__ tab_row, int i0, bool copy, const RowScale& sc) {
  uint32_t a[4] = {A.x, A.y, A.z, A.w};
  constexpr int PW = (DTYPE == 0) ? 1 : 2, BITS = (DTYPE == 0) ? 16 : 8;     // pairs per 32-bit word
  constexpr uint32_t MASK = (DTYPE == 0) ? 0xFFFFu : 0xFFu;
#pragma unroll
  for (int k = 0; k < 4; ++k) {
    uint32_t w = 0;
#pragma unroll
    for (int m = 0; m < PW; ++m) {
      uint32_t ua = (a[k] >> (2 * BITS * m)) & MASK, ub = (a[k] >> (2 * BITS * m + BITS)) & MASK;
      rot_pair<DTYPE>(ua, ub, tab_row[i0 + k * PW + m], copy, sc);
      w |= ((ua & MASK) << (2 * BITS * m)) | ((ub & MASK) << (2 * BITS * m + BITS));
    }
    a[k] = w;
  }
  A = make_uint4(a[0], a[1], a[2], a[3]);
}

// fp8 pass-through dims when source and destination scales differ: requantise every code (kvr_generic.cu).
__device__ __forceinline__ void requant_vec(uint4& A, const RowScale& sc) {
  uint32_t a[4] = {A.x, A.y, A.z, A.w};
#pragma unroll
  for (int k = 0; k < 4; ++k) {
    uint32_t w = 0;
#pragma unroll
    for (int m = 0; m < 4; ++m) {
      const uint32_t q = (a[k] >> (8 * m)) & 0xFFu;
      w |= (f32_to_e4m3_sat(__fmul_rn(__fmul_rn(e4m3_to_f32(q), sc.s_src), sc.inv_dst)) & 0xFFu) << (8 * m);
    }
    a[k] = w;
  }
  A = make_uint4(a[0], a[1], a[2], a[3]);
}

// Launch shape, measured on B200 over configs[1] / [3] fp8 / [4] forced through this kernel (GB/s): 2 items in flight per
// thread with >= 4 CTAs per SM (<= 64 registers) 2895 / 2761 / 3855; 4 items, 2 CTAs 2650 / 2601 / 3291; 1 item, 6 CTAs
// 2719 / 2585 / 3141; 4 items, 3 CTAs 2314 / 1907 / 3368: more resident warps beat more loads per warp.
#ifndef KVR_GVEC_UNROLL
#define KVR_GVEC_UNROLL 2
#endif
#ifndef KVR_GVEC_COPY_UNROLL
#define KVR_GVEC_COPY_UNROLL KVR_GVEC_UNROLL
#endif
#ifndef KVR_GVEC_MIN_CTAS
#define KVR_GVEC_MIN_CTAS 4
#endif
constexpr int kUnroll = KVR_GVEC_UNROLL;            // rotary items (NeoX: pair-vectors) a thread has in flight per iteration
constexpr int kCopyUnroll = KVR_GVEC_COPY_UNROLL;   // plain 16-byte copies (pass-through dims, V) in flight per iteration

template <int DTYPE, int PAIRING>
__global__ void __launch_bounds__(256, KVR_GVEC_MIN_CTAS) kvr_generic_vec_kernel(const __grid_constant__ CallParams P) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  float4* tab = reinterpret_cast<float4*>(smem_raw);                 // [cg][R/2]
  int32_t* is_copy = reinterpret_cast<int32_t*>(tab + (size_t)P.cg * (P.rotary_dim / 2));  // [cg]
  constexpr int E = (DTYPE == 0) ? 2 : 1, VE = 16 / E;
  const int half = P.rotary_dim / 2, D = P.head_dim, R = P.rotary_dim;
  const int nrot = (PAIRING == 0) ? half / VE : R / VE;              // rotary items per row (NeoX: two vectors each)
  const int npass = (D - R) / VE, nvec = D / VE;
  const int pass_lo = P.rotary_offset / VE;                          // pass-through vectors below the window

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
    const bool per_token = s.pos_map != nullptr || s.pre_rope != 0;
    const int tab_rows = per_token ? ch.n_tok : 1;
    for (int idx = threadIdx.x; idx < tab_rows * half; idx += blockDim.x) {
      const int t = idx / half, i = idx % half;
      tab[t * half + i] = angle_entry(token_delta(s, ch.t0 + t), P.inv_freq[i]);
    }
    for (int t = threadIdx.x; t < ch.n_tok; t += blockDim.x) is_copy[t] = (token_delta(s, ch.t0 + t) == 0);
    const int32_t blk = P.block_table[(int64_t)s.dst_seq * P.max_blocks + ch.blk_index];
    __syncthreads();
    if (blk < 0 || blk >= P.num_blocks) {
      if (threadIdx.x == 0) report_bad_block(P.status, s.index, ch.t0);
      continue;
    }
    const int64_t dst_base = (int64_t)blk * P.d_sb + (int64_t)ch.off * P.d_st;
    const int rows = (l1 - l0) * P.heads * ch.n_tok;
    auto row_of = [&](int row, int& t, int& h, int& l) {
      t = row % ch.n_tok; h = (row / ch.n_tok) % P.heads; l = l0 + row / (ch.n_tok * P.heads);
    };
    auto k_dst = [&](int t, int h, int l) {
      return P.k_cache + ((int64_t)l * P.d_sl + (int64_t)h * P.d_sh + (int64_t)t * P.d_st + dst_base) * E;
    };
    auto k_src = [&](int t, int h, int l, uint8_t* dst) -> const uint8_t* {
      return P.inplace ? dst : s.k_src + ((int64_t)l * s.sl + (int64_t)h * s.sh + (int64_t)(ch.t0 + t) * s.st) * E;
    };
    auto scale_of = [&](int h, int l) {
      RowScale sc{1.0f, 1.0f, 1.0f, true};
      if (DTYPE == 1) {
        sc.s_src = s.k_scale_src[l * P.heads + h]; sc.s_dst = P.k_scale_dst[l * P.heads + h];
        sc.equal = sc.s_src == sc.s_dst; sc.inv_dst = __frcp_rn(sc.s_dst);
      }
      return sc;
    };

    // ---- K rotary window: kUnroll items per thread, loads before stores ----
    const int64_t n_rot = (int64_t)rows * nrot;
    for (int64_t base = threadIdx.x; base < n_rot; base += (int64_t)blockDim.x * kUnroll) {
      uint4 A[kUnroll], B[kUnroll];
      uint8_t* dp[kUnroll];
      int tt[kUnroll], i0[kUnroll];
      RowScale sc[kUnroll];
#pragma unroll
      for (int u = 0; u < kUnroll; ++u) {
        const int64_t idx = base + (int64_t)u * blockDim.x;
        dp[u] = nullptr;
        if (idx >= n_rot) continue;
        const int v = (int)(idx % nrot);
        int t, h, l;
        row_of((int)(idx / nrot), t, h, l);
        uint8_t* d = k_dst(t, h, l);
        const uint8_t* sp = k_src(t, h, l, d);
        const int e0 = P.rotary_offset + v * VE;                       // first element of the (first-half) vector
        dp[u] = d + (int64_t)e0 * E;
        tt[u] = t;
        i0[u] = (PAIRING == 0) ? v * VE : v * (VE / 2);
        sc[u] = scale_of(h, l);
        A[u] = ld16(sp + (int64_t)e0 * E);
        if (PAIRING == 0) B[u] = ld16(sp + (int64_t)(e0 + half) * E);
      }
#pragma unroll
      for (int u = 0; u < kUnroll; ++u) {
        if (!dp[u]) continue;
        const float4* row = tab + (per_token ? tt[u] : 0) * half;
        const bool copy = is_copy[tt[u]] != 0;
        if (PAIRING == 0) {
          rot_vec_neox<DTYPE>(A[u], B[u], row, i0[u], copy, sc[u]);
          st16(dp[u], A[u]);
          st16(dp[u] + (int64_t)half * E, B[u]);
        } else {
          rot_vec_gptj<DTYPE>(A[u], row, i0[u], copy, sc[u]);
          st16(dp[u], A[u]);
        }
      }
    }
    if (P.inplace) continue;   // pass-through dims and V already hold their bytes

    // ---- K pass-through vectors ([0, rotary_offset) and [rotary_offset + R, D)) and all V vectors: copies ----
    const int per_row = npass + (P.no_v ? 0 : nvec);
    const int64_t n_copy = (int64_t)rows * per_row;
    for (int64_t base = threadIdx.x; base < n_copy; base += (int64_t)blockDim.x * kCopyUnroll) {
      uint4 A[kCopyUnroll];
      uint8_t* dp[kCopyUnroll];
#pragma unroll
      for (int u = 0; u < kCopyUnroll; ++u) {
        const int64_t idx = base + (int64_t)u * blockDim.x;
        dp[u] = nullptr;
        if (idx >= n_copy) continue;
        int item = (int)(idx % per_row);
        int t, h, l;
        row_of((int)(idx / per_row), t, h, l);
        const int64_t src_row = ((int64_t)l * s.sl + (int64_t)h * s.sh + (int64_t)(ch.t0 + t) * s.st) * E;
        const int64_t dst_row = ((int64_t)l * P.d_sl + (int64_t)h * P.d_sh + (int64_t)t * P.d_st + dst_base) * E;
        if (item < npass) {
          const int v = item < pass_lo ? item : item + R / VE;           // vector index within the row
          A[u] = ld16(s.k_src + src_row + (int64_t)v * 16);
          if (DTYPE == 1) {
            const RowScale sc = scale_of(h, l);
            if (!sc.equal) requant_vec(A[u], sc);
          }
          dp[u] = P.k_cache + dst_row + (int64_t)v * 16;
        } else {
          item -= npass;
          A[u] = ld16(s.v_src + src_row + (int64_t)item * 16);
          dp[u] = P.v_cache + dst_row + (int64_t)item * 16;
        }
      }
#pragma unroll
      for (int u = 0; u < kCopyUnroll; ++u)
        if (dp[u]) st16(dp[u], A[u]);
    }
  }
}

}  // namespace

bool generic_vec_supported(const CallParams& P) {
  const int E = P.dtype == 0 ? 2 : 1;
  const int rotB = P.rotary_dim * E;
  return P.pairing == 0 ? rotB % 32 == 0 : rotB % 16 == 0;   // rows, offsets and strides are 16-byte multiples by the API's rules
}

cudaError_t launch_generic_vec(const CallParams& P, int sm_count, cudaStream_t stream, int* grid, int* block, int* smem) {
  size_t sm = (size_t)P.cg * (P.rotary_dim / 2) * sizeof(float4) + (size_t)P.cg * sizeof(int32_t);
  int64_t g = P.total_units < (int64_t)sm_count * 32 ? P.total_units : (int64_t)sm_count * 32;
  if (g < 1) g = 1;
  *grid = (int)g; *block = 256; *smem = (int)sm;
  if (P.dtype == 0) {
    if (P.pairing == 0) kvr_generic_vec_kernel<0, 0><<<(unsigned)g, 256, sm, stream>>>(P);
    else kvr_generic_vec_kernel<0, 1><<<(unsigned)g, 256, sm, stream>>>(P);
  } else {
    if (P.pairing == 0) kvr_generic_vec_kernel<1, 0><<<(unsigned)g, 256, sm, stream>>>(P);
    else kvr_generic_vec_kernel<1, 1><<<(unsigned)g, 256, sm, stream>>>(P);
  }
  return cudaGetLastError();
}

}  // namespace kvr
