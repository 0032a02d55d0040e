// kvr_window.cu -- in-place re-float of a ROTARY WINDOW inside a longer cached row, for sm_100a.
//
// kvr_reposition_inplace on a cache whose rows carry position-free dims besides the rotary ones -- the MLA
// [latent c_t | k_pe] row of DeepSeek-V2 ("repositioning re-rotates only k_pe and copies the latent
// as-is", :514 Fig. 22a; R23) re-floated each turn (R20).  Only the window moves: 2 * layers *
// kv_heads * rotary_dim * esz bytes per token (128 of the 1152 bytes of an MLA row), so the TMA ring of kvr_ring.cu,
// which stages whole rows, would read nine times the bytes that matter; this kernel touches the window alone.
//
// Work units are the API's (segment, chunk of <= cg tokens inside one block, layer group); a CTA walks units
// grid-stride, rebuilds the segment's angle table (fp64 sincos -> fp32 hi/lo, step a1) in shared memory only when
// the segment changes, resolves the chunk's block (a4) and then treats every (layer, head, token) row of the unit
// with rotary_dim * esz / 32 lanes per row: a lane loads the two 16-byte vectors that hold both halves of its pairs
// straight from the paged slot (a2), rotates them in registers with the same word-level routines as the ring
// kernel (a3) and stores them back to where they came from (a5) -- each pair is read and written by one thread, so the
// call is aliasing-safe by construction.  Per-segment shifts only (a position map takes the generic kernel).

#include "kvr_rotate.cuh"

namespace kvr {

template <int DTYPE, int PAIRING>
__global__ void __launch_bounds__(256) kvr_window_inplace_kernel(const __grid_constant__ CallParams P, int log_lpr) {
  using G = Geo<DTYPE, PAIRING>;
  constexpr int E = (DTYPE == 0) ? 2 : 1;
  __shared__ float4 tab[512];                      // (cos_hi, cos_lo, sin_hi, sin_lo) of pair p for the current segment
  const int half_R = P.rotary_dim >> 1;
  const int lpr = 1 << log_lpr;                    // lanes per row = rotary vectors / 2
  const int q = threadIdx.x & (lpr - 1);           // this thread's slot in a row: vectors q and q + lpr of the window
  const int va16 = q * 16, vb16 = (q + lpr) * 16;
  float4 T4[DTYPE == 0 ? G::NT : 1];
  float2 T2[DTYPE == 1 ? G::NT : 1];
  int cur_si = -1;
  const SegDev* segs = seg_array(P);

  for (int64_t unit = blockIdx.x; unit < P.total_units; unit += gridDim.x) {
    const int si = find_segment(segs, P.n_segs, unit);
    const SegDev s = segs[si];
    if (si != cur_si) {                            // uniform over the CTA
      __syncthreads();                             // the previous table is no longer read
      for (int p = threadIdx.x; p < half_R; p += blockDim.x) tab[p] = angle_entry((int64_t)s.delta, P.inv_freq[p]);
      __syncthreads();
      // pairs of this lane: NeoX -- vector q holds the "a" halves of pairs q*EPV.., vector q + lpr their partners;
      // GPT-J -- vector v holds pairs v*PPV.. whole, the lane rotates its two vectors independently
#pragma unroll
      for (int k = 0; k < G::NT; ++k) {
        const int p = (PAIRING == 0) ? q * G::EPV + k : ((k < G::PPV) ? q * G::PPV + k : (q + lpr) * G::PPV + (k - G::PPV));
        const float4 e = tab[p];
        if (DTYPE == 0) T4[k] = e; else T2[k] = make_float2(e.x, e.z);
      }
      cur_si = si;
    }
    if (s.delta == 0) continue;                    // nothing moves
    const int64_t local = unit - s.unit_begin;
    const int lg = (int)(local / s.n_chunks), c = (int)(local - (int64_t)lg * s.n_chunks);
    const Chunk ch = chunk_of(s, c, P.cg, P.block_size);
    const int l0 = lg * P.lpu, l1 = min(P.layers, l0 + P.lpu);
    const int32_t blk = P.block_table[(int64_t)s.dst_seq * P.max_blocks + ch.blk_index];
    if (blk < 0 || blk >= P.num_blocks) {
      if (threadIdx.x == 0) report_bad_block(P.status, s.index, ch.t0);
      continue;
    }
    uint8_t* const base = P.k_cache + ((int64_t)blk * P.d_sb + (int64_t)ch.off * P.d_st + P.rotary_offset) * E;
    const int rows_per_layer = P.heads * ch.n_tok;
    const int tasks = ((l1 - l0) * rows_per_layer) << log_lpr;
    // four rows per thread and pass: all loads first (a store to the pool could alias a later load as far as the
    // compiler knows, so without this the passes would run one memory latency after the other)
    constexpr int U = 4;
    for (int task0 = threadIdx.x; task0 < tasks; task0 += U * blockDim.x) {
      uint8_t* p[U];
      uint4 A[U], B[U];
#pragma unroll
      for (int u = 0; u < U; ++u) {
        const int task = task0 + u * blockDim.x;
        const int row = min(task, tasks - 1) >> log_lpr;
        const int l = l0 + row / rows_per_layer, r2 = row % rows_per_layer;
        const int h = r2 / ch.n_tok, t = r2 - h * ch.n_tok;
        p[u] = base + ((int64_t)l * P.d_sl + (int64_t)h * P.d_sh + (int64_t)t * P.d_st) * E;
        A[u] = *reinterpret_cast<const uint4*>(p[u] + va16);
        B[u] = *reinterpret_cast<const uint4*>(p[u] + vb16);
      }
#pragma unroll
      for (int u = 0; u < U; ++u) {
        if (task0 + u * blockDim.x >= tasks) break;
        if constexpr (DTYPE == 0) {
          if constexpr (PAIRING == 0) rot_bf16_neox(A[u], B[u], T4);
          else { rot_bf16_gptj(A[u], T4); rot_bf16_gptj(B[u], T4 + G::PPV); }
        } else {                                   // in place the source and destination scales are the same number: they cancel
          if constexpr (PAIRING == 0) rot_fp8_neox<false>(A[u], B[u], T2, 1.0f, 1.0f, true);
          else { rot_fp8_gptj<false>(A[u], T2, 1.0f, 1.0f, true); rot_fp8_gptj<false>(B[u], T2 + G::PPV, 1.0f, 1.0f, true); }
        }
        *reinterpret_cast<uint4*>(p[u] + va16) = A[u];
        *reinterpret_cast<uint4*>(p[u] + vb16) = B[u];
      }
    }
  }
}

// rotary windows the kernel takes: rotary_dim * esz = 32 * 2^k bytes (k <= 5), at most 512 pairs, per-segment shifts
bool window_inplace_supported(const CallParams& P) {
  const int E = P.dtype == 0 ? 2 : 1;
  const int rotB = P.rotary_dim * E;
  if (!P.inplace || P.any_pos_map) return false;
  if (rotB % 32 || rotB > 1024 || ((rotB / 32) & (rotB / 32 - 1))) return false;
  return P.rotary_dim / 2 <= 512;
}

cudaError_t launch_window_inplace(const CallParams& P, int sm_count, cudaStream_t stream, int* grid, int* block, int* smem) {
  const int E = P.dtype == 0 ? 2 : 1;
  int log_lpr = 0;
  while ((1 << log_lpr) < P.rotary_dim * E / 32) ++log_lpr;
  int64_t g = P.total_units < (int64_t)sm_count * 8 ? P.total_units : (int64_t)sm_count * 8;
  if (g < 1) g = 1;
  *grid = (int)g; *block = 256; *smem = (int)sizeof(float4) * 512;
  if (P.dtype == 0) {
    if (P.pairing == 0) kvr_window_inplace_kernel<0, 0><<<(unsigned)g, 256, 0, stream>>>(P, log_lpr);
    else kvr_window_inplace_kernel<0, 1><<<(unsigned)g, 256, 0, stream>>>(P, log_lpr);
  } else {
    if (P.pairing == 0) kvr_window_inplace_kernel<1, 0><<<(unsigned)g, 256, 0, stream>>>(P, log_lpr);
    else kvr_window_inplace_kernel<1, 1><<<(unsigned)g, 256, 0, stream>>>(P, log_lpr);
  }
  return cudaGetLastError();
}

}  // namespace kvr
