// kvr_attend.cu -- ROTATE-ON-READ decode attention over precompiled skills, for sm_100a (tcgen05 + TMEM + TMA).
//
// include/kvr.h, kvr_rotate_on_read_attention (reading R25): a
// decode-step query attends the cached K/V of the skills where they lie; the re-rotation to the target positions is
// applied as the keys are read.  Because rotations are orthogonal,  q . R(Delta) k = (R(-Delta) q) . k :  the kernel
// counter-rotates the (tiny) query once per segment and streams the cached keys and values ONCE, untouched.  HBM-bound
// (2 * kv_heads * 128 * 2 bytes per token and layer); the two contractions run on the tensor cores, because at 6.5 TB/s
// the fp32 pipes could not keep up with 4..16 query heads per kv head.
//
// Both products are computed TRANSPOSED so that the 128 rows of the MMA are real work instead of padding (a decode
// step has only q_heads / kv_heads = 1..16 query rows per kv head):
//     S^T [128 keys x 16]  = K  [128 keys x 128 dims] . Q'^T      A = K tile   (K-major, SWIZZLE_128B, straight from TMA)
//                                                                 B = Q'       (16 rows x 128 dims, K-major, SW128)
//     O^T [128 dims x 16] += V^T[128 dims x 128 keys] . P^T       A = V tile   (MN-major, SW128, straight from TMA)
//                                                                 B = P        (16 rows x 128 keys, K-major, SW128)
// One CTA per SM, persistent over work items (segment, kv head, run of <= kTilesMax key tiles), warp-specialised:
//   warp 0      TMA producer: K and V tiles (2 x 64-dim panels of 128 keys each) into a ring of kStages stages
//   warp 1      MMA issuer (one elected lane): tcgen05.mma kind::f16, accumulators in TMEM (S double-buffered, O)
//   warps 2-3   query warps: fp64 sincos of -Delta * inv_freq, rotate the item's query heads, round once to bf16,
//               write Q' in the swizzled operand layout (double-buffered, one item ahead)
//   warps 4-7   softmax: thread i owns key i of the tile (TMEM lane i): tcgen05.ld of its <= 16 scores, tile maximum by
//               warp shuffles + one named barrier, exp2, P^T to shared memory as the next MMA's B operand; the running
//               reference maximum only moves when a tile exceeds it by 2^8 (O^T is then rescaled in TMEM: 16 columns,
//               one tcgen05.ld/st pair per thread); at the end of an item O^T, the row sums and the reference go to
//               the partial buffer and the LAST item of a (request, kv head) group merges the group's partials.
#include <mutex>

#include "kvr_attend.cuh"
#include "kvr_ptx.cuh"

namespace kvr {

namespace {

constexpr int kD = 128;                 // head_dim this kernel is built for
constexpr int kTile = 128;              // keys per tile = rows of one MMA
constexpr int kStages = 3;              // K+V tiles in flight per CTA (64 KB each)
constexpr int kPanelB = kTile * 128;    // one 64-dim panel of a tile: 128 rows x 128 bytes
constexpr int kTileB = 2 * kPanelB;     // K (or V) tile: 32 KB
constexpr int kQB = 2 * 16 * 128;       // Q' / P operand: 2 panels x 16 rows x 128 bytes
constexpr int kThreads = 256;
constexpr int kRescaleLog2 = 8;         // the reference maximum moves only when a tile exceeds it by 2^8

// shared-memory layout (offsets from a 1024-byte aligned base)
constexpr int kOffK = 0;
constexpr int kOffV = kStages * kTileB;
constexpr int kOffQ = 2 * kStages * kTileB;
constexpr int kOffP = kOffQ + 2 * kQB;
constexpr int kOffBar = kOffP + 2 * kQB;
constexpr int kNumBars = 3 * kStages + 2 * 2 + 2 * 2 + 2 * 2 + 2;   // kfull, vfull, empty | s_full/empty | p_full/empty | q_full/empty | o_full/empty
constexpr int kOffRed = kOffBar + 8 * kNumBars;
constexpr int kOffMisc = kOffRed + 4 * 16 * 4;
constexpr int kSmemBytes = kOffMisc + 64 + 1024;   // + slack for the 1024-byte alignment of the base

// ---- tcgen05 wrappers ---------------------------------------------------------------------------------------------
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void fence_async_smem() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
__device__ __forceinline__ void tc_commit(uint32_t bar) {
  asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(bar) : "memory");
}
// D[tmem] (+)= A[smem desc] . B[smem desc]
__device__ __forceinline__ void tc_mma(uint32_t d_tmem, uint64_t a_desc, uint64_t b_desc, uint32_t idesc, uint32_t accumulate) {
  asm volatile(
      "{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
      "tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n\t}"
      ::"r"(d_tmem), "l"(a_desc), "l"(b_desc), "r"(idesc), "r"(accumulate) : "memory");
}
template <int N> struct TmemVec;
template <> struct TmemVec<4> {
  static __device__ __forceinline__ void ld(uint32_t a, float* r) {
    uint32_t v[4];
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x4.b32 {%0,%1,%2,%3}, [%4];" : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]) : "r"(a));
    asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
#pragma unroll
    for (int i = 0; i < 4; ++i) r[i] = __uint_as_float(v[i]);
  }
  static __device__ __forceinline__ void st(uint32_t a, const float* r) {
    asm volatile("tcgen05.st.sync.aligned.32x32b.x4.b32 [%0], {%1,%2,%3,%4};" ::"r"(a), "r"(__float_as_uint(r[0])),
                 "r"(__float_as_uint(r[1])), "r"(__float_as_uint(r[2])), "r"(__float_as_uint(r[3])) : "memory");
    asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
  }
};
template <> struct TmemVec<8> {
  static __device__ __forceinline__ void ld(uint32_t a, float* r) {
    uint32_t v[8];
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
                 : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]) : "r"(a));
    asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
#pragma unroll
    for (int i = 0; i < 8; ++i) r[i] = __uint_as_float(v[i]);
  }
  static __device__ __forceinline__ void st(uint32_t a, const float* r) {
    asm volatile("tcgen05.st.sync.aligned.32x32b.x8.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8};" ::"r"(a),
                 "r"(__float_as_uint(r[0])), "r"(__float_as_uint(r[1])), "r"(__float_as_uint(r[2])), "r"(__float_as_uint(r[3])),
                 "r"(__float_as_uint(r[4])), "r"(__float_as_uint(r[5])), "r"(__float_as_uint(r[6])), "r"(__float_as_uint(r[7])) : "memory");
    asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
  }
};
template <> struct TmemVec<16> {
  static __device__ __forceinline__ void ld(uint32_t a, float* r) {
    uint32_t v[16];
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];"
                 : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]),
                   "=r"(v[8]), "=r"(v[9]), "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15]) : "r"(a));
    asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
#pragma unroll
    for (int i = 0; i < 16; ++i) r[i] = __uint_as_float(v[i]);
  }
  static __device__ __forceinline__ void st(uint32_t a, const float* r) {
    asm volatile("tcgen05.st.sync.aligned.32x32b.x16.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16};" ::"r"(a),
                 "r"(__float_as_uint(r[0])), "r"(__float_as_uint(r[1])), "r"(__float_as_uint(r[2])), "r"(__float_as_uint(r[3])),
                 "r"(__float_as_uint(r[4])), "r"(__float_as_uint(r[5])), "r"(__float_as_uint(r[6])), "r"(__float_as_uint(r[7])),
                 "r"(__float_as_uint(r[8])), "r"(__float_as_uint(r[9])), "r"(__float_as_uint(r[10])), "r"(__float_as_uint(r[11])),
                 "r"(__float_as_uint(r[12])), "r"(__float_as_uint(r[13])), "r"(__float_as_uint(r[14])), "r"(__float_as_uint(r[15])) : "memory");
    asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
  }
};

// Shared-memory matrix descriptor (tcgen05 "smem descriptor", version 1): start address, leading / stride byte offsets
// (all >> 4), SWIZZLE_128B.  K-major operands: LBO unused (1), SBO = 1024 (8 rows x 128 bytes).  MN-major operand (V):
// LBO = stride between the two 64-dim panels, SBO = 1024 (8 keys x 128 bytes).
__device__ __forceinline__ uint64_t smem_desc(uint32_t addr, uint32_t lbo_bytes, uint32_t sbo_bytes) {
  return (uint64_t)((addr & 0x3FFFFu) >> 4) | ((uint64_t)(lbo_bytes >> 4) << 16) | ((uint64_t)(sbo_bytes >> 4) << 32) |
         (1ull << 46) | (2ull << 61);
}
// Instruction descriptor, kind::f16: D = fp32, A = B = bf16, N = 16, M = 128; a_mn: A is MN-major.
__host__ __device__ constexpr uint32_t instr_desc(bool a_mn) {
  return (1u << 4) | (1u << 7) | (1u << 10) | ((a_mn ? 1u : 0u) << 15) | ((16u >> 3) << 17) | ((128u >> 4) << 24);
}
// byte offset of element (row r < 16, column c < 128) of a 16-row K-major SW128 operand (Q' or P): two panels of 64
// columns; inside a panel rows are 128 bytes and the 16-byte chunk index is XORed with (row % 8)
__device__ __forceinline__ uint32_t opnd_off(int r, int c) {
  const int panel = c >> 6, cb = (c & 63) * 2;
  return (uint32_t)(panel * 2048 + r * 128 + ((((cb >> 4) ^ (r & 7))) << 4) + (cb & 15));
}

__device__ __forceinline__ void named_bar_sync(int id, int n) { asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(n) : "memory"); }

}  // namespace

template <int GP>    // query heads per kv head, padded to 4 / 8 / 16 (columns of S^T and O^T that are read back)
__global__ void __launch_bounds__(kThreads, 1) kvr_attend_kernel(const __grid_constant__ AttnParams P) {
  extern __shared__ unsigned char smem_raw[];
  const uint32_t s_base = (smem_u32(smem_raw) + 1023u) & ~1023u;
  unsigned char* const smem = smem_raw + (s_base - smem_u32(smem_raw));
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int G = P.group;

  // barriers
  auto bar = [&](int i) { return s_base + kOffBar + 8u * i; };
  const int B_KFULL = 0, B_VFULL = kStages, B_EMPTY = 2 * kStages, B_SFULL = 3 * kStages, B_SEMPTY = B_SFULL + 2,
            B_PFULL = B_SEMPTY + 2, B_PEMPTY = B_PFULL + 2, B_QFULL = B_PEMPTY + 2, B_QEMPTY = B_QFULL + 2,
            B_OFULL = B_QEMPTY + 2, B_OEMPTY = B_OFULL + 1;
  uint32_t* const tmem_slot = reinterpret_cast<uint32_t*>(smem + kOffMisc);

  if (threadIdx.x == 0) {
    for (int s = 0; s < kStages; ++s) { mbar_init(bar(B_KFULL + s), 1); mbar_init(bar(B_VFULL + s), 1); mbar_init(bar(B_EMPTY + s), 1); }
    for (int b = 0; b < 2; ++b) {
      mbar_init(bar(B_SFULL + b), 1); mbar_init(bar(B_SEMPTY + b), 128);
      mbar_init(bar(B_PFULL + b), 128); mbar_init(bar(B_PEMPTY + b), 1);
      mbar_init(bar(B_QFULL + b), 64); mbar_init(bar(B_QEMPTY + b), 1);
    }
    mbar_init(bar(B_OFULL), 1); mbar_init(bar(B_OEMPTY), 128);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  // zero both Q' and both P operands once: their rows >= G stay zero for the whole launch
  for (int i = threadIdx.x; i < (4 * kQB) / 16; i += kThreads) reinterpret_cast<uint4*>(smem + kOffQ)[i] = make_uint4(0, 0, 0, 0);
  if (warp == 1) {    // TMEM: 64 columns (S0 at 0, S1 at 16, O^T at 32), allocated and freed by the MMA warp
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(tmem_slot)), "r"(64u) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
  }
  fence_async_smem();
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = *tmem_slot;
  const uint32_t tm_s0 = tmem, tm_o = tmem + 32u;

  auto item_tiles = [&](const AttnItem& it) { return (it.n_keys + kTile - 1) / kTile; };

  if (warp == 0) {
    // =========================================================================== TMA PRODUCER
    if (lane == 0) {
      const uint64_t pol = policy_evict_first();
      uint32_t gt = 0;
      for (int ii = blockIdx.x; ii < P.n_items; ii += gridDim.x) {
        const AttnItem it = P.items[ii];
        const AttnSeg* sg = P.segs + it.seg;
        const int nt = item_tiles(it);
        for (int t = 0; t < nt; ++t, ++gt) {
          const int st = gt % kStages;
          const uint32_t ph = (gt / kStages) & 1u;
          mbar_wait(bar(B_EMPTY + st), ph ^ 1u, 10);
          const int tok = it.key0 + t * kTile;
          const uint32_t sk = s_base + kOffK + st * kTileB, sv = s_base + kOffV + st * kTileB;
          mbar_arrive_expect_tx(bar(B_KFULL + st), kTileB);
          tensor_g2s_4d(sk, &sg->k, 0, tok, it.head, P.layer, bar(B_KFULL + st), pol);
          tensor_g2s_4d(sk + kPanelB, &sg->k, 64, tok, it.head, P.layer, bar(B_KFULL + st), pol);
          mbar_arrive_expect_tx(bar(B_VFULL + st), kTileB);
          tensor_g2s_4d(sv, &sg->v, 0, tok, it.head, P.layer, bar(B_VFULL + st), pol);
          tensor_g2s_4d(sv + kPanelB, &sg->v, 64, tok, it.head, P.layer, bar(B_VFULL + st), pol);
        }
      }
    }
    __syncwarp();
  } else if (warp == 1) {
    // =========================================================================== MMA ISSUER
    if (lane == 0) {
      constexpr uint32_t idesc_qk = instr_desc(false), idesc_pv = instr_desc(true);
      uint32_t gt = 0, ic = 0;
      auto issue_qk = [&](uint32_t g, int qb) {      // S[g & 1] = K tile (stage g % kStages) . Q'[qb]^T
        const int st = g % kStages, sb = g & 1u;
        const uint32_t u = g >> 1;
        mbar_wait(bar(B_KFULL + st), (g / kStages) & 1u, 20);
        if (u > 0) mbar_wait(bar(B_SEMPTY + sb), (u - 1u) & 1u, 21);
        tc_fence_after();
        const uint32_t ka = s_base + kOffK + st * kTileB, qa = s_base + kOffQ + qb * kQB;
#pragma unroll
        for (int k = 0; k < 8; ++k) {               // 8 x 16 dims; dims 64.. are the second panel
          const uint32_t ko = (k >> 2) * kPanelB + (k & 3) * 32, qo = (k >> 2) * 2048 + (k & 3) * 32;
          tc_mma(tm_s0 + 16u * sb, smem_desc(ka + ko, 16, 1024), smem_desc(qa + qo, 16, 1024), idesc_qk, k > 0);
        }
        tc_commit(bar(B_SFULL + sb));
      };
      for (int ii = blockIdx.x; ii < P.n_items; ii += gridDim.x, ++ic) {
        const AttnItem it = P.items[ii];
        const int nt = item_tiles(it);
        const int qb = ic & 1u;
        mbar_wait(bar(B_QFULL + qb), (ic >> 1) & 1u, 22);
        issue_qk(gt, qb);
        for (int t = 0; t < nt; ++t) {
          const uint32_t g = gt + t;
          if (t + 1 < nt) issue_qk(g + 1, qb);
          else tc_commit(bar(B_QEMPTY + qb));        // every QK of this item has been issued: Q'[qb] is free once they complete
          const int st = g % kStages, pb = g & 1u;
          mbar_wait(bar(B_PFULL + pb), (g >> 1) & 1u, 23);
          mbar_wait(bar(B_VFULL + st), (g / kStages) & 1u, 24);
          if (t == 0 && ic > 0) mbar_wait(bar(B_OEMPTY), (ic - 1u) & 1u, 25);
          tc_fence_after();
          const uint32_t va = s_base + kOffV + st * kTileB, pa = s_base + kOffP + pb * kQB;
#pragma unroll
          for (int k = 0; k < 8; ++k) {             // 8 x 16 keys
            const uint32_t po = (k >> 2) * 2048 + (k & 3) * 32;
            tc_mma(tm_o, smem_desc(va + k * 2048, kPanelB, 1024), smem_desc(pa + po, 16, 1024), idesc_pv, (t > 0 || k > 0) ? 1u : 0u);
          }
          tc_commit(bar(B_EMPTY + st));             // K and V of this stage are consumed
          tc_commit(bar(B_PEMPTY + pb));
          if (t + 1 == nt) tc_commit(bar(B_OFULL));
        }
        gt += nt;
      }
    }
    __syncwarp();
  } else if (warp < 4) {
    // =========================================================================== QUERY WARPS
    const int tid = threadIdx.x - 64;              // 0..63
    const int half_R = P.rotary_dim >> 1;
    uint32_t ic = 0;
    for (int ii = blockIdx.x; ii < P.n_items; ii += gridDim.x, ++ic) {
      const AttnItem it = P.items[ii];
      const AttnSeg* sg = P.segs + it.seg;
      const int qb = ic & 1u;
      if (ic >= 2) mbar_wait(bar(B_QEMPTY + qb), ((ic >> 1) - 1u) & 1u, 30);
      unsigned char* const qs = smem + kOffQ + qb * kQB;
      const uint16_t* const qg = P.q + ((int64_t)sg->request * P.q_heads + (int64_t)it.head * G) * kD;
      // dims outside the rotary window are position-free: copied
      for (int idx = tid; idx < G * kD; idx += 64) {
        const int g = idx >> 7, d = idx & 127;
        if (d < P.rotary_offset || d >= P.rotary_offset + P.rotary_dim)
          *reinterpret_cast<uint16_t*>(qs + opnd_off(g, d)) = qg[g * kD + d];
      }
      // q' = R(-Delta) q: (a, b) -> (a c + b s, b c - a s) with (c, s) = cos / sin(Delta * inv_freq[i]), fp64, one rounding
      const int64_t delta = sg->delta;
      for (int i = tid; i < half_R; i += 64) {
        double sn, cs;
        sincos((double)delta * P.inv_freq[i], &sn, &cs);
        const int ia = P.rotary_offset + (P.pairing == 0 ? i : 2 * i), ib = P.rotary_offset + (P.pairing == 0 ? i + half_R : 2 * i + 1);
        for (int g = 0; g < G; ++g) {
          const double a = (double)bf16_bits_to_f32(qg[g * kD + ia]), b = (double)bf16_bits_to_f32(qg[g * kD + ib]);
          const double ra = a * cs + b * sn, rb = b * cs - a * sn;
          *reinterpret_cast<uint16_t*>(qs + opnd_off(g, ia)) = (uint16_t)f32_to_bf16_bits((float)ra);
          *reinterpret_cast<uint16_t*>(qs + opnd_off(g, ib)) = (uint16_t)f32_to_bf16_bits((float)rb);
        }
      }
      fence_async_smem();
      mbar_arrive(bar(B_QFULL + qb));
    }
  } else {
    // =========================================================================== SOFTMAX + EPILOGUE
    const int tid = threadIdx.x - 128;             // 0..127 = TMEM lane = key of the tile (softmax) / dim (epilogue)
    const int w4 = warp - 4;
    const uint32_t lane_base = (uint32_t)(w4 * 32) << 16;
    float* const red = reinterpret_cast<float*>(smem + kOffRed);       // [4 warps][16]
    uint32_t gt = 0, ic = 0;
    for (int ii = blockIdx.x; ii < P.n_items; ii += gridDim.x, ++ic) {
      const AttnItem it = P.items[ii];
      const int nt = item_tiles(it);
      float m_ref[GP], l_thr[GP];
#pragma unroll
      for (int g = 0; g < GP; ++g) { m_ref[g] = -INFINITY; l_thr[g] = 0.0f; }
      for (int t = 0; t < nt; ++t, ++gt) {
        const int sb = gt & 1u;
        const uint32_t u = gt >> 1;
        mbar_wait(bar(B_SFULL + sb), u & 1u, 40);
        tc_fence_after();
        float x[GP];
        TmemVec<GP>::ld(tm_s0 + 16u * sb + lane_base, x);
        tc_fence_before();
        mbar_arrive(bar(B_SEMPTY + sb));
        const bool valid = t * kTile + tid < it.n_keys;
        float mx[GP];
#pragma unroll
        for (int g = 0; g < GP; ++g) { x[g] = valid ? x[g] * P.scale_log2 : -INFINITY; mx[g] = x[g]; }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1)
#pragma unroll
          for (int g = 0; g < GP; ++g) mx[g] = fmaxf(mx[g], __shfl_xor_sync(0xFFFFFFFFu, mx[g], o));
        named_bar_sync(1, 128);                    // the previous tile's readers of `red` are done
        if (lane == 0)
#pragma unroll
          for (int g = 0; g < GP; ++g) red[w4 * 16 + g] = mx[g];
        named_bar_sync(1, 128);
        bool move = false;
#pragma unroll
        for (int g = 0; g < GP; ++g) {
          mx[g] = fmaxf(fmaxf(red[g], red[16 + g]), fmaxf(red[32 + g], red[48 + g]));
          move |= mx[g] > m_ref[g] + (float)kRescaleLog2;
        }
        if (move) {     // uniform over the 128 threads (every thread sees the same tile maxima)
          float alpha[GP];
#pragma unroll
          for (int g = 0; g < GP; ++g) {
            const float nm = fmaxf(m_ref[g], mx[g]);
            alpha[g] = (m_ref[g] == -INFINITY) ? 0.0f : exp2f(m_ref[g] - nm);
            l_thr[g] *= alpha[g];
            m_ref[g] = nm;
          }
          if (t > 0) {  // O^T holds the tiles before this one: wait for the last P.V to complete, then rescale its columns
            const uint32_t gp = gt - 1u;
            mbar_wait(bar(B_PEMPTY + (gp & 1u)), (gp >> 1) & 1u, 41);
            tc_fence_after();
            float o[GP];
            TmemVec<GP>::ld(tm_o + lane_base, o);
#pragma unroll
            for (int g = 0; g < GP; ++g) o[g] *= alpha[g];
            TmemVec<GP>::st(tm_o + lane_base, o);
            tc_fence_before();
          }
        }
        const int pb = gt & 1u;
        if (u > 0) mbar_wait(bar(B_PEMPTY + pb), (u - 1u) & 1u, 42);     // the P.V that read this buffer two tiles ago
        unsigned char* const ps = smem + kOffP + pb * kQB;
#pragma unroll
        for (int g = 0; g < GP; ++g) {
          const float p = exp2f(x[g] - m_ref[g]);
          // the row sum adds what the tensor core will multiply: p rounded to bf16
          const uint32_t pbits = f32_to_bf16_bits(p);
          l_thr[g] += bf16_bits_to_f32(pbits);
          if (g < G) *reinterpret_cast<uint16_t*>(ps + opnd_off(g, tid)) = (uint16_t)pbits;
        }
        fence_async_smem();
        tc_fence_before();
        mbar_arrive(bar(B_PFULL + pb));
      }
      // ---- end of the item: O^T (thread = dim), row sums, reference maxima ----
      mbar_wait(bar(B_OFULL), ic & 1u, 43);
      tc_fence_after();
      float o[GP];
      TmemVec<GP>::ld(tm_o + lane_base, o);
      tc_fence_before();
      mbar_arrive(bar(B_OEMPTY));
#pragma unroll
      for (int off = 16; off > 0; off >>= 1)
#pragma unroll
        for (int g = 0; g < GP; ++g) l_thr[g] += __shfl_xor_sync(0xFFFFFFFFu, l_thr[g], off);
      named_bar_sync(1, 128);
      if (lane == 0)
#pragma unroll
        for (int g = 0; g < GP; ++g) red[w4 * 16 + g] = l_thr[g];
      named_bar_sync(1, 128);
      float l[GP];
#pragma unroll
      for (int g = 0; g < GP; ++g) l[g] = (red[g] + red[16 + g]) + (red[32 + g] + red[48 + g]);
      const int64_t out_row = (int64_t)it.out_q0;          // first query head row of this group in o / lse
      if (it.group_count == 1) {
#pragma unroll
        for (int g = 0; g < GP; ++g)
          if (g < G) {
            P.o[(out_row + g) * kD + tid] = o[g] / l[g];
            if (tid == 0) P.lse[out_row + g] = (m_ref[g] + log2f(l[g])) * 0.6931471805599453f;
          }
      } else {
        float* const po = P.part_o + (int64_t)ii * G * kD;
#pragma unroll
        for (int g = 0; g < GP; ++g)
          if (g < G) {
            po[g * kD + tid] = o[g];
            if (tid == 0) { P.part_ml[((int64_t)ii * G + g) * 2] = m_ref[g]; P.part_ml[((int64_t)ii * G + g) * 2 + 1] = l[g]; }
          }
        __threadfence();
        named_bar_sync(1, 128);
        int* const flag = reinterpret_cast<int*>(smem + kOffMisc + 16);
        if (tid == 0) *flag = (atomicAdd(P.tickets + it.group, 1u) == (unsigned)it.group_count - 1u) ? 1 : 0;
        named_bar_sync(1, 128);
        if (*flag) {     // the last item of the group merges the group's partials (thread = dim)
          __threadfence();
          for (int g = 0; g < G; ++g) {
            float M = -INFINITY;
            for (int j = 0; j < it.group_count; ++j) M = fmaxf(M, __ldcg(P.part_ml + ((int64_t)(it.group_first + j) * G + g) * 2));
            float L = 0.0f, acc = 0.0f;
            for (int j = 0; j < it.group_count; ++j) {
              const int64_t pi = (int64_t)(it.group_first + j);
              const float w = exp2f(__ldcg(P.part_ml + (pi * G + g) * 2) - M);
              L += w * __ldcg(P.part_ml + (pi * G + g) * 2 + 1);
              acc += w * __ldcg(P.part_o + (pi * G + g) * kD + tid);
            }
            P.o[(out_row + g) * kD + tid] = acc / L;
            if (tid == 0) P.lse[out_row + g] = (M + log2f(L)) * 0.6931471805599453f;
          }
          if (tid == 0) P.tickets[it.group] = 0u;      // re-armed for the next launch
        }
      }
    }
  }
  // teardown: every tcgen05 operation of this CTA has completed once the softmax warps have seen their last o_full
  tc_fence_before();
  __syncthreads();
  if (warp == 1) {
    tc_fence_after();
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem), "r"(64u) : "memory");
  }
}

// ------------------------------------------------------------------------------- host side
template <int GP>
static cudaError_t launch_attend_inst(const AttnParams& P, int grid, cudaStream_t st) {
  static std::mutex mu;
  static bool configured[64] = {};
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  {
    std::lock_guard<std::mutex> lock(mu);
    if (dev < 0 || dev >= 64 || !configured[dev]) {
      e = cudaFuncSetAttribute(kvr_attend_kernel<GP>, cudaFuncAttributeMaxDynamicSharedMemorySize, kSmemBytes);
      if (e != cudaSuccess) return e;
      if (dev >= 0 && dev < 64) configured[dev] = true;
    }
  }
  kvr_attend_kernel<GP><<<grid, kThreads, kSmemBytes, st>>>(P);
  return cudaGetLastError();
}

cudaError_t launch_attend(const AttnParams& P, int sm_count, cudaStream_t stream, int* grid_out, int* block_out, int* smem_out) {
  int grid = P.n_items < sm_count ? P.n_items : sm_count;
  if (grid < 1) grid = 1;
  *grid_out = grid; *block_out = kThreads; *smem_out = kSmemBytes;
  if (P.group <= 4) return launch_attend_inst<4>(P, grid, stream);
  if (P.group <= 8) return launch_attend_inst<8>(P, grid, stream);
  return launch_attend_inst<16>(P, grid, stream);
}

}  // namespace kvr
