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
// One CTA per SM (384 threads, ~211 KB of shared memory, 64 TMEM columns), persistent over work items = (segment, kv
// head, run of 4..8 key tiles of 128 keys), warp-specialised:
//   warp 0 / 2  TMA producers (one elected lane each): K tiles / V tiles, each a pair of 64-dim panels of 128 keys
//               (SWIZZLE_128B tensor loads), into rings of kKS / kVS slots of 32 KB.  The rings are separate because
//               a K slot is free as soon as S^T is computed, while a V slot is held until P^T has multiplied it.
//   warp 1      MMA issuer (one elected lane): tcgen05.mma kind::f16 (M 128, N 16, K 16), accumulators in TMEM: S^T
//               double-buffered by tile, O^T double-buffered by item; the first S^T of the next item is issued before
//               the last P.V of this one is waited for.
//   warp 3      scheduler + query warp: lane 0 draws items (the first statically, the rest from one global counter, a
//               draw ahead) and publishes them to the other roles through a 4-slot ring in shared memory; the warp
//               then builds the item's Q' = R(-Delta) q (fp64 sincos, one rounding to bf16) in the swizzled operand
//               layout, double-buffered, an item ahead of the MMAs.
//   warps 4-7   softmax: thread i owns key i of the tile (TMEM lane i): tcgen05.ld of its <= 16 scores, tile maximum by
//               warp shuffles + ONE named barrier, exp2, P^T to shared memory as the next MMA's B operand.  The
//               reference maximum only moves when a tile exceeds it by 2^8 (O^T is then rescaled in TMEM: 16 columns,
//               one tcgen05.ld/st pair per thread).  At the end of an item the reference and the row sums go to the
//               epilogue warps through shared memory and the next item starts at once.
//   warps 8-11  epilogue, off the critical path: O^T (thread = dim) of a finished item goes to the output (a group of
//               one item) or to the partial buffer.  A (request, kv head) group of few partials is merged by its last
//               item (device-scope fence + ticket); a group of many is left to kvr_attend_merge_kernel after the
//               grid, because under a saturated HBM every dependent load of an in-kernel merge costs microseconds
//               (measured: a 512-partial in-kernel merge was a 600 us serial tail).
// Programmatic dependent launch: the prologue (barriers, TMEM allocation) and -- for precompiled skills
// (KVR_SEG_SRC_STABLE) -- the K / V loads of the first item overlap the tail of the previous launch.
#include <mutex>

#include "kvr_attend.cuh"
#include "kvr_ptx.cuh"

namespace kvr {

namespace {

constexpr int kD = 128;                 // head_dim this kernel is built for
constexpr int kTile = 128;              // keys per tile = rows of one MMA
#ifndef KVR_ATTN_KS
#define KVR_ATTN_KS 3
#endif
#ifndef KVR_ATTN_VS
#define KVR_ATTN_VS 3
#endif
constexpr int kKS = KVR_ATTN_KS;                // K tiles in flight per CTA (32 KB each); a K slot is free as soon as S^T is computed
constexpr int kVS = KVR_ATTN_VS;                // V tiles in flight per CTA (32 KB each); a V slot is held until P^T has multiplied it
constexpr int kIR = 4;                  // work items the scheduler may publish ahead
constexpr int kPanelB = kTile * 128;    // one 64-dim panel of a tile: 128 rows x 128 bytes
constexpr int kTileB = 2 * kPanelB;     // K (or V) tile: 32 KB
constexpr int kQB = 2 * 16 * 128;       // Q' / P operand: 2 panels x 16 rows x 128 bytes
constexpr int kThreads = 384;           // 12 warps: K producer, MMA, V producer, query + scheduler, 4 softmax, 4 epilogue
constexpr int kRescaleLog2 = 8;         // the reference maximum moves only when a tile exceeds it by 2^8

// shared-memory layout (offsets from a 1024-byte aligned base)
constexpr int kOffK = 0;
constexpr int kOffV = kKS * kTileB;
constexpr int kOffQ = (kKS + kVS) * kTileB;
constexpr int kOffP = kOffQ + 2 * kQB;
constexpr int kOffBar = kOffP + 2 * kQB;
// barriers: kfull, kempty | vfull, vempty | s_full/empty, p_full/empty, q_full/empty, o_full/empty, st_full/empty | item full/empty
constexpr int kNumBars = 2 * kKS + 2 * kVS + 10 * 2 + 2 * kIR;
constexpr int kOffRed = kOffBar + 8 * kNumBars;            // softmax tile maxima: [2 tile parities][4 warps][16]
constexpr int kOffStat = kOffRed + 2 * 4 * 16 * 4;         // item statistics handed to the epilogue: [2][16 m_ref + 4 x 16 row sums]
constexpr int kOffItem = kOffStat + 2 * 80 * 4;            // published work items: [kIR] AttnItem
constexpr int kOffMisc = kOffItem + kIR * 32;
constexpr int kSmemBytes = kOffMisc + 64 + 1024;   // + slack for the 1024-byte alignment of the base
static_assert(sizeof(AttnItem) == 32, "AttnItem layout");
static_assert(kSmemBytes <= 227 * 1024, "shared memory");

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
  constexpr int B_KFULL = 0, B_KEMPTY = kKS, B_VFULL = 2 * kKS, B_VEMPTY = 2 * kKS + kVS, B0 = 2 * kKS + 2 * kVS,
                B_SFULL = B0, B_SEMPTY = B0 + 2, B_PFULL = B0 + 4, B_PEMPTY = B0 + 6, B_QFULL = B0 + 8, B_QEMPTY = B0 + 10,
                B_OFULL = B0 + 12, B_OEMPTY = B0 + 14, B_STFULL = B0 + 16, B_STEMPTY = B0 + 18, B_IFULL = B0 + 20,
                B_IEMPTY = B_IFULL + kIR;
  uint32_t* const tmem_slot = reinterpret_cast<uint32_t*>(smem + kOffMisc);
  const AttnItem* const item_ring = reinterpret_cast<const AttnItem*>(smem + kOffItem);

  if (threadIdx.x == 0) {
    for (int s = 0; s < kKS; ++s) { mbar_init(bar(B_KFULL + s), 1); mbar_init(bar(B_KEMPTY + s), 1); }
    for (int s = 0; s < kVS; ++s) { mbar_init(bar(B_VFULL + s), 1); mbar_init(bar(B_VEMPTY + s), 1); }
    for (int b = 0; b < 2; ++b) {
      mbar_init(bar(B_SFULL + b), 1); mbar_init(bar(B_SEMPTY + b), 128);
      mbar_init(bar(B_PFULL + b), 128); mbar_init(bar(B_PEMPTY + b), 1);
      mbar_init(bar(B_QFULL + b), 32); mbar_init(bar(B_QEMPTY + b), 1);
      mbar_init(bar(B_OFULL + b), 1); mbar_init(bar(B_OEMPTY + b), 128);
      mbar_init(bar(B_STFULL + b), 128); mbar_init(bar(B_STEMPTY + b), 128);
    }
    // an item is read by the K producer, the MMA issuer, the V producer, 128 softmax and 128 epilogue threads
    for (int s = 0; s < kIR; ++s) { mbar_init(bar(B_IFULL + s), 1); mbar_init(bar(B_IEMPTY + s), 3 + 128 + 128); }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  // zero both Q' and both P operands once: their rows >= G stay zero for the whole launch
  for (int i = threadIdx.x; i < (4 * kQB) / 16; i += kThreads) reinterpret_cast<uint4*>(smem + kOffQ)[i] = make_uint4(0, 0, 0, 0);
  if (warp == 1) {    // TMEM: 64 columns (S0 at 0, S1 at 16, O0^T at 32, O1^T at 48), allocated and freed by the MMA warp
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(tmem_slot)), "r"(64u) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
  }
  fence_async_smem();
  tc_fence_before();
  // Programmatic dependent launch: everything above touches only this CTA's shared memory and TMEM and may overlap
  // the tail of the previous launch on the stream.  That launch's partial buffers, tickets, item counter and outputs are
  // reused by this one, and the query may be its product: griddepcontrol.wait is executed per role, by the threads that
  // touch such memory -- the scheduler / query warp (the query, the item counter) and the epilogue warps (outputs,
  // partials, tickets).  The work items and tensor maps were staged before this kernel could start.  With P.early (every segment carries
  // KVR_SEG_SRC_STABLE: precompiled skills) the TMA producers do NOT wait: the K / V tiles of the CTA's first item
  // stream in while the previous kernel on the stream drains; otherwise they wait as well.
  asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
  __syncthreads();
  tc_fence_after();
  auto dependency_wait = [] { asm volatile("griddepcontrol.wait;" ::: "memory"); };
  const uint32_t tmem = *tmem_slot;
  const uint32_t tm_s0 = tmem, tm_o0 = tmem + 32u;

  // Work items come from the scheduler (query warp) through a small ring in shared memory: item number n of this CTA
  // sits in slot n % kIR once its "full" barrier has completed phase n / kIR; seg < 0 ends the stream.
  auto take_item = [&](uint32_t n, int who) -> AttnItem {
    const int slot = n % kIR;
    mbar_wait(bar(B_IFULL + slot), (n / kIR) & 1u, who);
    const AttnItem it = item_ring[slot];
    mbar_arrive(bar(B_IEMPTY + slot));
    return it;
  };
  auto item_tiles = [&](const AttnItem& it) { return (it.n_keys + kTile - 1) / kTile; };

  if (warp == 0 || warp == 2) {
    // =========================================================================== TMA PRODUCERS (warp 0: K, warp 2: V)
    if (lane == 0) {
      if (!P.early) dependency_wait();
      const bool is_k = warp == 0;
      const int NS = is_k ? kKS : kVS;
      const int b_full = is_k ? B_KFULL : B_VFULL, b_empty = is_k ? B_KEMPTY : B_VEMPTY;
      const uint32_t s_tiles = s_base + (is_k ? kOffK : kOffV);
      const uint64_t pol = policy_evict_first();
      uint32_t gt = 0;
      for (uint32_t n = 0;; ++n) {
        const AttnItem it = take_item(n, 10);
        if (it.seg < 0) break;
        const AttnSeg* sg = P.segs + it.seg;
        const CUtensorMap* map = is_k ? &sg->k : &sg->v;
        const int nt = item_tiles(it);
        for (int t = 0; t < nt; ++t, ++gt) {
          const int st = gt % NS;
          mbar_wait(bar(b_empty + st), ((gt / NS) & 1u) ^ 1u, 11);
          const int tok = it.key0 + t * kTile;
          const uint32_t dst = s_tiles + st * kTileB;
          mbar_arrive_expect_tx(bar(b_full + st), kTileB);
          tensor_g2s_4d(dst, map, 0, tok, it.head, P.layer, bar(b_full + st), pol);
          tensor_g2s_4d(dst + kPanelB, map, 64, tok, it.head, P.layer, bar(b_full + st), pol);
        }
      }
    }
    __syncwarp();
  } else if (warp == 1) {
    // =========================================================================== MMA ISSUER
    if (lane == 0) {
      constexpr uint32_t idesc_qk = instr_desc(false), idesc_pv = instr_desc(true);
      uint32_t gt = 0;
      auto issue_qk = [&](uint32_t g, int qb) {      // S[g & 1] = K tile (slot g % kKS) . Q'[qb]^T
        const int st = g % kKS, sb = g & 1u;
        const uint32_t u = g >> 1;
        mbar_wait(bar(B_KFULL + st), (g / kKS) & 1u, 20);
        if (u > 0) mbar_wait(bar(B_SEMPTY + sb), (u - 1u) & 1u, 21);
        tc_fence_after();
        const uint32_t ka = s_base + kOffK + st * kTileB, qa = s_base + kOffQ + qb * kQB;
#pragma unroll
        for (int k = 0; k < 8; ++k) {               // 8 x 16 dims; dims 64.. are the second panel
          const uint32_t ko = (k >> 2) * kPanelB + (k & 3) * 32, qo = (k >> 2) * 2048 + (k & 3) * 32;
          tc_mma(tm_s0 + 16u * sb, smem_desc(ka + ko, 16, 1024), smem_desc(qa + qo, 16, 1024), idesc_qk, k > 0);
        }
        tc_commit(bar(B_KEMPTY + st));               // the K slot is free as soon as these have read it
        tc_commit(bar(B_SFULL + sb));
      };
      // The first S^T of the NEXT item is issued before this item's last P.V is waited for (the softmax warps then find
      // it ready when they cross the item boundary), so items are taken one ahead.
      AttnItem it = take_item(0, 22);
      if (it.seg >= 0) {
        mbar_wait(bar(B_QFULL + 0), 0u, 23);
        issue_qk(0, 0);
      }
      for (uint32_t ic = 0; it.seg >= 0; ++ic) {
        const int nt = item_tiles(it);
        const int qb = ic & 1u;
        const uint32_t tm_o = tm_o0 + 16u * (ic & 1u);
        AttnItem nx{};
        nx.seg = -1;
        for (int t = 0; t < nt; ++t) {
          const uint32_t g = gt + t;
          if (t + 1 < nt) {
            issue_qk(g + 1, qb);
          } else {
            tc_commit(bar(B_QEMPTY + qb));           // every QK of this item has been issued: Q'[qb] is free once they complete
            nx = take_item(ic + 1u, 22);
            if (nx.seg >= 0) {
              mbar_wait(bar(B_QFULL + (qb ^ 1)), ((ic + 1u) >> 1) & 1u, 23);
              issue_qk(g + 1, qb ^ 1);
            }
          }
          const int st = g % kVS, pb = g & 1u;
          mbar_wait(bar(B_PFULL + pb), (g >> 1) & 1u, 24);
          mbar_wait(bar(B_VFULL + st), (g / kVS) & 1u, 25);
          if (t == 0 && ic >= 2) mbar_wait(bar(B_OEMPTY + (ic & 1u)), ((ic >> 1) - 1u) & 1u, 26);
          tc_fence_after();
          const uint32_t va = s_base + kOffV + st * kTileB, pa = s_base + kOffP + pb * kQB;
#pragma unroll
          for (int k = 0; k < 8; ++k) {             // 8 x 16 keys
            const uint32_t po = (k >> 2) * 2048 + (k & 3) * 32;
            tc_mma(tm_o, smem_desc(va + k * 2048, kPanelB, 1024), smem_desc(pa + po, 16, 1024), idesc_pv, (t > 0 || k > 0) ? 1u : 0u);
          }
          tc_commit(bar(B_VEMPTY + st));
          tc_commit(bar(B_PEMPTY + pb));
          if (t + 1 == nt) tc_commit(bar(B_OFULL + (ic & 1u)));
        }
        gt += nt;
        it = nx;
      }
    }
    __syncwarp();
  } else if (warp == 3) {
    // =========================================================================== SCHEDULER + QUERY WARP
    // Lane 0 draws work items (the first one statically, the rest from one global counter, each draw requested an
    // item ahead so its latency is hidden) and publishes them to the CTA; the warp then builds the item's Q'.
    const int half_R = P.rotary_dim >> 1;
    AttnItem* const ring_w = reinterpret_cast<AttnItem*>(smem + kOffItem);
    unsigned long long nxt = 0;
    int64_t idx = blockIdx.x;
    uint32_t n_pub = 0;
    // lane 0: fetch the next item (or the end marker), publish it, request the draw after it
    auto publish_next = [&](bool first) -> AttnItem {
      AttnItem it{};
      it.seg = -1;
      if (idx < P.n_items) it = P.items[idx];
      if (!first) {
        idx = (int64_t)gridDim.x + (int64_t)nxt;
        if (it.seg >= 0 && idx < P.n_items) nxt = atomicAdd(P.sched, 1ull);
      }
      const int slot = n_pub % kIR;
      if (n_pub >= (uint32_t)kIR) mbar_wait(bar(B_IEMPTY + slot), ((n_pub / kIR) - 1u) & 1u, 30);
      ring_w[slot] = it;
      mbar_arrive(bar(B_IFULL + slot));
      ++n_pub;
      return it;
    };
    AttnItem nx{};
    nx.seg = -1;
    // the first item is static (items[blockIdx.x]) and is published BEFORE the dependency wait, so that the producers
    // can start on it; the item counter (re-armed by the previous launch's last CTA) is only touched after the wait
    if (lane == 0) nx = publish_next(true);
    dependency_wait();
    if (lane == 0) {
      nxt = atomicAdd(P.sched, 1ull);
      idx = (int64_t)gridDim.x + (int64_t)nxt;
      if (idx < P.n_items) nxt = atomicAdd(P.sched, 1ull);
    }
    for (uint32_t ic = 0;; ++ic) {
      AttnItem it = nx;                    // the item whose Q' is built now; the one after it is published first, so
      if (lane == 0 && it.seg >= 0) nx = publish_next(false);   // that the producers can run an item ahead of the query
      it.seg = __shfl_sync(0xFFFFFFFFu, it.seg, 0);
      if (it.seg < 0) break;
      it.head = __shfl_sync(0xFFFFFFFFu, it.head, 0);
      const AttnSeg* sg = P.segs + it.seg;
      const int qb = ic & 1u;
      if (ic >= 2) mbar_wait(bar(B_QEMPTY + qb), ((ic >> 1) - 1u) & 1u, 31);
      unsigned char* const qs = smem + kOffQ + qb * kQB;
      const uint16_t* const qg = P.q + ((int64_t)sg->request * P.q_heads + (int64_t)it.head * G) * kD;
      // dims outside the rotary window are position-free: copied
      if (P.rotary_dim < kD)
        for (int idx2 = lane; idx2 < G * kD; idx2 += 32) {
          const int g = idx2 >> 7, d = idx2 & 127;
          if (d < P.rotary_offset || d >= P.rotary_offset + P.rotary_dim)
            *reinterpret_cast<uint16_t*>(qs + opnd_off(g, d)) = qg[g * kD + d];
        }
      // q' = R(-Delta) q: (a, b) -> (a c + b s, b c - a s) with (c, s) = cos / sin(Delta * inv_freq[i]), fp64, one rounding.
      // A lane's query elements are fetched first, all loads in flight at once (one memory latency per item, not one
      // per head), then rotated.
      const int64_t delta = sg->delta;
      for (int i0 = 0; i0 < half_R; i0 += 32) {
        const int i = i0 + lane;
        const bool on = i < half_R;
        const int ia = P.rotary_offset + (P.pairing == 0 ? i : 2 * i), ib = P.rotary_offset + (P.pairing == 0 ? i + half_R : 2 * i + 1);
        uint16_t qa[GP], qbv[GP];
#pragma unroll
        for (int g = 0; g < GP; ++g) {
          qa[g] = (on && g < G) ? __ldg(qg + g * kD + ia) : (uint16_t)0;
          qbv[g] = (on && g < G) ? __ldg(qg + g * kD + ib) : (uint16_t)0;
        }
        double sn = 0.0, cs = 1.0;
        if (on) sincos((double)delta * P.inv_freq[i], &sn, &cs);
#pragma unroll
        for (int g = 0; g < GP; ++g)
          if (on && g < G) {
            const double a = (double)bf16_bits_to_f32(qa[g]), b = (double)bf16_bits_to_f32(qbv[g]);
            const double ra = a * cs + b * sn, rb = b * cs - a * sn;
            *reinterpret_cast<uint16_t*>(qs + opnd_off(g, ia)) = (uint16_t)f32_to_bf16_bits((float)ra);
            *reinterpret_cast<uint16_t*>(qs + opnd_off(g, ib)) = (uint16_t)f32_to_bf16_bits((float)rb);
          }
      }
      fence_async_smem();
      mbar_arrive(bar(B_QFULL + qb));
    }
    // every CTA's last draw has returned >= n_items once all of them are here: the last one re-arms the counter
    if (lane == 0) {
      __threadfence();
      if (atomicAdd(P.sched + 1, 1ull) == (unsigned long long)gridDim.x - 1ull) {
        P.sched[0] = 0ull; P.sched[1] = 0ull;
        __threadfence();
      }
    }
  } else if (warp < 8) {
    // =========================================================================== SOFTMAX
    const int tid = threadIdx.x - 128;             // 0..127 = TMEM lane = key of the tile
    const int w4 = warp - 4;
    const uint32_t lane_base = (uint32_t)(w4 * 32) << 16;
    float* const red = reinterpret_cast<float*>(smem + kOffRed);       // [2][4 warps][16]
    float* const stat = reinterpret_cast<float*>(smem + kOffStat);     // [2][16 + 4 x 16]
    uint32_t gt = 0;
    for (uint32_t ic = 0;; ++ic) {
      const AttnItem it = take_item(ic, 40);
      if (it.seg < 0) break;
      const int nt = item_tiles(it);
      const uint32_t tm_o = tm_o0 + 16u * (ic & 1u);
      float m_ref[GP], l_thr[GP];
#pragma unroll
      for (int g = 0; g < GP; ++g) { m_ref[g] = -INFINITY; l_thr[g] = 0.0f; }
      for (int t = 0; t < nt; ++t, ++gt) {
        const int sb = gt & 1u;
        const uint32_t u = gt >> 1;
        mbar_wait(bar(B_SFULL + sb), u & 1u, 41);
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
        float* const rd = red + sb * 64;           // double-buffered by tile parity: one barrier per tile
        if (lane == 0)
#pragma unroll
          for (int g = 0; g < GP; ++g) rd[w4 * 16 + g] = mx[g];
        named_bar_sync(1, 128);
        bool move = false;
#pragma unroll
        for (int g = 0; g < GP; ++g) {
          mx[g] = fmaxf(fmaxf(rd[g], rd[16 + g]), fmaxf(rd[32 + g], rd[48 + g]));
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
            mbar_wait(bar(B_PEMPTY + (gp & 1u)), (gp >> 1) & 1u, 42);
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
        if (u > 0) mbar_wait(bar(B_PEMPTY + pb), (u - 1u) & 1u, 43);     // the P.V that read this buffer two tiles ago
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
      // ---- end of the item: hand the reference maxima and the row sums (per warp) to the epilogue warps ----
#pragma unroll
      for (int off = 16; off > 0; off >>= 1)
#pragma unroll
        for (int g = 0; g < GP; ++g) l_thr[g] += __shfl_xor_sync(0xFFFFFFFFu, l_thr[g], off);
      const int sp = ic & 1u;
      if (ic >= 2) mbar_wait(bar(B_STEMPTY + sp), ((ic >> 1) - 1u) & 1u, 44);
      float* const stp = stat + sp * 80;
      if (lane == 0)
#pragma unroll
        for (int g = 0; g < GP; ++g) { stp[16 + w4 * 16 + g] = l_thr[g]; if (w4 == 0) stp[g] = m_ref[g]; }
      __syncwarp();
      mbar_arrive(bar(B_STFULL + sp));
    }
  } else {
    // =========================================================================== EPILOGUE
    // Off the softmax warps' critical path: O^T (thread = dim) of a finished item goes to the output or to the partial
    // buffer; the last item of a (request, kv head) group merges the group's partials.
    const int tid = threadIdx.x - 256;             // 0..127 = TMEM lane = dim
    const int w4 = warp - 8;
    const uint32_t lane_base = (uint32_t)(w4 * 32) << 16;
    const float* const stat = reinterpret_cast<const float*>(smem + kOffStat);
    dependency_wait();
    for (uint32_t ic = 0;; ++ic) {
      const AttnItem it = take_item(ic, 50);
      if (it.seg < 0) break;
      const int sp = ic & 1u;
      const uint32_t ph = (ic >> 1) & 1u;
      mbar_wait(bar(B_STFULL + sp), ph, 51);
      float m_ref[GP], l[GP];
#pragma unroll
      for (int g = 0; g < GP; ++g) {
        const float* stp = stat + sp * 80;
        m_ref[g] = stp[g];
        l[g] = (stp[16 + g] + stp[32 + g]) + (stp[48 + g] + stp[64 + g]);
      }
      mbar_arrive(bar(B_STEMPTY + sp));
      mbar_wait(bar(B_OFULL + sp), ph, 52);
      tc_fence_after();
      float o[GP];
      TmemVec<GP>::ld(tm_o0 + 16u * sp + lane_base, o);
      tc_fence_before();
      mbar_arrive(bar(B_OEMPTY + sp));
      const int64_t out_row = (int64_t)P.segs[it.seg].request * P.q_heads + (int64_t)it.head * G;   // the group's first row of o / lse
      if (it.group_count == 1) {
#pragma unroll
        for (int g = 0; g < GP; ++g)
          if (g < G) {
            P.o[(out_row + g) * kD + tid] = o[g] / l[g];
            if (tid == 0) P.lse[out_row + g] = (m_ref[g] + log2f(l[g])) * 0.6931471805599453f;
          }
      } else {
        const int64_t ii = it.index;
        float* const po = P.part_o + ii * G * kD;
#pragma unroll
        for (int g = 0; g < GP; ++g)
          if (g < G) {
            po[g * kD + tid] = o[g];
            if (tid == 0) { P.part_ml[(ii * G + g) * 2] = m_ref[g]; P.part_ml[(ii * G + g) * 2 + 1] = l[g]; }
          }
        // A group with more partials than one merge step takes is merged by kvr_attend_merge_kernel after this grid
        // (group_count < 0): its items only leave their partials -- no fence, no ticket.
        if (it.group_count < 0) continue;
        // release: the barrier orders the 128 threads' partial writes before thread 0's (cumulative) device-scope fence
        named_bar_sync(2, 128);
        int* const flag = reinterpret_cast<int*>(smem + kOffMisc + 16);
        if (tid == 0) {
          __threadfence();
          const int last = atomicAdd(P.tickets + it.group, 1u) == (unsigned)it.group_count - 1u;
          if (last) __threadfence();      // acquire: the other items' partials, released before their tickets, are visible
          *flag = last;
        }
        named_bar_sync(2, 128);
        const bool do_merge = *flag != 0;
        named_bar_sync(2, 128);     // everyone has read the flag before thread 0 may write the next item's
        if (do_merge) {  // the last item of the group merges the group's partials (thread = dim)
          __threadfence();
          // One pass over the group's partials, all query heads at once and JB partials per step (their loads are
          // independent: one L2 latency per step), merged online: the running maximum rescales what has been summed.
          float M[GP], L[GP], acc[GP];
#pragma unroll
          for (int g = 0; g < GP; ++g) { M[g] = -INFINITY; L[g] = 0.0f; acc[g] = 0.0f; }
          const int cnt = it.group_count;
          constexpr int JB = GP == 4 ? 8 : (GP == 8 ? 2 : 1);        // partials per step (registers: 3 * JB * GP values)
          for (int j0 = 0; j0 < cnt; j0 += JB) {
            float mv[JB][GP], lv[JB][GP], ov[JB][GP];
#pragma unroll
            for (int jj = 0; jj < JB; ++jj)
#pragma unroll
              for (int g = 0; g < GP; ++g) {
                // unconditional loads at clamped indices (a predicated load would serialise the step), masked afterwards
                const bool ok = j0 + jj < cnt && g < G;
                const int64_t pi = (int64_t)(it.group_first + min(j0 + jj, cnt - 1));
                const int gc = min(g, G - 1);
                const float2 ml = __ldcg(reinterpret_cast<const float2*>(P.part_ml + (pi * G + gc) * 2));
                const float ovv = __ldcg(P.part_o + (pi * G + gc) * kD + tid);
                mv[jj][g] = ok ? ml.x : -INFINITY;
                lv[jj][g] = ok ? ml.y : 0.0f;
                ov[jj][g] = ok ? ovv : 0.0f;
              }
#pragma unroll
            for (int g = 0; g < GP; ++g) {
              float nm = M[g];
#pragma unroll
              for (int jj = 0; jj < JB; ++jj) nm = fmaxf(nm, mv[jj][g]);
              const float a0 = (M[g] == -INFINITY) ? 0.0f : exp2f(M[g] - nm);
              float Ls = L[g] * a0, as = acc[g] * a0;
#pragma unroll
              for (int jj = 0; jj < JB; ++jj) {
                const float w = (mv[jj][g] == -INFINITY) ? 0.0f : exp2f(mv[jj][g] - nm);
                Ls += w * lv[jj][g];
                as += w * ov[jj][g];
              }
              M[g] = nm; L[g] = Ls; acc[g] = as;
            }
          }
#pragma unroll
          for (int g = 0; g < GP; ++g)
            if (g < G) {
              P.o[(out_row + g) * kD + tid] = acc[g] / L[g];
              if (tid == 0) P.lse[out_row + g] = (M[g] + log2f(L[g])) * 0.6931471805599453f;
            }
          if (tid == 0) P.tickets[it.group] = 0u;      // re-armed for the next launch
        }
      }
    }
  }
  // teardown: every tcgen05 operation of this CTA has completed once the epilogue warps have seen their last o_full
  tc_fence_before();
  __syncthreads();
  if (warp == 1) {
    tc_fence_after();
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem), "r"(64u) : "memory");
  }
}

// Merge of the partials of the LARGE groups (more partials than the in-kernel merge takes in one step), after the
// attention grid: one CTA per (group, query head); thread = (slice of the group's partials, dim).  Under a saturated
// HBM a dependent load costs several microseconds, so the in-kernel merge of a long group would be a serial tail of
// (partials / 8) such latencies; here the machine is idle, every thread has 32 loads in flight and 4 slices share a group.
template <int kMergeSlices>      // 4: long groups; 1: every group has <= 32 partials (a slice per group, 4x the CTAs per SM)
__global__ void __launch_bounds__(128 * kMergeSlices) kvr_attend_merge_kernel(const AttnMerge* __restrict__ merges, int G,
                                                                              const float* __restrict__ part_o,
                                                                              const float* __restrict__ part_ml,
                                                                              float* __restrict__ o, float* __restrict__ lse) {
  __shared__ float s_m[kMergeSlices], s_l[kMergeSlices], s_acc[kMergeSlices][kD];
  asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
  asm volatile("griddepcontrol.wait;" ::: "memory");      // every partial of the attention grid is complete and visible
  const AttnMerge mg = merges[blockIdx.x / G];
  const int g = blockIdx.x % G, dim = threadIdx.x & (kD - 1), sl = threadIdx.x >> 7;
  const int per = (mg.count + kMergeSlices - 1) / kMergeSlices, j_lo = sl * per, j_hi = min(mg.count, j_lo + per);
  float M = -INFINITY, L = 0.0f, acc = 0.0f;
  constexpr int JB = 16;
  for (int j0 = j_lo; j0 < j_hi; j0 += JB) {
    float2 ml[JB];
    float ov[JB];
#pragma unroll
    for (int jj = 0; jj < JB; ++jj) {
      const int64_t pi = (int64_t)mg.first + min(j0 + jj, j_hi - 1);
      ml[jj] = __ldcg(reinterpret_cast<const float2*>(part_ml + (pi * G + g) * 2));
      ov[jj] = __ldcg(part_o + (pi * G + g) * kD + dim);
    }
    float nm = M;
#pragma unroll
    for (int jj = 0; jj < JB; ++jj) if (j0 + jj < j_hi) nm = fmaxf(nm, ml[jj].x);
    const float a0 = (M == -INFINITY) ? 0.0f : exp2f(M - nm);
    L *= a0; acc *= a0;
#pragma unroll
    for (int jj = 0; jj < JB; ++jj)
      if (j0 + jj < j_hi) {
        const float w = exp2f(ml[jj].x - nm);
        L += w * ml[jj].y;
        acc += w * ov[jj];
      }
    M = nm;
  }
  if (dim == 0) { s_m[sl] = M; s_l[sl] = L; }
  s_acc[sl][dim] = acc;
  __syncthreads();
  if (sl == 0) {
    float Mx = -INFINITY;
#pragma unroll
    for (int k = 0; k < kMergeSlices; ++k) Mx = fmaxf(Mx, s_m[k]);
    float Ls = 0.0f, as = 0.0f;
#pragma unroll
    for (int k = 0; k < kMergeSlices; ++k) {
      const float w = (s_m[k] == -INFINITY) ? 0.0f : exp2f(s_m[k] - Mx);
      Ls += w * s_l[k];
      as += w * s_acc[k][dim];
    }
    o[((int64_t)mg.out_q0 + g) * kD + dim] = as / Ls;
    if (dim == 0) lse[mg.out_q0 + g] = (Mx + log2f(Ls)) * 0.6931471805599453f;
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
  cudaLaunchConfig_t lc{};
  lc.gridDim = dim3((unsigned)grid); lc.blockDim = dim3(kThreads); lc.dynamicSmemBytes = kSmemBytes; lc.stream = st;
  cudaLaunchAttribute at[1];
  at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  at[0].val.programmaticStreamSerializationAllowed = 1;
  lc.attrs = at; lc.numAttrs = 1;
  return cudaLaunchKernelEx(&lc, kvr_attend_kernel<GP>, P);
}

cudaError_t launch_attend(const AttnParams& P, int sm_count, cudaStream_t stream, int* grid_out, int* block_out, int* smem_out) {
  int grid = P.n_items < sm_count ? P.n_items : sm_count;
  if (grid < 1) grid = 1;
  *grid_out = grid; *block_out = kThreads; *smem_out = kSmemBytes;
  cudaError_t e = P.group <= 4 ? launch_attend_inst<4>(P, grid, stream)
                : P.group <= 8 ? launch_attend_inst<8>(P, grid, stream) : launch_attend_inst<16>(P, grid, stream);
  if (e != cudaSuccess || P.n_merges == 0) return e;
  cudaLaunchConfig_t lc{};
  const int slices = P.merge_max_count <= 32 ? 1 : 4;
  lc.gridDim = dim3((unsigned)(P.n_merges * P.group)); lc.blockDim = dim3(128 * slices); lc.dynamicSmemBytes = 0; lc.stream = stream;
  cudaLaunchAttribute at[1];
  at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  at[0].val.programmaticStreamSerializationAllowed = 1;
  lc.attrs = at; lc.numAttrs = 1;
  return slices == 1
      ? cudaLaunchKernelEx(&lc, kvr_attend_merge_kernel<1>, P.merges, (int)P.group, (const float*)P.part_o, (const float*)P.part_ml, P.o, P.lse)
      : cudaLaunchKernelEx(&lc, kvr_attend_merge_kernel<4>, P.merges, (int)P.group, (const float*)P.part_o, (const float*)P.part_ml, P.o, P.lse);
}

// partials the in-kernel merge takes in one step (the loads of a step are in flight together)
int attend_inline_merge_limit(int group) { return group <= 4 ? 8 : (group <= 8 ? 2 : 1); }

}  // namespace kvr
