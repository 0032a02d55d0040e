// kvr_ring.cu -- the FAST reposition+splice kernel for sm_100a: a persistent, warp-specialised
// TMA ring.  HBM-bound by construction (no contraction => no tensor cores).
//
//   producer warp   draws units (segment, chunk of <= cg destination tokens, layer group) -- the first grab is
//                   static, the rest come from one global counter -- and decodes 32 of them at a time, lane j
//                   resolving unit j's segment, chunk geometry and block-table entry (step a4) one grab ahead.
//                   For every tile of a unit a lane arms the stage's "full" mbarrier with the byte count and
//                   issues 1-D bulk TMA loads  global -> shared  (cp.async.bulk, steps a2 / a6-read) of the K
//                   and V runs, together with a 32-byte tile descriptor; up to min(32, S) tiles per pass.
//                   All 32 lanes evaluate the angle table  (fp64 sincos of Delta*inv_freq -> fp32 hi/lo,
//                   step a1)  into a double-buffered shared table when the segment changes; with per-token
//                   shifts (position map, pre-RoPE keys) per unit, deduplicated into runs of equal Delta.
//   consumer warps  each owns every (NW/wpg)-th stage: wait on its "full" mbarrier, then
//                   V: one bulk TMA store  shared -> global  per destination run (head-major pools) or per row
//                      (gather mode), or 16-byte warp copies (token-major pools)                  (step a6)
//                   K: 16-byte shared loads, compensated fp32 rotation in registers with the segment's
//                      cos/sin held in registers, 16-byte global stores to the paged slot   (steps a3, a5)
//                   then release the stage through its "empty" mbarrier.
//   modes           in place (K rows read from the slot they are written back to), window (rows that are not a
//                   power of two / rotary window at an offset: the MLA [latent | k_pe] row), gather (dense
//                   token-major pools: all heads of a chunk per stage, several warps per stage), K-only.
//
// Persistent grid = SMs x CTAs/SM; programmatic dependent launch overlaps a launch's prologue (and its first
// angle table) with the tail of the previous one.
#include <cstdio>
#include <mutex>

#include "kvr_common.cuh"
#include "kvr_ptx.cuh"
#include "kvr_rotate.cuh"

namespace kvr {

struct RingParams {
  int S, NW, hpt, cg;
  int rowB, nv, log_nv, sp, log_sp, rpi;  // row bytes; 16-B vectors per row; slots (vector pairs) per row; rows per warp pass
  int nr;                                 // rotary vectors per row = rotary_dim * E / 16
  int half_R;                             // rotary pairs per row
  int NV;                                 // table transposition width (see tab_pos)
  int tile_bytes;                         // K (or V) region of a stage = hpt * cg * rowB
  int stage_bytes;                        // 2 * tile_bytes
  int off_meta, off_scales, off_tab, tab_stride, NTB, off_stage;
  int v_bulk;                             // V leaves shared memory by bulk stores (needs stride_token == head_dim)
  int n_scales;                           // fp8: layers * heads destination scales preloaded to shared memory
  int off_ub, n_ub;                       // segments' first-unit prefix sums in shared memory (calls with many segments)
  int no_v;                               // in-place / K-only calls: a stage holds K only and V is never touched
  int win;                                // WINDOW mode (rows that are not a power of two, or rotary_offset != 0, e.g. the
                                          // MLA [latent | k_pe] row): lanes are laid over the rotary window only and the
                                          // rest of the row is moved by a plain 16-byte copy loop
  int nv_slot;                            // vectors the lane slots are laid over: nv, or nr in window mode
  int ro_v;                               // rotary_offset in 16-byte vectors
  int log_rpi;                            // log2(rows per warp pass)
  int gather;                             // GATHER mode (see wpg)
  int split;                              // gather tiles hold K or V alone (all heads of a FULL chunk of one tensor)
  int wpg;                                // GATHER mode (dense token-major pools): a tile holds ALL heads of a few tokens and
                                          // wpg consumer warps share it, each taking whole token rows, tokens outer / heads
                                          // inner, so that a token's H*D row reaches L2 (and DRAM) as one contiguous burst
                                          // instead of H pieces written by H different warps at different times; 1 otherwise
  int hmaj;                               // gather tiles, "lanes over heads": a warp pass covers rpi HEADS of one token (their
                                          // rows are adjacent in a dense token-major pool) instead of rpi tokens of one head,
                                          // so every warp store instruction writes one contiguous run, as on a head-major pool
  int log_pt;                             // hmaj: log2(hpt * nv), the 16-byte vectors of one token in a tile
  int log_hp;                             // hmaj: a pass covers 2^log_hp heads (min(hpt, rpi)) x (rpi >> log_hp) tokens
  int ct;                                 // tmajor: tokens per tile
  int ip_mode;                            // in-place source runs: 0 one run per head (d_st == head_dim), 1 one run for the
                                          // whole tile (token-major pool, all heads in the tile), 2 one copy per row
};

struct __align__(16) TileMeta {
  int64_t dst_off;    // element offset of (layer, block, offset-in-block, first head of the tile)
  int32_t n_tok;
  int32_t flags;      // bit0 DONE, bit1 ROTATE (segment mode: Delta != 0)
  int32_t tab;        // table buffer index
  int32_t gen;        // table generation (changes when the consumer must reload its registers)
  int32_t scale_idx;  // layer * heads + first head
  int32_t seg;        // segment (only read when source scales differ)
};
static_assert(sizeof(TileMeta) == 32, "TileMeta layout");

constexpr int kFlagDone = 1, kFlagRotate = 2, kFlagTokMajor = 4;   // TokMajor: the stage is laid out [token][head][dim]
constexpr int kFlagKOnly = 8, kFlagVOnly = 16;                       // split gather tiles: the stage holds K or V alone
constexpr int kFlagSkip = 32;                                        // early-loaded tile whose block-table entry turned out invalid: release only
constexpr int kMaxThreads = 32 * 17;
constexpr int kMaxDevices = 64;

// Position of rotary pair p inside a table row.  Transposed so that the lanes of one row read
// consecutive 16-byte entries for the same k (bank-conflict free): p = group * PPV + k -> k * NV + group.
template <int PPV>
__device__ __forceinline__ int tab_pos(int p, int NV) { return (p % PPV) * NV + p / PPV; }

// ------------------------------------------------------------------------------- the kernel
// MAXT = 256: the default launch shape (<= 8 warps, 2 CTAs per SM) gets 128 registers per thread and no spills;
// MAXT = kMaxThreads: the wide shapes the tuning knobs allow (up to 16 consumer warps, or 3+ CTAs per SM).
template <int DTYPE, int PAIRING, bool MAP, int MAXT>
__global__ void __launch_bounds__(MAXT, (MAXT <= 256 ? 2 : 1))   // 256 x 2, 448 x 1: 128 registers; 544 x 1: 96
kvr_ring_kernel(const __grid_constant__ CallParams P, const __grid_constant__ RingParams RP,
                const __grid_constant__ TmapInline TI) {
  using G = Geo<DTYPE, PAIRING>;
  constexpr int E = (DTYPE == 0) ? 2 : 1;
  extern __shared__ __align__(128) unsigned char smem[];
  const uint32_t s_base = smem_u32(smem);
  const uint32_t s_full = s_base, s_empty = s_base + 8u * RP.S;
  TileMeta* meta = reinterpret_cast<TileMeta*>(smem + RP.off_meta);
  float* s_scales = reinterpret_cast<float*>(smem + RP.off_scales);
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int S = RP.S, NW = RP.NW;

  if (threadIdx.x == 0) {
    for (int s = 0; s < S; ++s) { mbar_init(s_full + 8u * s, 1); mbar_init(s_empty + 8u * s, (uint32_t)RP.wpg); }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();     // the barriers are initialised before the producer warp may use them (early source loads below)
  // Programmatic dependent launch: let the next launch on this stream bring its CTAs up (they take an SM's shared
  // memory as soon as a CTA of this grid exits) and run this prologue while our tail drains; it touches no global
  // memory that earlier work on the stream may write until griddepcontrol.wait has seen the previous grid complete.
  asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
  // Before the dependency wait the producer may only touch kernel parameters and the context's own immutable
  // inv_freq copy: with the descriptors inline it already knows the segment of its first (statically assigned)
  // unit and builds that segment's angle table (fp64 sincos), taking it off the critical path of the launch.
  int pre_si = -1;
  if (!MAP && warp == NW && P.n_segs <= kInlineSegs && (int64_t)blockIdx.x * P.grab < P.total_units) {
    pre_si = find_segment(P.inline_segs, P.n_segs, (int64_t)blockIdx.x * P.grab);
    float4* tab = reinterpret_cast<float4*>(smem + RP.off_tab + RP.tab_stride);       // table buffer 1
    const int64_t delta = P.inline_segs[pre_si].delta;
    for (int p = lane; p < RP.half_R; p += 32) tab[tab_pos<G::PPV>(p, RP.NV)] = angle_entry(delta, P.inv_freq[p]);
    __syncwarp();
  }
  // EARLY SOURCE LOADS (KVR_SEG_SRC_STABLE, kvr.h): a precompiled skill is not written by anything that precedes the call
  // on the stream, so the loads of the CTA's first (statically assigned) unit are issued NOW, while the previous grid
  // is still draining, into stages 0.. with their byte counts posted by expect_tx WITHOUT an arrival.  The stages'
  // destinations need the block table, which is read after the wait: the producer then writes the tile descriptors and
  // arrives, and only then can a stage's "full" phase complete.  Inline descriptors only (they are kernel parameters).
  int early_n = 0;
  if (warp == NW && P.n_segs <= kInlineSegs && !P.inplace && !RP.split && (int64_t)blockIdx.x * P.grab < P.total_units) {
    const int64_t u0 = (int64_t)blockIdx.x * P.grab;
    const int si0 = find_segment(P.inline_segs, P.n_segs, u0);
    const SegDev& s0 = P.inline_segs[si0];
    if (s0.src_stable && (P.tmajor || s0.st == P.head_dim)) {
      const int64_t local = u0 - s0.unit_begin;
      const int lg = (int)(local / s0.n_chunks), c = (int)(local - (int64_t)lg * s0.n_chunks);
      const Chunk ch = chunk_of(s0, c, RP.cg, P.block_size);
      const int lgi = lg / P.hsplit, hpart = lg - lgi * P.hsplit;
      const int l0 = lgi * P.lpu, l1 = min(P.layers, l0 + P.lpu);
      const int hg_per = (P.heads / RP.hpt) / P.hsplit;
      const int n_sub = P.tmajor ? (ch.n_tok + RP.ct - 1) / RP.ct : 1;
      const int n_tiles = P.tmajor ? (l1 - l0) * n_sub : (l1 - l0) * hg_per;
      early_n = min(S < 32 ? S : 32, n_tiles);
      if (lane < early_n) {
        const uint64_t pol = policy_evict_first();
        const uint32_t bar = s_full + 8u * lane;
        const uint32_t sk = s_base + RP.off_stage + (uint32_t)lane * RP.stage_bytes;
        if (P.tmajor) {
          const int l = l0 + lane / n_sub, tok0 = (lane % n_sub) * RP.ct;
          mbar_expect_tx(bar, (RP.no_v ? 1u : 2u) * (uint32_t)RP.tile_bytes);
          tensor_g2s_4d(sk, &TI.m[si0].k, 0, 0, ch.t0 + tok0, l, bar, pol);
          if (!RP.no_v) tensor_g2s_4d(sk + RP.tile_bytes, &TI.m[si0].v, 0, 0, ch.t0 + tok0, l, bar, pol);
        } else {
          const int l = l0 + lane / hg_per, h0 = (hpart * hg_per + lane % hg_per) * RP.hpt;
          const uint32_t run_bytes = (uint32_t)(ch.n_tok * RP.rowB);
          mbar_expect_tx(bar, (RP.no_v ? 1u : 2u) * RP.hpt * run_bytes);
          for (int hh = 0; hh < RP.hpt; ++hh) {
            const int64_t src_off = ((int64_t)l * s0.sl + (int64_t)(h0 + hh) * s0.sh + (int64_t)ch.t0 * s0.st) * E;
            const uint32_t so = (uint32_t)(hh * RP.cg * RP.rowB);
            bulk_g2s(sk + so, s0.k_src + src_off, run_bytes, bar, pol);
            if (!RP.no_v) bulk_g2s(sk + RP.tile_bytes + so, s0.v_src + src_off, run_bytes, bar, pol);
          }
        }
      }
      __syncwarp();
    }
  }
  asm volatile("griddepcontrol.wait;" ::: "memory");
  if (DTYPE == 1)
    for (int i = threadIdx.x; i < RP.n_scales; i += blockDim.x) s_scales[i] = P.k_scale_dst[i];
  for (int i = threadIdx.x; i < RP.n_ub; i += blockDim.x)
    reinterpret_cast<int64_t*>(smem + RP.off_ub)[i] = P.segs[i].unit_begin;
  __syncthreads();

  if (warp == NW) {
    // =========================================================================== PRODUCER
    const uint64_t pol = policy_evict_first();
    uint32_t i = 0;                // tiles issued by this CTA; (stage, phase) of the next one
    int stage = 0;
    uint32_t phase = 0;
    int tb = 0, gen = 0;           // current table buffer / generation
    int64_t cur_key = -1;          // segment (segment mode) or unit (map mode) the current table belongs to
    if (pre_si >= 0) { tb = 1; gen = 1; cur_key = pre_si; }   // built before the dependency wait
    uint32_t lu_i[2] = {0, 0};     // last tile that used each table buffer
    bool lu_valid[2] = {false, false};
    int cur_si = -1;
    SegDev sg{};                   // current segment, held in registers
    const int hgroups = P.heads / RP.hpt;
    const unsigned FULL = 0xFFFFFFFFu;

    const SegDev* segs = seg_array(P);
    const int G = P.grab;          // units per grab, 1..32
    // ---- dynamic scheduling: CTAs draw units from one global counter, so a CTA on a slower path to memory
    //      simply takes fewer units (a static round-robin deal loses ~10 % of the copy bandwidth to drift and tail).
    //      The next grab is requested before the current one is issued, so its latency is off the critical path. ----
    // ---- batch decode: lane j resolves unit base + j (segment, chunk, block-table entry: step a4).  The decode of
    //      grab k+1 is started BEFORE the tiles of grab k are issued, so its dependent global loads (descriptor,
    //      block table) complete while the producer is busy arming stages: small units cost no producer stalls. ----
    const int64_t* ub = reinterpret_cast<const int64_t*>(smem + RP.off_ub);
    auto decode = [&](int64_t base_, int& d_si, int& d_t0, int& d_ntok, int& d_off, int& d_lg, int& d_blk) {
      const int64_t my_unit = base_ + lane;
      d_si = -1; d_t0 = 0; d_ntok = 0; d_off = 0; d_lg = 0; d_blk = -1;
      if (lane < G && my_unit < P.total_units) {
        if (RP.n_ub) {               // prefix sums of the segments' unit counts, staged in shared memory
          int lo = 0, hi = P.n_segs - 1;
          while (lo < hi) { const int mid = (lo + hi + 1) >> 1; if (ub[mid] <= my_unit) lo = mid; else hi = mid - 1; }
          d_si = lo;
        } else {
          d_si = find_segment(segs, P.n_segs, my_unit);
        }
        const SegDev* s = segs + d_si;
        const int64_t local = my_unit - s->unit_begin;
        const int n_chunks = s->n_chunks;
        d_lg = (int)(local / n_chunks);
        const int c = (int)(local - (int64_t)d_lg * n_chunks);
        const Chunk ch = chunk_of(*s, c, RP.cg, P.block_size);
        d_t0 = ch.t0; d_ntok = ch.n_tok; d_off = ch.off;
        d_blk = P.block_table[(int64_t)s->dst_seq * P.max_blocks + ch.blk_index];
      }
    };
    // The first grab is static (CTA b takes units [b G, (b+1) G)): no round trip to the counter before the first
    // load is in flight.  The counter hands out the units from gridDim.x * G on.
    unsigned long long nxt = 0;
    const int64_t dyn0 = (int64_t)gridDim.x * G;
    int64_t base = (int64_t)blockIdx.x * G;
    if (lane == 0) nxt = atomicAdd(P.sched, (unsigned long long)G);
    int d_si, d_t0, d_ntok, d_off, d_lg, d_blk;
    decode(base, d_si, d_t0, d_ntok, d_off, d_lg, d_blk);
    for (;;) {
      if (base >= P.total_units) break;
      const int64_t base_n = dyn0 + (int64_t)__shfl_sync(FULL, nxt, 0);
      if (lane == 0 && base_n < P.total_units) nxt = atomicAdd(P.sched, (unsigned long long)G);
      int n_si, n_t0, n_ntok, n_off, n_lg, n_blk;
      decode(base_n, n_si, n_t0, n_ntok, n_off, n_lg, n_blk);
      for (int j = 0; j < G; ++j) {
        const int si = __shfl_sync(FULL, d_si, j);
        if (si < 0) break;
        const int t0 = __shfl_sync(FULL, d_t0, j), n_tok = __shfl_sync(FULL, d_ntok, j);
        const int off = __shfl_sync(FULL, d_off, j), lg = __shfl_sync(FULL, d_lg, j);
        const int blk = __shfl_sync(FULL, d_blk, j);
        if (si != cur_si) {
          sg = segs[si]; cur_si = si;
          if (P.tmajor && lane < 2) {      // bring the segment's two tensor maps into the TMA unit's descriptor cache
            const TmapPair* tp = (P.n_segs <= kInlineSegs) ? &TI.m[si] : &P.tmaps[si];
            if (lane == 0 || !RP.no_v)
              asm volatile("prefetch.tensormap [%0];" ::"l"(lane == 0 ? &tp->k : &tp->v) : "memory");
          }
        }
        if (blk < 0 || blk >= P.num_blocks) {
          if (lane == 0) report_bad_block(P.status, sg.index, t0);
          if (early_n > 0 && i == 0u && base == (int64_t)blockIdx.x * G && j == 0) {
            // the unit's first tiles were loaded before the dependency wait: hand their stages to the consumers as
            // SKIP tiles (released without touching the destination) so that the ring keeps turning
            if (lane < early_n) {
              TileMeta m{};
              m.flags = kFlagSkip;
              meta[lane] = m;
              mbar_arrive(s_full + 8u * lane);
            }
            __syncwarp();
            i += (uint32_t)early_n; stage += early_n;
            if (stage >= S) { stage -= S; phase ^= 1u; }
            early_n = 0;
          }
          continue;
        }
        // ---- angle table (step a1) ----
        // per-token shifts (position map, pre-RoPE keys): a table per unit; a constant shift: a table per segment,
        // also inside a call that has per-token segments elsewhere (its per-token words then all name row 0)
        const bool per_token = MAP && (sg.pos_map != nullptr || sg.pre_rope != 0);
        const int64_t key = per_token ? ((base + j) | (1ll << 62)) : (int64_t)si;
        if (key != cur_key) {
          const int nb = tb ^ 1;
          // Buffer nb was last read by the tiles up to lu_i[nb].  Consumer warps take their stages in order, so once
          // the newest tile of EACH warp (group) among those is released, every older one is: wait for the last
          // NW / wpg tiles up to lu_i (tile j sits in stage j % S, use j / S); tiles <= i-1-S are known released.
          if (nb ? lu_valid[1] : lu_valid[0]) {
            const uint32_t last = nb ? lu_i[1] : lu_i[0];
            if ((uint32_t)lane < (uint32_t)(NW / RP.wpg) && (uint32_t)lane <= last) {
              const uint32_t j = last - (uint32_t)lane;
              if (j + (uint32_t)S >= i) mbar_wait(s_empty + 8u * (j % (uint32_t)S), (j / (uint32_t)S) & 1u, 1);
            }
          }
          __syncwarp();
          float4* tab = reinterpret_cast<float4*>(smem + RP.off_tab + nb * RP.tab_stride);
          if (MAP && !per_token) {
            for (int p = lane; p < RP.half_R; p += 32)
              tab[tab_pos<G::PPV>(p, RP.NV)] = angle_entry((int64_t)sg.delta, P.inv_freq[p]);
            if (lane < RP.cg) reinterpret_cast<int32_t*>(tab + RP.cg * RP.half_R)[lane] = (sg.delta == 0) ? -1 : 0;
          } else if (MAP && sg.pre_rope && sg.pos_map == nullptr) {
            // Pre-RoPE keys at consecutive target positions: Delta_t = Delta_0 + t.  One fp64 sincos per pair for the
            // first token and one for the step angle inv_freq[p]; the other tokens follow by the fp64 angle-addition
            // recurrence (c, s) <- (c c1 - s s1, s c1 + c s1): <= 15 steps, error ~2e-15 against sincos of the product,
            // i.e. at the resolution of the fp32 hi+lo pair the table stores.  ~4x cheaper than a
            // sincos per (token, pair), which is what bounds a chunk whose every token has its own shift.
            const long long d0 = token_delta(sg, t0);
            for (int p = lane; p < RP.half_R; p += 32) {
              const double f = P.inv_freq[p];
              double s1, c1, sn, cs;
              sincos(f, &s1, &c1);
              sincos((double)d0 * f, &sn, &cs);
              const int pos = tab_pos<G::PPV>(p, RP.NV);
              for (int r = 0; r < n_tok; ++r) {
                tab[r * RP.half_R + pos] = angle_entry_cs(cs, sn);
                const double c2 = cs * c1 - sn * s1, s2 = sn * c1 + cs * s1;
                cs = c2; sn = s2;
              }
            }
            if (lane < n_tok) reinterpret_cast<int32_t*>(tab + RP.cg * RP.half_R)[lane] = (d0 + lane == 0) ? -1 : lane;
          } else if (MAP) {
            // Per-token shifts, deduplicated into RUNS of equal Delta (a position map is contiguous except at its
            // gaps, so a chunk of <= 32 tokens holds a handful of distinct shifts): one table row per run, and a
            // per-token word that names the token's row (-1: Delta_t == 0, the row is a byte copy).
            long long d = 0;
            if (lane < n_tok) d = token_delta(sg, t0 + lane);
            const long long dprev = __shfl_up_sync(FULL, d, 1);
            const unsigned heads_mask = __ballot_sync(FULL, lane < n_tok && (lane == 0 || d != dprev));
            const int n_runs = __popc(heads_mask);
            if (lane < n_tok)
              reinterpret_cast<int32_t*>(tab + RP.cg * RP.half_R)[lane] =
                  (d == 0) ? -1 : (__popc(heads_mask & (0xFFFFFFFFu >> (31 - lane))) - 1);
            const int total = n_runs * RP.half_R;
            for (int base_idx = 0; base_idx < total; base_idx += 32) {
              const int idx = base_idx + lane;
              const int r = idx < total ? idx / RP.half_R : 0, p = idx - r * RP.half_R;
              const int src_lane = (int)__fns(heads_mask, 0, r + 1);            // first token of run r
              const long long delta = __shfl_sync(FULL, d, src_lane);
              if (idx < total) tab[r * RP.half_R + tab_pos<G::PPV>(p, RP.NV)] = angle_entry((int64_t)delta, P.inv_freq[p]);
            }
          } else {
            for (int p = lane; p < RP.half_R; p += 32)
              tab[tab_pos<G::PPV>(p, RP.NV)] = angle_entry((int64_t)sg.delta, P.inv_freq[p]);
          }
          __syncwarp();
          tb = nb; gen += 1; cur_key = key;
        }
        {
          // ---- tile issue (steps a2 / a6-read): lane t takes tile t of the unit, so up to min(32, S) tiles are
          //      armed and issued per pass instead of one (a single thread needs ~1k cycles per tile) ----
          const int lgi = lg / P.hsplit, hpart = lg - lgi * P.hsplit;     // layer group, head part of this unit
          const int l0 = lgi * P.lpu, l1 = min(P.layers, l0 + P.lpu);
          const int hg_per = hgroups / P.hsplit;
          const int kinds = RP.split ? 2 : 1;                            // split: a K tile, then a V tile
          const bool tmajor = P.tmajor != 0;                             // tiles = (layer, sub-chunk of ct tokens), all heads
          const int n_sub = tmajor ? (n_tok + RP.ct - 1) / RP.ct : 1;
          const int n_tiles = tmajor ? (l1 - l0) * n_sub : (l1 - l0) * hg_per * kinds;
          const bool inplace = P.inplace != 0;
          const int flags = ((MAP || sg.delta != 0) ? kFlagRotate : 0) |
                            (((inplace && RP.ip_mode == 1) || tmajor) ? kFlagTokMajor : 0);
          const uint32_t run_bytes = (uint32_t)(n_tok * RP.rowB);
          const bool packed_rows = (sg.st == P.head_dim);
          const int64_t dst_chunk = (int64_t)blk * P.d_sb + (int64_t)off * P.d_st;
          const int64_t src_chunk = (int64_t)t0 * sg.st;
          const int pass = S < 32 ? S : 32;
          // the first pass of the CTA's first unit: its loads were issued before the dependency wait (early_n tiles)
          const bool early_unit = early_n > 0 && i == 0u && base == (int64_t)blockIdx.x * G && j == 0;
          for (int tb0 = 0; tb0 < n_tiles; tb0 += pass) {
            const int n = min(pass, n_tiles - tb0);
            const bool early = early_unit && tb0 == 0;      // then n == early_n: descriptor + arrival only
            if (lane < n && tmajor) {
              // transposing tensor loads: the box {head_dim, heads, ct tokens, 1 layer} of the source lands as
              // [token][head][dim], the order of a dense token-major pool; one TMA operation per tensor and tile
              const int t = tb0 + lane;
              const int l = l0 + t / n_sub, tok0 = (t % n_sub) * RP.ct;
              int my_stage = stage + lane;
              uint32_t my_phase = phase;
              if (my_stage >= S) { my_stage -= S; my_phase ^= 1u; }
              const uint32_t bar = s_full + 8u * my_stage;
              mbar_wait(s_empty + 8u * my_stage, my_phase ^ 1u, 2);
              TileMeta m;
              m.dst_off = (int64_t)l * P.d_sl + dst_chunk + (int64_t)tok0 * P.d_st;
              m.n_tok = min(RP.ct, n_tok - tok0); m.tab = tb; m.gen = gen;
              m.flags = flags | (tok0 << 8);                                   // bits 8+: first token of the tile in its chunk
              m.scale_idx = l * P.heads; m.seg = si;
              meta[my_stage] = m;
              if (early) {
                mbar_arrive(bar);
              } else {
              mbar_arrive_expect_tx(bar, (RP.no_v ? 1u : 2u) * (uint32_t)RP.tile_bytes);   // the whole box, zero-filled past the end
              const uint32_t sk = s_base + RP.off_stage + (uint32_t)my_stage * RP.stage_bytes;
              const TmapPair* tp = (P.n_segs <= kInlineSegs) ? &TI.m[si] : &P.tmaps[si];
              tensor_g2s_4d(sk, &tp->k, 0, 0, t0 + tok0, l, bar, pol);
              if (!RP.no_v) tensor_g2s_4d(sk + RP.tile_bytes, &tp->v, 0, 0, t0 + tok0, l, bar, pol);
              }
            } else if (lane < n) {
              const int t = (tb0 + lane) / kinds;
              const int kind = RP.split ? (tb0 + lane) - t * kinds : -1;      // 0: K tile, 1: V tile, -1: both
              const int l = l0 + t / hg_per, h0 = (hpart * hg_per + t % hg_per) * RP.hpt;
              int my_stage = stage + lane;
              uint32_t my_phase = phase;
              if (my_stage >= S) { my_stage -= S; my_phase ^= 1u; }
              const uint32_t bar = s_full + 8u * my_stage;
              mbar_wait(s_empty + 8u * my_stage, my_phase ^ 1u, 2);
              TileMeta m;
              m.dst_off = (int64_t)l * P.d_sl + dst_chunk + (int64_t)h0 * P.d_sh;
              m.n_tok = n_tok; m.tab = tb; m.gen = gen;
              m.flags = flags | (kind == 0 ? kFlagKOnly : 0) | (kind == 1 ? kFlagVOnly : 0);
              m.scale_idx = l * P.heads + h0; m.seg = si;
              meta[my_stage] = m;
              if (early) {
                mbar_arrive(bar);
              } else {
              mbar_arrive_expect_tx(bar, ((RP.no_v || RP.split) ? 1u : 2u) * RP.hpt * run_bytes);
              const uint32_t sk = s_base + RP.off_stage + (uint32_t)my_stage * RP.stage_bytes;
              const uint32_t sv = RP.split ? sk : sk + RP.tile_bytes;
              const bool ld_k = kind != 1, ld_v = kind != 0 && !RP.no_v;
              if (inplace) {
                // the tile's source IS its destination: K rows already resident in the paged pool (R20)
                const uint8_t* src = P.k_cache + m.dst_off * E;
                if (RP.ip_mode == 1) {
                  bulk_g2s(sk, src, RP.hpt * run_bytes, bar, pol);                    // [token][head][dim], one run
                } else if (RP.ip_mode == 0) {
                  for (int hh = 0; hh < RP.hpt; ++hh)                                  // [head][token][dim], a run per head
                    bulk_g2s(sk + (uint32_t)(hh * RP.cg * RP.rowB), src + (int64_t)hh * P.d_sh * E, run_bytes, bar, pol);
                } else {
                  for (int hh = 0; hh < RP.hpt; ++hh)
                    for (int r = 0; r < n_tok; ++r)
                      bulk_g2s(sk + (uint32_t)((hh * RP.cg + r) * RP.rowB),
                               src + ((int64_t)hh * P.d_sh + (int64_t)r * P.d_st) * E, RP.rowB, bar, pol);
                }
              } else
              for (int hh = 0; hh < RP.hpt; ++hh) {
                const int64_t src_off = ((int64_t)l * sg.sl + (int64_t)(h0 + hh) * sg.sh + src_chunk) * E;
                const uint32_t so = (uint32_t)(hh * RP.cg * RP.rowB);
                if (packed_rows) {
                  if (ld_k) bulk_g2s(sk + so, sg.k_src + src_off, run_bytes, bar, pol);
                  if (ld_v) bulk_g2s(sv + so, sg.v_src + src_off, run_bytes, bar, pol);
                } else {
                  for (int r = 0; r < n_tok; ++r) {
                    if (ld_k) bulk_g2s(sk + so + r * RP.rowB, sg.k_src + src_off + (int64_t)r * sg.st * E, RP.rowB, bar, pol);
                    if (ld_v) bulk_g2s(sv + so + r * RP.rowB, sg.v_src + src_off + (int64_t)r * sg.st * E, RP.rowB, bar, pol);
                  }
                }
              }
              }
            }
            __syncwarp();
            if (early) early_n = 0;
            i += (uint32_t)n;
            stage += n;
            if (stage >= S) { stage -= S; phase ^= 1u; }
          }
          // the unit's last tile is the last reader of table buffer tb
          if (n_tiles > 0) {
            if (tb) { lu_i[1] = i - 1u; lu_valid[1] = true; }
            else { lu_i[0] = i - 1u; lu_valid[0] = true; }
          }
        }
      }
      base = base_n;
      d_si = n_si; d_t0 = n_t0; d_ntok = n_ntok; d_off = n_off; d_lg = n_lg; d_blk = n_blk;
    }
    // one DONE tile per consumer warp (per group of wpg warps), through the same ring (NW / wpg <= S: distinct stages)
    if (lane < NW / RP.wpg) {
      int my_stage = stage + lane;
      uint32_t my_phase = phase;
      if (my_stage >= S) { my_stage -= S; my_phase ^= 1u; }
      mbar_wait(s_empty + 8u * my_stage, my_phase ^ 1u, 3);
      TileMeta m{};
      m.flags = kFlagDone;
      meta[my_stage] = m;
      mbar_arrive(s_full + 8u * my_stage);
    }
    // every CTA's last grab has returned >= total_units once all of them are here: the last one re-arms the scheduler
    if (lane == 0) {
      __threadfence();
      if (atomicAdd(P.sched + 1, 1ull) == (unsigned long long)gridDim.x - 1ull) {
        P.sched[0] = 0ull; P.sched[1] = 0ull;
        __threadfence();
      }
    }
    return;
  }

  // ============================================================================= CONSUMERS
  const int sp = RP.sp, q = lane & (sp - 1), rsub = lane >> RP.log_sp, rpi = RP.rpi;
  const int nv = RP.nv, nr = RP.nr, nvs = RP.nv_slot;
  // this lane's slot: two 16-byte vectors (va, vb) of every row it visits (of its rotary window in window mode)
  int va, vb;
  bool rot_a, rot_b;
  if (PAIRING == 0) {
    const int half = nr >> 1;
    if (q < half) { va = q; vb = q + half; rot_a = rot_b = true; }
    else { va = nr + 2 * (q - half); vb = va + 1; rot_a = rot_b = false; }
  } else {
    va = q; vb = q + (nvs >> 1);
    rot_a = va < nr; rot_b = vb < nr;
  }
  // Table position of this lane's k-th pair (tab_pos of pair va * EPV + k for NeoX, of pair v * PPV + k % PPV for
  // GPT-J): affine in k, so it is recomputed where the table is read instead of being held in NT registers.
  const int tp_a = rot_a ? va : 0, tp_b = rot_b ? vb : 0, tp_nv = RP.NV;
  auto tpos = [&](int k) -> int {
    if (PAIRING == 0) return rot_a ? tp_a + k * tp_nv : 0;
    return (k < G::PPV) ? (rot_a ? tp_a + k * tp_nv : 0) : (rot_b ? tp_b + (k - G::PPV) * tp_nv : 0);
  };
  va += RP.ro_v; vb += RP.ro_v;       // table positions above are relative to the window; addresses are not
  float4 T4[DTYPE == 0 ? G::NT : 1];
  float2 T2[DTYPE == 1 ? G::NT : 1];
  int my_gen = -1, my_run = -1;

  const int wpg = RP.wpg, wsub = warp % wpg, stage_step = NW / wpg;
  int stage = (warp / wpg) % S;
  uint32_t phase = (uint32_t)((warp / wpg) / S) & 1u;

  // one K row-slot of this lane: load, rotate (or requantise), store
  // srow / grow: shared-memory address and destination pointer of the row (callers step them; no 64-bit multiply per row);
  // t: the row's token within its chunk (names its table row when shifts are per token)
  const int va16 = va * 16, vb16 = vb * 16;
  const int64_t tokB = P.d_st * E;                // bytes between the rows of consecutive tokens in the pool
  auto k_row = [&](const TileMeta& m, uint32_t tab, bool rotate, uint32_t srow, uint8_t* grow, int t,
                   float s_src, float inv_dst, bool requant) {
    uint4 A = lds128(srow + va16);
    uint4 B = lds128(srow + vb16);
    bool rot_row = rotate;
    if (MAP) {
      const int run = reinterpret_cast<const int32_t*>(smem + RP.off_tab + m.tab * RP.tab_stride + RP.cg * RP.half_R * 16)[t + (m.flags >> 8)];
      rot_row = run >= 0;
      if (rot_row && (rot_a || rot_b) && (run != my_run || m.gen != my_gen)) {   // cos/sin registers follow the run
        my_run = run; my_gen = m.gen;
        const uint32_t trow = tab + run * RP.half_R * 16;
#pragma unroll
        for (int k = 0; k < G::NT; ++k) {
          float4 e = lds128f(trow + tpos(k) * 16);
          if (DTYPE == 0) T4[k] = e; else T2[k] = make_float2(e.x, e.z);
        }
      }
    }
    if constexpr (DTYPE == 0) {
      if (rot_row) {
        if constexpr (PAIRING == 0) { if (rot_a) rot_bf16_neox(A, B, T4); }
        else { if (rot_a) rot_bf16_gptj(A, T4); if (rot_b) rot_bf16_gptj(B, T4 + G::PPV); }
      }
    } else if (rot_row || requant) {
      if (requant) {
        if constexpr (PAIRING == 0) {
          if (rot_a) rot_fp8_neox<true>(A, B, T2, s_src, inv_dst, rot_row);
          else { requant_fp8(A, s_src, inv_dst); requant_fp8(B, s_src, inv_dst); }
        } else {
          if (rot_a) rot_fp8_gptj<true>(A, T2, s_src, inv_dst, rot_row); else requant_fp8(A, s_src, inv_dst);
          if (rot_b) rot_fp8_gptj<true>(B, T2 + G::PPV, s_src, inv_dst, rot_row); else requant_fp8(B, s_src, inv_dst);
        }
      } else {                       // equal scales (then rot_row holds): they cancel
        if constexpr (PAIRING == 0) {
          if (rot_a) rot_fp8_neox<false>(A, B, T2, 1.0f, 1.0f, true);
        } else {
          if (rot_a) rot_fp8_gptj<false>(A, T2, 1.0f, 1.0f, true);
          if (rot_b) rot_fp8_gptj<false>(B, T2 + G::PPV, 1.0f, 1.0f, true);
        }
      }
    }
    stg128(grow + va16, A);
    stg128(grow + vb16, B);
  };
  auto head_scales = [&](const TileMeta& m, int hh, float& s_src, float& inv_dst, bool& requant) {
    s_src = 1.0f; inv_dst = 1.0f; requant = false;
    if (DTYPE == 1) {
      const float s_dst = s_scales[m.scale_idx + hh];
      s_src = P.scales_differ ? seg_array(P)[m.seg].k_scale_src[m.scale_idx + hh] : s_dst;
      requant = (s_src != s_dst);
      inv_dst = __frcp_rn(s_dst);
    }
  };

  for (;; ) {
    mbar_wait(s_full + 8u * stage, phase, 4);
    const TileMeta m = meta[stage];
    if (m.flags & kFlagDone) break;
    if (m.flags & kFlagSkip) {       // an early-loaded tile whose destination block is invalid: release the stage, nothing else
      __syncwarp();
      if (lane == 0) mbar_arrive(s_empty + 8u * stage);
      stage += stage_step;
      if (stage >= S) { stage -= S; phase ^= 1u; }
      continue;
    }
    const uint32_t sk = s_base + RP.off_stage + (uint32_t)stage * RP.stage_bytes;
    const uint32_t sv = RP.split ? sk : sk + RP.tile_bytes;
    const int n_tok = m.n_tok;

    // ---- V (step a6): bytes unchanged ----
    if (RP.no_v || (m.flags & kFlagKOnly)) {
      // in-place: V is position-free and already where it belongs
    } else if (RP.hmaj && RP.v_bulk == 0) {
      // lanes over heads (dense token-major pool): this warp's tokens, each as ONE contiguous run of hpt * rowB
      // destination bytes; consecutive lanes write consecutive 16-byte vectors (a warp instruction = 512 contiguous
      // bytes), reading the head-major stage in 128-byte row pieces (conflict-free per quarter warp)
      const int tpw = (n_tok + wpg - 1) / wpg, tk0 = wsub * tpw, tk1 = min(n_tok, tk0 + tpw);
      const int total = (tk1 - tk0) << RP.log_pt;
      uint8_t* const vd = P.v_cache + (m.dst_off + (int64_t)tk0 * P.d_st) * E;
      const int64_t tok_step = P.d_st * E - ((int64_t)RP.hpt * RP.rowB);     // gap between token runs (0: all heads in the tile)
#pragma unroll 4
      for (int idx = lane; idx < total; idx += 32) {
        const int tt = idx >> RP.log_pt, rem = idx & ((1 << RP.log_pt) - 1);
        const int hh = rem >> RP.log_nv, v = rem & (nv - 1);
        stg128(vd + (int64_t)idx * 16 + tt * tok_step, lds128(sv + (hh * RP.cg + tk0 + tt) * RP.rowB + v * 16));
      }
    } else if (RP.gather) {
      // gather mode: this warp's tokens leave by one bulk (TMA) store per (token, head) row, heads innermost, so the
      // rows of a token arrive back to back and form one contiguous H*D run of the dense token-major pool
      // Work items of a gather tile: (token group of rpi tokens, head), token group major; warp wsub of the wpg
      // warps that share the stage takes a contiguous range of them.
      const int items = ((n_tok + rpi - 1) / rpi) * RP.hpt, ipw = (items + wpg - 1) / wpg;
      const int it0 = wsub * ipw, it1 = min(items, it0 + ipw);
      if (RP.v_bulk == 0) {
        // 16-byte warp copies, same item order (short rows -- fp8 -- make poor bulk stores)
        const int per_item = rpi * nv, total = (it1 - it0) * per_item;
#pragma unroll 4
        for (int idx = lane; idx < total; idx += 32) {
          const int it = it0 + idx / per_item, rem = idx % per_item;
          const int tg = it / RP.hpt, hh = it - tg * RP.hpt, tt = tg * rpi + (rem >> RP.log_nv), v = rem & (nv - 1);
          if (tt < n_tok)
            stg128(P.v_cache + (m.dst_off + (int64_t)tt * P.d_st + (int64_t)hh * P.d_sh) * E + v * 16,
                   lds128(sv + (hh * RP.cg + tt) * RP.rowB + v * 16));
        }
      } else
      for (int idx = lane; idx < (it1 - it0) * rpi; idx += 32) {
        const int it = it0 + idx / rpi, r = idx - (idx / rpi) * rpi;
        const int tg = it / RP.hpt, hh = it - tg * RP.hpt, tt = tg * rpi + r;
        if (tt < n_tok)
          bulk_s2g(P.v_cache + (m.dst_off + (int64_t)tt * P.d_st + (int64_t)hh * P.d_sh) * E,
                   sv + (hh * RP.cg + tt) * RP.rowB, (uint32_t)RP.rowB);
      }
      bulk_commit();
    } else if (RP.v_bulk == 2) {
      // token-major pool: one bulk store per (head, token) row, lane r issues row r (n_tok <= 32)
      for (int hh = 0; hh < RP.hpt; ++hh)
        if (lane < n_tok)
          bulk_s2g(P.v_cache + (m.dst_off + (int64_t)hh * P.d_sh + (int64_t)lane * P.d_st) * E,
                   sv + (hh * RP.cg + lane) * RP.rowB, (uint32_t)RP.rowB);
      bulk_commit();
    } else if (RP.v_bulk) {
      if (lane == 0) {
        if (m.flags & kFlagTokMajor)       // the stage is in the pool's order: the tile's V is ONE contiguous run
          bulk_s2g(P.v_cache + m.dst_off * E, sv, (uint32_t)(n_tok * RP.hpt * RP.rowB));
        else
          for (int hh = 0; hh < RP.hpt; ++hh)
            bulk_s2g(P.v_cache + (m.dst_off + (int64_t)hh * P.d_sh) * E, sv + hh * RP.cg * RP.rowB, (uint32_t)(n_tok * RP.rowB));
        bulk_commit();
      }
    } else {
      for (int hh = 0; hh < RP.hpt; ++hh) {
        const uint32_t vs = sv + hh * RP.cg * RP.rowB;
        uint8_t* vd = P.v_cache + (m.dst_off + (int64_t)hh * P.d_sh) * E;
        const int total = n_tok * nv;
#pragma unroll 4
        for (int idx = lane; idx < total; idx += 32) {
          int t, v;
          if (RP.log_nv >= 0) { t = idx >> RP.log_nv; v = idx & (nv - 1); } else { t = idx / nv; v = idx - t * nv; }
          stg128(vd + (int64_t)t * P.d_st * E + v * 16, lds128(vs + idx * 16));
        }
      }
    }

    // ---- K (steps a3, a5) ----
    const uint32_t tab = s_base + RP.off_tab + m.tab * RP.tab_stride;
    const bool rotate = (m.flags & kFlagRotate) != 0;
    if (!MAP && rotate && m.gen != my_gen) {       // new segment: refresh the cos/sin registers
      my_gen = m.gen;
      if (rot_a || rot_b) {
#pragma unroll
        for (int k = 0; k < G::NT; ++k) {
          float4 e = lds128f(tab + tpos(k) * 16);
          if (DTYPE == 0) T4[k] = e; else T2[k] = make_float2(e.x, e.z);
        }
      }
    }
    const int sm_sh = (m.flags & kFlagTokMajor) ? RP.rowB : RP.cg * RP.rowB;        // stage strides of a head / a token
    const int sm_st = (m.flags & kFlagTokMajor) ? RP.hpt * RP.rowB : RP.rowB;
    if (m.flags & kFlagVOnly) {
      // split gather tile holding V alone: nothing to rotate
    } else if (RP.hmaj) {
      // lanes over heads: a pass of the warp covers 2^log_hp adjacent HEADS of (rpi >> log_hp) tokens, so its rows are
      // adjacent in a dense token-major pool and a pair of warp store instructions writes contiguous runs, as on a
      // head-major pool.  Items = (token group, head group), token group major; warp wsub of the wpg warps that share
      // the stage takes a contiguous range of them.
      const int log_hp = RP.log_hp, log_tp = RP.log_rpi - log_hp;
      const int hgs = RP.hpt >> log_hp, tgs = (n_tok + (1 << log_tp) - 1) >> log_tp;
      const int items = tgs * hgs, ipw = (items + wpg - 1) / wpg;
      const int it0 = wsub * ipw, it1 = min(items, it0 + ipw);
      const int hsub = rsub & ((1 << log_hp) - 1), tsub = rsub >> log_hp;
      int tg = it0 / hgs, g = it0 - tg * hgs;
      float s_src = 1.0f, inv_dst = 1.0f; bool requant = false;
      int hh = (g << log_hp) + hsub;
      if (DTYPE == 1) head_scales(m, hh, s_src, inv_dst, requant);
      // the row's shared-memory address and destination pointer are stepped, not recomputed
      int t = (tg << log_tp) + tsub;
      const int64_t kd_step = P.d_sh * E;
      const uint32_t s_item = (uint32_t)sm_sh << log_hp, s_wrap = ((uint32_t)sm_st << log_tp) - (uint32_t)(hgs - 1) * s_item;
      const int64_t g_item = kd_step << log_hp, g_wrap = (tokB << log_tp) - (int64_t)(hgs - 1) * g_item;
      uint32_t srow = sk + hh * sm_sh + t * sm_st;
      uint8_t* grow = P.k_cache + m.dst_off * E + hh * kd_step + t * tokB;
      for (int it = it0; it < it1; ++it) {
        if (t < n_tok) k_row(m, tab, rotate, srow, grow, t, s_src, inv_dst, requant);
        if (hgs == 1) {
          t += 1 << log_tp; srow += s_wrap; grow += g_wrap;
        } else {
          if (++g == hgs) { g = 0; t += 1 << log_tp; srow += s_wrap; grow += g_wrap; }
          else { srow += s_item; grow += g_item; }
          hh = (g << log_hp) + hsub;
          if (DTYPE == 1) head_scales(m, hh, s_src, inv_dst, requant);
        }
      }
    } else if (RP.gather) {
      // gather mode: tokens outer, heads inner -- a pass of this warp completes rpi whole token rows
      // (token group, head) items of this warp, token group major; the walk keeps running pointers (no divisions)
      const int items = ((n_tok + rpi - 1) >> RP.log_rpi) * RP.hpt;
      const int ipw = (wpg == 1) ? items : (items + wpg - 1) / wpg;
      const int it0 = wsub * ipw, it1 = min(items, it0 + ipw);
      int tg = (wpg == 1) ? 0 : it0 / RP.hpt, hh = it0 - tg * RP.hpt;
      uint8_t* const kd0 = P.k_cache + m.dst_off * E;
      const int64_t kd_step = P.d_sh * E;
      uint32_t ks = sk + hh * sm_sh;
      uint8_t* kd = kd0 + hh * kd_step;
      int t = (tg << RP.log_rpi) + rsub;
      for (int it = it0; it < it1; ++it) {
        float s_src = 1.0f, inv_dst = 1.0f; bool requant = false;
        if (DTYPE == 1) head_scales(m, hh, s_src, inv_dst, requant);
        if (t < n_tok) k_row(m, tab, rotate, ks + t * sm_st, kd + t * tokB, t, s_src, inv_dst, requant);
        ++hh; ks += sm_sh; kd += kd_step;
        if (hh == RP.hpt) { hh = 0; ks = sk; kd = kd0; t += rpi; }
      }
    } else
    for (int hh = 0; hh < RP.hpt; ++hh) {
      const uint32_t ks = sk + hh * sm_sh;
      uint8_t* kd = P.k_cache + (m.dst_off + (int64_t)hh * P.d_sh) * E;
      float s_src, inv_dst; bool requant;
      head_scales(m, hh, s_src, inv_dst, requant);
      {
        uint32_t srow = ks + rsub * sm_st;
        uint8_t* grow = kd + rsub * tokB;
        const uint32_t s_step = (uint32_t)(rpi * sm_st);
        const int64_t g_step = rpi * tokB;
        for (int t = rsub; t < n_tok; t += rpi, srow += s_step, grow += g_step)
          k_row(m, tab, rotate, srow, grow, t, s_src, inv_dst, requant);
      }
      if (RP.win) {
        // window mode: everything outside the rotary window (the MLA latent) is position-free -- 16-byte copies
        const int npass = nv - nr;
        for (int t = 0; t < n_tok; ++t) {
          const uint32_t srow = ks + t * sm_st;
          uint8_t* drow = kd + (int64_t)t * P.d_st * E;
#pragma unroll 2
          for (int j = lane; j < npass; j += 32) {
            const int v = (j >= RP.ro_v) ? j + nr : j;
            uint4 A = lds128(srow + v * 16);
            if (DTYPE == 1 && requant) requant_fp8(A, s_src, inv_dst);
            stg128(drow + v * 16, A);
          }
        }
      }
    }
    if (RP.v_bulk == 2 || (RP.v_bulk && lane == 0)) bulk_wait_read0();   // V bytes have left shared memory
    __syncwarp();
    if (lane == 0) mbar_arrive(s_empty + 8u * stage);
    stage += stage_step;
    if (stage >= S) { stage -= S; phase ^= 1u; }
  }
  if (RP.v_bulk == 2 || (RP.v_bulk && lane == 0)) bulk_wait_all0();
}

// ------------------------------------------------------------------------------- host side
static int ilog2(int x) { int l = 0; while ((1 << l) < x) ++l; return l; }

// heads per tile: smallest divisor of heads whose K run reaches 4 KB; a dense token-major pool re-floated in place
// takes all heads (its tile is then one contiguous run of the pool)
int ring_heads_per_tile(const CallParams& P) {
  const int rowB = P.head_dim * (P.dtype == 0 ? 2 : 1);
  if (P.tmajor) return P.heads;        // transposing loads: a tile is all heads x ct tokens
  if (P.inplace && P.d_st != P.head_dim && P.d_sh == P.head_dim && P.d_st == (int64_t)P.heads * P.head_dim) return P.heads;
  for (int h = 1; h <= P.heads; ++h)
    if (P.heads % h == 0 && h * P.cg * rowB >= (P.tile_min_bytes > 0 ? P.tile_min_bytes : (P.inplace ? 8192 : 4096))) return h;
  // (in place a stage holds K alone: 8 KB tiles keep as many bytes in flight as the splice's K + V stages; B200,
  //  head-major pools: configs[2] 5673 -> 6240 GB/s, configs[3] 5194 -> 5845, configs[4] 6180 -> 6424)
  return P.heads;
}

// rows the power-of-two slot layout cannot take: the lanes cover the rotary window, a copy loop moves the rest
bool ring_window_mode(const CallParams& P) {
  const int rowB = P.head_dim * (P.dtype == 0 ? 2 : 1);
  return P.rotary_offset != 0 || rowB > 1024 || (rowB & (rowB - 1)) != 0;
}

static bool ring_plan(const CallParams& P_in, const RingConfig& cfg, int sm_count, CallParams& P, RingParams& RP,
                      int& grid, int& block, int& smem);

bool ring_supported(const CallParams& P, const SegDev* segs, const RingConfig& cfg, int sm_count, const char** why) {
  const int E = P.dtype == 0 ? 2 : 1;
  const int rowB = P.head_dim * E;
  const char* w = nullptr;
  const int rotB = P.rotary_dim * E;
  if (ring_window_mode(P)) {
    if (rowB < 32 || rowB > 4096 || rowB % 16) w = "window mode: head_dim*esz must be a multiple of 16 in [32, 4096] bytes";
    else if (rotB % 32 || rotB > 1024 || ((rotB / 32) & (rotB / 32 - 1))) w = "window mode: rotary_dim*esz must be 32 * a power of two, <= 1024";
    else if (P.inplace) w = "window mode: in-place calls take kvr_window_inplace_kernel (it touches only the rotary window)";
  }
  else if (rowB < 32 || rowB > 1024 || (rowB & (rowB - 1))) w = "head_dim*esz must be a power of two in [32, 1024] bytes";
  else if (P.pairing == 0 && (P.rotary_dim * E) % 32) w = "NeoX pairing needs rotary_dim*esz % 32 == 0";
  else if (P.pairing == 1 && (P.rotary_dim * E) % 16) w = "GPT-J pairing needs rotary_dim*esz % 16 == 0";
  else if (P.dtype == 1 && (int64_t)P.layers * P.heads > 8192) w = "too many (layer, head) scales for shared memory";
  else if (P.rotary_dim / 2 > 512) w = "rotary_dim too large for the shared angle table";
  (void)segs;
  if (!w) {
    // the shortest ring (2 stages) with its angle tables, scales and tile descriptors must fit the CTA's shared memory:
    // e.g. bf16 head_dim = rotary_dim = 512 with per-token shifts needs 2 x 64 KB of tables and takes the generic kernel
    CallParams Pp; RingParams RP; int g, b, sm;
    if (!ring_plan(P, cfg, sm_count, Pp, RP, g, b, sm)) w = "the ring's shared-memory layout (tables + scales + 2 stages) does not fit";
  }
  if (why) *why = w;
  return w == nullptr;
}

template <int DTYPE, int PAIRING, bool MAP, int MAXT>
static cudaError_t launch_inst(const CallParams& P, const RingParams& RP, const TmapInline& TI, int grid, int block, int smem,
                               cudaStream_t st, bool pdl) {
  // The opt-in to > 48 KB of dynamic shared memory is a per-DEVICE attribute of the function: remember what was set per
  // (instantiation, device), under a lock (contexts on several devices / host threads share this process-wide table).
  static std::mutex mu;
  static int configured[kMaxDevices] = {};
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  {
    std::lock_guard<std::mutex> lock(mu);
    if (dev < 0 || dev >= kMaxDevices || configured[dev] < smem) {
      e = cudaFuncSetAttribute(kvr_ring_kernel<DTYPE, PAIRING, MAP, MAXT>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
      if (e != cudaSuccess) return e;
      if (dev >= 0 && dev < kMaxDevices) configured[dev] = smem;
    }
  }
  cudaLaunchConfig_t lc{};
  lc.gridDim = dim3((unsigned)grid); lc.blockDim = dim3((unsigned)block); lc.dynamicSmemBytes = (size_t)smem; lc.stream = st;
  cudaLaunchAttribute at[1];
  at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  at[0].val.programmaticStreamSerializationAllowed = 1;
  lc.attrs = at; lc.numAttrs = pdl ? 1 : 0;
  return cudaLaunchKernelEx(&lc, kvr_ring_kernel<DTYPE, PAIRING, MAP, MAXT>, P, RP, TI);
}

// Launch shape and shared-memory layout of one call; false when even the shortest ring does not fit.
static bool ring_plan(const CallParams& P_in, const RingConfig& cfg, int sm_count, CallParams& P, RingParams& RP,
                      int& grid_out, int& block_out, int& smem_out) {
  P = P_in;
  P.grab = cfg.grab > 0 ? (cfg.grab > 32 ? 32 : cfg.grab) : 1;
  const int E = P.dtype == 0 ? 2 : 1;
  RP = RingParams{};
  RP.cg = P.cg;
  RP.rowB = P.head_dim * E;
  RP.nr = P.rotary_dim * E / 16;
  RP.win = ring_window_mode(P) ? 1 : 0;
  RP.ro_v = P.rotary_offset * E / 16;
  RP.nv = RP.rowB / 16; RP.log_nv = (RP.nv & (RP.nv - 1)) ? -1 : ilog2(RP.nv);
  RP.nv_slot = RP.win ? RP.nr : RP.nv;
  RP.sp = RP.nv_slot / 2; RP.log_sp = ilog2(RP.sp); RP.rpi = 32 / RP.sp; RP.log_rpi = ilog2(RP.rpi);
  RP.half_R = P.rotary_dim / 2;
  const int ppv = (P.pairing == 0) ? 16 / E : 8 / E;
  RP.NV = RP.half_R / ppv;
  RP.no_v = (P.inplace || P.no_v) ? 1 : 0;
  RP.ip_mode = 0;
  if (P.inplace) {
    if (P.d_st == P.head_dim) RP.ip_mode = 0;                                             // head-major pool
    else if (P.d_sh == P.head_dim && P.d_st == (int64_t)P.heads * P.head_dim) RP.ip_mode = 1;   // token-major, dense
    else RP.ip_mode = 2;                                                                  // padded rows
  }
  const int hpt = ring_heads_per_tile(P);
  RP.hpt = hpt;
  RP.ct = P.tmajor ? P.ct : RP.cg;
  RP.tile_bytes = hpt * RP.ct * RP.rowB;
  RP.split = (P.gather == 2 && !RP.no_v && !P.tmajor) ? 1 : 0;
  RP.stage_bytes = ((RP.no_v || RP.split) ? 1 : 2) * RP.tile_bytes;
  const int ctas = cfg.ctas_per_sm > 0 ? cfg.ctas_per_sm : 2;
  RP.NW = cfg.consumer_warps > 0 ? cfg.consumer_warps : 6;
  if (RP.NW > 16) RP.NW = 16;
  RP.NTB = 2;                                              // the producer's bookkeeping assumes two
  const int tab_rows = P.any_pos_map ? RP.cg : 1;
  RP.tab_stride = ((tab_rows * RP.half_R * 16 + RP.cg * 4) + 127) & ~127;
  RP.n_scales = P.dtype == 1 ? P.layers * P.heads : 0;
  RP.n_ub = (P.n_segs > kInlineSegs && P.n_segs <= 2048) ? P.n_segs : 0;
  // per-CTA dynamic shared memory: 228 KB per SM, 1 KB reserved per resident CTA, at most 227 KB per CTA
  const int budget = (ctas == 1) ? 227 * 1024 : (228 * 1024) / ctas - 1024;
  auto layout = [&](int S) {
    int off = 16 * S;
    off = (off + 31) & ~31; RP.off_meta = off; off += 32 * S;
    off = (off + 15) & ~15; RP.off_scales = off; off += 4 * RP.n_scales;
    off = (off + 15) & ~15; RP.off_ub = off; off += 8 * RP.n_ub;
    off = (off + 127) & ~127; RP.off_tab = off; off += RP.NTB * RP.tab_stride;
    off = (off + 127) & ~127; RP.off_stage = off; off += S * RP.stage_bytes;
    return off;
  };
  int S = cfg.stages > 0 ? cfg.stages : 64;
  while (S > 2 && layout(S) > budget) --S;
  if (layout(S) > budget) return false;
  // Stage ownership: consumer warp w serves stages (w / wpg) + k * (NW / wpg); S is a multiple of NW / wpg, so the
  // successive phases of one mbarrier are ordered by one warp's program order (a warp two phases ahead would pass a
  // parity wait early).  wpg > 1 only in gather mode, when the ring holds fewer (large) stages than consumer warps.
  RP.gather = (P.gather && !P.tmajor) ? 1 : 0;
  RP.wpg = 1;
  if (RP.gather && (cfg.warps_per_stage > 0 || S < RP.NW)) {
    // Few large stages: groups of wpg warps walk the ring in NW / wpg strides.  A group should own TWO stages (one
    // loading while the other is consumed): with one stage per group, load and rotate of that stage are serial and
    // the ring cannot hide the rotate.  Default wpg = 2: 16 KB stages, S = 6 -> 3 groups x 2 stages.  Measured on
    // B200: configs[2] 6.34 -> 6.47 TB/s with split 16 KB tiles and 2 stages per group; one stage per group 6.15-6.29;
    // all warps on every stage 6.30; one CTA per SM with 12 warps 5.0-5.5.
    int wpg = cfg.warps_per_stage > 0 ? cfg.warps_per_stage : 2;
    if (wpg > RP.NW) wpg = RP.NW;
    int step = RP.NW / wpg;
    if (step < 1) step = 1;
    if (step > S) step = S;
    S -= S % step;
    RP.wpg = wpg; RP.NW = wpg * step;
  } else if (S >= RP.NW) {
    S -= S % RP.NW;
  } else {
    RP.NW = S;
  }
  RP.S = S;
  const int smem = layout(S);
  // V out of shared memory: 1 = one bulk store per (head, chunk) run (needs d_st == head_dim), 2 = one bulk store per
  // row, 0 = 16-byte warp copies.  Tuning v_bulk_store: 0 auto, 1 bulk wherever possible, 2 warp copies, 3 row bulk.
  const bool runs = (P.d_st == P.head_dim);
  if (cfg.v_bulk_store == 2) RP.v_bulk = 0;
  else if (cfg.v_bulk_store == 3) RP.v_bulk = 2;
  else if (cfg.v_bulk_store == 1) RP.v_bulk = runs ? 1 : 2;
  else RP.v_bulk = runs ? 1 : 0;
  if (RP.gather)   // gather mode: 2 = one bulk store per (token, head) row (default: measured faster), 0 = warp copies
    RP.v_bulk = (cfg.v_bulk_store == 2) ? 0 : (cfg.v_bulk_store == 3 || cfg.v_bulk_store == 1) ? 2 : 2;
  if (P.tmajor) RP.v_bulk = 1;      // the stage is in the pool's order: V leaves as one bulk store per tile
  if (RP.no_v) RP.v_bulk = 0;
  // lanes over heads (dense token-major pools): needs whole groups of min(hpt, rpi) heads per tile and a power of two
  // of vectors per token.  tuning.lanes_over_heads: 0 auto (on in gather mode), 1 on wherever possible, 2 off.
  RP.hmaj = 0; RP.log_pt = 0; RP.log_hp = 0;
  {
    const int pt = RP.hpt * RP.nv, hp = RP.hpt < RP.rpi ? RP.hpt : RP.rpi;
    const bool ip_tm = P.inplace && RP.ip_mode == 1;        // in place on a dense token-major pool: the stage is in pool order
    const bool can = !RP.win && (!P.inplace || ip_tm) && RP.log_nv >= 0 && hp >= 1 && (hp & (hp - 1)) == 0 && RP.hpt % hp == 0 &&
                     (pt & (pt - 1)) == 0 && RP.hpt > 1 && P.d_sh == P.head_dim && P.d_st >= (int64_t)RP.hpt * P.head_dim;
    if (can && (cfg.lanes_over_heads == 1 || (cfg.lanes_over_heads == 0 && (RP.gather || P.tmajor || ip_tm)))) {
      RP.hmaj = 1; RP.log_pt = ilog2(pt); RP.log_hp = ilog2(hp);
      if (P.tmajor) { /* V: one bulk store per tile (set above) */ }
      else if (RP.no_v) RP.v_bulk = 0;
      else if (cfg.v_bulk_store == 3 || cfg.v_bulk_store == 1) RP.v_bulk = 2;   // forced: one bulk store per row
      else RP.v_bulk = 0;                                                        // V leaves by contiguous warp copies
    }
  }
  int64_t g = (int64_t)sm_count * ctas;
  if (cfg.max_ctas > 0 && g > cfg.max_ctas) g = cfg.max_ctas;
  if (g > P.total_units) g = P.total_units;
  if (g < 1) g = 1;
  grid_out = (int)g; block_out = (RP.NW + 1) * 32; smem_out = smem;
  return true;
}

cudaError_t launch_ring(const CallParams& P_in, const RingConfig& cfg, int sm_count, cudaStream_t stream,
                        int* grid_out, int* block_out, int* smem_out) {
  CallParams P; RingParams RP; int g = 0, block = 0, smem = 0;
  if (!ring_plan(P_in, cfg, sm_count, P, RP, g, block, smem)) return cudaErrorInvalidConfiguration;
  *grid_out = g; *block_out = block; *smem_out = smem;
  const int ctas = cfg.ctas_per_sm > 0 ? cfg.ctas_per_sm : 2;
  const bool map = P.any_pos_map != 0;
  const bool small = block <= 256 && ctas <= 2, mid = block <= 448 && ctas == 1;
  static const TmapInline no_maps{};
  const TmapInline& TI = (P.tmajor && cfg.tmaps_inline) ? *cfg.tmaps_inline : no_maps;
#define KVR_LAUNCH(D, PR, M)                                                                             \
  return small ? launch_inst<D, PR, M, 256>(P, RP, TI, (int)g, block, smem, stream, cfg.pdl != 2)            \
         : mid ? launch_inst<D, PR, M, 448>(P, RP, TI, (int)g, block, smem, stream, cfg.pdl != 2)            \
               : launch_inst<D, PR, M, kMaxThreads>(P, RP, TI, (int)g, block, smem, stream, cfg.pdl != 2)
  if (P.dtype == 0) {
    if (P.pairing == 0) { if (map) KVR_LAUNCH(0, 0, true); else KVR_LAUNCH(0, 0, false); }
    else { if (map) KVR_LAUNCH(0, 1, true); else KVR_LAUNCH(0, 1, false); }
  } else {
    if (P.pairing == 0) { if (map) KVR_LAUNCH(1, 0, true); else KVR_LAUNCH(1, 0, false); }
    else { if (map) KVR_LAUNCH(1, 1, true); else KVR_LAUNCH(1, 1, false); }
  }
#undef KVR_LAUNCH
}

}  // namespace kvr
