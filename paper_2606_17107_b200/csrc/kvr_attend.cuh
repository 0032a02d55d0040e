// kvr_attend.cuh -- device-side structures of the rotate-on-read attention kernel (kvr_attend.cu) and its launcher.
// Product code (sm_100a).  Shares nothing with oracle/.
#pragma once
#include "kvr_common.cuh"

namespace kvr {

// One segment of a rotate-on-read call: TMA tensor maps of its K and V sources, dims ordered (dim, token, head, layer),
// box {64 dims, 128 tokens, 1, 1}, SWIZZLE_128B -- a tile of 128 keys lands as two 64-dim panels of 128-byte rows, the
// canonical K-major (K) / MN-major (V) shared-memory operand layout of tcgen05.mma.
struct alignas(64) AttnSeg {
  CUtensorMap k, v;
  int32_t delta, len, request, pad_;
};

// One work item: keys [key0, key0 + n_keys) of kv head `head` of segment `seg`.  Items of one (request, kv head) group
// are numbered consecutively: [group_first, group_first + |group_count|); group_count < 0: the group is merged after
// the grid (AttnMerge), its items only write their partials.
struct AttnItem {
  int32_t seg, head, key0, n_keys;
  int32_t group, group_first, group_count;
  int32_t index;           // this item's own number (its slot in the partial buffers); items are handed out dynamically
};

// A group whose partials are merged after the attention grid (kvr_attend_merge_kernel): partials [first, first + count).
struct AttnMerge { int32_t first, count, out_q0, pad_; };

struct AttnParams {
  const uint16_t* q;       // bf16 [n_req][q_heads][128]
  float* o;                // [n_req][q_heads][128]
  float* lse;              // [n_req][q_heads]
  const AttnSeg* segs;
  const AttnItem* items;
  const AttnMerge* merges;
  int32_t n_items, n_merges;
  int32_t merge_max_count; // largest group among `merges`
  int32_t early;           // every segment carries KVR_SEG_SRC_STABLE: the TMA producers need not wait for the previous kernel
  int32_t q_heads, group;  // group = q_heads / kv_heads
  int32_t layer, rotary_dim, rotary_offset, pairing;
  float scale_log2;        // softmax_scale * log2(e)
  const double* inv_freq;  // DEVICE, rotary_dim / 2
  float* part_o;           // [n_items][group][128]: unnormalised O^T of an item, relative to its reference maximum
  float* part_ml;          // [n_items][group][2]: reference maximum (log2 units), row sum
  unsigned int* tickets;   // [groups]: items of the group that have finished; zero between launches
  unsigned long long* sched;   // [0] next item to hand out (beyond the first, static one per CTA), [1] CTAs that have
                               // finished; both zero between launches (the last CTA to finish resets them)
};

int attend_inline_merge_limit(int group);   // groups with more partials are merged by the merge kernel
cudaError_t launch_attend(const AttnParams& P, int sm_count, cudaStream_t stream, int* grid, int* block, int* smem);

}  // namespace kvr
