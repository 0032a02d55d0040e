// kvr_api.cu -- the C ABI of include/kvr.h: context, host-side validation, work decomposition,
// descriptor staging and kernel dispatch.  No arithmetic of the method happens on the host.
#include <algorithm>
#include <cmath>
#include <cstddef>
#include <cstdio>
#include <cstring>
#include <mutex>
#include <new>
#include <string>
#include <vector>

#include "../../include/kvr.h"
#include "kvr_attend.cuh"
#include "kvr_common.cuh"

using namespace kvr;

namespace {

constexpr int kSlots = 16;          // descriptor staging ring (launches in flight per context)
constexpr int kStageBufs = 2;       // host-source path: device staging buffers (copy of group g+1 overlaps kernel g)
constexpr int kInitialSegCap = 256;
constexpr bool kTransposeAuto = true;    // tuning.transpose_load == 0: on (B200: every BASELINE config gains)

struct Slot {
  SegDev* host = nullptr;           // pinned
  SegDev* dev = nullptr;
  size_t cap = 0;
  TmapPair* tm_host = nullptr;      // pinned: tensor maps of the segments' sources (transposing loads), allocated on demand
  TmapPair* tm_dev = nullptr;
  size_t tm_cap = 0;
  cudaEvent_t ev = nullptr;
  bool pending = false;
};

// cuTensorMapEncodeTiled, fetched from the driver the runtime has already loaded (no link against libcuda)
typedef CUresult (*TmapEncodeFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                 const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                 CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
TmapEncodeFn tmap_encoder() {
  static TmapEncodeFn fn = nullptr;
  static std::once_flag once;
  std::call_once(once, [] {
    void* p = nullptr;
    cudaDriverEntryPointQueryResult qr;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &qr) == cudaSuccess &&
        qr == cudaDriverEntryPointSuccess)
      fn = reinterpret_cast<TmapEncodeFn>(p);
    (void)cudaGetLastError();
  });
  return fn;
}

// Tensor map of one source tensor [layers][heads][len][head_dim] (element strides sl, sh, st) with its dimensions ordered
// (dim, head, token, layer): a box {head_dim, heads, ct, 1} then lands in shared memory as [token][head][dim].
bool encode_source_map(CUtensorMap* out, const void* base, int dtype, int head_dim, int heads, int len, int layers,
                       int64_t sl, int64_t sh, int64_t st, int ct) {
  TmapEncodeFn enc = tmap_encoder();
  if (!enc || !base) return false;
  const uint64_t E = dtype == KVR_BF16 ? 2 : 1, rowB = (uint64_t)head_dim * E;
  // a dimension of extent 1 never uses its stride: give it a legal one
  uint64_t s_h = (uint64_t)sh * E, s_t = (uint64_t)st * E, s_l = (uint64_t)sl * E;
  if (heads == 1 && s_h == 0) s_h = rowB;
  if (len == 1 && s_t == 0) s_t = rowB;
  if (layers == 1 && s_l == 0) s_l = rowB;
  if (s_h == 0 || s_t == 0 || s_l == 0) return false;
  const cuuint64_t dims[4] = {(cuuint64_t)head_dim, (cuuint64_t)heads, (cuuint64_t)len, (cuuint64_t)layers};
  const cuuint64_t strides[3] = {s_h, s_t, s_l};
  const cuuint32_t box[4] = {(cuuint32_t)head_dim, (cuuint32_t)heads, (cuuint32_t)ct, 1u};
  const cuuint32_t es[4] = {1u, 1u, 1u, 1u};
  const CUtensorMapL2promotion promo = rowB >= 256 ? CU_TENSOR_MAP_L2_PROMOTION_L2_256B
                                     : rowB >= 128 ? CU_TENSOR_MAP_L2_PROMOTION_L2_128B : CU_TENSOR_MAP_L2_PROMOTION_NONE;
  return enc(out, dtype == KVR_BF16 ? CU_TENSOR_MAP_DATA_TYPE_UINT16 : CU_TENSOR_MAP_DATA_TYPE_UINT8, 4,
             const_cast<void*>(base), dims, strides, box, es, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
             promo, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

inline int elt_bytes(int dtype) { return dtype == KVR_BF16 ? 2 : 1; }

kvr_status check_model(const kvr_model_desc* m) {
  if (!m || !m->inv_freq) return KVR_ERR_INVALID_ARG;
  if (m->layers <= 0 || m->kv_heads <= 0 || m->head_dim <= 0) return KVR_ERR_INVALID_ARG;
  if (m->rotary_dim < 2 || (m->rotary_dim & 1) || m->rotary_offset < 0 || m->reserved_ != 0 ||
      (int64_t)m->rotary_offset + m->rotary_dim > m->head_dim)
    return KVR_ERR_INVALID_ARG;
  if (m->pairing != KVR_PAIR_NEOX_HALF && m->pairing != KVR_PAIR_GPTJ_INTERLEAVED) return KVR_ERR_INVALID_ARG;
  if (m->dtype != KVR_BF16 && m->dtype != KVR_FP8_E4M3) return KVR_ERR_INVALID_ARG;
  if (((int64_t)m->head_dim * elt_bytes(m->dtype)) % 16 != 0) return KVR_ERR_ALIGNMENT;
  if (((int64_t)m->rotary_offset * elt_bytes(m->dtype)) % 16 != 0) return KVR_ERR_ALIGNMENT;
  return KVR_OK;
}

inline bool aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }

kvr_status check_call(const kvr_model_desc* m, const kvr_paged_dst* d, const kvr_segment* segs, int32_t n) {
  kvr_status st = check_model(m);
  if (st != KVR_OK) return st;
  if (!d || n < 0 || (n > 0 && !segs)) return KVR_ERR_INVALID_ARG;
  if (!d->k_cache || !d->block_table) return KVR_ERR_INVALID_ARG;
  const bool k_only = (d->v_cache == nullptr);   // a [latent | k_pe] cache: one tensor per token (kvr.h, NEXT-3)
  if (d->num_blocks <= 0 || d->block_size <= 0 || d->num_seqs <= 0 || d->max_blocks_per_seq <= 0)
    return KVR_ERR_INVALID_ARG;
  if (d->stride_layer < 0 || d->stride_block <= 0 || (d->stride_token < m->head_dim && d->block_size > 1))
    return KVR_ERR_INVALID_ARG;
  if (d->stride_head < m->head_dim && m->kv_heads > 1) return KVR_ERR_INVALID_ARG;
  if (m->dtype == KVR_FP8_E4M3 && !d->k_scale) return KVR_ERR_INVALID_ARG;
  const int E = elt_bytes(m->dtype);
  if (!aligned16(d->k_cache) || !aligned16(d->v_cache)) return KVR_ERR_ALIGNMENT;
  const int64_t ds[4] = {d->stride_layer, d->stride_block, d->stride_token, d->stride_head};
  for (int64_t s : ds)
    if ((s * E) % 16 != 0) return KVR_ERR_ALIGNMENT;
  const int64_t cap = (int64_t)d->max_blocks_per_seq * d->block_size;
  for (int32_t i = 0; i < n; ++i) {
    const kvr_segment& s = segs[i];
    if (!s.k_src || (s.v_src == nullptr) != k_only) return KVR_ERR_INVALID_ARG;
    if (s.len <= 0 || s.dst_seq < 0 || s.dst_seq >= d->num_seqs || s.dst_token_start < 0)
      return KVR_ERR_INVALID_ARG;
    if (s.old_start < 0 || (!s.pos_map && s.new_start < 0)) return KVR_ERR_INVALID_ARG;
    if (s.src_stride_token < m->head_dim && s.len > 1) return KVR_ERR_INVALID_ARG;
    if (s.src_stride_layer < 0 || s.src_stride_head < 0) return KVR_ERR_INVALID_ARG;
    if ((int64_t)s.dst_token_start + s.len > cap) return KVR_ERR_OUT_OF_RANGE;
    if (!aligned16(s.k_src) || !aligned16(s.v_src)) return KVR_ERR_ALIGNMENT;
    const int64_t ss[3] = {s.src_stride_layer, s.src_stride_head, s.src_stride_token};
    for (int64_t x : ss)
      if ((x * E) % 16 != 0) return KVR_ERR_ALIGNMENT;
    if (s.pos_map && (reinterpret_cast<uintptr_t>(s.pos_map) & 3u)) return KVR_ERR_ALIGNMENT;
    if (s.flags & ~(KVR_SEG_PRE_ROPE | KVR_SEG_SRC_STABLE)) return KVR_ERR_INVALID_ARG;
  }
  return KVR_OK;
}

// largest divisor of block_size that is <= limit
int chunk_granularity(int block_size, int limit) {
  if (limit < 1) limit = 1;
  for (int c = (block_size < limit ? block_size : limit); c >= 1; --c)
    if (block_size % c == 0) return c;
  return 1;
}

}  // namespace

struct kvr_ctx {
  kvr_model_desc model{};
  std::vector<double> inv_freq;
  double* d_inv_freq = nullptr;
  int32_t* d_status = nullptr;
  int32_t* h_status = nullptr;      // pinned
  unsigned long long* d_sched = nullptr;   // ring kernel's unit counter + finished-CTA counter (zero between launches)
  int device = 0, sm_count = 0;
  Slot slots[kSlots];
  int next_slot = 0;
  SegDev inline_scratch[kInlineSegs];   // host-side descriptors of calls that carry them in the kernel parameters
  kvr_tuning tuning{};
  uint64_t launches = 0;
  int last_path = 0, last_grid = 0, last_block = 0, last_smem = 0;
  cudaStream_t last_stream = nullptr;
  std::string last_err;
  // host-source path (kvr_reposition_splice_host)
  cudaStream_t copy_stream = nullptr;
  uint8_t* stage[kStageBufs] = {nullptr, nullptr};
  size_t stage_cap = 0;
  cudaEvent_t stage_filled[kStageBufs] = {nullptr, nullptr};   // recorded on copy_stream
  cudaEvent_t stage_drained[kStageBufs] = {nullptr, nullptr};  // recorded on the caller's stream
  bool stage_drained_valid[kStageBufs] = {false, false};
  cudaEvent_t fork_ev = nullptr;
  void* aux_dev = nullptr;            // pos_map / k_scale_src copies
  size_t aux_cap = 0;
  uint64_t h2d_bytes = 0;             // bytes the last host-source call copied host -> device
  // rotate-on-read attention (kvr_rotate_on_read_attention): descriptor staging ring, partial results, group tickets
  // A slot keeps the device-resident descriptors (tensor maps, work items) of one call, keyed by the call's segment
  // array: a decode loop reads the same skills at every step and every layer, so the same call comes back and then
  // enqueues nothing but its kernel.
  struct AttnSlot {
    unsigned char* host = nullptr; unsigned char* dev = nullptr; size_t cap = 0; cudaEvent_t ev = nullptr; bool pending = false;
    std::vector<unsigned char> key; int32_t n_req = 0, q_heads = 0, tpi_tuning = 0, n_groups = 0;
    size_t n_items = 0, seg_bytes = 0, n_merges = 0; int32_t merge_max = 0; uint64_t last_use = 0;
    bool pinned = false;          // captured in a CUDA graph: never evicted
    cudaStream_t last_stream = nullptr;   // stream of the last eager call on this entry (`ev` was recorded there)
  };
  static constexpr int kAttnSlots = 8;
  AttnSlot attn_slots[kAttnSlots];
  uint64_t attn_clock = 0;
  float* attn_part = nullptr;         // [items][group][128 + 2]
  size_t attn_part_cap = 0;           // bytes
  unsigned int* attn_tickets = nullptr;
  size_t attn_ticket_cap = 0;         // entries
  std::vector<void*> attn_retired;    // outgrown buffers a captured graph may still point at

  kvr_status cuda_fail(cudaError_t e, const char* what) {
    last_err = std::string(what) + ": " + cudaGetErrorString(e);
    (void)cudaGetLastError();
    return KVR_ERR_CUDA;
  }
};

#define KVR_CUDA(ctx, call)                                  \
  do {                                                       \
    cudaError_t e_ = (call);                                 \
    if (e_ != cudaSuccess) return (ctx)->cuda_fail(e_, #call); \
  } while (0)

static kvr_status slot_reserve_tmaps(kvr_ctx* c, Slot& s, size_t n);
static kvr_status slot_reserve(kvr_ctx* c, Slot& s, size_t n) {
  if (n <= s.cap) return KVR_OK;
  size_t cap = s.cap ? s.cap : kInitialSegCap;
  while (cap < n) cap *= 2;
  if (s.host) cudaFreeHost(s.host);
  if (s.dev) cudaFree(s.dev);
  s.host = nullptr; s.dev = nullptr; s.cap = 0;
  KVR_CUDA(c, cudaMallocHost(&s.host, cap * sizeof(SegDev)));
  KVR_CUDA(c, cudaMalloc(&s.dev, cap * sizeof(SegDev)));
  s.cap = cap;
  return KVR_OK;
}

static kvr_status slot_reserve_tmaps(kvr_ctx* c, Slot& s, size_t n) {
  if (n <= s.tm_cap) return KVR_OK;
  size_t cap = s.tm_cap ? s.tm_cap : kInitialSegCap;
  while (cap < n) cap *= 2;
  if (s.tm_host) cudaFreeHost(s.tm_host);
  if (s.tm_dev) cudaFree(s.tm_dev);
  s.tm_host = nullptr; s.tm_dev = nullptr; s.tm_cap = 0;
  KVR_CUDA(c, cudaMallocHost(&s.tm_host, cap * sizeof(TmapPair)));
  KVR_CUDA(c, cudaMalloc(&s.tm_dev, cap * sizeof(TmapPair)));
  s.tm_cap = cap;
  return KVR_OK;
}

extern "C" {

kvr_status kvr_create(kvr_ctx** out, const kvr_model_desc* model, int cuda_device) {
  if (!out) return KVR_ERR_INVALID_ARG;
  *out = nullptr;
  kvr_status st = check_model(model);
  if (st != KVR_OK) return st;
  int count = 0;
  if (cudaGetDeviceCount(&count) != cudaSuccess || cuda_device < 0 || cuda_device >= count) {
    (void)cudaGetLastError();
    return KVR_ERR_CUDA;   // no CUDA device: this library has no CPU fallback
  }
  cudaDeviceProp prop{};
  if (cudaGetDeviceProperties(&prop, cuda_device) != cudaSuccess) return KVR_ERR_CUDA;
  if (prop.major != 10) return KVR_ERR_UNSUPPORTED;   // built for sm_100a only
  kvr_ctx* c = new (std::nothrow) kvr_ctx();
  if (!c) return KVR_ERR_NOMEM;
  c->model = *model;
  c->inv_freq.assign(model->inv_freq, model->inv_freq + model->rotary_dim / 2);
  c->model.inv_freq = c->inv_freq.data();
  c->device = cuda_device;
  c->sm_count = prop.multiProcessorCount;
  int prev = 0;
  cudaGetDevice(&prev);
  cudaError_t e = cudaSetDevice(cuda_device);
  if (e == cudaSuccess) e = cudaMalloc(&c->d_inv_freq, c->inv_freq.size() * sizeof(double));
  if (e == cudaSuccess) e = cudaMemcpy(c->d_inv_freq, c->inv_freq.data(), c->inv_freq.size() * sizeof(double),
                                       cudaMemcpyHostToDevice);
  if (e == cudaSuccess) e = cudaMalloc(&c->d_status, 4 * sizeof(int32_t));
  if (e == cudaSuccess) e = cudaMemset(c->d_status, 0, 4 * sizeof(int32_t));
  if (e == cudaSuccess) e = cudaMallocHost(&c->h_status, 4 * sizeof(int32_t));
  if (e == cudaSuccess) e = cudaMalloc(&c->d_sched, 4 * sizeof(unsigned long long));   // [0..1] ring kernel, [2..3] attention kernel
  if (e == cudaSuccess) e = cudaMemset(c->d_sched, 0, 4 * sizeof(unsigned long long));
  for (int i = 0; i < kSlots && e == cudaSuccess; ++i)
    e = cudaEventCreateWithFlags(&c->slots[i].ev, cudaEventDisableTiming);
  // every staging slot is usable from the first call on (a call under stream capture cannot allocate)
  for (int i = 0; i < kSlots && e == cudaSuccess; ++i)
    if (slot_reserve(c, c->slots[i], kInitialSegCap) != KVR_OK) e = cudaErrorMemoryAllocation;
  cudaSetDevice(prev);
  if (e != cudaSuccess) {
    kvr_destroy(c);
    (void)cudaGetLastError();
    return KVR_ERR_CUDA;
  }
  *out = c;
  return KVR_OK;
}

kvr_status kvr_destroy(kvr_ctx* c) {
  if (!c) return KVR_OK;
  int prev = 0;
  cudaGetDevice(&prev);
  cudaSetDevice(c->device);
  cudaDeviceSynchronize();
  for (Slot& s : c->slots) {
    if (s.host) cudaFreeHost(s.host);
    if (s.dev) cudaFree(s.dev);
    if (s.tm_host) cudaFreeHost(s.tm_host);
    if (s.tm_dev) cudaFree(s.tm_dev);
    if (s.ev) cudaEventDestroy(s.ev);
  }
  for (int b = 0; b < kStageBufs; ++b) {
    if (c->stage[b]) cudaFree(c->stage[b]);
    if (c->stage_filled[b]) cudaEventDestroy(c->stage_filled[b]);
    if (c->stage_drained[b]) cudaEventDestroy(c->stage_drained[b]);
  }
  if (c->fork_ev) cudaEventDestroy(c->fork_ev);
  for (auto& a : c->attn_slots) {
    if (a.host) cudaFreeHost(a.host);
    if (a.dev) cudaFree(a.dev);
    if (a.ev) cudaEventDestroy(a.ev);
  }
  if (c->attn_part) cudaFree(c->attn_part);
  if (c->attn_tickets) cudaFree(c->attn_tickets);
  for (void* p : c->attn_retired) cudaFree(p);
  if (c->aux_dev) cudaFree(c->aux_dev);
  if (c->copy_stream) cudaStreamDestroy(c->copy_stream);
  if (c->d_inv_freq) cudaFree(c->d_inv_freq);
  if (c->d_status) cudaFree(c->d_status);
  if (c->d_sched) cudaFree(c->d_sched);
  if (c->h_status) cudaFreeHost(c->h_status);
  cudaSetDevice(prev);
  (void)cudaGetLastError();
  delete c;
  return KVR_OK;
}

kvr_status kvr_set_tuning(kvr_ctx* c, const kvr_tuning* t) {
  if (!c) return KVR_ERR_INVALID_ARG;
  if (t) c->tuning = *t; else c->tuning = kvr_tuning{};
  return KVR_OK;
}

kvr_status kvr_validate(const kvr_model_desc* model, const kvr_paged_dst* dst, const kvr_segment* segs,
                        int32_t n_segs) {
  return check_call(model, dst, segs, n_segs);
}

uint64_t kvr_bytes_moved(const kvr_model_desc* m, const kvr_segment* segs, int32_t n) {
  if (!m || (n > 0 && !segs)) return 0;
  uint64_t tokens = 0;
  for (int32_t i = 0; i < n; ++i) tokens += segs[i].len > 0 ? (uint64_t)segs[i].len : 0u;
  const uint64_t tensors = (n > 0 && segs[0].v_src == nullptr) ? 2ull : 4ull;   // K-only: read K, write K
  return tensors * (uint64_t)m->layers * (uint64_t)m->kv_heads * (uint64_t)m->head_dim *
         (uint64_t)elt_bytes(m->dtype) * tokens;
}

}  // extern "C"

// One launch over layers [l0, l0 + nl) of the model.  All segment pointers are DEVICE pointers.  The
// destination, its scales and the source scales are advanced to layer l0; the K/V sources are advanced too
// unless `src_group_local` (the host-source path stages exactly the group's layers at layer index 0).
static kvr_status enqueue_layers(kvr_ctx* c, const kvr_paged_dst* d, const kvr_segment* segs, int32_t n,
                                 cudaStream_t stream, int l0, int nl, bool src_group_local, bool inplace = false) {
  kvr_status st = KVR_OK;
  cudaStreamCaptureStatus cap = cudaStreamCaptureStatusNone;
  KVR_CUDA(c, cudaStreamIsCapturing(stream, &cap));
  const bool capturing = cap != cudaStreamCaptureStatusNone;

  // Descriptors.  Calls with <= kInlineSegs segments carry them in the kernel parameters: they are built in a
  // context-owned host scratch array, enqueue nothing but the kernel and may be captured in a CUDA graph.  Larger calls
  // stage them through a ring of pinned slots + one H2D copy; a captured copy node would read its pinned slot again at
  // every replay, long after later calls have overwritten it, so such calls are refused under capture (kvr.h).
  const bool inline_descs = n <= kInlineSegs;
  if (capturing && !inline_descs) {
    c->last_err = "more than 8 segments (spans) per call cannot be captured in a CUDA graph";
    return KVR_ERR_UNSUPPORTED;
  }
  Slot* slot_p = nullptr;
  if (!inline_descs) {
    slot_p = &c->slots[c->next_slot];
    c->next_slot = (c->next_slot + 1) % kSlots;
    if (slot_p->pending) {
      KVR_CUDA(c, cudaEventSynchronize(slot_p->ev));   // the call that used this slot kSlots calls ago
      slot_p->pending = false;
    }
    if ((size_t)n > slot_p->cap) {
      st = slot_reserve(c, *slot_p, (size_t)n);
      if (st != KVR_OK) return st;
    }
  }
  SegDev* const host_descs = inline_descs ? c->inline_scratch : slot_p->host;

  kvr_model_desc m = c->model;
  m.layers = nl;
  const int E = elt_bytes(m.dtype);
  CallParams P{};
  P.layers = m.layers; P.heads = m.kv_heads; P.head_dim = m.head_dim; P.rotary_dim = m.rotary_dim;
  P.rotary_offset = m.rotary_offset;
  P.no_v = (inplace || d->v_cache == nullptr) ? 1 : 0;
  P.pairing = m.pairing; P.dtype = m.dtype; P.inv_freq = c->d_inv_freq;
  P.k_cache = static_cast<uint8_t*>(d->k_cache) + (int64_t)l0 * d->stride_layer * E;
  P.v_cache = d->v_cache ? static_cast<uint8_t*>(d->v_cache) + (int64_t)l0 * d->stride_layer * E : nullptr;
  P.inplace = inplace ? 1 : 0;
  P.d_sl = d->stride_layer; P.d_sb = d->stride_block; P.d_st = d->stride_token; P.d_sh = d->stride_head;
  P.block_table = d->block_table;
  P.k_scale_dst = d->k_scale ? d->k_scale + (int64_t)l0 * m.kv_heads : nullptr;
  P.num_blocks = d->num_blocks; P.block_size = d->block_size; P.num_seqs = d->num_seqs;
  P.max_blocks = d->max_blocks_per_seq;
  P.segs = inline_descs ? nullptr : slot_p->dev; P.n_segs = n; P.status = c->d_status;
  P.sched = c->d_sched;

  bool any_map = false, scales_differ = false;
  for (int32_t i = 0; i < n; ++i) {
    any_map |= segs[i].pos_map != nullptr || (segs[i].flags & KVR_SEG_PRE_ROPE);   // per-token shifts
    scales_differ |= (m.dtype == KVR_FP8_E4M3 && segs[i].k_scale_src && segs[i].k_scale_src != d->k_scale);
  }
  P.any_pos_map = any_map; P.scales_differ = scales_differ;

  // ---- work decomposition: (segment, chunk of <= cg destination tokens, group of lpu layers) ----
  auto decompose = [&](int cg, int lpu_request, int hsplit_request, bool ring) {
    P.cg = cg;
    // head split (ring kernel only): must divide the number of head groups of a unit
    int hsplit = 1;
    if (hsplit_request > 1 && !any_map && !P.tmajor) {
      const int hgroups = m.kv_heads / ring_heads_per_tile(P);
      hsplit = hsplit_request > hgroups ? hgroups : hsplit_request;
      while (hsplit > 1 && hgroups % hsplit) --hsplit;
    }
    P.hsplit = hsplit;
    int64_t chunks_total = 0;
    for (int32_t i = 0; i < n; ++i) {
      const kvr_segment& s = segs[i];
      SegDev& o = host_descs[i];
      const int64_t src_adv = src_group_local ? 0 : (int64_t)l0 * s.src_stride_layer * E;
      o.k_src = static_cast<const uint8_t*>(s.k_src) + src_adv;
      o.v_src = s.v_src ? static_cast<const uint8_t*>(s.v_src) + src_adv : nullptr;
      o.pos_map = s.pos_map;
      o.k_scale_src = s.k_scale_src ? s.k_scale_src : d->k_scale;
      if (o.k_scale_src) o.k_scale_src += (int64_t)l0 * m.kv_heads;
      o.sl = s.src_stride_layer; o.sh = s.src_stride_head; o.st = s.src_stride_token;
      o.len = s.len; o.old_start = s.old_start; o.delta = (int32_t)((int64_t)s.new_start - s.old_start);
      o.dst_seq = s.dst_seq; o.dst_token_start = s.dst_token_start;
      o.first_q = s.dst_token_start / cg;
      o.n_chunks = (int32_t)(((int64_t)s.dst_token_start + s.len - 1) / cg - o.first_q + 1);
      o.index = i; o.pre_rope = (s.flags & KVR_SEG_PRE_ROPE) ? 1 : 0;
      o.src_stable = (!src_group_local && (s.flags & KVR_SEG_SRC_STABLE)) ? 1 : 0; o.pad_ = 0;
      chunks_total += o.n_chunks;
    }
    int lpu = lpu_request;
    if (lpu <= 0 && ring) {
      // Ring kernel: a unit should hold enough tiles to amortise its decode in the producer warp (~8 tiles = 64 KB)
      // and no more -- units are handed out in (layer, chunk) order, so with few layers per unit the CTAs that run
      // concurrently read neighbouring source rows of one layer (DRAM page locality: +3 % on configs[2] against
      // 11 layers per unit) and the tail is short.  With a position map the per-chunk angle table is rebuilt per
      // unit, so a unit holds ~24 tiles there.
      const int tiles_per_layer = P.tmajor ? (cg + P.ct - 1) / P.ct
                                           : ((m.kv_heads / ring_heads_per_tile(P)) / hsplit) * (P.gather == 2 ? 2 : 1);
      // (with pre-RoPE keys every token has its own shift, nothing deduplicates: ~96 tiles per unit.  One value per
      //  call: giving the constant-shift segments of such a call their own, smaller units measured slower.)
      bool any_pre = false;
      for (int32_t i = 0; i < n; ++i) any_pre |= (segs[i].flags & KVR_SEG_PRE_ROPE) != 0;
      const int want = (any_pre ? 96 : any_map ? 24 : 8) / (P.gather ? 4 : 1);   // gather tiles are 32 KB, ordinary ones 8 KB
      lpu = (want + tiles_per_layer - 1) / tiles_per_layer;
      if (lpu > m.layers) lpu = m.layers;
      // small calls: prefer more, smaller units so that every SM gets one (latency, not bandwidth, is the bound)
      while (lpu > 1 && chunks_total * ((m.layers + lpu - 1) / lpu) * hsplit < (int64_t)4 * c->sm_count) lpu = (lpu + 1) / 2;
    } else if (lpu <= 0) {
      if (any_map) lpu = m.layers;   // the per-token angle table is built once per chunk and reused by all layers
      else {
        int64_t target = (int64_t)c->sm_count * 32;
        int64_t v = (chunks_total * m.layers) / target;
        lpu = (int)(v < 1 ? 1 : (v > m.layers ? m.layers : v));
      }
    }
    if (lpu > m.layers) lpu = m.layers;
    P.lpu = lpu; P.n_lgroups = ((m.layers + lpu - 1) / lpu) * hsplit;
    int64_t at = 0;
    for (int32_t i = 0; i < n; ++i) {
      host_descs[i].unit_begin = at;
      at += (int64_t)host_descs[i].n_chunks * P.n_lgroups;
    }
    P.total_units = at;
  };

  const kvr_tuning& tu = c->tuning;
  int path = tu.path;
  const char* why = nullptr;
  TmapInline tmaps_inline;             // tensor maps of a call with inline descriptors (transposing loads)
  bool use_tmaps = false;
  for (int attempt = 0; attempt < 2 && (path == 0 || path == 2); ++attempt) {
    int cg_limit = (tu.chunk_tokens > 0 && tu.chunk_tokens < 16) ? tu.chunk_tokens : 16;
    P.tile_min_bytes = tu.tile_bytes;
    // TRANSPOSING loads (kvr_ring.cu, TmapPair): dense token-major (NHD) pool, several heads, power-of-two rows, not in
    // place: a tile = ALL heads x ct tokens, loaded by one TMA tensor operation per tensor so that it lands in shared
    // memory in the pool's own order; V then leaves as one contiguous bulk store and K as contiguous warp stores.
    // tuning.transpose_load: 0 auto, 1 on, 2 off.  Second attempt (the encoder refused a source): off.
    P.tmajor = 0; P.ct = 0; P.tmaps = nullptr;
    {
      const int64_t rowB = (int64_t)m.head_dim * E;
      const bool pow2_row = rowB >= 32 && rowB <= 1024 && (rowB & (rowB - 1)) == 0 && m.rotary_offset == 0;
      const bool dense_nhd = d->stride_head == m.head_dim && d->stride_token == (int64_t)m.kv_heads * m.head_dim;
      const bool want = tu.transpose_load == 1 || (tu.transpose_load == 0 && kTransposeAuto);
      if (attempt == 0 && want && !inplace && pow2_row && dense_nhd && m.kv_heads >= 2 && m.kv_heads <= 256 &&
          m.head_dim <= 256 && tu.hsplit <= 1 && (tu.gather == 0 || tu.gather == 2) && tmap_encoder()) {
        const int cg_full = chunk_granularity(d->block_size, cg_limit);
        const int64_t tokB = (int64_t)m.kv_heads * rowB;                         // one token, all heads, one tensor
        const int64_t target = tu.tile_bytes > 0 ? tu.tile_bytes : 4096;
        const int ct = chunk_granularity(cg_full, (int)(target / tokB > 1 ? target / tokB : 1));
        if (tokB * ct <= 32768) { P.tmajor = 1; P.ct = ct; }
      }
    }
    // GATHER mode (kvr_ring.cu): dense token-major (NHD) pool, several heads, power-of-two rows, not in place:
    // a tile = all heads x cg tokens with K (and V) <= 16 KB each, so that a token's H*D destination row is written
    // by one warp in one burst.  tuning.gather: 0 auto (on), 1 on, 2 off.
    P.gather = 0;
    if (!P.tmajor) {
      const int64_t rowB = (int64_t)m.head_dim * E;
      const bool pow2_row = rowB >= 32 && rowB <= 1024 && (rowB & (rowB - 1)) == 0 && m.rotary_offset == 0;
      const bool dense_nhd = d->stride_head == m.head_dim && d->stride_token == (int64_t)m.kv_heads * m.head_dim;
      // A gather stage is <= 32 KB: K and V of all heads of a full chunk together if they fit (mode 1), else K and V
      // in tiles of their own (mode 2, "split": a full chunk of ONE tensor), else a shorter chunk (mode 1).
      const int cg_full = chunk_granularity(d->block_size, 16);
      const int64_t chunk_bytes = (int64_t)m.kv_heads * cg_full * rowB;          // one tensor, all heads, a full chunk
      int mode = 1;
      int64_t tile_target = tu.tile_bytes > 0 ? tu.tile_bytes : 16384;             // K bytes of a gather tile
      // More than 16 KB per tensor (8 heads of 128 bf16): K and V in 16 KB tiles of their own, each holding HALF the
      // heads of a full chunk (a token then leaves as two contiguous 1 KB pieces), ring of 6, two stages per warp group
      // (kvr_ring.cu).  B200: configs[1] 6.15 -> 6.25, configs[2] 6.34 -> 6.47, Qwen3-VL image-KV 6.35 -> 6.48 TB/s.
      // Not with per-token shifts (measured: no gain) and not in fp8 (-15 %: 128-byte rows make poor bulk stores).
      bool split16 = false;
      if (tu.gather == 0 && tu.tile_bytes <= 0 && m.dtype == KVR_BF16 && !any_map && d->v_cache &&
          chunk_bytes > 16384 && 16384 % (cg_full * rowB) == 0) {
        const int hpt = (int)(16384 / (cg_full * rowB));
        if (hpt >= 2 && m.kv_heads % hpt == 0) { mode = 2; tile_target = chunk_bytes; split16 = true; }
      }
      if (tu.gather == 3) { mode = 2; if (tu.tile_bytes <= 0) tile_target = 32768; }
      int64_t lim = tile_target / (m.kv_heads * rowB);
      const int cg_g = chunk_granularity(d->block_size, (int)(lim > 16 ? 16 : lim));
      // auto: only where it was measured to pay (B200): bf16 and source runs that are not shortened.
      const bool pays = m.dtype == KVR_BF16 && cg_g == cg_full;
      if (tu.gather != 2 && (tu.gather == 1 || tu.gather == 3 || pays) && tu.chunk_tokens <= 0 &&
          (tu.tile_bytes <= 0 || tu.gather == 1 || tu.gather == 3) && tu.hsplit <= 1 && !inplace && pow2_row && dense_nhd &&
          m.kv_heads > 1 && m.kv_heads * rowB <= 8192 && cg_g >= 2) {
        P.gather = (mode == 2 && d->v_cache) ? 2 : 1;
        cg_limit = cg_g;
        P.tile_min_bytes = (int32_t)(m.kv_heads * cg_g * rowB);
        // forced, with a tile smaller than all heads of a full chunk: keep the full chunk and take a SUBSET of the heads
        // per tile (a token then leaves as heads/hpt contiguous pieces instead of one)
        if (tu.tile_bytes > 0 && tu.tile_bytes >= cg_full * rowB && tu.tile_bytes < chunk_bytes) {
          cg_limit = cg_full;
          P.tile_min_bytes = tu.tile_bytes;
        }
        if (split16) { cg_limit = cg_full; P.tile_min_bytes = 16384; }
      }
    }
    if (inplace && d->stride_token != m.head_dim) {
      // token-major pool, in place: a tile is cg tokens x ALL heads (one contiguous run); keep it near 8 KB
      cg_limit = (int)((tu.tile_bytes > 0 ? tu.tile_bytes : 8192) / ((int64_t)m.kv_heads * m.head_dim * E));
      cg_limit = cg_limit < 1 ? 1 : (cg_limit > 16 ? 16 : cg_limit);
    }
    if ((int64_t)m.head_dim * E > 1024) {
      // long rows (MLA [latent | k_pe] = 1152 B): keep a tile near 8-16 KB so the ring still holds >= 6 stages
      cg_limit = (int)(16384 / ((int64_t)m.head_dim * E));
      cg_limit = cg_limit < 1 ? 1 : (cg_limit > 16 ? 16 : cg_limit);
    }
    decompose(chunk_granularity(d->block_size, cg_limit), tu.layers_per_unit, tu.hsplit, true);
    const RingConfig rc0{tu.ctas_per_sm, tu.consumer_warps, tu.stages, tu.v_bulk_store, tu.max_ctas, tu.grab, tu.pdl, tu.warps_per_stage,
                         tu.lanes_over_heads, nullptr};
    bool ok = ring_supported(P, host_descs, rc0, c->sm_count, &why);
    if (ok && P.tmajor) {
      // one tensor map per source tensor; the token extent is the segment's length, so a box that runs past the last
      // row is zero-filled instead of reading past the source allocation
      TmapPair* maps = tmaps_inline.m;
      if (!inline_descs) {
        st = slot_reserve_tmaps(c, *slot_p, (size_t)n);
        if (st != KVR_OK) return st;
        maps = slot_p->tm_host;
      }
      bool enc_ok = true;
      for (int32_t i = 0; i < n && enc_ok; ++i) {
        const SegDev& o = host_descs[i];
        enc_ok = encode_source_map(&maps[i].k, o.k_src, m.dtype, m.head_dim, m.kv_heads, o.len, m.layers, o.sl, o.sh, o.st, P.ct);
        if (enc_ok && o.v_src && !P.no_v)
          enc_ok = encode_source_map(&maps[i].v, o.v_src, m.dtype, m.head_dim, m.kv_heads, o.len, m.layers, o.sl, o.sh, o.st, P.ct);
      }
      if (!enc_ok) continue;                 // plan again without transposing loads
      use_tmaps = true;
      if (!inline_descs) P.tmaps = slot_p->tm_dev;
    } else if (!ok && P.tmajor) {
      continue;                              // e.g. the layout does not fit: plan again without transposing loads
    }
    if (!ok && path == 2) { c->last_err = std::string("ring kernel unsupported: ") + (why ? why : ""); return KVR_ERR_UNSUPPORTED; }
    path = ok ? 2 : 1;
    break;
  }
  if (path == 1 && tu.path == 0 && window_inplace_supported(P)) {
    // in place on rows that carry position-free dims besides the rotary window (the MLA [latent | k_pe] row): the window
    // kernel touches the window alone.  Units of all layers x one chunk, halved while there are fewer than 4 per SM.
    P.tmajor = 0; P.ct = 0; P.tmaps = nullptr; P.gather = 0;
    const int cg = chunk_granularity(d->block_size, 16);
    int64_t chunks_total = 0;
    for (int32_t i = 0; i < n; ++i)
      chunks_total += ((int64_t)segs[i].dst_token_start + segs[i].len - 1) / cg - segs[i].dst_token_start / cg + 1;
    int lpu = tu.layers_per_unit > 0 ? tu.layers_per_unit : m.layers;
    if (tu.layers_per_unit <= 0)
      while (lpu > 1 && chunks_total * ((m.layers + lpu - 1) / lpu) < (int64_t)4 * c->sm_count) lpu = (lpu + 1) / 2;
    decompose(cg, lpu, 1, false);
    path = 4;
  }
  if (path == 1 || path == 5) {
    P.tmajor = 0; P.ct = 0; P.tmaps = nullptr; P.gather = 0;
    // generic kernels: chunk table [cg][R/2] float4 must fit 48 KB of static-limit shared memory
    int limit = (int)(47 * 1024 / ((m.rotary_dim / 2) * 16 + 4));
    if (limit < 1) return KVR_ERR_UNSUPPORTED;
    decompose(chunk_granularity(d->block_size, limit < 16 ? limit : 16), tu.layers_per_unit, 1, false);
    // Auto dispatch prefers the 16-byte-access form where the rotary window splits into whole vectors; tuning.path = 1
    // keeps the scalar kernel (the on-device cross-check), tuning.path = 5 insists on the vector one.
    const bool vec_ok = generic_vec_supported(P);
    if (path == 5 && !vec_ok) { c->last_err = "vectorised generic kernel: rotary_dim * esz must be a multiple of 32 (NeoX) or 16 (GPT-J) bytes"; return KVR_ERR_UNSUPPORTED; }
    if (path == 1 && tu.path == 0 && vec_ok) path = 5;
  }

  if (inline_descs) {
    for (int32_t i = 0; i < n; ++i) P.inline_segs[i] = host_descs[i];   // descriptors ride in the kernel parameters
  } else {
    KVR_CUDA(c, cudaMemcpyAsync(slot_p->dev, slot_p->host, (size_t)n * sizeof(SegDev), cudaMemcpyHostToDevice, stream));
    if (use_tmaps && path == 2)
      KVR_CUDA(c, cudaMemcpyAsync(slot_p->tm_dev, slot_p->tm_host, (size_t)n * sizeof(TmapPair), cudaMemcpyHostToDevice, stream));
  }
  cudaError_t e;
  if (path == 2) {
    RingConfig rc{tu.ctas_per_sm, tu.consumer_warps, tu.stages, tu.v_bulk_store, tu.max_ctas, tu.grab, tu.pdl, tu.warps_per_stage,
                  tu.lanes_over_heads, (use_tmaps && inline_descs) ? &tmaps_inline : nullptr};
    e = launch_ring(P, rc, c->sm_count, stream, &c->last_grid, &c->last_block, &c->last_smem);
  } else if (path == 4) {
    e = launch_window_inplace(P, c->sm_count, stream, &c->last_grid, &c->last_block, &c->last_smem);
  } else if (path == 5) {
    e = launch_generic_vec(P, c->sm_count, stream, &c->last_grid, &c->last_block, &c->last_smem);
  } else {
    e = launch_generic(P, c->sm_count, stream, &c->last_grid, &c->last_block, &c->last_smem);
  }
  if (e != cudaSuccess) return c->cuda_fail(e, path == 2 ? "launch_ring" : path == 4 ? "launch_window_inplace" : path == 5 ? "launch_generic_vec" : "launch_generic");
  c->launches += 1;
  c->last_path = path;
  c->last_stream = stream;
  if (slot_p) {
    KVR_CUDA(c, cudaEventRecord(slot_p->ev, stream));   // the slot may be rewritten once its copy and kernel have run
    slot_p->pending = true;
  }
  return KVR_OK;
}

static kvr_status check_deltas(const kvr_segment* segs, int32_t n) {
  for (int32_t i = 0; i < n; ++i) {
    int64_t delta = (int64_t)segs[i].new_start - (int64_t)segs[i].old_start;
    if (!segs[i].pos_map && (delta > INT32_MAX || delta < INT32_MIN)) return KVR_ERR_INVALID_ARG;
  }
  return KVR_OK;
}

struct DeviceGuard {
  int prev = 0, cur = 0;
  explicit DeviceGuard(int dev) : cur(dev) { cudaGetDevice(&prev); if (prev != cur) cudaSetDevice(cur); }
  ~DeviceGuard() { if (prev != cur) cudaSetDevice(prev); }
};

// ---- NEXT-4, first alternative: rotate-on-read decode attention (kvr.h; R25) ----
namespace {

// Tensor map of one source tensor [layers][heads][len][128] bf16 with dims ordered (dim, token, head, layer): a box of
// {64 dims, 128 tokens} lands as 128 rows of 128 bytes, 128-byte swizzled -- the tcgen05 shared-memory operand layout.
bool encode_attn_map(CUtensorMap* out, const void* base, int heads, int len, int layers, int64_t sl, int64_t sh, int64_t st) {
  TmapEncodeFn enc = tmap_encoder();
  if (!enc || !base) return false;
  uint64_t s_t = (uint64_t)st * 2, s_h = (uint64_t)sh * 2, s_l = (uint64_t)sl * 2;
  if (len == 1 && s_t == 0) s_t = 256;          // a dimension of extent 1 never uses its stride: give it a legal one
  if (heads == 1 && s_h == 0) s_h = 256;
  if (layers == 1 && s_l == 0) s_l = 256;
  if (s_t == 0 || s_h == 0 || s_l == 0) return false;
  const cuuint64_t dims[4] = {128u, (cuuint64_t)len, (cuuint64_t)heads, (cuuint64_t)layers};
  const cuuint64_t strides[3] = {s_t, s_h, s_l};
  const cuuint32_t box[4] = {64u, 128u, 1u, 1u};
  const cuuint32_t es[4] = {1u, 1u, 1u, 1u};
  return enc(out, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 4, const_cast<void*>(base), dims, strides, box, es,
             CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
             CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

}  // namespace

extern "C" {

uint64_t kvr_attention_bytes_read(const kvr_model_desc* m, const kvr_read_segment* segs, int32_t n) {
  if (!m || (n > 0 && !segs)) return 0;
  uint64_t tokens = 0;
  for (int32_t i = 0; i < n; ++i) tokens += segs[i].len > 0 ? (uint64_t)segs[i].len : 0u;
  return 2ull * (uint64_t)m->kv_heads * (uint64_t)m->head_dim * (uint64_t)elt_bytes(m->dtype) * tokens;
}

// Host-only validation of a rotate-on-read call (no CUDA call is made): the status the call itself returns before it
// enqueues anything.
kvr_status kvr_validate_read(const kvr_model_desc* mp, const void* q, int32_t n_req, int32_t q_heads, int32_t layer,
                             float softmax_scale, const kvr_read_segment* segs, int32_t n, const float* o, const float* lse) {
  kvr_status st = check_model(mp);
  if (st != KVR_OK) return st;
  const kvr_model_desc& m = *mp;
  if (!q || !o || !lse || !segs || n <= 0 || n_req <= 0 || q_heads <= 0 || layer < 0 || layer >= m.layers) return KVR_ERR_INVALID_ARG;
  if (q_heads % m.kv_heads != 0 || !(softmax_scale > 0.0f) || !std::isfinite(softmax_scale)) return KVR_ERR_INVALID_ARG;
  if (!aligned16(q) || !aligned16(o) || (reinterpret_cast<uintptr_t>(lse) & 3u)) return KVR_ERR_ALIGNMENT;
  if (m.dtype != KVR_BF16 || m.head_dim != 128 || q_heads / m.kv_heads > 16) return KVR_ERR_UNSUPPORTED;
  if (n_req > n) return KVR_ERR_INVALID_ARG;      // every request must own a segment (also bounds the vector below)
  std::vector<int32_t> per_req;
  try { per_req.assign((size_t)n_req, 0); } catch (const std::bad_alloc&) { return KVR_ERR_NOMEM; }
  for (int32_t i = 0; i < n; ++i) {
    const kvr_read_segment& s = segs[i];
    if (!s.k_src || !s.v_src || s.len <= 0 || s.request < 0 || s.request >= n_req || (s.flags & ~KVR_SEG_SRC_STABLE)) return KVR_ERR_INVALID_ARG;
    if ((s.src_stride_token < m.head_dim && s.len > 1) || s.src_stride_layer < 0 || s.src_stride_head < 0) return KVR_ERR_INVALID_ARG;
    if ((s.src_stride_head < m.head_dim && m.kv_heads > 1)) return KVR_ERR_INVALID_ARG;
    if (!aligned16(s.k_src) || !aligned16(s.v_src)) return KVR_ERR_ALIGNMENT;
    if ((s.src_stride_layer * 2) % 16 || (s.src_stride_head * 2) % 16 || (s.src_stride_token * 2) % 16) return KVR_ERR_ALIGNMENT;
    // what a TMA tensor map can describe (encode_attn_map): a dimension of extent > 1 needs a non-zero stride, strides
    // stay below 2^40 bytes
    if ((s.src_stride_layer == 0 && m.layers > 1) || (s.src_stride_head == 0 && m.kv_heads > 1)) return KVR_ERR_UNSUPPORTED;
    const int64_t lim = (int64_t)1 << 39;           // elements of 2 bytes
    if (s.src_stride_layer >= lim || s.src_stride_head >= lim || s.src_stride_token >= lim) return KVR_ERR_UNSUPPORTED;
    per_req[(size_t)s.request] += 1;
  }
  for (int32_t r = 0; r < n_req; ++r)
    if (per_req[(size_t)r] == 0) return KVR_ERR_INVALID_ARG;      // every request must own at least one segment
  return KVR_OK;
}

static kvr_status attend_call(kvr_ctx* c, const void* q, int32_t n_req, int32_t q_heads, int32_t layer,
                              float softmax_scale, const kvr_read_segment* segs, int32_t n, float* o, float* lse,
                              void* cuda_stream);

// The C ABI never throws: the host-side decomposition builds std::vectors sized by the caller's numbers.
kvr_status kvr_rotate_on_read_attention(kvr_ctx* c, const void* q, int32_t n_req, int32_t q_heads, int32_t layer,
                                        float softmax_scale, const kvr_read_segment* segs, int32_t n, float* o, float* lse,
                                        void* cuda_stream) {
  try {
    return attend_call(c, q, n_req, q_heads, layer, softmax_scale, segs, n, o, lse, cuda_stream);
  } catch (const std::bad_alloc&) {
    if (c) c->last_err = "rotate-on-read attention: out of host memory while building the work items";
    return KVR_ERR_NOMEM;
  }
}

static kvr_status attend_call(kvr_ctx* c, const void* q, int32_t n_req, int32_t q_heads, int32_t layer,
                              float softmax_scale, const kvr_read_segment* segs, int32_t n, float* o, float* lse,
                              void* cuda_stream) {
  if (!c) return KVR_ERR_INVALID_ARG;
  c->last_err.clear();
  const kvr_model_desc& m = c->model;
  const kvr_status vst = kvr_validate_read(&m, q, n_req, q_heads, layer, softmax_scale, segs, n, o, lse);
  if (vst != KVR_OK) {
    if (vst == KVR_ERR_UNSUPPORTED) c->last_err = "rotate-on-read attention: bf16 caches, head_dim 128 and q_heads / kv_heads <= 16 only";
    return vst;
  }
  const int group = q_heads / m.kv_heads;
  if (!tmap_encoder()) { c->last_err = "cuTensorMapEncodeTiled is not available"; return KVR_ERR_UNSUPPORTED; }
  DeviceGuard guard(c->device);
  cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
  cudaStreamCaptureStatus cap = cudaStreamCaptureStatusNone;
  KVR_CUDA(c, cudaStreamIsCapturing(stream, &cap));
  const bool capturing = cap != cudaStreamCaptureStatusNone;

  // ---- descriptors: cached per distinct segment array ----
  const size_t key_bytes = (size_t)n * sizeof(kvr_read_segment);
  kvr_ctx::AttnSlot* slot_p = nullptr;
  for (auto& a : c->attn_slots)
    if (a.key.size() == key_bytes && a.n_req == n_req && a.q_heads == q_heads && a.tpi_tuning == c->tuning.layers_per_unit + 1000 * c->tuning.hsplit &&
        std::memcmp(a.key.data(), segs, key_bytes) == 0) { slot_p = &a; break; }
  const bool hit = slot_p != nullptr;
  if (!hit) {
    // CUDA graphs: a call whose descriptors are cached enqueues nothing but kernels and may be captured; its cache
    // entry is then PINNED (never evicted: every replay reads it).  A call that would have to build and copy its
    // descriptors is refused under capture -- issue it once eagerly first.
    if (capturing) {
      c->last_err = "rotate-on-read attention: descriptors of this segment array are not cached yet; issue the call once outside the capture";
      return KVR_ERR_UNSUPPORTED;
    }
    for (auto& a : c->attn_slots)
      if (!a.pinned && (!slot_p || a.last_use < slot_p->last_use)) slot_p = &a;      // least recently used, not pinned
    if (!slot_p) { c->last_err = "rotate-on-read attention: every descriptor cache entry is pinned by a captured graph"; return KVR_ERR_NOMEM; }
  }
  kvr_ctx::AttnSlot& slot = *slot_p;
  slot.last_use = ++c->attn_clock;
  if (!slot.ev) KVR_CUDA(c, cudaEventCreateWithFlags(&slot.ev, cudaEventDisableTiming));
  if (!hit) {
    if (slot.pending) { KVR_CUDA(c, cudaEventSynchronize(slot.ev)); slot.pending = false; }
    slot.key.clear();
    // ---- work decomposition: items = (segment, kv head, run of key tiles); groups = (request, kv head) ----
    std::vector<int32_t> order((size_t)n);
    for (int32_t i = 0; i < n; ++i) order[(size_t)i] = i;
    std::stable_sort(order.begin(), order.end(), [&](int32_t a, int32_t b) { return segs[a].request < segs[b].request; });
    int64_t total_tiles = 0;
    for (int32_t i = 0; i < n; ++i) total_tiles += ((int64_t)segs[i].len + 127) / 128;
    total_tiles *= m.kv_heads;
    // ~8 items per SM when the call is large enough (items are handed out dynamically: the tail is at most one item);
    // 4..8 tiles (512..1024 keys) per item -- B200: 8 beats 16 by 1-4 % on the serving and 32k workloads, 4 beats 8 on
    // the small compose call; tuning.layers_per_unit doubles as "tiles per item" for experiments (this call has no
    // layers to group)
    int64_t tpi = (total_tiles + 8ll * c->sm_count - 1) / (8ll * c->sm_count);
    tpi = tpi < 4 ? 4 : (tpi > 8 ? 8 : tpi);
    if (c->tuning.layers_per_unit > 0) tpi = c->tuning.layers_per_unit;
    std::vector<AttnItem> items;
    std::vector<AttnMerge> merges;
    items.reserve((size_t)(total_tiles / tpi + (int64_t)n * m.kv_heads));
    int32_t n_groups = 0;
    for (size_t a = 0; a < order.size();) {
      size_t b = a;
      while (b < order.size() && segs[order[b]].request == segs[order[a]].request) ++b;
      for (int32_t h = 0; h < m.kv_heads; ++h) {
        const int32_t first = (int32_t)items.size();
        for (size_t j = a; j < b; ++j) {
          const int32_t si = order[j], len = segs[si].len;
          for (int32_t k0 = 0; k0 < len; k0 += (int32_t)tpi * 128) {
            AttnItem it{};
            it.seg = si; it.head = h; it.key0 = k0; it.n_keys = std::min<int32_t>((int32_t)tpi * 128, len - k0);
            it.group = n_groups; it.group_first = first; it.index = (int32_t)items.size();
            items.push_back(it);
          }
        }
        const int32_t cnt = (int32_t)items.size() - first;
        const bool defer = cnt > (c->tuning.hsplit > 0 ? c->tuning.hsplit : attend_inline_merge_limit(group));   // merged after the grid (tuning.hsplit overrides the limit)
        for (int32_t j = first; j < first + cnt; ++j) items[(size_t)j].group_count = defer ? -cnt : cnt;
        if (defer) merges.push_back(AttnMerge{first, cnt, segs[order[a]].request * q_heads + h * group, 0});
        ++n_groups;
      }
      a = b;
    }
    // ---- staging: [AttnSeg x n][AttnItem x n_items] through the slot's pinned buffer and one H2D copy ----
    const size_t seg_bytes = (size_t)n * sizeof(AttnSeg), item_bytes = items.size() * sizeof(AttnItem),
                 bytes = seg_bytes + item_bytes + merges.size() * sizeof(AttnMerge);
    if (bytes > slot.cap) {
      size_t cap = slot.cap ? slot.cap : (size_t)1 << 16;
      while (cap < bytes) cap *= 2;
      if (slot.host) cudaFreeHost(slot.host);
      if (slot.dev) cudaFree(slot.dev);
      slot.host = nullptr; slot.dev = nullptr; slot.cap = 0;
      KVR_CUDA(c, cudaMallocHost(&slot.host, cap));
      KVR_CUDA(c, cudaMalloc(&slot.dev, cap));
      slot.cap = cap;
    }
    AttnSeg* hs = reinterpret_cast<AttnSeg*>(slot.host);
    for (int32_t i = 0; i < n; ++i) {
      const kvr_read_segment& sg = segs[i];
      if (!encode_attn_map(&hs[i].k, sg.k_src, m.kv_heads, sg.len, m.layers, sg.src_stride_layer, sg.src_stride_head, sg.src_stride_token) ||
          !encode_attn_map(&hs[i].v, sg.v_src, m.kv_heads, sg.len, m.layers, sg.src_stride_layer, sg.src_stride_head, sg.src_stride_token)) {
        c->last_err = "rotate-on-read attention: a source tensor cannot be described by a TMA tensor map";
        return KVR_ERR_UNSUPPORTED;
      }
      hs[i].delta = sg.delta; hs[i].len = sg.len; hs[i].request = sg.request; hs[i].pad_ = 0;
    }
    std::memcpy(slot.host + seg_bytes, items.data(), item_bytes);
    if (!merges.empty()) std::memcpy(slot.host + seg_bytes + item_bytes, merges.data(), merges.size() * sizeof(AttnMerge));
    KVR_CUDA(c, cudaMemcpyAsync(slot.dev, slot.host, bytes, cudaMemcpyHostToDevice, stream));
    slot.n_items = items.size(); slot.seg_bytes = seg_bytes; slot.n_groups = n_groups; slot.n_merges = merges.size();
    slot.merge_max = 0;
    for (const AttnMerge& mg : merges) slot.merge_max = std::max(slot.merge_max, mg.count);
    slot.n_req = n_req; slot.q_heads = q_heads; slot.tpi_tuning = c->tuning.layers_per_unit + 1000 * c->tuning.hsplit;
    slot.key.assign(reinterpret_cast<const unsigned char*>(segs), reinterpret_cast<const unsigned char*>(segs) + key_bytes);
  }
  if (hit && slot.pending && stream != slot.last_stream) {
    // The descriptors were copied in on another stream: order this stream behind that copy.  Under capture an event
    // recorded outside the capture cannot be waited on, so the caller must have synchronised that stream (kvr.h).
    if (!capturing) KVR_CUDA(c, cudaStreamWaitEvent(stream, slot.ev, 0));
  }
  const size_t n_items = slot.n_items, seg_bytes = slot.seg_bytes;
  const int32_t n_groups = slot.n_groups;
  // partial results and tickets (grown on demand; a regrowth waits for the launches that may still use the old buffers)
  const size_t part_bytes = n_items * (size_t)group * (128 + 2) * sizeof(float);
  if (part_bytes > c->attn_part_cap || (size_t)n_groups > c->attn_ticket_cap) {
    if (capturing) { c->last_err = "rotate-on-read attention: partial buffers must grow; issue the call once outside the capture"; return KVR_ERR_UNSUPPORTED; }
    KVR_CUDA(c, cudaDeviceSynchronize());
    bool any_pinned = false;
    for (auto& a : c->attn_slots) any_pinned |= a.pinned;
    if (any_pinned) {           // a captured graph still points at the old buffers: keep them until kvr_destroy
      if (part_bytes > c->attn_part_cap && c->attn_part) { c->attn_retired.push_back(c->attn_part); c->attn_part = nullptr; }
      if ((size_t)n_groups > c->attn_ticket_cap && c->attn_tickets) { c->attn_retired.push_back(c->attn_tickets); c->attn_tickets = nullptr; }
    }
    if (part_bytes > c->attn_part_cap) {
      if (c->attn_part) cudaFree(c->attn_part);
      c->attn_part = nullptr; c->attn_part_cap = 0;
      size_t cap = std::max<size_t>(part_bytes * 2, (size_t)1 << 20);
      KVR_CUDA(c, cudaMalloc(&c->attn_part, cap));
      c->attn_part_cap = cap;
    }
    if ((size_t)n_groups > c->attn_ticket_cap) {
      if (c->attn_tickets) cudaFree(c->attn_tickets);
      c->attn_tickets = nullptr; c->attn_ticket_cap = 0;
      size_t cap = std::max<size_t>((size_t)n_groups * 2, 1024);
      KVR_CUDA(c, cudaMalloc(&c->attn_tickets, cap * sizeof(unsigned int)));
      KVR_CUDA(c, cudaMemset(c->attn_tickets, 0, cap * sizeof(unsigned int)));
      c->attn_ticket_cap = cap;
    }
  }

  AttnParams P{};
  P.q = static_cast<const uint16_t*>(q); P.o = o; P.lse = lse;
  P.segs = reinterpret_cast<const AttnSeg*>(slot.dev);
  P.items = reinterpret_cast<const AttnItem*>(slot.dev + seg_bytes);
  P.n_items = (int32_t)n_items;
  P.merges = reinterpret_cast<const AttnMerge*>(slot.dev + seg_bytes + n_items * sizeof(AttnItem));
  P.n_merges = (int32_t)slot.n_merges;
  P.merge_max_count = slot.merge_max;
  P.early = 1;
  for (int32_t i = 0; i < n; ++i) if (!(segs[i].flags & KVR_SEG_SRC_STABLE)) P.early = 0;
  P.q_heads = q_heads; P.group = group; P.layer = layer;
  P.rotary_dim = m.rotary_dim; P.rotary_offset = m.rotary_offset; P.pairing = m.pairing;
  P.scale_log2 = (float)((double)softmax_scale * 1.4426950408889634);
  P.inv_freq = c->d_inv_freq;
  P.part_o = c->attn_part;
  P.part_ml = c->attn_part + n_items * (size_t)group * 128;
  P.tickets = c->attn_tickets;
  P.sched = c->d_sched + 2;
  cudaError_t e = launch_attend(P, c->tuning.max_ctas > 0 ? std::min(c->tuning.max_ctas, c->sm_count) : c->sm_count, stream,
                                &c->last_grid, &c->last_block, &c->last_smem);
  if (e != cudaSuccess) return c->cuda_fail(e, "launch_attend");
  c->launches += 1 + (slot.n_merges ? 1 : 0);
  c->last_path = 3;
  c->last_stream = stream;
  if (capturing) {
    slot.pinned = true;
  } else if (!slot.pinned) {
    KVR_CUDA(c, cudaEventRecord(slot.ev, stream));      // the entry may be replaced once this launch has run
    slot.pending = true;
    slot.last_stream = stream;
  }
  return KVR_OK;
}

}  // extern "C"

extern "C" {

kvr_status kvr_reposition_splice(kvr_ctx* c, const kvr_paged_dst* d, const kvr_segment* segs, int32_t n,
                                 void* cuda_stream) {
  if (!c) return KVR_ERR_INVALID_ARG;
  c->last_err.clear();
  kvr_status st = check_call(&c->model, d, segs, n);
  if (st != KVR_OK) return st;
  if (n == 0) return KVR_OK;
  if ((st = check_deltas(segs, n)) != KVR_OK) return st;
  DeviceGuard guard(c->device);
  return enqueue_layers(c, d, segs, n, static_cast<cudaStream_t>(cuda_stream), 0, c->model.layers, false);
}

// Host-resident sources (a skill library kept in host RAM): stage layer groups through two context-owned device
// buffers; the H2D copies of group g+1 run on the context's copy stream while the kernel of group g runs on the
// caller's stream.  No arithmetic happens on the host: the staged bytes go through the same kernels.
kvr_status kvr_reposition_splice_host(kvr_ctx* c, const kvr_paged_dst* d, const kvr_segment* segs, int32_t n,
                                      void* cuda_stream) {
  if (!c) return KVR_ERR_INVALID_ARG;
  c->last_err.clear();
  c->h2d_bytes = 0;
  const kvr_model_desc& m = c->model;
  const int E = elt_bytes(m.dtype);
  // validate with stand-in device addresses for the host pointers (alignment rules are the same)
  kvr_status st = check_call(&m, d, segs, n);
  if (st != KVR_OK) return st;
  if (n == 0) return KVR_OK;
  if ((st = check_deltas(segs, n)) != KVR_OK) return st;
  int64_t tokens = 0;
  size_t aux_need = 0;
  for (int32_t i = 0; i < n; ++i) {
    const kvr_segment& s = segs[i];
    // host sources must be dense [layers][kv_heads][len][head_dim] so that a layer group is one contiguous run
    if (s.src_stride_token != m.head_dim || s.src_stride_head != (int64_t)s.len * m.head_dim ||
        s.src_stride_layer != (int64_t)m.kv_heads * s.len * m.head_dim)
      return KVR_ERR_UNSUPPORTED;
    tokens += s.len;
    if (s.pos_map) aux_need += (((size_t)s.len * 4) + 15) & ~(size_t)15;
    if (s.k_scale_src) aux_need += (((size_t)m.layers * m.kv_heads * 4) + 15) & ~(size_t)15;
  }
  cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
  DeviceGuard guard(c->device);
  cudaStreamCaptureStatus cap = cudaStreamCaptureStatusNone;
  KVR_CUDA(c, cudaStreamIsCapturing(stream, &cap));
  if (cap != cudaStreamCaptureStatusNone) return KVR_ERR_UNSUPPORTED;   // allocates and uses a second stream

  // ---- layer-group size: staging buffer of <= ~256 MB, at least one layer ----
  const bool k_only = (d->v_cache == nullptr);
  const size_t layer_bytes = (k_only ? 1u : 2u) * (size_t)tokens * m.kv_heads * m.head_dim * E;   // K (+ V) of one layer, all segments
  int lg = (int)((256ull << 20) / (layer_bytes ? layer_bytes : 1));
  if (lg < 1) lg = 1;
  if (lg > m.layers) lg = m.layers;
  if (m.layers >= 4 && lg > m.layers / 4) lg = m.layers / 4;                        // keep >= 4 groups so copy and kernel overlap
  const size_t need = (size_t)lg * layer_bytes;
  if (need > c->stage_cap) {
    KVR_CUDA(c, cudaDeviceSynchronize());
    for (int b = 0; b < kStageBufs; ++b) { if (c->stage[b]) cudaFree(c->stage[b]); c->stage[b] = nullptr; }
    c->stage_cap = 0;
    for (int b = 0; b < kStageBufs; ++b) KVR_CUDA(c, cudaMalloc(&c->stage[b], need));
    c->stage_cap = need;
    c->stage_drained_valid[0] = c->stage_drained_valid[1] = false;
  }
  if (aux_need > c->aux_cap) {
    KVR_CUDA(c, cudaDeviceSynchronize());
    if (c->aux_dev) cudaFree(c->aux_dev);
    c->aux_dev = nullptr; c->aux_cap = 0;
    KVR_CUDA(c, cudaMalloc(&c->aux_dev, aux_need));
    c->aux_cap = aux_need;
  }
  if (!c->copy_stream) {
    KVR_CUDA(c, cudaStreamCreateWithFlags(&c->copy_stream, cudaStreamNonBlocking));
    for (int b = 0; b < kStageBufs; ++b) {
      KVR_CUDA(c, cudaEventCreateWithFlags(&c->stage_filled[b], cudaEventDisableTiming));
      KVR_CUDA(c, cudaEventCreateWithFlags(&c->stage_drained[b], cudaEventDisableTiming));
    }
    KVR_CUDA(c, cudaEventCreateWithFlags(&c->fork_ev, cudaEventDisableTiming));
  }
  // the copy stream starts after everything already enqueued on the caller's stream
  KVR_CUDA(c, cudaEventRecord(c->fork_ev, stream));
  KVR_CUDA(c, cudaStreamWaitEvent(c->copy_stream, c->fork_ev, 0));

  // ---- per-token maps and source scales: small, copied once ----
  std::vector<kvr_segment> dsegs(segs, segs + n);
  {
    uint8_t* at = static_cast<uint8_t*>(c->aux_dev);
    for (int32_t i = 0; i < n; ++i) {
      if (segs[i].pos_map) {
        const size_t b = (size_t)segs[i].len * 4;
        KVR_CUDA(c, cudaMemcpyAsync(at, segs[i].pos_map, b, cudaMemcpyHostToDevice, c->copy_stream));
        dsegs[i].pos_map = reinterpret_cast<const int32_t*>(at);
        at += (b + 15) & ~(size_t)15; c->h2d_bytes += b;
      }
      if (segs[i].k_scale_src) {
        const size_t b = (size_t)m.layers * m.kv_heads * 4;
        KVR_CUDA(c, cudaMemcpyAsync(at, segs[i].k_scale_src, b, cudaMemcpyHostToDevice, c->copy_stream));
        dsegs[i].k_scale_src = reinterpret_cast<const float*>(at);
        at += (b + 15) & ~(size_t)15; c->h2d_bytes += b;
      }
    }
  }
  int g = 0;
  for (int l0 = 0; l0 < m.layers; l0 += lg, ++g) {
    const int nl = (m.layers - l0 < lg) ? (m.layers - l0) : lg;
    const int b = g % kStageBufs;
    if (c->stage_drained_valid[b]) KVR_CUDA(c, cudaStreamWaitEvent(c->copy_stream, c->stage_drained[b], 0));
    uint8_t* at = c->stage[b];
    for (int32_t i = 0; i < n; ++i) {
      const kvr_segment& s = segs[i];
      const size_t run = (size_t)nl * s.src_stride_layer * E;
      const size_t off = (size_t)l0 * s.src_stride_layer * E;
      KVR_CUDA(c, cudaMemcpyAsync(at, static_cast<const uint8_t*>(s.k_src) + off, run, cudaMemcpyHostToDevice, c->copy_stream));
      dsegs[i].k_src = at; at += run;
      c->h2d_bytes += run;
      if (k_only) continue;
      KVR_CUDA(c, cudaMemcpyAsync(at, static_cast<const uint8_t*>(s.v_src) + off, run, cudaMemcpyHostToDevice, c->copy_stream));
      dsegs[i].v_src = at; at += run;
      c->h2d_bytes += run;
    }
    KVR_CUDA(c, cudaEventRecord(c->stage_filled[b], c->copy_stream));
    KVR_CUDA(c, cudaStreamWaitEvent(stream, c->stage_filled[b], 0));
    st = enqueue_layers(c, d, dsegs.data(), n, stream, l0, nl, true);
    if (st != KVR_OK) return st;
    KVR_CUDA(c, cudaEventRecord(c->stage_drained[b], stream));
    c->stage_drained_valid[b] = true;
  }
  return KVR_OK;
}

uint64_t kvr_last_h2d_bytes(const kvr_ctx* c) { return c ? c->h2d_bytes : 0; }

// ---- NEXT-1: in-place reposition of resident spans (R20) ----
static kvr_status check_inplace(const kvr_model_desc* m, const kvr_paged_dst* d, const kvr_resident_span* sp, int32_t n) {
  kvr_status st = check_model(m);
  if (st != KVR_OK) return st;
  if (!d || n < 0 || (n > 0 && !sp)) return KVR_ERR_INVALID_ARG;
  if (!d->k_cache || !d->block_table) return KVR_ERR_INVALID_ARG;
  if (d->num_blocks <= 0 || d->block_size <= 0 || d->num_seqs <= 0 || d->max_blocks_per_seq <= 0)
    return KVR_ERR_INVALID_ARG;
  if (d->stride_layer < 0 || d->stride_block <= 0 || (d->stride_token < m->head_dim && d->block_size > 1))
    return KVR_ERR_INVALID_ARG;
  if (d->stride_head < m->head_dim && m->kv_heads > 1) return KVR_ERR_INVALID_ARG;
  if (m->dtype == KVR_FP8_E4M3 && !d->k_scale) return KVR_ERR_INVALID_ARG;
  const int E = elt_bytes(m->dtype);
  if (!aligned16(d->k_cache)) return KVR_ERR_ALIGNMENT;
  const int64_t ds[4] = {d->stride_layer, d->stride_block, d->stride_token, d->stride_head};
  for (int64_t s : ds)
    if ((s * E) % 16 != 0) return KVR_ERR_ALIGNMENT;
  const int64_t cap = (int64_t)d->max_blocks_per_seq * d->block_size;
  for (int32_t i = 0; i < n; ++i) {
    const kvr_resident_span& s = sp[i];
    if (s.len <= 0 || s.seq < 0 || s.seq >= d->num_seqs || s.token_start < 0) return KVR_ERR_INVALID_ARG;
    if (s.old_start < 0 || (!s.pos_map && s.new_start < 0)) return KVR_ERR_INVALID_ARG;
    if ((int64_t)s.token_start + s.len > cap) return KVR_ERR_OUT_OF_RANGE;
    if (s.pos_map && (reinterpret_cast<uintptr_t>(s.pos_map) & 3u)) return KVR_ERR_ALIGNMENT;
  }
  return KVR_OK;
}

kvr_status kvr_reposition_inplace(kvr_ctx* c, const kvr_paged_dst* pool, const kvr_resident_span* spans, int32_t n,
                                  void* cuda_stream) {
  if (!c) return KVR_ERR_INVALID_ARG;
  c->last_err.clear();
  kvr_status st = check_inplace(&c->model, pool, spans, n);
  if (st != KVR_OK) return st;
  if (n == 0) return KVR_OK;
  std::vector<kvr_segment> segs((size_t)n);
  for (int32_t i = 0; i < n; ++i) {
    kvr_segment& g = segs[(size_t)i];
    g = kvr_segment{};
    g.k_src = pool->k_cache; g.v_src = pool->k_cache;      // placeholders: the kernels read the pool slot itself
    g.src_stride_layer = g.src_stride_head = 0; g.src_stride_token = c->model.head_dim;
    g.len = spans[i].len; g.old_start = spans[i].old_start; g.new_start = spans[i].new_start;
    g.dst_seq = spans[i].seq; g.dst_token_start = spans[i].token_start;
    g.pos_map = spans[i].pos_map; g.k_scale_src = nullptr;
  }
  if ((st = check_deltas(segs.data(), n)) != KVR_OK) return st;
  DeviceGuard guard(c->device);
  return enqueue_layers(c, pool, segs.data(), n, static_cast<cudaStream_t>(cuda_stream), 0, c->model.layers, false, true);
}

uint64_t kvr_inplace_bytes_moved(const kvr_model_desc* m, const kvr_resident_span* spans, int32_t n) {
  if (!m || (n > 0 && !spans)) return 0;
  uint64_t tokens = 0;
  for (int32_t i = 0; i < n; ++i) tokens += spans[i].len > 0 ? (uint64_t)spans[i].len : 0u;
  // a [latent | k_pe] row (rotary_offset != 0): only the k_pe window is read and written, the latent stays put
  const uint64_t width = m->rotary_offset != 0 ? (uint64_t)m->rotary_dim : (uint64_t)m->head_dim;
  return 2ull * (uint64_t)m->layers * (uint64_t)m->kv_heads * width * (uint64_t)elt_bytes(m->dtype) * tokens;
}

// ---- NEXT-2: span overwrite = the delta == 0 splice (R21) ----
kvr_status kvr_write_span(kvr_ctx* c, const kvr_paged_dst* dst, const kvr_span* spans, int32_t n, void* cuda_stream) {
  if (!c) return KVR_ERR_INVALID_ARG;
  c->last_err.clear();
  if (n < 0 || (n > 0 && !spans)) return KVR_ERR_INVALID_ARG;
  std::vector<kvr_segment> segs((size_t)n);
  for (int32_t i = 0; i < n; ++i) {
    kvr_segment& g = segs[(size_t)i];
    g = kvr_segment{};
    g.k_src = spans[i].k_src; g.v_src = spans[i].v_src;
    g.src_stride_layer = spans[i].src_stride_layer; g.src_stride_head = spans[i].src_stride_head;
    g.src_stride_token = spans[i].src_stride_token;
    g.len = spans[i].len; g.old_start = 0; g.new_start = 0;          // delta = 0: K rows are byte copies
    g.dst_seq = spans[i].dst_seq; g.dst_token_start = spans[i].dst_token_start;
  }
  return kvr_reposition_splice(c, dst, segs.data(), n, cuda_stream);
}

kvr_status kvr_last_device_status(kvr_ctx* c, int32_t* bad_segment, int32_t* bad_token) {
  if (!c) return KVR_ERR_INVALID_ARG;
  int prev = 0;
  cudaGetDevice(&prev);
  if (prev != c->device) cudaSetDevice(c->device);
  cudaError_t e = cudaMemcpyAsync(c->h_status, c->d_status, 4 * sizeof(int32_t), cudaMemcpyDeviceToHost, c->last_stream);
  if (e == cudaSuccess) e = cudaMemsetAsync(c->d_status, 0, 4 * sizeof(int32_t), c->last_stream);
  if (e == cudaSuccess) e = cudaStreamSynchronize(c->last_stream);
  if (prev != c->device) cudaSetDevice(prev);
  if (e != cudaSuccess) return c->cuda_fail(e, "kvr_last_device_status");
  if (c->h_status[0] == 0) return KVR_OK;
  if (bad_segment) *bad_segment = c->h_status[1];
  if (bad_token) *bad_token = c->h_status[2];
  return KVR_ERR_OUT_OF_RANGE;
}

uint64_t kvr_launch_count(const kvr_ctx* c) { return c ? c->launches : 0; }

kvr_status kvr_last_launch_info(const kvr_ctx* c, int32_t* path, int32_t* grid, int32_t* block, int32_t* smem) {
  if (!c) return KVR_ERR_INVALID_ARG;
  if (path) *path = c->last_path;
  if (grid) *grid = c->last_grid;
  if (block) *block = c->last_block;
  if (smem) *smem = c->last_smem;
  return KVR_OK;
}

const char* kvr_status_string(kvr_status s) {
  switch (s) {
    case KVR_OK: return "KVR_OK";
    case KVR_ERR_INVALID_ARG: return "KVR_ERR_INVALID_ARG";
    case KVR_ERR_UNSUPPORTED: return "KVR_ERR_UNSUPPORTED";
    case KVR_ERR_ALIGNMENT: return "KVR_ERR_ALIGNMENT";
    case KVR_ERR_OUT_OF_RANGE: return "KVR_ERR_OUT_OF_RANGE";
    case KVR_ERR_CUDA: return "KVR_ERR_CUDA";
    case KVR_ERR_NOMEM: return "KVR_ERR_NOMEM";
  }
  return "KVR_ERR_UNKNOWN";
}

const char* kvr_last_cuda_error(const kvr_ctx* c) { return c ? c->last_err.c_str() : ""; }

const char* kvr_version(void) { return "kvr 0.1 (sm_100a)"; }

}  // extern "C"

// ---- reposition + splice for callers that must not allocate (kvr.h: kvr_reposition_splice_noalloc) ----
// Everything a context keeps in device memory for this path, in one array that belongs to the library's device image
// (one copy per GPU that loads the library, alive until the process exits).  Layout = NoAllocScratch below.
namespace {

constexpr int kNoAllocMaxPairs = KVR_NOALLOC_MAX_ROTARY_DIM / 2;
struct NoAllocScratch {
  unsigned long long sched[4];      // ring kernel: next unit, finished CTAs (zero when a launch starts)
  int32_t status[4];                // sticky {flag, segment, token, -} when the caller passes no device_status
  int32_t pad_[4];
  double inv_freq[kNoAllocMaxPairs];
};
constexpr size_t kNoAllocHeaderBytes = 64;   // sched + status + pad_: what every call clears
static_assert(offsetof(NoAllocScratch, inv_freq) == kNoAllocHeaderBytes, "header is 64 bytes");
static_assert(sizeof(NoAllocScratch) <= KVR_NOALLOC_SCRATCH_BYTES, "kvr.h states the size of the array");

// In HOST code this name is only a handle for cudaGetSymbolAddress: it is not a device address and must never be given
// to a kernel or a cudaMemcpy as one.  noalloc_device_state() asks the runtime for the real address, once per device.
static __device__ __align__(256) unsigned char g_noalloc_scratch[KVR_NOALLOC_SCRATCH_BYTES];

struct NoAllocDevice {
  bool ready = false;
  unsigned char* base = nullptr;    // device address of g_noalloc_scratch on this device
  kvr_ctx* ctx = nullptr;           // host-only bookkeeping (owns no CUDA resource); its device pointers aim into `base`
};
constexpr int kNoAllocMaxDevices = 64;
NoAllocDevice g_noalloc_dev[kNoAllocMaxDevices];
std::mutex g_noalloc_mu;

kvr_status noalloc_fail(kvr_status st, char* err, int32_t err_len, const char* fmt, long long a = 0, long long b = 0) {
  if (err && err_len > 0) std::snprintf(err, (size_t)err_len, fmt, a, b);
  return st;
}

// Set-up, once per device, with that device current (the caller holds g_noalloc_mu and a DeviceGuard).
kvr_status noalloc_device_state(int dev, NoAllocDevice** out, char* err, int32_t err_len) {
  NoAllocDevice& d = g_noalloc_dev[dev];
  if (!d.ready) {
    int major = 0, sms = 0;
    cudaError_t e = cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    if (e != cudaSuccess) {
      (void)cudaGetLastError();
      return noalloc_fail(KVR_ERR_CUDA, err, err_len, "kvr_reposition_splice_noalloc: cannot query device %lld (CUDA error %lld)", dev, (long long)e);
    }
    if (major != 10)
      return noalloc_fail(KVR_ERR_UNSUPPORTED, err, err_len, "kvr_reposition_splice_noalloc: device %lld has compute capability %lld.x; the library is built for sm_100a", dev, major);
    void* p = nullptr;
    e = cudaGetSymbolAddress(&p, g_noalloc_scratch);
    if (e != cudaSuccess || !p) {
      (void)cudaGetLastError();
      return noalloc_fail(KVR_ERR_CUDA, err, err_len, "kvr_reposition_splice_noalloc: cudaGetSymbolAddress failed on device %lld (CUDA error %lld)", dev, (long long)e);
    }
    if (!d.ctx) d.ctx = new (std::nothrow) kvr_ctx();
    if (!d.ctx) return noalloc_fail(KVR_ERR_NOMEM, err, err_len, "kvr_reposition_splice_noalloc: out of host memory");
    d.base = static_cast<unsigned char*>(p);
    d.ctx->device = dev;
    d.ctx->sm_count = sms;
    d.ctx->d_sched = reinterpret_cast<unsigned long long*>(d.base + offsetof(NoAllocScratch, sched));
    d.ctx->d_inv_freq = reinterpret_cast<double*>(d.base + offsetof(NoAllocScratch, inv_freq));
    d.ready = true;
  }
  *out = &d;
  return KVR_OK;
}

}  // namespace

extern "C" {

kvr_status kvr_reposition_splice_noalloc(const kvr_model_desc* model, int cuda_device, const kvr_paged_dst* dst,
                                         const kvr_segment* segs, int32_t n, int32_t* device_status, void* cuda_stream,
                                         char* err, int32_t err_len) {
  if (err && err_len > 0) err[0] = 0;
  // ---- host-only checks: nothing below this block runs unless the call fits the fixed array ----
  kvr_status st = check_call(model, dst, segs, n);
  if (st == KVR_OK && n > 0) st = check_deltas(segs, n);
  if (st != KVR_OK) return noalloc_fail(st, err, err_len, "kvr_reposition_splice_noalloc: invalid arguments (see kvr_validate)");
  if (n > KVR_NOALLOC_MAX_SEGMENTS)
    return noalloc_fail(KVR_ERR_UNSUPPORTED, err, err_len,
                        "kvr_reposition_splice_noalloc: %lld segments, but a call without allocations carries at most %lld "
                        "(KVR_NOALLOC_MAX_SEGMENTS); split the call", n, KVR_NOALLOC_MAX_SEGMENTS);
  if (model->rotary_dim > KVR_NOALLOC_MAX_ROTARY_DIM)
    return noalloc_fail(KVR_ERR_UNSUPPORTED, err, err_len,
                        "kvr_reposition_splice_noalloc: rotary_dim %lld, but the fixed device array has room for %lld "
                        "(KVR_NOALLOC_MAX_ROTARY_DIM)", model->rotary_dim, KVR_NOALLOC_MAX_ROTARY_DIM);
  if (device_status && (reinterpret_cast<uintptr_t>(device_status) & 3u))
    return noalloc_fail(KVR_ERR_ALIGNMENT, err, err_len, "kvr_reposition_splice_noalloc: device_status is not 4-byte aligned");
  if (cuda_device < 0 || cuda_device >= kNoAllocMaxDevices)
    return noalloc_fail(KVR_ERR_INVALID_ARG, err, err_len, "kvr_reposition_splice_noalloc: cuda_device %lld out of range", cuda_device);
  if (n == 0) return KVR_OK;

  std::lock_guard<std::mutex> lock(g_noalloc_mu);      // orders the HOST side only; GPU work of overlapping calls races (kvr.h)
  int count = 0;
  if (cudaGetDeviceCount(&count) != cudaSuccess || cuda_device >= count) {
    (void)cudaGetLastError();
    return noalloc_fail(KVR_ERR_CUDA, err, err_len, "kvr_reposition_splice_noalloc: no CUDA device %lld (there is no CPU fallback)", cuda_device);
  }
  DeviceGuard guard(cuda_device);
  NoAllocDevice* d = nullptr;
  if ((st = noalloc_device_state(cuda_device, &d, err, err_len)) != KVR_OK) return st;
  kvr_ctx* c = d->ctx;
  cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
  c->last_err.clear();
  c->model = *model;                       // inv_freq stays the caller's HOST pointer: only the copy below reads it
  c->tuning = kvr_tuning{};
  c->d_status = device_status ? device_status : reinterpret_cast<int32_t*>(d->base + offsetof(NoAllocScratch, status));

  // The array keeps whatever the last call left: the counters and the status word must be zero when the kernel starts.
  cudaError_t e = cudaMemsetAsync(d->base, 0, kNoAllocHeaderBytes, stream);
  if (e == cudaSuccess && device_status) e = cudaMemsetAsync(device_status, 0, 4 * sizeof(int32_t), stream);
  if (e == cudaSuccess)
    e = cudaMemcpyAsync(c->d_inv_freq, model->inv_freq, (size_t)(model->rotary_dim / 2) * sizeof(double),
                        cudaMemcpyHostToDevice, stream);
  if (e != cudaSuccess) {
    (void)cudaGetLastError();
    return noalloc_fail(KVR_ERR_CUDA, err, err_len, "kvr_reposition_splice_noalloc: staging the scratch array failed (CUDA error %lld)", (long long)e);
  }
  // n <= kInlineSegs: enqueue_layers builds the descriptors in c->inline_scratch (host) and passes them in the kernel
  // parameters; it touches no staging slot and allocates nothing.
  static_assert(KVR_NOALLOC_MAX_SEGMENTS <= kInlineSegs, "descriptors must fit the kernel parameters");
  st = enqueue_layers(c, dst, segs, n, stream, 0, model->layers, false);
  if (st != KVR_OK && err && err_len > 0) std::snprintf(err, (size_t)err_len, "kvr_reposition_splice_noalloc: %s", c->last_err.c_str());
  return st;
}

}  // extern "C"
