/*
 * kvr.h -- C ABI of the kvr library: RoPE REPOSITIONING + SPLICE of precompiled
 * key/value segments into a paged KV cache, on one NVIDIA B200 (sm_100a).
 *
 * The operation is the data-parallel hot path behind the "composable" KV cache of
 * arxiv/paper_2606_17107 ("Models Take Notes at Prefill: KV Cache Can Be Editable and
 * Composable").  PAPER.md = the paper text; line numbers refer to it.
 *
 *   PAPER.md:131 (sec. 5): "we precompile a long skill ... and because the attention library
 *     caches post-RoPE keys, we re-rotate the chunk's keys from their source positions to the
 *     target positions (values are position-free) before concatenating (Figure 4b)."
 *   PAPER.md:393 (App. B): "The skill is prefilled once in isolation (positions 0..L-1), its keys
 *     re-rotated to the target offset, and spliced after the system prompt".
 *   PAPER.md:143 (sec. 5): "transplant is O(L) (a re-rotation pass plus the suffix)".
 *   PAPER.md:528 (App. H): the memory chunk is "RoPE-repositioned ... each turn (an O(L_mem)
 *     re-rotation, no re-prefill)".
 *   PAPER.md:209 (sec. 8): the operation is compatible with "paged attention/vLLM, and GQA/MQA".
 *
 * For every spliced segment s, layer l, kv head h and token t in [0, len_s):
 *     Delta_t = new_start - old_start            (or pos_map[t] - (old_start + t) if pos_map)
 *     for each rotary pair i < rotary_dim/2, with phi = Delta_t * inv_freq[i]:
 *         (ia, ib) = (i, i + rotary_dim/2)  [KVR_PAIR_NEOX_HALF]  or  (2i, 2i+1)  [KVR_PAIR_GPTJ_INTERLEAVED]
 *         K'[ia] = K[ia] cos(phi) - K[ib] sin(phi) ;  K'[ib] = K[ib] cos(phi) + K[ia] sin(phi)
 *     dims [rotary_dim, head_dim) of K and all of V are copied unchanged
 *     j = dst_token_start + t ; blk = block_table[dst_seq][j / block_size] ; off = j % block_size
 *     K', V are written at element offset  l*stride_layer + blk*stride_block + off*stride_token + h*stride_head
 * Delta_t == 0 copies the K row byte for byte.  In KVR_FP8_E4M3 mode K is dequantised with the
 * source scale, rotated, and requantised (round-to-nearest-even, saturating to +-448) with the
 * destination scale; where the two scales of a (layer, head) are the same number they cancel exactly
 * ((q s cos - q' s sin) / s = q cos - q' sin) and every kernel rotates the e4m3 codes as they are.
 * V bytes are always copied unchanged.
 *
 * Every step above runs in hand-written CUDA kernels; there is no CPU fallback.  All entry points
 * return kvr_status and never throw.  Nothing here synchronises the device except where stated.
 */
#ifndef KVR_H_
#define KVR_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define KVR_API __attribute__((visibility("default")))

typedef struct kvr_ctx kvr_ctx; /* opaque; owned by the library */

typedef enum {
  KVR_OK = 0,
  KVR_ERR_INVALID_ARG = -1,  /* NULL pointer, bad enum, odd rotary_dim, len <= 0, dst_seq out of range ... */
  KVR_ERR_UNSUPPORTED = -2,  /* valid but not implemented on this build / device (e.g. not sm_100)          */
  KVR_ERR_ALIGNMENT = -3,    /* a base pointer or stride is not a multiple of 16 bytes                     */
  KVR_ERR_OUT_OF_RANGE = -4, /* segment runs past its block-table row; device: bad block-table entry        */
  KVR_ERR_CUDA = -5,         /* a CUDA runtime call failed (see kvr_last_cuda_error)                        */
  KVR_ERR_NOMEM = -6
} kvr_status;

typedef enum { KVR_BF16 = 0, KVR_FP8_E4M3 = 1 } kvr_dtype;
typedef enum { KVR_PAIR_NEOX_HALF = 0, KVR_PAIR_GPTJ_INTERLEAVED = 1 } kvr_pairing;

/* Fixed per model.  inv_freq is a HOST array of rotary_dim/2 doubles, copied by kvr_create; the caller
 * applies any frequency scaling (standard theta^(-2i/R), llama3, YaRN ...; "RoPE [28] and
 * their extensions [25]").  rotary_dim is even, 2 <= rotary_dim, rotary_offset + rotary_dim <= head_dim
 * (partial rotary allowed).  head_dim * sizeof(element) must be a multiple of 16 bytes.
 *
 * Representation adapters (NEXT-3; Fig. 22), all expressed through this struct:
 *  - M-RoPE, "moving an image within a trajectory re-rotates only the temporal channels": give the height /
 *    width pairs inv_freq = 0 (their angle is then 0 for every Delta); sectioned and interleaved layouts differ
 *    only in WHICH entries are zero.
 *  - MLA, "repositioning re-rotates only k_pe and copies the latent as-is": a cached row is
 *    [latent c_t | k_pe]; set kv_heads = 1, head_dim = latent width + rope width, rotary_offset = latent width,
 *    rotary_dim = rope width.  Rotary pair i then is dims rotary_offset + (i, i + rotary_dim/2)  [NEOX_HALF] or
 *    rotary_offset + (2i, 2i+1)  [GPTJ_INTERLEAVED]; every dim outside the window is copied unchanged.  Such a
 *    cache has ONE tensor per token: pass v_cache = NULL in kvr_paged_dst and v_src = NULL in every segment
 *    ("K-only" call; all-or-none, else KVR_ERR_INVALID_ARG).
 * rotary_offset * sizeof(element) must be a multiple of 16 bytes. */
typedef struct {
  int32_t layers, kv_heads, head_dim, rotary_dim;
  int32_t pairing; /* kvr_pairing */
  int32_t dtype;   /* kvr_dtype   */
  const double* inv_freq;
  int32_t rotary_offset; /* first rotary dim of a row; 0 for ordinary K caches */
  int32_t reserved_;     /* must be 0 */
} kvr_model_desc;

/* Destination paged pool: caller-owned DEVICE memory.  K and V pools share the four element strides;
 * head_dim elements are contiguous.  Covers token-major ("NHD": stride_token = kv_heads*head_dim,
 * stride_head = head_dim) and head-major ("HND": stride_head = block_size*head_dim, stride_token =
 * head_dim) block layouts, with the layer dimension outside or inside the block dimension.
 * block_table is a DEVICE array [num_seqs][max_blocks_per_seq] of physical block ids; an entry the call
 * touches that is < 0 or >= num_blocks makes the kernel skip that token range and raise the sticky
 * device status (kvr_last_device_status).  k_scale: DEVICE [layers*kv_heads] fp32 destination K scales,
 * KVR_FP8_E4M3 only (NULL otherwise). */
typedef struct {
  void* k_cache;
  void* v_cache;
  int64_t stride_layer, stride_block, stride_token, stride_head; /* elements */
  int32_t num_blocks, block_size;
  const int32_t* block_table;
  int32_t num_seqs, max_blocks_per_seq;
  const float* k_scale;
} kvr_paged_dst;

/* One spliced segment.  The ARRAY of segments lives on the HOST and is copied before the call returns.
 * k_src / v_src: DEVICE, logical [layers][kv_heads][len][head_dim] addressed by the three element
 * strides (head_dim contiguous).  delta = new_start - old_start (any sign).  Token t is written to logical
 * token dst_token_start + t of block-table row dst_seq (slots are dense; positions only set angles).
 * pos_map: DEVICE int32 [len] or NULL; if given, token t moves to position pos_map[t], i.e.
 * delta_t = pos_map[t] - (old_start + t), and new_start is ignored.
 * k_scale_src: DEVICE fp32 [layers*kv_heads] source K scales (fp8 only); NULL = same as destination.
 * Two segments that write the same slot, or a source that aliases the destination, are undefined. */
/* flags: KVR_SEG_PRE_ROPE (NEXT-4, "splice fused with the suffix-prefill KV write"; "TTFT is a
 * re-rotation pass plus the suffix"): the segment's keys are not yet position-encoded -- the suffix keys a model has
 * just projected -- i.e. EVERY source token sits at position old_start (0 for plain pre-RoPE keys: RoPE at 0 is the
 * identity) and token t goes to its target position new_start + t (or pos_map[t]): delta_t = target_t - old_start.
 * One kvr_reposition_splice call can thus carry the spliced skills (delta per segment), repaired seam tokens
 * (delta = 0) and the fresh suffix (RoPE applied on the way into the cache): K is never materialised twice. */
#define KVR_SEG_PRE_ROPE 1
/* KVR_SEG_SRC_STABLE: a promise about ordering, never about results.  The segment's k_src / v_src bytes are not written
 * by any work enqueued on `cuda_stream` before this call -- the normal state of a PRECOMPILED skill ("we
 * precompile a long skill", :393 "prefilled once in isolation"), unlike suffix keys a kernel has just produced.  The
 * kernels are launched with programmatic dependent launch; with this flag a CTA may start READING the segment's
 * sources while the previous kernel on the stream is still draining (nothing is written, and the block table, position
 * maps and scales are only read, before that kernel has completed).  Setting it on sources that earlier work on the
 * stream does write is a data race.  Ignored by kvr_reposition_splice_host. */
#define KVR_SEG_SRC_STABLE 2
typedef struct {
  const void* k_src;
  const void* v_src;
  int64_t src_stride_layer, src_stride_head, src_stride_token; /* elements */
  int32_t len, old_start, new_start;
  int32_t dst_seq, dst_token_start;
  int32_t flags; /* 0 or an OR of KVR_SEG_* (occupies what used to be padding: the struct size is unchanged) */
  const int32_t* pos_map;
  const float* k_scale_src;
} kvr_segment;

/* Optional tuning knobs (0 = library default).  Never changes results, only the launch shape. */
typedef struct {
  int32_t path;            /* 0 auto, 1 force the scalar generic kernel, 2 force the TMA-ring kernel, 5 force the generic kernel with 16-byte accesses */
  int32_t ctas_per_sm;     /* persistent CTAs per SM for the ring kernel                       */
  int32_t consumer_warps;  /* consumer warps per CTA                                           */
  int32_t stages;          /* ring depth (tiles in flight per CTA)                             */
  int32_t layers_per_unit; /* layers one scheduled unit covers                                  */
  int32_t v_bulk_store;    /* 0 auto, 1 V leaves shared memory by bulk (TMA) stores, 2 by warps, 3 one bulk store per row */
  int32_t max_ctas;        /* cap on the persistent grid (tests use it to force many tiles per CTA)  */
  int32_t grab;            /* units a CTA draws from the dynamic scheduler per atomic (1..32)               */
  int32_t pdl;             /* programmatic dependent launch of the ring kernel: 0 auto (on), 1 on, 2 off            */
  int32_t hsplit;          /* split a unit's heads into this many units (finer tail); 0 auto                        */
  int32_t chunk_tokens;    /* ring kernel: upper bound on the tokens of a chunk (default 16); the chunk is the largest
                              divisor of block_size below it                                                          */
  int32_t tile_bytes;      /* ring kernel: a tile takes the fewest heads whose K run reaches this size (default 4096) */
  int32_t gather;          /* ring kernel, dense token-major pools: tiles of all heads x few tokens, several consumer
                              warps per tile (see kvr_ring.cu): 0 auto, 1 on, 2 off, 3 on with K and V in tiles of their own                            */
  int32_t warps_per_stage; /* gather mode: consumer warps that share one stage (default: all of them)                  */
  int32_t lanes_over_heads; /* gather mode: a warp pass covers several HEADS of one token (adjacent rows of a dense
                              token-major pool) instead of several tokens of one head: 0 auto, 1 on, 2 off */
  int32_t transpose_load;  /* dense token-major pools: tiles of all heads x few tokens loaded by TMA tensor maps whose
                              dimension order transposes them into the pool's order on the way in: 0 auto, 1 on, 2 off */
} kvr_tuning;

/* Creates a context on CUDA device `cuda_device` (must be compute capability 10.x).  Allocates a few
 * hundred KB of device and pinned host memory (descriptor staging, status word).  Synchronous. */
KVR_API kvr_status kvr_create(kvr_ctx** out, const kvr_model_desc* model, int cuda_device);
KVR_API kvr_status kvr_destroy(kvr_ctx* ctx); /* synchronises the device; NULL is a no-op */
KVR_API kvr_status kvr_set_tuning(kvr_ctx* ctx, const kvr_tuning* t); /* NULL restores defaults */

/* Host-only validation of one call's arguments (no CUDA call is made; usable without a GPU).
 * Returns the status kvr_reposition_splice would return before launching anything. */
KVR_API kvr_status kvr_validate(const kvr_model_desc* model, const kvr_paged_dst* dst,
                                const kvr_segment* segs, int32_t n_segs);

/* THE HOT PATH.  Enqueues, on `cuda_stream` (a cudaStream_t; NULL = the legacy
 * default stream), the reposition + splice of n_segs segments into dst.  Asynchronous: returns once the
 * work is enqueued; there is no device synchronisation.  Host-detectable faults are rejected before any
 * launch and leave the destination untouched.  Calls on one context must be issued to one stream at a
 * time (the context owns per-call staging).  Every destination byte not addressed keeps its value.
 * CUDA graphs: a call with at most 8 segments carries its descriptors in the kernel parameters, enqueues nothing
 * but its kernel and may be captured (stream capture) and replayed; the pointers it was given must stay valid for
 * every replay.  A call with more than 8 segments stages its descriptors through context-owned pinned memory that
 * later calls reuse, so under capture it is refused with KVR_ERR_UNSUPPORTED before anything is enqueued (split it
 * into calls of <= 8 segments to capture it).  The same rule holds for kvr_reposition_inplace and kvr_write_span
 * (spans); kvr_reposition_splice_host is never capturable. */
KVR_API kvr_status kvr_reposition_splice(kvr_ctx* ctx, const kvr_paged_dst* dst, const kvr_segment* segs,
                                         int32_t n_segs, void* cuda_stream);

/* The same operation with HOST-resident sources (a library of precompiled skills kept in host RAM,
 * PAPER.md:131 "we precompile a long skill", :393 "prefilled once in isolation"): every segment's k_src,
 * v_src, pos_map and k_scale_src are HOST pointers; dst (pools, block_table, k_scale) stays DEVICE memory.
 * Sources must be dense [layers][kv_heads][len][head_dim] (else KVR_ERR_UNSUPPORTED) and should be pinned
 * (cudaHostAlloc / cudaHostRegister); pageable memory works but makes the copies synchronous.  The library
 * stages groups of layers through two context-owned device buffers (allocated on first use, <= ~256 MB
 * each, or one layer if that is larger): the host->device copies of group g+1 run on a context-owned copy
 * stream while the kernel of group g runs on `cuda_stream`.  Returns when everything is enqueued; the host
 * buffers must stay valid and unchanged until `cuda_stream` has passed this call.  Not capturable in a CUDA
 * graph.  kvr_last_h2d_bytes reports the bytes the last such call copied host -> device. */
KVR_API kvr_status kvr_reposition_splice_host(kvr_ctx* ctx, const kvr_paged_dst* dst, const kvr_segment* segs,
                                              int32_t n_segs, void* cuda_stream);
KVR_API uint64_t kvr_last_h2d_bytes(const kvr_ctx* ctx);

/* ---- The hot path for callers that must not allocate ------------------------------------------------------
 * kvr_create, and now and then the calls above, reserve device and pinned memory (cudaMalloc / cudaMallocHost).
 * Some hosts of this library cannot let that happen:
 *   - a serving engine that sized its KV pool to whatever HBM was left at start-up: a later cudaMalloc of even a
 *     few KB can fail there, and the engine's memory accounting would not see it if it succeeded;
 *   - a process in which some thread is recording a CUDA graph in the default (global) capture mode: cudaMalloc
 *     from ANY thread then fails and invalidates that recording;
 *   - a latency-critical step that cannot afford the device-wide synchronisation cudaMalloc / cudaFree may imply;
 *   - a plug-in loaded under an allocator policy ("all device memory comes from the host application's pool") that
 *     forbids driver allocations outright.
 * For them: the same reposition + splice as kvr_reposition_splice -- same validation, same kernels, same results
 * bit for bit -- WITHOUT a context and without a single CUDA allocation (no cudaMalloc, cudaMallocHost, cudaFree,
 * stream or event creation).  What a context would hold on the device -- the unit scheduler's two counters, the
 * sticky status word and the model's inv_freq table -- lives in ONE fixed array of KVR_NOALLOC_SCRATCH_BYTES bytes
 * that is part of the library's device image: every GPU that loads the library carries it until the process exits,
 * whether or not this call is ever made.
 * Limits, rejected with KVR_ERR_UNSUPPORTED and a message in `err` before anything is enqueued:
 *   n_segs <= KVR_NOALLOC_MAX_SEGMENTS (the descriptors then travel in the kernel parameters; split larger calls),
 *   model->rotary_dim <= KVR_NOALLOC_MAX_ROTARY_DIM (room for its inv_freq in the array).
 * Arguments: model / dst / segs / n_segs / cuda_stream as for kvr_create + kvr_reposition_splice (library default
 * tuning); cuda_device = the device that owns every pointer and the stream.  device_status: NULL, or DEVICE int32[4]
 * that this call zeroes and the kernel then fills if it meets a bad block-table entry ([0] != 0, [1] = segment,
 * [2] = token; those tokens are skipped) -- read it after the stream has passed the call; with NULL the word stays
 * in the array and is dropped.  err / err_len: NULL / 0, or a HOST buffer that receives a 0-terminated message
 * whenever the result is not KVR_OK.
 * First call on a device: looks up the array's device address (this can make the CUDA runtime load the library's
 * device code), so make that call outside any stream capture; a one-token splice into a spare block will do.
 * Every call: enqueues, on cuda_stream, a 64-byte clear of the counters and status word, a copy of inv_freq
 * (rotary_dim/2 doubles, from pageable host memory: it is consumed before the call returns), and the kernel.
 * Sharing: all calls on one device use the same array, and each one overwrites what the previous left there.  Calls
 * on ONE stream are ordered and safe.  Two calls that can overlap on the GPU (different streams without an event
 * between them, or two host threads' streams) race on the counters and the table and give undefined results; the
 * host side is serialised by a lock, which does not order the GPU work. */
#define KVR_NOALLOC_MAX_SEGMENTS 8
#define KVR_NOALLOC_MAX_ROTARY_DIM 1024
#define KVR_NOALLOC_SCRATCH_BYTES 4352
KVR_API kvr_status kvr_reposition_splice_noalloc(const kvr_model_desc* model, int cuda_device, const kvr_paged_dst* dst,
                                                 const kvr_segment* segs, int32_t n_segs, int32_t* device_status,
                                                 void* cuda_stream, char* err, int32_t err_len);

/* ---- NEXT-1: in-place reposition of a chunk that is ALREADY RESIDENT in the paged pool -------------------
 * PAPER.md:528 (App. H): "the user-memory chunk is precompiled once in isolation and RoPE-repositioned to float
 * just before the query each turn (an O(L_mem) re-rotation, no re-prefill)"; PAPER.md:167 (sec. 7).
 * A resident span is logical tokens [token_start, token_start + len) of block-table row `seq`.  Every K row of it
 * is rotated by delta = new_start - old_start (or, with pos_map (DEVICE int32 [len]), by
 * delta_t = pos_map[t] - (old_start + t)) exactly as in kvr_reposition_splice and written back to the slot it was
 * read from.  V is position-free and is neither read nor written: pool->v_cache may be NULL.
 * fp8: pool->k_scale is both the source and the destination scale.  delta_t == 0 leaves the row's bytes alone.
 * Traffic is 2 * layers*kv_heads*head_dim*esz bytes per token (kvr_inplace_bytes_moved), half of a re-splice; with
 * rotary_offset != 0 (a [latent | k_pe] cache) only the rotary window is read and written: 2 * layers*kv_heads*
 * rotary_dim*esz bytes per token.
 * Spans of one call must not overlap (undefined).  Same asynchrony, validation and error rules as the splice:
 * host-detectable faults are rejected before any launch; an invalid block-table entry skips its tokens and
 * raises the sticky device status. */
typedef struct {
  int32_t seq, token_start, len;
  int32_t old_start, new_start;
  const int32_t* pos_map;
} kvr_resident_span;

KVR_API kvr_status kvr_reposition_inplace(kvr_ctx* ctx, const kvr_paged_dst* pool, const kvr_resident_span* spans,
                                          int32_t n_spans, void* cuda_stream);
KVR_API uint64_t kvr_inplace_bytes_moved(const kvr_model_desc* model, const kvr_resident_span* spans, int32_t n_spans);

/* ---- NEXT-2: span overwrite -----------------------------------------------------------------------------
 * PAPER.md:348 (App. B) / :112 (sec. 4): the field-only edit overwrites the KV of a short value span in place;
 * PAPER.md:141 (sec. 5) / :171 / :528: one (or a few) boundary tokens of a transplanted chunk are recomputed
 * ("seam repair").  Producing the new K/V needs a model and is the caller's business; writing them into the paged
 * pool is this call: K and V rows k_src / v_src (DEVICE, logical [layers][kv_heads][len][head_dim], element
 * strides as in kvr_segment; K already RoPE'd at its final positions) are copied byte for byte to logical tokens
 * [dst_token_start, dst_token_start + len) of block-table row dst_seq.  It is the delta = 0 case of
 * kvr_reposition_splice and runs through the same kernels. */
typedef struct {
  const void* k_src;
  const void* v_src;
  int64_t src_stride_layer, src_stride_head, src_stride_token; /* elements */
  int32_t len, dst_seq, dst_token_start;
} kvr_span;

KVR_API kvr_status kvr_write_span(kvr_ctx* ctx, const kvr_paged_dst* dst, const kvr_span* spans, int32_t n_spans,
                                  void* cuda_stream);

/* ---- NEXT-4, first alternative: ROTATE-ON-READ decode attention ---------------------------------------------
 * "fusing the rotate into a consumer (rotate-on-read in the attention K load ...) so K is never
 * materialised twice"; "we re-rotate the chunk's keys from their source positions to the target positions
 * (values are position-free)"; PAPER.md:143 (the pass is O(L)); PAPER.md:209 (works under FlashAttention / paged
 * attention, GQA/MQA).  DESIGN.md reading R25.
 * A decode-step query attends the cached keys and values of precompiled skills WHERE THEY LIE -- nothing is spliced,
 * nothing is written back.  For request r, query head g (kv head h = g / (q_heads / kv_heads)), over every token t of
 * every segment s with segs[s].request == r, at model layer `layer`:
 *     x_{s,t} = softmax_scale * sum_d q[r][g][d] * (R(delta_s) k_{s,t})[d]      R = the re-rotation of kvr_reposition_splice
 *     lse[r][g] = ln sum exp(x)            o[r][g][:] = sum exp(x_{s,t} - lse[r][g]) * v_{s,t}[:]
 * (o, lse) is the partial-attention pair the caller merges with its attention over the rest of the context.
 * q: DEVICE bf16 [n_req][q_heads][head_dim], the query as the model produced it (RoPE'd at its own position).
 * o: DEVICE fp32 [n_req][q_heads][head_dim]; lse: DEVICE fp32 [n_req][q_heads] (natural logarithm).
 * Arithmetic: the kernel uses q . R(delta) k = (R(-delta) q) . k: the counter-rotated query is evaluated in fp64 and
 * rounded once to bf16; both contractions run on the tensor cores (bf16 operands, fp32 accumulation), the softmax
 * weights are rounded to bf16 before they multiply V and their row sum adds the rounded weights.
 * Limits (else KVR_ERR_UNSUPPORTED): KVR_BF16 caches, head_dim == 128, q_heads / kv_heads <= 16.  Every request must
 * own at least one segment; k_src / v_src as in kvr_segment (DEVICE, [layers][kv_heads][len][head_dim], element strides,
 * 16-byte aligned).  Asynchronous on `cuda_stream`; descriptors (TMA tensor maps, work items) are built on the host,
 * staged through context-owned pinned memory and CACHED per distinct segment array (8 entries, least recently used
 * replaced): a decode loop that reads the same skills at every step and layer enqueues nothing but its kernels from
 * the second call on.  CUDA graphs: a call whose descriptors are cached (it has been issued once eagerly with the same
 * segment array and its buffers have not grown since) enqueues nothing but kernels and may be captured and replayed
 * with other q / o / lse / layer arguments per node; its cache entry is then pinned until kvr_destroy.  Any other call
 * is refused under capture with KVR_ERR_UNSUPPORTED before anything is enqueued.  One or two kernels per
 * call (the second merges the partial results of (request, kv head) groups that were split over many CTAs).  Reads
 * 2 * kv_heads * head_dim * 2 bytes per token (kvr_attention_bytes_read): K and V of one layer, once.  Outputs are
 * written only by this call's kernels; partial results live in context-owned device memory, so calls on one context
 * must be issued to one stream at a time (as for every other call).  Changing streams between calls: an eager call
 * that finds its descriptors cached but was issued on another stream than the previous one first waits (on the
 * device) for that stream's call; a CAPTURED call cannot do so, so capture on the stream of the eager call or
 * synchronise that stream before the capture begins. */
typedef struct {
  const void* k_src;
  const void* v_src;
  int64_t src_stride_layer, src_stride_head, src_stride_token; /* elements */
  int32_t len;
  int32_t delta;   /* new_start - old_start: where the skill sits in this request's context minus where it was compiled */
  int32_t request; /* row of q / o / lse that attends this segment */
  int32_t flags;   /* 0 or KVR_SEG_SRC_STABLE (as in kvr_segment: the K / V loads may then overlap the previous kernel's tail) */
} kvr_read_segment;

KVR_API kvr_status kvr_rotate_on_read_attention(kvr_ctx* ctx, const void* q, int32_t n_req, int32_t q_heads, int32_t layer,
                                                float softmax_scale, const kvr_read_segment* segs, int32_t n_segs,
                                                float* o, float* lse, void* cuda_stream);
KVR_API uint64_t kvr_attention_bytes_read(const kvr_model_desc* model, const kvr_read_segment* segs, int32_t n_segs);
/* Host-only validation of a kvr_rotate_on_read_attention call (no CUDA call is made; usable without a GPU): the status
 * the call returns before it enqueues anything (pointers are only checked for NULL and alignment; what a TMA tensor
 * map cannot describe -- a zero layer stride with layers > 1, a stride of 2^40 bytes or more -- is
 * KVR_ERR_UNSUPPORTED; n_req > n_segs is KVR_ERR_INVALID_ARG since every request must own a segment). */
KVR_API kvr_status kvr_validate_read(const kvr_model_desc* model, const void* q, int32_t n_req, int32_t q_heads, int32_t layer,
                                     float softmax_scale, const kvr_read_segment* segs, int32_t n_segs, const float* o,
                                     const float* lse);

/* Algorithmic bytes of a call: read K, read V, write K, write V = 4 * layers*kv_heads*head_dim*esz * sum(len)
 * (2 * ... for a K-only call, i.e. when segs[0].v_src == NULL).
 * This is the O(L) of PAPER.md:143 and the numerator of every GB/s this repository reports. */
KVR_API uint64_t kvr_bytes_moved(const kvr_model_desc* model, const kvr_segment* segs, int32_t n_segs);

/* Waits for the stream of the last call, then reports and clears the sticky device status:
 * KVR_OK, or KVR_ERR_OUT_OF_RANGE with the first offending segment index and token (either may be NULL). */
KVR_API kvr_status kvr_last_device_status(kvr_ctx* ctx, int32_t* bad_segment, int32_t* bad_token);

/* Introspection for benchmarks: kernels launched by this context so far; the kernel path the last call took
 * (1 generic, 2 TMA ring, 3 rotate-on-read attention, 4 window in place, 5 generic with 16-byte accesses); grid size, CTA size and dynamic shared memory of its main kernel. */
KVR_API uint64_t kvr_launch_count(const kvr_ctx* ctx);
KVR_API kvr_status kvr_last_launch_info(const kvr_ctx* ctx, int32_t* path, int32_t* grid, int32_t* block,
                                        int32_t* smem_bytes);

KVR_API const char* kvr_status_string(kvr_status s);
KVR_API const char* kvr_last_cuda_error(const kvr_ctx* ctx); /* "" if none; valid until the next call */
KVR_API const char* kvr_version(void);

#ifdef __cplusplus
}
#endif
#endif /* KVR_H_ */
